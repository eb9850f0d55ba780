"""Pins of the per-neuron external current (SURVEY 8(f) row 1 remainder; "I_ext,i are parameters,
independently sampled following a Gamma distribution"; property table; reading R31 in DESIGN.md) against
scipy's Gamma quantile function, the moments of the law, the pinned Philox words and the closed form of the membrane
equation under a constant current.  CPU only."""
import math

import numpy as np
import pytest
from scipy import stats

import db_inputs


def _lone(oracle_mod, N, types, ntype=None, seed=5, fp64=True, dt=0.1):
    sim = db_inputs.sim_params(dt_ms=dt, types=types)
    net = dict(N=N, n_regions=1, region_start=np.array([0, N]), ntype=np.zeros(N, np.uint8) if ntype is None else ntype,
               row_ptr=np.zeros(N + 1, np.int64), tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32),
               delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))
    return oracle_mod.OracleSim(sim, net, seed=seed, fp64=fp64)


@pytest.mark.parametrize("shape,scale", [(2.0, 0.1), (0.5, 0.3), (9.0, 0.02), (1.0, 1.0), (40.0, 0.005)])
def test_gamma_quantile_table_matches_scipy(oracle_mod, shape, scale):
    tab = oracle_mod.gamma_table(shape, scale)
    q = (np.arange(65536) + 0.5) / 65536.0
    want = stats.gamma.ppf(q, shape, scale=scale)
    assert np.all(np.abs(tab - want) <= 1.2e-7 * want + 1e-30)          # one fp32 rounding
    assert np.all(np.diff(tab) >= 0) and tab[0] >= 0
    for p in (1e-9, 0.003, 0.5, 0.97, 1 - 1.0 / 131072):                 # the table's own range of p
        assert abs(oracle_mod.lib().orc_gamma_ppf(p, shape, scale) - stats.gamma.ppf(p, shape, scale=scale)) \
            < 1e-10 * max(1.0, stats.gamma.ppf(p, shape, scale=scale))
    # midpoint rule over the quantiles reproduces the mean of the law, k theta
    assert abs(tab.astype(np.float64).mean() - shape * scale) < 2e-4 * shape * scale + 2e-5


@pytest.mark.parametrize("fp64", [True, False])
def test_external_currents_are_the_table_at_the_pinned_philox_words(oracle_mod, fp64):
    a = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    a.update(Iext=0.1, iext_gamma_shape=2.0, iext_gamma_scale=0.05)
    b = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    b.update(Iext=-0.2)                                                   # no Gamma part: the constant
    N, seed = 6001, 0xABCDEF0123456789
    ntype = (np.arange(N) % 4 == 1).astype(np.uint8)
    s = _lone(oracle_mod, N, [a, b], ntype=ntype, seed=seed, fp64=fp64)
    got = s.iext()
    tab = stats.gamma.ppf((np.arange(65536) + 0.5) / 65536.0, 2.0, scale=0.05).astype(np.float32)
    real = np.float64 if fp64 else np.float32
    draws = np.empty(N)
    for i in range(N):
        u = int(oracle_mod.philox([i, 9 << 24, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])[0])
        draws[i] = tab[u >> 16]
        want = real(-0.2) if ntype[i] else real(0.1) + real(tab[u >> 16])
        assert abs(got[i] - float(want)) <= 1.3e-7 * abs(float(want)), i      # (table entries: one fp32 ulp between two libms)
    x = draws[ntype == 0]
    k, th = 2.0, 0.05
    assert abs(x.mean() - k * th) < 4 * math.sqrt(k) * th / math.sqrt(len(x))
    assert abs(x.var() - k * th * th) < 0.12 * k * th * th
    assert stats.kstest(x, "gamma", args=(k, 0, th)).pvalue > 1e-3


def test_every_neuron_relaxes_to_the_fixed_point_of_its_own_current(oracle_mod):
    # sub-threshold constant current, no synapses: V_inf,i = VL + I_ext,i / gL and V_n = V_inf + (V_0 - V_inf)(1 - dt gL / C)^n
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    t.update(Iext=0.05, iext_gamma_shape=3.0, iext_gamma_scale=0.04, Vth=1e9)
    N = 300
    s = _lone(oracle_mod, N, [t, dict(t)])
    I = s.iext()
    assert I.min() >= 0.05 and I.std() > 0.03
    V0, g, ref = s.state()
    V0 = np.linspace(-80.0, -60.0, N)
    s.set_state(V0, g, ref)
    q = 1.0 - 0.1 * t["gL"] / t["C"]
    for n in (1, 17, 400):
        s.step(n - s.step_index)
        want = (t["VL"] + I / t["gL"]) + (V0 - (t["VL"] + I / t["gL"])) * q ** n
        assert np.max(np.abs(s.state()[0] - want)) < 1e-10
    assert np.array_equal(s.iext(), I)                                       # a parameter: it does not move


def test_zero_shape_means_the_constant_of_the_type(oracle_mod):
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    t.update(Iext=0.33)
    s = _lone(oracle_mod, 50, [t, dict(t)])
    assert np.all(s.iext() == 0.33)
