"""Pins of the oracle's Balloon-Windkessel read-out (Extended Data Table 4; reading R30) against what
the mathematics fixes: the resting fixed point, the steady state under constant activity, the closed form of the
linear (s, f) subsystem, a quadrature of the autonomous volume equation, and the linear q equation.  CPU only."""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle as orc

P = dict(orc.BOLD_DEFAULTS)


def _run(z, T, h, state=None):
    st = orc.bold_rest(1) if state is None else np.array(state, np.float64).reshape(1, 4)
    out = [st[0].copy()]
    for _ in range(int(round(T / h))):
        st = orc.bold_step(st, np.array([z]), h, P)
        out.append(st[0].copy())
    return np.array(out)


def test_rest_is_a_fixed_point_with_zero_signal():
    tr = _run(0.0, 5.0, 1e-3)
    assert np.all(tr[:, 0] == 0.0) and np.all(tr[:, 1:] == 1.0)
    assert np.all(orc.bold_signal(tr, P) == 0.0)


@pytest.mark.parametrize("z", [0.05, 0.4, 1.5])
def test_steady_state_under_constant_activity(z):
    # s* = 0, f* = 1 + z / gamma, v* = f*^alpha, q* = v* E(f*, rho) / rho
    tr = _run(z, 120.0, 2e-3)
    f = 1.0 + z / P["gamma"]
    v = f ** P["alpha"]
    q = v * (1.0 - (1.0 - P["rho"]) ** (1.0 / f)) / P["rho"]
    assert np.allclose(tr[-1], [0.0, f, v, q], rtol=0, atol=1e-9)
    y = P["V0"] * (P["k1"] * (1 - q) + P["k2"] * (1 - q / v) + P["k3"] * (1 - v))
    assert abs(orc.bold_signal(tr[-1], P) - y) < 1e-10
    assert y > 0                                              # activation raises the signal


def test_flow_subsystem_follows_the_damped_oscillator_closed_form():
    # s' = z - kappa s - gamma (f - 1), f' = s is linear: f - 1 = (z / gamma)(1 - e^(-kappa t / 2)(cos wt + kappa / (2w) sin wt))
    z, T = 0.7, 20.0
    w = math.sqrt(P["gamma"] - P["kappa"] ** 2 / 4)
    errs = []
    for h in (2e-3, 1e-3):
        tr = _run(z, T, h)
        t = np.arange(len(tr)) * h
        env = np.exp(-P["kappa"] * t / 2)
        f = 1 + z / P["gamma"] * (1 - env * (np.cos(w * t) + P["kappa"] / (2 * w) * np.sin(w * t)))
        s = z / w * env * np.sin(w * t)
        errs.append(max(np.abs(tr[:, 1] - f).max(), np.abs(tr[:, 0] - s).max()))
    assert errs[1] < 2e-3 and 1.8 < errs[0] / errs[1] < 2.2  # explicit Euler: first order


def test_volume_equation_matches_quadrature_of_its_inverse():
    # hold the inflow at f0 (s = 0, z = gamma (f0 - 1)): tau v' = f0 - v^(1/alpha) is autonomous, so the time to go
    # from v0 to v1 is tau * integral dv / (f0 - v^(1/alpha))
    f0, h = 1.6, 2e-4
    z = P["gamma"] * (f0 - 1)
    tr = _run(z, 3.0, h, state=[0.0, f0, 1.0, 1.0])
    assert np.all(np.abs(tr[:, 1] - f0) < 1e-12) and np.all(np.abs(tr[:, 0]) < 1e-12)
    for k in (500, 2500, 10000):
        v1 = tr[k, 2]
        t_quad, _ = integrate.quad(lambda v: P["tau"] / (f0 - v ** (1 / P["alpha"])), 1.0, v1)
        assert abs(t_quad - k * h) < max(3 * h, 1e-3 * k * h)     # Euler: O(h) in v, divided by a shrinking slope
    assert tr[-1, 2] < f0 ** P["alpha"] and tr[-1, 2] > 1.1


def test_deoxyhemoglobin_equation_is_linear_at_fixed_flow_and_volume():
    # f = f0, v = f0^alpha fixed: tau q' = a - b q with a = f0 E / rho, b = v^(1/alpha) / v = f0 / v
    f0, h = 1.4, 2e-4
    v0 = f0 ** P["alpha"]
    tr = _run(P["gamma"] * (f0 - 1), 2.0, h, state=[0.0, f0, v0, 1.0])
    assert np.all(np.abs(tr[:, 2] - v0) < 1e-12)
    a = f0 * (1 - (1 - P["rho"]) ** (1 / f0)) / P["rho"]
    b = f0 / v0
    t = np.arange(len(tr)) * h
    q = a / b + (1 - a / b) * np.exp(-b * t / P["tau"])
    assert np.abs(tr[:, 3] - q).max() < 1e-4
    assert abs(tr[-1, 3] - q[-1]) > 0 and q[-1] < 1.0


def test_bold_run_turns_counts_into_rates_per_region():
    # 2 regions of different size with the same rate give the same signal; the count -> Hz conversion is R24
    sizes = np.array([1000, 250])
    win_s = 1e-3
    counts = np.tile(np.array([[8, 2]]), (3000, 1))          # 8 Hz in both
    ys, st = orc.bold_run(counts, sizes, win_s, P)
    assert ys.shape == (3000, 2) and np.allclose(ys[:, 0], ys[:, 1], rtol=0, atol=1e-15)
    tr = _run(P["z_scale"] * 8.0, 3.0, win_s)
    assert np.allclose(st[0], tr[-1], rtol=0, atol=1e-12)
