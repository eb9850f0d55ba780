"""Pins of the parts of the oracle's step that VERDICT round 1 found unpinned: the synaptic current of every
receptor (G_u g_u (E_u - V), P:L110 / P:L382; oracle step 4), which g the membrane step sees (R8, P:L475 / P:L479)
to the step, the V0 draw (R-RNG), and the fixed-point wrap with its sticky overflow flag (R28).  Every expected
value here is a closed form of the Euler map or an integer computed from the pinned Philox words -- nothing is
read from the oracle itself.  CPU only."""
import math

import numpy as np
import pytest

import db_inputs

# per-receptor-distinct gains and reversal potentials: a swap of two E's or two G's moves every fixed point below
G_DISTINCT = [1.3, 0.21, 0.77, 1.9]
E_DISTINCT = [3.0, -11.0, -68.0, -97.0]
TAU_FROZEN = 1e30            # exp(-dt / tau) == 1.0 to the last bit of fp64: the conductance is held constant


def _lone_neurons(oracle_mod, N, dt, types, fp64=True, seed=3, ntype=None):
    sim = db_inputs.sim_params(dt_ms=dt, types=types)
    net = dict(N=N, n_regions=1, region_start=np.array([0, N]), ntype=np.zeros(N, np.uint8) if ntype is None else ntype,
               row_ptr=np.zeros(N + 1, np.int64), tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32),
               delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))
    return oracle_mod.OracleSim(sim, net, seed=seed, fp64=fp64), sim


def _frozen_type(**kw):
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    t.update(G=list(G_DISTINCT), E=list(E_DISTINCT), tau_ms=[TAU_FROZEN] * 4, Vth=1e9)
    t.update(kw)
    return t


@pytest.mark.parametrize("dt", [0.1, 1.0])
@pytest.mark.parametrize("u", [0, 1, 2, 3])
def test_each_receptor_current_fixed_point_and_euler_approach(oracle_mod, u, dt):
    # one conductance g_u held constant, the others zero: the membrane equation is linear,
    #   C dV/dt = -gL (V - VL) + G_u g_u (E_u - V)   =>   V_inf = (gL VL + G_u g_u E_u) / (gL + G_u g_u)
    # and the Euler map contracts geometrically: V_n = V_inf + (V_0 - V_inf) (1 - dt (gL + G_u g_u) / C)^n
    t = _frozen_type()
    s, _ = _lone_neurons(oracle_mod, 1, dt, [t, dict(t)])
    gu, V0 = 0.045, -61.0
    V, g, ref = s.state()
    V[0] = V0
    g[0, u] = gu
    s.set_state(V, g, ref)
    a = t["G"][u] * gu
    Vinf = (t["gL"] * t["VL"] + a * t["E"][u]) / (t["gL"] + a)
    q = 1.0 - dt * (t["gL"] + a) / t["C"]
    for n in range(1, 300):
        s.step(1)
        Vn, gn, _ = s.state()
        assert gn[0, u] == gu and np.all(np.delete(gn[0], u) == 0.0)          # frozen, and nothing leaks between receptors
        assert abs(Vn[0] - (Vinf + (V0 - Vinf) * q ** n)) < 1e-10, (u, n)
    s.step(int(40.0 / (dt * (t["gL"] + a))))
    assert abs(s.state()[0][0] - Vinf) < 1e-9
    # the fixed point separates the receptors: using another receptor's E or G would miss it by far more than the tolerance
    for v in range(4):
        if v != u:
            wrongE = (t["gL"] * t["VL"] + a * t["E"][v]) / (t["gL"] + a)
            wrongG = (t["gL"] * t["VL"] + t["G"][v] * gu * t["E"][u]) / (t["gL"] + t["G"][v] * gu)
            assert abs(wrongE - Vinf) > 0.1 and abs(wrongG - Vinf) > 0.1


def test_all_receptors_and_iext_together_fixed_point(oracle_mod):
    # all four conductances on, plus a constant external current:
    #   V_inf = (gL VL + sum_u G_u g_u E_u + I_ext) / (gL + sum_u G_u g_u)
    t = _frozen_type(Iext=0.37)
    s, _ = _lone_neurons(oracle_mod, 1, 0.1, [t, dict(t)])
    gs = [0.011, 0.05, 0.023, 0.007]
    V, g, ref = s.state()
    V[0] = -80.0
    g[0] = gs
    s.set_state(V, g, ref)
    a = [t["G"][u] * gs[u] for u in range(4)]
    tot = t["gL"] + sum(a)
    Vinf = (t["gL"] * t["VL"] + sum(a[u] * t["E"][u] for u in range(4)) + t["Iext"]) / tot
    q = 1.0 - 0.1 * tot / t["C"]
    for n in range(1, 200):
        s.step(1)
        assert abs(s.state()[0][0] - (Vinf + (-80.0 - Vinf) * q ** n)) < 1e-10
    # a sign slip on any single term moves the fixed point
    for u in range(4):
        flipped = (t["gL"] * t["VL"] + sum(a[v] * t["E"][v] * (-1 if v == u else 1) for v in range(4)) + t["Iext"]) / tot
        assert abs(flipped - Vinf) > 1e-3 or abs(a[u] * t["E"][u]) < 1e-3


def test_types_use_their_own_constants(oracle_mod):
    # neuron 0 of type 0, neuron 1 of type 1 with different gL, VL, G, E and I_ext: each relaxes to ITS fixed point
    t0 = _frozen_type(Iext=0.2)
    t1 = _frozen_type(Iext=-0.1, gL=0.05, VL=-70.0, G=[0.5, 0.9, 1.4, 0.3], E=[-5.0, 2.0, -80.0, -90.0])
    s, _ = _lone_neurons(oracle_mod, 2, 0.1, [t0, t1], ntype=np.array([0, 1], np.uint8))
    V, g, ref = s.state()
    V[:] = -66.0
    g[:] = [0.02, 0.01, 0.03, 0.015]
    s.set_state(V, g, ref)
    s.step(20000)
    for i, t in enumerate((t0, t1)):
        a = [t["G"][u] * g[i, u] for u in range(4)]
        Vinf = (t["gL"] * t["VL"] + sum(a[u] * t["E"][u] for u in range(4)) + t["Iext"]) / (t["gL"] + sum(a))
        assert abs(s.state()[0][i] - Vinf) < 1e-9


@pytest.mark.parametrize("rec", [0, 1, 2, 3])
@pytest.mark.parametrize("delay", [1, 3])
def test_membrane_sees_old_conductance_to_the_step(oracle_mod, rec, delay):
    # R8 (P:L475 / P:L479: both right-hand sides at time t), at the paper's production step dt = 1 ms.  Neuron 0 is
    # flagged in step 0; over a synapse of delay d the event is read in step d and g jumps at the END of step d
    # (state after d + 1 updates); V of the target must NOT move in that step -- it sits exactly at V_L, where the
    # leak is zero -- and moves in the next one by exactly kappa G_u (wq 2^-S) (E_u - V_L).
    dt, w = 1.0, 0.0123
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    t.update(G=list(G_DISTINCT), E=list(E_DISTINCT))
    sim = db_inputs.sim_params(dt_ms=dt, D=8, types=[t, dict(t)])
    net = dict(N=2, n_regions=1, region_start=np.array([0, 2]), ntype=np.array([0 if rec < 2 else 1, 0], np.uint8),
               row_ptr=np.array([0, 1, 1], np.int64), tgt=np.array([1], np.int32),
               w=np.array([w], np.float32), delay=np.array([delay], np.uint8), rec=np.array([rec], np.uint8))
    s = oracle_mod.OracleSim(sim, net, seed=1, fp64=True)
    V, g, ref = s.state()
    V[0], V[1] = -40.0, t["VL"]
    s.set_state(V, g, ref)
    wq = int(np.rint(np.float32(w) * np.float32(2.0 ** sim["S"]))) * 2.0 ** -sim["S"]
    for n in range(delay + 1):                     # steps 0 .. d
        s.step(1)
        Vn, gn, _ = s.state()
        assert Vn[1] == t["VL"]                     # untouched up to and including the step in which g jumps
        assert (gn[1, rec] == wq) == (n == delay) and (n == delay or gn[1, rec] == 0.0)
    s.step(1)                                       # step d + 1: the first one whose current holds the new g
    want = t["VL"] + (dt / t["C"]) * (t["G"][rec] * wq) * (t["E"][rec] - t["VL"])
    assert abs(s.state()[0][1] - want) < 1e-12 and abs(want - t["VL"]) > 1e-3
    assert list(s.spikes()[0]) == [0] and list(s.spikes()[1]) == [0]


@pytest.mark.parametrize("fp64", [True, False])
def test_initial_potential_from_the_pinned_philox_words(oracle_mod, fp64):
    # R-RNG: V0 = Vreset + (Vth - Vreset) * (u >> 8) * 2^-24, u = word 0 of Philox(key = seed, counter = (i, stream 1 << 24, 0, 0)),
    # from the generator pinned by the published known-answer vectors -- integers here, one rounding per operation
    a = db_inputs.type_params()
    b = db_inputs.type_params()
    b.update(Vth=-48.5, Vreset=-61.25)
    N, seed = 4097, 0x1234567890ABCDEF
    ntype = (np.arange(N) % 3 == 0).astype(np.uint8)
    s, _ = _lone_neurons(oracle_mod, N, 0.1, [a, b], fp64=fp64, seed=seed, ntype=ntype)
    V = s.state()[0]
    real = np.float64 if fp64 else np.float32
    U = np.empty(N)
    for i in range(N):
        u = int(oracle_mod.philox([i, 1 << 24, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])[0])
        U[i] = (u >> 8) * 2.0 ** -24                  # exact in fp32 and fp64
        t = b if ntype[i] else a
        want = real(t["Vreset"]) + (real(t["Vth"]) - real(t["Vreset"])) * real(U[i])
        assert V[i] == float(want), i
    # and the draw is uniform on [0, 1): all below 1, mean 1/2, variance 1/12 (4 sigma)
    assert U.max() < 1.0 and U.min() >= 0.0
    assert abs(U.mean() - 0.5) < 4 * math.sqrt(1 / 12 / N) and abs(U.var() - 1 / 12) < 4 * math.sqrt(1 / 180 / N)
    g, ref = s.state()[1], s.state()[2]
    assert np.all(g == 0.0) and np.all(ref == 0)


def _to_i32(x):
    return int(np.array([x & 0xFFFFFFFF], np.uint64).astype(np.uint32).view(np.int32)[0])


@pytest.mark.parametrize("fp64", [True, False])
def test_ring_wraps_in_twos_complement_and_raises_the_sticky_flag(oracle_mod, fp64):
    # R28: accumulation is 32-bit two's complement on both sides; a consumed cell beyond 2^30 in magnitude raises a
    # sticky flag.  Neurons 0, 1, 2 all push w = 300 (wq = 300 * 2^22 = 1,258,291,200) into (neuron 3, AMPA) with
    # delay 2 and fire together in step 0: the cell must hold 3 wq mod 2^32 = 3,774,873,600 - 2^32 = -520,093,696.
    S, D = 22, 8
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    sim = db_inputs.sim_params(dt_ms=0.1, S=S, D=D, types=[t, dict(t)])
    net = dict(N=4, n_regions=1, region_start=np.array([0, 4]), ntype=np.zeros(4, np.uint8),
               row_ptr=np.array([0, 1, 2, 3, 3], np.int64), tgt=np.array([3, 3, 3], np.int32),
               w=np.array([300.0] * 3, np.float32), delay=np.array([2, 2, 2], np.uint8), rec=np.zeros(3, np.uint8))
    s = oracle_mod.OracleSim(sim, net, seed=1, fp64=fp64)
    V, g, ref = s.state()
    V[:3], V[3] = -40.0, t["VL"]
    s.set_state(V, g, ref)
    s.step(1)
    wq = 300 * 2 ** S
    cell = _to_i32(3 * wq)
    assert cell == -520093696
    ring = s.ring()
    assert ring[2, 3, 0] == cell and np.count_nonzero(ring) == 1
    assert s.counters()["overflow"] == 0                 # nothing consumed yet
    s.step(2)                                            # step 2 consumes the cell
    assert s.counters()["overflow"] == 0                 # |-520,093,696| < 2^30: wrapped, but inside the bound
    assert s.state()[1][3, 0] == cell * 2.0 ** -S        # the wrapped integer is what enters g (exact in fp32 too: 2^9 * 2^-22 grid)
    assert np.count_nonzero(s.ring()) == 0
    # the bound itself: exactly 2^30 passes, 2^30 + 1 trips, on either sign; the flag is sticky
    lone = dict(net, row_ptr=np.zeros(5, np.int64), tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32),
                delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))       # no synapses: nothing else enters the ring
    for val, trips in ((1 << 30, False), (-(1 << 30), False), ((1 << 30) + 1, True), (-(1 << 30) - 1, True)):
        o = oracle_mod.OracleSim(sim, lone, seed=1, fp64=fp64)
        r = o.ring()
        r[0, 1, 2] = val
        o.set_ring(r)
        o.step(1)
        assert o.counters()["overflow"] == int(trips), val
        o.step(5)
        assert o.counters()["overflow"] == int(trips)


def test_eight_types_each_relax_to_their_own_fixed_point(oracle_mod):
    # up to eight neuron types with their own constants (the populations of a micro-column, Ext. Table 3, or
    # (region group, type) pairs): neuron i of type i mod 8 relaxes to ITS fixed point
    types = []
    for k in range(8):
        types.append(_frozen_type(Iext=0.05 * k - 0.1, gL=0.02 + 0.005 * k, VL=-78.0 + 1.5 * k, C=0.7 + 0.1 * k,
                                  G=[1.3 - 0.1 * k, 0.21 + 0.02 * k, 0.77 + 0.05 * k, 1.9 - 0.15 * k],
                                  E=[3.0 - k, -11.0 + k, -68.0 - 0.5 * k, -97.0 + k]))
    N = 64
    ntype = (np.arange(N) % 8).astype(np.uint8)
    s, _ = _lone_neurons(oracle_mod, N, 0.1, types, ntype=ntype)
    V, g, ref = s.state()
    V[:] = -66.0
    g[:] = [0.02, 0.01, 0.03, 0.015]
    s.set_state(V, g, ref)
    s.step(40000)
    got = s.state()[0]
    for i in range(N):
        t = types[i % 8]
        a = [t["G"][u] * g[i, u] for u in range(4)]
        Vinf = (t["gL"] * t["VL"] + sum(a[u] * t["E"][u] for u in range(4)) + t["Iext"]) / (t["gL"] + sum(a))
        assert abs(got[i] - Vinf) < 1e-9, i
