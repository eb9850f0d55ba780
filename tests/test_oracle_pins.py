"""Pins of the oracle's pieces against things that are not the oracle:
published known-answer vectors, library routines (scipy / numpy), closed
forms, invariants and brute force.  CPU only."""
import math
import os

import numpy as np
import pytest
from scipy import stats

import db_inputs

HERE = os.path.dirname(os.path.abspath(__file__))


# ---------------------------------------------------------------- generators
def test_philox_known_answers(oracle_mod):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle_mod.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_draw_counter_layout(oracle_mod):
    # draw(seed, stream, a, b) = philox(counter=(a_lo, a_hi|stream<<24, b_lo, b_hi), key=seed)
    seed, stream, a, b = 0x0123456789ABCDEF, 5, (3 << 32) | 77, (9 << 32) | 12345
    exp = oracle_mod.philox([77, 3 | (5 << 24), 12345, 9], [0x89ABCDEF, 0x01234567])
    assert (oracle_mod.draw(seed, stream, a, b) == exp).all()


@pytest.mark.parametrize("lam", [0.0, 0.01, 0.1, 1.0, 3.7])
def test_poisson_thresholds_match_scipy_cdf(oracle_mod, lam):
    T = oracle_mod.poisson_thresholds(lam)
    if lam == 0.0:
        assert len(T) == 0
        return
    cdf = stats.poisson.cdf(np.arange(len(T) + 1), lam)
    # floor(cdf * 2^32), allowing the last-bit difference of two double evaluations
    want = np.floor(cdf * 2.0 ** 32)
    assert np.all(np.abs(T.astype(np.float64) - want[:len(T)]) <= 2)
    assert np.all(np.diff(T.astype(np.int64)) > 0)
    assert want[len(T)] >= 2 ** 32 - 1            # the table stops only when saturated


def test_poisson_sample_moments(oracle_mod):
    lam = 0.1
    T = oracle_mod.poisson_thresholds(lam)
    n = 200_000
    ks = np.empty(n)
    for i in range(n // 4):
        u = oracle_mod.draw(7, 2, i, 3)
        for j in range(4):
            ks[4 * i + j] = oracle_mod.poisson_count(int(u[j]), T)
    se = math.sqrt(lam / n)
    assert abs(ks.mean() - lam) < 4 * se
    assert abs(ks.var() - lam) < 6 * math.sqrt(lam * (1 + 2 * lam) / n) + 4 * se
    # exact counting definition k = #{m: u >= T_m}
    assert oracle_mod.poisson_count(0, T) == 0
    assert oracle_mod.poisson_count(int(T[0]), T) == 1
    assert oracle_mod.poisson_count(int(T[0]) - 1, T) == 0
    assert oracle_mod.poisson_count(2 ** 32 - 1, T) == len(T)


def test_norm_ppf_and_half_rounding(oracle_mod):
    for p in [1e-6, 0.001, 0.2, 0.5, 0.77, 0.999, 1 - 1e-6]:
        assert abs(oracle_mod.lib().orc_norm_ppf(p) - stats.norm.ppf(p)) < 1e-9
    rng = np.random.default_rng(0)
    xs = np.concatenate([rng.lognormal(-6, 2, 2000), [0.0, 65504.0, 65519.9, 1e-8, 6.0e-5, 5.96e-8, 0.1]])
    xs = np.concatenate([xs, -xs]).astype(np.float32)
    for x in xs:
        got = oracle_mod.lib().orc_round_to_half(float(x))
        want = float(np.float32(np.float16(x)))
        assert got == want, (x, got, want)


# independent Python restatement of the keyed permutation (Feistel + cycle walking)
def _fmix32(h):
    h &= 0xFFFFFFFF
    h ^= h >> 16
    h = (h * 0x85EBCA6B) & 0xFFFFFFFF
    h ^= h >> 13
    h = (h * 0xC2B2AE35) & 0xFFFFFFFF
    h ^= h >> 16
    return h


def _prp_py(x, M, key):
    if M <= 1:
        return 0
    nb = max(2, (M - 1).bit_length())
    a, b = nb // 2, nb - nb // 2
    while True:
        L, R = x >> b, x & ((1 << b) - 1)
        nl, nr = a, b
        for r in range(8):
            rk = (int(key[r & 3]) + (r >> 2) * 0x9E3779B9) & 0xFFFFFFFF
            F = _fmix32((R + rk) & 0xFFFFFFFF) & ((1 << nl) - 1)
            L, R = R, L ^ F
            nl, nr = nr, nl
        x = (L << nr) | R
        if x < M:
            return x


@pytest.mark.parametrize("M", [1, 2, 3, 4, 5, 17, 64, 100, 1000, 4097])
def test_prp_is_a_permutation(oracle_mod, M):
    key = oracle_mod.draw(11, 3, M, 0)
    out = [oracle_mod.prp(x, M, key) for x in range(M)]
    assert sorted(out) == list(range(M))
    assert out == [_prp_py(x, M, key) for x in range(M)]


def test_prp_first_elements_are_uniform(oracle_mod):
    # perm_key(0) over many keys is uniform on [0, M): chi-square
    M, n = 50, 20000
    cnt = np.zeros(M)
    for i in range(n):
        cnt[oracle_mod.prp(0, M, oracle_mod.draw(5, 3, i, 0))] += 1
    chi2 = ((cnt - n / M) ** 2 / (n / M)).sum()
    assert chi2 < stats.chi2.ppf(0.9999, M - 1)
    # and pairs (perm(0), perm(1)) are uniform over ordered pairs
    M = 12
    cnt = np.zeros((M, M))
    for i in range(n):
        k = oracle_mod.draw(6, 3, i, 0)
        cnt[oracle_mod.prp(0, M, k), oracle_mod.prp(1, M, k)] += 1
    assert np.all(np.diag(cnt) == 0)
    off = cnt[~np.eye(M, dtype=bool)]
    chi2 = ((off - n / off.size) ** 2 / (n / off.size)).sum()
    assert chi2 < stats.chi2.ppf(0.9999, off.size - 1)


# ---------------------------------------------------------------- single neuron closed forms
def _single(oracle_mod, Iext=0.0, dt=0.1, fp64=True, bg_rate=0.0, bg_weight=0.0, N=1, V0=None, **kw):
    t = db_inputs.type_params(bg_weight=bg_weight, bg_rate_hz=bg_rate)
    t["Iext"] = Iext
    t.update(kw)
    sim = db_inputs.sim_params(dt_ms=dt, types=[t, dict(t)])
    net = dict(N=N, n_regions=1, region_start=np.array([0, N]), ntype=np.zeros(N, np.uint8),
               row_ptr=np.zeros(N + 1, np.int64), tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32),
               delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))
    s = oracle_mod.OracleSim(sim, net, seed=3, fp64=fp64)
    if V0 is not None:
        V, g, ref = s.state()
        V[:] = V0
        s.set_state(V, g, ref)
    return s, t


def test_lif_discrete_and_continuous_closed_form(oracle_mod):
    # sub-threshold constant current: V_n = Vinf + (V0 - Vinf)(1 - dt gL/C)^n  (exact for the Euler map)
    I = 0.6                                   # Vinf = -75 + 0.6/0.03 = -55 < Vth
    for dt in (0.1, 1.0):
        s, t = _single(oracle_mod, Iext=I, dt=dt, V0=-70.0)
        Vinf = t["VL"] + I / t["gL"]
        q = 1.0 - dt * t["gL"] / t["C"]
        for n in range(1, 400):
            s.step(1)
            V = s.state()[0][0]
            assert abs(V - (Vinf + (-70.0 - Vinf) * q ** n)) < 1e-11
        # continuous solution approached to first order in dt
        tt = 400 * dt - dt
        cont = Vinf + (-70.0 - Vinf) * math.exp(-tt * t["gL"] / t["C"])
        assert abs(V - cont) < 15.0 * dt * t["gL"]    # O(dt) global error
        assert len(s.spikes()[1]) == 0


def test_first_spike_time_and_isi(oracle_mod):
    # supra-threshold constant current: first spike step n*, then period n*(Vreset) + R  (R6)
    I, dt = 1.2, 0.1                          # Vinf = -35
    s, t = _single(oracle_mod, Iext=I, dt=dt, V0=-72.0)
    Vinf = t["VL"] + I / t["gL"]
    q = 1.0 - dt * t["gL"] / t["C"]
    R = round(t["Tref_ms"] / dt)

    def nstar(V0):   # smallest n with Vinf + (V0-Vinf) q^n >= Vth
        return math.ceil(math.log((t["Vth"] - Vinf) / (V0 - Vinf)) / math.log(q))

    s.step(3000)
    st, ids = s.spikes()
    assert len(st) >= 5
    # V(t_{n+1}) >= Vth is flagged in step n: the spike of the n-th update has step index n-1
    assert int(st[0]) == nstar(-72.0) - 1
    isi = np.diff(st.astype(np.int64))
    assert np.all(isi == nstar(t["Vreset"]) + R)
    # continuous first-spike time
    tstar = (t["C"] / t["gL"]) * math.log((Vinf - (-72.0)) / (Vinf - t["Vth"]))
    assert abs((int(st[0]) + 1) * dt - tstar) < 0.3


def test_refractory_clamp_values(oracle_mod):
    # at the spike step and during the next R steps V is Vreset; integration resumes after (R6)
    s, t = _single(oracle_mod, Iext=1.2, dt=0.1, V0=-50.5)
    R = round(t["Tref_ms"] / 0.1)
    vs, refs = [], []
    for n in range(R + 30):
        s.step(1)
        V, g, ref = s.state()
        vs.append(V[0]); refs.append(ref[0])
    st, _ = s.spikes()
    n0 = int(st[0])
    assert all(v == t["Vreset"] for v in vs[n0:n0 + R + 1])
    assert vs[n0 + R + 1] > t["Vreset"]
    assert refs[n0] == R and refs[n0 + R] == 0


def _two_neuron(oracle_mod, w, rec, delay, dt=0.1, fp64=True, D=32):
    """neuron 0 -> neuron 1, one synapse; no background."""
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    sim = db_inputs.sim_params(dt_ms=dt, D=D, types=[t, dict(t)])
    net = dict(N=2, n_regions=1, region_start=np.array([0, 2]), ntype=np.array([0 if rec < 2 else 1, 0], np.uint8),
               row_ptr=np.array([0, 1, 1], np.int64), tgt=np.array([1], np.int32),
               w=np.array([w], np.float32), delay=np.array([delay], np.uint8), rec=np.array([rec], np.uint8))
    s = oracle_mod.OracleSim(sim, net, seed=1, fp64=fp64)
    return s, t, sim


@pytest.mark.parametrize("rec", [0, 1, 2, 3])
@pytest.mark.parametrize("delay", [1, 7])
def test_single_event_conductance_kernel(oracle_mod, rec, delay):
    # one event of weight w: g jumps instantly then decays exactly exponentially (SI Eq.(3))
    w, dt = 0.0123, 0.1
    s, t, sim = _two_neuron(oracle_mod, w, rec, delay, dt)
    V, g, ref = s.state()
    V[0] = -40.0     # above threshold: neuron 0 is flagged in step 0 (after its Euler step it stays >= Vth)
    V[1] = t["VL"]
    s.set_state(V, g, ref)
    wq = int(np.rint(np.float32(w) * np.float32(2.0 ** sim["S"])))
    alpha = math.exp(-dt / t["tau_ms"][rec])
    na = 0 + delay          # read in step na, enters g at the end of step na
    for n in range(na + 200):
        s.step(1)
        g1 = s.state()[1][1]
        if n < na:
            assert np.all(g1 == 0.0)
        else:
            want = wq * 2.0 ** -sim["S"] * alpha ** (n - na)
            assert abs(g1[rec] - want) <= 1e-13 * want
            assert np.all(np.delete(g1, rec) == 0.0)
            # continuous kernel w exp(-(t - t_a)/tau)
            assert abs(g1[rec] - w * math.exp(-(n - na) * dt / t["tau_ms"][rec])) < 2e-7 + 1e-6 * w
    assert list(s.spikes()[0][:1]) == [0]


def test_psp_shape_small_weight(oracle_mod):
    # small-w AMPA event on a neuron at rest: difference of exponentials
    w, dt = 1e-4, 0.01
    s, t, sim = _two_neuron(oracle_mod, w, 0, 1, dt, D=4)
    V, g, ref = s.state()
    V[0] = -40.0
    V[1] = t["VL"]
    s.set_state(V, g, ref)
    tau_m, tau_s = t["C"] / t["gL"], t["tau_ms"][0]
    wq = np.rint(np.float32(w) * np.float32(2.0 ** sim["S"])) * 2.0 ** -sim["S"]
    amp = t["G"][0] * wq * (t["E"][0] - t["VL"]) / t["C"] * tau_m * tau_s / (tau_m - tau_s)
    peak_seen = 0.0
    for n in range(1500):
        s.step(1)
        tt = (n - 1) * dt                 # g jumps at the end of step 1, moves V from step 2 on
        dv = s.state()[0][1] - t["VL"]
        if tt > 0:
            want = amp * (math.exp(-tt / tau_m) - math.exp(-tt / tau_s))
            assert abs(dv - want) < 0.02 * amp * 0.8 + 1e-9     # O(dt) + O(w) corrections
            peak_seen = max(peak_seen, dv)
    tpk = math.log(tau_m / tau_s) * tau_m * tau_s / (tau_m - tau_s)
    assert abs(peak_seen - amp * (math.exp(-tpk / tau_m) - math.exp(-tpk / tau_s))) < 0.02 * amp


def test_background_mean_conductance(oracle_mod):
    # no recurrent input: E[g_AMPA] = lambda * w_bg / (1 - alpha)
    N = 4000
    s, t = _single(oracle_mod, N=N, bg_rate=1000.0, bg_weight=0.004, fp64=True, Vth=1e9)
    s.step(1500)
    g = s.state()[1][:, 0]
    lam = 1000.0 * 0.1 * 1e-3
    alpha = math.exp(-0.1 / t["tau_ms"][0])
    wq = round(0.004 * 2 ** 22) * 2.0 ** -22
    mean = lam * wq / (1 - alpha)
    sd = wq * math.sqrt(lam / (1 - alpha ** 2))
    assert abs(g.mean() - mean) < 5 * sd / math.sqrt(N)
    assert abs(g.std() - sd) < 0.1 * sd
    assert s.counters()["bg_events"] > 0 and s.counters()["events"] == 0


def test_dt_convergence_first_order(oracle_mod):
    # Euler: error vs a fine reference shrinks ~linearly in dt (~5 % at 1 ms)
    def v_at(dt, T=20.0):
        s, t = _single(oracle_mod, Iext=0.7, dt=dt, V0=-74.0)
        s.step(int(round(T / dt)))
        return s.state()[0][0]
    ref = v_at(0.001)
    e1, e2 = abs(v_at(1.0) - ref), abs(v_at(0.1) - ref)
    assert 7.0 < e1 / e2 < 13.0


# ---------------------------------------------------------------- network-level pins
def _driven_sim(oracle_mod, net, fp64=False, D=32, bg_weight=0.02):
    t = db_inputs.type_params(bg_weight=bg_weight, bg_rate_hz=1000.0)
    sim = db_inputs.sim_params(D=D, types=[t, dict(t)])
    return oracle_mod.OracleSim(sim, net, seed=5, fp64=fp64), sim, t


def test_delivery_equals_dense_brute_force(oracle_mod):
    net = db_inputs.random_csr(N=48, mean_outdeg=9, seed=4, max_delay=20)
    s, sim, t = _driven_sim(oracle_mod, net)
    s.log_arrivals(True)
    T = 1000
    s.step(T)
    st, ids = s.spikes()
    assert len(ids) > 200
    spikes = np.zeros((T, 48), np.uint8)
    spikes[st.astype(np.int64), ids] = 1
    dense = oracle_mod.dense_arrivals(net, sim["S"], spikes)
    got = s.arrivals().astype(np.int64)
    assert got.shape == dense.shape
    assert np.array_equal(got, dense)
    # conservation: events = sum of out-degrees of the spiking neurons
    outdeg = np.diff(net["row_ptr"])
    assert s.counters()["events"] == int(outdeg[ids].sum())
    # everything ever delivered is either consumed or still in the ring
    wq = np.rint(net["w"] * np.float32(2.0 ** sim["S"])).astype(np.int64)
    row_sum = np.add.reduceat(np.concatenate([wq, [0]]), net["row_ptr"][:-1]) * (outdeg > 0)
    assert got.sum() + s.ring().astype(np.int64).sum() == int(row_sum[ids].sum())


# ---- time bin for transferring spikes, b_t (SI "Numerical method"; R29)
@pytest.mark.parametrize("B", [2, 10])
def test_binned_transfer_equals_dense_definition_of_A(oracle_mod, B):
    # A_j(t) = 1 iff t is a bin boundary and j fired in (t - b_t, t], written out densely from
    # the raster in numpy; the delivered sums are then the dense matrix x delayed A vectors (Eq.(3), 2nd term)
    net = db_inputs.random_csr(N=48, mean_outdeg=9, seed=4, max_delay=20)
    t = db_inputs.type_params(bg_weight=0.02, bg_rate_hz=1000.0)
    sim = db_inputs.sim_params(D=64, types=[t, dict(t)], spike_bin_steps=B)
    s = oracle_mod.OracleSim(sim, net, seed=5)
    s.log_arrivals(True)
    T = 1000
    s.step(T)
    st, ids = s.spikes()
    assert len(ids) > 200
    spikes = np.zeros((T, 48), np.uint8)
    spikes[st.astype(np.int64), ids] = 1
    A = np.zeros_like(spikes)
    for m in range(B - 1, T, B):                     # step m closes the bin (m - B, m]
        A[m] = spikes[m - B + 1:m + 1].max(axis=0)
    assert A.sum() == spikes.sum()                   # T_ref > b_t: nobody fires twice in a bin
    dense = oracle_mod.dense_arrivals(net, sim["S"], A)
    got = s.arrivals().astype(np.int64)
    assert np.array_equal(got, dense)
    plain = oracle_mod.dense_arrivals(net, sim["S"], spikes)
    assert not np.array_equal(got, plain)            # and it is not the unbinned scheme
    outdeg = np.diff(net["row_ptr"])
    assert s.counters()["events"] == int(outdeg[ids].sum())


@pytest.mark.parametrize("n_s", [0, 3, 9, 10, 17])
def test_binned_transfer_timing_of_one_event(oracle_mod, n_s):
    # neuron 0 fires in step n_s; with b_t = 10 steps the spike is transferred at the end of the step
    # n_k = 10 floor(n_s / 10) + 9 and, over a synapse of delay d, read in step n_k + d
    B, d, w, rec = 10, 3, 0.0123, 0
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    sim = db_inputs.sim_params(D=32, types=[t, dict(t)], spike_bin_steps=B)
    net = dict(N=2, n_regions=1, region_start=np.array([0, 2]), ntype=np.array([0, 0], np.uint8),
               row_ptr=np.array([0, 1, 1], np.int64), tgt=np.array([1], np.int32),
               w=np.array([w], np.float32), delay=np.array([d], np.uint8), rec=np.array([rec], np.uint8))
    s = oracle_mod.OracleSim(sim, net, seed=1, fp64=True)
    V, g, ref = s.state()
    V[:] = t["VL"]
    s.set_state(V, g, ref)
    s.step(n_s)
    V, g, ref = s.state()
    V[0] = -40.0                                     # flagged in step n_s
    s.set_state(V, g, ref)
    na = (n_s // B) * B + B - 1 + d
    wq = int(np.rint(np.float32(w) * np.float32(2.0 ** sim["S"])))
    alpha = math.exp(-sim["dt_ms"] / t["tau_ms"][rec])
    for n in range(n_s, na + 30):
        s.step(1)
        g1 = s.state()[1][1][rec]
        if n < na:
            assert g1 == 0.0
        else:
            want = wq * 2.0 ** -sim["S"] * alpha ** (n - na)
            assert abs(g1 - want) <= 1e-13 * want
    assert list(s.spikes()[0]) == [n_s]


def test_bin_of_one_step_is_the_plain_scheme(oracle_mod):
    net = db_inputs.random_csr(N=200, mean_outdeg=20, seed=2)
    t = db_inputs.type_params(bg_weight=0.03)
    out = []
    for B in (0, 1):
        sim = db_inputs.sim_params(types=[t, dict(t)], spike_bin_steps=B)
        s = oracle_mod.OracleSim(sim, net, seed=5)
        s.step(600)
        out.append((s.spikes(), s.ring()))
    assert np.array_equal(out[0][0][0], out[1][0][0]) and np.array_equal(out[0][0][1], out[1][0][1])
    assert np.array_equal(out[0][1], out[1][1]) and len(out[0][0][1]) > 100


def test_refractoriness_invariant(oracle_mod):
    net = db_inputs.random_csr(N=300, mean_outdeg=30, seed=9)
    s, sim, t = _driven_sim(oracle_mod, net, bg_weight=0.05)
    s.step(1500)
    st, ids = s.spikes()
    R = round(t["Tref_ms"] / sim["dt_ms"])
    order = np.lexsort((st, ids))
    st, ids = st[order].astype(np.int64), ids[order]
    same = ids[1:] == ids[:-1]
    assert same.sum() > 100
    assert np.all((st[1:] - st[:-1])[same] >= R + 1)
    # region counts add up to the raster
    rc = s.region_counts()
    assert rc.sum() == len(ids)
    assert rc.shape[0] == 1500 // sim["window_steps"]


def test_region_counts_by_window(oracle_mod):
    net = db_inputs.random_csr(N=200, mean_outdeg=10, seed=2, n_regions=4)
    s, sim, t = _driven_sim(oracle_mod, net, bg_weight=0.04)
    s.step(230)
    st, ids = s.spikes()
    rc = s.region_counts()
    want = np.zeros_like(rc)
    reg = np.searchsorted(net["region_start"], ids, side="right") - 1
    np.add.at(want, (st.astype(np.int64) // sim["window_steps"], reg), 1)
    assert np.array_equal(rc, want)


def test_fp32_mode_tracks_fp64_mode_early(oracle_mod):
    # the fp32 contract mode is the same algorithm: identical raster early on, small V drift
    net = db_inputs.random_csr(N=400, mean_outdeg=40, seed=12)
    a, sim, _ = _driven_sim(oracle_mod, net, fp64=False)
    b, _, _ = _driven_sim(oracle_mod, net, fp64=True)
    a.step(100); b.step(100)
    assert np.array_equal(a.spikes()[1], b.spikes()[1])
    assert np.max(np.abs(a.state()[0] - b.state()[0])) < 1e-3
    assert np.array_equal(a.ring(), b.ring())


# ------------------------------------------------------------------ OU background current
def _ou_net(N):
    return dict(N=N, E=0, n_regions=1, region_start=np.array([0, N]), ntype=np.zeros(N, np.uint8),
                row_ptr=np.zeros(N + 1, np.int64), tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32),
                delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))


def _ou_sim(mu, sigma, tau_ms, dt_ms=0.1, **kw):
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    t.update(ou_mu=mu, ou_sigma=sigma, ou_tau_ms=tau_ms, **kw)
    return db_inputs.sim_params(dt_ms=dt_ms, types=[t])


def test_normal_table_is_the_standard_normal_quantile_function(oracle_mod):
    from scipy.stats import norm
    tab = oracle_mod.normal_table()
    want = norm.ppf((np.arange(65536) + 0.5) / 65536.0)
    assert np.all(np.abs(tab - want) <= 2e-7 * np.maximum(1.0, np.abs(want)))      # fp32 rounding of the double quantile
    assert np.all(np.diff(tab) > 0) and np.array_equal(tab, -tab[::-1])             # strictly increasing, antisymmetric
    assert abs(float(tab.astype(np.float64).mean())) < 1e-9
    assert abs(float((tab.astype(np.float64) ** 2).mean()) - 1.0) < 2e-4          # variance of the 65536-point quantisation


def test_ou_without_noise_relaxes_geometrically_to_mu(oracle_mod):
    # sigma = 0: I_n = mu + (I_0 - mu)(1 - dt/tau)^n, the Euler map of dI/dt = (mu - I)/tau (main Eq.(1))
    mu, tau, dt = 0.66, 10.0, 0.1
    o = oracle_mod.OracleSim(_ou_sim(mu, 0.0, tau, dt), _ou_net(3), 1, fp64=True)
    o.set_iou(np.array([0.0, 2.0, mu]))
    n = 400
    o.step(n)
    want = mu + (np.array([0.0, 2.0, mu]) - mu) * (1.0 - dt / tau) ** n
    assert np.allclose(o.iou(), want, rtol=0, atol=1e-12)


def test_ou_stationary_mean_sd_and_autocorrelation(oracle_mod):
    # Ext. Table 2: mu = 0.66, sigma = 0.12, tau = 10.  The discrete map has stationary mean mu,
    # variance sigma^2 (2a)/(1-(1-a)^2) = sigma^2/(1 - a/2), a = dt/tau, and lag-k autocorrelation (1-a)^k ~ e^{-k dt/tau}
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "ou_extended_data_table2.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    mu, sigma, tau, dt = vals["mu_ext"], vals["sigma_ext"], vals["tau_ext"], 1.0     # the paper's printed values
    assert (mu, sigma, tau) == (0.66, 0.12, 10.0)
    N, burn, T = 4000, 200, 400
    sim = _ou_sim(mu, sigma, tau, dt, Vth=1e9)                  # no spikes: the membrane is irrelevant here
    o = oracle_mod.OracleSim(sim, _ou_net(N), 7, fp64=True)
    assert np.array_equal(o.iou(), np.full(N, mu))               # starts at its mean
    o.step(burn)
    xs = []
    for _ in range(T):
        xs.append(o.iou().copy())
        o.step(1)
    x = np.array(xs)                                             # [T][N]
    a = dt / tau
    sd_want = sigma / np.sqrt(1.0 - a / 2.0)
    assert abs(x.mean() - mu) < 4 * sd_want / np.sqrt(N * T * a)            # about a*T*N independent samples
    assert abs(x.std() / sd_want - 1.0) < 0.02
    for lag in (1, 5, 10, 20):
        c = np.mean((x[:-lag] - mu) * (x[lag:] - mu)) / x.var()
        assert abs(c - (1.0 - a) ** lag) < 0.02
        assert abs(c - np.exp(-lag * dt / tau)) < 0.03


def test_ou_current_enters_the_membrane_equation_as_a_current(oracle_mod):
    # sigma = 0 and I_ou(0) = mu: a constant current mu, so V follows the constant-current closed form
    # V_n = V_inf + (V_0 - V_inf)(1 - dt gL / C)^n with V_inf = VL + mu / gL (below threshold here)
    mu, dt = 0.5, 0.1
    sim = _ou_sim(mu, 0.0, 10.0, dt)
    tp = sim["types"][0]
    o = oracle_mod.OracleSim(sim, _ou_net(1), 1, fp64=True)
    V0 = o.state()[0][0]
    n = 300
    o.step(n)
    Vinf = tp["VL"] + mu / tp["gL"]
    assert Vinf < tp["Vth"]
    want = Vinf + (V0 - Vinf) * (1.0 - dt * tp["gL"] / tp["C"]) ** n
    assert abs(o.state()[0][0] - want) < 1e-10
