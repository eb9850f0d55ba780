"""Parity cases for the kernel paths VERDICT round 1 found unreached: I_ext != 0 with different constants per neuron
type, the paper's production step dt = 1 ms (long Poisson table, R = 5 steps), region-rate windows of 1, 2 and 3 steps,
a synchronised burst that overflows the per-block spike and heavy-row lists of the persistent kernel, and the ring's
wrap / overflow flag.  Same bars as tests/test_gpu_parity.py (ring and counters bit-exact, raster identical, state
within 1e-5 -- in fact equal), through the C ABI, in all three execution modes."""
import numpy as np
import pytest

import db_inputs

pytestmark = pytest.mark.gpu

MODES = [1, 2, 3]   # DB_EXEC_KERNELS, DB_EXEC_PERSISTENT, DB_EXEC_KERNELS_DEFERRED


@pytest.fixture(scope="module")
def db():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2211_15963_b200 as m
    m.load()
    return m


def _check(g, o, steps, ring=True, rel=1e-5):
    Vg, gg, rg = g.state()
    Vo, go, ro = o.state()
    assert np.array_equal(rg, ro)
    assert np.all(np.abs(Vg - Vo) <= rel * np.abs(Vo)) and np.all(np.abs(gg - go) <= rel * np.abs(go))
    assert np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32))
    if ring:
        assert np.array_equal(g.db_read_state(7), o.ring())
    sg, ig = g.db_read_spikes(0, steps)
    so, io = o.spikes()
    order = np.lexsort((io, so))
    assert np.array_equal(sg, so[order]) and np.array_equal(ig, io[order])
    cg, co = g.db_get_counters(), o.counters()
    for k in ("steps", "spikes", "events", "bg_events"):
        assert cg[k] == co[k], k
    assert cg["ring_overflow"] == co["overflow"]
    return len(ig)


def _distinct_types():
    exc = db_inputs.type_params(bg_weight=0.009)
    exc.update(Iext=0.21, G=[1.1, 0.3, 0.9, 1.2], E=[2.0, -3.0, -72.0, -95.0], tau_ms=[2.5, 35.0, 8.0, 60.0])
    inh = db_inputs.type_params(bg_weight=0.006, bg_rate_hz=1500.0)
    inh.update(Iext=-0.05, C=0.8, gL=0.04, VL=-70.0, Vth=-52.0, Vreset=-60.0, Tref_ms=2.0,
               G=[0.8, 0.2, 1.3, 0.7], E=[0.0, 1.0, -75.0, -90.0], tau_ms=[1.5, 50.0, 12.0, 40.0])
    return exc, inh


@pytest.mark.parametrize("mode", MODES)
def test_iext_and_different_constants_per_type(db, oracle_mod, mode):
    # I_ext is non-zero and of opposite sign on the two types; every other constant differs too
    exc, inh = _distinct_types()
    sim = db_inputs.sim_params(types=[exc, inh])
    N = 6000 + 19
    net = db_inputs.random_csr(N=N, mean_outdeg=30, seed=31, n_regions=3)       # type boundaries inside 4-neuron groups
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    for upto in (1, 2, 60, 500):
        g.db_step(upto - int(g.db_get_counters()["steps"])); o.step(upto - o.step_index)
        n = _check(g, o, upto)
    ids = g.db_read_spikes(0, 500)[1]
    assert np.count_nonzero(net["ntype"][ids] == 0) > 100 and np.count_nonzero(net["ntype"][ids] == 1) > 100
    # the external current matters: without it the raster is another one
    exc0, inh0 = dict(exc, Iext=0.0), dict(inh, Iext=0.0)
    h = db.Sim.db_create_from_csr(db_inputs.sim_params(types=[exc0, inh0]), net, exec_mode=mode)
    h.db_step(500)
    assert len(h.db_read_spikes(0, 500)[1]) != n


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("bin_steps", [1])
def test_production_step_dt_1ms(db, oracle_mod, mode, bin_steps):
    # the paper's production step: dt = 1 ms, so lambda = 1 background event per step (the long Poisson
    # table: up to 12 thresholds are walked), R = 5 steps, b_t = 1 step = 1 ms, delays 1..20 ms
    t = db_inputs.type_params(bg_weight=0.005, bg_rate_hz=1000.0)
    sim = db_inputs.sim_params(dt_ms=1.0, D=32, window_steps=5, types=[t, dict(t)], spike_bin_steps=bin_steps)
    N = 8000 + 5
    net = db_inputs.random_csr(N=N, mean_outdeg=40, seed=17, heavy_rows={3: 2500})
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    for upto in (1, 5, 100, 1000):                                  # 1 s of biological time
        g.db_step(upto - int(g.db_get_counters()["steps"])); o.step(upto - o.step_index)
        n = _check(g, o, upto)
    rate = n / N / 1.0
    assert 1.0 < rate < 60.0, rate
    assert g.db_get_counters()["bg_events"] > 0.9 * N * 1000
    cnt, first = g.db_region_counts()
    assert np.array_equal(cnt, o.region_counts()[first:first + len(cnt)]) and len(cnt) == 200


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("window", [1, 2, 3])
def test_region_windows_shorter_than_the_pipeline(db, oracle_mod, mode, window):
    # windows of 1, 2 and 3 steps with several regions: the persistent kernel's blocks run up to two units apart, so the
    # window that is cleared ahead and the windows still being counted are only a few cells apart
    t = db_inputs.type_params(bg_weight=0.03)
    sim = db_inputs.sim_params(window_steps=window, types=[t, dict(t)])
    N, R = 20000 + 3, 6
    net = db_inputs.random_csr(N=N, mean_outdeg=15, seed=23, n_regions=R)
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode, max_windows=64)     # a short history: it wraps many times
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    done = 0
    for upto in (1, 2, 3, 7, 150, 151, 400):
        g.db_step(upto - done); o.step(upto - done)
        done = upto
        cnt, first = g.db_region_counts()
        want = o.region_counts()
        assert len(cnt) == min(upto // window, 64 - 1 - (2 // window + 1))
        assert first + len(cnt) == upto // window
        assert np.array_equal(cnt, want[first:first + len(cnt)]), (upto, first)
    assert cnt.sum() > 100 and np.all(cnt.sum(axis=0) > 0)
    _check(g, o, 400)
    # single region, same windows (counted per block and unit in the persistent kernel)
    net1 = db_inputs.random_csr(N=5000, mean_outdeg=15, seed=24)
    g1 = db.Sim.db_create_from_csr(sim, net1, exec_mode=mode, max_windows=32)
    o1 = oracle_mod.OracleSim(sim, net1, db_inputs.DYN_SEED)
    g1.db_step(333); o1.step(333)
    cnt, first = g1.db_region_counts()
    assert np.array_equal(cnt, o1.region_counts()[first:first + len(cnt)]) and cnt.sum() > 50


@pytest.mark.parametrize("mode", MODES)
def test_synchronised_burst_overflows_the_block_lists(db, oracle_mod, mode):
    # P:L490 worries about synchronised activity; here EVERY neuron of a 400,037-neuron network fires in step 0.  One block
    # of the persistent kernel owns ~2,800 neurons (> kSpkCap = 1024 staged spikes: the rest reserve raster positions
    # straight from the global cursor) and 640 of the first 2,700 rows are longer than kInlineMax = 1024 synapses
    # (> kHeavyListCap = 512 deferred heavy rows: the rest are pushed by the warp that found them).
    N = 400_000 + 37
    rng = np.random.default_rng(5)
    heavy = {int(r): int(d) for r, d in zip(rng.choice(2700, 640, replace=False), rng.integers(1025, 1400, 640))}
    heavy.update({150_000: 20_000, 399_999: 3000})
    net = db_inputs.bulk_csr(N, base_outdeg=3, seed=9, heavy_rows=heavy)
    t = db_inputs.type_params(bg_weight=0.03)
    sim = db_inputs.sim_params(types=[t, dict(t)])
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    assert g.db_get_counters()["exec_mode"] == mode
    V, gg, ref = o.state()
    V[:] = -45.0                                                   # above threshold: flagged in step 0
    o.set_state(V, gg, ref); g.set_state(V.astype(np.float32), gg.astype(np.float32), ref)
    g.db_step(1); o.step(1)
    assert g.db_get_counters()["spikes"] == N
    assert _check(g, o, 1) == N
    g.db_step(1); o.step(1)
    _check(g, o, 2)
    g.db_step(118); o.step(118)                                    # past the refractory period: ordinary activity again
    n = _check(g, o, 120)
    assert n > N + 1000
    # a second burst in the middle of a run (odd unit parity of the kernel's double-buffered lists)
    V, gg, ref = o.state()
    V[:] = -45.0
    ref[:] = 0
    o.set_state(V, gg, ref); g.set_state(V.astype(np.float32), gg.astype(np.float32), ref)
    g.db_step(3); o.step(3)
    assert g.db_get_counters()["spikes"] >= n + N
    _check(g, o, 123)        # (deferred mode: the near segments pending across the state write are still pushed)


@pytest.mark.parametrize("mode", MODES)
def test_ring_wrap_and_overflow_flag(db, oracle_mod, mode):
    # R28: the same two's-complement wrap and the same sticky flag on both sides (tests/test_oracle_pins_current.py pins
    # the oracle's: three pushes of 300 * 2^22 wrap to -520,093,696; a consumed cell beyond 2^30 raises the flag)
    t = db_inputs.type_params(bg_weight=0.0, bg_rate_hz=0.0)
    sim = db_inputs.sim_params(D=8, types=[t, dict(t)])
    net = dict(N=4, n_regions=1, region_start=np.array([0, 4]), ntype=np.zeros(4, np.uint8),
               row_ptr=np.array([0, 1, 2, 3, 3], np.int64), tgt=np.array([3, 3, 3], np.int32),
               w=np.array([300.0] * 3, np.float32), delay=np.array([2, 2, 2], np.uint8), rec=np.zeros(3, np.uint8))
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    V, gg, ref = o.state()
    V[:3], V[3] = -40.0, t["VL"]
    o.set_state(V, gg, ref); g.set_state(V.astype(np.float32), gg.astype(np.float32), ref)
    g.db_step(1); o.step(1)
    ring = g.db_read_state(7)
    assert ring[2, 3, 0] == -520093696 and np.array_equal(ring, o.ring())
    g.db_step(2); o.step(2)
    _check(g, o, 3)
    assert g.db_get_counters()["ring_overflow"] == 0
    g.db_step(3); o.step(3)
    _check(g, o, 6)
    # trip the flag: a cell of 2^30 + 1 (and -2^30 - 1), consumed in the next step; 2^30 itself does not trip it
    lone = dict(net, row_ptr=np.zeros(5, np.int64), tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32),
                delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))
    for val, trips in ((1 << 30, 0), (-(1 << 30), 0), ((1 << 30) + 1, 1), (-(1 << 30) - 1, 1)):
        g = db.Sim.db_create_from_csr(sim, lone, exec_mode=mode)
        o = oracle_mod.OracleSim(sim, lone, db_inputs.DYN_SEED)
        r = np.zeros((8, 4, 4), np.int32)
        r[0, 1, 2] = val
        g.db_write_state(7, r); o.set_ring(r)
        g.db_step(1); o.step(1)
        assert g.db_get_counters()["ring_overflow"] == trips == o.counters()["overflow"]
        g.db_step(4); o.step(4)
        assert g.db_get_counters()["ring_overflow"] == trips == o.counters()["overflow"]     # sticky
        assert np.array_equal(g.state()[1], o.state()[1].astype(np.float32))


def test_deferred_mode_ring_write_after_the_first_step_is_refused(db):
    # in deferred mode the ring the API shows is the device ring plus the near segments not pushed yet; once spikes may be
    # pending a write could not be read back as written, so it is refused (include/db_b200.h, db_write_state)
    net = db_inputs.random_csr(N=600, mean_outdeg=10, seed=2)
    sim = db_inputs.sim_params()
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=3)
    assert g.db_get_counters()["exec_mode"] == 3
    r = np.zeros((sim["D"], 600, 4), np.int32)
    r[3, 5, 1] = 77
    g.db_write_state(7, r)                         # step 0: nothing pending
    assert np.array_equal(g.db_read_state(7), r)
    g.db_step(2)
    with pytest.raises(db.DbError) as e:
        g.db_write_state(7, r)
    assert e.value.code == db.binding.DB_ESTATE
    g.db_write_state(0, np.full(600, -60.0, np.float32))            # the other fields stay writable


@pytest.mark.parametrize("mode", MODES)
def test_per_neuron_external_current_from_a_gamma_law(db, oracle_mod, mode):
    # SURVEY 8(f) row 1, remainder: I_ext,i "independently sampled following a Gamma distribution" (R31) on
    # one type, the constant of the type on the other; the plane is one more stream of the update (read only)
    exc, inh = _distinct_types()
    exc.update(Iext=0.05, iext_gamma_shape=2.5, iext_gamma_scale=0.06)
    sim = db_inputs.sim_params(types=[exc, inh])
    N = 7000 + 21
    net = db_inputs.random_csr(N=N, mean_outdeg=25, seed=33, n_regions=2)
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    Ig, Io = g.db_read_state(db.FIELD_IEXT), o.iext().astype(np.float32)
    assert np.array_equal(Ig, Io)                                     # same table, same Philox words, one fp32 addition
    assert np.all(Ig[net["ntype"] == 1] == np.float32(-0.05)) and Ig[net["ntype"] == 0].std() > 0.05
    for upto in (1, 2, 80, 400):
        g.db_step(upto - int(g.db_get_counters()["steps"])); o.step(upto - o.step_index)
        n = _check(g, o, upto)
    assert n > 300
    assert np.array_equal(g.db_read_state(db.FIELD_IEXT), Io)         # a parameter: the step loop does not touch it
    # the plane can be rewritten (e.g. by an assimilation loop): the dynamics follow the written values
    g.db_write_state(db.FIELD_IEXT, np.full(N, 0.05, np.float32))
    h = db.Sim.db_create_from_csr(db_inputs.sim_params(types=[dict(exc, iext_gamma_shape=0.0), inh]), net, exec_mode=mode)
    assert np.all(h.db_read_state(db.FIELD_IEXT)[net["ntype"] == 0] == np.float32(0.05))      # no plane: the constants
    with pytest.raises(db.DbError) as e:
        h.db_write_state(db.FIELD_IEXT, Io)
    assert e.value.code == db.binding.DB_ESTATE


def _run_shards(db, shards, bounds, steps, every, window=False, peer=False):
    """Step the handles `shards` (owning [bounds[k], bounds[k + 1])) together: every `every` steps each one's new spikes go
    to all the others (db_read_spikes -> db_deliver_external step by step, or db_deliver_external_window once).  Returns
    the merged raster."""
    done, all_st, all_id = 0, [], []
    while done < steps:
        n = min(every, steps - done)
        for s in shards:
            s.db_step(n)
        fresh = [s.db_read_spikes(done, done + n) for s in shards]
        for k, dst in enumerate(shards):
            for j, (st, ids) in enumerate(fresh):
                if j == k:
                    continue
                if peer:
                    dst.db_exchange_peer(shards[j], done, done + n)
                    continue
                if window:
                    dst.db_deliver_external_window(done, n, st, ids)
                    continue
                for step in np.unique(st):
                    dst.db_deliver_external(int(step), ids[st == step])
        for st, ids in fresh:
            all_st.append(st); all_id.append(ids)
        done += n
    st, ids = np.concatenate(all_st), np.concatenate(all_id)
    order = np.lexsort((ids, st))
    return st[order], ids[order]


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("source", ["csr", "generator", "peer"])     # exchange: one call per step / per window / device to device
def test_two_handles_that_own_half_of_the_targets_each_reproduce_the_whole(db, oracle_mod, mode, source):
    # SURVEY 8(f) row 3, the half that one GPU can test (SI Eq.(6); layout P:L494): each handle owns a range of
    # targets -- state, ring and the synapses onto them from EVERY source -- and receives the other's spikes as id lists
    # every d_min steps.  Raster, state, ring and counters must be those of the oracle's single whole network, bit for bit.
    cfg = db_inputs.config(2, scale=0.004)                       # 20,000 neurons in regions, K = 160 + 40, inter delays 20..200
    cfg["net"].update(n_regions=8, delay_intra_min=3, delay_inter_min=20)
    t = db_inputs.type_params(bg_weight=0.02)
    t.update(G=[0.5, 0.125, 0.5, 0.5], ou_mu=0.3, ou_sigma=0.1, ou_tau_ms=10.0)       # Poisson and OU draws: both keyed by global id
    cfg["sim"]["types"] = [t, dict(t)]
    N = cfg["net"]["N"]
    net = oracle_mod.generate(cfg["net"], db_inputs.GEN_SEED)
    o = oracle_mod.OracleSim(cfg["sim"], net, db_inputs.DYN_SEED)
    cut = 9 * 1024                                               # not a region boundary, not half
    bounds = [0, cut, N]
    if source == "csr":
        shards = [db.Sim.db_create_from_csr(cfg["sim"], net, exec_mode=mode, own=(bounds[k], bounds[k + 1] - bounds[k])) for k in range(2)]
    else:
        # a small raster ring makes db_exchange_peer check the sender's counters first (its slower, validating path)
        shards = [db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, exec_mode=mode,
                                   raster_capacity=(1 << 14) if (source == "peer" and mode != 2) else 0,
                                   own=(bounds[k], bounds[k + 1] - bounds[k])) for k in range(2)]
    Vo = o.state()[0].astype(np.float32)
    for k, s in enumerate(shards):
        assert np.array_equal(s.db_read_state(db.FIELD_V), Vo[bounds[k]:bounds[k + 1]])          # V0 keyed by global id
        assert np.array_equal(s.db_read_state(db.FIELD_TYPE), net["ntype"][bounds[k]:bounds[k + 1]])
    steps, d_min = 300, 3
    st, ids = _run_shards(db, shards, bounds, steps, d_min, window=(source == "generator"), peer=(source == "peer"))
    o.step(steps)
    so, io = o.spikes()
    order = np.lexsort((io, so))
    assert np.array_equal(st, so[order]) and np.array_equal(ids, io[order]) and len(ids) > 500
    assert np.count_nonzero(ids < cut) > 100 and np.count_nonzero(ids >= cut) > 100
    Vo, go, ro = o.state()
    ring = o.ring()
    for k, s in enumerate(shards):
        a, b = bounds[k], bounds[k + 1]
        Vg, gg, rg = s.state()
        assert np.array_equal(Vg, Vo[a:b].astype(np.float32)) and np.array_equal(gg, go[a:b].astype(np.float32)) and np.array_equal(rg, ro[a:b])
        assert np.array_equal(s.db_read_state(db.FIELD_RING), ring[:, a:b, :])
        assert np.array_equal(s.db_read_state(db.FIELD_IOU), o.iou()[a:b].astype(np.float32))
    cs = [s.db_get_counters() for s in shards]
    co = o.counters()
    assert sum(c["events"] for c in cs) == co["events"] and sum(c["spikes"] for c in cs) == co["spikes"]
    assert sum(c["bg_events"] for c in cs) == co["bg_events"]
    # argument checks: an owned id, an id out of range, a spike whose arrivals are already in the past
    with pytest.raises(db.DbError):
        shards[0].db_deliver_external(steps - 1, np.array([5], np.int32))
    with pytest.raises(db.DbError):
        shards[0].db_deliver_external(steps - 1, np.array([N], np.int32))
    with pytest.raises(db.DbError) as e:
        shards[0].db_deliver_external(steps - 10, np.array([cut + 1], np.int32))
    assert e.value.code == db.binding.DB_ERANGE
    with pytest.raises(db.DbError):
        shards[1].db_read_state(db.FIELD_V, first=0, count=10)       # not its neurons
    with pytest.raises(db.DbError) as e:                              # device-to-device: too late, not simulated yet, same handle
        shards[0].db_exchange_peer(shards[1], steps - 12, steps - 6)
    assert e.value.code == db.binding.DB_ERANGE
    with pytest.raises(db.DbError) as e:
        shards[0].db_exchange_peer(shards[1], steps - 1, steps + 1)
    assert e.value.code == db.binding.DB_ERANGE
    with pytest.raises(db.DbError):
        shards[0].db_exchange_peer(shards[0], steps - 1, steps)
    with pytest.raises(db.DbError) as e:                              # window: the first step that carries spikes is too late
        shards[0].db_deliver_external_window(steps - 12, 12, np.array([steps - 10, steps - 1]), np.array([cut + 1, cut + 2], np.int32))
    assert e.value.code == db.binding.DB_ERANGE
    with pytest.raises(db.DbError):
        shards[0].db_deliver_external_window(steps - 2, 2, np.array([steps - 1]), np.array([5], np.int32))      # owned id


@pytest.mark.parametrize("mode", MODES)
def test_eight_neuron_types_with_their_own_constants(db, oracle_mod, mode):
    # R-D1: the property table is held per type; eight types cover the populations of a micro-column (Ext. Table 3)
    # or (region group, type) pairs.  Types are interleaved neuron by neuron, so almost every 4-neuron group of a thread
    # mixes types (the slow path of neuron_group), and every constant differs between types.
    rng = np.random.default_rng(77)
    types = []
    for k in range(8):
        t = db_inputs.type_params(bg_weight=0.006 + 0.001 * k, bg_rate_hz=800.0 + 100.0 * k)
        t.update(Iext=0.02 * k - 0.05, C=0.8 + 0.05 * k, gL=0.025 + 0.002 * k, VL=-76.0 + 0.5 * k, Vth=-51.0 + 0.3 * k,
                 Vreset=-66.0 + 0.4 * k, Tref_ms=2.0 + 0.5 * k,
                 G=[1.0 + 0.05 * k, 0.25 - 0.01 * k, 1.0 - 0.03 * k, 1.0 + 0.02 * k],
                 E=[0.0 + 0.5 * k, -1.0 * k, -70.0 - k, -100.0 + k], tau_ms=[2.0 + 0.1 * k, 40.0 - k, 10.0 + 0.5 * k, 50.0 - 2 * k])
        if k in (2, 5):
            t.update(ou_mu=0.5, ou_sigma=0.1, ou_tau_ms=8.0 + k)
        if k in (3, 5):
            t.update(iext_gamma_shape=2.0, iext_gamma_scale=0.03)
        types.append(t)
    sim = db_inputs.sim_params(types=types)
    N = 5000 + 11
    net = db_inputs.random_csr(N=N, mean_outdeg=25, seed=55)
    net["ntype"] = rng.integers(0, 8, N).astype(np.uint8)
    net["rec"] = (2 * (net["ntype"][np.repeat(np.arange(N), np.diff(net["row_ptr"]))] % 2) + (net["rec"] % 2)).astype(np.uint8)
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    assert np.array_equal(g.db_read_state(db.FIELD_TYPE), net["ntype"])
    assert np.array_equal(g.db_read_state(db.FIELD_IEXT), o.iext().astype(np.float32))
    for upto in (1, 3, 90, 500):
        g.db_step(upto - int(g.db_get_counters()["steps"])); o.step(upto - o.step_index)
        n = _check(g, o, upto)
        assert np.array_equal(g.db_read_state(db.FIELD_IOU), o.iou().astype(np.float32))
    ids = g.db_read_spikes(0, 500)[1]
    assert all(np.count_nonzero(net["ntype"][ids] == k) > 5 for k in range(8)), np.bincount(net["ntype"][ids], minlength=8)
    with pytest.raises(db.DbError):
        db.Sim.db_create_from_csr(db_inputs.sim_params(types=types + [types[0]]), net)      # nine types


def test_bold_readout_keeps_up_inside_db_step_profiled(db, oracle_mod):
    # db_step_profiled (CUDA events around every kernel) lets the BOLD read-out catch up before its short count history wraps
    N, R = 3000, 5
    net = db_inputs.random_csr(N=N, mean_outdeg=25, seed=8, n_regions=R)
    t = db_inputs.type_params(bg_weight=0.02)
    sim = db_inputs.sim_params(types=[t, dict(t)])
    sim["bold"] = dict(oracle_mod.BOLD_DEFAULTS)
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=1, max_windows=16)     # history of 13 windows = 130 steps
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    prof = g.db_step_profiled(700)
    o.step(700)
    assert prof["steps"] == 700 and prof["update_ms"] > 0 and prof["deliver_ms"] > 0
    y, st, n = g.db_read_bold()
    sizes = np.diff(net["region_start"])
    ys, so = oracle_mod.bold_run(o.region_counts()[:n], sizes, sim["window_steps"] * sim["dt_ms"] * 1e-3, sim["bold"])
    assert n == 70 and np.max(np.abs(st - so)) < 1e-10 and np.max(np.abs(y - ys[-1])) < 1e-10


@pytest.mark.parametrize("mode", MODES)
def test_cortical_microcolumn_workload(db, oracle_mod, mode):
    # SURVEY 8(f), unranked extra: voxels of the cortical laminar model (Extended Data Table 3),
    # ten populations per voxel with the table's population-specific in-degrees, cortico-cortical input from the
    # excitatory neurons of the other voxels (db_inputs.microcolumn_csr; 8 voxels x 4,000 neurons, d_in = 100:
    # 3.2e6 synapses, in-degrees 38-180, out-degrees 0-~500).  Voxel = region, so a4 gives the voxel rates.
    net = db_inputs.microcolumn_csr(8, 4000, 100, seed=21)
    t = db_inputs.type_params(bg_weight=0.0072)
    sim = db_inputs.sim_params(types=[t, dict(t)], D=32)
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    assert g.db_get_counters()["exec_mode"] == mode
    for steps in (1, 50, 400):
        g.db_step(steps - int(g.db_get_counters()["steps"])); o.step(steps - int(o.counters()["steps"]))
        n = _check(g, o, steps)
    assert n > 2000                                                # ~14 Hz (tests/test_inputs_microcolumn.py)
    cnt, first = g.db_region_counts()
    assert len(cnt) >= 30 and np.array_equal(cnt, o.region_counts()[first:first + len(cnt)])
    # e1 neurons (the first 640 of every voxel) send nothing inside their voxel: only their cortico-cortical share
    deg = np.diff(net["row_ptr"])
    assert deg[:640].mean() < 0.5 * deg[800:1440].mean()


@pytest.mark.parametrize("mode", [1, 3])
def test_graph_replay_starts_on_an_even_step_whatever_the_batch_sizes(db, oracle_mod, mode):
    # The step graph of the two-kernel modes (32 steps) carries the parity of the work-list half in its launches, so it may
    # only be replayed from an even step.  Found by tests/test_gpu_parity_random.py: a db_step call that reached the graph
    # with an odd step count and EXACTLY 32 steps left replayed it misaligned (list mode: wrong arrival lists consumed).
    net = db_inputs.random_csr(N=3000 + 21, mean_outdeg=40, seed=33, max_delay=20)
    t = db_inputs.type_params(bg_weight=0.012)
    sim = db_inputs.sim_params(types=[t, dict(t)])
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    assert g.db_get_counters()["exec_mode"] == mode
    done = 0
    for b in (40, 33, 32, 31, 65, 33, 1, 32, 64, 34):      # graph built by the first call; 33 = prologue + 32 from an odd step
        g.db_step(b); o.step(b); done += b
        _check(g, o, done)
    assert g.db_get_counters()["spikes"] > 500


@pytest.mark.parametrize("mode", MODES)
def test_long_run_past_the_wrap_of_the_step_log_and_the_raster_ring(db, oracle_mod, mode):
    # 70,000 steps (7 s of model time at dt 0.1 ms): the step log (2^16 entries) and a small raster ring wrap several
    # times, the rotating arrival counters of the persistent kernel run through 70,000 units in a few launches, the region
    # history wraps.  State, ring, counters and the recent raster must still be the oracle's; old ranges are refused.
    N = 1500 + 11
    net = db_inputs.random_csr(N=N, mean_outdeg=15, seed=44, max_delay=20, n_regions=3)
    t = db_inputs.type_params(bg_weight=0.012)
    sim = db_inputs.sim_params(types=[t, dict(t)], window_steps=7)
    g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode, raster_capacity=1 << 13, max_windows=64)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    done = 0
    for b in (1, 33001, 999, 32768, 3231):
        g.db_step(b); o.step(b); done += b
        Vg, gg, rg = g.state()
        Vo, go, ro = o.state()
        assert np.array_equal(rg, ro) and np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32)), done
        assert np.array_equal(g.db_read_state(db.FIELD_RING), o.ring()), done
    assert done == 70000
    cg, co = g.db_get_counters(), o.counters()
    for k in ("steps", "spikes", "events", "bg_events"):
        assert cg[k] == co[k], k
    assert co["spikes"] > 5 * (1 << 13)                               # the raster ring has wrapped several times
    so, io = o.spikes()
    for a, b in ((done - 300, done), (done - 1200, done - 900), (done - 1, done)):      # ~4.6 spikes per step: 8192 entries hold ~1,700 steps
        sg, ig = g.db_read_spikes(a, b)
        sel = (so >= a) & (so < b)
        order = np.lexsort((io[sel], so[sel]))
        assert np.array_equal(sg, so[sel][order]) and np.array_equal(ig, io[sel][order]), (a, b)
    with pytest.raises(db.DbError) as e:
        g.db_read_spikes(0, 100)                                       # overwritten long ago
    assert e.value.code == db.binding.DB_ERANGE
    cnt, first = g.db_region_counts()
    assert first > 0 and np.array_equal(cnt, o.region_counts()[first:first + len(cnt)])


def test_device_to_device_exchange_between_handles_on_different_streams(db, oracle_mod):
    # db_exchange_peer orders the receiver's stream after the sender's steps with an event when the two handles run on
    # different streams (the handles of the other tests share torch's current stream).  Nothing here synchronises the
    # host between the steps and the exchanges.
    import torch
    cfg = db_inputs.config(2, scale=0.004)
    cfg["net"].update(n_regions=8, delay_intra_min=4, delay_inter_min=20)
    t = db_inputs.type_params(bg_weight=0.02)
    t.update(G=[0.5, 0.125, 0.5, 0.5])
    cfg["sim"]["types"] = [t, dict(t)]
    N = cfg["net"]["N"]
    net = oracle_mod.generate(cfg["net"], db_inputs.GEN_SEED)
    o = oracle_mod.OracleSim(cfg["sim"], net, db_inputs.DYN_SEED)
    bounds = [0, 7 * 1024, 13 * 1024, N]
    streams = [torch.cuda.Stream() for _ in range(3)]
    shards = []
    for k in range(3):
        with torch.cuda.stream(streams[k]):              # the handle keeps the stream that is current when it is created
            shards.append(db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, exec_mode=[2, 1, 3][k],
                                           own=(bounds[k], bounds[k + 1] - bounds[k])))
    from paper_2211_15963_b200 import sharded
    sharded.run_local(shards, 240, 4)
    torch.cuda.synchronize()
    o.step(240)
    so, io = o.spikes()
    order = np.lexsort((io, so))
    parts = [s.db_read_spikes(0, 240) for s in shards]
    st, ids = np.concatenate([a for a, _ in parts]), np.concatenate([b for _, b in parts])
    od = np.lexsort((ids, st))
    assert np.array_equal(st[od], so[order]) and np.array_equal(ids[od], io[order]) and len(ids) > 300
    Vo, go, ro = o.state()
    ring = o.ring()
    for k, s in enumerate(shards):
        a, b = bounds[k], bounds[k + 1]
        Vg, gg, rg = s.state()
        assert np.array_equal(Vg, Vo[a:b].astype(np.float32)) and np.array_equal(gg, go[a:b].astype(np.float32)) and np.array_equal(rg, ro[a:b])
        assert np.array_equal(s.db_read_state(db.FIELD_RING), ring[:, a:b, :])
    assert sum(s.db_get_counters()["events"] for s in shards) == o.counters()["events"]
