"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (db_create on the
device, DB_EXEC_AUTO).

configs[1] (the bench workload, 1e6 neurons / 1e8 synapses): the oracle generates the same network itself (the export must equal it array
for array) and runs it closed loop: raster, fp32 state and the fixed-point ring must be identical.

configs[2] / [3] (5e6 / 1e7 neurons, 1e9 / 1e10 synapses): open-loop replay of a chunk T of target
neurons (SURVEY 8(c) "Oracle at scale").  The oracle's generator yields the incoming synapses of T
only (oracle.OwnerEdges); the arrivals into T are recomputed from the GPU's full raster with the plain
definition a_n[i][u] = sum_s wq_s spike_src(s)(n - d_s); the oracle steps T on those arrivals and T's
spikes and state must equal the GPU's.  By induction over the steps this checks generator, delivery and
update for the sampled targets.  Properties that hold at any size cover the rest: event conservation
(events = sum of out-degrees of the spiking neurons), region counts recounted from the raster, and the
two execution modes agreeing bit for bit.

configs[4] (out-degree mode, 2e6 neurons): sampled rows against the oracle's generator, the same
properties, and the two modes agreeing.
"""
import numpy as np
import pytest

import db_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def db():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2211_15963_b200 as m
    m.load()
    return m


def _free():
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()


def _raster_props(s, db, steps, n_regions, region_start, window):
    """events = sum of out-degrees of the spiking neurons; region counts = recount of the raster."""
    st, ids = s.db_read_spikes(0, steps)
    outdeg = s.db_read_state(db.FIELD_OUTDEG)
    c = s.db_get_counters()
    assert c["steps"] == steps and c["spikes"] == len(ids) and c["ring_overflow"] == 0
    assert c["events"] == int(outdeg[ids].astype(np.int64).sum())
    cnt, first = s.db_region_counts()
    assert first == 0 and len(cnt) == steps // window
    reg = np.searchsorted(region_start, ids, side="right") - 1
    win = (st // window).astype(np.int64)
    keep = win < len(cnt)
    want = np.zeros((len(cnt), n_regions), np.int64)
    np.add.at(want, (win[keep], reg[keep]), 1)
    assert np.array_equal(cnt.astype(np.int64), want)
    return st, ids


def test_config1_full_size_closed_loop(db, oracle_mod):
    cfg = db_inputs.config(1)
    steps = 60
    s = db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, dyn_seed=db_inputs.DYN_SEED,
                         raster_capacity=1 << 25)
    assert s.db_get_counters()["exec_mode"] == db.EXEC_PERSISTENT          # what AUTO picks here and bench.py times
    net = oracle_mod.generate(cfg["net"], db_inputs.GEN_SEED)        # the oracle's own network (about 45 s of CPU)
    got = s.db_export_csr()
    for key in ("N", "E", "n_regions"):
        assert got[key] == net[key], key
    for key in ("region_start", "ntype", "row_ptr", "tgt", "rec", "delay", "w"):
        assert np.array_equal(got[key], net[key]), key
    del got
    N, K = cfg["net"]["N"], cfg["net"]["K"]
    assert net["E"] == N * K
    assert np.array_equal(np.bincount(net["tgt"], minlength=N), np.full(N, K))       # exact in-degree
    src = np.repeat(np.arange(N, dtype=np.int32), np.diff(net["row_ptr"]))
    assert not np.any(src == net["tgt"])                                            # no autapse
    assert np.all((net["rec"] >> 1) == net["ntype"][src])                           # receptor class follows the source
    assert net["delay"].min() == 1 and net["delay"].max() == 20
    del src
    o = oracle_mod.OracleSim(cfg["sim"], net, db_inputs.DYN_SEED)
    s.db_step(steps)
    o.step(steps)
    sg, ig = s.db_read_spikes(0, steps)
    so, io = o.spikes()
    k = np.lexsort((io, so))
    assert len(ig) > 1000 and np.array_equal(sg, so[k]) and np.array_equal(ig, io[k])
    Vg, gg, rg = s.state()
    Vo, go, ro = o.state()
    assert np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32))
    assert np.array_equal(rg, ro)
    assert np.array_equal(s.db_read_state(db.FIELD_RING), o.ring())                 # bit-exact fixed point
    cg, co = s.db_get_counters(), o.counters()
    for key in ("steps", "spikes", "events", "bg_events"):
        assert cg[key] == co[key], key
    s.db_destroy()
    o.close()
    _free()
    # the same network in the paper's production mode (`bench.py --drive ou --spike-bin 10`): OU drive, b_t = 10 steps
    import copy
    sim2 = db_inputs.ou_drive(copy.deepcopy(cfg["sim"]))
    sim2["spike_bin_steps"] = 10
    s = db.Sim.db_create(cfg["net"], sim2, seed=db_inputs.GEN_SEED, dyn_seed=db_inputs.DYN_SEED, raster_capacity=1 << 25)
    assert s.db_get_counters()["exec_mode"] == db.EXEC_PERSISTENT
    o = oracle_mod.OracleSim(sim2, net, db_inputs.DYN_SEED)
    s.db_step(40)
    o.step(40)
    sg, ig = s.db_read_spikes(0, 40)
    so, io = o.spikes()
    k = np.lexsort((io, so))
    assert len(ig) > 300 and np.array_equal(sg, so[k]) and np.array_equal(ig, io[k])
    Vg, gg, rg = s.state()
    Vo, go, ro = o.state()
    assert np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32)) and np.array_equal(rg, ro)
    assert np.array_equal(s.db_read_state(db.FIELD_IOU), o.iou().astype(np.float32))
    assert np.array_equal(s.db_read_state(db.FIELD_RING), o.ring())                 # 40 is a bin boundary
    s.db_destroy()
    o.close()
    _free()


def _replay_chunk(db, oracle_mod, cfg, s, steps, m, st, ids):
    """Open-loop replay of the target neurons [0, m) against the GPU's raster (st, ids) of `steps` steps."""
    net_spec, sim = cfg["net"], cfg["sim"]
    S, D = sim["S"], sim["D"]
    own = oracle_mod.OwnerEdges(net_spec, db_inputs.GEN_SEED)
    src, tgt, wq, dl, rec = [], [], [], [], []
    for i in range(m):
        e = own(i)
        assert np.all(e["tgt"] == i)
        src.append(e["src"]); tgt.append(e["tgt"]); dl.append(e["delay"]); rec.append(e["rec"])
        wq.append(np.rint(e["w"].astype(np.float32) * np.float32(2.0 ** S)).astype(np.int64))   # lrintf(w 2^S), SURVEY 8(c) step 9
    ntype = own.ntype(0, m)
    own.close()
    src, tgt, wq, dl, rec = (np.concatenate(x) for x in (src, tgt, wq, dl, rec))
    # spikes of every source, from the GPU raster
    k = np.argsort(ids, kind="stable")
    ids_s, st_s = ids[k], st[k].astype(np.int64)
    lo, hi = np.searchsorted(ids_s, src, side="left"), np.searchsorted(ids_s, src, side="right")
    cnt = hi - lo
    e_idx = np.repeat(np.arange(len(src)), cnt)
    pos = np.concatenate([np.arange(a, b) for a, b in zip(lo[cnt > 0], hi[cnt > 0])]) if cnt.sum() else np.zeros(0, np.int64)
    when = st_s[pos] + dl[e_idx]
    A = np.zeros((steps + D, m, 4), np.int64)
    np.add.at(A, (when, tgt[e_idx], rec[e_idx]), wq[e_idx])
    A = A.astype(np.int32)                          # two's-complement wrap (never reached here)
    assert int(np.count_nonzero(A[:steps])) > 100
    # the chunk as a network without synapses; its arrivals are injected slot by slot
    assert np.array_equal(s.db_read_state(db.FIELD_TYPE, 0, m), ntype)
    sub = dict(N=m, E=0, n_regions=1, region_start=np.array([0, m]), ntype=ntype, row_ptr=np.zeros(m + 1, np.int64),
               tgt=np.zeros(0, np.int32), w=np.zeros(0, np.float32), delay=np.zeros(0, np.uint8), rec=np.zeros(0, np.uint8))
    o = oracle_mod.OracleSim(sim, sub, db_inputs.DYN_SEED)
    ring = np.zeros((D, m, 4), np.int32)
    for n in range(steps):
        ring[:] = 0
        ring[n % D] = A[n]
        o.set_ring(ring)
        o.step(1)
    so, io = o.spikes()
    sel = ids < m
    k = np.lexsort((ids[sel], st[sel]))
    ko = np.lexsort((io, so))
    assert len(io) > 0
    assert np.array_equal(st[sel][k], so[ko]) and np.array_equal(ids[sel][k], io[ko])
    Vo, go, ro = o.state()
    assert np.array_equal(s.db_read_state(db.FIELD_V, 0, m), Vo.astype(np.float32))
    for u in range(4):
        assert np.array_equal(s.db_read_state(db.FIELD_G_AMPA + u, 0, m), go[:, u].astype(np.float32))
    assert np.array_equal(s.db_read_state(db.FIELD_REF, 0, m), ro)
    # and the arrivals still in flight for the chunk are the GPU's ring
    got = s.db_read_state(db.FIELD_RING, 0, m)
    want = np.zeros((D, m, 4), np.int32)
    for n in range(steps, steps + D):
        want[n % D] = A[n]
    assert np.array_equal(got, want)


@pytest.mark.parametrize("idx,steps,m", [(2, 300, 1536), (3, 120, 512)])
def test_region_configs_full_size_replay_and_properties(db, oracle_mod, idx, steps, m):
    cfg = db_inputs.config(idx)
    region_start = None
    keep = {}
    for mode in (db.EXEC_AUTO, "other"):
        if mode == "other":                     # the execution mode AUTO did not pick: an independent schedule
            mode = db.EXEC_KERNELS if keep["mode"] == db.EXEC_PERSISTENT else db.EXEC_PERSISTENT
        s = db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, dyn_seed=db_inputs.DYN_SEED,
                             exec_mode=mode, raster_capacity=1 << 26)
        if region_start is None:
            sizes = oracle_mod.region_sizes(db_inputs.GEN_SEED, cfg["net"]["N"], cfg["net"]["n_regions"],
                                            cfg["net"]["region_size_sigma"])
            region_start = np.concatenate([[0], np.cumsum(sizes)])
        s.db_step(steps)
        st, ids = _raster_props(s, db, steps, cfg["net"]["n_regions"], region_start, cfg["sim"]["window_steps"])
        assert len(ids) > 10 * steps
        if mode == db.EXEC_AUTO:
            _replay_chunk(db, oracle_mod, cfg, s, steps, m, st, ids)
            keep = dict(st=st, ids=ids, V=s.db_read_state(db.FIELD_V), mode=s.db_get_counters()["exec_mode"])
        else:                                   # an independent schedule of the same arithmetic: identical results
            assert np.array_equal(st, keep["st"]) and np.array_equal(ids, keep["ids"])
            assert np.array_equal(s.db_read_state(db.FIELD_V), keep["V"])
        s.db_destroy()
        del s
        _free()


def test_config4_full_size_rows_and_properties(db, oracle_mod):
    cfg = db_inputs.config(4)
    steps = 150
    N = cfg["net"]["N"]
    keep = {}
    for mode in (db.EXEC_AUTO, "other"):
        if mode == "other":
            mode = db.EXEC_KERNELS if keep["mode"] == db.EXEC_PERSISTENT else db.EXEC_PERSISTENT
        s = db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, dyn_seed=db_inputs.DYN_SEED,
                             exec_mode=mode, raster_capacity=1 << 26)
        if mode == db.EXEC_AUTO:
            outdeg = s.db_read_state(db.FIELD_OUTDEG)
            assert outdeg.max() == cfg["net"]["outdeg_cap"] or outdeg.max() > 5000      # the heavy tail is there
            assert abs(outdeg.mean() / cfg["net"]["outdeg_mean"] - 1.0) < 0.02
            own = oracle_mod.OwnerEdges(cfg["net"], db_inputs.GEN_SEED)
            for j in (0, 1, N - 1, int(np.argmax(outdeg)), int(np.argmin(outdeg)), 1_234_567):
                assert len(own(j)["tgt"]) == outdeg[j]                              # row lengths = the oracle's draws
            own.close()
        s.db_step(steps)
        st, ids = _raster_props(s, db, steps, 1, np.array([0, N]), cfg["sim"]["window_steps"])
        assert len(ids) > 10 * steps
        if mode == db.EXEC_AUTO:
            keep = dict(st=st, ids=ids, V=s.db_read_state(db.FIELD_V), ring0=s.db_read_state(db.FIELD_RING, 0, 4096),
                        mode=s.db_get_counters()["exec_mode"])
        else:
            assert np.array_equal(st, keep["st"]) and np.array_equal(ids, keep["ids"])
            assert np.array_equal(s.db_read_state(db.FIELD_V), keep["V"])
            assert np.array_equal(s.db_read_state(db.FIELD_RING, 0, 4096), keep["ring0"])
        s.db_destroy()
        del s
        _free()
