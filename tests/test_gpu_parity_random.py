"""Randomised differential test: networks, constants and run-time options drawn at random (seeded), the CUDA path against
the oracle in all three execution modes.  Every case combines options the hand-written cases cover one or two at a
time: 1-8 neuron types with their own constants, dt 0.1 / 1 ms, ring depth, region windows of 1-12 steps, spike time
bin, OU current and Poisson background side by side, per-neuron I_ext, fp16 weights, heavy rows, ragged sizes, regions,
uneven db_step batches.  Bars as in tests/test_gpu_parity.py: ring, raster and counters bit-exact, state equal."""
import os

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


def _draw_case(seed):
    rng = np.random.default_rng(1000 + seed)
    n_types = int(rng.integers(1, 9))
    dt = 1.0 if seed % 4 == 3 else 0.1
    types = []
    for k in range(n_types):
        t = db_inputs.type_params(bg_weight=float(rng.uniform(0.004, 0.02)) * (0.15 if dt == 1.0 else 1.0),
                                  bg_rate_hz=float(rng.choice([0.0, 500.0, 1000.0, 2000.0])))
        t.update(C=float(rng.uniform(0.6, 1.2)), gL=float(rng.uniform(0.02, 0.06)), VL=float(rng.uniform(-76.0, -68.0)),
                 Vth=float(rng.uniform(-54.0, -48.0)), Vreset=float(rng.uniform(-66.0, -58.0)), Tref_ms=float(rng.choice([0.0, 1.0, 2.0, 5.0])),
                 Iext=float(rng.uniform(-0.05, 0.25)),
                 G=[float(x) for x in rng.uniform(0.2, 1.3, 4)], E=[float(rng.uniform(-5, 5)), float(rng.uniform(-5, 5)),
                                                                   float(rng.uniform(-80, -65)), float(rng.uniform(-100, -85))],
                 tau_ms=[float(rng.uniform(1.5, 4)), float(rng.uniform(20, 60)), float(rng.uniform(5, 12)), float(rng.uniform(30, 80))])
        if rng.random() < 0.4:
            t.update(ou_mu=float(rng.uniform(0.1, 0.5)), ou_sigma=float(rng.uniform(0.05, 0.2)), ou_tau_ms=float(rng.uniform(2.0, 20.0)))
        if rng.random() < 0.3:
            t.update(iext_gamma_shape=float(rng.uniform(1.0, 6.0)), iext_gamma_scale=float(rng.uniform(0.005, 0.03)))
        types.append(t)
    max_delay = int(rng.choice([1, 3, 20, 60]))
    bin_steps = int(rng.choice([1, 1, 2, 5])) if dt == 0.1 else 1
    if bin_steps > 1:                                  # the library wants b_t <= round(Tref / dt) + 1 for every type (R29)
        for t in types:
            t["Tref_ms"] = max(t["Tref_ms"], 1.0)
    D = 32
    while D < max_delay + 3 + bin_steps:
        D *= 2
    sim = db_inputs.sim_params(dt_ms=dt, D=D, window_steps=int(rng.integers(1, 13)), types=types, spike_bin_steps=bin_steps)
    N = [4097, 31, 2, 1000, 20011, 129, 1, 5000, 2048, 777, 20011, 4097, 1000, 12345][seed % 14]
    n_regions = int(rng.choice([1, 1, 3, 7])) if N >= 1000 else 1
    fp16 = bool(rng.random() < 0.3)
    heavy = {}
    if N >= 4097 and rng.random() < 0.5:
        heavy = {int(r): int(d) for r, d in zip(rng.choice(N, 3, replace=False), rng.integers(1100, min(N - 1, 3000), 3))}
    net = db_inputs.random_csr(N=N, mean_outdeg=float(rng.choice([0.0, 3.0, 20.0, 60.0])) if N > 2 else 1.0, seed=int(seed),
                               max_delay=max_delay, n_regions=n_regions, fp16=fp16, heavy_rows=heavy or None)
    net["ntype"] = (rng.integers(0, n_types, N)).astype(np.uint8) if n_types > 2 else np.minimum(net["ntype"], n_types - 1).astype(np.uint8)
    batches = [int(x) for x in rng.integers(1, 40, 6)]
    return sim, net, fp16, batches


@pytest.mark.parametrize("seed", range(int(os.environ.get("DB_RANDOM_CASES", "14"))))    # more cases: DB_RANDOM_CASES=200 pytest ...
def test_random_configuration_matches_the_oracle(db, oracle_mod, seed):
    sim, net, fp16, batches = _draw_case(seed)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    rings = []
    for b in batches:
        o.step(b)
        rings.append(o.ring().copy())
    done = sum(batches)
    Vo, go, ro = o.state()
    so, io = o.spikes()
    order = np.lexsort((io, so))
    co = o.counters()
    ou = any("ou_mu" in t for t in sim["types"])
    for mode in (1, 2, 3):
        g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode, fp16=fp16)
        used = g.db_get_counters()["exec_mode"]
        assert used == mode or (mode == 3 and used == 1)      # no arrival lists where every delay is one step
        at = 0
        for b, ring in zip(batches, rings):
            g.db_step(b)
            at += b
            if at % sim["spike_bin_steps"] == 0:         # inside a time bin the device ring already holds the open bin's pushes
                assert np.array_equal(g.db_read_state(db.FIELD_RING), ring), (seed, mode, at)
        Vg, gg, rg = g.state()
        assert np.array_equal(rg, ro) and np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32)), (seed, mode)
        sg, ig = g.db_read_spikes(0, done)
        assert np.array_equal(sg, so[order]) and np.array_equal(ig, io[order]), (seed, mode)
        cg = g.db_get_counters()
        for k in ("steps", "spikes", "events", "bg_events"):
            assert cg[k] == co[k], (k, seed, mode)
        assert cg["ring_overflow"] == co["overflow"]
        cnt, first = g.db_region_counts()
        assert np.array_equal(cnt, o.region_counts()[first:first + len(cnt)]), (seed, mode)
        if ou:
            assert np.array_equal(g.db_read_state(db.FIELD_IOU), o.iou().astype(np.float32)), (seed, mode)
        g.db_destroy()


def _draw_spec(seed):
    """A random network SPEC for the on-device generator (both sides generate it themselves) and plain constants."""
    rng = np.random.default_rng(5000 + seed)
    mode = int(rng.random() < 0.3)
    n_regions = 1 if mode else int(rng.choice([1, 1, 4, 9]))           # the out-degree recipe has one region
    N = int(rng.choice([3000, 5037, 8192, 12001]))
    K = int(rng.choice([20, 60, 120]))
    d_lo = int(rng.choice([1, 1, 3]))
    net = db_inputs._net(N=N, n_regions=n_regions, region_size_sigma=float(rng.choice([0.0, 0.7])), mode=mode,
                         K=0 if mode else K, intra_frac=1.0 if n_regions == 1 else float(rng.choice([0.6, 0.8])),
                         outdeg_mean=float(rng.choice([30.0, 80.0])), outdeg_sigma=float(rng.choice([0.5, 1.0])), outdeg_cap=int(rng.choice([400, 2500])),
                         delay_intra_min=d_lo, delay_intra_max=int(rng.choice([d_lo, 8, 20])),
                         delay_inter_min=int(rng.choice([5, 20])), delay_inter_max=int(rng.choice([20, 40, 90])),
                         weight_fp16=int(rng.random() < 0.3))
    max_delay = max(net["delay_intra_max"], net["delay_inter_max"] if n_regions > 1 else 0)
    D = 32
    while D < max_delay + 4:
        D *= 2
    t = db_inputs.type_params(bg_weight=float(rng.uniform(0.008, 0.02)))
    u = dict(t)
    u.update(Vth=-51.0, Tref_ms=1.0, G=[0.9, 0.3, 1.1, 0.8])
    sim = db_inputs.sim_params(D=D, window_steps=int(rng.integers(1, 12)), types=[t, u])
    return rng, net, sim


@pytest.mark.parametrize("seed", range(int(os.environ.get("DB_RANDOM_CASES", "8"))))
def test_random_call_sequences_on_generated_networks(db, oracle_mod, seed):
    # db_step, db_step_profiled (two-kernel modes), state writes and partial read-backs interleaved at random
    rng, net, sim = _draw_spec(seed)
    try:
        csr = oracle_mod.generate(net, db_inputs.GEN_SEED + seed)
    except ValueError:                                 # a region smaller than the in-degree drawn from it: not a network
        pytest.skip("random spec not realisable")
    N = net["N"]
    bold = seed % 2 == 1                               # BOLD read-out with a short count history: db_step lets it catch up
    if bold:
        sim["bold"] = dict(oracle_mod.BOLD_DEFAULTS)
    max_windows = int(rng.choice([16, 64])) if bold else 0
    sizes = np.diff(csr["region_start"])
    win_s = sim["window_steps"] * sim["dt_ms"] * 1e-3
    ops = []
    for _ in range(10):
        r = rng.random()
        if r < 0.55:
            ops.append(("step", int(rng.integers(1, 70))))
        elif r < 0.75:
            ops.append(("prof", int(rng.integers(1, 40))))
        elif r < 0.9:
            ops.append(("write", int(rng.integers(0, 1 << 30))))
        else:
            ops.append(("read", None))
    for mode in (1, 2, 3):
        g = db.Sim.db_create(net, sim, seed=db_inputs.GEN_SEED + seed, exec_mode=mode, max_windows=max_windows)
        o = oracle_mod.OracleSim(sim, csr, db_inputs.DYN_SEED)
        used = g.db_get_counters()["exec_mode"]
        done = 0
        for op, arg in ops:
            if op == "step" or (op == "prof" and used == 2):
                g.db_step(arg); o.step(arg); done += arg
            elif op == "prof":
                g.db_step_profiled(arg); o.step(arg); done += arg
            elif op == "write":
                r2 = np.random.default_rng(arg)
                V = r2.uniform(-75.0, -49.5, N).astype(np.float32)
                gg = r2.gamma(1.0, 0.03, (N, 4)).astype(np.float32)
                ref = np.where(r2.random(N) < 0.1, r2.integers(1, 15, N), 0).astype(np.int32)
                g.set_state(V, gg, ref); o.set_state(V, gg, ref)
            elif done:
                a = int(rng.integers(0, done)); b = int(rng.integers(a, done + 1))
                sg, ig = g.db_read_spikes(a, b)
                so, io = o.spikes()
                sel = (so >= a) & (so < b)
                order = np.lexsort((io[sel], so[sel]))
                assert np.array_equal(sg, so[sel][order]) and np.array_equal(ig, io[sel][order]), (seed, mode, a, b)
            assert np.array_equal(g.db_read_state(db.FIELD_RING), o.ring()), (seed, mode, op, done)
        Vg, gg, rg = g.state()
        Vo, go, ro = o.state()
        assert np.array_equal(rg, ro) and np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32)), (seed, mode)
        sg, ig = g.db_read_spikes(0, done)
        so, io = o.spikes()
        order = np.lexsort((io, so))
        assert np.array_equal(sg, so[order]) and np.array_equal(ig, io[order]), (seed, mode)
        cg, co = g.db_get_counters(), o.counters()
        for k in ("steps", "spikes", "events", "bg_events"):
            assert cg[k] == co[k], (k, seed, mode)
        cnt, first = g.db_region_counts()
        assert np.array_equal(cnt, o.region_counts()[first:first + len(cnt)]), (seed, mode)
        if bold:
            y, stb, n = g.db_read_bold()
            assert n == done // sim["window_steps"]
            if n:
                ys, sob = oracle_mod.bold_run(o.region_counts()[:n], sizes, win_s, sim["bold"])
                assert np.max(np.abs(stb - sob)) < 1e-10 and np.max(np.abs(y - ys[-1])) < 1e-10, (seed, mode)
        g.db_destroy()


@pytest.mark.parametrize("seed", range(int(os.environ.get("DB_RANDOM_CASES", "6"))))
def test_random_shardings_reproduce_the_whole_network(db, oracle_mod, seed):
    # two to four handles that own random 1024-aligned ranges, random exchange window <= the smallest delay, the three
    # exchange calls chosen at random per window
    rng, net, sim = _draw_spec(seed)
    net.update(mode=0, K=int(rng.choice([40, 100])) if net["N"] >= 5000 else 40, delay_intra_min=int(rng.choice([2, 3, 6])))
    if net["n_regions"] > 1 and net["N"] < 5000:
        net["region_size_sigma"] = 0.0                 # small regions must still hold K distinct sources
    net["delay_intra_max"] = max(net["delay_intra_max"], net["delay_intra_min"])
    net["delay_inter_min"] = max(net["delay_inter_min"], net["delay_intra_min"])
    net["delay_inter_max"] = max(net["delay_inter_max"], net["delay_inter_min"])
    try:
        csr = oracle_mod.generate(net, db_inputs.GEN_SEED + seed)
    except ValueError:                                 # a region smaller than the in-degree drawn from it: not a network
        pytest.skip("random spec not realisable")
    N = net["N"]
    n_sh = min(int(rng.integers(2, 5)), (N - 1) // 1024 + 1)
    cuts = sorted(int(c) * 1024 for c in rng.choice(np.arange(1, (N - 1) // 1024 + 1), n_sh - 1, replace=False))
    bounds = [0] + cuts + [N]
    d_min = int(rng.integers(1, net["delay_intra_min"] + 1))
    o = oracle_mod.OracleSim(sim, csr, db_inputs.DYN_SEED)
    mode = int(rng.integers(1, 4))
    shards = [db.Sim.db_create(net, sim, seed=db_inputs.GEN_SEED + seed, exec_mode=mode, own=(bounds[k], bounds[k + 1] - bounds[k]))
              for k in range(n_sh)]
    steps, done = 90, 0
    while done < steps:
        n = min(d_min, steps - done)
        for s in shards:
            s.db_step(n)
        how = int(rng.integers(0, 3))
        fresh = [s.db_read_spikes(done, done + n) for s in shards] if how < 2 else None
        for k, dst in enumerate(shards):
            for j, src in enumerate(shards):
                if j == k:
                    continue
                if how == 2:
                    dst.db_exchange_peer(src, done, done + n)
                elif how == 1:
                    if len(fresh[j][1]):
                        dst.db_deliver_external_window(done, n, fresh[j][0], fresh[j][1])
                else:
                    for step in np.unique(fresh[j][0]):
                        dst.db_deliver_external(int(step), fresh[j][1][fresh[j][0] == step])
        done += n
    o.step(steps)
    Vo, go, ro = o.state()
    ring = o.ring()
    so, io = o.spikes()
    order = np.lexsort((io, so))
    st = np.concatenate([s.db_read_spikes(0, steps)[0] for s in shards])
    ids = np.concatenate([s.db_read_spikes(0, steps)[1] for s in shards])
    od = np.lexsort((ids, st))
    assert np.array_equal(st[od], so[order]) and np.array_equal(ids[od], io[order]), (seed, mode, bounds, d_min)
    for k, s in enumerate(shards):
        a, b = bounds[k], bounds[k + 1]
        Vg, gg, rg = s.state()
        assert np.array_equal(Vg, Vo[a:b].astype(np.float32)) and np.array_equal(gg, go[a:b].astype(np.float32)) and np.array_equal(rg, ro[a:b]), (seed, k)
        assert np.array_equal(s.db_read_state(db.FIELD_RING), ring[:, a:b, :]), (seed, k)
    assert sum(s.db_get_counters()["events"] for s in shards) == o.counters()["events"]
    for s in shards:
        s.db_destroy()


@pytest.mark.parametrize("seed", range(int(os.environ.get("DB_RANDOM_CASES", "4"))))
def test_random_bursts_in_networks_where_a_block_owns_thousands_of_neurons(db, oracle_mod, seed):
    # 60,000 - 300,000 neurons (a block of the persistent kernel owns 400 - 2,000 of them, several tasks per warp), a
    # random number of rows longer than kInlineMax = 1024 synapses, and synchronised bursts of a random share of the
    # neurons at random times: the per-block spike and heavy-row lists fill to random levels, overflow or not
    rng = np.random.default_rng(9000 + seed)
    N = int(rng.choice([60_000, 160_000, 300_000])) + int(rng.integers(0, 128))
    n_heavy = int(rng.choice([0, 5, 300, 900]))
    heavy = {int(r): int(d) for r, d in zip(rng.choice(N, n_heavy, replace=False), rng.integers(1025, 1800, n_heavy))} if n_heavy else None
    net = db_inputs.bulk_csr(N, base_outdeg=int(rng.choice([2, 6])), seed=seed, heavy_rows=heavy, max_delay=int(rng.choice([3, 20])),
                             n_regions=int(rng.choice([1, 5])))
    t = db_inputs.type_params(bg_weight=float(rng.uniform(0.01, 0.03)))
    sim = db_inputs.sim_params(types=[t, dict(t)], window_steps=int(rng.integers(1, 12)))
    plan = []
    for _ in range(4):
        plan.append((int(rng.integers(1, 30)), float(rng.choice([0.0, 0.02, 0.4, 1.0]))))     # (steps, share of the neurons set above threshold first)
    o = oracle_mod.OracleSim(sim, net, db_inputs.DYN_SEED)
    snaps = []
    for steps, share in plan:
        V, gg, ref = o.state()
        sel = np.random.default_rng(int(share * 1000) + steps).random(N) < share
        V[sel] = -45.0
        ref[sel] = 0
        o.set_state(V, gg, ref)
        o.step(steps)
        snaps.append((sel, o.ring().copy(), o.counters()["spikes"]))
    Vo, go, ro = o.state()
    so, io = o.spikes()
    order = np.lexsort((io, so))
    done = sum(s for s, _ in plan)
    for mode in (1, 2, 3):
        g = db.Sim.db_create_from_csr(sim, net, exec_mode=mode)
        for (steps, share), (sel, ring, n_sp) in zip(plan, snaps):
            V, gg, ref = g.state()
            V[sel] = -45.0
            ref[sel] = 0
            g.set_state(V, gg, ref)
            g.db_step(steps)
            assert g.db_get_counters()["spikes"] == n_sp, (seed, mode)
            assert np.array_equal(g.db_read_state(db.FIELD_RING), ring), (seed, mode)
        Vg, gg, rg = g.state()
        assert np.array_equal(rg, ro) and np.array_equal(Vg, Vo.astype(np.float32)) and np.array_equal(gg, go.astype(np.float32)), (seed, mode)
        sg, ig = g.db_read_spikes(0, done)
        assert np.array_equal(sg, so[order]) and np.array_equal(ig, io[order]), (seed, mode)
        assert g.db_get_counters()["events"] == o.counters()["events"]
        g.db_destroy()
