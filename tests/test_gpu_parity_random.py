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
