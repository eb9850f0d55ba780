"""Host-side logic of bench.py that needs no GPU: the reference arm (the oracle timed on the host
cores), its behaviour under torchrun (rank 0 alone works and prints), and the whole-job reduction
over ranks (MAX of the device time, SUM of the counters) on a world_size-2 gloo group."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env=None, timeout=300):
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT, env=e,
                          capture_output=True, text=True, timeout=timeout)


def test_reference_arm_prints_the_contract_line():
    r = _run(["--impl", "reference", "--steps", "1", "--warmup", "0", "--ref-scale", "0.01",
              "--ref-warm-steps", "50", "--ref-sim-steps", "20"])
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "synaptic_events_per_s" and line["unit"] == "events/s"
    assert line["higher_is_better"] is True and line["value"] > 0 and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["config"]["workload"].startswith("configs[1]")


def test_reference_arm_other_ranks_exit_silently():
    r = _run(["--impl", "reference", "--gpus", "2"], env={"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"})
    assert r.returncode == 0 and r.stdout.strip() == ""


_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["PORT"],
                        rank=int(os.environ["RANK"]), world_size=2)
rank = dist.get_rank()
ms, sums = bench.reduce_over_ranks(dist, "cpu", 10.0 + 5.0 * rank, [100 * (rank + 1), 7, rank])
print(json.dumps({"rank": rank, "ms": ms, "sums": sums}))
dist.barrier()
dist.destroy_process_group()
""" % ROOT


def test_whole_job_reduction_over_two_ranks_gloo():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = [subprocess.Popen([sys.executable, "-c", _WORKER], cwd=ROOT, text=True, stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, env=dict(os.environ, RANK=str(r), PORT=str(port)))
             for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    for o, _ in outs:
        d = json.loads(o.strip().splitlines()[-1])
        assert d["ms"] == 15.0                       # MAX over ranks
        assert d["sums"] == [300.0, 14.0, 1.0]       # SUM over ranks


def test_single_process_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    ms, sums = bench.reduce_over_ranks(None, "cpu", 3.5, [1, 2])
    assert ms == 3.5 and sums == [1.0, 2.0]


def test_all_cores_build_of_the_oracle_gives_the_oracles_results(oracle_mod):
    # bench.py's cpu_baseline times the oracle on one core and on all of them (same source, -fopenmp: parallel for over
    # neurons and over spikes, integer atomics): the two builds must agree bit for bit, or the second figure is not the oracle's
    import numpy as np
    import db_inputs
    cfg = db_inputs.config(0, scale=0.5)
    net = oracle_mod.generate(cfg["net"], 3)
    try:
        a = oracle_mod.OracleSim(cfg["sim"], net, 2)
        a.step(400)
        ra = (a.spikes(), a.ring(), a.state(), a.counters(), a.region_counts())
        a.close()
        oracle_mod.use_all_cores(True)
        b = oracle_mod.OracleSim(cfg["sim"], net, 2)
        b.step(400)
        rb = (b.spikes(), b.ring(), b.state(), b.counters(), b.region_counts())
        b.close()
    finally:
        oracle_mod.use_all_cores(False)
    assert len(ra[0][1]) > 500 and ra[3] == rb[3]
    assert np.array_equal(ra[0][0], rb[0][0]) and np.array_equal(ra[0][1], rb[0][1])
    assert np.array_equal(ra[1], rb[1]) and np.array_equal(ra[4], rb[4])
    for x, y in zip(ra[2], rb[2]):
        assert np.array_equal(x, y)


def test_cpu_baseline_reports_one_core_all_cores_and_the_host():
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    args = argparse.Namespace(rate=7, ref_scale=0.01, ref_warm_steps=50)
    c = bench.cpu_baseline(args, steps_one=40, steps_all=40)
    assert c["kind"] == "oracle" and c["cores"] == 1 and c["value"] > 0
    assert c["all_cores"]["cores"] == os.cpu_count() == c["nproc"] and c["all_cores"]["value"] > 0
    assert c["cpu_model"] and "linear" in c["extrapolation"] and "no code" in c["external_reference"]


def test_ncu_traffic_is_tied_to_the_kernel_sources():
    sys.path.insert(0, ROOT)
    import bench
    v, why = bench._ncu_traffic("no such kernel")
    assert v is None and isinstance(why, str)
    assert len(bench._csrc_sha16()) == 16


_SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_2211_15963_b200 import sharded
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["PORT"], rank=int(os.environ["RANK"]), world_size=2)
rank = dist.get_rank()

class FakeSim:                       # stands in for the CUDA handle: the exchange is host logic
    def __init__(self):
        self.got, self.steps = [], 0
    def db_get_counters(self):
        return {"steps": self.steps}
    def db_step(self, k):
        self.steps += k
    def db_read_spikes(self, a, b):  # rank r fires neuron 1000 r + step in every step, twice in step 7 for rank 1
        st = np.arange(a, b, dtype=np.uint64)
        ids = (1000 * rank + st).astype(np.int32)
        if rank == 1 and a <= 7 < b:
            st, ids = np.append(st, np.uint64(7)), np.append(ids, np.int32(1999))
        return st, ids
    def db_deliver_external_window(self, step_begin, n_steps, steps, ids):
        assert np.all(np.diff(steps.astype(np.int64)) >= 0) and steps.min() >= step_begin and steps.max() < step_begin + n_steps
        for step in np.unique(steps):
            self.got.append((int(step), [int(x) for x in ids[steps == step]]))

sim = FakeSim()
sharded.run(dist, torch, sim, 10, 4)
print(json.dumps({"rank": rank, "got": sim.got, "own": [sharded.own_range(5000, r, 2) for r in range(2)]}))
dist.barrier()
dist.destroy_process_group()
""" % ROOT


def test_sharded_exchange_over_two_ranks_gloo():
    # the host side of the region-sharded path: all-gather of the variable-length spike lists every d_min
    # steps, delivery of the OTHER ranks' spikes window by window; world_size 2 on the CPU (gloo)
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = [subprocess.Popen([sys.executable, "-c", _SHARD_WORKER], cwd=ROOT, text=True, stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, env=dict(os.environ, RANK=str(r), PORT=str(port)))
             for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    res = {json.loads(o.strip().splitlines()[-1])["rank"]: json.loads(o.strip().splitlines()[-1]) for o, _ in outs}
    assert res[0]["own"] == [[0, 3072], [3072, 1928]]
    want0 = [(s, [1000 + s] + ([1999] if s == 7 else [])) for s in range(10)]        # rank 0 receives rank 1's spikes
    want1 = [(s, [s]) for s in range(10)]
    assert [(s, sorted(i)) for s, i in res[0]["got"]] == [(s, sorted(i)) for s, i in want0]
    assert [(s, i) for s, i in res[1]["got"]] == want1


def test_sharded_run_local_orders_steps_and_exchanges():
    # single-process sharding (handles on one GPU or on peer GPUs): every window each handle steps, then pulls the window
    # of every OTHER handle with db_exchange_peer; host logic only, with stand-ins for the CUDA handles
    from paper_2211_15963_b200 import sharded
    log = []

    class Fake:
        def __init__(self, name):
            self.name, self.steps = name, 0
        def db_get_counters(self):
            return {"steps": self.steps}
        def db_step(self, k):
            log.append(("step", self.name, self.steps, k)); self.steps += k
        def db_exchange_peer(self, src, a, b):
            assert src is not self and src.steps >= b and self.steps >= b      # both have simulated the window
            log.append(("pull", self.name, src.name, a, b))

    shards = [Fake("a"), Fake("b"), Fake("c")]
    sharded.run_local(shards, 10, 4)
    assert [s.steps for s in shards] == [10, 10, 10]
    windows = [(0, 4), (4, 8), (8, 10)]
    for (a, b) in windows:
        pulls = [e for e in log if e[0] == "pull" and e[3:] == (a, b)]
        assert sorted((e[1], e[2]) for e in pulls) == [(x, y) for x in "abc" for y in "abc" if x != y]
    # inside a window every step precedes every pull
    for (a, b) in windows:
        idx_steps = [i for i, e in enumerate(log) if e[0] == "step" and e[2] == a]
        idx_pulls = [i for i, e in enumerate(log) if e[0] == "pull" and e[3] == a]
        assert max(idx_steps) < min(idx_pulls)
