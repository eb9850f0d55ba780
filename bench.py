#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (a1 update, a2 compaction, a3 delivery, a4 region
rates) on BASELINE.json configs[1]: 1,000,000 LIF neurons, in-degree 100
(1e8 synapses), dt = 0.1 ms, background tuned for ~7 Hz (``--rate 15|30`` for the other two).

One bench "step" = one ``db_step(sim_steps)`` call = ``--sim-steps`` (default 1000) consecutive
simulation time steps = 0.1 s of biological time.  The default run (``--steps 10``) is therefore
the 10,000 steps / 1 s biological that configs[1] names, after ``--warmup`` (default 3) untimed
bench steps that also carry the network past its start-up transient.

Prints ONE JSON line (rank 0):
  value         synaptic events/s (sum of out-degrees of spiking neurons / device time), whole job
  e2e           same metric through the C ABI with HOST buffers: every bench step restores the neuron
                state from pinned host memory (db_write_state), steps, and reads the raster, the
                region rates and V back to the host (db_read_spikes / db_region_rates / db_read_state)
  roofline      the dominant kernel of the timed region (k_run in persistent mode: one launch = all the time
                steps of a db_step call; k_update_stream or k_deliver in two-kernel mode) against the measured HBM copy peak
  cpu_baseline  the oracle (oracle/, as it stands) on the host cores, on a bounded sample
``--impl reference`` times the oracle instead (same metric, unit and config).

Multi-GPU (torchrun): the path does not shard inside this build (replicas
only) -- every rank simulates an independent replica (its own seeds); value = all ranks' events /
max-over-ranks device time; scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

import db_inputs

METRIC = "synaptic_events_per_s"
UNIT = "events/s"

# Algorithmic bytes.
UPDATE_BYTES_PER_NEURON_STEP = 58      # read V 4 + g 16 + rt 2 + ring slot 16; write V 4 + g 16 (compulsory)
UPDATE_BYTES_SURVEY = (72, 80)         # plus ref and the zeroed slot written back every step (2- or 4-byte ref)
DELIVER_BYTES_PER_EVENT = {0: 17, 1: 15}   # tgt|rec 4 + w 4 (fp32) / 2 (fp16) + delay 1 + accumulator read 4 + write 4
LIST_BYTES_PER_EVENT = 16              # list mode: the 8-byte record of an event is written once and read once on top of that


STEP_KERNEL_SOURCES = ("db_device.cuh", "db_philox.cuh", "db_step.cu")     # where every kernel of the step loop is defined


def _csrc_sha16() -> str:
    """Hash of the sources of the step kernels: ties a committed ncu capture to the kernels it was taken from."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2211_15963_b200", "csrc")
    for f in STEP_KERNEL_SOURCES:
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def _ncu_traffic(key: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of a kernel from the committed `ncu --set
    full` capture, or None when the capture was not taken from this tree (profiles/ncu_traffic.json holds the hash of
    the kernel sources it belongs to)."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    try:
        d = json.load(open(p))
    except Exception:
        return None, "no profiles/ncu_traffic.json"
    if d.get("csrc_sha16") != _csrc_sha16():
        return None, f"stale: capture belongs to kernel sources {d.get('csrc_sha16')}, tree is {_csrc_sha16()}"
    v = d.get("kernels", {}).get(key)
    return (float(v["dram_bytes"]) if v else None), (v.get("source") if v else "kernel not in the capture")


def _host_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except Exception:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device: int):
        self.device = device
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.device), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------- oracle arm
def oracle_sample(rate_hz: int, scale: float, warm_steps: int, timed_steps: int, repeats: int = 1, all_cores: bool = False):
    """Times the oracle as it stands on configs[1] shrunk to `scale` (same in-degree, weights, delays, background):
    returns a list of (seconds, events, neuron_updates) per repeat.  all_cores: the -fopenmp build of the same source
    (loops over neurons and over spikes shared among the host cores; identical results)."""
    import oracle
    oracle.use_all_cores(all_cores)
    cfg = db_inputs.config(1, rate_hz=rate_hz, scale=scale)
    net = oracle.generate(cfg["net"], db_inputs.GEN_SEED)
    o = oracle.OracleSim(cfg["sim"], net, db_inputs.DYN_SEED)
    o.step(warm_steps)
    out = []
    for _ in range(repeats):
        e0 = o.counters()["events"]
        t0 = time.perf_counter()
        o.step(timed_steps)
        dt = time.perf_counter() - t0
        out.append((dt, o.counters()["events"] - e0, timed_steps * cfg["net"]["N"]))
    o.close()
    oracle.use_all_cores(False)
    return out, cfg


EXTRAPOLATION = ("linear in neuron-updates and synaptic events: the oracle's cost per neuron-step and per event does not depend on "
                 "N at fixed in-degree (apart from cache effects: the sample's state and ring are 4x smaller), so events/s of the "
                 "sample stands for the full-size workload")


def cpu_baseline(args, steps_one: int, steps_all: int) -> dict:
    """The oracle on the host: one core (the oracle as it stands) and all cores (same source built with -fopenmp)."""
    host = _host_info()
    res, ocfg = oracle_sample(args.rate, args.ref_scale, warm_steps=args.ref_warm_steps, timed_steps=steps_one)
    dt1, ev1, up1 = res[0]
    resa, _ = oracle_sample(args.rate, args.ref_scale, warm_steps=args.ref_warm_steps, timed_steps=steps_all, all_cores=True)
    dta, eva, upa = resa[0]
    n = ocfg["net"]["N"]
    return {"value": ev1 / dt1, "unit": UNIT, "cores": 1, "kind": "oracle", "neuron_updates_per_s": up1 / dt1,
            "all_cores": {"value": eva / dta, "unit": UNIT, "cores": host["nproc"], "neuron_updates_per_s": upa / dta,
                          "how": "same oracle source built with -fopenmp: parallel for over neurons (update) and over spikes "
                                 "(delivery, integer atomic adds); results identical to the one-core build",
                          "steps": steps_all, "seconds": dta},
            "nproc": host["nproc"], "cpu_model": host["cpu_model"],
            "sample": f"configs[1] shrunk to N={n} (in-degree 100, same distributions), {steps_one} time steps after "
                      f"{args.ref_warm_steps} warm-up steps on one core ({dt1:.1f} s), {steps_all} on all {host['nproc']} cores "
                      f"({dta:.1f} s), + network generation",
            "extrapolation": EXTRAPOLATION,
            "external_reference": "none: the paper ships no code, so nothing outside this repository pins the oracle's speed or results "
                                  "(its arithmetic is pinned by tests/: closed forms, invariants, brute force)"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    scale = args.ref_scale
    # the start-up transient runs at several times the steady rate: warm the oracle past part of it
    warm = max(args.ref_sim_steps * args.warmup, args.ref_warm_steps)
    res, cfg = oracle_sample(args.rate, scale, warm_steps=warm, timed_steps=args.ref_sim_steps, repeats=args.steps)
    secs = sum(r[0] for r in res)
    events = sum(r[1] for r in res)
    updates = sum(r[2] for r in res)
    value = events / secs
    host = _host_info()
    sample = (f"configs[1] shrunk to N={cfg['net']['N']} (in-degree 100, same distributions), "
              f"{args.steps} x {args.ref_sim_steps} time steps after {warm} warm-up steps, "
              f"single thread")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": dict(_config_dict(args, int(1_000_000 * args.scale), args.sim_steps),
                       reference_sample={"n_neurons": cfg["net"]["N"], "sim_steps_per_bench_step": args.ref_sim_steps}),
        "neuron_updates_per_s": updates / secs,
        "rtf": secs / (args.steps * args.ref_sim_steps * cfg["sim"]["dt_ms"] * 1e-3),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "nproc": host["nproc"], "cpu_model": host["cpu_model"], "extrapolation": EXTRAPOLATION},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def _config_dict(args, n_neurons, sim_steps):
    if args.config != 1:           # configs 2-4 are parity-test cases; `--config` times them for profiles/ only
        return {"workload": f"configs[{args.config}] (DESIGN.md section 5): {n_neurons} LIF neurons, dt 0.1 ms",
                "n_neurons": n_neurons, "sim_steps_per_bench_step": sim_steps, "dt_ms": 1.0 if args.dt == 1 else 0.1,
                "l2": "no flush: device footprint far exceeds the 126 MB L2"}
    return {"workload": f"configs[1]: {n_neurons} LIF neurons, in-degree 100, dt 0.1 ms, ~{args.rate} Hz",
            "n_neurons": n_neurons, "in_degree": 100, "rate_hz_target": args.rate,
            "sim_steps_per_bench_step": sim_steps, "dt_ms": 1.0 if args.dt == 1 else 0.1,
            "l2": "no flush: device footprint (state + ring + CSR ~1.4 GB) exceeds the 126 MB L2; the step loop "
                  "runs back to back as in production"}


def reduce_over_ranks(dist, device, ms: float, sums: list):
    """Whole-job figures from per-rank ones: MAX of the device time over the ranks, SUM of the counters
    (replicas only).  `dist` is torch.distributed or None (single process)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    tot = torch.tensor([float(x) for x in sums], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(x) for x in tot.tolist()]


# --------------------------------------------------------------------------------------------- CUDA arm
def shard_pair(db, torch, local, n_sim=1000, d_min=10, peer=True):
    """SURVEY 8(f) row 3, the half one GPU can measure: configs[1] (delays U{d_min..20} so that the exchange window is
    d_min steps) split between TWO handles on this GPU, each owning half of the targets and the synapses onto them from
    every source (SI Eq.(6); layout P:L494).  They step d_min steps one after the other, then each one's
    spikes go to the other through the public API: device to device (db_exchange_peer: the receiver reads the sender's
    raster in device memory; peer=True), or through the host (db_read_spikes -> db_deliver_external_window, as between
    ranks of a multi-process run).  Wall clock with a device synchronise at the ends; on two GPUs the handles would run
    side by side, so the per-shard figure is half the pair's."""
    from paper_2211_15963_b200 import sharded
    cfg = _make_cfg(1, 7)
    cfg["net"].update(delay_intra_min=d_min)
    N = cfg["net"]["N"]
    cut = (N // 2) // 1024 * 1024
    bounds = [0, cut, N]
    shards = [db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED, dyn_seed=db_inputs.DYN_SEED, exec_mode=db.EXEC_AUTO,
                               raster_capacity=1 << 24, device=local, own=(bounds[k], bounds[k + 1] - bounds[k])) for k in range(2)]

    def window(done, clock):
        t0 = time.perf_counter()
        for sh in shards:
            sh.db_step(d_min)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        n_ext = 0
        if peer:
            for k, dst in enumerate(shards):
                dst.db_exchange_peer(shards[1 - k], done, done + d_min)
        else:
            fresh = [sh.db_read_spikes(done, done + d_min) for sh in shards]
            for k, dst in enumerate(shards):
                st, ids = fresh[1 - k]
                if len(ids):
                    dst.db_deliver_external_window(done, d_min, st, ids)
                    n_ext += len(ids)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        if clock is not None:
            clock[0] += t1 - t0; clock[1] += t2 - t1; clock[2] += n_ext

    done = 0
    for _ in range(300 // d_min):                      # past the start-up transient
        window(done, None); done += d_min
    c0 = [sh.db_get_counters() for sh in shards]
    clock = [0.0, 0.0, 0]
    for _ in range(n_sim // d_min):
        window(done, clock); done += d_min
    c1 = [sh.db_get_counters() for sh in shards]
    steps = n_sim // d_min * d_min
    free_us = None
    if peer:                                           # the same loop as a run would issue it: nothing waits on the host
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sharded.run_local(shards, steps, d_min)
        torch.cuda.synchronize()
        free_us = 1e6 * (time.perf_counter() - t0) / steps
    events = sum(b["events"] - a_["events"] for a_, b in zip(c0, c1))
    spikes = sum(b["spikes"] - a_["spikes"] for a_, b in zip(c0, c1))
    for sh in shards:
        sh.db_destroy()
    tot = clock[0] + clock[1]
    return {"n_neurons": N, "shards": 2, "owned": [cut, N - cut], "exchange_every_steps": d_min,
            "exec_mode": {1: "kernels+graph", 2: "persistent", 3: "kernels+graph, arrival lists"}.get(c1[0]["exec_mode"]),
            "pair_us_per_sim_step": 1e6 * tot / steps, "per_shard_us_per_sim_step": 0.5e6 * tot / steps,
            "step_us_per_sim_step_pair": 1e6 * clock[0] / steps, "exchange_us_per_sim_step_pair": 1e6 * clock[1] / steps,
            "external_spikes_per_sim_step": spikes / steps, "events_per_s_pair": events / tot,
            "mean_rate_hz": spikes / N / (steps * cfg["sim"]["dt_ms"] * 1e-3), "sim_steps_timed": steps,
            "pair_us_per_sim_step_no_host_sync": free_us,
            "exchange": "db_exchange_peer (device to device)" if peer else "db_read_spikes -> host -> db_deliver_external_window",
            "what": "two handles on ONE GPU run one after the other; wall clock (not a multi-GPU measurement)"}


def _make_cfg(idx, rate, scale=1.0, drive="poisson", spike_bin=1, dt_ms=0.1, iext_gamma=False):
    cfg = db_inputs.config(idx, rate_hz=(rate if idx == 1 else None), scale=scale)
    cfg["sim"]["dt_ms"] = dt_ms
    if iext_gamma:                              # per-neuron external currents (R31): zero-mean Gamma(4, 0.01) spread
        for t in cfg["sim"]["types"]:
            t.update(Iext=-0.04, iext_gamma_shape=4.0, iext_gamma_scale=0.01)
    if drive == "ou":                           # the paper's production drive instead of Poisson
        db_inputs.ou_drive(cfg["sim"], rate)
    cfg["sim"]["spike_bin_steps"] = spike_bin
    return cfg


def measure(db, torch, cfg, exec_mode, n_sim, steps, warmup, profile_steps, local, seed_off=0, barrier=None, drive="poisson",
            extra_bytes=0):
    """Creates the simulation, runs `warmup` untimed and `steps` timed db_step(n_sim) calls (CUDA events on the stream
    the library launches on, one per call) and, in the two-kernel modes, `profile_steps` steps with events around
    every kernel.  Returns (sim, record); the caller destroys sim."""
    N = cfg["net"]["N"]
    fp16 = int(cfg["net"]["weight_fp16"])
    t_create = time.perf_counter()
    sim = db.Sim.db_create(cfg["net"], cfg["sim"], seed=db_inputs.GEN_SEED + seed_off, dyn_seed=db_inputs.DYN_SEED + seed_off,
                           exec_mode=exec_mode, raster_capacity=1 << 25, device=local)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t_create
    for _ in range(warmup):
        sim.db_step(n_sim)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    c0 = sim.db_get_counters()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    if barrier:
        barrier()
    evs[0].record()
    for k in range(steps):
        sim.db_step(n_sim)
        evs[k + 1].record()
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    ms = evs[0].elapsed_time(evs[-1])
    launch_ms = [evs[k].elapsed_time(evs[k + 1]) for k in range(steps)]
    c1 = sim.db_get_counters()
    events, spikes = c1["events"] - c0["events"], c1["spikes"] - c0["spikes"]
    used = c1["exec_mode"]
    peak, peak_src = _peaks()
    upd_per = UPDATE_BYTES_PER_NEURON_STEP + (8 if drive == "ou" else 0) + extra_bytes      # + read and write of I_ou (+ read of I_ext)
    ev_bytes = DELIVER_BYTES_PER_EVENT[fp16]
    secs = ms * 1e-3
    bio_s = steps * n_sim * cfg["sim"]["dt_ms"] * 1e-3
    rec = {"n_neurons": N, "exec_mode": {1: "kernels+graph", 2: "persistent", 3: "kernels+graph, arrival lists"}.get(used, str(used)),
           "us_per_sim_step": 1e6 * secs / (steps * n_sim), "events_per_s": events / secs,
           "neuron_updates_per_s": N * steps * n_sim / secs, "rtf": secs / bio_s,
           "mean_rate_hz": spikes / N / bio_s, "events_per_sim_step": events / (steps * n_sim), "create_s": t_create,
           "sim_steps_timed": steps * n_sim, "list_spilled": c1["list_spilled"] - c0["list_spilled"],
           "_ms": ms, "_launch_ms": launch_ms, "_events": events, "_spikes": spikes, "_launches": c1["launches"] - c0["launches"],
           "_used": used}
    # whole step against the roofline: algorithmic bytes of a1 (58 B per neuron-step) + a3 (17 / 15 B per event) over the step time
    step_bytes = upd_per * N + ev_bytes * events / (steps * n_sim)
    step_s = secs / (steps * n_sim)
    rec["step"] = {"bytes_per_sim_step": step_bytes, "achieved_gbs": step_bytes / step_s / 1e9, "frac": step_bytes / step_s / 1e9 / peak}
    if used != db.EXEC_PERSISTENT and profile_steps > 0:
        prof = sim.db_step_profiled(profile_steps)
        upd_s = prof["update_ms"] * 1e-3 / prof["steps"]
        del_s = prof["deliver_ms"] * 1e-3 / prof["steps"]
        ev_step = prof["events"] / prof["steps"]
        upd_gbs = upd_per * N / upd_s / 1e9
        lists = used == db.EXEC_KERNELS_DEFERRED
        del_alg = ev_bytes * ev_step / del_s / 1e9
        rec["kernels"] = {
            "update": {"kernel": "k_update_stream", "us_per_launch": upd_s * 1e6, "bytes_per_launch": upd_per * N,
                       "achieved_gbs": upd_gbs, "frac": upd_gbs / peak,
                       "frac_survey_72_80B": [b * N / upd_s / 1e9 / peak for b in UPDATE_BYTES_SURVEY]},
            "delivery": {"kernel": "k_deliver_lists" if lists else "k_deliver", "us_per_launch": del_s * 1e6,
                         "events_per_launch": ev_step, "events_per_s": ev_step / del_s, "bytes_per_event": ev_bytes,
                         "achieved_gbs": del_alg, "frac": del_alg / peak},
            "method": f"db_step_profiled({profile_steps}): CUDA events around every kernel, kernels back to back on one stream",
        }
        if lists:   # what the list kernel has to stream per event on top of the accumulator: row + record written + record read
            b = ev_bytes + LIST_BYTES_PER_EVENT
            rec["kernels"]["delivery"].update(bytes_per_event_streamed=b, frac_streamed=b * ev_step / del_s / 1e9 / peak)
    return sim, rec


def _public(rec):
    return {k: v for k, v in rec.items() if not k.startswith("_")}


def run_ours(args):
    import torch
    import paper_2211_15963_b200 as db

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    db.load()

    dt_ms = 1.0 if args.dt == 1 else 0.1
    cfg = _make_cfg(args.config, args.rate, args.scale, args.drive, args.spike_bin, dt_ms)
    N = cfg["net"]["N"]
    n_sim = args.sim_steps
    mode = {"auto": db.EXEC_AUTO, "kernels": db.EXEC_KERNELS, "persistent": db.EXEC_PERSISTENT,
            "deferred": db.EXEC_KERNELS_DEFERRED}[args.exec_mode]
    fp16 = int(cfg["net"]["weight_fp16"])

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident throughput of the headline workload --------------------------
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    sim, rec = measure(db, torch, cfg, mode, n_sim, args.steps, args.warmup, 0, local, seed_off=rank, barrier=barrier, drive=args.drive)
    clk = clocks.stop() if rank == 0 else None
    ms, launch_ms, events, spikes = rec["_ms"], rec["_launch_ms"], rec["_events"], rec["_spikes"]
    exec_used = rec["_used"]
    ms_max, (events_all, spikes_all, launches_all) = reduce_over_ranks(dist, f"cuda:{local}", ms, [events, spikes, rec["_launches"]])
    secs = ms_max * 1e-3
    bio_s = args.steps * n_sim * cfg["sim"]["dt_ms"] * 1e-3
    value = events_all / secs
    rate_hz = spikes_all / (world * N) / bio_s

    # ---------------- roofline of the dominant kernel of the timed region ---------------------------
    peak, peak_src = _peaks()
    upd_per = UPDATE_BYTES_PER_NEURON_STEP + (8 if args.drive == "ou" else 0)
    ev_bytes = DELIVER_BYTES_PER_EVENT[fp16]
    if exec_used == db.EXEC_PERSISTENT:
        # k_run: ONE launch = n_sim fused steps (a1 + a2 + a3 + a4); algorithmic bytes per launch =
        # n_sim * 58 B * N (update) + 17 B (15 B fp16) * events of the launch (delivery)
        upd_bytes = float(upd_per) * N * n_sim
        del_bytes = float(ev_bytes) * events / max(args.steps, 1)
        dur_s = float(np.mean(launch_ms)) * 1e-3
        gbs = (upd_bytes + del_bytes) / dur_s / 1e9
        key = f"k_run:config{args.config}:rate{args.rate}:{args.drive}:bin{args.spike_bin}:dt{args.dt}"
        per_step, src = _ncu_traffic(key) if args.scale == 1.0 else (None, "scaled workload")
        traffic = per_step * n_sim if per_step else None
        l2_resident = traffic is not None and traffic < 0.9 * (upd_bytes + del_bytes)
        roofline = {
            "bound": "l2+issue" if l2_resident else "hbm",
            "kernel": "k_run (persistent: update + compaction + delivery + region counts, fused)",
            "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
            "frac_survey_72_80B": [(float(b) * N * n_sim + del_bytes) / dur_s / 1e9 / peak for b in UPDATE_BYTES_SURVEY],
            "traffic": traffic, "traffic_source": src,
            "frac_dram": (traffic / dur_s / 1e9 / peak) if traffic else None,
            "peak_source": peak_src, "bytes_per_launch": upd_bytes + del_bytes,
            "bytes_per_launch_update": upd_bytes, "bytes_per_launch_delivery": del_bytes,
            "sim_steps_per_launch": n_sim, "us_per_launch": dur_s * 1e6, "us_per_sim_step": dur_s * 1e6 / n_sim,
            "launch_ms": launch_ms, "frac_of_nominal_8000": gbs / 8000.0, "share_of_step": 1.0,
            "note": ("`frac` = algorithmic bytes (58 B per neuron-step + 17 B per event) / time / measured HBM copy peak; when `bound` is "
                     "l2+issue the per-step working set (state 22 MB + one ring slot 16 MB) sits in the 126 MB L2, DRAM moved only "
                     "`traffic` bytes per launch (ncu, profiles/) and ran at `frac_dram` of the peak: the figure is an L2 / issue-rate "
                     "number, not an HBM one"),
        }
    else:
        sim.db_destroy()
        sim, rec2 = measure(db, torch, cfg, mode, n_sim, 1, 1, args.profile_steps, local, seed_off=rank, drive=args.drive)
        k = rec2.get("kernels")
        if k and k["delivery"]["us_per_launch"] > k["update"]["us_per_launch"]:
            d = k["delivery"]
            roofline = {"bound": "hbm", "kernel": d["kernel"], "achieved": d["achieved_gbs"], "peak": peak, "unit": "GB/s",
                        "frac": d["frac"], "traffic": None, "peak_source": peak_src,
                        "bytes_per_launch": ev_bytes * d["events_per_launch"], "us_per_launch": d["us_per_launch"],
                        "update": k["update"], "delivery": d}
        elif k:
            u = k["update"]
            roofline = {"bound": "hbm", "kernel": u["kernel"], "achieved": u["achieved_gbs"], "peak": peak, "unit": "GB/s",
                        "frac": u["frac"], "traffic": None, "peak_source": peak_src, "bytes_per_launch": u["bytes_per_launch"],
                        "us_per_launch": u["us_per_launch"], "update": u, "delivery": k["delivery"]}
        else:
            roofline = {"bound": "hbm", "kernel": "k_update_stream + delivery", "achieved": None, "peak": peak, "unit": "GB/s",
                        "frac": None, "traffic": None, "note": "run with --profile-steps > 0 for per-kernel times"}
    # the ceilings of scatter delivery (a3) on this device: random 4-byte reductions into a region the size of the ring
    # (far larger than L2: random DRAM sectors) and into one the size of ONE ring slot (L2-resident), measured live
    if rank == 0 and not args.no_scatter_probe:
        ring_bytes = min(int(cfg["sim"]["D"]) * 16 * N, 8 << 30)
        slot_bytes = 16 * N
        roofline["scatter_probe"] = {
            "what": "db_probe_scatter (bench-only helper library): red.global.add.s32 to uniformly random cells, ops/s",
            "ring_sized_region": {"bytes": ring_bytes, "ops_per_s": db.binding.db_probe_scatter(ring_bytes, device=local)},
            "one_slot_region": {"bytes": slot_bytes, "ops_per_s": db.binding.db_probe_scatter(slot_bytes, device=local)}}

    # ---------------- end to end through the C ABI with host buffers --------------------------------
    V_h = torch.empty(N, dtype=torch.float32).pin_memory()
    g_h = [torch.empty(N, dtype=torch.float32).pin_memory() for _ in range(4)]
    ref_h = torch.empty(N, dtype=torch.int32).pin_memory()
    V_h.numpy()[:] = sim.db_read_state(db.FIELD_V)
    for u in range(4):
        g_h[u].numpy()[:] = sim.db_read_state(db.FIELD_G_AMPA + u)
    ref_h.numpy()[:] = sim.db_read_state(db.FIELD_REF)
    cap = int(3 * max(spikes / max(args.steps, 1), 1)) + 4096
    st_h = torch.empty(cap, dtype=torch.int64).pin_memory()
    id_h = torch.empty(cap, dtype=torch.int32).pin_memory()
    st_np, id_np = st_h.numpy().view(np.uint64), id_h.numpy()
    Vout_h = torch.empty(N, dtype=torch.float32).pin_memory()
    C = db.binding.C

    def e2e_step():
        s0 = sim.db_get_counters()["steps"]
        sim.db_write_state(db.FIELD_V, V_h.numpy())
        for u in range(4):
            sim.db_write_state(db.FIELD_G_AMPA + u, g_h[u].numpy())
        sim.db_write_state(db.FIELD_REF, ref_h.numpy())
        sim.db_step(n_sim)
        st, ids = sim.db_read_spikes(s0, s0 + n_sim, st_np, id_np)
        rates, _ = sim.db_region_rates()
        sim.L.db_read_state(sim.h, db.FIELD_V, 0, N, C.c_void_p(Vout_h.data_ptr()))
        return len(ids), rates.nbytes

    e2e_step()                                   # warm
    barrier()
    ce0 = sim.db_get_counters()
    t0 = time.perf_counter()
    n_sp = 0
    for _ in range(args.e2e_steps):
        k, rate_bytes = e2e_step()
        n_sp += k
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    ce1 = sim.db_get_counters()
    e2e_max, (e2e_events,) = reduce_over_ranks(dist, f"cuda:{local}", e2e_s, [ce1["events"] - ce0["events"]])
    e2e = {"value": e2e_events / e2e_max, "unit": UNIT,
           "h2d_bytes_per_step": int(N * (4 + 16 + 4)),
           "d2h_bytes_per_step": int(N * 4 + (n_sp // max(args.e2e_steps, 1)) * 12 + rate_bytes),
           "steps": args.e2e_steps, "ms_per_step": 1e3 * e2e_max / args.e2e_steps,
           "what": "db_write_state(V, g[4], ref) from pinned host + db_step + db_read_spikes + db_region_rates + "
                   "db_read_state(V) to pinned host, wall clock"}
    sim.db_destroy()
    del sim

    # ---------------- the other operating points north_star names (rank 0, N = 1, default workload only) ------------
    rates, configs, variants = {}, {}, {}
    if rank == 0 and world == 1 and not args.no_sweep and args.config == 1 and args.scale == 1.0 and args.drive == "poisson" \
            and args.dt == 0 and args.spike_bin == 1:
        def sub(cfg_s, n_sim_s, steps_s, warm_s, prof_s, drive="poisson", extra_bytes=0):
            torch.cuda.empty_cache()
            t0 = time.perf_counter()
            sm, r = measure(db, torch, cfg_s, db.EXEC_AUTO, n_sim_s, steps_s, warm_s, prof_s, local, drive=drive, extra_bytes=extra_bytes)
            sm.db_destroy()
            del sm
            r = _public(r)
            r["wall_s"] = time.perf_counter() - t0
            return r
        for r_hz in (15, 30):
            if r_hz != args.rate:
                rates[str(r_hz)] = sub(_make_cfg(1, r_hz), 1000, 5, 3, 0)
        rates[str(args.rate)] = "headline"
        # the paper's production mode: dt = 1 ms (b_t = dt), OU drive; RTF comparable in kind with BASELINE.md 1a
        variants["dt_1ms_ou"] = sub(_make_cfg(1, 7, drive="ou", dt_ms=1.0), 1000, 5, 3, 0, drive="ou")
        variants["dt_0.1ms_ou_bin10"] = sub(_make_cfg(1, 7, drive="ou", spike_bin=10), 1000, 5, 3, 0, drive="ou")
        # per-neuron external currents from a Gamma law (R31): one more fp32 plane read by the update (62 B per neuron-step)
        variants["iext_gamma_plane"] = sub(_make_cfg(1, 7, iext_gamma=True), 1000, 5, 3, 0, extra_bytes=4)
        # region sharding on one GPU: two handles that own half of the targets each, spikes exchanged every 10 steps
        try:
            torch.cuda.empty_cache()
            variants["two_shards_one_gpu"] = shard_pair(db, torch, local, peer=True)
            variants["two_shards_one_gpu_host_exchange"] = shard_pair(db, torch, local, peer=False)
        except Exception as ex:
            variants["two_shards_one_gpu"] = {"error": str(ex)[:200]}
        for idx, (n_s, st_s, wm_s) in {2: (500, 2, 3), 4: (500, 2, 3), 3: (150, 2, 4)}.items():
            if idx == 3 and args.skip_config3:
                configs["3"] = "skipped (--skip-config3)"
                continue
            try:
                configs[str(idx)] = sub(_make_cfg(idx, None), n_s, st_s, wm_s, 128)
            except Exception as ex:             # e.g. not enough device memory on a shared box
                configs[str(idx)] = {"error": str(ex)[:200]}

    # ---------------- CPU baseline: the oracle on the host cores (rank 0, N = 1 only) ----------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(args, steps_one=2000, steps_all=6000)     # ~12 s on one core, about as long on all of them

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": dict(_config_dict(args, N, n_sim), replicas=world, drive=args.drive, spike_bin_steps=args.spike_bin,
                           exec_mode={1: "kernels+graph", 2: "persistent", 3: "kernels+graph, arrival lists"}.get(exec_used, str(exec_used))),
            "neuron_updates_per_s": world * N * args.steps * n_sim / secs,
            "rtf": secs / bio_s, "mean_rate_hz": rate_hz, "us_per_sim_step": 1e6 * secs / (args.steps * n_sim),
            "paper_context": "paper RTF 65 / 78.8 / 118.8 at 7 / 15 / 30 Hz for 86e9 neurons on 14,012 GPUs (dt 1 ms): "
                             "another machine and workload, not a target",
            "roofline": roofline, "rates": rates, "configs": configs, "variants": variants,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches_all), "clocks": clk,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--rate", type=int, default=7, choices=[7, 15, 30])
    ap.add_argument("--config", type=int, default=1, choices=[1, 2, 3, 4],
                    help="BASELINE.json configs[i]; 1 is the bench workload (the default run adds sub-records for the others)")
    ap.add_argument("--sim-steps", type=int, default=1000, help="simulation time steps per bench step")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink configs[1] (debugging only)")
    ap.add_argument("--exec-mode", choices=["auto", "kernels", "persistent", "deferred"], default="auto")
    ap.add_argument("--drive", choices=["poisson", "ou"], default="poisson",
                    help="background drive: Poisson events into AMPA (BASELINE configs) or the paper's OU current (7 Hz only)")
    ap.add_argument("--dt", type=int, default=0, choices=[0, 1], help="1: the paper's production step dt = 1 ms instead of 0.1 ms")
    ap.add_argument("--spike-bin", type=int, default=1, help="time bin b_t for transferring spikes, in steps (paper: 10 at dt 0.1 ms)")
    ap.add_argument("--profile-steps", type=int, default=256, help="two-kernel modes: steps with CUDA events around every kernel")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-sweep", action="store_true", help="headline only: no sub-records for 15 / 30 Hz, configs 2-4, dt = 1 ms")
    ap.add_argument("--skip-config3", action="store_true", help="leave the 112 GB configs[3] out of the sweep")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-scatter-probe", action="store_true")
    ap.add_argument("--ref-scale", type=float, default=0.25, help="oracle sample: fraction of configs[1]'s neurons")
    ap.add_argument("--ref-warm-steps", type=int, default=1000, help="oracle: untimed steps past the start-up transient")
    ap.add_argument("--ref-sim-steps", type=int, default=50, help="oracle arm: time steps per bench step")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"bench.py: warmup {args.warmup} < 3 is below the timing rules", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
