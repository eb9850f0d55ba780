"""Region-sharded simulation over several processes (one exchange step): every rank owns a contiguous range
of neurons (db_create(..., own=(first, count))) and, every `d_min` time steps, all-gathers the compacted spike lists of
the window (SI Eq.(6): the second sum runs over the neurons of the other GPUs); the spikes of the other ranks
go into the local ring through db_deliver_external.  Plumbing only: torch.distributed moves the lists (NCCL on GPUs,
gloo on the CPU in the tests), the library does the delivery.  The single-GPU test of the same protocol
(tests/test_gpu_parity_paths.py) shows that it reproduces the unsharded simulation bit for bit."""
from __future__ import annotations

import numpy as np


def own_range(N: int, rank: int, world: int, align: int = 1024):
    """Contiguous, 1024-aligned ranges of about N / world neurons: (first, count) of `rank`."""
    per = -(-N // world)
    per = -(-per // align) * align
    first = min(rank * per, N)
    return first, max(min(N, first + per) - first, 0)


def pack_spikes(steps: np.ndarray, ids: np.ndarray, step_begin: int) -> np.ndarray:
    """(step - step_begin) << 32 | id, one int64 per spike."""
    return ((np.asarray(steps, np.int64) - int(step_begin)) << 32) | np.asarray(ids, np.int64)


def unpack_spikes(packed: np.ndarray, step_begin: int):
    packed = np.asarray(packed, np.int64)
    return (packed >> 32) + int(step_begin), (packed & 0xFFFFFFFF).astype(np.int32)


def all_gather_spikes(dist, torch, steps, ids, step_begin: int, device="cpu"):
    """Every rank's (steps, ids) of the window, as a list indexed by rank.  Two collectives: the counts, then the lists
    padded to the longest (message size ~ 8 bytes per spike)."""
    world = dist.get_world_size()
    mine = torch.from_numpy(pack_spikes(steps, ids, step_begin)).to(device)
    n = torch.tensor([mine.numel()], dtype=torch.int64, device=device)
    counts = [torch.zeros_like(n) for _ in range(world)]
    dist.all_gather(counts, n)
    counts = [int(c.item()) for c in counts]
    width = max(max(counts), 1)
    buf = torch.zeros(width, dtype=torch.int64, device=device)
    buf[:mine.numel()] = mine
    out = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return [unpack_spikes(out[r][:counts[r]].cpu().numpy(), step_begin) for r in range(world)]


def exchange(dist, torch, sim, step_begin: int, step_end: int, device="cpu"):
    """After every rank has stepped to `step_end`: gather the spikes of [step_begin, step_end) and deliver the other ranks'
    to `sim`.  Returns the number of outside spikes delivered.  step_end - step_begin must not exceed the smallest delay."""
    st, ids = sim.db_read_spikes(step_begin, step_end)
    gathered = all_gather_spikes(dist, torch, st, ids, step_begin, device)
    rank, n = dist.get_rank(), 0
    for r, (s_r, i_r) in enumerate(gathered):
        if r == rank or len(i_r) == 0:
            continue
        order = np.argsort(s_r, kind="stable")               # by step: the layout of the window call
        sim.db_deliver_external_window(step_begin, step_end - step_begin, s_r[order], i_r[order])
        n += len(i_r)
    return n


def run(dist, torch, sim, n_steps: int, d_min: int, device="cpu"):
    """n_steps time steps on every rank with an exchange every d_min steps."""
    done = int(sim.db_get_counters()["steps"])
    end = done + n_steps
    while done < end:
        k = min(d_min, end - done)
        sim.db_step(k)
        exchange(dist, torch, sim, done, done + k, device)
        done += k


def run_local(shards, n_steps: int, d_min: int):
    """The same for shards held by ONE process (handles on one GPU, or on GPUs with peer access): every d_min steps each
    handle pushes the rows of the others' new spikes straight out of their rasters in device memory
    (db_exchange_peer).  Nothing here waits on the host."""
    done = int(shards[0].db_get_counters()["steps"])
    end = done + n_steps
    while done < end:
        k = min(d_min, end - done)
        for sh in shards:
            sh.db_step(k)
        for dst in shards:
            for src in shards:
                if src is not dst:
                    dst.db_exchange_peer(src, done, done + k)
        done += k
