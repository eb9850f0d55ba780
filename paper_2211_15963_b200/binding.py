"""Thin ctypes binding of include/db_b200.h: argument marshalling only.

Every step of the hot path runs in the CUDA library; there is no CPU fallback
(create calls raise if the library or a CUDA device is missing).  PyTorch
supplies device memory (allocator callbacks backed by torch tensors) and the
stream.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

DB_OK, DB_EINVAL, DB_ENOMEM, DB_ECUDA, DB_ERANGE, DB_ESTATE = 0, -1, -2, -3, -4, -5
EXEC_AUTO, EXEC_KERNELS, EXEC_PERSISTENT, EXEC_KERNELS_DEFERRED = 0, 1, 2, 3
(FIELD_V, FIELD_G_AMPA, FIELD_G_NMDA, FIELD_G_GABAA, FIELD_G_GABAB, FIELD_REF, FIELD_TYPE, FIELD_RING,
 FIELD_OUTDEG, FIELD_IOU, FIELD_IEXT) = range(11)
EXTERNAL_STATIC_MAX = 65536   # DB_EXTERNAL_STATIC_MAX

EXPORTS = [
    "db_create", "db_create_from_csr", "db_destroy", "db_step", "db_deliver_external", "db_deliver_external_static", "db_deliver_external_window", "db_exchange_peer", "db_step_profiled", "db_read_spikes",
    "db_read_state", "db_write_state", "db_region_rates", "db_region_counts", "db_read_bold", "db_export_csr",
    "db_free_csr", "db_get_counters", "db_synchronize", "db_last_error",
]


class DbError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"db error {code}: {msg}")
        self.code = code


class TypeParams(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("C", "gL", "VL", "Vth", "Vreset", "Tref_ms", "Iext")] + [
        ("G", C.c_double * 4), ("E", C.c_double * 4), ("tau_ms", C.c_double * 4),
        ("bg_rate_hz", C.c_double), ("bg_weight", C.c_double),
        ("ou_mu", C.c_double), ("ou_sigma", C.c_double), ("ou_tau_ms", C.c_double),
        ("iext_gamma_shape", C.c_double), ("iext_gamma_scale", C.c_double)]


BOLD_KEYS = ("kappa", "gamma", "tau", "alpha", "rho", "V0", "k1", "k2", "k3", "z_scale")


class BoldParams(C.Structure):
    _fields_ = [("enabled", C.c_int32), ("reserved", C.c_int32)] + [(k, C.c_double) for k in BOLD_KEYS]


class SimParams(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("dt_ms", C.c_double), ("S", C.c_int32), ("D", C.c_int32),
                ("window_steps", C.c_int32), ("n_types", C.c_int32), ("type", TypeParams * 8),
                ("dyn_seed", C.c_uint64), ("raster_capacity", C.c_uint64), ("max_windows", C.c_uint32),
                ("exec_mode", C.c_int32), ("spike_bin_steps", C.c_int32), ("bold", BoldParams)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Runtime(C.Structure):
    _fields_ = [("alloc", ALLOC_FN), ("free", FREE_FN), ("user", C.c_void_p), ("stream", C.c_void_p),
                ("device", C.c_int32)]


class NetworkSpec(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("N", C.c_int64), ("n_regions", C.c_int32),
                ("region_size_sigma", C.c_double), ("exc_frac", C.c_double), ("mode", C.c_int32), ("K", C.c_int32),
                ("intra_frac", C.c_double), ("region_matrix_sigma", C.c_double), ("outdeg_mean", C.c_double),
                ("outdeg_sigma", C.c_double), ("outdeg_cap", C.c_int32), ("w_mu", C.c_double), ("w_sigma", C.c_double),
                ("w_scale", C.c_double), ("inh_mult", C.c_double), ("slow_frac", C.c_double),
                ("delay_intra_min", C.c_int32), ("delay_intra_max", C.c_int32), ("delay_inter_min", C.c_int32),
                ("delay_inter_max", C.c_int32), ("weight_fp16", C.c_int32), ("own_first", C.c_int64), ("own_count", C.c_int64),
                ("sim", SimParams),
                ("runtime", C.POINTER(Runtime))]


class CsrView(C.Structure):
    _fields_ = [("N", C.c_int64), ("E", C.c_int64), ("n_regions", C.c_int32), ("region_start", C.c_void_p),
                ("ntype", C.c_void_p), ("row_ptr", C.c_void_p), ("tgt", C.c_void_p), ("w", C.c_void_p),
                ("delay", C.c_void_p), ("rec", C.c_void_p), ("weight_fp16", C.c_int32), ("own_first", C.c_int64),
                ("own_count", C.c_int64)]


class CsrHost(C.Structure):
    _fields_ = [("N", C.c_int64), ("E", C.c_int64), ("n_regions", C.c_int32),
                ("region_start", C.POINTER(C.c_int64)), ("ntype", C.POINTER(C.c_uint8)),
                ("row_ptr", C.POINTER(C.c_int64)), ("tgt", C.POINTER(C.c_int32)), ("w", C.POINTER(C.c_float)),
                ("delay", C.POINTER(C.c_uint8)), ("rec", C.POINTER(C.c_uint8))]


class Counters(C.Structure):
    _fields_ = [("steps", C.c_uint64), ("spikes", C.c_uint64), ("events", C.c_uint64), ("bg_events", C.c_uint64),
                ("ring_overflow", C.c_uint32), ("exec_mode", C.c_uint32), ("launches", C.c_uint64), ("list_spilled", C.c_uint64)]


class PhaseTimes(C.Structure):
    _fields_ = [("update_ms", C.c_double), ("deliver_ms", C.c_double), ("total_ms", C.c_double),
                ("steps", C.c_uint64), ("spikes", C.c_uint64), ("events", C.c_uint64)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def load():
    """Load the C-ABI library (building it if the sources are newer).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libdb_b200.so is missing: the CUDA extension is required (no CPU fallback)")
        L = C.CDLL(path)
        L.db_create.argtypes = [C.POINTER(NetworkSpec), C.c_uint64, C.POINTER(C.c_void_p)]
        L.db_create_from_csr.argtypes = [C.POINTER(SimParams), C.POINTER(CsrView), C.POINTER(Runtime),
                                         C.POINTER(C.c_void_p)]
        L.db_destroy.argtypes = [C.c_void_p]
        L.db_step.argtypes = [C.c_void_p, C.c_uint32]
        L.db_deliver_external.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64]
        L.db_deliver_external_static.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64]
        L.db_deliver_external_window.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
        L.db_exchange_peer.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint64]
        L.db_step_profiled.argtypes = [C.c_void_p, C.c_uint32, C.POINTER(PhaseTimes)]
        L.db_read_spikes.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_uint64,
                                     C.POINTER(C.c_uint64)]
        L.db_read_state.argtypes = [C.c_void_p, C.c_uint32, C.c_int64, C.c_int64, C.c_void_p]
        L.db_write_state.argtypes = [C.c_void_p, C.c_uint32, C.c_int64, C.c_int64, C.c_void_p]
        L.db_region_rates.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.db_read_bold.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_uint64)]
        L.db_region_counts.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.db_export_csr.argtypes = [C.c_void_p, C.POINTER(CsrHost)]
        L.db_free_csr.argtypes = [C.POINTER(CsrHost)]
        L.db_get_counters.argtypes = [C.c_void_p, C.POINTER(Counters)]
        L.db_synchronize.argtypes = [C.c_void_p]
        L.db_last_error.argtypes = [C.c_void_p]
        L.db_last_error.restype = C.c_char_p
        for f in EXPORTS:
            if f != "db_last_error":
                getattr(L, f).restype = C.c_int32
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _fill_sim_params(p: SimParams, d: dict, dyn_seed: int, exec_mode: int, raster_capacity: int, max_windows: int):
    p.struct_size = C.sizeof(SimParams)
    p.dt_ms, p.S, p.D, p.window_steps = d["dt_ms"], d["S"], d["D"], d["window_steps"]
    p.n_types = len(d["types"])
    for i, t in enumerate(d["types"][:len(p.type)]):       # (more than DB_MAX_TYPES: n_types says so and the library refuses)
        q = p.type[i]
        for k in ("C", "gL", "VL", "Vth", "Vreset", "Tref_ms", "Iext", "bg_rate_hz", "bg_weight"):
            setattr(q, k, float(t[k]))
        for k in ("ou_mu", "ou_sigma", "ou_tau_ms", "iext_gamma_shape", "iext_gamma_scale"):   # off by default
            setattr(q, k, float(t.get(k, 0.0)))
        for k in ("G", "E", "tau_ms"):
            for u in range(4):
                getattr(q, k)[u] = float(t[k][u])
    p.dyn_seed = int(dyn_seed)
    p.raster_capacity = int(raster_capacity)
    p.max_windows = int(max_windows)
    p.exec_mode = int(exec_mode)
    p.spike_bin_steps = int(d.get("spike_bin_steps", 1))
    if d.get("bold"):                                         # Balloon-Windkessel read-out: dict with BOLD_KEYS
        p.bold.enabled = 1
        for k in BOLD_KEYS:
            setattr(p.bold, k, float(d["bold"][k]))


class _TorchRuntime:
    """Device memory from torch (one uint8 tensor per allocation) and torch's current stream."""

    def __init__(self, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_2211_15963_b200 has no CPU path")
        self.torch = torch
        self.device = device
        self.blocks = {}
        torch.cuda.set_device(device)

        def _alloc(nbytes, _user):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=f"cuda:{device}")
            except Exception:
                return None
            self.blocks[t.data_ptr()] = t
            return t.data_ptr()

        def _free(ptr, _user):
            self.blocks.pop(ptr, None)

        self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)
        self.rt = Runtime(self._alloc_cb, self._free_cb, None,
                          C.c_void_p(torch.cuda.current_stream(device).cuda_stream), device)


_probe_lib = None


def db_probe_scatter(region_bytes: int, n_ops: int = 1 << 24, reps: int = 5, device: int = 0) -> float:
    """Random 4-byte reductions per second into a region of `region_bytes`: bench-only measurement helper
    (libdb_probe.so, csrc/db_probe.cu), not part of the product ABI."""
    global _probe_lib
    if _probe_lib is None:
        _build.build()
        _probe_lib = C.CDLL(_build.PROBE_LIB)
        _probe_lib.db_probe_scatter.argtypes = [C.c_int32, C.c_uint64, C.c_uint64, C.c_uint32, C.POINTER(C.c_double)]
        _probe_lib.db_probe_scatter.restype = C.c_int32
    out = C.c_double()
    rc = _probe_lib.db_probe_scatter(int(device), int(region_bytes), int(n_ops), int(reps), C.byref(out))
    if rc != DB_OK:
        raise DbError(rc, "db_probe_scatter failed")
    return out.value


class Sim:
    """One simulation handle.  Methods carry the names of the C calls."""

    def __init__(self):
        self.h = C.c_void_p()
        self.L = load()
        self._rt = None
        self.N = self.D = self.R = 0
        self.dt_ms = 0.0
        self.window = 1

    # -- construction --------------------------------------------------------
    @classmethod
    def db_create(cls, net: dict, sim: dict, seed: int, dyn_seed: int = 1, exec_mode: int = EXEC_AUTO,
                  raster_capacity: int = 0, max_windows: int = 0, device: int = 0, own=None) -> "Sim":
        s = cls()
        s._rt = _TorchRuntime(device)
        spec = NetworkSpec()
        spec.struct_size = C.sizeof(NetworkSpec)
        for k, _ in NetworkSpec._fields_:
            if k in net:
                setattr(spec, k, net[k])
        _fill_sim_params(spec.sim, sim, dyn_seed, exec_mode, raster_capacity, max_windows)
        spec.runtime = C.pointer(s._rt.rt)
        if own is not None:                              # (first, count): the neurons this handle owns
            spec.own_first, spec.own_count = int(own[0]), int(own[1])
        rc = s.L.db_create(C.byref(spec), int(seed), C.byref(s.h))
        if rc != DB_OK:
            raise DbError(rc, s.L.db_last_error(None).decode())
        s._remember(net["N"], net["n_regions"], sim, own)
        return s

    @classmethod
    def db_create_from_csr(cls, sim: dict, net: dict, dyn_seed: int = 1, exec_mode: int = EXEC_AUTO,
                           raster_capacity: int = 0, max_windows: int = 0, fp16: bool = False,
                           device: int = 0, own=None) -> "Sim":
        s = cls()
        s._rt = _TorchRuntime(device)
        sp = SimParams()
        _fill_sim_params(sp, sim, dyn_seed, exec_mode, raster_capacity, max_windows)
        N = int(net["N"])
        R = int(net.get("n_regions", 1))
        keep = [np.ascontiguousarray(net.get("region_start", np.array([0, N])), np.int64),
                np.ascontiguousarray(net["ntype"], np.uint8), np.ascontiguousarray(net["row_ptr"], np.int64),
                np.ascontiguousarray(net["tgt"], np.int32), np.ascontiguousarray(net["w"], np.float32),
                np.ascontiguousarray(net["delay"], np.uint8), np.ascontiguousarray(net["rec"], np.uint8)]
        v = CsrView(N, int(keep[2][-1]), R, *[_p(a) for a in keep], int(fp16), *(own if own is not None else (0, 0)))
        rc = s.L.db_create_from_csr(C.byref(sp), C.byref(v), C.byref(s._rt.rt), C.byref(s.h))
        if rc != DB_OK:
            raise DbError(rc, s.L.db_last_error(None).decode())
        s._remember(N, R, sim, own)
        return s

    def _remember(self, N, R, sim, own=None):
        self.N, self.R, self.D = int(N), int(R), int(sim["D"])
        self.first, self.count = (int(own[0]), int(own[1])) if own is not None and own[1] else (0, int(N))
        self.dt_ms, self.window = float(sim["dt_ms"]), int(sim["window_steps"])

    def _ck(self, rc):
        if rc != DB_OK:
            raise DbError(rc, self.L.db_last_error(self.h).decode())

    def db_destroy(self):
        if self.h:
            self.L.db_destroy(self.h)
            self.h = C.c_void_p()

    close = db_destroy

    def __del__(self):
        try:
            self.db_destroy()
        except Exception:
            pass

    # -- stepping ----------------------------------------------------------------
    def db_step(self, n_steps: int):
        self._ck(self.L.db_step(self.h, int(n_steps)))

    def db_deliver_external(self, step: int, ids: np.ndarray):
        ids = np.ascontiguousarray(ids, np.int32)
        self._ck(self.L.db_deliver_external(self.h, int(step), _p(ids), len(ids)))

    def db_deliver_external_window(self, step_begin: int, n_steps: int, steps: np.ndarray, ids: np.ndarray):
        """The spikes (steps[k], ids[k]), sorted by step as db_read_spikes returns them, all inside
        [step_begin, step_begin + n_steps): one call, one launch."""
        ids = np.ascontiguousarray(ids, np.int32)
        offs = np.searchsorted(np.asarray(steps, np.int64), np.arange(step_begin, step_begin + n_steps + 1)).astype(np.uint64)
        assert offs[0] == 0 and offs[-1] == len(ids), "steps outside the window or not sorted"
        self._ck(self.L.db_deliver_external_window(self.h, int(step_begin), int(n_steps), _p(offs), _p(ids)))

    def db_exchange_peer(self, src: "Sim", step_begin: int, step_end: int):
        """Push the rows of the spikes `src` fired in [step_begin, step_end), read from its raster on the device."""
        self._ck(self.L.db_exchange_peer(self.h, src.h, int(step_begin), int(step_end)))

    def db_deliver_external_static(self, step: int, ids: np.ndarray):
        """db_deliver_external without any device allocation (at most EXTERNAL_STATIC_MAX ids per call)."""
        ids = np.ascontiguousarray(ids, np.int32)
        self._ck(self.L.db_deliver_external_static(self.h, int(step), _p(ids), len(ids)))

    def db_step_profiled(self, n_steps: int) -> dict:
        t = PhaseTimes()
        self._ck(self.L.db_step_profiled(self.h, int(n_steps), C.byref(t)))
        return {k: getattr(t, k) for k, _ in PhaseTimes._fields_}

    def db_synchronize(self):
        self._ck(self.L.db_synchronize(self.h))

    # -- read-back -----------------------------------------------------------------
    def db_get_counters(self) -> dict:
        c = Counters()
        self._ck(self.L.db_get_counters(self.h, C.byref(c)))
        return {k: getattr(c, k) for k, _ in Counters._fields_}

    def db_read_spikes(self, step_begin: int, step_end: int, steps_out=None, ids_out=None):
        """Returns (steps, ids) sorted by (step, id); optional preallocated host buffers."""
        n = C.c_uint64()
        if steps_out is None or ids_out is None:
            self._ck(self.L.db_read_spikes(self.h, step_begin, step_end, None, None, 0, C.byref(n)))
            steps_out = np.empty(n.value, np.uint64)
            ids_out = np.empty(n.value, np.int32)
        self._ck(self.L.db_read_spikes(self.h, step_begin, step_end, _p(steps_out), _p(ids_out),
                                       len(ids_out), C.byref(n)))
        m = min(n.value, len(ids_out))
        return steps_out[:m], ids_out[:m]

    def db_read_state(self, field: int, first: int | None = None, count: int | None = None) -> np.ndarray:
        first = self.first if first is None else first
        count = self.first + self.count - first if count is None else count
        if field == FIELD_RING:
            out = np.empty((self.D, count, 4), np.int32)
        elif field in (FIELD_REF, FIELD_OUTDEG):
            out = np.empty(count, np.int32)
        elif field == FIELD_TYPE:
            out = np.empty(count, np.uint8)
        else:
            out = np.empty(count, np.float32)
        self._ck(self.L.db_read_state(self.h, field, first, count, _p(out)))
        return out

    def db_write_state(self, field: int, values: np.ndarray, first: int | None = None):
        first = self.first if first is None else first
        dt = np.int32 if field in (FIELD_REF, FIELD_RING) else np.float32
        v = np.ascontiguousarray(values, dt)
        count = v.shape[1] if field == FIELD_RING else v.shape[0]
        self._ck(self.L.db_write_state(self.h, field, first, count, _p(v)))

    def db_region_counts(self):
        n, first = C.c_uint64(), C.c_uint64()
        self._ck(self.L.db_region_counts(self.h, None, 0, C.byref(n), C.byref(first)))
        out = np.empty((n.value, self.R), np.uint32)
        self._ck(self.L.db_region_counts(self.h, _p(out), n.value, C.byref(n), C.byref(first)))
        return out, first.value

    def db_read_bold(self):
        """(y [regions], state [regions][4] = s, f, v, q, windows consumed), fp64."""
        n = C.c_uint64()
        y = np.empty(self.R, np.float64)
        st = np.empty((self.R, 4), np.float64)
        self._ck(self.L.db_read_bold(self.h, _p(y), _p(st), C.byref(n)))
        return y, st, n.value

    def db_region_rates(self):
        n, first = C.c_uint64(), C.c_uint64()
        self._ck(self.L.db_region_rates(self.h, None, 0, C.byref(n), C.byref(first)))
        out = np.empty((n.value, self.R), np.float32)
        self._ck(self.L.db_region_rates(self.h, _p(out), n.value, C.byref(n), C.byref(first)))
        return out, first.value

    def db_export_csr(self) -> dict:
        c = CsrHost()
        self._ck(self.L.db_export_csr(self.h, C.byref(c)))
        N, E, R = c.N, c.E, c.n_regions
        arr = np.ctypeslib.as_array
        out = dict(N=N, E=E, n_regions=R, region_start=arr(c.region_start, (R + 1,)).copy(),
                   ntype=arr(c.ntype, (N,)).copy(), row_ptr=arr(c.row_ptr, (N + 1,)).copy(),
                   tgt=arr(c.tgt, (max(E, 1),))[:E].copy(), w=arr(c.w, (max(E, 1),))[:E].copy(),
                   delay=arr(c.delay, (max(E, 1),))[:E].copy(), rec=arr(c.rec, (max(E, 1),))[:E].copy())
        self.L.db_free_csr(C.byref(c))
        return out

    # -- convenience (pure marshalling) ---------------------------------------------
    def state(self):
        V = self.db_read_state(FIELD_V)
        g = np.stack([self.db_read_state(FIELD_G_AMPA + u) for u in range(4)], axis=1)
        ref = self.db_read_state(FIELD_REF)
        return V, g, ref

    def set_state(self, V, g, ref):
        self.db_write_state(FIELD_V, V)
        for u in range(4):
            self.db_write_state(FIELD_G_AMPA + u, np.ascontiguousarray(g[:, u]))
        self.db_write_state(FIELD_REF, ref)
