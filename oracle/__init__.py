"""ctypes binding of the ORACLE (test infrastructure, not product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "db_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_LIB_OMP = os.path.join(_HERE, "liboracle_omp.so")      # same source with -fopenmp: the all-cores timing leg of bench.py
_lib = None

CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", *CXXFLAGS, "-o", _LIB, _SRC])
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", *CXXFLAGS, "-fopenmp", "-o", _LIB_OMP, _SRC])
    return _LIB


def use_all_cores(on: bool = True):
    """Switch this process to the -fopenmp build of the same source (loops over neurons and over spikes shared among
    the host cores, integer atomics in delivery: same results) or back.  Handles created before the switch stay valid
    only with the library that made them: switch before creating simulators."""
    global _lib
    _lib = None
    globals()["_ACTIVE"] = _LIB_OMP if on else _LIB


class TypeParams(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("C", "gL", "VL", "Vth", "Vreset", "Tref_ms", "Iext")] + [
        ("G", C.c_double * 4), ("E", C.c_double * 4), ("tau_ms", C.c_double * 4),
        ("bg_rate_hz", C.c_double), ("bg_weight", C.c_double),
        ("ou_mu", C.c_double), ("ou_sigma", C.c_double), ("ou_tau_ms", C.c_double),
        ("iext_gamma_shape", C.c_double), ("iext_gamma_scale", C.c_double)]


class SimParams(C.Structure):
    _fields_ = [("dt_ms", C.c_double), ("S", C.c_int32), ("D", C.c_int32), ("window_steps", C.c_int32),
                ("n_types", C.c_int32), ("type", TypeParams * 8), ("spike_bin_steps", C.c_int32)]


class NetSpec(C.Structure):
    _fields_ = [("N", C.c_int64), ("n_regions", C.c_int32), ("region_size_sigma", C.c_double),
                ("exc_frac", C.c_double), ("mode", C.c_int32), ("K", C.c_int32), ("intra_frac", C.c_double),
                ("region_matrix_sigma", C.c_double), ("outdeg_mean", C.c_double), ("outdeg_sigma", C.c_double),
                ("outdeg_cap", C.c_int32), ("w_mu", C.c_double), ("w_sigma", C.c_double), ("w_scale", C.c_double),
                ("inh_mult", C.c_double), ("slow_frac", C.c_double),
                ("delay_intra_min", C.c_int32), ("delay_intra_max", C.c_int32),
                ("delay_inter_min", C.c_int32), ("delay_inter_max", C.c_int32), ("weight_fp16", C.c_int32)]


class Network(C.Structure):
    _fields_ = [("N", C.c_int64), ("E", C.c_int64), ("n_regions", C.c_int32),
                ("region_start", C.POINTER(C.c_int64)), ("region_nexc", C.POINTER(C.c_int64)),
                ("ntype", C.POINTER(C.c_uint8)), ("row_ptr", C.POINTER(C.c_int64)),
                ("tgt", C.POINTER(C.c_int32)), ("w", C.POINTER(C.c_float)),
                ("delay", C.POINTER(C.c_uint8)), ("rec", C.POINTER(C.c_uint8))]


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(globals().get("_ACTIVE", _LIB))
        L.orc_generate.restype = C.POINTER(Network)
        L.orc_generate.argtypes = [C.POINTER(NetSpec), C.c_uint64]
        L.orc_network_free.argtypes = [C.POINTER(Network)]
        L.orc_gen_create.restype = C.c_void_p
        L.orc_gen_create.argtypes = [C.POINTER(NetSpec), C.c_uint64]
        L.orc_gen_destroy.argtypes = [C.c_void_p]
        L.orc_gen_ntype.restype = C.c_int32
        L.orc_gen_ntype.argtypes = [C.c_void_p, C.c_int64]
        L.orc_gen_owner_edges.restype = C.c_int64
        L.orc_gen_owner_edges.argtypes = [C.c_void_p, C.c_int64, C.c_int64] + [C.c_void_p] * 5
        L.orc_sim_create.restype = C.c_void_p
        L.orc_sim_create.argtypes = [C.POINTER(SimParams), C.c_int64, C.c_void_p, C.c_int32, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_uint64, C.c_int32]
        L.orc_sim_destroy.argtypes = [C.c_void_p]
        L.orc_sim_step.argtypes = [C.c_void_p, C.c_int64]
        for f in ("orc_sim_step_index", "orc_sim_n_spikes", "orc_sim_n_events", "orc_sim_n_bg"):
            getattr(L, f).restype = C.c_uint64
            getattr(L, f).argtypes = [C.c_void_p]
        L.orc_sim_overflow.restype = C.c_int32
        L.orc_sim_overflow.argtypes = [C.c_void_p]
        L.orc_sim_get_spikes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_sim_get_state.argtypes = [C.c_void_p] * 4
        L.orc_sim_set_state.argtypes = [C.c_void_p] * 4
        L.orc_sim_get_ring.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_sim_set_ring.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_sim_get_iou.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_sim_set_iou.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_sim_get_iext.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_gamma_ppf.restype = C.c_double
        L.orc_gamma_ppf.argtypes = [C.c_double] * 3
        L.orc_gamma_table.argtypes = [C.c_double, C.c_double, C.c_void_p]
        L.orc_normal_table.argtypes = [C.c_void_p]
        L.orc_sim_region_counts.restype = C.c_int64
        L.orc_sim_region_counts.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_sim_log_arrivals.argtypes = [C.c_void_p, C.c_int32]
        L.orc_sim_get_arrivals.restype = C.c_uint64
        L.orc_sim_get_arrivals.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_philox.argtypes = [C.c_uint32] * 6 + [C.c_void_p]
        L.orc_draw.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint64, C.c_void_p]
        L.orc_poisson_thresholds.restype = C.c_int32
        L.orc_poisson_thresholds.argtypes = [C.c_double, C.c_void_p]
        L.orc_poisson_count.restype = C.c_int32
        L.orc_poisson_count.argtypes = [C.c_uint32, C.c_void_p, C.c_int32]
        L.orc_prp.restype = C.c_uint32
        L.orc_prp.argtypes = [C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_norm_ppf.restype = C.c_double
        L.orc_norm_ppf.argtypes = [C.c_double]
        L.orc_round_to_half.restype = C.c_float
        L.orc_round_to_half.argtypes = [C.c_float]
        L.orc_weight_table.argtypes = [C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.orc_outdeg_table.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_void_p]
        L.orc_region_sizes.argtypes = [C.c_uint64, C.c_int64, C.c_int32, C.c_double, C.c_void_p]
        L.orc_region_cdf.argtypes = [C.c_uint64, C.c_int32, C.c_double, C.c_void_p]
        L.orc_dense_arrivals.argtypes = [C.c_int64, C.c_int64, C.c_int32] + [C.c_void_p] * 7
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


# ---- raw pieces (pins) -------------------------------------------------------
def philox(c, k):
    out = np.zeros(4, np.uint32)
    lib().orc_philox(*[int(x) for x in c], *[int(x) for x in k], _p(out))
    return out


def draw(seed, stream, a, b):
    out = np.zeros(4, np.uint32)
    lib().orc_draw(int(seed), int(stream), int(a), int(b), _p(out))
    return out


def poisson_thresholds(lam):
    T = np.zeros(32, np.uint32)
    M = lib().orc_poisson_thresholds(float(lam), _p(T))
    return T[:M].copy()


def poisson_count(u, T):
    T = np.ascontiguousarray(T, np.uint32)
    return lib().orc_poisson_count(int(u), _p(T), len(T))


def prp(x, M, key4):
    key4 = np.ascontiguousarray(key4, np.uint32)
    return lib().orc_prp(int(x), int(M), _p(key4))


def weight_table(mu, sigma, scale):
    t = np.zeros(65536, np.float32)
    lib().orc_weight_table(mu, sigma, scale, _p(t))
    return t


def outdeg_table(mean, sigma, cap):
    t = np.zeros(65536, np.int32)
    lib().orc_outdeg_table(mean, sigma, cap, _p(t))
    return t


def region_sizes(seed, N, R, sigma):
    s = np.zeros(R, np.int64)
    lib().orc_region_sizes(int(seed), int(N), int(R), float(sigma), _p(s))
    return s


def region_cdf(seed, R, sigma):
    t = np.zeros((R, R - 1), np.uint32)
    lib().orc_region_cdf(int(seed), int(R), float(sigma), _p(t))
    return t


# ---- generator -------------------------------------------------------------------
def _net_spec(d: dict) -> NetSpec:
    s = NetSpec()
    for k, _ in NetSpec._fields_:
        setattr(s, k, d[k])
    return s


def generate(net: dict, seed: int) -> dict:
    """Run the oracle's network generator; returns numpy copies (CSR rows sorted by target)."""
    L = lib()
    sp = _net_spec(net)
    h = L.orc_generate(C.byref(sp), int(seed))
    if not h:
        raise ValueError("oracle.generate: a region is too small for the requested in-degree (sampling without replacement)")
    n = h.contents
    N, E, R = n.N, n.E, n.n_regions
    out = dict(
        N=N, E=E, n_regions=R,
        region_start=np.ctypeslib.as_array(n.region_start, (R + 1,)).copy(),
        region_nexc=np.ctypeslib.as_array(n.region_nexc, (R,)).copy(),
        ntype=np.ctypeslib.as_array(n.ntype, (N,)).copy(),
        row_ptr=np.ctypeslib.as_array(n.row_ptr, (N + 1,)).copy(),
        tgt=np.ctypeslib.as_array(n.tgt, (max(E, 1),))[:E].copy(),
        w=np.ctypeslib.as_array(n.w, (max(E, 1),))[:E].copy(),
        delay=np.ctypeslib.as_array(n.delay, (max(E, 1),))[:E].copy(),
        rec=np.ctypeslib.as_array(n.rec, (max(E, 1),))[:E].copy(),
    )
    L.orc_network_free(h)
    return out


class OwnerEdges:
    """The synapses owned by single neurons (their K inputs, or in out-degree mode their
    outputs), without building the whole network: sampled parity at full size."""

    def __init__(self, net: dict, seed: int):
        sp = _net_spec(net)
        self.h = lib().orc_gen_create(C.byref(sp), int(seed))
        self.cap = max(int(net["K"]), int(net["outdeg_cap"])) + 1

    def __call__(self, i: int) -> dict:
        cap = self.cap
        src, tgt = np.zeros(cap, np.int32), np.zeros(cap, np.int32)
        w, d, r = np.zeros(cap, np.float32), np.zeros(cap, np.uint8), np.zeros(cap, np.uint8)
        n = lib().orc_gen_owner_edges(self.h, int(i), cap, _p(src), _p(tgt), _p(w), _p(d), _p(r))
        assert n <= cap
        return dict(src=src[:n], tgt=tgt[:n], w=w[:n], delay=d[:n], rec=r[:n])

    def ntype(self, first: int, count: int) -> np.ndarray:
        return np.array([lib().orc_gen_ntype(self.h, int(i)) for i in range(first, first + count)], np.uint8)

    def close(self):
        if self.h:
            lib().orc_gen_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- simulator ------------------------------------------------------------------
def _sim_params(d: dict) -> SimParams:
    p = SimParams()
    p.dt_ms, p.S, p.D, p.window_steps = d["dt_ms"], d["S"], d["D"], d["window_steps"]
    p.n_types = len(d["types"])
    p.spike_bin_steps = int(d.get("spike_bin_steps", 1))      # time bin b_t for transferring spikes (R29), in steps
    for i, t in enumerate(d["types"]):
        q = p.type[i]
        for k in ("C", "gL", "VL", "Vth", "Vreset", "Tref_ms", "Iext", "bg_rate_hz", "bg_weight"):
            setattr(q, k, float(t[k]))
        for k in ("ou_mu", "ou_sigma", "ou_tau_ms", "iext_gamma_shape", "iext_gamma_scale"):   # off by default
            setattr(q, k, float(t.get(k, 0.0)))
        for k in ("G", "E", "tau_ms"):
            for u in range(4):
                getattr(q, k)[u] = float(t[k][u])
    return p


class OracleSim:
    """The oracle simulator on one network (fp32 parity mode, or fp64 for closed-form pins)."""

    def __init__(self, sim: dict, net: dict, seed: int, fp64: bool = False):
        self.N = int(net["N"])
        self.D = int(sim["D"])
        self.R = int(net.get("n_regions", 1))
        self.window = int(sim["window_steps"])
        self.dt_ms = float(sim["dt_ms"])
        rs = np.ascontiguousarray(net.get("region_start", np.array([0, self.N])), np.int64)
        self._keep = [np.ascontiguousarray(net["ntype"], np.uint8), rs,
                      np.ascontiguousarray(net["row_ptr"], np.int64), np.ascontiguousarray(net["tgt"], np.int32),
                      np.ascontiguousarray(net["w"], np.float32), np.ascontiguousarray(net["delay"], np.uint8),
                      np.ascontiguousarray(net["rec"], np.uint8)]
        k = self._keep
        p = _sim_params(sim)
        self.h = lib().orc_sim_create(C.byref(p), self.N, _p(k[0]), self.R, _p(k[1]), _p(k[2]), _p(k[3]),
                                      _p(k[4]), _p(k[5]), _p(k[6]), int(seed), int(fp64))

    def close(self):
        if self.h:
            lib().orc_sim_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def step(self, n=1):
        lib().orc_sim_step(self.h, int(n))

    @property
    def step_index(self):
        return lib().orc_sim_step_index(self.h)

    def counters(self):
        L = lib()
        return dict(steps=L.orc_sim_step_index(self.h), spikes=L.orc_sim_n_spikes(self.h),
                    events=L.orc_sim_n_events(self.h), bg_events=L.orc_sim_n_bg(self.h),
                    overflow=L.orc_sim_overflow(self.h))

    def spikes(self):
        n = lib().orc_sim_n_spikes(self.h)
        st = np.zeros(n, np.uint64)
        ids = np.zeros(n, np.int32)
        lib().orc_sim_get_spikes(self.h, _p(st), _p(ids))
        return st, ids

    def state(self):
        V = np.zeros(self.N, np.float64)
        g = np.zeros((self.N, 4), np.float64)
        ref = np.zeros(self.N, np.int32)
        lib().orc_sim_get_state(self.h, _p(V), _p(g), _p(ref))
        return V, g, ref

    def set_state(self, V, g, ref):
        V = np.ascontiguousarray(V, np.float64)
        g = np.ascontiguousarray(g, np.float64)
        ref = np.ascontiguousarray(ref, np.int32)
        lib().orc_sim_set_state(self.h, _p(V), _p(g), _p(ref))

    def iou(self):
        out = np.zeros(self.N, np.float64)
        lib().orc_sim_get_iou(self.h, _p(out))
        return out

    def iext(self):
        """External current of every neuron (R31): a parameter drawn once at creation."""
        out = np.zeros(self.N, np.float64)
        lib().orc_sim_get_iext(self.h, _p(out))
        return out

    def set_iou(self, v):
        v = np.ascontiguousarray(v, np.float64)
        assert v.shape == (self.N,)
        lib().orc_sim_set_iou(self.h, _p(v))

    def ring(self):
        r = np.zeros((self.D, self.N, 4), np.int32)
        lib().orc_sim_get_ring(self.h, _p(r))
        return r

    def set_ring(self, r):
        r = np.ascontiguousarray(r, np.int32)
        assert r.shape == (self.D, self.N, 4)
        lib().orc_sim_set_ring(self.h, _p(r))

    def region_counts(self):
        nw = lib().orc_sim_region_counts(self.h, None, 0)
        out = np.zeros((nw, self.R), np.uint32)
        lib().orc_sim_region_counts(self.h, _p(out), nw)
        return out

    def region_rates(self, region_sizes):
        """Hz: spikes in window / (region size * window seconds) (R24)."""
        c = self.region_counts().astype(np.float64)
        return c / (np.asarray(region_sizes, np.float64)[None, :] * self.window * self.dt_ms * 1e-3)

    def log_arrivals(self, on=True):
        lib().orc_sim_log_arrivals(self.h, int(on))

    def arrivals(self):
        n = lib().orc_sim_get_arrivals(self.h, None)
        a = np.zeros(n, np.int32)
        lib().orc_sim_get_arrivals(self.h, _p(a))
        return a.reshape(-1, self.N, 4)


def gamma_table(shape: float, scale: float) -> np.ndarray:
    """The 65536 Gamma(shape, scale) quantiles (fp32) the per-neuron external currents are drawn from."""
    tab = np.zeros(65536, np.float32)
    lib().orc_gamma_table(float(shape), float(scale), _p(tab))
    return tab


def normal_table() -> np.ndarray:
    """The 65536 standard-normal quantiles (fp32) the OU increments are drawn from."""
    tab = np.zeros(65536, np.float32)
    lib().orc_normal_table(_p(tab))
    return tab


def dense_arrivals(net: dict, S: int, spikes: np.ndarray) -> np.ndarray:
    """Plain definition of the delivered sums: dense matrix x delayed spike vectors."""
    T, N = spikes.shape
    out = np.zeros((T, N, 4), np.int64)
    sp = np.ascontiguousarray(spikes, np.uint8)
    a = [np.ascontiguousarray(net["row_ptr"], np.int64), np.ascontiguousarray(net["tgt"], np.int32),
         np.ascontiguousarray(net["w"], np.float32), np.ascontiguousarray(net["delay"], np.uint8),
         np.ascontiguousarray(net["rec"], np.uint8)]
    lib().orc_dense_arrivals(N, T, int(S), *[_p(x) for x in a], _p(sp), _p(out))
    return out


# ---- Balloon-Windkessel BOLD read-out (Extended Data Table 4) ---------------------------
# Test infrastructure like everything else in this package.  Reading R30: the table prints the
# equations only; "BW(.) is the Euler-Maruyama discrete-time version of the Balloon-Windkessel model",
# its noise term is not specified and is left out, so one explicit Euler step per region-rate window; the neural
# activity z_i is "the spike rate of a pool of neurons": z = z_scale * (region rate in Hz).
# The constants are not printed either; the defaults are the usual ones of the paper's reference 19
# (Friston et al. 2000) -- builder's choice, "parity unpinned" for their values.
BOLD_DEFAULTS = dict(kappa=0.65, gamma=0.41, tau=0.98, alpha=0.32, rho=0.34, V0=0.02,
                     k1=7 * 0.34, k2=2.0, k3=2 * 0.34 - 0.2, z_scale=0.1)


def bold_signal(state: np.ndarray, prm: dict) -> np.ndarray:
    """y_i = V0 [k1 (1 - q) + k2 (1 - q / v) + k3 (1 - v)]; state[..., 4] = s, f, v, q."""
    v, q = state[..., 2], state[..., 3]
    return prm["V0"] * (prm["k1"] * (1.0 - q) + prm["k2"] * (1.0 - q / v) + prm["k3"] * (1.0 - v))


def bold_step(state: np.ndarray, z: np.ndarray, h: float, prm: dict) -> np.ndarray:
    """One explicit Euler step of length h (seconds) of the four equations of, all right-hand
    sides taken at time t."""
    s, f, v, q = (state[..., k] for k in range(4))
    fout = v ** (1.0 / prm["alpha"])                                  # f_out = v^(1/alpha)
    E = 1.0 - (1.0 - prm["rho"]) ** (1.0 / f)                         # E(f, rho) = 1 - (1 - rho)^(1/f)
    ds = z - prm["kappa"] * s - prm["gamma"] * (f - 1.0)              # s' = z - kappa s - gamma (f - 1)
    df = s                                                            # f' = s
    dv = (f - fout) / prm["tau"]                                      # tau v' = f - v^(1/alpha)
    dq = (f * E / prm["rho"] - fout * q / v) / prm["tau"]             # tau q' = f E / rho - v^(1/alpha) q / v
    return np.stack([s + h * ds, f + h * df, v + h * dv, q + h * dq], axis=-1)


def bold_rest(n_regions: int) -> np.ndarray:
    """Resting state s = 0, f = v = q = 1 (y = 0)."""
    st = np.ones((n_regions, 4), np.float64)
    st[:, 0] = 0.0
    return st


def bold_run(counts: np.ndarray, region_sizes: np.ndarray, window_s: float, prm: dict, state: np.ndarray | None = None):
    """Feed region spike counts [windows][regions] through the model, one Euler step per window.
    Returns (y [windows][regions] after each step, final state [regions][4])."""
    counts = np.asarray(counts, np.float64)
    sizes = np.asarray(region_sizes, np.float64)
    st = bold_rest(counts.shape[1]) if state is None else np.array(state, np.float64)
    ys = np.zeros(counts.shape, np.float64)
    for w in range(counts.shape[0]):
        rate_hz = counts[w] / (sizes * window_s)                      # R24
        st = bold_step(st, prm["z_scale"] * rate_hz, window_s, prm)
        ys[w] = bold_signal(st, prm)
    return ys, st
