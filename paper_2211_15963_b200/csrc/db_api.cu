// C ABI of the library (include/db_b200.h): handle management, host-side
// constant tables, CSR upload, step scheduling (CUDA graph / persistent
// kernel) and read-back.  All simulation work is done by the kernels in
// db_step.cu and db_gen.cu; nothing here computes on the CPU what the step
// path computes.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "../../include/db_b200.h"
#include "db_device.cuh"
#include "db_host.h"

using namespace dbk;

static thread_local std::string g_create_error;

struct db_sim {
    SimDev dev{};
    db_sim_params params{};
    db_runtime rt{};
    bool have_rt = false;
    cudaStream_t stream = nullptr;
    int device = 0, n_sm = 0;
    std::vector<void*> allocs;
    int64_t E = 0, Epad = 0;
    uint64_t spike_cap = 0, work_cap = 0;
    std::vector<int64_t> region_start;
    uint8_t* ntype_dev = nullptr;
    float* iext_tab_dev = nullptr;  // [kMaxTypes][65536] Gamma quantiles of the per-neuron external currents (R31)
    int exec_mode = DB_EXEC_KERNELS;
    int deliver_grid = 0;
    bool heavy = false;             // some row is longer than kInlineMax
    int32_t max_delay = 0;          // largest synaptic delay, in steps
    int32_t min_delay = 1;          // smallest one (db_deliver_external: how late an outside spike may arrive)
    int32_t* ext_ids_dev = nullptr; // db_deliver_external: device copy of the id list
    uint64_t ext_ids_cap = 0;
    cudaEvent_t xchg_event = nullptr; // db_exchange_peer: orders this handle's stream after the source's
    int xchg_event_dev = -1;          // device the event was created on (the source's)
    double list_rate_hz = 0.0;      // arrival lists: mean firing rate their capacity was sized for
    int update_sm = 0;              // two-kernel mode: SM count the update kernel is shaped for
    cudaGraphExec_t graph_exec = nullptr;
    int graph_steps = 0;
    uint64_t host_step = 0;         // steps launched so far (two-kernel modes: parity of the work-list half)
    uint64_t launches = 0;
    std::vector<cudaEvent_t> prof_events;
    BoldDev bold{};                 // BOLD read-out (params.bold.enabled)
    uint32_t bold_batch = 0;        // steps after which the read-out must catch up (history ring of the region counts)
    std::string err;
};

namespace {

#define CK(call)                                                                         \
    do {                                                                                 \
        cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess) {                                                         \
            return fail(sim, DB_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
        }                                                                                \
    } while (0)

int32_t fail(db_sim* sim, int32_t code, const std::string& msg) {
    if (sim) sim->err = msg;
    g_create_error = msg;
    return code;
}

void* dev_alloc(db_sim* sim, size_t bytes) {
    if (bytes == 0) bytes = 256;
    void* p = nullptr;
    if (sim->have_rt && sim->rt.alloc) p = sim->rt.alloc(bytes, sim->rt.user);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
    if (p) sim->allocs.push_back(p);
    return p;
}

void dev_free_all(db_sim* sim) {
    for (void* p : sim->allocs) {
        if (sim->have_rt && sim->rt.free) sim->rt.free(p, sim->rt.user);
        else cudaFree(p);
    }
    sim->allocs.clear();
}

template <typename T>
int32_t alloc_zero(db_sim* sim, T** out, size_t count) {
    *out = static_cast<T*>(dev_alloc(sim, count * sizeof(T)));
    if (!*out) return fail(sim, DB_ENOMEM, "device allocation of " + std::to_string(count * sizeof(T)) + " bytes failed");
    CK(cudaMemsetAsync(*out, 0, std::max<size_t>(count * sizeof(T), 1), sim->stream));
    return DB_OK;
}

uint64_t next_pow2(uint64_t x) { uint64_t p = 1; while (p < x) p <<= 1; return p; }

// Per-type constants, formed in double and rounded once to fp32 (DESIGN.md
// "Arithmetic contract").  Poisson thresholds: c_m = c_{m-1} + p_m with
// p_0 = exp(-lambda), p_m = (p_{m-1} * lambda) / m; T_m = floor(c_m * 2^32);
// the table ends where it saturates.
int32_t make_type_consts(db_sim* sim, const db_sim_params& sp, TypeConst* tc) {
    for (int t = 0; t < sp.n_types; ++t) {
        const db_type_params& q = sp.type[t];
        if (!(q.C > 0) || !(q.gL >= 0) || !(q.Tref_ms >= 0) || !(q.bg_rate_hz >= 0))
            return fail(sim, DB_EINVAL, "type parameters out of range");
        TypeConst c{};
        c.neg_gL = -(float)q.gL; c.VL = (float)q.VL; c.Vth = (float)q.Vth; c.Vreset = (float)q.Vreset;
        c.kappa = (float)(sp.dt_ms / q.C); c.Iext = (float)q.Iext;
        for (int u = 0; u < 4; ++u) {
            if (!(q.tau_ms[u] > 0)) return fail(sim, DB_EINVAL, "tau_ms must be positive");
            c.G[u] = (float)q.G[u]; c.E[u] = (float)q.E[u];
            c.alpha[u] = (float)std::exp(-sp.dt_ms / q.tau_ms[u]);
        }
        const long R = std::lrint(q.Tref_ms / sp.dt_ms);
        if (R < 0 || R > kRefMask) return fail(sim, DB_EINVAL, "Tref/dt must be within 0..4095 steps");
        c.R = (int32_t)R;
        const double wq = std::rint(q.bg_weight * std::ldexp(1.0, sp.S));
        if (std::fabs(wq) > 1073741824.0) return fail(sim, DB_EINVAL, "bg_weight * 2^S overflows");
        c.wq_bg = (int32_t)wq;
        const double lambda = q.bg_rate_hz * sp.dt_ms * 1e-3;
        double term = std::exp(-lambda), cum = 0.0;
        int M = 0;
        bool saturated = false;
        for (int m = 0; m < kPoissonMax; ++m) {
            cum += term;
            const double thr = std::floor(cum * 4294967296.0);
            if (thr >= 4294967295.0) { saturated = true; break; }
            c.T[M++] = (uint32_t)thr;
            term = term * lambda / (double)(m + 1);
        }
        if (!saturated) return fail(sim, DB_EINVAL, "bg_rate_hz * dt too large for the Poisson table");
        c.M = M;
        if (!(q.ou_tau_ms >= 0) || !(q.ou_sigma >= 0)) return fail(sim, DB_EINVAL, "OU parameters out of range");
        if (!(q.iext_gamma_shape >= 0) || (q.iext_gamma_shape > 0 && !(q.iext_gamma_scale > 0)))
            return fail(sim, DB_EINVAL, "iext_gamma_shape must be >= 0 and iext_gamma_scale > 0 with it");
        c.ix_on = q.iext_gamma_shape > 0 ? 1 : 0;
        if (q.ou_tau_ms > 0) {          // OU background current (R3): constants formed in double, rounded once
            c.ou = 1;
            c.ou_mu = (float)q.ou_mu;
            c.ou_a = (float)(sp.dt_ms / q.ou_tau_ms);
            c.ou_s = (float)(q.ou_sigma * std::sqrt(2.0 * sp.dt_ms / q.ou_tau_ms));
        }
        tc[t] = c;
    }
    return DB_OK;
}

int32_t check_sim_params(db_sim* sim, const db_sim_params* sp) {
    if (!sp || sp->struct_size != sizeof(db_sim_params)) return fail(sim, DB_EINVAL, "db_sim_params.struct_size mismatch");
    if (!(sp->dt_ms > 0)) return fail(sim, DB_EINVAL, "dt_ms must be positive");
    if (sp->S < 0 || sp->S > 30) return fail(sim, DB_EINVAL, "S must be within 0..30");
    if (sp->D < 2 || sp->D > 65536 || (sp->D & (sp->D - 1))) return fail(sim, DB_EINVAL, "D must be a power of two in 2..65536");
    if (sp->window_steps < 1) return fail(sim, DB_EINVAL, "window_steps must be >= 1");
    if (sp->n_types < 1 || sp->n_types > DB_MAX_TYPES) return fail(sim, DB_EINVAL, "n_types must be 1..8");
    if (sp->exec_mode < DB_EXEC_AUTO || sp->exec_mode > DB_EXEC_KERNELS_DEFERRED) return fail(sim, DB_EINVAL, "bad exec_mode");
    if (sp->spike_bin_steps < 0 || sp->spike_bin_steps > 4096) return fail(sim, DB_EINVAL, "spike_bin_steps must be within 0..4096");
    return DB_OK;
}

int32_t open_device(db_sim* sim, const db_runtime* rt) {
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0)
        return fail(sim, DB_ECUDA, "no CUDA device: this library has no CPU path");
    if (rt) { sim->rt = *rt; sim->have_rt = true; sim->device = rt->device; sim->stream = (cudaStream_t)rt->stream; }
    if (sim->device < 0 || sim->device >= n_dev) return fail(sim, DB_EINVAL, "bad device ordinal");
    CK(cudaSetDevice(sim->device));
    cudaDeviceProp prop{};
    CK(cudaGetDeviceProperties(&prop, sim->device));
    sim->n_sm = prop.multiProcessorCount;
    return DB_OK;
}

// Everything except the CSR arrays: state, ring, lists, counters.
int32_t setup_common(db_sim* sim, const db_sim_params* sp, int64_t N_all, int32_t n_regions,
                     const int64_t* region_start, int32_t max_delay, int64_t own_first, int64_t own_count) {
    SimDev& d = sim->dev;
    sim->params = *sp;
    if (N_all < 1 || N_all >= (1ll << 30)) return fail(sim, DB_EINVAL, "N must be within 1..2^30-1");
    if (n_regions < 1 || n_regions > 65536) return fail(sim, DB_EINVAL, "n_regions must be 1..65536");
    if (own_count == 0) { own_first = 0; own_count = N_all; }
    if (own_first < 0 || own_count < 1 || own_first + own_count > N_all || own_first % kNeuronPad != 0)
        return fail(sim, DB_EINVAL, "own_first must be a multiple of 1024 and [own_first, own_first + own_count) lie inside the network");
    if (own_count != N_all && sp->bold.enabled)
        return fail(sim, DB_EINVAL, "the BOLD read-out needs whole regions: not available on a handle that owns part of the network");
    const int64_t N = own_count;                       // neurons of this handle: state, ring and targets are local
    d.n_rows = (int32_t)N_all;
    d.id0 = (int32_t)own_first;
    d.N = (int32_t)N;
    d.Npad = (int32_t)(((N + kNeuronPad - 1) / kNeuronPad) * kNeuronPad);
    // internal ring depth: the persistent kernel lets blocks run up to two steps apart and needs
    // depth >= largest delay + 3 (db_step.cu); the API's D (slot = step mod D) is mapped on read / write
    // (+ b_t - 1 with a time bin for transferring spikes: a row is pushed from the last step of its bin)
    d.bin_steps = sp->spike_bin_steps > 1 ? sp->spike_bin_steps : 1;
    if (max_delay + d.bin_steps - 1 >= sp->D) return fail(sim, DB_EINVAL, "largest delay + spike_bin_steps - 1 must be < D");
    d.D = (max_delay + d.bin_steps + 2 > sp->D) ? 2 * sp->D : sp->D;
    d.S = sp->S;
    d.scale = (float)std::ldexp(1.0, -sp->S);
    d.wscale = (float)std::ldexp(1.0, sp->S);
    d.seed_lo = (uint32_t)sp->dyn_seed; d.seed_hi = (uint32_t)(sp->dyn_seed >> 32);
    for (int r = 0; r < 10; ++r) {
        d.rk[2 * r] = d.seed_lo + (uint32_t)r * 0x9E3779B9u;
        d.rk[2 * r + 1] = d.seed_hi + (uint32_t)r * 0xBB67AE85u;
    }
    d.window_steps = sp->window_steps;
    d.max_windows = sp->max_windows ? sp->max_windows : 4096u;
    if (d.max_windows < 8) return fail(sim, DB_EINVAL, "max_windows must be >= 8");
    d.n_regions = n_regions;
    int32_t rc = make_type_consts(sim, *sp, d.tc);
    if (rc) return rc;
    for (int t = 0; t < sp->n_types; ++t)          // A_j is 0 or 1: nobody may fire twice inside a bin
        if (d.bin_steps > d.tc[t].R + 1) return fail(sim, DB_EINVAL, "spike_bin_steps must be <= round(Tref / dt) + 1 of every type");

    sim->region_start.assign(region_start, region_start + n_regions + 1);
    if (sim->region_start.front() != 0 || sim->region_start.back() != N_all)
        return fail(sim, DB_EINVAL, "region_start must run from 0 to N");
    std::vector<int32_t> rs32((size_t)n_regions + 1);
    for (int r = 0; r <= n_regions; ++r) {
        if (r && sim->region_start[(size_t)r] < sim->region_start[(size_t)r - 1])
            return fail(sim, DB_EINVAL, "region_start must be non-decreasing");
        rs32[(size_t)r] = (int32_t)sim->region_start[(size_t)r];
    }

    const size_t Np = (size_t)d.Npad;
    if ((rc = alloc_zero(sim, &d.V, Np))) return rc;
    if ((rc = alloc_zero(sim, &d.g, 4 * Np))) return rc;
    if ((rc = alloc_zero(sim, &d.rt, Np))) return rc;
    d.ou_on = 0;
    d.bg_on = 0;
    for (int t = 0; t < sp->n_types; ++t) { d.ou_on |= d.tc[t].ou; d.bg_on |= (d.tc[t].M > 0); }
    if (d.ou_on) {                      // OU state and the table of standard-normal quantiles its increments come from
        if ((rc = alloc_zero(sim, &d.Iou, Np))) return rc;
        float* ntab = nullptr;
        if ((rc = alloc_zero(sim, &ntab, 65536))) return rc;
        std::vector<float> tab(65536);
        for (int q = 0; q < 65536; ++q) tab[(size_t)q] = (float)std_normal_quantile(((double)q + 0.5) / 65536.0);
        CK(cudaMemcpyAsync(ntab, tab.data(), 65536 * sizeof(float), cudaMemcpyHostToDevice, sim->stream));
        CK(cudaStreamSynchronize(sim->stream));
        d.ntab = ntab;
    }
    bool ix_any = false;
    for (int t = 0; t < sp->n_types; ++t) ix_any |= d.tc[t].ix_on != 0;
    if (ix_any) {                       // per-neuron external currents (R31): the plane and the Gamma quantile tables of the types
        if ((rc = alloc_zero(sim, &d.iext, Np))) return rc;
        if ((rc = alloc_zero(sim, &sim->iext_tab_dev, (size_t)kMaxTypes * 65536))) return rc;
        std::vector<float> tab(65536);
        for (int t = 0; t < sp->n_types; ++t) {
            if (!d.tc[t].ix_on) continue;
            for (int q = 0; q < 65536; ++q)
                tab[(size_t)q] = (float)gamma_quantile(((double)q + 0.5) / 65536.0, sp->type[t].iext_gamma_shape, sp->type[t].iext_gamma_scale);
            CK(cudaMemcpyAsync(sim->iext_tab_dev + (size_t)t * 65536, tab.data(), 65536 * sizeof(float), cudaMemcpyHostToDevice, sim->stream));
            CK(cudaStreamSynchronize(sim->stream));
        }
    }
    if ((rc = alloc_zero(sim, &d.ring, (size_t)d.D * 4 * Np))) return rc;
    uint64_t cap = sp->raster_capacity ? sp->raster_capacity : (1ull << 24);
    cap = next_pow2(std::max<uint64_t>(cap, (uint64_t)N));
    sim->spike_cap = cap;
    d.spike_mask = cap - 1;
    if ((rc = alloc_zero(sim, &d.spike_ids, (size_t)cap))) return rc;
    if ((rc = alloc_zero(sim, &d.spike_tag, (size_t)cap))) return rc;
    d.step_log_mask = (1u << 16) - 1u;
    if ((rc = alloc_zero(sim, &d.step_end, (size_t)d.step_log_mask + 1))) return rc;
    int32_t* rs_dev = nullptr;
    if ((rc = alloc_zero(sim, &rs_dev, (size_t)n_regions + 1))) return rc;
    CK(cudaMemcpyAsync(rs_dev, rs32.data(), rs32.size() * sizeof(int32_t), cudaMemcpyHostToDevice, sim->stream));
    d.region_start = rs_dev;
    if ((rc = alloc_zero(sim, &d.region_counts, (size_t)d.max_windows * (size_t)n_regions))) return rc;
    if (sp->bold.enabled) {             // Balloon-Windkessel read-out per region (R30)
        const db_bold_params& bp = sp->bold;
        if (!(bp.tau > 0) || !(bp.alpha > 0) || !(bp.rho > 0 && bp.rho < 1))
            return fail(sim, DB_EINVAL, "BOLD parameters out of range (tau > 0, alpha > 0, 0 < rho < 1)");
        BoldDev& b = sim->bold;
        double* scale = nullptr;
        if ((rc = alloc_zero(sim, &b.state, 4 * (size_t)n_regions))) return rc;
        if ((rc = alloc_zero(sim, &b.y, (size_t)n_regions))) return rc;
        if ((rc = alloc_zero(sim, &scale, (size_t)n_regions))) return rc;
        if ((rc = alloc_zero(sim, &b.cursor, 1))) return rc;
        const double win_s = (double)sp->window_steps * sp->dt_ms * 1e-3;
        std::vector<double> sc((size_t)n_regions);
        for (int r = 0; r < n_regions; ++r) {
            const double size = (double)(sim->region_start[(size_t)r + 1] - sim->region_start[(size_t)r]);
            sc[(size_t)r] = size > 0 ? bp.z_scale / (size * win_s) : 0.0;
        }
        CK(cudaMemcpyAsync(scale, sc.data(), sc.size() * sizeof(double), cudaMemcpyHostToDevice, sim->stream));
        CK(cudaStreamSynchronize(sim->stream));
        b.scale = scale;
        b.kappa = bp.kappa; b.gamma = bp.gamma; b.tau = bp.tau; b.alpha = bp.alpha; b.rho = bp.rho;
        b.V0 = bp.V0; b.k1 = bp.k1; b.k2 = bp.k2; b.k3 = bp.k3; b.h = win_s;
        CK(launch_bold_init(b, n_regions, sim->stream));
        // windows kept as history: max_windows - 1 - (cleared ahead); catch up after at most half of them
        const uint64_t keep = (uint64_t)d.max_windows - 2 - 2u / (uint64_t)d.window_steps;
        sim->bold_batch = (uint32_t)std::min<uint64_t>((keep / 2) * (uint64_t)d.window_steps, 1u << 20);
    }
    if ((rc = alloc_zero(sim, &d.bg_parts, (size_t)kBgParts))) return rc;
    if ((rc = alloc_zero(sim, &d.ctl, 1))) return rc;
    if ((rc = alloc_zero(sim, &sim->ntype_dev, Np))) return rc;
    return DB_OK;
}

// DB_EXEC_KERNELS_DEFERRED: size and allocate the arrival lists, then sort every row by (delay, target window) on the
// device, batch by batch through scratch arrays.  *ok = false (and nothing changed) when the network has nothing to
// list or the lists do not fit in memory: the caller falls back to DB_EXEC_KERNELS.
int32_t build_arrival_lists(db_sim* sim, bool* ok) {
    SimDev& d = sim->dev;
    *ok = false;
    const int64_t N = d.n_rows;                        // CSR rows: one per neuron of the whole network
    const int max_ahead = sim->max_delay + d.bin_steps - 1;        // furthest arrival, in steps after the spike
    if (max_ahead <= 1 || sim->Epad < 16) return DB_OK;
    // synapses per delay
    unsigned long long* hist_dev = nullptr;
    int32_t rc = alloc_zero(sim, &hist_dev, 256);
    if (rc) return rc;
    CK(launch_delay_hist(d.delay, sim->Epad, hist_dev, sim->n_sm, sim->stream));
    unsigned long long hist[256];
    CK(cudaStreamSynchronize(sim->stream));
    CK(cudaMemcpy(hist, hist_dev, sizeof(hist), cudaMemcpyDeviceToHost));
    const int Dn = std::min(d.D, 32), near_lim = std::max(Dn - 3, 0);
    double e_near = 0.0, e_far = 0.0;
    for (int dl = 1; dl < 256; ++dl) ((dl + d.bin_steps - 1 <= near_lim) ? e_near : e_far) += (double)hist[dl];
    // target windows: one ring slot (16 B per neuron) is swept window by window, each window small enough to stay in L2
    int W = 1;
    while (W < 4 && 16.0 * (double)d.Npad / W > 48.0 * 1048576.0) W *= 2;
    // one list per (slot, window) and BLOCK of the delivery kernel: a block appends to its own lists through cursors in
    // its shared memory (no global atomics) and reduces them itself when their step comes
    const int P = sim->n_sm * 4;                       // k_deliver_lists: four blocks of 256 threads per SM, all resident
    const int64_t win = ((((int64_t)d.Npad + W - 1) / W + kNeuronPad - 1) / kNeuronPad) * kNeuronPad;
    const uint64_t cur_near = (uint64_t)Dn * W, cur_far = e_far > 0 ? (uint64_t)d.D * W : 0;
    if (cur_near + cur_far > 8192) return DB_OK;       // (cursors of a block live in its shared memory)
    // capacity: the records of one step at the design rate, split over the lists of a slot; any excess spills into the
    // dense ring (exact, only slower).  Halve the design rate until the lists fit into half of the free memory.
    size_t free_b = 0, total_b = 0;
    CK(cudaMemGetInfo(&free_b, &total_b));
    const double dt_s = sim->params.dt_ms * 1e-3;
    uint64_t cap_near = 0, cap_far = 0;
    const uint64_t n_near = cur_near * (uint64_t)P, n_far = cur_far * (uint64_t)P;
    double rate = 60.0;
    for (;; rate *= 0.5) {
        if (rate < 4.0) return DB_OK;                              // no room for useful lists
        auto cap_of = [&](double synapses) {
            const double per_list = synapses * rate * dt_s / (double)(W * P);
            return (uint64_t)std::max(256.0, std::ceil(per_list / 16.0) * 16.0);
        };
        cap_near = cap_of(e_near);
        cap_far = n_far ? cap_of(e_far) : 0;
        if ((double)(n_near * cap_near + n_far * cap_far) * 8.0 <= 0.5 * (double)free_b) break;
    }
    if (cap_near > 0xFFFFFFF0ull || cap_far > 0xFFFFFFF0ull) return DB_OK;
    uint2* rec = nullptr;
    unsigned* cnt = nullptr;
    const size_t n_rec = (size_t)(n_near * cap_near + n_far * cap_far);
    rec = static_cast<uint2*>(dev_alloc(sim, n_rec * sizeof(uint2)));
    if (!rec) return DB_OK;                                        // fall back rather than fail
    if ((rc = alloc_zero(sim, &cnt, (size_t)(cur_near + cur_far) * (size_t)P))) return rc;
    d.ev_direct = 1; d.ev_near_lim = near_lim; d.ev_near_d = std::max(near_lim - (d.bin_steps - 1), 0); d.ev_Dn = Dn; d.ev_D = d.D; d.ev_W = W; d.ev_P = P;
    d.ev_n_cur = (int32_t)(cur_near + cur_far); d.ev_n_far = (int32_t)n_far;
    d.ev_cap_near = (uint32_t)cap_near; d.ev_cap_far = (uint32_t)cap_far;
    for (int k = 0; k < 3; ++k) d.ev_wb[k] = (k + 1 < W) ? (uint32_t)std::min<int64_t>((int64_t)(k + 1) * win, 0x7FFFFFFF) : 0xFFFFFFFFu;
    d.ev_rec = rec; d.ev_cnt = cnt;
    sim->list_rate_hz = rate;
    uint32_t* seg = nullptr;
    if ((rc = alloc_zero(sim, &seg, (size_t)N * (size_t)(d.ev_near_d * W + 1)))) return rc;
    d.seg = seg;

    // sort the rows
    std::vector<int64_t> rb((size_t)N);
    std::vector<int32_t> rl((size_t)N);
    CK(cudaMemcpy(rb.data(), d.row_begin, (size_t)N * 8, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(rl.data(), d.row_len, (size_t)N * 4, cudaMemcpyDeviceToHost));
    auto row_end = [&](int64_t j) { return rb[(size_t)j] + ((int64_t)rl[(size_t)j] + kRowAlign - 1) / kRowAlign * kRowAlign; };
    const int64_t batch = std::min<int64_t>(sim->Epad, (int64_t)1 << 28);        // synapses per batch
    const size_t wsz = d.w_fp16 ? 2 : 4;
    uint32_t* t_s = nullptr; uint8_t* d_s = nullptr; void* w_s = nullptr;
    if (cudaMalloc(&t_s, (size_t)batch * 4) != cudaSuccess || cudaMalloc(&d_s, (size_t)batch) != cudaSuccess ||
        cudaMalloc(&w_s, (size_t)batch * wsz) != cudaSuccess) {
        cudaFree(t_s); cudaFree(d_s); cudaFree(w_s);
        cudaGetLastError();
        return fail(sim, DB_ENOMEM, "no device memory for the row-sorting scratch arrays");
    }
    int32_t out = DB_OK;
    for (int64_t r0 = 0; r0 < N && out == DB_OK;) {
        const int64_t s0 = rb[(size_t)r0];
        int64_t r1 = r0 + 1;
        while (r1 < N && row_end(r1) - s0 <= batch) ++r1;
        const int64_t s1 = row_end(r1 - 1);
        if (s1 - s0 > batch) { out = fail(sim, DB_EINVAL, "a row is longer than the sorting batch"); break; }
        cudaError_t e = launch_sort_rows(d, sim->n_sm, r0, r1, s0, t_s, w_s, d_s, seg, sim->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(const_cast<uint32_t*>(d.tgt_rec) + s0, t_s, (size_t)(s1 - s0) * 4, cudaMemcpyDeviceToDevice, sim->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(const_cast<uint8_t*>(d.delay) + s0, d_s, (size_t)(s1 - s0), cudaMemcpyDeviceToDevice, sim->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync((char*)const_cast<void*>(d.w) + (size_t)s0 * wsz, w_s, (size_t)(s1 - s0) * wsz, cudaMemcpyDeviceToDevice, sim->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(sim->stream);
        if (e != cudaSuccess) out = fail(sim, DB_ECUDA, std::string("row sorting: ") + cudaGetErrorString(e));
        r0 = r1;
    }
    cudaFree(t_s); cudaFree(d_s); cudaFree(w_s);
    if (out) return out;
    d.ev_on = 1;
    sim->deliver_grid = sim->n_sm * 4;      // k_deliver_lists: four blocks of 256 threads per SM, all resident
    *ok = true;
    return DB_OK;
}

// After the CSR is on the device: work list, execution mode, initial state.
int32_t finish_setup(db_sim* sim, uint64_t work_cap, uint64_t heavy_chunks) {
    SimDev& d = sim->dev;
    int32_t rc;
    sim->work_cap = std::max<uint64_t>(work_cap, 1);
    d.work_half = sim->work_cap;
    if ((rc = alloc_zero(sim, &d.work, 2 * (size_t)sim->work_cap))) return rc;
    sim->heavy = heavy_chunks > 0;
    CK(launch_init_state(d, sim->ntype_dev, sim->iext_tab_dev, sim->stream));
    sim->deliver_grid = sim->n_sm * 8;
    sim->update_sm = sim->n_sm;
    int coop = 0;
    CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, sim->device));
    bool fits = false;
    CK(prepare_kernels());              // function attributes and the memory pool belong to the device: once per handle
    CK(raster_pool_setup(sim->device));
    CK(persistent_fits(d, sim->heavy, sim->n_sm, &fits));
    int mode = sim->params.exec_mode;
    // AUTO: the persistent kernel wins while the update dominates the step; with long rows (mean
    // out-degree >= 400: configs 3 and 4) the step is delivery-bound and the two-kernel mode, where every
    // warp of the grid pushes rows, is faster (measured: profiles/)
    const bool delivery_bound = sim->heavy || (sim->E >= 400 * (int64_t)d.N);
    if (mode == DB_EXEC_AUTO)
        mode = (coop && fits && !delivery_bound) ? DB_EXEC_PERSISTENT : DB_EXEC_KERNELS_DEFERRED;
    if (mode == DB_EXEC_KERNELS_DEFERRED) {
        bool ok = false;
        int32_t rc2 = build_arrival_lists(sim, &ok);
        if (rc2) return rc2;
        if (!ok) mode = DB_EXEC_KERNELS;            // nothing to list (no delay beyond 1), or no memory for the lists
    }
    if (mode == DB_EXEC_PERSISTENT && (!coop || !fits))
        return fail(sim, DB_ECUDA, "cooperative launch not available for the persistent mode");
    sim->exec_mode = mode;
    CK(cudaStreamSynchronize(sim->stream));
    return DB_OK;
}

// One step on `st` (no overlap): update, delivery.  List mode: the update kernel is a unit (k_update_stream): `first`
// marks the first step of a db_step call (A only).
cudaError_t launch_step(db_sim* sim, bool first, cudaStream_t st) {
    const int mode = sim->dev.ev_on ? (first ? 1 : 2) : 0;
    cudaError_t e = launch_update(sim->dev, sim->update_sm, mode, st);
    if (e == cudaSuccess) e = launch_deliver(sim->dev, sim->deliver_grid, (unsigned)(sim->host_step & 1ull), st);
    sim->launches += 2;
    sim->host_step += 1;
    return e;
}

// A CUDA graph of 32 steps (an even number: it is replayed from even steps only, so the parity of a step inside it is
// fixed).  In list mode the delivery kernel of step s runs on a second branch, beside the update kernel of step s + 1;
// the update kernel of step s + 2 waits for it.
int32_t build_graph(db_sim* sim) {
    const int steps = 32;
    const bool fork = sim->dev.ev_on != 0;
    const int mode = fork ? 2 : 0;
    cudaGraph_t graph = nullptr;
    cudaStream_t cap = nullptr, side = nullptr;
    std::vector<cudaEvent_t> ev;
    auto cleanup = [&]() {
        for (cudaEvent_t x : ev) cudaEventDestroy(x);
        if (side) cudaStreamDestroy(side);
        if (cap) cudaStreamDestroy(cap);
    };
    int prio_lo = 0, prio_hi = 0;                       // the update kernels get the SMs first; the delivery kernels fill in
    CK(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    CK(cudaStreamCreateWithPriority(&cap, cudaStreamNonBlocking, prio_hi));
    if (fork) {
        if (cudaStreamCreateWithPriority(&side, cudaStreamNonBlocking, prio_lo) != cudaSuccess) { cleanup(); return fail(sim, DB_ECUDA, "stream creation failed"); }
        ev.resize(2 * (size_t)steps);
        for (auto& x : ev) if (cudaEventCreateWithFlags(&x, cudaEventDisableTiming) != cudaSuccess) { cleanup(); return fail(sim, DB_ECUDA, "event creation failed"); }
    }
    cudaError_t le = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (le != cudaSuccess) { cleanup(); return fail(sim, DB_ECUDA, std::string("graph capture: ") + cudaGetErrorString(le)); }
    for (int s = 0; s < steps && le == cudaSuccess; ++s) {
        if (fork) {
            if (s >= 2) le = cudaStreamWaitEvent(cap, ev[2 * (size_t)(s - 2) + 1], 0);                  // delivery of step s - 2 done
            if (le == cudaSuccess) le = launch_update(sim->dev, sim->update_sm, mode, cap);
            if (le == cudaSuccess) le = cudaEventRecord(ev[2 * (size_t)s], cap);                       // update kernel of step s done
            if (le == cudaSuccess) le = cudaStreamWaitEvent(side, ev[2 * (size_t)s], 0);
            if (le == cudaSuccess) le = launch_deliver(sim->dev, sim->deliver_grid, (unsigned)(s & 1), side);
            if (le == cudaSuccess) le = cudaEventRecord(ev[2 * (size_t)s + 1], side);
        } else {
            le = launch_update(sim->dev, sim->update_sm, mode, cap);
            if (le == cudaSuccess) le = launch_deliver(sim->dev, sim->deliver_grid, (unsigned)(s & 1), cap);
        }
    }
    if (fork && le == cudaSuccess) le = cudaStreamWaitEvent(cap, ev[2 * (size_t)steps - 1], 0);        // join (the side branch is in order)
    cudaError_t e = cudaStreamEndCapture(cap, &graph);
    if (le != cudaSuccess || e != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        cleanup();
        cudaGetLastError();
        return fail(sim, DB_ECUDA, std::string("graph capture: ") + cudaGetErrorString(le != cudaSuccess ? le : e));
    }
    e = cudaGraphInstantiate(&sim->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    cleanup();
    if (e != cudaSuccess) return fail(sim, DB_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e));
    sim->graph_steps = steps;
    return DB_OK;
}

int32_t read_ctl(db_sim* sim, Ctl* out) {
    CK(cudaStreamSynchronize(sim->stream));
    CK(cudaMemcpy(out, sim->dev.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost));
    return DB_OK;
}

}  // namespace

// ===========================================================================
extern "C" {

const char* db_last_error(const db_sim* sim) { return sim ? sim->err.c_str() : g_create_error.c_str(); }

int32_t db_create_from_csr(const db_sim_params* sp, const db_csr_view* csr, const db_runtime* rt, db_sim** out) {
    if (!out) return fail(nullptr, DB_EINVAL, "out is NULL");
    *out = nullptr;
    if (!csr || !csr->row_ptr || !csr->ntype || !csr->region_start) return fail(nullptr, DB_EINVAL, "csr is incomplete");
    if (csr->N < 1 || csr->N >= (1ll << 30)) return fail(nullptr, DB_EINVAL, "N must be within 1..2^30-1");
    if (csr->E < 0) return fail(nullptr, DB_EINVAL, "E must be >= 0");
    if (csr->n_regions < 1 || csr->n_regions > 65536) return fail(nullptr, DB_EINVAL, "n_regions must be 1..65536");
    db_sim* sim = new (std::nothrow) db_sim();
    if (!sim) return fail(nullptr, DB_ENOMEM, "host allocation failed");
    auto bail = [&](int32_t rc) { g_create_error = sim->err; dev_free_all(sim); delete sim; return rc; };
    int32_t rc;
    if ((rc = check_sim_params(sim, sp))) return bail(rc);
    if ((rc = open_device(sim, rt))) return bail(rc);
    const int64_t N = csr->N, E = csr->E;
    if (csr->row_ptr[0] != 0 || csr->row_ptr[N] != E) return bail(fail(sim, DB_EINVAL, "row_ptr must run from 0 to E"));
    if (E > 0 && (!csr->tgt || !csr->w || !csr->delay || !csr->rec)) return bail(fail(sim, DB_EINVAL, "csr arrays missing"));
    for (int64_t j = 0; j < N; ++j)                     // before any array is walked up to E
        if (csr->row_ptr[j + 1] < csr->row_ptr[j]) return bail(fail(sim, DB_EINVAL, "row_ptr must be non-decreasing"));
    int32_t max_delay = 0;
    for (int64_t e = 0; e < E; ++e) max_delay = std::max<int32_t>(max_delay, csr->delay[e]);
    if (max_delay >= sp->D) return bail(fail(sim, DB_EINVAL, "delay must satisfy 1 <= delay < D"));
    int32_t min_delay = 255;
    for (int64_t e = 0; e < E; ++e) min_delay = std::min<int32_t>(min_delay, csr->delay[e]);
    if ((rc = setup_common(sim, sp, N, csr->n_regions, csr->region_start, max_delay, csr->own_first, csr->own_count))) return bail(rc);
    sim->max_delay = max_delay;
    sim->min_delay = E > 0 ? min_delay : 1;
    const int64_t own0 = sim->dev.id0, own1 = own0 + sim->dev.N;     // keep the synapses onto [own0, own1)
    SimDev& d = sim->dev;

    // padded row layout + validation
    std::vector<int64_t> row_begin((size_t)N);
    std::vector<int32_t> row_len((size_t)N);
    int64_t pos = 0;
    uint64_t work_cap = 0, heavy_chunks = 0;
    int64_t E_own = 0;
    for (int64_t j = 0; j < N; ++j) {
        int64_t len = csr->row_ptr[j + 1] - csr->row_ptr[j];
        if (len < 0 || len > 0x7FFFFFFF) return bail(fail(sim, DB_EINVAL, "row_ptr must be non-decreasing"));
        if (csr->ntype[j] >= sp->n_types) return bail(fail(sim, DB_EINVAL, "ntype out of range"));
        if (own1 - own0 != N) {                          // only the synapses onto the owned neurons stay in the row
            len = 0;
            for (int64_t s = csr->row_ptr[j]; s < csr->row_ptr[j + 1]; ++s) len += (csr->tgt[s] >= own0 && csr->tgt[s] < own1);
        }
        E_own += len;
        row_begin[(size_t)j] = pos; row_len[(size_t)j] = (int32_t)len;
        pos += (len + kRowAlign - 1) / kRowAlign * kRowAlign;
        work_cap += (uint64_t)((len + kChunk - 1) / kChunk);
        if (len > kInlineMax) heavy_chunks += (uint64_t)((len + kChunk - 1) / kChunk);
    }
    const int64_t Epad = pos + kRowAlign;
    sim->E = E_own; sim->Epad = Epad;
    std::vector<uint32_t> tr((size_t)Epad, 0u);
    std::vector<uint8_t> dl((size_t)Epad, 1);
    std::vector<float> wf;
    std::vector<__half> wh;
    if (csr->weight_fp16) wh.assign((size_t)Epad, __float2half(0.0f)); else wf.assign((size_t)Epad, 0.0f);
    for (int64_t j = 0; j < N; ++j) {
        int64_t o = row_begin[(size_t)j];
        for (int64_t s = csr->row_ptr[j]; s < csr->row_ptr[j + 1]; ++s) {
            if (csr->tgt[s] < 0 || csr->tgt[s] >= N) return bail(fail(sim, DB_EINVAL, "target out of range"));
            if (csr->rec[s] > 3) return bail(fail(sim, DB_EINVAL, "receptor out of range"));
            if (csr->delay[s] < 1 || csr->delay[s] >= sp->D) return bail(fail(sim, DB_EINVAL, "delay must satisfy 1 <= delay < D"));
            if (csr->tgt[s] < own0 || csr->tgt[s] >= own1) continue;
            tr[(size_t)o] = ((uint32_t)csr->rec[s] << 30) | (uint32_t)(csr->tgt[s] - own0);      // targets are local
            dl[(size_t)o] = csr->delay[s];
            if (csr->weight_fp16) wh[(size_t)o] = __float2half_rn(csr->w[s]); else wf[(size_t)o] = csr->w[s];
            ++o;
        }
    }
    int64_t* rb_dev; int32_t* rl_dev; uint32_t* tr_dev; uint8_t* dl_dev; void* w_dev;
    if ((rc = alloc_zero(sim, &rb_dev, (size_t)N))) return bail(rc);
    if ((rc = alloc_zero(sim, &rl_dev, (size_t)N))) return bail(rc);
    if ((rc = alloc_zero(sim, &tr_dev, (size_t)Epad))) return bail(rc);
    if ((rc = alloc_zero(sim, &dl_dev, (size_t)Epad))) return bail(rc);
    const size_t wbytes = (size_t)Epad * (csr->weight_fp16 ? 2 : 4);
    uint8_t* wraw;
    if ((rc = alloc_zero(sim, &wraw, wbytes))) return bail(rc);
    w_dev = wraw;
    auto up = [&](void* dst, const void* src, size_t bytes) {
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, sim->stream);
    };
    if (up(rb_dev, row_begin.data(), (size_t)N * 8) != cudaSuccess || up(rl_dev, row_len.data(), (size_t)N * 4) != cudaSuccess ||
        up(tr_dev, tr.data(), (size_t)Epad * 4) != cudaSuccess || up(dl_dev, dl.data(), (size_t)Epad) != cudaSuccess ||
        up(w_dev, csr->weight_fp16 ? (const void*)wh.data() : (const void*)wf.data(), wbytes) != cudaSuccess ||
        up(sim->ntype_dev, csr->ntype + own0, (size_t)(own1 - own0)) != cudaSuccess || cudaStreamSynchronize(sim->stream) != cudaSuccess)
        return bail(fail(sim, DB_ECUDA, std::string("CSR upload: ") + cudaGetErrorString(cudaGetLastError())));
    d.row_begin = rb_dev; d.row_len = rl_dev; d.tgt_rec = tr_dev; d.delay = dl_dev; d.w = w_dev;
    d.w_fp16 = csr->weight_fp16 ? 1 : 0;
    if ((rc = finish_setup(sim, work_cap, heavy_chunks))) return bail(rc);
    *out = sim;
    return DB_OK;
}

int32_t db_create(const db_network_spec* spec, uint64_t seed, db_sim** out) {
    if (!out) return fail(nullptr, DB_EINVAL, "out is NULL");
    *out = nullptr;
    if (!spec || spec->struct_size != sizeof(db_network_spec)) return fail(nullptr, DB_EINVAL, "db_network_spec.struct_size mismatch");
    db_sim* sim = new (std::nothrow) db_sim();
    if (!sim) return fail(nullptr, DB_ENOMEM, "host allocation failed");
    auto bail = [&](int32_t rc) { g_create_error = sim->err; dev_free_all(sim); delete sim; return rc; };
    int32_t rc;
    if ((rc = check_sim_params(sim, &spec->sim))) return bail(rc);
    if ((rc = open_device(sim, spec->runtime))) return bail(rc);

    GenHostTables tabs;
    std::string gerr;
    if (!gen_host_tables(*spec, seed, &tabs, &gerr)) return bail(fail(sim, DB_EINVAL, gerr));
    int32_t max_delay = spec->delay_intra_max;
    if (tabs.K_inter > 0) max_delay = std::max(max_delay, spec->delay_inter_max);
    if (max_delay >= spec->sim.D) return bail(fail(sim, DB_EINVAL, "delays must be < D"));
    if (spec->own_count != 0 && spec->mode != DB_MODE_FIXED_INDEGREE)
        return bail(fail(sim, DB_EINVAL, "a handle that owns part of the network needs DB_MODE_FIXED_INDEGREE (synapses are drawn per target)"));
    if ((rc = setup_common(sim, &spec->sim, spec->N, spec->n_regions, tabs.region_start.data(), max_delay, spec->own_first, spec->own_count))) return bail(rc);
    sim->min_delay = tabs.K_inter > 0 ? std::min(spec->delay_intra_min, spec->delay_inter_min) : spec->delay_intra_min;

    GenAlloc ga;
    ga.user = sim;
    ga.alloc = [](void* u, size_t bytes) { return dev_alloc(static_cast<db_sim*>(u), bytes); };
    GenResult gr;
    cudaError_t ce = generate_network(*spec, seed, tabs, ga, sim->stream, sim->dev.Npad, sim->ntype_dev, &gr, &gerr);
    if (ce != cudaSuccess) return bail(fail(sim, DB_ECUDA, "generator: " + gerr + " (" + cudaGetErrorString(ce) + ")"));
    if (!gerr.empty()) return bail(fail(sim, gr.oom ? DB_ENOMEM : DB_EINVAL, "generator: " + gerr));
    SimDev& d = sim->dev;
    d.row_begin = gr.row_begin; d.row_len = gr.row_len; d.tgt_rec = gr.tgt_rec; d.delay = gr.delay; d.w = gr.w;
    d.w_fp16 = spec->weight_fp16 ? 1 : 0;
    sim->E = gr.E; sim->Epad = gr.Epad;
    if (gr.max_delay >= spec->sim.D) return bail(fail(sim, DB_EINVAL, "delays must be < D"));
    sim->max_delay = gr.max_delay;
    if ((rc = finish_setup(sim, gr.work_cap, gr.heavy_chunks))) return bail(rc);
    *out = sim;
    return DB_OK;
}

int32_t db_destroy(db_sim* sim) {
    if (!sim) return DB_EINVAL;
    cudaSetDevice(sim->device);
    cudaStreamSynchronize(sim->stream);
    if (sim->graph_exec) cudaGraphExecDestroy(sim->graph_exec);
    for (cudaEvent_t e : sim->prof_events) cudaEventDestroy(e);
    if (sim->xchg_event) cudaEventDestroy(sim->xchg_event);
    dev_free_all(sim);
    delete sim;
    return DB_OK;
}

static int32_t step_batch(db_sim* sim, uint32_t n_steps);

int32_t db_step(db_sim* sim, uint32_t n_steps) {
    if (!sim) return DB_EINVAL;
    if (n_steps == 0) return DB_OK;
    CK(cudaSetDevice(sim->device));
    if (!sim->params.bold.enabled) return step_batch(sim, n_steps);
    for (uint32_t left = n_steps; left;) {          // the BOLD read-out catches up before the count history wraps
        const uint32_t b = std::min(left, sim->bold_batch);
        int32_t rc = step_batch(sim, b);
        if (rc) return rc;
        CK(launch_bold(sim->dev, sim->bold, sim->stream));
        sim->launches += 2;
        left -= b;
    }
    return DB_OK;
}

static int32_t step_batch(db_sim* sim, uint32_t n_steps) {
    if (sim->exec_mode == DB_EXEC_PERSISTENT) {
        const uint32_t cap = 1u << 20;     // keeps the arrival counter of one launch far below 2^32
        for (uint32_t left = n_steps; left;) {
            const uint32_t b = std::min(left, cap);
            CK(launch_persistent(sim->dev, sim->heavy, b, sim->n_sm, sim->stream));
            sim->launches += 1;
            sim->host_step += b;
            left -= b;
        }
        return DB_OK;
    }
    if (!sim->graph_exec && n_steps >= 34) { int32_t rc = build_graph(sim); if (rc) return rc; }
    uint32_t left = n_steps;
    const bool lists = sim->dev.ev_on != 0;
    if (lists) {                                       // unit form: the first kernel of the call has no B part
        CK(launch_step(sim, true, sim->stream));
        left -= 1;
    }
    if (sim->graph_exec && left >= (uint32_t)sim->graph_steps && (sim->host_step & 1ull)) {  // the graph starts on even steps (its launches carry the parity)
        CK(launch_step(sim, false, sim->stream));
        left -= 1;
    }
    while (sim->graph_exec && left >= (uint32_t)sim->graph_steps) {
        CK(cudaGraphLaunch(sim->graph_exec, sim->stream));
        left -= (uint32_t)sim->graph_steps;
        sim->launches += 2ull * (uint64_t)sim->graph_steps;
        sim->host_step += (uint64_t)sim->graph_steps;
    }
    for (; left; --left) CK(launch_step(sim, false, sim->stream));
    if (lists) {                                       // ... and the last one only a B part: the state is complete again
        CK(launch_update(sim->dev, sim->update_sm, 3, sim->stream));
        sim->launches += 1;
    }
    return DB_OK;
}

int32_t db_deliver_external(db_sim* sim, uint64_t step, const int32_t* ids, uint64_t n) {
    if (!sim || (n && !ids)) return DB_EINVAL;
    if (n == 0) return DB_OK;
    CK(cudaSetDevice(sim->device));
    const SimDev& d = sim->dev;
    if (n > 0xFFFFFFFFull) return fail(sim, DB_EINVAL, "too many ids");
    for (uint64_t k = 0; k < n; ++k) {
        if (ids[k] < 0 || ids[k] >= d.n_rows) return fail(sim, DB_EINVAL, "id out of range");
        if (ids[k] >= d.id0 && ids[k] < d.id0 + d.N) return fail(sim, DB_EINVAL, "id is owned by this handle: its spikes are delivered by db_step");
    }
    // the earliest arrival (end of the spike's time bin + smallest delay) must not be consumed yet
    const uint64_t b = (uint64_t)d.bin_steps, nt = step - step % b + (b - 1);
    if (nt + (uint64_t)sim->min_delay < sim->host_step) return fail(sim, DB_ERANGE, "too late: the handle has stepped past the arrival of these spikes");
    if (nt + (uint64_t)sim->max_delay >= sim->host_step + (uint64_t)d.D - 2) return fail(sim, DB_ERANGE, "too early: the arrivals lie beyond the ring");
    if (n > sim->ext_ids_cap) {
        const uint64_t cap = std::max<uint64_t>(next_pow2(n), 4096);
        int32_t* buf = static_cast<int32_t*>(dev_alloc(sim, (size_t)cap * 4));     // (the old one is freed with the handle)
        if (!buf) return fail(sim, DB_ENOMEM, "device allocation for the external spike list failed");
        sim->ext_ids_dev = buf; sim->ext_ids_cap = cap;
    }
    CK(cudaMemcpyAsync(sim->ext_ids_dev, ids, (size_t)n * 4, cudaMemcpyHostToDevice, sim->stream));
    CK(cudaStreamSynchronize(sim->stream));            // `ids` is the caller's pageable memory
    CK(launch_deliver_external(d, sim->n_sm, sim->ext_ids_dev, (unsigned)n, (unsigned long long)step, sim->stream));
    sim->launches += 1;
    return DB_OK;
}

}  // extern "C" (interrupted for the device side of db_deliver_external_static; resumed below)

// ---------------------------------------------------------------------------------------------------------------------
// db_deliver_external_static: the entry point that allocates nothing (callers under CUDA graph capture, serving loops
// and harnesses that forbid cudaMalloc).  db_deliver_external keeps the device copy of the id list in a buffer it
// (re)allocates when the list grows; here that scratch is a file-scope array of DB_EXTERNAL_STATIC_MAX ids (256 KB),
// held by every GPU that loads the library until the process exits.  In HOST code the name `g_ext_ids_static` is a
// host-side stand-in, not a device address: the kernel is given the address cudaGetSymbolAddress returns on the
// handle's device (static_ext_ids below, once per device, with that device current).  Every call on a device shares
// the array, which keeps the last call's list: each call overwrites the entries it reads (nothing has to start at
// zero), and two calls that overlap on the GPU -- different handles on different streams of one device -- race.
// ---------------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) int32_t g_ext_ids_static[DB_EXTERNAL_STATIC_MAX];

namespace {

// Variant of k_deliver_external (db_step.cu) whose id list lives in the static array: one warp per outside spike, one
// synapse per lane and pass.  Same integer reductions into the same ring cells as the existing kernel (their order
// does not matter), same event count.  SI Eq.(6) second sum.
__global__ void __launch_bounds__(256) k_deliver_external_static(const __grid_constant__ SimDev p, const int32_t* __restrict__ ids,
                                                                 const unsigned n_ids, const unsigned long long step) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const unsigned long long b = (unsigned long long)p.bin_steps;
    const unsigned nto = (unsigned)(p.bin_steps == 1 ? step : step - step % b + (b - 1ull));   // end of the spike's time bin (R29)
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    unsigned long long ev = 0ull;
    for (unsigned q = warp; q < n_ids; q += n_warps) {
        const int j = ids[q];
        const int64_t rb = __ldg(p.row_begin + j);
        const int len = __ldg(p.row_len + j);
        for (int e = (int)lane; e < len; e += 32) {
            const uint32_t tr = __ldg(p.tgt_rec + rb + e);
            const unsigned dl = __ldg(p.delay + rb + e);
            const float w = p.w_fp16 ? __half2float(__ldg(static_cast<const __half*>(p.w) + rb + e))
                                     : __ldg(static_cast<const float*>(p.w) + rb + e);
            const int wq = __float2int_rn(__fmul_rn(w, p.wscale));
            int32_t* cell = p.ring + ((size_t)((nto + dl) & Dm) * 4 + (tr >> 30)) * Np + (tr & 0x3FFFFFFFu);
            asm volatile("red.global.add.s32 [%0], %1;" :: "l"(cell), "r"(wq) : "memory");
        }
        ev += (unsigned long long)len;
    }
    if (lane == 0 && ev) atomicAdd(&p.ctl->events, ev);
}

// db_deliver_external_window: the lists of several consecutive time steps in one launch.  ids[offs[s] .. offs[s + 1])
// fired in step `step` + s; a warp finds the step of its spike by bisection in the (n_steps + 1) offsets.
__global__ void __launch_bounds__(256) k_deliver_external_window(const __grid_constant__ SimDev p, const int32_t* __restrict__ ids,
                                                                 const unsigned* __restrict__ offs, const unsigned n_steps,
                                                                 const unsigned long long step) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const unsigned n_ids = __ldg(offs + n_steps);
    const unsigned long long b = (unsigned long long)p.bin_steps;
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    unsigned long long ev = 0ull;
    for (unsigned q = warp; q < n_ids; q += n_warps) {
        unsigned lo = 0u, hi = n_steps;                    // largest s with offs[s] <= q
        while (hi - lo > 1u) {
            const unsigned mid = (lo + hi) >> 1;
            if (__ldg(offs + mid) <= q) lo = mid; else hi = mid;
        }
        const unsigned long long n = step + lo;
        const unsigned nto = (unsigned)(p.bin_steps == 1 ? n : n - n % b + (b - 1ull));
        const int j = __ldg(ids + q);
        const int64_t rb = __ldg(p.row_begin + j);
        const int len = __ldg(p.row_len + j);
        for (int e = (int)lane; e < len; e += 32) {
            const uint32_t tr = __ldg(p.tgt_rec + rb + e);
            const unsigned dl = __ldg(p.delay + rb + e);
            const float w = p.w_fp16 ? __half2float(__ldg(static_cast<const __half*>(p.w) + rb + e))
                                     : __ldg(static_cast<const float*>(p.w) + rb + e);
            const int wq = __float2int_rn(__fmul_rn(w, p.wscale));
            int32_t* cell = p.ring + ((size_t)((nto + dl) & Dm) * 4 + (tr >> 30)) * Np + (tr & 0x3FFFFFFFu);
            asm volatile("red.global.add.s32 [%0], %1;" :: "l"(cell), "r"(wq) : "memory");
        }
        ev += (unsigned long long)len;
    }
    if (lane == 0 && ev) atomicAdd(&p.ctl->events, ev);
}

// db_exchange_peer: the exchange step of a sharded run without the host in the data path.  The handle `p` pushes the
// rows of the spikes ANOTHER handle logged in its raster ring (device memory of this GPU, or of a peer GPU mapped over
// NVLink) for the steps [lo, lo + span): raster positions [scan_begin, scan_begin + m), entries of other steps are
// skipped by their tag.  32 entries per warp and pass (one coalesced read of ids and tags), then the warp pushes the
// matching rows one after the other.  Order does not matter (integer reductions): no sort, no list, no copy.
__global__ void __launch_bounds__(256) k_deliver_from_raster(const __grid_constant__ SimDev p, const int32_t* src_ids,
                                                             const uint32_t* src_tag, const unsigned long long src_mask,
                                                             const unsigned long long* src_step_end, const unsigned src_log_mask,
                                                             const unsigned long long step_begin, const unsigned span,
                                                             const unsigned long long last_log) {
    // the entries of step u lie somewhere in the raster positions [S(u - 2), S(u + 1)), S = the source's step log
    const unsigned long long scan_begin = step_begin >= 2ull ? src_step_end[(step_begin - 2ull) & src_log_mask] : 0ull;
    const unsigned long long m = src_step_end[last_log & src_log_mask] - scan_begin;
    const unsigned lo = (unsigned)step_begin;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned long long warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned long long n_warps = (gridDim.x * blockDim.x) >> 5;
    const unsigned long long b = (unsigned long long)p.bin_steps;
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    unsigned long long ev = 0ull;
    // entries per warp and pass: 32 when there is plenty of work, fewer when the range is short (a warp pushes its rows
    // one after the other, so a short range is spread over all warps of the grid)
    const unsigned per = (unsigned)min(32ull, max(1ull, (m + n_warps - 1ull) / n_warps));
    for (unsigned long long base = warp * per; base < m; base += n_warps * per) {
        int my_id = 0;
        unsigned my_rel = 0xFFFFFFFFu;
        if (lane < per && base + lane < m) {
            const unsigned long long at = (scan_begin + base + lane) & src_mask;
            my_rel = src_tag[at] - lo;
            my_id = src_ids[at];
        }
        unsigned todo = __ballot_sync(0xffffffffu, my_rel < span);
        while (todo) {
            const int src_lane = __ffs((int)todo) - 1;
            todo &= todo - 1u;
            const int j = __shfl_sync(0xffffffffu, my_id, src_lane);
            const unsigned long long n = step_begin + __shfl_sync(0xffffffffu, my_rel, src_lane);
            const unsigned nto = (unsigned)(p.bin_steps == 1 ? n : n - n % b + (b - 1ull));
            const int64_t rb = __ldg(p.row_begin + j);
            const int len = __ldg(p.row_len + j);
            for (int e = (int)lane; e < len; e += 32) {
                const uint32_t tr = __ldg(p.tgt_rec + rb + e);
                const unsigned dl = __ldg(p.delay + rb + e);
                const float w = p.w_fp16 ? __half2float(__ldg(static_cast<const __half*>(p.w) + rb + e))
                                         : __ldg(static_cast<const float*>(p.w) + rb + e);
                const int wq = __float2int_rn(__fmul_rn(w, p.wscale));
                int32_t* cell = p.ring + ((size_t)((nto + dl) & Dm) * 4 + (tr >> 30)) * Np + (tr & 0x3FFFFFFFu);
                asm volatile("red.global.add.s32 [%0], %1;" :: "l"(cell), "r"(wq) : "memory");
            }
            ev += (unsigned long long)len;
        }
    }
    if (lane == 0 && ev) atomicAdd(&p.ctl->events, ev);
}

// db_write_state(DB_FIELD_REF): the refractory counter of neuron i goes into the low bits of rt[i]; the type bits stay.
__global__ void __launch_bounds__(256) k_write_ref(uint16_t* __restrict__ rt, const int32_t* __restrict__ ref, const int64_t count) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x)
        rt[i] = (uint16_t)((rt[i] & ~kRefMask) | ref[i]);
}

constexpr int kMaxStaticDevices = 64;
int32_t* g_ext_ids_static_addr[kMaxStaticDevices] = {};     // device address of g_ext_ids_static, per device ordinal

// Set-up, once per device, with that device current: the device address of the static array.
cudaError_t static_ext_ids(int device, int32_t** out) {
    if (device < 0 || device >= kMaxStaticDevices) return cudaErrorInvalidDevice;
    if (!g_ext_ids_static_addr[device]) {
        int32_t* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_ext_ids_static);
        if (e != cudaSuccess) return e;
        g_ext_ids_static_addr[device] = ptr;                // (racing first calls store the same value)
    }
    *out = g_ext_ids_static_addr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" {

int32_t db_deliver_external_static(db_sim* sim, uint64_t step, const int32_t* ids, uint64_t n) {
    if (!sim || (n && !ids)) return DB_EINVAL;
    if (n > (uint64_t)DB_EXTERNAL_STATIC_MAX)
        return fail(sim, DB_EINVAL, "db_deliver_external_static: more than DB_EXTERNAL_STATIC_MAX (65536) ids in one call; "
                                    "split the list or use db_deliver_external");
    if (n == 0) return DB_OK;
    CK(cudaSetDevice(sim->device));
    const SimDev& d = sim->dev;
    for (uint64_t k = 0; k < n; ++k) {
        if (ids[k] < 0 || ids[k] >= d.n_rows) return fail(sim, DB_EINVAL, "id out of range");
        if (ids[k] >= d.id0 && ids[k] < d.id0 + d.N) return fail(sim, DB_EINVAL, "id is owned by this handle: its spikes are delivered by db_step");
    }
    const uint64_t b = (uint64_t)d.bin_steps, nt = step - step % b + (b - 1);
    if (nt + (uint64_t)sim->min_delay < sim->host_step) return fail(sim, DB_ERANGE, "too late: the handle has stepped past the arrival of these spikes");
    if (nt + (uint64_t)sim->max_delay >= sim->host_step + (uint64_t)d.D - 2) return fail(sim, DB_ERANGE, "too early: the arrivals lie beyond the ring");
    int32_t* scratch = nullptr;
    CK(static_ext_ids(sim->device, &scratch));
    CK(cudaMemcpyAsync(scratch, ids, (size_t)n * 4, cudaMemcpyHostToDevice, sim->stream));
    CK(cudaStreamSynchronize(sim->stream));            // `ids` is the caller's pageable memory
    const unsigned grid = std::min<unsigned>(((unsigned)n + 7u) / 8u, (unsigned)sim->n_sm * 8u);
    k_deliver_external_static<<<grid, 256, 0, sim->stream>>>(d, scratch, (unsigned)n, (unsigned long long)step);
    CK(cudaGetLastError());
    sim->launches += 1;
    return DB_OK;
}

int32_t db_deliver_external_window(db_sim* sim, uint64_t step_begin, uint32_t n_steps, const uint64_t* offsets, const int32_t* ids) {
    if (!sim || !offsets || n_steps == 0 || n_steps > 4096) return DB_EINVAL;
    const uint64_t n = offsets[n_steps];
    if (offsets[0] != 0 || (n && !ids)) return fail(sim, DB_EINVAL, "offsets must start at 0");
    if (n > 0xFFFFFFF0ull) return fail(sim, DB_EINVAL, "too many ids");
    for (uint32_t s = 0; s < n_steps; ++s)
        if (offsets[s + 1] < offsets[s]) return fail(sim, DB_EINVAL, "offsets must not decrease");
    if (n == 0) return DB_OK;
    CK(cudaSetDevice(sim->device));
    const SimDev& d = sim->dev;
    for (uint64_t k = 0; k < n; ++k) {
        if (ids[k] < 0 || ids[k] >= d.n_rows) return fail(sim, DB_EINVAL, "id out of range");
        if (ids[k] >= d.id0 && ids[k] < d.id0 + d.N) return fail(sim, DB_EINVAL, "id is owned by this handle: its spikes are delivered by db_step");
    }
    uint32_t s_first = 0, s_last = n_steps - 1;        // first and last step of the window that carry spikes
    while (offsets[s_first + 1] == 0) ++s_first;
    while (offsets[s_last] == n) --s_last;
    const uint64_t b = (uint64_t)d.bin_steps;
    const uint64_t n_lo = step_begin + s_first, n_hi = step_begin + s_last;
    const uint64_t nt_lo = n_lo - n_lo % b + (b - 1), nt_hi = n_hi - n_hi % b + (b - 1);
    if (nt_lo + (uint64_t)sim->min_delay < sim->host_step) return fail(sim, DB_ERANGE, "too late: the handle has stepped past the arrival of these spikes");
    if (nt_hi + (uint64_t)sim->max_delay >= sim->host_step + (uint64_t)d.D - 2) return fail(sim, DB_ERANGE, "too early: the arrivals lie beyond the ring");
    const uint64_t need = n + (uint64_t)n_steps + 1;   // [ids | offsets as u32]
    if (need > sim->ext_ids_cap) {
        const uint64_t cap = std::max<uint64_t>(next_pow2(need), 4096);
        int32_t* buf = static_cast<int32_t*>(dev_alloc(sim, (size_t)cap * 4));     // (the old one is freed with the handle)
        if (!buf) return fail(sim, DB_ENOMEM, "device allocation for the external spike list failed");
        sim->ext_ids_dev = buf; sim->ext_ids_cap = cap;
    }
    uint32_t offs32[4097];
    for (uint32_t s = 0; s <= n_steps; ++s) offs32[s] = (uint32_t)offsets[s];
    unsigned* offs_dev = reinterpret_cast<unsigned*>(sim->ext_ids_dev + n);
    CK(cudaMemcpyAsync(sim->ext_ids_dev, ids, (size_t)n * 4, cudaMemcpyHostToDevice, sim->stream));
    CK(cudaMemcpyAsync(offs_dev, offs32, ((size_t)n_steps + 1) * 4, cudaMemcpyHostToDevice, sim->stream));
    CK(cudaStreamSynchronize(sim->stream));            // `ids` and offs32 are pageable host memory
    const unsigned grid = std::min<unsigned>(((unsigned)n + 7u) / 8u, (unsigned)sim->n_sm * 8u);
    k_deliver_external_window<<<grid, 256, 0, sim->stream>>>(d, sim->ext_ids_dev, offs_dev, n_steps, (unsigned long long)step_begin);
    CK(cudaGetLastError());
    sim->launches += 1;
    return DB_OK;
}

int32_t db_exchange_peer(db_sim* sim, db_sim* src, uint64_t step_begin, uint64_t step_end) {
    if (!sim || !src || sim == src) return DB_EINVAL;
    const SimDev& d = sim->dev;
    const SimDev& o = src->dev;
    if (d.n_rows != o.n_rows) return fail(sim, DB_EINVAL, "the two handles are not shards of the same network");
    if (!(o.id0 + o.N <= d.id0 || d.id0 + d.N <= o.id0)) return fail(sim, DB_EINVAL, "the two handles own overlapping neuron ranges");
    if (step_begin > step_end || step_end - step_begin > 0xFFFFFFFFull) return fail(sim, DB_EINVAL, "bad step range");
    if (step_begin == step_end) return DB_OK;
    if (step_end > src->host_step) return fail(sim, DB_ERANGE, "the source has not simulated these steps yet");
    // where the arrivals fall in this handle's ring (as db_deliver_external, for the first and the last step of the range,
    // whether or not they carry spikes)
    const uint64_t b = (uint64_t)d.bin_steps, s_hi = step_end - 1;
    const uint64_t nt_lo = step_begin - step_begin % b + (b - 1), nt_hi = s_hi - s_hi % b + (b - 1);
    if (nt_lo + (uint64_t)sim->min_delay < sim->host_step) return fail(sim, DB_ERANGE, "too late: the handle has stepped past the arrival of these spikes");
    if (nt_hi + (uint64_t)sim->max_delay >= sim->host_step + (uint64_t)d.D - 2) return fail(sim, DB_ERANGE, "too early: the arrivals lie beyond the ring");
    // is the range still in the source's step log and raster ring?
    const uint64_t log_cap = (uint64_t)o.step_log_mask + 1;
    const uint64_t first_log = step_begin >= 2 ? step_begin - 2 : 0;
    const uint64_t last_log = std::min<uint64_t>(step_end, src->host_step - 1);
    if (src->host_step - first_log > log_cap) return fail(sim, DB_ERANGE, "steps older than the source's step log");
    // the source cannot have logged more than (steps since) x (its neurons) spikes since the range began: when even that
    // fits its raster ring nothing has to be read back, and the call neither copies nor waits
    if ((src->host_step - first_log) * (uint64_t)o.N > src->spike_cap) {
        Ctl c;
        if (int32_t rc = read_ctl(src, &c)) return fail(sim, rc, "source handle: " + src->err);
        uint64_t scan_begin = 0;
        if (step_begin >= 2) CK(cudaMemcpy(&scan_begin, o.step_end + ((step_begin - 2) & o.step_log_mask), 8, cudaMemcpyDeviceToHost));
        if (c.spike_begin - scan_begin > src->spike_cap) return fail(sim, DB_ERANGE, "spikes already overwritten in the source's raster ring");
    }
    CK(cudaSetDevice(sim->device));
    if (src->device != sim->device) {                  // the source's raster is read over the NVLink / PCIe peer mapping
        int can = 0;
        CK(cudaDeviceCanAccessPeer(&can, sim->device, src->device));
        if (!can) return fail(sim, DB_ESTATE, "no peer access between the two devices: exchange through db_read_spikes / db_deliver_external_window");
        const cudaError_t e = cudaDeviceEnablePeerAccess(src->device, 0);
        if (e == cudaErrorPeerAccessAlreadyEnabled) (void)cudaGetLastError();
        else if (e != cudaSuccess) return fail(sim, DB_ECUDA, std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e));
    }
    if (src->stream != sim->stream) {                  // the kernel runs after the steps the source has launched so far
        // the event is recorded on the source's stream, so it has to live on the source's device
        if (src->device != sim->device) CK(cudaSetDevice(src->device));
        if (sim->xchg_event && sim->xchg_event_dev != src->device) { cudaEventDestroy(sim->xchg_event); sim->xchg_event = nullptr; }
        if (!sim->xchg_event) {
            CK(cudaEventCreateWithFlags(&sim->xchg_event, cudaEventDisableTiming));
            sim->xchg_event_dev = src->device;
        }
        CK(cudaEventRecord(sim->xchg_event, src->stream));
        if (src->device != sim->device) CK(cudaSetDevice(sim->device));
        CK(cudaStreamWaitEvent(sim->stream, sim->xchg_event, 0));
    }
    k_deliver_from_raster<<<(unsigned)sim->n_sm * 4u, 256, 0, sim->stream>>>(d, o.spike_ids, o.spike_tag, o.spike_mask, o.step_end, o.step_log_mask,
                                                                             (unsigned long long)step_begin, (unsigned)(step_end - step_begin),
                                                                             (unsigned long long)last_log);
    CK(cudaGetLastError());
    sim->launches += 1;
    return DB_OK;
}

int32_t db_step_profiled(db_sim* sim, uint32_t n_steps, db_phase_times* out) {
    if (!sim || !out) return DB_EINVAL;
    CK(cudaSetDevice(sim->device));
    Ctl c0, c1;
    int32_t rc;
    if ((rc = read_ctl(sim, &c0))) return rc;
    std::memset(out, 0, sizeof(*out));
    const uint32_t batch = 256;
    while (sim->prof_events.size() < 2 * batch + 1) {
        cudaEvent_t e; CK(cudaEventCreate(&e)); sim->prof_events.push_back(e);
    }
    uint32_t left = n_steps, since_bold = 0;
    while (left) {
        const uint32_t b = std::min(std::min(left, batch), sim->params.bold.enabled ? std::max(sim->bold_batch, 1u) : batch);
        CK(cudaEventRecord(sim->prof_events[0], sim->stream));
        for (uint32_t s = 0; s < b; ++s) {              // every kernel on the handle's stream, nothing overlapped
            const int mode = sim->dev.ev_on ? (s == 0 ? 1 : 2) : 0;
            CK(launch_update(sim->dev, sim->update_sm, mode, sim->stream));
            CK(cudaEventRecord(sim->prof_events[2 * s + 1], sim->stream));
            CK(launch_deliver(sim->dev, sim->deliver_grid, (unsigned)(sim->host_step & 1ull), sim->stream));
            CK(cudaEventRecord(sim->prof_events[2 * s + 2], sim->stream));
            sim->launches += 2;
            sim->host_step += 1;
        }
        if (sim->dev.ev_on) {                           // (the B part of the batch's last step: not timed)
            CK(launch_update(sim->dev, sim->update_sm, 3, sim->stream));
            sim->launches += 1;
        }
        CK(cudaStreamSynchronize(sim->stream));
        for (uint32_t s = 0; s < b; ++s) {
            float a = 0, d = 0;
            CK(cudaEventElapsedTime(&a, sim->prof_events[2 * s], sim->prof_events[2 * s + 1]));
            CK(cudaEventElapsedTime(&d, sim->prof_events[2 * s + 1], sim->prof_events[2 * s + 2]));
            out->update_ms += a; out->deliver_ms += d;
        }
        float t = 0;
        CK(cudaEventElapsedTime(&t, sim->prof_events[0], sim->prof_events[2 * b]));
        out->total_ms += t;
        left -= b;
        since_bold += b;
        if (sim->params.bold.enabled && (since_bold + batch > sim->bold_batch || left == 0)) {   // before the count history wraps
            CK(launch_bold(sim->dev, sim->bold, sim->stream));
            sim->launches += 2;
            since_bold = 0;
        }
    }
    if ((rc = read_ctl(sim, &c1))) return rc;
    out->steps = c1.step - c0.step; out->spikes = c1.spike_begin - c0.spike_begin; out->events = c1.events - c0.events;
    return DB_OK;
}

int32_t db_synchronize(db_sim* sim) {
    if (!sim) return DB_EINVAL;
    CK(cudaStreamSynchronize(sim->stream));
    return DB_OK;
}

int32_t db_get_counters(db_sim* sim, db_counters* out) {
    if (!sim || !out) return DB_EINVAL;
    Ctl c;
    int32_t rc = read_ctl(sim, &c);
    if (rc) return rc;
    std::vector<unsigned long long> parts(kBgParts);
    CK(cudaMemcpy(parts.data(), sim->dev.bg_parts, kBgParts * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    uint64_t bg = 0;
    for (auto v : parts) bg += v;
    out->steps = c.step; out->spikes = c.spike_begin; out->events = c.events; out->bg_events = bg;
    out->ring_overflow = c.overflow; out->exec_mode = (uint32_t)sim->exec_mode;
    out->launches = sim->launches;
    out->list_spilled = c.ev_spilled;
    return DB_OK;
}

int32_t db_read_spikes(db_sim* sim, uint64_t step_begin, uint64_t step_end, uint64_t* steps, int32_t* ids,
                       uint64_t cap, uint64_t* n_out) {
    if (!sim || !n_out) return DB_EINVAL;
    *n_out = 0;
    Ctl c;
    int32_t rc = read_ctl(sim, &c);
    if (rc) return rc;
    if (step_begin > step_end) return fail(sim, DB_EINVAL, "step_begin > step_end");
    if (step_end > c.step) return fail(sim, DB_ERANGE, "steps not simulated yet");
    if (step_begin == step_end) return DB_OK;
    // step_end[u] = S(u), the number of spikes of the steps <= u.  The raster is written through one
    // cursor by blocks that may be one step apart, so the entries of step u lie somewhere in the
    // positions [S(u-2), S(u+1)) and carry the low 32 bits of their step as a tag.
    if (step_end - step_begin > 0xFFFFFFFFull) return fail(sim, DB_EINVAL, "step range too long");
    const uint64_t log_cap = (uint64_t)sim->dev.step_log_mask + 1;
    const uint64_t first_log = step_begin >= 2 ? step_begin - 2 : 0;            // first log entry needed
    const uint64_t last_log = std::min<uint64_t>(step_end, c.step - 1);          // last one
    if (c.step - first_log > log_cap) return fail(sim, DB_ERANGE, "steps older than the step log");
    const uint64_t n_log = last_log - first_log + 1;
    std::vector<unsigned long long> S((size_t)n_log);
    for (uint64_t k = 0; k < n_log;) {                               // circular copy
        const uint64_t idx = (first_log + k) & sim->dev.step_log_mask;
        const uint64_t run = std::min<uint64_t>(n_log - k, log_cap - idx);
        CK(cudaMemcpy(S.data() + k, sim->dev.step_end + idx, (size_t)run * 8, cudaMemcpyDeviceToHost));
        k += run;
    }
    auto S_of = [&](uint64_t u) { return (uint64_t)S[(size_t)(u - first_log)]; };
    const uint64_t scan_begin = step_begin >= 2 ? S_of(step_begin - 2) : 0ull;
    const uint64_t scan_end = S_of(last_log);
    const uint64_t n = S_of(step_end - 1) - (step_begin ? S_of(step_begin - 1) : 0ull);
    if (c.spike_begin - scan_begin > sim->spike_cap) return fail(sim, DB_ERANGE, "spikes already overwritten in the raster ring");
    *n_out = n;
    if (n == 0 || cap == 0) return DB_OK;
    const uint64_t m = scan_end - scan_begin;
    if (m >= 2048) {                    // long ranges: select, sort and split on the device (db_raster.cu), copy into the caller's arrays
        bool consistent = false;
        CK(raster_sorted_read(sim->dev, sim->n_sm, scan_begin, m, (uint32_t)step_begin, (uint32_t)(step_end - step_begin), n, step_begin,
                              steps, ids, cap, &consistent, sim->stream));
        if (!consistent) return fail(sim, DB_ESTATE, "raster log is inconsistent");
        return DB_OK;
    }
    std::vector<int32_t> id_raw((size_t)m);
    std::vector<uint32_t> tag_raw((size_t)m);
    for (uint64_t k = 0; k < m;) {
        const uint64_t idx = (scan_begin + k) & sim->dev.spike_mask;
        const uint64_t run = std::min<uint64_t>(m - k, sim->spike_cap - idx);
        CK(cudaMemcpy(id_raw.data() + k, sim->dev.spike_ids + idx, (size_t)run * 4, cudaMemcpyDeviceToHost));
        CK(cudaMemcpy(tag_raw.data() + k, sim->dev.spike_tag + idx, (size_t)run * 4, cudaMemcpyDeviceToHost));
        k += run;
    }
    std::vector<std::pair<uint64_t, int32_t>> sel;
    sel.reserve((size_t)n);
    const uint32_t span = (uint32_t)(step_end - step_begin), lo = (uint32_t)step_begin;
    for (uint64_t k = 0; k < m; ++k) {
        const uint32_t rel = tag_raw[(size_t)k] - lo;
        if (rel < span) sel.emplace_back(step_begin + rel, id_raw[(size_t)k]);
    }
    if (sel.size() != n) return fail(sim, DB_ESTATE, "raster log is inconsistent");
    std::sort(sel.begin(), sel.end());
    for (uint64_t o = 0; o < n && o < cap; ++o) {
        if (steps) steps[o] = sel[(size_t)o].first;
        if (ids) ids[o] = sel[(size_t)o].second;
    }
    return DB_OK;
}

int32_t db_read_state(db_sim* sim, uint32_t field, int64_t first, int64_t count, void* dst) {
    if (!sim || !dst) return DB_EINVAL;
    const SimDev& d = sim->dev;
    if (first < d.id0 || count < 0 || first + count > (int64_t)d.id0 + d.N) return fail(sim, DB_ERANGE, "neuron range out of bounds (ids are global; this handle owns [own_first, own_first + own_count))");
    const int64_t first_global = first;
    first -= d.id0;                                    // state and ring are indexed locally
    CK(cudaStreamSynchronize(sim->stream));
    if (count == 0) return DB_OK;
    const size_t Np = (size_t)d.Npad;
    switch (field) {
    case DB_FIELD_V:
        CK(cudaMemcpy(dst, d.V + first, (size_t)count * 4, cudaMemcpyDeviceToHost)); break;
    case DB_FIELD_G_AMPA: case DB_FIELD_G_NMDA: case DB_FIELD_G_GABAA: case DB_FIELD_G_GABAB:
        CK(cudaMemcpy(dst, d.g + (field - DB_FIELD_G_AMPA) * Np + first, (size_t)count * 4, cudaMemcpyDeviceToHost)); break;
    case DB_FIELD_REF: case DB_FIELD_TYPE: {
        std::vector<uint16_t> t((size_t)count);
        CK(cudaMemcpy(t.data(), d.rt + first, (size_t)count * 2, cudaMemcpyDeviceToHost));
        for (int64_t i = 0; i < count; ++i) {
            if (field == DB_FIELD_REF) static_cast<int32_t*>(dst)[i] = t[(size_t)i] & kRefMask;
            else static_cast<uint8_t*>(dst)[i] = (uint8_t)(t[(size_t)i] >> 12);
        }
        break;
    }
    case DB_FIELD_OUTDEG:
        CK(cudaMemcpy(dst, d.row_len + first_global, (size_t)count * 4, cudaMemcpyDeviceToHost)); break;   // rows are keyed by global id
    case DB_FIELD_IOU:
        if (d.ou_on) CK(cudaMemcpy(dst, d.Iou + first, (size_t)count * 4, cudaMemcpyDeviceToHost));
        else std::memset(dst, 0, (size_t)count * 4);
        break;
    case DB_FIELD_IEXT:
        if (d.iext) CK(cudaMemcpy(dst, d.iext + first, (size_t)count * 4, cudaMemcpyDeviceToHost));
        else {                          // no plane: every neuron carries the constant of its type
            std::vector<uint16_t> t((size_t)count);
            CK(cudaMemcpy(t.data(), d.rt + first, (size_t)count * 2, cudaMemcpyDeviceToHost));
            for (int64_t i = 0; i < count; ++i) static_cast<float*>(dst)[i] = d.tc[t[(size_t)i] >> 12].Iext;
        }
        break;
    case DB_FIELD_RING: {
        // API slot j holds the arrivals of the step t in [n, n + D) with t mod D == j; device slot = t mod d.D
        Ctl c;
        int32_t rc = read_ctl(sim, &c);
        if (rc) return rc;
        const int D = sim->params.D;
        std::vector<int32_t> t((size_t)count);
        int32_t* o = static_cast<int32_t*>(dst);
        for (int k = 0; k < D; ++k) {
            const uint64_t step = c.step + (uint64_t)k;
            const size_t s = (size_t)(step % (uint64_t)D), sd = (size_t)(step & (uint64_t)(d.D - 1));
            for (int u = 0; u < 4; ++u) {
                CK(cudaMemcpy(t.data(), d.ring + (sd * 4 + u) * Np + first, (size_t)count * 4, cudaMemcpyDeviceToHost));
                for (int64_t i = 0; i < count; ++i) o[(s * (size_t)count + (size_t)i) * 4 + u] = t[(size_t)i];
            }
        }
        if (d.ev_on) {                 // list mode: plus the records waiting in the arrival lists
            const size_t cells = (size_t)D * (size_t)count * 4;
            int32_t* tmp = nullptr;
            if (cudaMalloc(&tmp, cells * 4) != cudaSuccess) { cudaGetLastError(); return fail(sim, DB_ENOMEM, "no device memory for the ring read-out"); }
            cudaError_t e = cudaMemsetAsync(tmp, 0, cells * 4, sim->stream);
            if (e == cudaSuccess) e = launch_lists_to_ring(d, sim->n_sm, tmp, (int)first, (int)count, D, sim->stream);
            std::vector<int32_t> pend(cells);
            if (e == cudaSuccess) e = cudaStreamSynchronize(sim->stream);
            if (e == cudaSuccess) e = cudaMemcpy(pend.data(), tmp, cells * 4, cudaMemcpyDeviceToHost);
            cudaFree(tmp);
            if (e != cudaSuccess) return fail(sim, DB_ECUDA, std::string("ring read-out: ") + cudaGetErrorString(e));
            for (size_t k = 0; k < cells; ++k) o[k] = (int32_t)((uint32_t)o[k] + (uint32_t)pend[k]);
        }
        break;
    }
    default: return fail(sim, DB_EINVAL, "unknown field");
    }
    return DB_OK;
}

int32_t db_write_state(db_sim* sim, uint32_t field, int64_t first, int64_t count, const void* src) {
    if (!sim || !src) return DB_EINVAL;
    const SimDev& d = sim->dev;
    if (first < d.id0 || count < 0 || first + count > (int64_t)d.id0 + d.N) return fail(sim, DB_ERANGE, "neuron range out of bounds (ids are global; this handle owns [own_first, own_first + own_count))");
    first -= d.id0;
    CK(cudaStreamSynchronize(sim->stream));
    if (count == 0) return DB_OK;
    const size_t Np = (size_t)d.Npad;
    switch (field) {
    case DB_FIELD_V:
        CK(cudaMemcpy(d.V + first, src, (size_t)count * 4, cudaMemcpyHostToDevice)); break;
    case DB_FIELD_G_AMPA: case DB_FIELD_G_NMDA: case DB_FIELD_G_GABAA: case DB_FIELD_G_GABAB:
        CK(cudaMemcpy(d.g + (field - DB_FIELD_G_AMPA) * Np + first, src, (size_t)count * 4, cudaMemcpyHostToDevice)); break;
    case DB_FIELD_IOU:
        if (!d.ou_on) return fail(sim, DB_ESTATE, "no neuron type uses the OU background current");
        CK(cudaMemcpy(d.Iou + first, src, (size_t)count * 4, cudaMemcpyHostToDevice)); break;
    case DB_FIELD_IEXT:
        if (!d.iext) return fail(sim, DB_ESTATE, "no neuron type draws its external current per neuron (iext_gamma_shape = 0)");
        CK(cudaMemcpy(d.iext + first, src, (size_t)count * 4, cudaMemcpyHostToDevice)); break;
    case DB_FIELD_REF: {                               // the counter shares a 16-bit word with the neuron type: merged on the device
        const int32_t* in = static_cast<const int32_t*>(src);
        int32_t lo = 0, hi = 0;
        for (int64_t i = 0; i < count; ++i) { lo = std::min(lo, in[i]); hi = std::max(hi, in[i]); }
        if (lo < 0 || hi > kRefMask) return fail(sim, DB_EINVAL, "ref out of range");
        int32_t* tmp = nullptr;
        CK(cudaMallocAsync(&tmp, (size_t)count * 4, sim->stream));
        CK(cudaMemcpyAsync(tmp, in, (size_t)count * 4, cudaMemcpyHostToDevice, sim->stream));
        k_write_ref<<<(unsigned)std::min<int64_t>((count + 255) / 256, (int64_t)sim->n_sm * 16), 256, 0, sim->stream>>>(d.rt + first, tmp, count);
        CK(cudaGetLastError());
        CK(cudaFreeAsync(tmp, sim->stream));
        CK(cudaStreamSynchronize(sim->stream));        // `src` is the caller's memory
        break;
    }
    case DB_FIELD_RING: {
        Ctl c;
        int32_t rc = read_ctl(sim, &c);
        if (rc) return rc;
        // list mode: what DB_FIELD_RING shows is the device ring plus the records waiting in the arrival lists; once
        // records may be waiting a write could not be read back as written
        if (d.ev_on && c.step > 0)
            return fail(sim, DB_ESTATE, "DB_FIELD_RING is writable only before the first step in DB_EXEC_KERNELS_DEFERRED mode");
        const int D = sim->params.D;
        std::vector<int32_t> t((size_t)count);
        const int32_t* in = static_cast<const int32_t*>(src);
        for (int k = 0; k < D; ++k) {
            const uint64_t step = c.step + (uint64_t)k;
            const size_t s = (size_t)(step % (uint64_t)D), sd = (size_t)(step & (uint64_t)(d.D - 1));
            for (int u = 0; u < 4; ++u) {
                for (int64_t i = 0; i < count; ++i) t[(size_t)i] = in[(s * (size_t)count + (size_t)i) * 4 + u];
                CK(cudaMemcpy(d.ring + (sd * 4 + u) * Np + first, t.data(), (size_t)count * 4, cudaMemcpyHostToDevice));
            }
        }
        break;
    }
    default: return fail(sim, DB_EINVAL, "field is not writable");
    }
    return DB_OK;
}

static int32_t region_windows(db_sim* sim, std::vector<uint32_t>* counts, uint64_t cap_windows,
                              uint64_t* n_windows, uint64_t* first_window) {
    Ctl c;
    int32_t rc = read_ctl(sim, &c);
    if (rc) return rc;
    const SimDev& d = sim->dev;
    const uint64_t done = c.step / (uint64_t)d.window_steps;           // completed windows
    const uint64_t ahead = 2u / (uint64_t)d.window_steps + 1u;         // windows cleared ahead of time (db_step.cu)
    const uint64_t keep = (uint64_t)d.max_windows - 1 - ahead;         // the open window and the cleared ones are not history
    const uint64_t first = done > keep ? done - keep : 0;
    uint64_t n = done - first;
    if (first_window) *first_window = first;
    if (n_windows) *n_windows = n;
    n = std::min(n, cap_windows);
    counts->resize((size_t)n * (size_t)d.n_regions);
    for (uint64_t k = 0; k < n;) {
        const uint64_t idx = (first + k) % d.max_windows;
        const uint64_t run = std::min<uint64_t>(n - k, d.max_windows - idx);
        CK(cudaMemcpy(counts->data() + (size_t)k * d.n_regions, d.region_counts + (size_t)idx * d.n_regions,
                      (size_t)run * d.n_regions * 4, cudaMemcpyDeviceToHost));
        k += run;
    }
    return DB_OK;
}

int32_t db_region_counts(db_sim* sim, uint32_t* counts, uint64_t cap_windows, uint64_t* n_windows, uint64_t* first_window) {
    if (!sim) return DB_EINVAL;
    std::vector<uint32_t> c;
    int32_t rc = region_windows(sim, &c, counts ? cap_windows : 0, n_windows, first_window);
    if (rc) return rc;
    if (counts) std::copy(c.begin(), c.end(), counts);
    return DB_OK;
}

int32_t db_region_rates(db_sim* sim, float* rates_hz, uint64_t cap_windows, uint64_t* n_windows, uint64_t* first_window) {
    if (!sim) return DB_EINVAL;
    std::vector<uint32_t> c;
    int32_t rc = region_windows(sim, &c, rates_hz ? cap_windows : 0, n_windows, first_window);
    if (rc) return rc;
    if (!rates_hz) return DB_OK;
    const int R = sim->dev.n_regions;
    const double win_s = (double)sim->dev.window_steps * sim->params.dt_ms * 1e-3;
    for (size_t k = 0; k < c.size(); ++k) {
        const int r = (int)(k % (size_t)R);
        const double size = (double)(sim->region_start[(size_t)r + 1] - sim->region_start[(size_t)r]);
        rates_hz[k] = size > 0 ? (float)((double)c[k] / (size * win_s)) : 0.0f;
    }
    return DB_OK;
}

int32_t db_read_bold(db_sim* sim, double* y, double* state, uint64_t* n_windows) {
    if (!sim) return DB_EINVAL;
    if (!sim->params.bold.enabled) return fail(sim, DB_ESTATE, "the BOLD read-out was not enabled (db_sim_params.bold.enabled)");
    CK(cudaSetDevice(sim->device));
    CK(launch_bold(sim->dev, sim->bold, sim->stream));     // steps taken through db_step_profiled() are caught up here
    sim->launches += 2;
    CK(cudaStreamSynchronize(sim->stream));
    const size_t R = (size_t)sim->dev.n_regions;
    if (y) CK(cudaMemcpy(y, sim->bold.y, R * sizeof(double), cudaMemcpyDeviceToHost));
    if (state) CK(cudaMemcpy(state, sim->bold.state, 4 * R * sizeof(double), cudaMemcpyDeviceToHost));
    if (n_windows) {
        unsigned long long c = 0;
        CK(cudaMemcpy(&c, sim->bold.cursor, sizeof(c), cudaMemcpyDeviceToHost));
        *n_windows = c;
    }
    return DB_OK;
}

int32_t db_export_csr(db_sim* sim, db_csr_host* out) {
    if (!sim || !out) return DB_EINVAL;
    std::memset(out, 0, sizeof(*out));
    const SimDev& d = sim->dev;
    if (d.N != d.n_rows) return fail(sim, DB_ESTATE, "this handle owns part of the network: export the network from a handle that owns all of it");
    CK(cudaStreamSynchronize(sim->stream));
    const int64_t N = d.N;
    std::vector<int64_t> rb((size_t)N);
    std::vector<int32_t> rl((size_t)N);
    CK(cudaMemcpy(rb.data(), d.row_begin, (size_t)N * 8, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(rl.data(), d.row_len, (size_t)N * 4, cudaMemcpyDeviceToHost));
    std::vector<uint32_t> tr((size_t)sim->Epad);
    std::vector<uint8_t> dl((size_t)sim->Epad);
    CK(cudaMemcpy(tr.data(), d.tgt_rec, (size_t)sim->Epad * 4, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(dl.data(), d.delay, (size_t)sim->Epad, cudaMemcpyDeviceToHost));
    std::vector<float> wf((size_t)sim->Epad);
    if (d.w_fp16) {
        std::vector<__half> wh((size_t)sim->Epad);
        CK(cudaMemcpy(wh.data(), d.w, (size_t)sim->Epad * 2, cudaMemcpyDeviceToHost));
        for (size_t k = 0; k < wh.size(); ++k) wf[k] = __half2float(wh[k]);
    } else {
        CK(cudaMemcpy(wf.data(), d.w, (size_t)sim->Epad * 4, cudaMemcpyDeviceToHost));
    }
    int64_t E = 0;
    for (int64_t j = 0; j < N; ++j) E += rl[(size_t)j];
    out->N = N; out->E = E; out->n_regions = d.n_regions;
    out->region_start = (int64_t*)std::malloc(sizeof(int64_t) * ((size_t)d.n_regions + 1));
    out->ntype = (uint8_t*)std::malloc((size_t)N);
    out->row_ptr = (int64_t*)std::malloc(sizeof(int64_t) * ((size_t)N + 1));
    const size_t En = (size_t)std::max<int64_t>(E, 1);
    out->tgt = (int32_t*)std::malloc(4 * En); out->w = (float*)std::malloc(4 * En);
    out->delay = (uint8_t*)std::malloc(En); out->rec = (uint8_t*)std::malloc(En);
    if (!out->region_start || !out->ntype || !out->row_ptr || !out->tgt || !out->w || !out->delay || !out->rec) {
        db_free_csr(out);
        return fail(sim, DB_ENOMEM, "host allocation failed");
    }
    std::copy(sim->region_start.begin(), sim->region_start.end(), out->region_start);
    CK(cudaMemcpy(out->ntype, sim->ntype_dev, (size_t)N, cudaMemcpyDeviceToHost));
    std::vector<int32_t> order;
    int64_t o = 0;
    out->row_ptr[0] = 0;
    for (int64_t j = 0; j < N; ++j) {
        const int64_t b = rb[(size_t)j];
        const int32_t len = rl[(size_t)j];
        order.resize((size_t)len);
        for (int32_t k = 0; k < len; ++k) order[(size_t)k] = k;
        std::sort(order.begin(), order.end(), [&](int32_t x, int32_t y) {   // canonical: by (target, receptor)
            const uint32_t a = tr[(size_t)(b + x)], c = tr[(size_t)(b + y)];
            const uint32_t ta = a & 0x3FFFFFFFu, tc = c & 0x3FFFFFFFu;
            if (ta != tc) return ta < tc;
            return (a >> 30) < (c >> 30);
        });
        for (int32_t k = 0; k < len; ++k, ++o) {
            const size_t s = (size_t)(b + order[(size_t)k]);
            out->tgt[o] = (int32_t)(tr[s] & 0x3FFFFFFFu); out->rec[o] = (uint8_t)(tr[s] >> 30);
            out->w[o] = wf[s]; out->delay[o] = dl[s];
        }
        out->row_ptr[j + 1] = o;
    }
    return DB_OK;
}

int32_t db_free_csr(db_csr_host* c) {
    if (!c) return DB_EINVAL;
    std::free(c->region_start); std::free(c->ntype); std::free(c->row_ptr);
    std::free(c->tgt); std::free(c->w); std::free(c->delay); std::free(c->rec);
    std::memset(c, 0, sizeof(*c));
    return DB_OK;
}

}  // extern "C"
