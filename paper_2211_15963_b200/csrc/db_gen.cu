// a0: seeded synthetic network generator (stand-in for the paper's HRGCME
// generator).  Every synapse is
// a pure function of (seed, owner neuron, slot), so the presynaptic-major CSR
// is built procedurally in two passes (count out-degrees, then regenerate and
// scatter) without ever materialising an edge list: 10^10 synapses fit.
#include <algorithm>
#include <cmath>
#include <cuda_fp16.h>
#include "db_host.h"
#include "db_philox.cuh"

namespace dbk {

// ---------------------------------------------------------------------------
// host tables
// ---------------------------------------------------------------------------
namespace {

double std_normal_cdf(double z) { return 0.5 * std::erfc(-z * 0.70710678118654752440); }

}  // namespace

// Inverse normal CDF: Newton iterations on erfc from a logistic starting guess.
double std_normal_quantile(double p) {
    double z = 0.0;
    {   // crude start: logit scaled to the normal
        const double l = std::log(p / (1.0 - p));
        z = l * 0.5513 * (1.0 + 0.02 * std::fabs(l));
        if (z > 8.0) z = 8.0;
        if (z < -8.0) z = -8.0;
    }
    for (int it = 0; it < 100; ++it) {
        const double f = std_normal_cdf(z) - p;
        const double pdf = 0.39894228040143267794 * std::exp(-0.5 * z * z);
        double step = f / pdf;
        if (step > 1.0) step = 1.0;
        if (step < -1.0) step = -1.0;
        const double zn = z - step;
        if (zn == z) break;
        z = zn;
        if (std::fabs(step) < 1e-17 * (1.0 + std::fabs(z))) break;
    }
    return z;
}

// Quantile of the Gamma(shape k, scale theta) law (per-neuron external currents, R31).  The regularised incomplete gamma
// function comes from Kummer's series for the lower part and from the even part of Legendre's continued fraction,
// summed by its forward (Wallis) recurrence, for the upper part; the root is found by a bracketed Newton iteration on
// whichever tail is the smaller one, started from the Wilson-Hilferty approximation.
static void gamma_tails(double a, double x, double* P, double* Q) {
    if (x <= 0.0) { *P = 0.0; *Q = 1.0; return; }
    const double front = std::exp(a * std::log(x) - x - std::lgamma(a));
    if (x < a + 1.0) {
        double term = 1.0 / a, sum = term;
        for (int n = 1; n < 200000; ++n) {
            term *= x / (a + (double)n);
            sum += term;
            if (term < sum * 1e-17) break;
        }
        *P = front * sum; *Q = 1.0 - *P;
        return;
    }
    // Q = front / (x + 1 - a - 1 (1 - a) / (x + 3 - a - 2 (2 - a) / (x + 5 - a - ...))): convergents A_n / B_n
    double A0 = 1.0, B0 = 0.0, A1 = 0.0, B1 = 1.0, prev = 0.0;      // A_{-1}, B_{-1}, A_0 = b_0 = 0, B_0 = 1
    for (int n = 1; n < 200000; ++n) {
        const double an = (n == 1) ? 1.0 : -((double)(n - 1)) * ((double)(n - 1) - a);
        const double bn = x + (double)(2 * n - 1) - a;
        const double A2 = bn * A1 + an * A0, B2 = bn * B1 + an * B0;
        A0 = A1; B0 = B1; A1 = A2; B1 = B2;
        if (std::fabs(B1) > 1e200) { A0 *= 1e-200; B0 *= 1e-200; A1 *= 1e-200; B1 *= 1e-200; }
        const double cur = A1 / B1;
        if (n > 1 && std::fabs(cur - prev) <= 1e-17 * std::fabs(cur)) { prev = cur; break; }
        prev = cur;
    }
    *Q = front * prev; *P = 1.0 - *Q;
}

double gamma_quantile(double p, double k, double theta) {
    const double z = std_normal_quantile(p), c = 1.0 / (9.0 * k);
    double x = k * std::pow(std::max(1.0 - c + z * std::sqrt(c), 1e-3), 3.0);
    double lo = 0.0, hi = std::max(4.0 * x, k + 20.0);
    for (;;) { double P, Q; gamma_tails(k, hi, &P, &Q); if (P >= p) break; hi *= 2.0; }
    for (int it = 0; it < 400; ++it) {
        double P, Q;
        gamma_tails(k, x, &P, &Q);
        const double f = (p <= 0.5) ? (P - p) : ((1.0 - p) - Q);      // the smaller tail carries the precision
        if (f > 0.0) hi = x; else lo = x;
        const double pdf = std::exp((k - 1.0) * std::log(x) - x - std::lgamma(k));
        double xn = (pdf > 0.0) ? x - f / pdf : 0.5 * (lo + hi);
        if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
        if (xn == x || hi - lo <= 1e-17 * hi) break;
        x = xn;
    }
    return theta * x;
}

namespace {

double normal_from_words(uint32_t u0, uint32_t u1) {     // Box-Muller, double
    const double a = ((double)u0 + 0.5) / 4294967296.0;
    const double b = ((double)u1 + 0.5) / 4294967296.0;
    return std::sqrt(-2.0 * std::log(a)) * std::cos(2.0 * M_PI * b);
}

}  // namespace

bool gen_host_tables(const db_network_spec& sp, uint64_t seed, GenHostTables* out, std::string* err) {
    const int64_t N = sp.N;
    const int R = sp.n_regions;
    const uint32_t slo = (uint32_t)seed, shi = (uint32_t)(seed >> 32);
    if (N < 2 || N >= (1ll << 30)) { *err = "N must be within 2..2^30-1"; return false; }
    if (R < 1 || R > 4096 || R > N) { *err = "n_regions must be within 1..4096"; return false; }
    if (!(sp.exc_frac > 0.0 && sp.exc_frac <= 1.0)) { *err = "exc_frac must be in (0, 1]"; return false; }
    if (!(sp.slow_frac >= 0.0 && sp.slow_frac < 1.0)) { *err = "slow_frac must be in [0, 1)"; return false; }
    if (sp.mode != DB_MODE_FIXED_INDEGREE && sp.mode != DB_MODE_OUTDEG_LOGNORMAL) { *err = "unknown mode"; return false; }
    auto bad_delay = [](int lo, int hi) { return lo < 1 || hi > 255 || lo > hi; };
    if (bad_delay(sp.delay_intra_min, sp.delay_intra_max) || (R > 1 && bad_delay(sp.delay_inter_min, sp.delay_inter_max))) {
        *err = "delays must satisfy 1 <= min <= max <= 255"; return false;
    }

    // region sizes: lognormal(0, sigma) shares, largest-remainder rounding
    std::vector<int64_t> size((size_t)R);
    if (R == 1) {
        size[0] = N;
    } else {
        std::vector<double> share((size_t)R);
        double total = 0.0;
        for (int r = 0; r < R; ++r) {
            const uint4 o = keyed_draw(slo, shi, kStreamREGION, (uint64_t)r, 0);
            share[(size_t)r] = std::exp(sp.region_size_sigma * normal_from_words(o.x, o.y));
            total += share[(size_t)r];
        }
        std::vector<std::pair<double, int>> rem((size_t)R);
        int64_t used = 0;
        for (int r = 0; r < R; ++r) {
            const double q = share[(size_t)r] / total * (double)N;
            const double fl = std::floor(q);
            size[(size_t)r] = (int64_t)fl;
            rem[(size_t)r] = { -(q - fl), r };
            used += size[(size_t)r];
        }
        std::sort(rem.begin(), rem.end());
        for (int64_t k = 0; k < N - used; ++k) size[(size_t)rem[(size_t)k].second] += 1;
    }
    out->region_start.assign((size_t)R + 1, 0);
    out->region_nexc.assign((size_t)R, 0);
    for (int r = 0; r < R; ++r) {
        out->region_start[(size_t)r + 1] = out->region_start[(size_t)r] + size[(size_t)r];
        out->region_nexc[(size_t)r] = (int32_t)std::floor(sp.exc_frac * (double)size[(size_t)r] + 0.5);
    }

    // weight quantiles
    out->weight_tab.resize(65536);
    for (int q = 0; q < 65536; ++q) {
        const double z = std_normal_quantile(((double)q + 0.5) / 65536.0);
        out->weight_tab[(size_t)q] = (float)(sp.w_scale * std::exp(sp.w_mu + sp.w_sigma * z));
    }

    if (sp.mode == DB_MODE_FIXED_INDEGREE) {
        if (sp.K < 1) { *err = "K must be >= 1"; return false; }
        out->K_intra = sp.K; out->K_inter = 0;
        if (R > 1) {
            out->K_intra = (int32_t)std::floor(sp.intra_frac * (double)sp.K + 0.5);
            out->K_inter = sp.K - out->K_intra;
            if (out->K_intra < 0 || out->K_inter < 0) { *err = "intra_frac must be in [0, 1]"; return false; }
        }
        for (int r = 0; r < R; ++r) {
            if (size[(size_t)r] - 1 < out->K_intra) { *err = "a region is smaller than the intra-region in-degree"; return false; }
            if (out->K_inter > 0 && out->region_nexc[(size_t)r] < out->K_inter) { *err = "a region has fewer excitatory neurons than the inter-region in-degree"; return false; }
        }
        if (out->K_inter > 0) {
            out->region_cdf.resize((size_t)R * (size_t)(R - 1));
            std::vector<double> p((size_t)R);
            for (int r = 0; r < R; ++r) {
                double s = 0.0;
                for (int c = 0; c < R; ++c) {
                    const uint4 o = keyed_draw(slo, shi, kStreamREGION, (uint64_t)r * (uint64_t)R + (uint64_t)c, 1);
                    p[(size_t)c] = (c == r) ? 0.0 : std::exp(sp.region_matrix_sigma * normal_from_words(o.x, o.y));
                    s += p[(size_t)c];
                }
                double cum = 0.0;
                for (int c = 0; c < R - 1; ++c) {
                    cum += p[(size_t)c] / s;
                    double t = std::floor(cum * 4294967296.0);
                    if (t > 4294967295.0) t = 4294967295.0;
                    out->region_cdf[(size_t)r * (size_t)(R - 1) + (size_t)c] = (uint32_t)t;
                }
            }
        }
    } else {
        if (R != 1) { *err = "out-degree mode supports one region"; return false; }
        if (!(sp.outdeg_mean >= 1.0) || sp.outdeg_cap < 1) { *err = "bad out-degree parameters"; return false; }
        out->outdeg_tab.resize(65536);
        const double mu = std::log(sp.outdeg_mean) - 0.5 * sp.outdeg_sigma * sp.outdeg_sigma;
        for (int q = 0; q < 65536; ++q) {
            const double z = std_normal_quantile(((double)q + 0.5) / 65536.0);
            double d = std::floor(std::exp(mu + sp.outdeg_sigma * z) + 0.5);
            if (d < 1.0) d = 1.0;
            if (d > (double)sp.outdeg_cap) d = (double)sp.outdeg_cap;
            out->outdeg_tab[(size_t)q] = (int32_t)d;
        }
    }
    return true;
}

// ---------------------------------------------------------------------------
// device side
// ---------------------------------------------------------------------------
struct GenDev {
    int32_t N, R, K, K_intra, K_inter;
    int32_t own0, ownN;            // the targets this handle owns: [own0, own0 + ownN) (the whole network: 0, N)
    uint32_t seed_lo, seed_hi;
    const int32_t* region_start;   // [R + 1]
    const int32_t* region_nexc;    // [R]
    const uint32_t* region_cdf;    // [R][R - 1]
    const float* weight_tab;       // [65536]
    const int32_t* outdeg_tab;     // [65536]
    float inh_mult;
    uint32_t slow_thr;
    int32_t d_intra_min, d_intra_span, d_inter_min, d_inter_span;
    int32_t w_fp16;
    // outputs
    int32_t* row_len;              // [N] out-degree
    int32_t* cursor;               // [N] fill position inside each row
    const int64_t* row_begin;      // [N]
    uint32_t* tgt_rec; void* w; uint8_t* delay;
};

__device__ __forceinline__ int gen_region_of(const GenDev& g, int i) {
    int lo = 0, hi = g.R;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(g.region_start + mid) <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// number of thresholds <= u (thresholds are non-decreasing)
__device__ __forceinline__ int cdf_pick(const uint32_t* T, int n, uint32_t u) {
    int lo = 0, hi = n;                     // invariant: T[0..lo) <= u, T[hi..n) > u
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(T + mid) <= u) lo = mid + 1; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void emit_synapse(const GenDev& g, uint64_t owner, uint64_t slot, int src, int tgt,
                                             bool inh, bool inter, int64_t pos) {
    const uint4 o = keyed_draw(g.seed_lo, g.seed_hi, kStreamSYN, owner, slot);
    float w = __ldg(g.weight_tab + (o.x >> 16));
    if (inh) w = __fmul_rn(w, g.inh_mult);
    const int dmin = inter ? g.d_inter_min : g.d_intra_min;
    const int span = inter ? g.d_inter_span : g.d_intra_span;
    const uint32_t d = (uint32_t)dmin + __umulhi(o.y, (uint32_t)span);
    const uint32_t rec = (inh ? 2u : 0u) + (o.z < g.slow_thr ? 1u : 0u);
    g.tgt_rec[pos] = (rec << 30) | (uint32_t)tgt;
    g.delay[pos] = (uint8_t)d;
    if (g.w_fp16) static_cast<__half*>(g.w)[pos] = __float2half_rn(w);
    else          static_cast<float*>(g.w)[pos] = w;
    (void)src;
}

__global__ void k_gen_types(const __grid_constant__ GenDev g, uint8_t* ntype) {       // ntype[] is local: the owned neurons
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= g.ownN) return;
    const int i = g.own0 + l;
    const int r = gen_region_of(g, i);
    ntype[l] = (uint8_t)((i - g.region_start[r]) >= g.region_nexc[r]);
}

// Mode 0, one warp per target neuron i.  kFill = false: count out-degrees of
// the sources; kFill = true: regenerate and scatter into the rows.
template <bool kFill>
__global__ void __launch_bounds__(256) k_gen_indegree(const __grid_constant__ GenDev g) {
    const unsigned lane = threadIdx.x & 31u;
    const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    // (a handle that owns part of the network draws the inputs of ITS neurons only: the same draws, keyed by the global id)
    for (long long i = g.own0 + (((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5); i < g.own0 + g.ownN; i += n_warps) {
        int r = 0;
        uint4 key_in = make_uint4(0, 0, 0, 0), key_out = key_in;
        if (lane == 0) {
            r = gen_region_of(g, (int)i);
            key_in = keyed_draw(g.seed_lo, g.seed_hi, kStreamSRC, (uint64_t)i, 0);
            key_out = keyed_draw(g.seed_lo, g.seed_hi, kStreamSRC, (uint64_t)i, 1);
        }
        r = __shfl_sync(0xffffffffu, r, 0);
        key_in.x = __shfl_sync(0xffffffffu, key_in.x, 0); key_in.y = __shfl_sync(0xffffffffu, key_in.y, 0);
        key_in.z = __shfl_sync(0xffffffffu, key_in.z, 0); key_in.w = __shfl_sync(0xffffffffu, key_in.w, 0);
        key_out.x = __shfl_sync(0xffffffffu, key_out.x, 0); key_out.y = __shfl_sync(0xffffffffu, key_out.y, 0);
        key_out.z = __shfl_sync(0xffffffffu, key_out.z, 0); key_out.w = __shfl_sync(0xffffffffu, key_out.w, 0);
        const int base = __ldg(g.region_start + r);
        const int size = __ldg(g.region_start + r + 1) - base;
        const int nexc = __ldg(g.region_nexc + r);
        const int li = (int)i - base;
        for (int k = (int)lane; k < g.K; k += 32) {
            int src; bool inh, inter;
            if (k < g.K_intra) {                                  // own region, any type, never itself
                uint32_t j = feistel_perm((uint32_t)k, (uint32_t)(size - 1), key_in);
                if ((int)j >= li) ++j;
                src = base + (int)j; inh = (int)j >= nexc; inter = false;
            } else {                                              // another region, excitatory only
                const int s = k - g.K_intra;
                const uint32_t u = keyed_draw(g.seed_lo, g.seed_hi, kStreamINTER, (uint64_t)i, (uint64_t)s).x;
                const int rs = cdf_pick(g.region_cdf + (size_t)r * (size_t)(g.R - 1), g.R - 1, u);
                const uint32_t j = feistel_perm((uint32_t)s, (uint32_t)__ldg(g.region_nexc + rs), key_out);
                src = __ldg(g.region_start + rs) + (int)j; inh = false; inter = true;
            }
            if (!kFill) {
                atomicAdd(g.row_len + src, 1);
            } else {
                const int64_t pos = __ldg(g.row_begin + src) + atomicAdd(g.cursor + src, 1);
                emit_synapse(g, (uint64_t)i, (uint64_t)k, src, (int)i - g.own0, inh, inter, pos);      // targets are stored locally
            }
        }
    }
}

// Mode 1: out-degree of every neuron from the quantile table.
__global__ void k_gen_outdeg(const __grid_constant__ GenDev g) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= g.N) return;
    int deg = __ldg(g.outdeg_tab + (keyed_draw(g.seed_lo, g.seed_hi, kStreamDEG, (uint64_t)j, 0).x >> 16));
    if (deg > g.N - 1) deg = g.N - 1;
    g.row_len[j] = deg;
}

// Mode 1 fill: one warp per source row; targets = first deg elements of a keyed permutation.
__global__ void __launch_bounds__(256) k_gen_outrows(const __grid_constant__ GenDev g) {
    const unsigned lane = threadIdx.x & 31u;
    const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long j = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; j < g.N; j += n_warps) {
        const uint4 key = keyed_draw(g.seed_lo, g.seed_hi, kStreamSRC, (uint64_t)j, 0);
        const int deg = g.row_len[j];
        const int64_t rb = __ldg(g.row_begin + j);
        const bool inh = (int)j >= __ldg(g.region_nexc);
        for (int m = (int)lane; m < deg; m += 32) {
            uint32_t t = feistel_perm((uint32_t)m, (uint32_t)(g.N - 1), key);
            if ((long long)t >= j) ++t;
            emit_synapse(g, (uint64_t)j, (uint64_t)m, (int)j, (int)t, inh, false, rb + m);
        }
    }
}

// ---------------------------------------------------------------------------
cudaError_t generate_network(const db_network_spec& sp, uint64_t seed, const GenHostTables& tabs,
                             const GenAlloc& ga, cudaStream_t st, int32_t Npad, uint8_t* ntype_dev,
                             GenResult* out, std::string* err) {
    (void)Npad;
    const int64_t N = sp.N;
    const int R = sp.n_regions;
    cudaError_t e;
    auto A = [&](size_t bytes) -> void* {
        void* p = ga.alloc(ga.user, bytes);
        if (!p) { out->oom = true; *err = "device allocation of " + std::to_string(bytes) + " bytes failed"; }
        return p;
    };
#define GCK(x) do { e = (x); if (e != cudaSuccess) { *err = #x; return e; } } while (0)

    GenDev g{};
    g.own0 = sp.own_count ? (int32_t)sp.own_first : 0; g.ownN = sp.own_count ? (int32_t)sp.own_count : (int32_t)N;
    g.N = (int32_t)N; g.R = R; g.K = sp.K; g.K_intra = tabs.K_intra; g.K_inter = tabs.K_inter;
    g.seed_lo = (uint32_t)seed; g.seed_hi = (uint32_t)(seed >> 32);
    g.inh_mult = (float)sp.inh_mult;
    g.slow_thr = (uint32_t)std::floor(sp.slow_frac * 4294967296.0);
    g.d_intra_min = sp.delay_intra_min; g.d_intra_span = sp.delay_intra_max - sp.delay_intra_min + 1;
    g.d_inter_min = sp.delay_inter_min; g.d_inter_span = sp.delay_inter_max - sp.delay_inter_min + 1;
    g.w_fp16 = sp.weight_fp16 ? 1 : 0;
    out->max_delay = sp.delay_intra_max;
    if (tabs.K_inter > 0) out->max_delay = std::max(out->max_delay, sp.delay_inter_max);

    // small tables
    std::vector<int32_t> rs32((size_t)R + 1);
    for (int r = 0; r <= R; ++r) rs32[(size_t)r] = (int32_t)tabs.region_start[(size_t)r];
    int32_t* rs_dev = (int32_t*)A(rs32.size() * 4); if (!rs_dev) return cudaSuccess;
    int32_t* ne_dev = (int32_t*)A((size_t)R * 4); if (!ne_dev) return cudaSuccess;
    float* wt_dev = (float*)A(65536 * 4); if (!wt_dev) return cudaSuccess;
    GCK(cudaMemcpyAsync(rs_dev, rs32.data(), rs32.size() * 4, cudaMemcpyHostToDevice, st));
    GCK(cudaMemcpyAsync(ne_dev, tabs.region_nexc.data(), (size_t)R * 4, cudaMemcpyHostToDevice, st));
    GCK(cudaMemcpyAsync(wt_dev, tabs.weight_tab.data(), 65536 * 4, cudaMemcpyHostToDevice, st));
    g.region_start = rs_dev; g.region_nexc = ne_dev; g.weight_tab = wt_dev;
    if (!tabs.region_cdf.empty()) {
        uint32_t* cdf_dev = (uint32_t*)A(tabs.region_cdf.size() * 4); if (!cdf_dev) return cudaSuccess;
        GCK(cudaMemcpyAsync(cdf_dev, tabs.region_cdf.data(), tabs.region_cdf.size() * 4, cudaMemcpyHostToDevice, st));
        g.region_cdf = cdf_dev;
    }
    if (!tabs.outdeg_tab.empty()) {
        int32_t* od_dev = (int32_t*)A(65536 * 4); if (!od_dev) return cudaSuccess;
        GCK(cudaMemcpyAsync(od_dev, tabs.outdeg_tab.data(), 65536 * 4, cudaMemcpyHostToDevice, st));
        g.outdeg_tab = od_dev;
    }
    int32_t* row_len = (int32_t*)A((size_t)N * 4); if (!row_len) return cudaSuccess;
    int32_t* cursor = (int32_t*)A((size_t)N * 4); if (!cursor) return cudaSuccess;
    int64_t* row_begin = (int64_t*)A((size_t)N * 8); if (!row_begin) return cudaSuccess;
    GCK(cudaMemsetAsync(row_len, 0, (size_t)N * 4, st));
    GCK(cudaMemsetAsync(cursor, 0, (size_t)N * 4, st));
    g.row_len = row_len; g.cursor = cursor; g.row_begin = row_begin;

    k_gen_types<<<(unsigned)((g.ownN + 255) / 256), 256, 0, st>>>(g, ntype_dev);
    GCK(cudaGetLastError());

    int dev = 0, n_sm = 0;
    GCK(cudaGetDevice(&dev));
    GCK(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    const unsigned warp_grid = (unsigned)std::min<int64_t>((N + 7) / 8, (int64_t)n_sm * 64);
    if (sp.mode == DB_MODE_FIXED_INDEGREE) {
        k_gen_indegree<false><<<warp_grid, 256, 0, st>>>(g);
    } else {
        k_gen_outdeg<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(g);
    }
    GCK(cudaGetLastError());

    // row offsets: exclusive scan of the padded out-degrees (one-off; on the host)
    std::vector<int32_t> len_h((size_t)N);
    GCK(cudaMemcpyAsync(len_h.data(), row_len, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
    GCK(cudaStreamSynchronize(st));
    std::vector<int64_t> begin_h((size_t)N);
    int64_t pos = 0, E = 0;
    uint64_t work_cap = 0, heavy_chunks = 0;
    for (int64_t j = 0; j < N; ++j) {
        const int64_t len = len_h[(size_t)j];
        begin_h[(size_t)j] = pos;
        pos += (len + kRowAlign - 1) / kRowAlign * kRowAlign;
        E += len;
        work_cap += (uint64_t)((len + kChunk - 1) / kChunk);
        if (len > kInlineMax) heavy_chunks += (uint64_t)((len + kChunk - 1) / kChunk);
    }
    out->E = E; out->Epad = pos + kRowAlign; out->work_cap = work_cap; out->heavy_chunks = heavy_chunks;
    GCK(cudaMemcpyAsync(row_begin, begin_h.data(), (size_t)N * 8, cudaMemcpyHostToDevice, st));

    uint32_t* tgt_rec = (uint32_t*)A((size_t)out->Epad * 4); if (!tgt_rec) return cudaSuccess;
    uint8_t* delay = (uint8_t*)A((size_t)out->Epad); if (!delay) return cudaSuccess;
    void* w = A((size_t)out->Epad * (sp.weight_fp16 ? 2 : 4)); if (!w) return cudaSuccess;
    g.tgt_rec = tgt_rec; g.delay = delay; g.w = w;
    if (sp.mode == DB_MODE_FIXED_INDEGREE) k_gen_indegree<true><<<warp_grid, 256, 0, st>>>(g);
    else                                   k_gen_outrows<<<warp_grid, 256, 0, st>>>(g);
    GCK(cudaGetLastError());
    GCK(cudaStreamSynchronize(st));
    out->row_begin = row_begin; out->row_len = row_len; out->tgt_rec = tgt_rec; out->w = w; out->delay = delay;
#undef GCK
    return cudaSuccess;
}

}  // namespace dbk
