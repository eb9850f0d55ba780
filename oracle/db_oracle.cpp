// =============================================================================
// db_oracle.cpp -- ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Plain, slow, single-threaded CPU implementation of the per-time-step hot path
// of the Digital Brain spiking-network simulator (arXiv 2211.15963), written
// from /root/reference/PAPER.md ("P:L<n>" = line n of that file) and the
// readings listed in DESIGN.md ("R<n>").  It shares NO code with the CUDA path
// under paper_2211_15963_b200/: no headers, helpers, tables or generators.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load this library.
//
// What is here
//   1. Philox4x32-10 counter-based generator (Salmon et al., SC'11) + the
//      keyed draws the method uses (V0, Poisson background, generator).
//   2. Integer Poisson inverse-CDF thresholds (background drive).
//   3. The synthetic network generator (stand-in for the paper's HRGCME
//      generator): fixed in-degree / lognormal
//      out-degree, regions, no autapses, no multapses.
//   4. The simulator: one iteration = SI Eq.(3) conductances,
//      SI Eq.(5) membrane step read with the CV equation,
//      threshold / reset / refractory, push-based spike
//      delivery (Supp. Alg. 2) into a delayed fixed-point ring.
//   5. Dense brute-force delivery (plain definition of the delivered sums).
//
// Pins (tests/, -m "not gpu"): Philox known-answer vectors; Poisson moments;
// discrete + continuous LIF closed forms, first-spike time, ISI = n*+R;
// single-event conductance kernel; PSP shape; dense brute force + event
// conservation; generator degree/no-dup/receptor/moment checks and a second
// independent (Python) implementation of the draws.
// Parity unpinned: the numeric neuron constants (paper prints none, R13) and
// the absolute firing rates they produce.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -shared -fPIC
//        (no FMA contraction: the fp32 mode is an arithmetic contract, R-FP).
// =============================================================================
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <vector>

namespace {

// ----------------------------------------------------------------------------
// 1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as
//    easy as 1, 2, 3", SC'11).  10 rounds; multipliers / Weyl constants as
//    published.  counter c[4], key k[2] -> 4 output words.
// ----------------------------------------------------------------------------
struct u32x4 { uint32_t w[4]; };

u32x4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                    uint32_t k0, uint32_t k1) {
    const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    u32x4 o; o.w[0] = c0; o.w[1] = c1; o.w[2] = c2; o.w[3] = c3;
    return o;
}

// Keyed draw used everywhere (R-RNG): key = seed, counter =
// (a_lo, a_hi | stream<<24, b_lo, b_hi); a < 2^56 is an entity id, b a second
// index (time step, slot).
enum : uint32_t {
    STREAM_V0 = 1,     // initial membrane potential
    STREAM_BG = 2,     // Poisson background counts
    STREAM_SRC = 3,    // permutation round keys (source / target selection)
    STREAM_SYN = 4,    // per-synapse weight / delay / receptor
    STREAM_REGION = 5, // region sizes and region matrix (host-side normals)
    STREAM_INTER = 6,  // source-region choice of an inter-region input
    STREAM_DEG = 7,    // out-degree of a neuron (out-degree mode)
    STREAM_OU = 8,     // Gaussian increments of the OU background current
    STREAM_IEXT = 9    // per-neuron external current (Gamma quantile table)
};

u32x4 draw(uint64_t seed, uint32_t stream, uint64_t a, uint64_t b) {
    return philox4x32_10((uint32_t)a, (uint32_t)(a >> 32) | (stream << 24),
                         (uint32_t)b, (uint32_t)(b >> 32),
                         (uint32_t)seed, (uint32_t)(seed >> 32));
}

// ----------------------------------------------------------------------------
// 2. Poisson inverse CDF on a 32-bit uniform (background drive: "independent
//    homogeneous Poisson spike trains"; R14).
//    T_m = floor(CDF(m; lambda) * 2^32), k = #{m : u >= T_m}.
// ----------------------------------------------------------------------------
const int POISSON_MAX = 32;

int poisson_thresholds(double lambda, uint32_t* T /*[POISSON_MAX]*/) {
    double pm = std::exp(-lambda);   // P(0)
    double cdf = 0.0;
    int M = 0;
    for (int m = 0; m < POISSON_MAX; ++m) {
        cdf += pm;
        double t = std::floor(cdf * 4294967296.0);
        if (t >= 4294967295.0) break;          // CDF saturated at 32-bit resolution
        T[M++] = (uint32_t)t;
        pm = pm * lambda / (double)(m + 1);
    }
    return M;
}

int poisson_count(uint32_t u, const uint32_t* T, int M) {
    int k = 0;
    for (int m = 0; m < M; ++m) if (u >= T[m]) ++k;
    return k;
}

// ----------------------------------------------------------------------------
// 3a. Keyed pseudo-random permutation of [0, M): 8-round alternating Feistel
//     network on nb = max(2, ceil(log2 M)) bits with cycle walking (round r
//     uses key[r & 3] + (r >> 2) * 0x9E3779B9).  Taking
//     perm(0), perm(1), ... gives sources "sampled with equal probability
//     without replacement" with no rejection state.
// ----------------------------------------------------------------------------
uint32_t fmix32(uint32_t h) {      // MurmurHash3 finaliser (public domain)
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}

uint32_t prp(uint32_t x, uint32_t M, const uint32_t key[4]) {
    if (M <= 1) return 0;
    int nb = 2;
    while (nb < 32 && (1ull << nb) < (uint64_t)M) ++nb;
    const int a = nb / 2, b = nb - a;           // left a bits, right b bits
    do {
        uint32_t L = x >> b, R = x & ((1u << b) - 1u);
        int nl = a, nr = b;
        for (int r = 0; r < 8; ++r) {
            uint32_t rk = key[r & 3] + (uint32_t)(r >> 2) * 0x9E3779B9u;
            uint32_t F = fmix32(R + rk) & ((1u << nl) - 1u);
            uint32_t newR = L ^ F;              // nl bits
            L = R; R = newR;
            int t = nl; nl = nr; nr = t;
        }
        x = (L << nr) | R;                      // even round count: (nl, nr) == (a, b) again
    } while (x >= M);
    return x;
}

// ----------------------------------------------------------------------------
// 3b. Host-side helpers for distribution tables.
// ----------------------------------------------------------------------------
double norm_cdf(double z) { return 0.5 * std::erfc(-z / std::sqrt(2.0)); }

double norm_ppf(double p) {                      // bisection on the CDF
    double lo = -40.0, hi = 40.0;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (norm_cdf(mid) < p) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

// Regularised lower incomplete gamma function P(a, x) = gamma(a, x) / Gamma(a): power series for x < a + 1, else one minus
// the continued fraction of Q(a, x) (modified Lentz); a > 0, x >= 0.
double gamma_p(double a, double x) {
    if (x <= 0.0) return 0.0;
    const double lg = std::lgamma(a);
    if (x < a + 1.0) {
        double ap = a, sum = 1.0 / a, del = sum;
        for (int n = 0; n < 100000; ++n) {
            ap += 1.0; del *= x / ap; sum += del;
            if (std::fabs(del) < std::fabs(sum) * 1e-17) break;
        }
        return sum * std::exp(-x + a * std::log(x) - lg);
    }
    const double tiny = 1e-300;
    double b = x + 1.0 - a, c = 1.0 / tiny, d = 1.0 / b, h = d;
    for (int i = 1; i < 100000; ++i) {
        const double an = -(double)i * ((double)i - a);
        b += 2.0;
        d = an * d + b; if (std::fabs(d) < tiny) d = tiny;
        c = b + an / c; if (std::fabs(c) < tiny) c = tiny;
        d = 1.0 / d;
        const double del = d * c;
        h *= del;
        if (std::fabs(del - 1.0) < 1e-16) break;
    }
    return 1.0 - std::exp(-x + a * std::log(x) - lg) * h;
}
// Quantile of the Gamma(shape k, scale theta) distribution: bisection on P(k, x / theta) = p.
double gamma_ppf(double p, double k, double theta) {
    double lo = 0.0, hi = k + 10.0;
    while (gamma_p(k, hi) < p) hi *= 2.0;
    for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (gamma_p(k, mid) < p) lo = mid; else hi = mid;
    }
    return theta * 0.5 * (lo + hi);
}

// IEEE binary16 round-to-nearest-even of a float, returned as float.
float round_to_half(float f) {
    uint32_t x; std::memcpy(&x, &f, 4);
    uint32_t sign = x & 0x80000000u;
    uint32_t ax = x & 0x7FFFFFFFu;
    float r;
    if (ax >= 0x7F800000u) return f;                      // inf / nan
    float af; std::memcpy(&af, &ax, 4);
    if (af >= 65520.0f) { uint32_t inf = sign | 0x7F800000u; std::memcpy(&r, &inf, 4); return r; }
    if (af < 6.103515625e-05f) {                          // subnormal half: multiples of 2^-24
        float q = std::nearbyintf(af * 16777216.0f) / 16777216.0f;
        uint32_t qb; std::memcpy(&qb, &q, 4); qb |= sign; std::memcpy(&r, &qb, 4); return r;
    }
    uint32_t rem = ax & 0x1FFFu, base = ax & ~0x1FFFu;    // drop 13 mantissa bits
    if (rem > 0x1000u || (rem == 0x1000u && (base & 0x2000u))) base += 0x2000u;
    base |= sign; std::memcpy(&r, &base, 4);
    return r;
}

}  // namespace

// =============================================================================
// C interface (ctypes).  All structs are plain data.
// =============================================================================
extern "C" {

// Per neuron type (0 = excitatory, 1 = inhibitory).  Names follow the paper's
// property table (Supp. Table 5).  Units: ms, mV; C = 1 makes
// g_L = 1/tau_m.
struct orc_type_params {
    double C, gL, VL, Vth, Vreset, Tref_ms, Iext;
    double G[4];        // g_u: maximal conductance per receptor
    double E[4];        // V_u: reversal potential
    double tau_ms[4];   // tau_u
    double bg_rate_hz;  // Poisson background rate per neuron (R14)
    double bg_weight;   // its weight, delivered to AMPA
    // OU background current (main Eq.(1), SI Eq.(4); mu = 0.66, sigma = 0.12, tau = 10 in
    // Ext. Table 2), read per R3: I += (mu - I) dt/tau + sigma sqrt(2 dt/tau) xi, xi ~ N(0,1).
    // ou_tau_ms = 0 switches it off.
    double ou_mu, ou_sigma, ou_tau_ms;
    // External current per neuron ("independently sampled following a Gamma distribution"; property table
    // P:L821), reading R31: I_ext,i = Iext + Gamma(shape, scale) drawn once per neuron through a 65,536-point quantile table
    // indexed by the top 16 bits of a Philox word (stream 9, counter = neuron).  iext_gamma_shape = 0: every neuron gets Iext.
    double iext_gamma_shape, iext_gamma_scale;
};

struct orc_sim_params {
    double dt_ms;
    int32_t S;            // fixed-point shift of the ring (R28)
    int32_t D;            // ring depth, power of two, > max delay
    int32_t window_steps; // region-rate window (R24)
    int32_t n_types;
    orc_type_params type[8];
    // Time bin for transferring spikes, b_t, in steps (SI "Numerical method"; the paper sets
    // b_t = 1 ms even at dt = 0.1 ms).  Reading R29: A_j(t) = 1 only at the bin boundaries t = k b_t,
    // for the neurons that fired in (t - b_t, t].  0 or 1: every step is a boundary.
    int32_t spike_bin_steps;
};

struct orc_net_spec {
    int64_t N;
    int32_t n_regions;
    double region_size_sigma;    // region sizes ~ lognormal(0, sigma), normalised
    double exc_frac;             // 0.8
    int32_t mode;                // 0 fixed in-degree, 1 lognormal out-degree
    int32_t K;                   // in-degree (mode 0)
    double intra_frac;           // fraction of K from the own region (n_regions > 1)
    double region_matrix_sigma;  // inter-region weights ~ lognormal(0, sigma), zero diag, row-normalised
    double outdeg_mean, outdeg_sigma; int32_t outdeg_cap;   // mode 1 (R27)
    double w_mu, w_sigma, w_scale, inh_mult, slow_frac;     // weights (R11), receptors (R12)
    int32_t delay_intra_min, delay_intra_max, delay_inter_min, delay_inter_max; // steps
    int32_t weight_fp16;
};

// ---- raw generator access for the pins --------------------------------------
void orc_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                uint32_t k0, uint32_t k1, uint32_t* out4) {
    u32x4 o = philox4x32_10(c0, c1, c2, c3, k0, k1);
    for (int i = 0; i < 4; ++i) out4[i] = o.w[i];
}
void orc_draw(uint64_t seed, uint32_t stream, uint64_t a, uint64_t b, uint32_t* out4) {
    u32x4 o = draw(seed, stream, a, b);
    for (int i = 0; i < 4; ++i) out4[i] = o.w[i];
}
int32_t orc_poisson_thresholds(double lambda, uint32_t* T) { return poisson_thresholds(lambda, T); }
int32_t orc_poisson_count(uint32_t u, const uint32_t* T, int32_t M) { return poisson_count(u, T, M); }
uint32_t orc_prp(uint32_t x, uint32_t M, const uint32_t* key4) { return prp(x, M, key4); }
double orc_norm_ppf(double p) { return norm_ppf(p); }
double orc_gamma_ppf(double p, double k, double theta) { return gamma_ppf(p, k, theta); }
void orc_gamma_table(double k, double theta, float* tab /*[65536]*/) {
    for (int q = 0; q < 65536; ++q) tab[q] = (float)gamma_ppf(((double)q + 0.5) / 65536.0, k, theta);
}
float orc_round_to_half(float f) { return round_to_half(f); }

// =============================================================================
// 3c. Network generator.  Output: presynaptic-major CSR (one row per source
//     neuron = the paper's per-neuron destination-address list), rows
//     sorted by (target, receptor).  Regions are contiguous id ranges,
//     excitatory neurons first inside each region.
// =============================================================================
struct orc_network {
    int64_t N, E;
    int32_t n_regions;
    int64_t* region_start;   // [n_regions+1]
    int64_t* region_nexc;    // [n_regions]
    uint8_t* ntype;          // [N] 0 exc / 1 inh
    int64_t* row_ptr;        // [N+1]
    int32_t* tgt;            // [E]
    float* w;                // [E] (already rounded to binary16 if weight_fp16)
    uint8_t* delay;          // [E] steps
    uint8_t* rec;            // [E] receptor 0..3
};

void orc_network_free(orc_network* n) {
    if (!n) return;
    std::free(n->region_start); std::free(n->region_nexc); std::free(n->ntype);
    std::free(n->row_ptr); std::free(n->tgt); std::free(n->w); std::free(n->delay); std::free(n->rec);
    std::free(n);
}

namespace {
struct Edge { int32_t src, tgt; float w; uint8_t delay, rec; };

// Standard normal from two 32-bit words (Box-Muller, double); host tables only.
double normal_from(uint32_t u0, uint32_t u1) {
    double a = ((double)u0 + 0.5) / 4294967296.0;
    double b = ((double)u1 + 0.5) / 4294967296.0;
    return std::sqrt(-2.0 * std::log(a)) * std::cos(2.0 * M_PI * b);
}

// Largest-remainder apportionment of `total` into parts proportional to x[].
std::vector<int64_t> apportion(const std::vector<double>& x, int64_t total) {
    size_t n = x.size();
    double s = 0; for (double v : x) s += v;
    std::vector<int64_t> out(n);
    std::vector<std::pair<double, size_t>> frac(n);
    int64_t used = 0;
    for (size_t i = 0; i < n; ++i) {
        double q = x[i] / s * (double)total;
        out[i] = (int64_t)std::floor(q);
        frac[i] = { -(q - std::floor(q)), i };   // sort: largest remainder first, then index
        used += out[i];
    }
    std::sort(frac.begin(), frac.end());
    for (int64_t r = 0; r < total - used; ++r) out[frac[(size_t)r].second] += 1;
    return out;
}

int region_of(const int64_t* region_start, int n_regions, int64_t i) {
    int r = 0;
    while (r + 1 < n_regions && region_start[r + 1] <= i) ++r;   // plain linear scan
    return r;
}
}  // namespace

// Weight quantile table (65536 entries): w_q = scale * exp(mu + sigma * Phi^-1((q+0.5)/65536)).
void orc_weight_table(double mu, double sigma, double scale, float* tab /*[65536]*/) {
    for (int q = 0; q < 65536; ++q) {
        double z = norm_ppf(((double)q + 0.5) / 65536.0);
        tab[q] = (float)(scale * std::exp(mu + sigma * z));
    }
}

// Out-degree quantile table (mode 1, R27): mean of the lognormal = outdeg_mean.
void orc_outdeg_table(double mean, double sigma, int32_t cap, int32_t* tab /*[65536]*/) {
    double mu = std::log(mean) - 0.5 * sigma * sigma;
    for (int q = 0; q < 65536; ++q) {
        double z = norm_ppf(((double)q + 0.5) / 65536.0);
        double d = std::floor(std::exp(mu + sigma * z) + 0.5);
        if (d < 1) d = 1;
        if (d > cap) d = cap;
        tab[q] = (int32_t)d;
    }
}

// Region sizes (lognormal, normalised, largest remainder) -- config 2 / 3.
void orc_region_sizes(uint64_t seed, int64_t N, int32_t R, double sigma, int64_t* sizes) {
    std::vector<double> x((size_t)R);
    for (int r = 0; r < R; ++r) {
        u32x4 o = draw(seed, STREAM_REGION, (uint64_t)r, 0);
        x[(size_t)r] = std::exp(sigma * normal_from(o.w[0], o.w[1]));
    }
    std::vector<int64_t> s = apportion(x, N);
    for (int r = 0; r < R; ++r) sizes[r] = s[(size_t)r];
}

// Inter-region cumulative thresholds: row r holds R-1 uint32 thresholds; the
// source region of a draw u is #{m : u >= T[r][m]}.
void orc_region_cdf(uint64_t seed, int32_t R, double sigma, uint32_t* T /*[R][R-1]*/) {
    for (int r = 0; r < R; ++r) {
        std::vector<double> p((size_t)R);
        double s = 0;
        for (int c = 0; c < R; ++c) {
            u32x4 o = draw(seed, STREAM_REGION, (uint64_t)r * (uint64_t)R + (uint64_t)c, 1);
            p[(size_t)c] = (c == r) ? 0.0 : std::exp(sigma * normal_from(o.w[0], o.w[1]));
            s += p[(size_t)c];
        }
        double cum = 0;
        for (int c = 0; c < R - 1; ++c) {
            cum += p[(size_t)c] / s;
            double t = std::floor(cum * 4294967296.0);
            if (t > 4294967295.0) t = 4294967295.0;
            T[(size_t)r * (size_t)(R - 1) + (size_t)c] = (uint32_t)t;
        }
    }
}

// Tables and per-neuron draws of the generator.  `owner_edges(i)` appends the
// synapses owned by neuron i: its K inputs (mode 0) or its outputs (mode 1).
struct orc_gen {
    orc_net_spec sp; uint64_t seed;
    std::vector<int64_t> region_start, region_nexc;
    std::vector<uint32_t> cdf;
    std::vector<float> wtab;
    std::vector<int32_t> dtab;
    int K_intra, K_inter;

    bool is_inh(int64_t j) const {
        int r = region_of(region_start.data(), sp.n_regions, j);
        return (j - region_start[(size_t)r]) >= region_nexc[(size_t)r];
    }
    // attributes of the synapse drawn as (owner, slot): weight, delay, receptor
    Edge make_edge(int64_t owner, int64_t slot, int64_t src, int64_t tgt, bool inter) const {
        u32x4 o = draw(seed, STREAM_SYN, (uint64_t)owner, (uint64_t)slot);
        Edge e;
        e.src = (int32_t)src; e.tgt = (int32_t)tgt;
        bool inh = is_inh(src);
        float w = wtab[o.w[0] >> 16];
        if (inh) w = w * (float)sp.inh_mult;
        if (sp.weight_fp16) w = round_to_half(w);
        e.w = w;
        int dmin = inter ? sp.delay_inter_min : sp.delay_intra_min;
        int dmax = inter ? sp.delay_inter_max : sp.delay_intra_max;
        e.delay = (uint8_t)(dmin + (int)(((uint64_t)o.w[1] * (uint64_t)(dmax - dmin + 1)) >> 32));
        uint32_t slow_thr = (uint32_t)std::floor(sp.slow_frac * 4294967296.0);
        int slow = (o.w[2] < slow_thr) ? 1 : 0;       // NMDA / GABA_B w.p. slow_frac (R12)
        e.rec = (uint8_t)((inh ? 2 : 0) + slow);       // receptor class follows the SOURCE type
        return e;
    }
    void owner_edges(int64_t i, std::vector<Edge>& edges) const {
        const int R = sp.n_regions;
        const int64_t N = sp.N;
        if (sp.mode == 0) {
            // fixed in-degree K per target ("for each neuron, the number of
            // synaptic inputs from each neuron population ...")
            int r = region_of(region_start.data(), R, i);
            int64_t base = region_start[(size_t)r];
            int64_t size = region_start[(size_t)r + 1] - base;
            int64_t li = i - base;
            u32x4 k0 = draw(seed, STREAM_SRC, (uint64_t)i, 0);
            for (int k = 0; k < K_intra; ++k) {        // own region, any type, not self
                uint32_t j = prp((uint32_t)k, (uint32_t)(size - 1), k0.w);
                if ((int64_t)j >= li) j += 1;          // skip self: no autapse
                edges.push_back(make_edge(i, k, base + j, i, false));
            }
            u32x4 k1 = draw(seed, STREAM_SRC, (uint64_t)i, 1);
            for (int s = 0; s < K_inter; ++s) {        // other regions, excitatory only
                uint32_t u = draw(seed, STREAM_INTER, (uint64_t)i, (uint64_t)s).w[0];
                const uint32_t* T = &cdf[(size_t)r * (size_t)(R - 1)];
                int rs = 0;
                for (int m = 0; m < R - 1; ++m) if (u >= T[m]) ++rs;
                // distinct slots s map to distinct neurons of region rs (prp is injective)
                uint32_t j = prp((uint32_t)s, (uint32_t)region_nexc[(size_t)rs], k1.w);
                edges.push_back(make_edge(i, K_intra + s, region_start[(size_t)rs] + j, i, true));
            }
        } else {
            // lognormal out-degree per source, targets uniform without replacement (R27)
            int32_t deg = dtab[draw(seed, STREAM_DEG, (uint64_t)i, 0).w[0] >> 16];
            if ((int64_t)deg > N - 1) deg = (int32_t)(N - 1);
            u32x4 k0 = draw(seed, STREAM_SRC, (uint64_t)i, 0);
            for (int m = 0; m < deg; ++m) {
                uint32_t t = prp((uint32_t)m, (uint32_t)(N - 1), k0.w);
                if ((int64_t)t >= i) t += 1;
                edges.push_back(make_edge(i, m, i, t, false));
            }
        }
    }
};

orc_gen* orc_gen_create(const orc_net_spec* sp, uint64_t seed) {
    orc_gen* g = new orc_gen();
    g->sp = *sp; g->seed = seed;
    const int64_t N = sp->N;
    const int R = sp->n_regions;
    std::vector<int64_t> sizes((size_t)R);
    if (R == 1) sizes[0] = N; else orc_region_sizes(seed, N, R, sp->region_size_sigma, sizes.data());
    g->region_start.assign((size_t)R + 1, 0);
    g->region_nexc.assign((size_t)R, 0);
    for (int r = 0; r < R; ++r) {
        g->region_start[(size_t)r + 1] = g->region_start[(size_t)r] + sizes[(size_t)r];
        g->region_nexc[(size_t)r] = (int64_t)std::floor(sp->exc_frac * (double)sizes[(size_t)r] + 0.5);
    }
    g->wtab.resize(65536);
    orc_weight_table(sp->w_mu, sp->w_sigma, sp->w_scale, g->wtab.data());
    g->K_intra = sp->K; g->K_inter = 0;
    if (sp->mode == 0 && R > 1) {
        g->K_intra = (int)std::floor(sp->intra_frac * (double)sp->K + 0.5);
        g->K_inter = sp->K - g->K_intra;
        g->cdf.resize((size_t)R * (size_t)(R - 1));
        orc_region_cdf(seed, R, sp->region_matrix_sigma, g->cdf.data());
    }
    if (sp->mode == 1) {
        g->dtab.resize(65536);
        orc_outdeg_table(sp->outdeg_mean, sp->outdeg_sigma, sp->outdeg_cap, g->dtab.data());
    }
    return g;
}
void orc_gen_destroy(orc_gen* g) { delete g; }

// neuron type of neuron i (0 excitatory, 1 inhibitory): excitatory neurons come first in each region
int32_t orc_gen_ntype(const orc_gen* g, int64_t i) { return g->is_inh(i) ? 1 : 0; }

// The synapses owned by neuron i, in slot order (sampled parity at full size).
// Returns the count; writes at most cap entries.
int64_t orc_gen_owner_edges(const orc_gen* g, int64_t i, int64_t cap, int32_t* src, int32_t* tgt,
                            float* w, uint8_t* delay, uint8_t* rec) {
    std::vector<Edge> e;
    g->owner_edges(i, e);
    for (int64_t k = 0; k < (int64_t)e.size() && k < cap; ++k) {
        src[k] = e[(size_t)k].src; tgt[k] = e[(size_t)k].tgt; w[k] = e[(size_t)k].w;
        delay[k] = e[(size_t)k].delay; rec[k] = e[(size_t)k].rec;
    }
    return (int64_t)e.size();
}

// 1 if the spec can be generated: every region must hold the K_intra distinct
// non-self sources and the K_inter distinct excitatory sources a target draws
// from it ("without replacement"); otherwise prp() has no answer.
int32_t orc_gen_valid(const orc_gen* g) {
    const orc_net_spec& sp = g->sp;
    if (sp.N < 2 || sp.n_regions < 1) return 0;
    for (int r = 0; r < sp.n_regions; ++r) {
        int64_t size = g->region_start[(size_t)r + 1] - g->region_start[(size_t)r];
        if (sp.mode == 0 && size - 1 < g->K_intra) return 0;
        if (sp.mode == 0 && g->K_inter > 0 && g->region_nexc[(size_t)r] < g->K_inter) return 0;
    }
    return 1;
}

orc_network* orc_generate(const orc_net_spec* sp, uint64_t seed) {
    const int64_t N = sp->N;
    const int R = sp->n_regions;
    orc_gen* g = orc_gen_create(sp, seed);
    if (!orc_gen_valid(g)) { orc_gen_destroy(g); return nullptr; }
    orc_network* net = (orc_network*)std::calloc(1, sizeof(orc_network));
    net->N = N; net->n_regions = R;
    net->region_start = (int64_t*)std::calloc((size_t)R + 1, sizeof(int64_t));
    net->region_nexc = (int64_t*)std::calloc((size_t)R, sizeof(int64_t));
    net->ntype = (uint8_t*)std::calloc((size_t)N, 1);
    for (int r = 0; r <= R; ++r) net->region_start[r] = g->region_start[(size_t)r];
    for (int r = 0; r < R; ++r) net->region_nexc[r] = g->region_nexc[(size_t)r];
    for (int64_t i = 0; i < N; ++i) net->ntype[i] = g->is_inh(i) ? 1 : 0;

    std::vector<Edge> edges;
    for (int64_t i = 0; i < N; ++i) g->owner_edges(i, edges);
    orc_gen_destroy(g);

    // presynaptic-major CSR, rows sorted by target ---------------------------------
    std::sort(edges.begin(), edges.end(), [](const Edge& a, const Edge& b) {
        if (a.src != b.src) return a.src < b.src;
        if (a.tgt != b.tgt) return a.tgt < b.tgt;
        return a.rec < b.rec;
    });
    const int64_t E = (int64_t)edges.size();
    net->E = E;
    net->row_ptr = (int64_t*)std::calloc((size_t)N + 1, sizeof(int64_t));
    net->tgt = (int32_t*)std::malloc(sizeof(int32_t) * (size_t)std::max<int64_t>(E, 1));
    net->w = (float*)std::malloc(sizeof(float) * (size_t)std::max<int64_t>(E, 1));
    net->delay = (uint8_t*)std::malloc((size_t)std::max<int64_t>(E, 1));
    net->rec = (uint8_t*)std::malloc((size_t)std::max<int64_t>(E, 1));
    for (int64_t e = 0; e < E; ++e) {
        net->row_ptr[edges[(size_t)e].src + 1] += 1;
        net->tgt[e] = edges[(size_t)e].tgt; net->w[e] = edges[(size_t)e].w;
        net->delay[e] = edges[(size_t)e].delay; net->rec[e] = edges[(size_t)e].rec;
    }
    for (int64_t i = 0; i < N; ++i) net->row_ptr[i + 1] += net->row_ptr[i];
    return net;
}

// =============================================================================
// 4. The simulator.  `real` = float is the parity mode (fp32, fixed operation
//    order, no FMA: R-FP); `real` = double is used only for closed-form and
//    dt-convergence pins.
// =============================================================================
}  // extern "C"

namespace {

template <typename real>
struct TypeConst {
    real gL, VL, Vth, Vreset, kappa, Iext;
    real G[4], E[4], alpha[4];
    int32_t R;              // refractory steps
    int32_t wq_bg;
    uint32_t T[POISSON_MAX]; int M;
    bool ou = false;        // OU background current on
    double ix_shape = 0, ix_scale = 0;   // Gamma law of the per-neuron external current (0: constant)
    real ou_mu = 0, ou_a = 0, ou_s = 0;   // mean, dt/tau, sigma sqrt(2 dt/tau): formed in double, rounded once
};

template <typename real>
struct Sim {
    int64_t N = 0, E = 0;
    int D = 0, S = 0, window = 0, n_regions = 1;
    int bin = 1;                      // b_t in steps (R29)
    std::vector<int32_t> A;           // neurons that fired in the current time bin: the non-zero A_j of its boundary
    uint64_t seed = 0;
    uint64_t step = 0;
    std::vector<TypeConst<real>> tc;
    std::vector<uint8_t> ntype;
    std::vector<int64_t> region_start;
    // network (borrowed copies)
    std::vector<int64_t> row_ptr; std::vector<int32_t> tgt; std::vector<float> w;
    std::vector<uint8_t> delay, rec;
    // state
    std::vector<real> V, g;           // g[4*i+u]
    std::vector<real> Iou;            // OU background current (R3)
    std::vector<real> Iext;           // external current of every neuron (R31): a parameter, drawn once
    std::vector<float> ntab;          // 65536 standard-normal quantiles, Phi^-1((q + 0.5) / 65536), as fp32
    std::vector<int32_t> ref;
    std::vector<int32_t> ring;        // ring[(slot*N + i)*4 + u]
    // outputs
    std::vector<uint64_t> spike_step; std::vector<int32_t> spike_id;
    std::vector<uint32_t> region_count;   // [window][region]
    uint64_t n_events = 0, n_bg = 0;
    int32_t overflow = 0;
    bool log_arrivals = false;            // pins only: what step 1 consumed, [n][i][u]
    std::vector<uint8_t> spike_flag;      // scratch of one_step: neuron i was flagged in this step
    std::vector<int32_t> arrivals_log;

    void one_step() {
        const uint64_t n = step;
        const real scale = (real)std::ldexp(1.0, -S);
        int32_t* slot = &ring[(size_t)(n % (uint64_t)D) * (size_t)N * 4];
        std::vector<int32_t> L;                           // SpikeList (Alg. 2 line 2)
        // The loop body reads and writes neuron i's own state and ring cells only, so its iterations are independent:
        // built with -fopenmp (the all-cores timing leg of bench.py, liboracle_omp.so) they are shared among the host
        // cores -- same arithmetic, same results; the plain build runs them in order on one core.
        spike_flag.assign((size_t)N, 0);
        if (log_arrivals) arrivals_log.resize(arrivals_log.size() + (size_t)N * 4);
        int32_t* const alog = log_arrivals ? &arrivals_log[arrivals_log.size() - (size_t)N * 4] : nullptr;
        uint64_t bg_sum = 0;
        int32_t ovf = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : bg_sum) reduction(| : ovf)
#endif
        for (int64_t i = 0; i < N; ++i) {
            const TypeConst<real>& c = tc[ntype[(size_t)i]];
            // 1. arrivals due now; the slot is consumed
            int32_t a[4];
            for (int u = 0; u < 4; ++u) { a[u] = slot[i * 4 + u]; slot[i * 4 + u] = 0; }
            if (alog) for (int u = 0; u < 4; ++u) alog[i * 4 + u] = a[u];
            for (int u = 0; u < 4; ++u)
                if (a[u] > (1 << 30) || a[u] < -(1 << 30)) ovf |= 1;
            // 2. Poisson background into AMPA (R14); one Philox block serves 4 neurons
            uint32_t uu = draw(seed, STREAM_BG, (uint64_t)(i >> 2), n).w[i & 3];
            int k = poisson_count(uu, c.T, c.M);
            a[0] = (int32_t)((uint32_t)a[0] + (uint32_t)k * (uint32_t)c.wq_bg);
            bg_sum += (uint64_t)k;
            // 3. fixed point -> real
            real x[4];
            for (int u = 0; u < 4; ++u) x[u] = (real)a[u] * scale;
            // 4. synaptic current I_u = g_u (V_u - V) J_u, fixed summation order
            real v = V[(size_t)i];
            real* gi = &g[(size_t)i * 4];
            real t0 = (c.G[0] * gi[0]) * (c.E[0] - v);
            real t1 = (c.G[1] * gi[1]) * (c.E[1] - v);
            real t2 = (c.G[2] * gi[2]) * (c.E[2] - v);
            real t3 = (c.G[3] * gi[3]) * (c.E[3] - v);
            real I = (((t0 + t1) + t2) + t3) + Iext[(size_t)i];
            // 4b. OU background current (SI Eq.(4); R3): the membrane step sees I_ou(t), then
            //     I_ou(t+dt) = I_ou + ((mu - I_ou) dt/tau + sigma sqrt(2 dt/tau) xi); one Philox block serves 4
            //     neurons, xi = table[top 16 bits of the word]
            if (c.ou) {
                real io = Iou[(size_t)i];
                I = I + io;
                uint32_t uo = draw(seed, STREAM_OU, (uint64_t)(i >> 2), n).w[i & 3];
                real xi = (real)ntab[uo >> 16];
                Iou[(size_t)i] = io + ((c.ou_mu - io) * c.ou_a + c.ou_s * xi);
            }
            // 5. membrane step: CV equation with Euler step (SI Eq.(5); R1)
            real leak = (-c.gL) * (v - c.VL);
            real vn = v + c.kappa * (leak + I);
            // 6. conductances: exact exponential decay + arrivals (SI Eq.(3))
            for (int u = 0; u < 4; ++u) gi[u] = gi[u] * c.alpha[u] + x[u];
            // 7. refractory clamp / threshold / reset (R5, R6)
            int spike = 0;
            if (ref[(size_t)i] > 0) { vn = c.Vreset; ref[(size_t)i] -= 1; }
            else if (vn >= c.Vth) { spike = 1; vn = c.Vreset; ref[(size_t)i] = c.R; }
            V[(size_t)i] = vn;
            spike_flag[(size_t)i] = (uint8_t)spike;
        }
        n_bg += bg_sum;
        overflow |= ovf;
        for (int64_t i = 0; i < N; ++i) if (spike_flag[(size_t)i]) L.push_back((int32_t)i);
        // 8. record + region counts
        const size_t win = (size_t)(n / (uint64_t)window);
        if (region_count.size() < (win + 1) * (size_t)n_regions) region_count.resize((win + 1) * (size_t)n_regions, 0);
        for (int32_t j : L) {
            spike_step.push_back(n); spike_id.push_back(j);
            int r = 0;
            while (r + 1 < n_regions && region_start[(size_t)r + 1] <= j) ++r;
            region_count[win * (size_t)n_regions + (size_t)r] += 1;
        }
        // 9. accumulated spikes A_j (SI "Numerical method"; R29): a neuron that fires inside the time
        //    bin (t - b_t, t] is transferred at the boundary t = k b_t, once (A_j is 0 or 1).  In steps: the bin
        //    of step n closes at the end of the step n with (n + 1) mod b_t = 0; b_t = 1 step is the plain
        //    scheme (every step a boundary).
        for (int32_t j : L) {
            A.push_back(j);
            n_events += (uint64_t)(row_ptr[(size_t)j + 1] - row_ptr[(size_t)j]);   // counted when the spike is emitted
        }
        if ((n + 1) % (uint64_t)bin == 0) {
            // push delivery along the destination lists (Alg. 2 lines 3-4), w A_j(t) of Eq.(3)
            // (-fopenmp build: the spikes are shared among the cores and the additions are atomic; integer sums do not
            // depend on their order, so the ring is the same)
            const int64_t nA = (int64_t)A.size();
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16)
#endif
            for (int64_t k = 0; k < nA; ++k) {
                const int32_t j = A[(size_t)k];
                for (int64_t s = row_ptr[(size_t)j]; s < row_ptr[(size_t)j + 1]; ++s) {
                    int32_t wq = (int32_t)std::lrintf(w[(size_t)s] * (float)std::ldexp(1.0, S));
                    size_t sl = (size_t)((n + delay[(size_t)s]) % (uint64_t)D);
                    int32_t* cell = &ring[(sl * (size_t)N + (size_t)tgt[(size_t)s]) * 4 + rec[(size_t)s]];
#ifdef _OPENMP
                    __atomic_fetch_add(reinterpret_cast<uint32_t*>(cell), (uint32_t)wq, __ATOMIC_RELAXED);   // wraps the same way
#else
                    *cell = (int32_t)((uint32_t)*cell + (uint32_t)wq);      // two's-complement wrap
#endif
                }
            }
            A.clear();
        }
        step += 1;
    }
};

template <typename real>
Sim<real>* sim_create(const orc_sim_params* p, int64_t N, const uint8_t* ntype,
                      int32_t n_regions, const int64_t* region_start,
                      const int64_t* row_ptr, const int32_t* tgt, const float* w,
                      const uint8_t* delay, const uint8_t* rec, uint64_t seed) {
    Sim<real>* s = new Sim<real>();
    s->N = N; s->E = row_ptr[N]; s->D = p->D; s->S = p->S; s->window = p->window_steps;
    s->seed = seed; s->n_regions = n_regions;
    s->bin = p->spike_bin_steps > 1 ? p->spike_bin_steps : 1;
    s->ntype.assign(ntype, ntype + N);
    s->region_start.assign(region_start, region_start + n_regions + 1);
    s->row_ptr.assign(row_ptr, row_ptr + N + 1);
    s->tgt.assign(tgt, tgt + s->E); s->w.assign(w, w + s->E);
    s->delay.assign(delay, delay + s->E); s->rec.assign(rec, rec + s->E);
    for (int t = 0; t < p->n_types; ++t) {
        const orc_type_params& q = p->type[t];
        TypeConst<real> c;
        // constants are formed in double, then rounded once to `real`
        c.gL = (real)q.gL; c.VL = (real)q.VL; c.Vth = (real)q.Vth; c.Vreset = (real)q.Vreset;
        c.kappa = (real)(p->dt_ms / q.C); c.Iext = (real)q.Iext;
        for (int u = 0; u < 4; ++u) {
            c.G[u] = (real)q.G[u]; c.E[u] = (real)q.E[u];
            c.alpha[u] = (real)std::exp(-p->dt_ms / q.tau_ms[u]);
        }
        c.R = (int32_t)std::lrint(q.Tref_ms / p->dt_ms);
        c.wq_bg = (int32_t)std::lrint(q.bg_weight * std::ldexp(1.0, p->S));
        c.M = poisson_thresholds(q.bg_rate_hz * p->dt_ms * 1e-3, c.T);
        c.ix_shape = q.iext_gamma_shape; c.ix_scale = q.iext_gamma_scale;
        if (q.ou_tau_ms > 0) {
            c.ou = true;
            c.ou_mu = (real)q.ou_mu;
            c.ou_a = (real)(p->dt_ms / q.ou_tau_ms);
            c.ou_s = (real)(q.ou_sigma * std::sqrt(2.0 * p->dt_ms / q.ou_tau_ms));
        }
        s->tc.push_back(c);
    }
    s->ntab.resize(65536);
    for (int q = 0; q < 65536; ++q) s->ntab[(size_t)q] = (float)norm_ppf(((double)q + 0.5) / 65536.0);
    s->Iou.resize((size_t)N);
    for (int64_t i = 0; i < N; ++i) s->Iou[(size_t)i] = s->tc[ntype[i]].ou ? s->tc[ntype[i]].ou_mu : (real)0;
    // per-neuron external current (R31): Iext + table[top 16 bits of Philox(stream 9, neuron)], one fp32 addition
    s->Iext.resize((size_t)N);
    {
        std::vector<std::vector<float>> gtab(s->tc.size());
        for (size_t t = 0; t < s->tc.size(); ++t)
            if (s->tc[t].ix_shape > 0) {
                gtab[t].resize(65536);
                for (int q = 0; q < 65536; ++q) gtab[t][(size_t)q] = (float)gamma_ppf(((double)q + 0.5) / 65536.0, s->tc[t].ix_shape, s->tc[t].ix_scale);
            }
        for (int64_t i = 0; i < N; ++i) {
            const size_t t = ntype[i];
            real v = s->tc[t].Iext;
            if (s->tc[t].ix_shape > 0) v = v + (real)gtab[t][draw(seed, STREAM_IEXT, (uint64_t)i, 0).w[0] >> 16];
            s->Iext[(size_t)i] = v;
        }
    }
    s->V.resize((size_t)N); s->g.assign((size_t)N * 4, (real)0); s->ref.assign((size_t)N, 0);
    s->ring.assign((size_t)p->D * (size_t)N * 4, 0);
    for (int64_t i = 0; i < N; ++i) {
        const TypeConst<real>& c = s->tc[ntype[i]];
        uint32_t u = draw(seed, STREAM_V0, (uint64_t)i, 0).w[0];
        real U = (real)(u >> 8) * (real)std::ldexp(1.0, -24);
        s->V[(size_t)i] = c.Vreset + (c.Vth - c.Vreset) * U;
    }
    return s;
}

struct Handle { int fp64; Sim<float>* f; Sim<double>* d; };

}  // namespace

extern "C" {

void* orc_sim_create(const orc_sim_params* p, int64_t N, const uint8_t* ntype,
                     int32_t n_regions, const int64_t* region_start,
                     const int64_t* row_ptr, const int32_t* tgt, const float* w,
                     const uint8_t* delay, const uint8_t* rec, uint64_t seed, int32_t fp64) {
    Handle* h = new Handle{fp64, nullptr, nullptr};
    if (fp64) h->d = sim_create<double>(p, N, ntype, n_regions, region_start, row_ptr, tgt, w, delay, rec, seed);
    else      h->f = sim_create<float>(p, N, ntype, n_regions, region_start, row_ptr, tgt, w, delay, rec, seed);
    return h;
}
void orc_sim_destroy(void* hv) { Handle* h = (Handle*)hv; delete h->f; delete h->d; delete h; }

void orc_sim_get_iou(void* hv, double* out) {
    Handle* h = (Handle*)hv;
    const int64_t N = h->fp64 ? h->d->N : h->f->N;
    for (int64_t i = 0; i < N; ++i) out[i] = h->fp64 ? h->d->Iou[(size_t)i] : (double)h->f->Iou[(size_t)i];
}
void orc_sim_get_iext(void* hv, double* out) {
    Handle* h = (Handle*)hv;
    const int64_t N = h->fp64 ? h->d->N : h->f->N;
    for (int64_t i = 0; i < N; ++i) out[i] = h->fp64 ? h->d->Iext[(size_t)i] : (double)h->f->Iext[(size_t)i];
}
void orc_sim_set_iou(void* hv, const double* in) {
    Handle* h = (Handle*)hv;
    const int64_t N = h->fp64 ? h->d->N : h->f->N;
    for (int64_t i = 0; i < N; ++i) { if (h->fp64) h->d->Iou[(size_t)i] = in[i]; else h->f->Iou[(size_t)i] = (float)in[i]; }
}
void orc_normal_table(float* tab /*[65536]*/) {
    for (int q = 0; q < 65536; ++q) tab[q] = (float)norm_ppf(((double)q + 0.5) / 65536.0);
}

void orc_sim_step(void* hv, int64_t n_steps) {
    Handle* h = (Handle*)hv;
    for (int64_t k = 0; k < n_steps; ++k) { if (h->fp64) h->d->one_step(); else h->f->one_step(); }
}

#define BOTH(expr_f, expr_d) (h->fp64 ? (expr_d) : (expr_f))

uint64_t orc_sim_step_index(void* hv) { Handle* h = (Handle*)hv; return BOTH(h->f->step, h->d->step); }
uint64_t orc_sim_n_spikes(void* hv) { Handle* h = (Handle*)hv; return BOTH(h->f->spike_id.size(), h->d->spike_id.size()); }
uint64_t orc_sim_n_events(void* hv) { Handle* h = (Handle*)hv; return BOTH(h->f->n_events, h->d->n_events); }
uint64_t orc_sim_n_bg(void* hv) { Handle* h = (Handle*)hv; return BOTH(h->f->n_bg, h->d->n_bg); }
int32_t orc_sim_overflow(void* hv) { Handle* h = (Handle*)hv; return BOTH(h->f->overflow, h->d->overflow); }

void orc_sim_get_spikes(void* hv, uint64_t* steps, int32_t* ids) {
    Handle* h = (Handle*)hv;
    const std::vector<uint64_t>& st = h->fp64 ? h->d->spike_step : h->f->spike_step;
    const std::vector<int32_t>& id = h->fp64 ? h->d->spike_id : h->f->spike_id;
    std::copy(st.begin(), st.end(), steps); std::copy(id.begin(), id.end(), ids);
}

void orc_sim_log_arrivals(void* hv, int32_t on) { Handle* h = (Handle*)hv; if (h->fp64) h->d->log_arrivals = on; else h->f->log_arrivals = on; }
uint64_t orc_sim_get_arrivals(void* hv, int32_t* out) {     // [steps][N][4]; returns element count
    Handle* h = (Handle*)hv;
    const std::vector<int32_t>& a = h->fp64 ? h->d->arrivals_log : h->f->arrivals_log;
    if (out) std::copy(a.begin(), a.end(), out);
    return a.size();
}

// state as double (exact for the fp32 mode): V[N], g[N][4]; ref[N]
void orc_sim_get_state(void* hv, double* V, double* g, int32_t* ref) {
    Handle* h = (Handle*)hv;
    int64_t N = BOTH(h->f->N, h->d->N);
    for (int64_t i = 0; i < N; ++i) {
        V[i] = BOTH((double)h->f->V[(size_t)i], h->d->V[(size_t)i]);
        for (int u = 0; u < 4; ++u) g[i * 4 + u] = BOTH((double)h->f->g[(size_t)i * 4 + u], h->d->g[(size_t)i * 4 + u]);
        ref[i] = BOTH(h->f->ref[(size_t)i], h->d->ref[(size_t)i]);
    }
}
void orc_sim_set_state(void* hv, const double* V, const double* g, const int32_t* ref) {
    Handle* h = (Handle*)hv;
    int64_t N = BOTH(h->f->N, h->d->N);
    for (int64_t i = 0; i < N; ++i) {
        if (h->fp64) h->d->V[(size_t)i] = V[i]; else h->f->V[(size_t)i] = (float)V[i];
        for (int u = 0; u < 4; ++u) {
            if (h->fp64) h->d->g[(size_t)i * 4 + u] = g[i * 4 + u]; else h->f->g[(size_t)i * 4 + u] = (float)g[i * 4 + u];
        }
        if (h->fp64) h->d->ref[(size_t)i] = ref[i]; else h->f->ref[(size_t)i] = ref[i];
    }
}
// ring[D][N][4] int32
void orc_sim_get_ring(void* hv, int32_t* out) {
    Handle* h = (Handle*)hv;
    const std::vector<int32_t>& r = h->fp64 ? h->d->ring : h->f->ring;
    std::copy(r.begin(), r.end(), out);
}
void orc_sim_set_ring(void* hv, const int32_t* in) {
    Handle* h = (Handle*)hv;
    std::vector<int32_t>& r = h->fp64 ? h->d->ring : h->f->ring;
    std::copy(in, in + r.size(), r.begin());
}
// spike counts per (window, region); returns number of windows available
int64_t orc_sim_region_counts(void* hv, uint32_t* out, int64_t cap_windows) {
    Handle* h = (Handle*)hv;
    const std::vector<uint32_t>& rc = h->fp64 ? h->d->region_count : h->f->region_count;
    int R = BOTH(h->f->n_regions, h->d->n_regions);
    int64_t nw = (int64_t)(rc.size() / (size_t)R);
    int64_t m = std::min(nw, cap_windows);
    if (out) std::copy(rc.begin(), rc.begin() + (size_t)(m * R), out);
    return nw;
}

// =============================================================================
// 5. Dense brute force: the plain definition of what delivery sums (R-DENSE).
//    arrivals[n][i][u] = sum_j Wq[u][i][j] * spike_j(n - d[i][j]), with the
//    dense matrices built from the CSR and spikes given as a [T][N] 0/1 array.
//    Integer arithmetic; must equal what the ring delivered, exactly.
// =============================================================================
void orc_dense_arrivals(int64_t N, int64_t T, int32_t S, const int64_t* row_ptr, const int32_t* tgt,
                        const float* w, const uint8_t* delay, const uint8_t* rec,
                        const uint8_t* spikes /*[T][N]*/, int64_t* arrivals /*[T][N][4]*/) {
    std::vector<int64_t> Wq((size_t)4 * (size_t)N * (size_t)N, 0);
    std::vector<int32_t> dd((size_t)N * (size_t)N, 0);
    for (int64_t j = 0; j < N; ++j)
        for (int64_t s = row_ptr[j]; s < row_ptr[j + 1]; ++s) {
            int64_t i = tgt[s];
            Wq[((size_t)rec[s] * (size_t)N + (size_t)i) * (size_t)N + (size_t)j] +=
                (int64_t)std::lrintf(w[s] * (float)std::ldexp(1.0, S));
            dd[(size_t)i * (size_t)N + (size_t)j] = delay[s];
        }
    for (int64_t n = 0; n < T; ++n)
        for (int64_t i = 0; i < N; ++i)
            for (int u = 0; u < 4; ++u) {
                int64_t acc = 0;
                for (int64_t j = 0; j < N; ++j) {
                    int64_t d = dd[(size_t)i * (size_t)N + (size_t)j];
                    if (d == 0 || n - d < 0) continue;
                    acc += Wq[((size_t)u * (size_t)N + (size_t)i) * (size_t)N + (size_t)j] *
                           (int64_t)spikes[(size_t)(n - d) * (size_t)N + (size_t)j];
                }
                arrivals[((size_t)n * (size_t)N + (size_t)i) * 4 + (size_t)u] = acc;
            }
}

}  // extern "C"
