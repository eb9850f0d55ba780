// Step kernels: neuron update + spike compaction (a1, a2, a4) and spike
// delivery (a3), as two kernels per step or as one persistent cooperative
// kernel.  Compiled with -fmad=false; every floating-point operation of the
// state update is an explicit round-to-nearest intrinsic in the fixed order of
// DESIGN.md "Arithmetic contract", so the fp32 state is bit-identical to a
// strict IEEE evaluation of the same expressions.
//
// Paper: SI Eq.(3) P:L475 (conductances), CV equation P:L382 + SI Eq.(5)
// (membrane), P:L108 / P:L481-482 (threshold, reset, refractory), Supp. Alg. 2
// P:L879-884 and P:L490 (push delivery with atomics along the destination list).
#include <algorithm>
#include <cuda_fp16.h>
#include <cooperative_groups.h>
#include "db_device.cuh"
#include "db_philox.cuh"

namespace cg = cooperative_groups;

namespace dbk {

// ---------------------------------------------------------------------------
// memory helpers: streaming 128-bit accesses that do not pollute L1
// ---------------------------------------------------------------------------
__device__ __forceinline__ int4 ld_stream_i4(const int32_t* p) {
    int4 r;
    asm volatile("ld.global.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ld_stream_f4(const float* p) {
    float4 r;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream_f4(float* p, float4 v) {
    asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void st_stream_i4(int32_t* p, int4 v) {
    asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void red_add_s32(int32_t* p, int32_t v) {
    asm volatile("red.global.add.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

// Region-count windows are cleared this many windows ahead of the one that is being closed: far
// enough that no block (up to three steps ahead of the step being logged) writes into it yet.
__device__ __forceinline__ unsigned window_clear_ahead(const int window_steps) { return 2u / (unsigned)window_steps + 1u; }

// Step whose end transfers the spikes of step n: the last step of n's time bin (R29); n itself when b_t = 1.
__device__ __forceinline__ unsigned long long transfer_step(const SimDev& p, const unsigned long long n) {
    if (p.bin_steps == 1) return n;
    const unsigned long long b = (unsigned long long)p.bin_steps;
    return n - n % b + (b - 1ull);
}

// The same for the persistent kernel, low word only (slots are taken modulo the power of two D), from the phase of
// the launch's first step (32-bit arithmetic: no 64-bit division on the spike path).
template <bool kBin>
__device__ __forceinline__ unsigned transfer_step_lo(const SimDev& p, const unsigned n_lo, const unsigned n0_lo,
                                                     const unsigned phase0) {
    if (!kBin) return n_lo;
    const unsigned b = (unsigned)p.bin_steps;
    return n_lo - (phase0 + (n_lo - n0_lo)) % b + (b - 1u);
}

__device__ __forceinline__ int region_of(const SimDev& p, int i) {
    int lo = 0, hi = p.n_regions;                 // region_start[lo] <= i < region_start[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(p.region_start + mid) <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// ---------------------------------------------------------------------------
// a3: one work item = up to kChunk consecutive synapses of one spiking neuron's
// row, handled by one warp; each lane takes 4 synapses per 128-bit load.
// ---------------------------------------------------------------------------
template <bool kHalf>
__device__ __forceinline__ void deliver_item(const SimDev& p, const unsigned long long n,
                                             const int2 wk, const unsigned lane) {
    const int j = wk.x;
    const int64_t rb = __ldg(p.row_begin + j) + (int64_t)wk.y * kChunk;
    int len = __ldg(p.row_len + j) - wk.y * kChunk;
    len = len < kChunk ? len : kChunk;
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    const unsigned nlo = (unsigned)n;
    constexpr int kIter = kChunk / 128;
    uint4 tr[kIter];
    float4 wv[kIter];
    uchar4 dl[kIter];
#pragma unroll
    for (int it = 0; it < kIter; ++it) {
        const int e = it * 128 + (int)lane * 4;
        if (e < len) {
            tr[it] = __ldg(reinterpret_cast<const uint4*>(p.tgt_rec + rb + e));
            dl[it] = __ldg(reinterpret_cast<const uchar4*>(p.delay + rb + e));
            if (kHalf) {
                const uint2 h = __ldg(reinterpret_cast<const uint2*>(static_cast<const __half*>(p.w) + rb + e));
                const __half2 h0 = *reinterpret_cast<const __half2*>(&h.x);
                const __half2 h1 = *reinterpret_cast<const __half2*>(&h.y);
                wv[it] = make_float4(__low2float(h0), __high2float(h0), __low2float(h1), __high2float(h1));
            } else {
                wv[it] = __ldg(reinterpret_cast<const float4*>(static_cast<const float*>(p.w) + rb + e));
            }
        }
    }
#pragma unroll
    for (int it = 0; it < kIter; ++it) {
        const int e = it * 128 + (int)lane * 4;
        if (e < len) {
            const unsigned t4[4] = {tr[it].x, tr[it].y, tr[it].z, tr[it].w};
            const float w4[4] = {wv[it].x, wv[it].y, wv[it].z, wv[it].w};
            const unsigned d4[4] = {dl[it].x, dl[it].y, dl[it].z, dl[it].w};
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (e + k < len) {
                    const int wq = __float2int_rn(__fmul_rn(w4[k], p.wscale));
                    const unsigned sl = (nlo + d4[k]) & Dm;
                    const unsigned rec = t4[k] >> 30, tg = t4[k] & 0x3FFFFFFFu;
                    red_add_s32(p.ring + ((size_t)sl * 4 + rec) * Np + tg, wq);
                }
        }
    }
}

// End of step n: publish the bookkeeping (one thread).  The counter cell of
// step n is cleared here and next used by step n + 2; the region-count window
// that starts two windows ahead is cleared one window early, so this may run
// concurrently with the update of step n + 1 (persistent mode).
__device__ __forceinline__ void finalize_step(const SimDev& p, const unsigned long long n,
                                              const unsigned long long counts) {
    Ctl* c = p.ctl;
    const unsigned long long end = c->spike_begin + (counts >> 32);
    c->spike_begin = end;
    c->spike_cursor = end;
    p.step_end[n & p.step_log_mask] = end;
    c->step_counts[(n + 2ull) & 3ull] = 0ull;            // the cell of step n - 2: every kernel of that step is done; next used by step n + 2
    if ((n + 1) % (unsigned long long)p.window_steps == 0) {
        const unsigned w = (unsigned)(((n + 1) / (unsigned long long)p.window_steps + window_clear_ahead(p.window_steps)) % p.max_windows);
        for (int r = 0; r < p.n_regions; ++r) p.region_counts[(size_t)w * p.n_regions + r] = 0u;
    }
    c->step = n + 1;
}

// ===========================================================================
// Mode DB_EXEC_KERNELS: two kernels per step.
// ===========================================================================
template <bool kHalf>
__global__ void __launch_bounds__(256) k_deliver(const __grid_constant__ SimDev p) {
    const unsigned long long n = p.ctl->step;
    const unsigned long long counts = p.ctl->step_counts[n & 3ull];
    const unsigned n_work = (unsigned)counts;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const unsigned long long nt = transfer_step(p, n);       // slot of a synapse = nt + delay
    const int2* const work = p.work + (size_t)(n & 1ull) * p.work_half;
    for (unsigned q = warp; q < n_work; q += n_warps) deliver_item<kHalf>(p, nt, work[q], lane);
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned ticket = atomicAdd(&p.ctl->done_blocks, 1u);
        if (ticket == gridDim.x - 1) {            // every block has read n / counts: safe to advance
            p.ctl->done_blocks = 0u;
            finalize_step(p, n, counts);
        }
    }
}

// ===========================================================================
// Mode DB_EXEC_PERSISTENT: one cooperative kernel runs all the steps, one block
// per SM.  Every block owns a fixed, contiguous range of 128-neuron tasks, so a
// thread meets the same neurons in every step.
//
// Software pipeline across the step boundary.  The membrane step is fully
// explicit (SI Eq.(5) takes J at time t, R8): V(n+1) and the spike decision of
// step n depend on the state after step n-1 only, NOT on the arrivals consumed
// in step n; only g(n+1) = alpha g(n) + x(n) needs ring slot n.  A step is
// therefore split into
//   A_n: V(n) -> V(n+1), refractory / threshold / reset, spike list L_n, and the
//        push of L_n along its rows into slots n + d          (needs g(n))
//   B_n: consume slot n, g(n) -> g(n+1)                       (needs L_m, m < n)
// and the kernel runs "units": unit 0 = A_n0, unit j = B_(n0+j-1) then A_(n0+j)
// in ONE pass over the data (same bytes as an unfused step), unit n_steps =
// B_(n0+n_steps-1).  The result is the oracle's, operation for operation.
// Unit j+1 needs only the deliveries of units <= j-1, so a block waits on a
// monotonic arrival counter for "everyone has finished unit j-1" while it may
// itself run a whole unit ahead: the barrier latency and the tail of the
// deliveries are off the critical path.  Slots written by the fastest block
// (up to n+1+d_max) must not meet the slot the slowest still consumes (n-1):
// the ring depth is kept >= d_max + 3 (+ b_t - 1 with a time bin for transferring spikes).
//
// All global->SM traffic of the update is staged through shared memory with
// cp.async (16 bytes per thread and plane: ring x4, V, g x4, rt), which keeps
// the loaded data out of the register file; while plane u of a task is
// consumed, plane u of the warp's next task is requested into the same cells,
// and the state planes of the first task of the next unit are requested before
// the wait.  Spikes are pushed by the warp that found them; rows longer than
// kInlineMax are shared by the warps of the block at the end of the unit.
// The raster is written through one global cursor with a step tag per entry
// (entries of adjacent steps may interleave); per-step counts go to
// Ctl::unit_spikes and are folded into the step log by block 0.
// ===========================================================================
struct alignas(16) TypeSmem {        // TypeConst regrouped into 128-bit words for broadcast LDS.128
    float4 rec[4];                   // per receptor u: G_u, E_u, alpha_u, -
    float4 m0;                       // neg_gL, VL, kappa, Iext
    float4 m1;                       // Vth, Vreset, R (int bits), wq_bg (int bits)
    uint4 m2;                        // M, T[0], T[1], T[2] (0xFFFFFFFF where m >= M)
    float4 m3;                       // OU background: mu, dt / tau, sigma sqrt(2 dt / tau), on (int bits)
};

constexpr int kStageBytesPerThread = 9 * 16 + 8;   // ring x4, V, g x4 (16 B each), rt (8 B)
constexpr uint32_t kPlaneStride = kRunThreads * 16;   // bytes between staging planes (fixed: immediate offsets)
constexpr int kStageBytes = kRunThreads * kStageBytesPerThread;

__device__ __forceinline__ unsigned ld_cg_u32(const unsigned* p) {
    unsigned r;
    asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long r;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(r) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ uint4 ld_cg_u4(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
// cache-streaming accesses (evict-first in L2): data that is read or written once and must not push the hot ring window out
__device__ __forceinline__ uint4 ld_cs_u4(const uint4* p) {
    uint4 r;
    asm volatile("ld.global.cs.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_cs_u2(uint2* p, const uint2 v) {
    asm volatile("st.global.cs.v2.u32 [%0], {%1,%2};" :: "l"(p), "r"(v.x), "r"(v.y) : "memory");
}
__device__ __forceinline__ float4 ld_cg_f4(const float* p) {
    float4 r;
    asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_cg_f4(float* p, float4 v) {
    asm volatile("st.global.cg.v4.f32 [%0], {%1,%2,%3,%4};" :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ void st_cg_i4(int32_t* p, int4 v) {
    asm volatile("st.global.cg.v4.s32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void cp_async16(const uint32_t smem, const void* g) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(smem), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async8(const uint32_t smem, const void* g) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(smem), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ uint4 lds128(const uint32_t smem) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(smem) : "memory");
    return r;
}
__device__ __forceinline__ uint2 lds64(const uint32_t smem) {
    uint2 r;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(smem) : "memory");
    return r;
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned r;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(r) : "l"(p) : "memory");
    return r;
}
// Spin until every block has finished unit u of this launch: counter [u & 3] collects the arrivals
// of the units u, u + 4, ... and only grows, so "all G blocks finished unit u" is count >= (u/4 + 1) G.
__device__ __forceinline__ void bar_wait(const unsigned* bar, const unsigned u, const unsigned G) {
    const unsigned* word = bar + (u & 3u);
    const unsigned target = (u / 4u + 1u) * G;
    while (ld_acquire_u32(word) < target) __nanosleep(20);
}

// Push one row (or one chunk of a row): 4 synapses per lane and 128-bit load,
// two batches of loads in flight before the first reduction is issued.
template <bool kHalf>
__device__ __forceinline__ void deliver_span(const SimDev& p, const unsigned nlo, const int64_t rb, const int len,
                                             const unsigned lane) {
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    for (int base = 0; base < len; base += 256) {
        uint4 tr[2];
        float4 wv[2];
        uchar4 dl[2];
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int e = base + it * 128 + (int)lane * 4;
            if (e < len) {
                tr[it] = __ldg(reinterpret_cast<const uint4*>(p.tgt_rec + rb + e));
                dl[it] = __ldg(reinterpret_cast<const uchar4*>(p.delay + rb + e));
                if (kHalf) {
                    const uint2 h = __ldg(reinterpret_cast<const uint2*>(static_cast<const __half*>(p.w) + rb + e));
                    const __half2 h0 = *reinterpret_cast<const __half2*>(&h.x);
                    const __half2 h1 = *reinterpret_cast<const __half2*>(&h.y);
                    wv[it] = make_float4(__low2float(h0), __high2float(h0), __low2float(h1), __high2float(h1));
                } else {
                    wv[it] = __ldg(reinterpret_cast<const float4*>(static_cast<const float*>(p.w) + rb + e));
                }
            }
        }
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int e = base + it * 128 + (int)lane * 4;
            if (e < len) {
                const unsigned t4[4] = {tr[it].x, tr[it].y, tr[it].z, tr[it].w};
                const float w4[4] = {wv[it].x, wv[it].y, wv[it].z, wv[it].w};
                const unsigned d4[4] = {dl[it].x, dl[it].y, dl[it].z, dl[it].w};
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (e + k < len) {
                        const int wq = __float2int_rn(__fmul_rn(w4[k], p.wscale));
                        const unsigned sl = (nlo + d4[k]) & Dm;
                        const unsigned rec = t4[k] >> 30, tg = t4[k] & 0x3FFFFFFFu;
                        red_add_s32(p.ring + ((size_t)sl * 4 + rec) * Np + tg, wq);
                    }
            }
        }
    }
}

struct RunCfg { unsigned n_steps; int n_tasks; int tasks_per_block; int iters; };

// Shared-memory staging cells of one thread: plane k at sbase + k * kPlaneStride (k = 0..3 ring,
// 4 V, 5..8 g), rt at srt.
struct Stage { uint32_t sbase, srt; };

__device__ __forceinline__ void request_state(const SimDev& p, const Stage& sg, const int i0) {
    const size_t Np = (size_t)p.Npad;
    cp_async16(sg.sbase + 4u * kPlaneStride, p.V + i0);
    cp_async8(sg.srt, p.rt + i0);
#pragma unroll
    for (int u = 0; u < 4; ++u) cp_async16(sg.sbase + (unsigned)(5 + u) * kPlaneStride, p.g + u * Np + i0);
}
__device__ __forceinline__ void request_ring(const SimDev& p, const Stage& sg, const int32_t* slot_i0) {
    const size_t Np = (size_t)p.Npad;
#pragma unroll
    for (int u = 0; u < 4; ++u) cp_async16(sg.sbase + (unsigned)u * kPlaneStride, slot_i0 + u * Np);
}

// The four neurons of one thread, receptor by receptor, out of the staging cells.
//   kB: consume the ring planes of step nB (slot), add the Poisson background, g <- g alpha + x, store g
//   kA: membrane step with the (new) g, refractory / threshold / reset, store V and rt; returns spike bits
// While plane u is consumed the same plane of the next task (next_off neurons further, if != 0)
// is requested (ring planes only if kB).  tp0..tp3 are the neuron types; the caller passes the
// same variable four times when they agree, which lets the constant loads (broadcast LDS.128)
// be shared.  Operation order: DESIGN.md "Arithmetic contract".
template <bool kB, bool kA, bool kClassic = false, bool kOU = false>
__device__ __forceinline__ unsigned neuron_group(const SimDev& p, const TypeSmem* s_tc,
                                                 const uint32_t (*s_T)[kPoissonMax], const Stage& sg,
                                                 const int tp0, const int tp1, const int tp2, const int tp3,
                                                 const int i0, int32_t* slot, const int next_off,
                                                 const uint4 v_bits, const uint2 rt_bits, const uint4 rnd,
                                                 unsigned& bg_acc, float4* iou = nullptr,
                                                 const float4 xi_ou = make_float4(0.0f, 0.0f, 0.0f, 0.0f),
                                                 const float4 ix = make_float4(0.0f, 0.0f, 0.0f, 0.0f)) {
    const size_t Np = (size_t)p.Npad;
    const int tp[4] = {tp0, tp1, tp2, tp3};
    const uint32_t rw[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
    const float v[4] = {__uint_as_float(v_bits.x), __uint_as_float(v_bits.y), __uint_as_float(v_bits.z),
                        __uint_as_float(v_bits.w)};
    const bool tail = (i0 + 3) >= p.N;              // only the last group can hold padding neurons
    float I[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        uint4 ab = make_uint4(0u, 0u, 0u, 0u);
        if (kB) ab = lds128(sg.sbase + (unsigned)u * kPlaneStride);
        const uint4 gb = lds128(sg.sbase + (unsigned)(5 + u) * kPlaneStride);
        if (next_off) {
            if (kB) cp_async16(sg.sbase + (unsigned)u * kPlaneStride, slot + u * Np + next_off);
            cp_async16(sg.sbase + (unsigned)(5 + u) * kPlaneStride, p.g + u * Np + i0 + next_off);
        }
        float gn[4] = {__uint_as_float(gb.x), __uint_as_float(gb.y), __uint_as_float(gb.z), __uint_as_float(gb.w)};
        // kClassic (whole step n in one pass, two-kernel mode): the membrane step sees g(n), the value loaded
        const float gc[4] = {gn[0], gn[1], gn[2], gn[3]};
        if (kB) {
            int a[4] = {(int)ab.x, (int)ab.y, (int)ab.z, (int)ab.w};
            if ((a[0] | a[1] | a[2] | a[3]) != 0) {  // consumed: zero the cells again, check the overflow bound
                st_cg_i4(slot + u * Np, make_int4(0, 0, 0, 0));
                const int lim = 1 << 30;
                if (a[0] > lim || a[0] < -lim || a[1] > lim || a[1] < -lim ||
                    a[2] > lim || a[2] < -lim || a[3] > lim || a[3] < -lim) p.ctl->overflow = 1u;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (u == 0) {           // Poisson background joins the AMPA arrivals (R14)
                    // k = #{m < M : u >= T_m}; thresholds increase, so the first three decide almost always
                    // m2.y / z / w hold 2^32 - T_m: u >= T_m is the carry of u + (2^32 - T_m)
                    const uint4 m2 = s_tc[tp[q]].m2;
                    unsigned k, scratch;
                    asm("add.cc.u32 %1, %2, %3;\n\taddc.u32 %0, 0, 0;\n\t"
                        "add.cc.u32 %1, %2, %4;\n\taddc.u32 %0, %0, 0;\n\t"
                        "add.cc.u32 %1, %2, %5;\n\taddc.u32 %0, %0, 0;"
                        : "=r"(k), "=r"(scratch) : "r"(rw[q]), "r"(m2.y), "r"(m2.z), "r"(m2.w));
                    if (k == 3u) {
                        if (m2.x > 3u) { while (k < m2.x && rw[q] >= s_T[tp[q]][k]) ++k; }
                        else k = m2.x;  // padded thresholds (u = 0xFFFFFFFF) do not count
                    }
                    if (tail && (i0 + q) >= p.N) k = 0u;
                    bg_acc += k;
                    a[q] = (int)((unsigned)a[q] + k * (unsigned)__float_as_int(s_tc[tp[q]].m1.w));
                }
                const float x = __fmul_rn(__int2float_rn(a[q]), p.scale);
                gn[q] = __fadd_rn(__fmul_rn(gn[q], s_tc[tp[q]].rec[u].z), x);
            }
            st_cg_f4(p.g + u * Np + i0, make_float4(gn[0], gn[1], gn[2], gn[3]));
        }
        if (kA) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 r = s_tc[tp[q]].rec[u];
                const float t = __fmul_rn(__fmul_rn(r.x, kClassic ? gc[q] : gn[q]), __fsub_rn(r.y, v[q]));
                I[q] = (u == 0) ? t : __fadd_rn(I[q], t);
            }
        }
    }
    unsigned spike_bits = 0;
    if (kA) {
        unsigned rt[4] = {rt_bits.x & 0xFFFFu, rt_bits.x >> 16, rt_bits.y & 0xFFFFu, rt_bits.y >> 16};
        float vn[4];
        unsigned rt_changed = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float4 m0 = s_tc[tp[q]].m0, m1 = s_tc[tp[q]].m1;
            // external current: the neuron's own (R31, when the plane exists) or the constant of its type
            const float ie = p.iext ? ((q == 0) ? ix.x : (q == 1) ? ix.y : (q == 2) ? ix.z : ix.w) : m0.w;
            float Iq = __fadd_rn(I[q], ie);
            if (kOU) {                 // OU background current (R3): the membrane step sees I_ou(t); then
                const float4 m3 = s_tc[tp[q]].m3;   // I_ou += (mu - I_ou) dt/tau + sigma sqrt(2 dt/tau) xi
                if (__float_as_int(m3.w)) {
                    float* io = reinterpret_cast<float*>(iou) + q;
                    const float xi = (q == 0) ? xi_ou.x : (q == 1) ? xi_ou.y : (q == 2) ? xi_ou.z : xi_ou.w;
                    Iq = __fadd_rn(Iq, *io);
                    *io = __fadd_rn(*io, __fadd_rn(__fmul_rn(__fsub_rn(m3.x, *io), m3.y), __fmul_rn(m3.z, xi)));
                }
            }
            const float leak = __fmul_rn(m0.x, __fsub_rn(v[q], m0.y));
            float w = __fadd_rn(v[q], __fmul_rn(m0.z, __fadd_rn(leak, Iq)));
            if ((rt[q] & (unsigned)kRefMask) > 0u) { w = m1.y; rt[q] -= 1u; rt_changed = 1u; }
            else if (w >= m1.x) {
                const unsigned R = (unsigned)__float_as_int(m1.z);
                w = m1.y; rt[q] |= R; rt_changed |= (unsigned)(R != 0u);
                if (!tail || (i0 + q) < p.N) spike_bits |= 1u << q;
            }
            vn[q] = w;
        }
        st_cg_f4(p.V + i0, make_float4(vn[0], vn[1], vn[2], vn[3]));
        if (rt_changed) *reinterpret_cast<uint2*>(p.rt + i0) = make_uint2(rt[0] | (rt[1] << 16), rt[2] | (rt[3] << 16));
    }
    return spike_bits;
}

constexpr int kSpkCap = 1024;        // spikes one block can stage per unit; beyond that the finder reserves raster positions itself
constexpr int kHeavyListCap = 512;   // heavy rows one block can defer per unit; beyond that the finder pushes them itself

struct BlockShared {                 // small per-block scratch of the persistent kernel
    unsigned unit_spikes[2];         // [unit & 1] spikes found by this block in the unit
    unsigned staged[2];              // [unit & 1] how many of them wait in spk[] for their raster position
    unsigned long long events;       // synaptic events of this block's spikes (whole launch)
    int spk[2][kSpkCap];             // [unit & 1] spikes of the unit, copied to the raster after the unit's barrier
    unsigned done[2];                // [unit & 1] update warps that have finished the unit (networks without heavy rows)
    unsigned grid_ok;                // units up to this one may start: the grid has closed everything they depend on
    unsigned heavy_n[2];             // [unit & 1] deferred heavy rows of the unit
    unsigned n0_lo, bin_phase0;      // step at launch (low word) and its position inside its time bin (R29)
    int heavy_row[2][kHeavyListCap];
};

// One 128-neuron task of one warp in unit (kB: B of step nB, kA: A of step nA).  next_off != 0:
// distance (in neurons) to the warp's next task of this unit, whose planes are requested while
// this one is consumed.
template <bool kHalf, bool kHeavy, bool kB, bool kA, bool kOU, bool kBin>
__device__ __forceinline__ void run_task(const SimDev& p, const TypeSmem* s_tc, const uint32_t (*s_T)[kPoissonMax],
                                         BlockShared* bs, const Stage& sg, const unsigned long long nB,
                                         const unsigned long long nA, const int task, const unsigned lane,
                                         const int next_off, unsigned& bg_acc) {
    const int grp = task * 32 + (int)lane;
    const int i0 = grp * 4;
    const size_t Np = (size_t)p.Npad;
    int32_t* slot = p.ring + (size_t)(nB & (unsigned long long)(p.D - 1)) * 4 * Np + i0;
    // one Philox block serves the four neurons (word q -> neuron i0 + q); drawn while the copies fly
    uint4 rnd = make_uint4(0u, 0u, 0u, 0u);
    if (kB && (!kOU || p.bg_on))       // (with the OU drive the Poisson background is usually off: no draw then)
        rnd = philox4x32_10_rk(make_uint4((uint32_t)(grp + (p.id0 >> 2)), kStreamBG << 24, (uint32_t)nB, (uint32_t)(nB >> 32)), p.rk);
    float4 iou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    float4 rnd_ou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    const bool ou = kOU && kA;
    if (ou) {                          // OU current of the four neurons and their N(0,1) draws (quantile table, top 16 bits of
        iou = ld_cg_f4(p.Iou + i0);    // a Philox word each); gathered here so that the latency hides behind the staged copies
        const uint4 wo = philox4x32_10_rk(make_uint4((uint32_t)(grp + (p.id0 >> 2)), kStreamOU << 24, (uint32_t)nA, (uint32_t)(nA >> 32)), p.rk);
        rnd_ou = make_float4(__ldg(p.ntab + (wo.x >> 16)), __ldg(p.ntab + (wo.y >> 16)), __ldg(p.ntab + (wo.z >> 16)),
                             __ldg(p.ntab + (wo.w >> 16)));
    }
    float4 ix = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (kA && p.iext) ix = ld_cg_f4(p.iext + i0);   // per-neuron external currents (R31): one more plane, read only
    cp_async_wait_all();
    const uint4 v_bits = lds128(sg.sbase + 4u * kPlaneStride);
    const uint2 rt_bits = lds64(sg.srt);
    if (next_off) {
        cp_async16(sg.sbase + 4u * kPlaneStride, p.V + i0 + next_off);
        cp_async8(sg.srt, p.rt + i0 + next_off);
    }
    const int tp0 = (int)((rt_bits.x >> 12) & 0xFu), tp1 = (int)(rt_bits.x >> 28);
    const int tp2 = (int)((rt_bits.y >> 12) & 0xFu), tp3 = (int)(rt_bits.y >> 28);
    unsigned spike_bits;
    if (tp0 == tp1 && tp0 == tp2 && tp0 == tp3)
        spike_bits = neuron_group<kB, kA, false, kOU>(p, s_tc, s_T, sg, tp0, tp0, tp0, tp0, i0, slot, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou, ix);
    else                                // a type boundary inside the group (rare)
        spike_bits = neuron_group<kB, kA, false, kOU>(p, s_tc, s_T, sg, tp0, tp1, tp2, tp3, i0, slot, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou, ix);
    if (ou) st_cg_f4(p.Iou + i0, iou);
    cp_async_commit();
    if (!kA) return;

    // ---- a2 + a4 + a3: spikes are rare (rate * dt per neuron-step); whole warps skip this
    unsigned any = __ballot_sync(0xffffffffu, spike_bits != 0);
    if (any == 0) return;
    int len[4] = {0, 0, 0, 0};
    int64_t rb[4] = {0, 0, 0, 0};
    unsigned my_events = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if (spike_bits & (1u << q)) {
            len[q] = __ldg(p.row_len + p.id0 + i0 + q);      // rows are keyed by the global id of the source
            rb[q] = __ldg(p.row_begin + p.id0 + i0 + q);
            my_events += (unsigned)len[q];
        }
    const unsigned my_spk = (unsigned)__popc(spike_bits);
    unsigned inc = my_spk;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= (unsigned)d) inc += o;
    }
    const unsigned tot = __shfl_sync(0xffffffffu, inc, 31);
    const unsigned ev_warp = __reduce_add_sync(0xffffffffu, my_events);
    // a2: the ids go to the block's list of the unit (shared memory); one warp copies the list to the
    // raster after the unit's barrier, with ONE reservation on the global cursor per block and unit
    const unsigned par = (unsigned)nA & 1u;
    unsigned lbase = 0;
    if (lane == 0) {
        lbase = atomicAdd(&bs->unit_spikes[par], tot);
        atomicAdd(&bs->events, (unsigned long long)ev_warp);   // flushed once per block at the end of the launch
        if (lbase + tot <= (unsigned)kSpkCap) atomicMax(&bs->staged[par], lbase + tot);
    }
    lbase = __shfl_sync(0xffffffffu, lbase, 0);
    const bool staged = (lbase + tot <= (unsigned)kSpkCap);   // else (list full): positions straight from the cursor
    unsigned long long base = 0;
    if (!staged) {
        if (lane == 0) base = atomicAdd(&p.ctl->spike_cursor, (unsigned long long)tot);
        base = __shfl_sync(0xffffffffu, base, 0);
    }
    unsigned at = lbase + (inc - my_spk);
    unsigned long long pos = base + (inc - my_spk);
    const unsigned win = (unsigned)((nA / (unsigned long long)p.window_steps) % p.max_windows);
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if (spike_bits & (1u << q)) {
            const int i = p.id0 + i0 + q;                   // the raster, the regions and the rows use global ids
            if (staged) bs->spk[par][at++] = i;
            else {
                p.spike_ids[pos & p.spike_mask] = i;
                p.spike_tag[pos & p.spike_mask] = (uint32_t)nA;
                ++pos;
            }
            if (p.n_regions > 1) atomicAdd(p.region_counts + (size_t)win * p.n_regions + region_of(p, i), 1u);
        }                                                      // one region: added per block and unit (run_unit)
    // a3: the warp pushes the rows of its own spikes, one row at a time
    const unsigned nlo = (unsigned)nA;
    const unsigned nto = transfer_step_lo<kBin>(p, nlo, bs->n0_lo, bs->bin_phase0);   // slot of a synapse = nto + delay
    while (any) {
        const int src = __ffs(any) - 1;
        any &= any - 1u;
        const unsigned bits = __shfl_sync(0xffffffffu, spike_bits, src);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int l = __shfl_sync(0xffffffffu, len[q], src);
            const long long b = __shfl_sync(0xffffffffu, (long long)rb[q], src);
            if (!(bits & (1u << q))) continue;
            if (kHeavy && l > kInlineMax) {                      // leave it to the whole block (end of the unit)
                unsigned at = 0;
                if (lane == 0) at = atomicAdd(&bs->heavy_n[nlo & 1u], 1u);
                at = __shfl_sync(0xffffffffu, at, 0);
                if (at < (unsigned)kHeavyListCap) {
                    if (lane == 0) bs->heavy_row[nlo & 1u][at] = p.id0 + (task * 32 + src) * 4 + q;
                    continue;
                }
            }
            deliver_span<kHalf>(p, nto, (int64_t)b, l, lane);
        }
    }
}

struct RunCtx {                      // per-thread constants of the persistent kernel
    unsigned long long n0;           // step at launch
    int task0, last, i00, task_stride;
    unsigned lane, warp, n_warps, G;
    bool keeper;
};

// Unit j of the launch (see the header comment): B of step n0 + j - 1 (if kB), A of step n0 + j (if kA).
template <bool kHalf, bool kHeavy, bool kB, bool kA, bool kOU, bool kBin>
__device__ __forceinline__ void run_unit(const SimDev& p, const RunCfg& cfg, const RunCtx& c, const TypeSmem* s_tc,
                                         const uint32_t (*s_T)[kPoissonMax], BlockShared* bs, const Stage& sg,
                                         const unsigned j, unsigned& bg_acc) {
    const unsigned long long nA = c.n0 + j, nB = c.n0 + j - 1ull;
    if (j >= 2u) {                     // every delivery of the units <= j - 2 must have landed: the service warp
        if (c.lane == 0)               // of the block polls the grid ahead of time and raises the flag
            while (*reinterpret_cast<volatile unsigned*>(&bs->grid_ok) < j) __nanosleep(20);
        __syncwarp();
        __threadfence_block();
    }
    if (c.task0 < c.last) {
        if (kB) request_ring(p, sg, p.ring + (size_t)(nB & (unsigned long long)(p.D - 1)) * 4 * (size_t)p.Npad + c.i00);
        cp_async_commit();
        for (int task = c.task0; task < c.last; task += (int)c.n_warps) {
            const int next_off = (task + (int)c.n_warps < c.last) ? c.task_stride : 0;
            run_task<kHalf, kHeavy, kB, kA, kOU, kBin>(p, s_tc, s_T, bs, sg, nB, nA, task, c.lane, next_off, bg_acc);
        }
        if (j < cfg.n_steps) { request_state(p, sg, c.i00); cp_async_commit(); }   // own data: no need to wait for the grid
    }
    if (!kHeavy) {                     // no block barrier: the warp reports to the service warp and moves on
        __syncwarp();
        if (c.lane == 0) {
            __threadfence_block();     // cta-scope release of this warp's pushes; the closer's gpu-scope fence is cumulative
            atomicAdd(&bs->done[(unsigned)nA & 1u], 1u);
        }
        return;
    }
    __syncthreads();
    if (kHeavy && kA) {                // rows too long for one warp: shared by the warps of the block
        const unsigned hp = (unsigned)nA & 1u;
        const unsigned nh = min(bs->heavy_n[hp], (unsigned)kHeavyListCap);
        if (nh) {
            const unsigned nto = transfer_step_lo<kBin>(p, (unsigned)nA, bs->n0_lo, bs->bin_phase0);
            unsigned idx = 0;
            for (unsigned r = 0; r < nh; ++r) {
                const int row = bs->heavy_row[hp][r];
                const int64_t rb = __ldg(p.row_begin + row);
                const int len = __ldg(p.row_len + row);
                for (int off = 0; off < len; off += kChunk, ++idx)
                    if (idx % c.n_warps == c.warp)
                        deliver_span<kHalf>(p, nto, rb + off, min(kChunk, len - off), c.lane);
            }
            __syncthreads();
        }
    }
}

// The service warp of a block (its last warp; it owns no neurons).  Per unit j:
//   1. ahead of time, while the update warps work on unit j: wait until the whole grid has closed unit
//      j - 1 (acquire polls of the arrival counter), in block 0 fold that unit's spike count into the
//      step log, and raise grid_ok to j + 1 -- the update warps find the flag up when they get there;
//   2. join the end-of-unit barrier (and the second one of a unit with shared heavy rows);
//   3. close the unit: reserve the raster positions of the block's spikes (before the arrival, so
//      that the entries of step n lie between the cumulative counts of the steps n - 2 and n + 1, as
//      db_read_spikes assumes), add the counters, fence, arrive, then copy the spike list out.  The
//      list and the counters of a unit are reused two units later, behind the next unit's barrier.
template <bool kHeavy>
__device__ __noinline__ void service_warp(const SimDev& p, const RunCfg& cfg, const RunCtx& c, BlockShared* bs) {
    Ctl* const ctl = p.ctl;
    const bool keeper = (blockIdx.x == 0);
    unsigned long long sb = ctl->spike_begin;       // raster bookkeeping (block 0)
    unsigned fin = 0u;                              // units whose step the keeper has logged
    auto log_unit = [&](const unsigned u) {
        sb += (unsigned long long)ld_cg_u32(&ctl->unit_spikes[u & 3u]);
        ctl->unit_spikes[u & 3u] = 0u;
        const unsigned long long np = c.n0 + u;
        p.step_end[np & p.step_log_mask] = sb;
        if ((np + 1) % (unsigned long long)p.window_steps == 0) {
            const unsigned w = (unsigned)(((np + 1) / (unsigned long long)p.window_steps + window_clear_ahead(p.window_steps)) % p.max_windows);
            for (int r = 0; r < p.n_regions; ++r) p.region_counts[(size_t)w * p.n_regions + r] = 0u;
        }
    };
    for (unsigned j = 0; j <= cfg.n_steps; ++j) {
        const unsigned long long nA = c.n0 + j;
        const bool kA = j < cfg.n_steps;
        if (j >= 1u && kA) {                        // unit j + 1 needs the grid to have closed unit j - 1
            if (c.lane == 0) {
                bar_wait(ctl->bar, j - 1u, c.G);
                if (keeper) { log_unit(j - 1u); fin = j; }
                __threadfence_block();
                *reinterpret_cast<volatile unsigned*>(&bs->grid_ok) = j + 1u;
            }
            __syncwarp();
        }
        const unsigned par = (unsigned)nA & 1u;
        if (kHeavy) __syncthreads();                // every update warp has finished unit j
        else {
            if (c.lane == 0) {
                while (*reinterpret_cast<volatile unsigned*>(&bs->done[par]) < c.n_warps) __nanosleep(20);
                __threadfence_block();
                bs->done[par] = 0u;                 // next used two units later, after this unit has been closed grid-wide
            }
            __syncwarp();
        }
        if (kHeavy && kA) {
            const unsigned nh = min(bs->heavy_n[par], (unsigned)kHeavyListCap);
            if (nh) __syncthreads();                // the update warps share the heavy rows, then meet again
            if (c.lane == 0) bs->heavy_n[par] = 0u;
        }
        unsigned st = 0;
        unsigned long long base = 0;
        if (c.lane == 0) {
            const unsigned k = bs->unit_spikes[par];
            st = bs->staged[par];
            bs->unit_spikes[par] = 0u;
            bs->staged[par] = 0u;
            if (k) {
                if (st) base = atomicAdd(&ctl->spike_cursor, (unsigned long long)st);
                atomicAdd(&ctl->unit_spikes[j & 3u], k);
                if (p.n_regions == 1)
                    atomicAdd(p.region_counts + (size_t)((nA / (unsigned long long)p.window_steps) % p.max_windows), k);
            }
            __threadfence();
            atomicAdd(&ctl->bar[j & 3u], 1u);
        }
        st = __shfl_sync(0xffffffffu, st, 0);
        if (st) {
            base = __shfl_sync(0xffffffffu, base, 0);
            for (unsigned k2 = c.lane; k2 < st; k2 += 32u) {
                p.spike_ids[(base + k2) & p.spike_mask] = bs->spk[par][k2];
                p.spike_tag[(base + k2) & p.spike_mask] = (uint32_t)nA;
            }
        }
        __syncwarp();                               // lane 0 must not let the unit that reuses spk[par] start while the others still copy
    }
    if (c.lane == 0) {
        if (bs->events) atomicAdd(&ctl->events, bs->events);     // every emit of the block lies before the last barrier
        if (keeper) {                               // close the launch: log the remaining steps, publish the position
            if (cfg.n_steps >= 1u) bar_wait(ctl->bar, cfg.n_steps - 1u, c.G);   // the last unit that produces spikes
            bar_wait(ctl->bar, cfg.n_steps, c.G);
            for (unsigned u = fin; u < cfg.n_steps; ++u) log_unit(u);
            ctl->spike_begin = sb;
            ctl->step = c.n0 + cfg.n_steps;
        }
    }
}

template <bool kHalf, bool kHeavy, bool kOU, bool kBin>
__global__ void __launch_bounds__(kRunThreads, 1) k_run(const __grid_constant__ SimDev p, const RunCfg cfg) {
    extern __shared__ uint4 s_stage[];                 // kStageBytes: plane k of thread t at k * kPlaneStride + 16 t
    __shared__ TypeSmem s_tc[kMaxTypes];
    __shared__ uint32_t s_T[kMaxTypes][kPoissonMax];
    __shared__ BlockShared bs;
    RunCtx c;
    c.lane = threadIdx.x & 31u; c.warp = threadIdx.x >> 5; c.n_warps = (blockDim.x >> 5) - 1u; c.G = gridDim.x;   // update warps; the last warp is the service warp
    for (int t = (int)threadIdx.x; t < kMaxTypes; t += (int)blockDim.x) {
        const TypeConst& tc = p.tc[t];
        TypeSmem r;
        for (int u = 0; u < 4; ++u) r.rec[u] = make_float4(tc.G[u], tc.E[u], tc.alpha[u], 0.0f);
        r.m0 = make_float4(tc.neg_gL, tc.VL, tc.kappa, tc.Iext);
        r.m1 = make_float4(tc.Vth, tc.Vreset, __int_as_float(tc.R), __int_as_float(tc.wq_bg));
        r.m2 = make_uint4((unsigned)tc.M, 0u - (tc.M > 0 ? tc.T[0] : 0xFFFFFFFFu), 0u - (tc.M > 1 ? tc.T[1] : 0xFFFFFFFFu),
                          0u - (tc.M > 2 ? tc.T[2] : 0xFFFFFFFFu));   // negated thresholds (carry trick in neuron_group)
        r.m3 = make_float4(tc.ou_mu, tc.ou_a, tc.ou_s, __int_as_float(tc.ou));
        s_tc[t] = r;
    }
    for (int k = (int)threadIdx.x; k < kMaxTypes * kPoissonMax; k += (int)blockDim.x)
        s_T[k / kPoissonMax][k % kPoissonMax] = p.tc[k / kPoissonMax].T[k % kPoissonMax];
    if (threadIdx.x == 0) { bs.unit_spikes[0] = bs.unit_spikes[1] = 0u; bs.staged[0] = bs.staged[1] = 0u; bs.heavy_n[0] = bs.heavy_n[1] = 0u; bs.grid_ok = 0u; bs.done[0] = bs.done[1] = 0u; bs.events = 0ull;
                            const unsigned long long n0 = p.ctl->step;
                            bs.n0_lo = (unsigned)n0; bs.bin_phase0 = (unsigned)(n0 % (unsigned long long)p.bin_steps); }
    __syncthreads();

    Stage sg;
    sg.sbase = (uint32_t)__cvta_generic_to_shared(s_stage) + threadIdx.x * 16u;
    sg.srt = (uint32_t)__cvta_generic_to_shared(s_stage) + 9u * kPlaneStride + threadIdx.x * 8u;

    c.n0 = p.ctl->step;                               // nobody writes it before the end of the launch
    const int first = (int)blockIdx.x * cfg.tasks_per_block;
    c.last = min(first + cfg.tasks_per_block, cfg.n_tasks);
    c.task0 = first + (int)c.warp;                    // the warp's first task of every unit
    c.i00 = (c.task0 * 32 + (int)c.lane) * 4;
    c.task_stride = (int)c.n_warps * 128;             // neurons between consecutive tasks of a warp
    unsigned bg_acc = 0u;
    if (cfg.n_steps == 0) return;
    if (c.warp == c.n_warps) { service_warp<kHeavy>(p, cfg, c, &bs); return; }

    if (c.task0 < c.last) { request_state(p, sg, c.i00); cp_async_commit(); }
    run_unit<kHalf, kHeavy, false, true, kOU, kBin>(p, cfg, c, s_tc, s_T, &bs, sg, 0u, bg_acc);
    for (unsigned j = 1; j < cfg.n_steps; ++j)
        run_unit<kHalf, kHeavy, true, true, kOU, kBin>(p, cfg, c, s_tc, s_T, &bs, sg, j, bg_acc);
    run_unit<kHalf, kHeavy, true, false, kOU, kBin>(p, cfg, c, s_tc, s_T, &bs, sg, cfg.n_steps, bg_acc);

    const unsigned bg_warp = __reduce_add_sync(0xffffffffu, bg_acc);
    if (c.lane == 0 && bg_warp)
        atomicAdd(p.bg_parts + ((blockIdx.x * c.n_warps + c.warp) & (kBgParts - 1)), (unsigned long long)bg_warp);
}

// ===========================================================================
// Mode DB_EXEC_KERNELS, update kernel: the neuron update of ONE step (a1 + a2 + a4) with the machinery
// of the persistent kernel -- one block per SM, fixed contiguous task ranges, every plane staged
// through shared memory with cp.async and requested one task ahead -- instead of one thread block
// per 1024 neurons: no tail wave, deeper prefetch.  Whole step n in one pass (classic order: the
// membrane step sees g(n), then slot n is consumed into g(n+1)); spikes go to the global work list
// of k_deliver as in update_group.
// ===========================================================================
__device__ __noinline__ void emit_global(const SimDev& p, const unsigned long long n, const unsigned long long spike_begin,
                                         const int i0, const unsigned lane, const unsigned spike_bits) {
    unsigned my_spk = __popc(spike_bits), my_work = 0, my_events = 0;
    int len[4] = {0, 0, 0, 0};
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if (spike_bits & (1u << q)) {
            len[q] = __ldg(p.row_len + p.id0 + i0 + q);
            my_events += (unsigned)len[q];
            my_work += (unsigned)((len[q] + kChunk - 1) / kChunk);
        }
    // inclusive warp scan of (spikes, work items) packed in one 64-bit word
    unsigned long long pk = ((unsigned long long)my_spk << 32) | my_work;
    unsigned long long inc = pk;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        unsigned long long o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= (unsigned)d) inc += o;
    }
    const unsigned long long tot = __shfl_sync(0xffffffffu, inc, 31);
    const unsigned ev_warp = __reduce_add_sync(0xffffffffu, my_events);
    unsigned long long base = 0;
    if (lane == 0) {
        base = atomicAdd(&p.ctl->step_counts[n & 3ull], tot);
        atomicAdd(&p.ctl->events, (unsigned long long)ev_warp);
    }
    base = __shfl_sync(0xffffffffu, base, 0);
    const unsigned long long mine = base + inc - pk;          // exclusive offsets
    unsigned long long spk_pos = spike_begin + (mine >> 32);
    unsigned work_pos = (unsigned)mine;
    const unsigned win = (unsigned)((n / (unsigned long long)p.window_steps) % p.max_windows);
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if (spike_bits & (1u << q)) {
            const int i = p.id0 + i0 + q;                   // global id
            p.spike_ids[spk_pos & p.spike_mask] = i;
            p.spike_tag[spk_pos & p.spike_mask] = (uint32_t)n;
            ++spk_pos;
            const int nch = (len[q] + kChunk - 1) / kChunk;
            for (int c = 0; c < nch; ++c) p.work[(size_t)(n & 1ull) * p.work_half + work_pos++] = make_int2(i, c);
            const int r = (p.n_regions > 1) ? region_of(p, i) : 0;
            atomicAdd(p.region_counts + (size_t)win * p.n_regions + r, 1u);
        }
}

// kMode 0: whole step n in one pass, classic order (DB_EXEC_KERNELS; the delivery kernel closes the step).
// List mode runs the UNITS of the persistent kernel instead (see its header: A_n = membrane step and spikes of step n,
// B_n = consume ring slot n), so that slot n is read one kernel later than in the classic order and the delivery of the
// spikes of step n -- all of it, delay 1 included -- has the whole next update kernel to run beside:
//   kMode 1: A_n only (first kernel of a db_step call);  kMode 2: B_(n-1) then A_n;  kMode 3: B_(n-1) only (last kernel of a
//   call: the state is complete again).  n = Ctl::step; the kernels with an A part close step n themselves.
template <bool kOU, int kMode>
__global__ void __launch_bounds__(kRunThreads, 1) k_update_stream(const __grid_constant__ SimDev p, const RunCfg cfg) {
    constexpr bool kClassic = (kMode == 0), kB = (kMode != 1), kA = (kMode != 3);
    extern __shared__ uint4 s_stage[];                 // kStageBytes: plane k of thread t at k * kPlaneStride + 16 t
    __shared__ TypeSmem s_tc[kMaxTypes];
    __shared__ uint32_t s_T[kMaxTypes][kPoissonMax];
    const unsigned lane = threadIdx.x & 31u;
    const int warp = (int)(threadIdx.x >> 5), n_warps = (int)(blockDim.x >> 5);
    for (int t = (int)threadIdx.x; t < kMaxTypes; t += (int)blockDim.x) {
        const TypeConst& tc = p.tc[t];
        TypeSmem r;
        for (int u = 0; u < 4; ++u) r.rec[u] = make_float4(tc.G[u], tc.E[u], tc.alpha[u], 0.0f);
        r.m0 = make_float4(tc.neg_gL, tc.VL, tc.kappa, tc.Iext);
        r.m1 = make_float4(tc.Vth, tc.Vreset, __int_as_float(tc.R), __int_as_float(tc.wq_bg));
        r.m2 = make_uint4((unsigned)tc.M, 0u - (tc.M > 0 ? tc.T[0] : 0xFFFFFFFFu), 0u - (tc.M > 1 ? tc.T[1] : 0xFFFFFFFFu),
                          0u - (tc.M > 2 ? tc.T[2] : 0xFFFFFFFFu));   // negated thresholds (carry trick in neuron_group)
        r.m3 = make_float4(tc.ou_mu, tc.ou_a, tc.ou_s, __int_as_float(tc.ou));
        s_tc[t] = r;
    }
    for (int k = (int)threadIdx.x; k < kMaxTypes * kPoissonMax; k += (int)blockDim.x)
        s_T[k / kPoissonMax][k % kPoissonMax] = p.tc[k / kPoissonMax].T[k % kPoissonMax];
    __syncthreads();

    Stage sg;
    sg.sbase = (uint32_t)__cvta_generic_to_shared(s_stage) + threadIdx.x * 16u;
    sg.srt = (uint32_t)__cvta_generic_to_shared(s_stage) + 9u * kPlaneStride + threadIdx.x * 8u;
    const unsigned long long n = p.ctl->step;              // step of the A part
    const unsigned long long nB = kClassic ? n : n - 1ull;  // step whose ring slot is consumed
    const unsigned long long sb = p.ctl->spike_begin;
    if (kA && blockIdx.x == 0 && threadIdx.x == 0) p.ctl->work_step[n & 1ull] = n;     // for the delivery kernel of this step (list mode)
    const int first = (int)blockIdx.x * cfg.tasks_per_block;
    const int last = min(first + cfg.tasks_per_block, cfg.n_tasks);
    const int task0 = first + warp;
    const size_t Np = (size_t)p.Npad;
    int32_t* const slot0 = p.ring + (size_t)(nB & (unsigned long long)(p.D - 1)) * 4 * Np;
    const int i00 = (task0 * 32 + (int)lane) * 4;
    const int task_stride = n_warps * 128;
    unsigned bg_acc = 0u;
    if (task0 < last) {
        request_state(p, sg, i00);
        if (kB) request_ring(p, sg, slot0 + i00);
        cp_async_commit();
    }
    for (int task = task0; task < last; task += n_warps) {
        const int next_off = (task + n_warps < last) ? task_stride : 0;
        const int grp = task * 32 + (int)lane;
        const int i0 = grp * 4;
        // one Philox block serves the four neurons (word q -> neuron i0 + q); drawn while the copies fly
        uint4 rnd = make_uint4(0u, 0u, 0u, 0u);
        if (kB && (!kOU || p.bg_on)) rnd = philox4x32_10_rk(make_uint4((uint32_t)(grp + (p.id0 >> 2)), kStreamBG << 24, (uint32_t)nB, (uint32_t)(nB >> 32)), p.rk);
        float4 iou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        float4 rnd_ou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (kOU && kA) {
            iou = ld_cg_f4(p.Iou + i0);
            const uint4 wo = philox4x32_10_rk(make_uint4((uint32_t)(grp + (p.id0 >> 2)), kStreamOU << 24, (uint32_t)n, (uint32_t)(n >> 32)), p.rk);
            rnd_ou = make_float4(__ldg(p.ntab + (wo.x >> 16)), __ldg(p.ntab + (wo.y >> 16)), __ldg(p.ntab + (wo.z >> 16)),
                                 __ldg(p.ntab + (wo.w >> 16)));
        }
        float4 ix = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (kA && p.iext) ix = ld_cg_f4(p.iext + i0);   // per-neuron external currents (R31)
        cp_async_wait_all();
        const uint4 v_bits = lds128(sg.sbase + 4u * kPlaneStride);
        const uint2 rt_bits = lds64(sg.srt);
        if (next_off) {
            cp_async16(sg.sbase + 4u * kPlaneStride, p.V + i0 + next_off);
            cp_async8(sg.srt, p.rt + i0 + next_off);
        }
        const int tp0 = (int)((rt_bits.x >> 12) & 0xFu), tp1 = (int)(rt_bits.x >> 28);
        const int tp2 = (int)((rt_bits.y >> 12) & 0xFu), tp3 = (int)(rt_bits.y >> 28);
        unsigned spike_bits;
        if (tp0 == tp1 && tp0 == tp2 && tp0 == tp3)
            spike_bits = neuron_group<kB, kA, kClassic, kOU>(p, s_tc, s_T, sg, tp0, tp0, tp0, tp0, i0, slot0 + i0, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou, ix);
        else                            // a type boundary inside the group (rare)
            spike_bits = neuron_group<kB, kA, kClassic, kOU>(p, s_tc, s_T, sg, tp0, tp1, tp2, tp3, i0, slot0 + i0, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou, ix);
        if (kOU && kA) st_cg_f4(p.Iou + i0, iou);
        cp_async_commit();
        if (kA && __ballot_sync(0xffffffffu, spike_bits != 0)) emit_global(p, n, sb, i0, lane, spike_bits);
    }
    const unsigned bg_warp = __reduce_add_sync(0xffffffffu, bg_acc);
    if (lane == 0 && bg_warp)
        atomicAdd(p.bg_parts + ((blockIdx.x * (unsigned)n_warps + (unsigned)warp) & (kBgParts - 1)), (unsigned long long)bg_warp);
    if (!kClassic && kA) {               // list mode: step n is closed here (its delivery runs beside the next update kernel)
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            const unsigned ticket = atomicAdd(&p.ctl->done_blocks, 1u);
            if (ticket == gridDim.x - 1) {    // every block has read n and has added its spikes
                p.ctl->done_blocks = 0u;
                __threadfence();
                finalize_step(p, n, *reinterpret_cast<volatile unsigned long long*>(&p.ctl->step_counts[n & 3ull]));
            }
        }
    }
}

// ---------------------------------------------------------------------------
// State initialisation: V0 = Vreset + (Vth - Vreset) * U, U = (u >> 8) * 2^-24
// keyed by (dyn_seed, STREAM_V0, i); g = 0, ref = 0.
// ---------------------------------------------------------------------------
__global__ void k_init_state(const __grid_constant__ SimDev p, const uint8_t* __restrict__ ntype, const float* __restrict__ iext_tab) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.Npad) return;
    const int tp = (i < p.N) ? ntype[i] : 0;
    const TypeConst& c = p.tc[tp];
    const uint4 r = philox4x32_10(make_uint4((uint32_t)(i + p.id0), kStreamV0 << 24, 0u, 0u), p.seed_lo, p.seed_hi);   // keyed by the global id
    const float U = __fmul_rn(__uint2float_rn(r.x >> 8), 5.9604644775390625e-08f);
    p.V[i] = (i < p.N) ? __fadd_rn(c.Vreset, __fmul_rn(__fsub_rn(c.Vth, c.Vreset), U)) : 0.0f;
    for (int u = 0; u < 4; ++u) p.g[(size_t)u * p.Npad + i] = 0.0f;
    p.rt[i] = (uint16_t)(tp << 12);
    if (p.ou_on) p.Iou[i] = (i < p.N && c.ou) ? c.ou_mu : 0.0f;   // the OU current starts at its mean
    if (p.iext) {                      // external current of the neuron (R31): Iext + Gamma quantile at the top 16 bits of a Philox word
        float v = 0.0f;
        if (i < p.N) {
            v = c.Iext;
            if (c.ix_on) v = __fadd_rn(v, iext_tab[(size_t)tp * 65536u + (philox4x32_10(make_uint4((uint32_t)(i + p.id0), kStreamIEXT << 24, 0u, 0u), p.seed_lo, p.seed_hi).x >> 16)]);
        }
        p.iext[i] = v;
    }
}

// ===========================================================================
// Mode DB_EXEC_KERNELS_DEFERRED: arrival lists.  Pushing a spike's whole row when it fires scatters 4-byte
// reductions over every ring slot the row's delays reach: with a ring far larger than L2 every event is a random
// 32-byte-sector read-modify-write in DRAM (~20 G/s on this device, profiles/), and pulling the (row, delay) segments
// out of the CSR when they arrive (round 1) turns the same events into random DRAM sector READS instead.  Here a row
// is read ONCE, when its neuron fires (contiguous: DRAM streams it), and every synapse becomes an 8-byte record
// (receptor | target, fixed-point weight) appended to the LIST OF ITS ARRIVAL STEP; the rows are sorted by (delay,
// target window) at db_create, so the records of a row fall into a few contiguous runs and one atomic on a list
// cursor reserves a whole run.  In the kernel of step n the list of step n + 1 is streamed back and reduced into
// ring slot n + 1 -- the only slot that takes reductions (16 B x N: L2-sized, window by window when it is not), so
// the reductions run at the L2 rate and DRAM only streams: row 7-9 B + record written 8 B + record read 8 B per
// event.  Records whose arrival step is the next one (delay 1) are reduced into the slot directly; a list that is
// full spills into the dense ring as in the other modes.  The sums are the same integers, whatever the order.
//   near lists: ring of ev_Dn slots for arrivals <= ev_near_lim steps ahead (most events: large capacity per slot);
//   far lists:  ring of D slots for the others (inter-region delays: few events per slot for many slots).
// ===========================================================================
__device__ __forceinline__ unsigned ev_window(const SimDev& p, const unsigned tg) {
    return (unsigned)(tg >= p.ev_wb[0]) + (unsigned)(tg >= p.ev_wb[1]) + (unsigned)(tg >= p.ev_wb[2]);
}

// Sort the rows [row0, row1) by (delay, target window) into scratch arrays (indexed by synapse - s0); one warp per
// row, counting sort over 256 W keys.
constexpr int kSortWarps = 8;
constexpr int kSortBins = 1024;      // 256 delays x up to 4 target windows
template <bool kHalf>
__global__ void __launch_bounds__(kSortWarps * 32) k_sort_rows(const __grid_constant__ SimDev p, const int64_t row0,
        const int64_t row1, const int64_t s0, uint32_t* __restrict__ tgt_out, void* __restrict__ w_out,
        uint8_t* __restrict__ delay_out, uint32_t* __restrict__ seg) {
    __shared__ unsigned s_cnt[kSortWarps][kSortBins];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned* cnt = s_cnt[warp];
    const unsigned W = (unsigned)p.ev_W;
    const int nb = 256 * (int)W, per = nb / 32;
    const long long n_warps = (long long)gridDim.x * kSortWarps;
    for (long long j = row0 + (long long)blockIdx.x * kSortWarps + warp; j < row1; j += n_warps) {
        const int64_t rb = p.row_begin[j];
        const int len = p.row_len[j];
        for (int k = (int)lane; k < nb; k += 32) cnt[k] = 0u;
        __syncwarp();
        for (int e = (int)lane; e < len; e += 32)
            atomicAdd(&cnt[(unsigned)p.delay[rb + e] * W + ev_window(p, p.tgt_rec[rb + e] & 0x3FFFFFFFu)], 1u);
        __syncwarp();
        // exclusive scan of the counters: lane l owns the bins per * l .. per * l + per - 1
        unsigned sum = 0u;
        for (int k = 0; k < per; ++k) { const unsigned c = cnt[(int)lane * per + k]; cnt[(int)lane * per + k] = sum; sum += c; }
        unsigned inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= (unsigned)d) inc += o;
        }
        const unsigned base = inc - sum;
        for (int k = 0; k < per; ++k) cnt[(int)lane * per + k] += base;       // start of every key inside the row
        __syncwarp();
        // segment table of the near part: seg[q] = first synapse with key >= q, q = (d - 1) W + w for d = 1 .. ev_near_d,
        // and seg[K] = start of the far part (delays are >= 1: the bins 0 .. W - 1 are empty)
        const int K = p.ev_near_d * (int)W;
        for (int q = (int)lane; q <= K; q += 32) seg[(size_t)j * (size_t)(K + 1) + (size_t)q] = (q + (int)W < nb) ? cnt[q + (int)W] : (unsigned)len;
        __syncwarp();
        for (int e = (int)lane; e < len; e += 32) {
            const unsigned d = p.delay[rb + e];
            const uint32_t t = p.tgt_rec[rb + e];
            const int64_t o = rb - s0 + (int64_t)atomicAdd(&cnt[d * W + ev_window(p, t & 0x3FFFFFFFu)], 1u);
            tgt_out[o] = t;
            delay_out[o] = (uint8_t)d;
            if (kHalf) static_cast<__half*>(w_out)[o] = static_cast<const __half*>(p.w)[rb + e];
            else       static_cast<float*>(w_out)[o] = static_cast<const float*>(p.w)[rb + e];
        }
        const int padded = (len + kRowAlign - 1) / kRowAlign * kRowAlign;      // keep the row padding inert
        for (int e = len + (int)lane; e < padded; e += 32) {
            const int64_t o = rb - s0 + e;
            tgt_out[o] = 0u;
            delay_out[o] = 1;
            if (kHalf) static_cast<__half*>(w_out)[o] = __float2half(0.0f);
            else       static_cast<float*>(w_out)[o] = 0.0f;
        }
        __syncwarp();
    }
}

// Lists are private to the blocks of the delivery kernel: block b appends to its own list of every (arrival slot,
// window) and reduces its own lists when their step comes, so the list cursors live in the block's shared memory during
// a launch (ev_cnt[b * ev_n_cur + cursor] between launches) and no append needs a global atomic.  Cursor index of the
// list that takes a record arriving `ahead` steps after step n (ahead > ev_direct) at target tg: near family first.
__device__ __forceinline__ unsigned ev_cursor_of(const SimDev& p, const unsigned arrival, const unsigned ahead, const unsigned tg) {
    const unsigned w = ev_window(p, tg);
    if (ahead <= (unsigned)p.ev_near_lim) return (arrival & (unsigned)(p.ev_Dn - 1)) * (unsigned)p.ev_W + w;
    return (unsigned)(p.ev_Dn * p.ev_W) + (arrival & (unsigned)(p.ev_D - 1)) * (unsigned)p.ev_W + w;
}
__device__ __forceinline__ uint2* ev_records(const SimDev& p, const unsigned cur, const unsigned block) {
    const unsigned n_near = (unsigned)(p.ev_Dn * p.ev_W);
    return cur < n_near ? p.ev_rec + ((size_t)cur * p.ev_P + block) * p.ev_cap_near
                        : p.ev_rec + (size_t)n_near * p.ev_P * p.ev_cap_near + ((size_t)(cur - n_near) * p.ev_P + block) * p.ev_cap_far;
}
__device__ __forceinline__ unsigned ev_capacity(const SimDev& p, const unsigned cur) {
    return cur < (unsigned)(p.ev_Dn * p.ev_W) ? p.ev_cap_near : p.ev_cap_far;
}

// Turn `len` synapses starting at `rb` into records: the lanes take 32 consecutive synapses per pass, four passes of
// loads in flight; the lanes of a pass whose records go to the same list (a run of the sorted row) reserve their
// positions with ONE atomic on the list's cursor.  n = step of the spike, nto = its transfer step (R29).
template <bool kHalf>
__device__ __forceinline__ void bin_span(const SimDev& p, const unsigned n_lo, const unsigned nto_lo, const int64_t rb,
                                         const int len, const unsigned lane, unsigned* s_cur, unsigned& spilled) {
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    const unsigned shift = nto_lo - n_lo;                // steps until the end of the spike's time bin
    constexpr int kRounds = 4;                           // passes of 32 synapses in flight: loads first, then the cursor
    for (int base = 0; base < len; base += 32 * kRounds) {   // atomics of all passes, then the stores
        unsigned tr[kRounds], dl[kRounds], list[kRounds], pos[kRounds], peers[kRounds];
        float wf[kRounds];
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const int e = base + r * 32 + (int)lane;
            tr[r] = 0u; dl[r] = 0u; wf[r] = 0.0f;
            if (e < len) {
                tr[r] = __ldg(p.tgt_rec + rb + e);
                dl[r] = __ldg(p.delay + rb + e);
                if (kHalf) wf[r] = __half2float(__ldg(static_cast<const __half*>(p.w) + rb + e));
                else       wf[r] = __ldg(static_cast<const float*>(p.w) + rb + e);
            }
        }
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            list[r] = 0xFFFFFFFFu; pos[r] = 0u; peers[r] = 0u;
            if (base + r * 32 >= len) continue;          // warp-uniform
            const bool valid = base + r * 32 + (int)lane < len;
            const unsigned ahead = shift + dl[r];
            if (valid && ahead > (unsigned)p.ev_direct) list[r] = ev_cursor_of(p, nto_lo + dl[r], ahead, tr[r] & 0x3FFFFFFFu);
            peers[r] = __match_any_sync(0xffffffffu, list[r]);
            if (lane == (unsigned)__ffs(peers[r]) - 1u && list[r] != 0xFFFFFFFFu)
                pos[r] = atomicAdd(s_cur + list[r], (unsigned)__popc(peers[r]));      // shared memory: the block's own cursor
        }
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            if (base + r * 32 >= len) continue;          // warp-uniform
            const unsigned at = __shfl_sync(0xffffffffu, pos[r], __ffs(peers[r]) - 1) + (unsigned)__popc(peers[r] & ((1u << lane) - 1u));
            if (base + r * 32 + (int)lane >= len) continue;
            const int wq = __float2int_rn(__fmul_rn(wf[r], p.wscale));
            if (list[r] != 0xFFFFFFFFu && at < ev_capacity(p, list[r])) {
                st_cs_u2(ev_records(p, list[r], blockIdx.x) + at, make_uint2(tr[r], (unsigned)wq));
            } else {                                     // next step's arrivals, or a full list: straight into the ring
                red_add_s32(p.ring + ((size_t)((nto_lo + dl[r]) & Dm) * 4 + (tr[r] >> 30)) * Np + (tr[r] & 0x3FFFFFFFu), wq);
                if (list[r] != 0xFFFFFFFFu) ++spilled;
            }
        }
    }
}

// The near part of one work item: the synapses [c0, c1) (relative to the row start rb0) of row j with delay <= ev_near_d.
// The row is sorted by (delay, window) and seg[] holds where every (delay, window) run starts, so the lanes reserve the
// list positions of ALL runs of the item at once (one atomic per run, issued together: one round trip), leave
// "list position - synapse index" per run in a table of the warp, and then copy the synapses as one flat range:
// no atomic and no vote inside the copy loop, whose loads are all independent.
constexpr int kEvKeysMax = 128;      // (delay, window) runs of the near part: ev_near_d <= 29 delays x W <= 4 windows
template <bool kHalf>
__device__ __forceinline__ void bin_near(const SimDev& p, const unsigned n_lo, const unsigned nto_lo, const int j, const int64_t rb0,
                                         const int c0, const int c1, const unsigned lane, unsigned* s_cur,
                                         int* tab_off, unsigned* tab_list, unsigned& spilled) {
    const unsigned W = (unsigned)p.ev_W;
    const int K = p.ev_near_d * (int)W;
    const uint32_t* sg = p.seg + (size_t)j * (size_t)(K + 1);
    const unsigned shift = nto_lo - n_lo;
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    constexpr int kRounds = 4;                           // 128 synapses per batch; two batches in flight
    auto load = [&](const int base, unsigned (&tr)[kRounds], unsigned (&dl)[kRounds], float (&wf)[kRounds]) {
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const int e = base + r * 32 + (int)lane;
            tr[r] = 0u; dl[r] = 1u; wf[r] = 0.0f;
            if (e < c1) {
                tr[r] = __ldg(p.tgt_rec + rb0 + e);
                dl[r] = __ldg(p.delay + rb0 + e);
                if (kHalf) wf[r] = __half2float(__ldg(static_cast<const __half*>(p.w) + rb0 + e));
                else       wf[r] = __ldg(static_cast<const float*>(p.w) + rb0 + e);
            }
        }
    };
    auto store = [&](const int base, const unsigned (&tr)[kRounds], const unsigned (&dl)[kRounds], const float (&wf)[kRounds]) {
#pragma unroll
        for (int r = 0; r < kRounds; ++r) {
            const int e = base + r * 32 + (int)lane;
            if (e >= c1) continue;
            const unsigned tg = tr[r] & 0x3FFFFFFFu;
            const unsigned q = (dl[r] - 1u) * W + ev_window(p, tg);
            const unsigned list = tab_list[q];
            const unsigned pos = (unsigned)(tab_off[q] + e);
            const int wq = __float2int_rn(__fmul_rn(wf[r], p.wscale));
            if (list != 0xFFFFFFFFu && pos < p.ev_cap_near) {
                st_cs_u2(p.ev_rec + ((size_t)list * p.ev_P + blockIdx.x) * p.ev_cap_near + pos, make_uint2(tr[r], (unsigned)wq));
            } else {                                     // a full list, or next step's arrivals: straight into the ring
                red_add_s32(p.ring + ((size_t)((nto_lo + dl[r]) & Dm) * 4 + (tr[r] >> 30)) * Np + tg, wq);
                if (list != 0xFFFFFFFFu) ++spilled;
            }
        }
    };
    unsigned trA[kRounds], dlA[kRounds], trB[kRounds], dlB[kRounds];
    float wfA[kRounds], wfB[kRounds];
    load(c0, trA, dlA, wfA);                             // on their way while the positions are reserved
    for (int q = (int)lane; q < K; q += 32) {
        const int s0 = max((int)__ldg(sg + q), c0), s1 = min((int)__ldg(sg + q + 1), c1);
        unsigned list = 0xFFFFFFFFu;
        int off = 0;
        if (s1 > s0) {
            const unsigned d = (unsigned)q / W + 1u, w = (unsigned)q % W;
            if (shift + d > (unsigned)p.ev_direct) {
                list = ((nto_lo + d) & (unsigned)(p.ev_Dn - 1)) * W + w;              // cursor index (near family)
                off = (int)atomicAdd(s_cur + list, (unsigned)(s1 - s0)) - s0;
            }
        }
        tab_off[q] = off;
        tab_list[q] = list;
    }
    __syncwarp();
    for (int base = c0; base < c1; base += 64 * kRounds) {
        const bool two = base + 32 * kRounds < c1;
        if (two) load(base + 32 * kRounds, trB, dlB, wfB);
        store(base, trA, dlA, wfA);
        if (two) {
            if (base + 64 * kRounds < c1) load(base + 64 * kRounds, trA, dlA, wfA);
            store(base + 32 * kRounds, trB, dlB, wfB);
        }
    }
    __syncwarp();
}

// How many synapses carry each delay (db_create: sizes the arrival lists); padding entries count as delay 1.
__global__ void __launch_bounds__(256) k_delay_hist(const uint8_t* __restrict__ delay, const int64_t n, unsigned long long* __restrict__ hist) {
    __shared__ unsigned s_h[256];
    s_h[threadIdx.x] = 0u;
    __syncthreads();
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * 16;
    for (int64_t e = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 16; e < n; e += stride) {
        if (e + 16 <= n) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(delay + e));
            const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 16; ++k) atomicAdd(&s_h[(w[k >> 2] >> ((k & 3) * 8)) & 0xFFu], 1u);
        } else {
            for (int64_t f = e; f < n; ++f) atomicAdd(&s_h[delay[f]], 1u);
        }
    }
    __syncthreads();
    if (s_h[threadIdx.x]) atomicAdd(hist + threadIdx.x, (unsigned long long)s_h[threadIdx.x]);
}

constexpr int kEvChunk = 2048;       // records per pass of a block over one of its lists (256 threads x 8)

// The delivery kernel of step n in list mode.  It touches nothing the NEXT update kernel (B_n, A_(n+1): reads ring slot
// n) reads -- ring slot n + 1 and later, the lists, the work list of step n -- so it sits on a second branch of the step
// graph (db_api.cu) and has to be done before the update kernel after that one (B_(n+1)) starts.  Every block
//   1. streams ITS OWN lists of arrival step n + 1 (filled by its earlier launches) into ring slot n + 1, window by
//      window -- all blocks sweep the windows together, so the reductions of the whole grid stay inside one L2-sized
//      part of the slot at a time -- and empties them;
//   2. takes its share of the rows that fired in step n: the synapses that arrive in step n + 1 are reduced into that
//      slot straight from the CSR, the later ones become records in its lists of their arrival steps.
// It takes n from the cell the update kernel left for it (Ctl::step moves on meanwhile).
template <bool kHalf>
__global__ void __maxnreg__(64) k_deliver_lists(const __grid_constant__ SimDev p, const unsigned parity) {
    extern __shared__ unsigned s_cur[];              // [ev_n_cur] cursors of this block's lists
    __shared__ int s_tab_off[8][kEvKeysMax];
    __shared__ unsigned s_tab_list[8][kEvKeysMax];
    const unsigned long long n = p.ctl->work_step[parity];
    const unsigned n_work = (unsigned)p.ctl->step_counts[n & 3ull];
    const unsigned lane = threadIdx.x & 31u;
    unsigned* const g_cur = p.ev_cnt + (size_t)blockIdx.x * p.ev_n_cur;
    for (unsigned k = threadIdx.x; k < (unsigned)p.ev_n_cur; k += blockDim.x) s_cur[k] = g_cur[k];
    __syncthreads();
    // ---- 1. this block's lists of step m = n + 1: (window, family) in window-major order
    const unsigned m = (unsigned)n + (unsigned)p.ev_direct;
    const size_t Np = (size_t)p.Npad;
    int32_t* const ring_slot = p.ring + (size_t)(m & (unsigned)(p.D - 1)) * 4 * Np;
    const unsigned fams = p.ev_n_far ? 2u : 1u;
    // The slot is cold: nobody has touched it since it was consumed D steps ago, so the FIRST reduction into each of its
    // sectors would be a random DRAM read (a third of all reductions at configs 3 / 4: measured, profiles/).  Instead
    // the blocks stream the window they are about to sweep into L2 with sequential prefetches (one per 128-byte line,
    // 16 B x window neurons in all), one window ahead of the reductions.
    auto prefetch_window = [&](const unsigned w) {
        const unsigned lo = w ? p.ev_wb[w - 1] : 0u;
        const unsigned hi = min(w + 1u < (unsigned)p.ev_W ? p.ev_wb[w] : (unsigned)p.Npad, (unsigned)p.Npad);
        if (hi <= lo) return;
        const unsigned lines = (hi - lo) / 32u;          // per receptor plane (window bounds are multiples of 1024 neurons)
        for (unsigned l = blockIdx.x * blockDim.x + threadIdx.x; l < 4u * lines; l += gridDim.x * blockDim.x) {
            const int32_t* a = ring_slot + (size_t)(l / lines) * Np + lo + (size_t)(l % lines) * 32u;
            asm volatile("prefetch.global.L2 [%0];" :: "l"(a));
        }
    };
    prefetch_window(0u);
    for (unsigned k = 0; k < (unsigned)p.ev_W * fams; ++k) {
        const unsigned w = k / fams, fam = k % fams;
        if (fam == 0u && w + 1u < (unsigned)p.ev_W) prefetch_window(w + 1u);
        const unsigned cur = fam ? (unsigned)(p.ev_Dn * p.ev_W) + (m & (unsigned)(p.ev_D - 1)) * (unsigned)p.ev_W + w
                                 : (m & (unsigned)(p.ev_Dn - 1)) * (unsigned)p.ev_W + w;
        const unsigned c = min(s_cur[cur], ev_capacity(p, cur));
        const uint2* rec = ev_records(p, cur, blockIdx.x);
        for (unsigned r0 = 0u; r0 < c; r0 += (unsigned)kEvChunk) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {                // two records per 128-bit load, four loads in flight
                const unsigned r = r0 + ((unsigned)u * 256u + threadIdx.x) * 2u;
                v[u] = make_uint4(0u, 0u, 0u, 0u);
                if (r + 1u < c) v[u] = ld_cs_u4(reinterpret_cast<const uint4*>(rec + r));
                else if (r < c) { const uint2 a = rec[r]; v[u] = make_uint4(a.x, a.y, 0u, 0u); }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const unsigned r = r0 + ((unsigned)u * 256u + threadIdx.x) * 2u;
                if (r < c) red_add_s32(ring_slot + (size_t)(v[u].x >> 30) * Np + (v[u].x & 0x3FFFFFFFu), (int)v[u].y);
                if (r + 1u < c) red_add_s32(ring_slot + (size_t)(v[u].z >> 30) * Np + (v[u].z & 0x3FFFFFFFu), (int)v[u].w);
            }
        }
        __syncthreads();                                 // every thread has read the count
        if (threadIdx.x == 0) s_cur[cur] = 0u;           // consumed (the appends below go to later steps: other cursors)
    }
    __syncthreads();
    // ---- 2. the rows that fired in step n
    {
        const unsigned bwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
        const unsigned n_bwarps = (gridDim.x * blockDim.x) >> 5;
        const unsigned nto = (unsigned)transfer_step(p, n);
        unsigned spilled = 0u;
        int* const tab_off = s_tab_off[threadIdx.x >> 5];
        unsigned* const tab_list = s_tab_list[threadIdx.x >> 5];
        const int K = p.ev_near_d * p.ev_W;
        const int2* const work = p.work + (size_t)(n & 1ull) * p.work_half;
        // the descriptor of the next item (work entry two ahead, row start / length / end of the near part one ahead) is
        // requested while this one is processed
        int2 wk = make_int2(0, 0), wk1 = make_int2(0, 0);
        if (bwarp < n_work) wk = work[bwarp];
        if (bwarp + n_bwarps < n_work) wk1 = work[bwarp + n_bwarps];
        int64_t rb0 = 0, rb0n = 0;
        int rlen = 0, rlenn = 0, near_end = 0, near_endn = 0;
        if (bwarp < n_work) {
            rb0 = __ldg(p.row_begin + wk.x); rlen = __ldg(p.row_len + wk.x);
            near_end = (int)__ldg(p.seg + (size_t)wk.x * (size_t)(K + 1) + (size_t)K);
        }
        for (unsigned q = bwarp; q < n_work; q += n_bwarps) {
            int2 wk2 = make_int2(0, 0);
            if (q + 2u * n_bwarps < n_work) wk2 = work[q + 2u * n_bwarps];
            if (q + n_bwarps < n_work) {
                rb0n = __ldg(p.row_begin + wk1.x); rlenn = __ldg(p.row_len + wk1.x);
                near_endn = (int)__ldg(p.seg + (size_t)wk1.x * (size_t)(K + 1) + (size_t)K);
            }
            const int c0 = wk.y * kChunk, c1 = min(c0 + kChunk, rlen);
            if (c0 < near_end) bin_near<kHalf>(p, (unsigned)n, nto, wk.x, rb0, c0, min(c1, near_end), lane, s_cur, tab_off, tab_list, spilled);
            if (c1 > near_end) {                         // far part: runs of about one synapse, positions by vote + shared-memory atomic
                const int f0 = max(c0, near_end);
                bin_span<kHalf>(p, (unsigned)n, nto, rb0 + f0, c1 - f0, lane, s_cur, spilled);
            }
            wk = wk1; wk1 = wk2; rb0 = rb0n; rlen = rlenn; near_end = near_endn;
        }
        spilled = __reduce_add_sync(0xffffffffu, spilled);
        if (lane == 0 && spilled) atomicAdd(&p.ctl->ev_spilled, (unsigned long long)spilled);
    }
    __syncthreads();
    for (unsigned k = threadIdx.x; k < (unsigned)p.ev_n_cur; k += blockDim.x) g_cur[k] = s_cur[k];     // for the next launch
}

// Read-back of the ring in list mode: the arrivals still to come are the ring's content PLUS the records waiting in
// the lists.  Adds them for the targets [first, first + count) into `out`, which has the layout of DB_FIELD_RING:
// out[(slot * count + i) * 4 + receptor], slot = arrival step mod D_api.  One block per list at a time.
__global__ void __launch_bounds__(256) k_lists_to_ring(const __grid_constant__ SimDev p, int32_t* __restrict__ out,
                                                       const int first, const int count, const int D_api) {
    const unsigned long long n = p.ctl->step;
    const unsigned n_near = (unsigned)(p.ev_Dn * p.ev_W);
    const unsigned total = (unsigned)p.ev_n_cur * (unsigned)p.ev_P;
    for (unsigned l = blockIdx.x; l < total; l += gridDim.x) {
        const unsigned block = l / (unsigned)p.ev_n_cur, cur = l % (unsigned)p.ev_n_cur;
        const bool far = cur >= n_near;
        const unsigned depth = far ? (unsigned)p.ev_D : (unsigned)p.ev_Dn;
        const unsigned slot = (far ? cur - n_near : cur) / (unsigned)p.ev_W;
        // the one step in [n, n + depth) that maps to this slot
        const unsigned long long arrive = n + (unsigned long long)((slot - (unsigned)n) & (depth - 1u));
        const size_t api_slot = (size_t)(arrive % (unsigned long long)D_api);
        const unsigned c = min(p.ev_cnt[(size_t)block * p.ev_n_cur + cur], ev_capacity(p, cur));
        const uint2* rec = ev_records(p, cur, block);
        for (unsigned r = threadIdx.x; r < c; r += blockDim.x) {
            const uint2 v = rec[r];
            const int tg = (int)(v.x & 0x3FFFFFFFu) - first;
            if (tg >= 0 && tg < count) atomicAdd(out + (api_slot * (size_t)count + (size_t)tg) * 4 + (v.x >> 30), (int)v.y);
        }
    }
}

// f3 (SI Eq.(6) second sum): a handle that owns the targets [id0, id0 + N) holds, for
// EVERY source neuron of the network, the synapses onto its own targets (the paper's layout).  The
// spikes of the neurons it does not own arrive from outside as a list of global ids that fired in step `step`; one warp
// per (spike, 512-synapse chunk) pushes the row into the ring, exactly as k_deliver does for the handle's own spikes.
template <bool kHalf>
__global__ void __launch_bounds__(256) k_deliver_external(const __grid_constant__ SimDev p, const int32_t* __restrict__ ids,
                                                          const unsigned n_ids, const unsigned long long step) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const unsigned nto = (unsigned)transfer_step(p, step);
    unsigned long long ev = 0ull;
    for (unsigned q = warp; q < n_ids; q += n_warps) {
        const int j = __ldg(ids + q);
        const int64_t rb = __ldg(p.row_begin + j);
        const int len = __ldg(p.row_len + j);
        deliver_span<kHalf>(p, nto, rb, len, lane);
        ev += (unsigned long long)len;
    }
    if (lane == 0 && ev) atomicAdd(&p.ctl->events, ev);
}

// ---------------------------------------------------------------------------
// host-side launchers (called from db_api.cu)
// ---------------------------------------------------------------------------
cudaError_t launch_init_state(const SimDev& p, const uint8_t* ntype_dev, const float* iext_tab_dev, cudaStream_t st) {
    k_init_state<<<(p.Npad + 255) / 256, 256, 0, st>>>(p, ntype_dev, iext_tab_dev);
    return cudaGetLastError();
}

void run_shape(const SimDev& p, int n_sm, int* grid, int* threads, RunCfg* cfg);

// Function attributes belong to the device context: called once per handle (finish_setup), on the handle's device.
template <bool kOU>
static const void* update_fn(int mode) {
    switch (mode) {
    case 1: return (const void*)k_update_stream<kOU, 1>;
    case 2: return (const void*)k_update_stream<kOU, 2>;
    case 3: return (const void*)k_update_stream<kOU, 3>;
    default: return (const void*)k_update_stream<kOU, 0>;
    }
}

cudaError_t prepare_kernels() {
    cudaError_t e = cudaSuccess;
    for (int mode = 0; mode < 4 && e == cudaSuccess; ++mode) {
        e = cudaFuncSetAttribute(update_fn<false>(mode), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStageBytes);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(update_fn<true>(mode), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStageBytes);
    }
    return e;
}

// mode: 0 = classic whole step; list mode: 1 = A only, 2 = B then A, 3 = B only (k_update_stream)
cudaError_t launch_update(const SimDev& p, int n_sm, int mode, cudaStream_t st) {
    int grid = 0, threads = 0;
    RunCfg cfg{};
    run_shape(p, n_sm, &grid, &threads, &cfg);
    void* args[] = {(void*)&p, (void*)&cfg};
    return cudaLaunchKernel(p.ou_on ? update_fn<true>(mode) : update_fn<false>(mode), dim3(grid), dim3(threads - 32), args,
                            (size_t)kStageBytes, st);                                               // no service warp here
}

cudaError_t launch_deliver(const SimDev& p, int grid, unsigned parity, cudaStream_t st) {
    if (p.ev_on) {
        const size_t smem = (size_t)p.ev_n_cur * sizeof(unsigned);
        if (p.w_fp16) k_deliver_lists<true><<<p.ev_P, 256, smem, st>>>(p, parity);        // the grid the lists were laid out for
        else          k_deliver_lists<false><<<p.ev_P, 256, smem, st>>>(p, parity);
    } else {
        if (p.w_fp16) k_deliver<true><<<grid, 256, 0, st>>>(p);
        else          k_deliver<false><<<grid, 256, 0, st>>>(p);
    }
    return cudaGetLastError();
}

cudaError_t launch_sort_rows(const SimDev& p, int n_sm, int64_t row0, int64_t row1, int64_t s0, uint32_t* tgt_out, void* w_out,
                             uint8_t* delay_out, uint32_t* seg, cudaStream_t st) {
    const int grid = (int)std::min<int64_t>((row1 - row0 + kSortWarps - 1) / kSortWarps, (int64_t)n_sm * 16);
    if (grid <= 0) return cudaSuccess;
    if (p.w_fp16) k_sort_rows<true><<<grid, kSortWarps * 32, 0, st>>>(p, row0, row1, s0, tgt_out, w_out, delay_out, seg);
    else          k_sort_rows<false><<<grid, kSortWarps * 32, 0, st>>>(p, row0, row1, s0, tgt_out, w_out, delay_out, seg);
    return cudaGetLastError();
}

cudaError_t launch_deliver_external(const SimDev& p, int n_sm, const int32_t* ids_dev, unsigned n_ids, unsigned long long step, cudaStream_t st) {
    const int grid = (int)std::min<unsigned>((n_ids + 7u) / 8u, (unsigned)n_sm * 8u);
    if (grid <= 0) return cudaSuccess;
    if (p.w_fp16) k_deliver_external<true><<<grid, 256, 0, st>>>(p, ids_dev, n_ids, step);
    else          k_deliver_external<false><<<grid, 256, 0, st>>>(p, ids_dev, n_ids, step);
    return cudaGetLastError();
}

cudaError_t launch_delay_hist(const uint8_t* delay, int64_t n, unsigned long long* hist, int n_sm, cudaStream_t st) {
    k_delay_hist<<<n_sm * 8, 256, 0, st>>>(delay, n, hist);
    return cudaGetLastError();
}

cudaError_t launch_lists_to_ring(const SimDev& p, int n_sm, int32_t* out, int first, int count, int D_api, cudaStream_t st) {
    k_lists_to_ring<<<n_sm * 4, 256, 0, st>>>(p, out, first, count, D_api);
    return cudaGetLastError();
}

// One block per SM; tasks (128 neurons) are dealt out in contiguous ranges, and the block size is
// chosen so that the warps of a block take the same number of tasks (no ragged last iteration).
void run_shape(const SimDev& p, int n_sm, int* grid, int* threads, RunCfg* cfg) {
    const int n_tasks = p.Npad / 128;
    const int max_warps = kRunThreads / 32 - 1;        // update warps; one more warp per block is the service warp
    const int tpb = (n_tasks + n_sm - 1) / n_sm;
    const int iters = (tpb + max_warps - 1) / max_warps;
    const int warps = (tpb + iters - 1) / iters;
    cfg->n_tasks = n_tasks; cfg->tasks_per_block = tpb; cfg->iters = iters;
    *grid = (n_tasks + tpb - 1) / tpb;
    *threads = (warps + 1) * 32;
}

template <bool kOU, bool kBin>
static const void* run_fn2(const SimDev& p, bool heavy) {
    if (p.w_fp16) return heavy ? (const void*)k_run<true, true, kOU, kBin> : (const void*)k_run<true, false, kOU, kBin>;
    return heavy ? (const void*)k_run<false, true, kOU, kBin> : (const void*)k_run<false, false, kOU, kBin>;
}

static const void* run_fn(const SimDev& p, bool heavy) {
    const bool bin = p.bin_steps > 1;       // OU drive and time-binned transfer are template arms: the plain kernel pays for neither
    if (p.ou_on) return bin ? run_fn2<true, true>(p, heavy) : run_fn2<true, false>(p, heavy);
    return bin ? run_fn2<false, true>(p, heavy) : run_fn2<false, false>(p, heavy);
}

cudaError_t persistent_fits(const SimDev& p, bool heavy, int n_sm, bool* ok) {
    int grid = 0, threads = 0, per_sm = 0;
    RunCfg cfg{};
    run_shape(p, n_sm, &grid, &threads, &cfg);
    const size_t smem = (size_t)kStageBytes;
    cudaError_t e = cudaFuncSetAttribute(run_fn(p, heavy), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, run_fn(p, heavy), threads, smem);
    *ok = (e == cudaSuccess) && (per_sm * n_sm >= grid);
    return e;
}

cudaError_t launch_persistent(const SimDev& p, bool heavy, unsigned n_steps, int n_sm, cudaStream_t st) {
    int grid = 0, threads = 0;
    RunCfg cfg{};
    run_shape(p, n_sm, &grid, &threads, &cfg);
    cfg.n_steps = n_steps;
    cudaError_t e = cudaMemsetAsync(p.ctl->bar, 0, sizeof(p.ctl->bar) + sizeof(p.ctl->unit_spikes), st);   // adjacent
    if (e != cudaSuccess) return e;
    void* args[] = {(void*)&p, (void*)&cfg};
    return cudaLaunchCooperativeKernel(run_fn(p, heavy), dim3(grid), dim3(threads), args,
                                       (size_t)kStageBytes, st);
}

}  // namespace dbk
