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
    c->step_counts[n & 1ull] = 0ull;
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
    const unsigned long long counts = p.ctl->step_counts[n & 1ull];
    const unsigned n_work = (unsigned)counts;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const unsigned long long nt = transfer_step(p, n);       // slot of a synapse = nt + delay
    for (unsigned q = warp; q < n_work; q += n_warps) deliver_item<kHalf>(p, nt, p.work[q], lane);
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
                                                 const float4 xi_ou = make_float4(0.0f, 0.0f, 0.0f, 0.0f)) {
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
            float Iq = __fadd_rn(I[q], m0.w);
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
        rnd = philox4x32_10_rk(make_uint4((uint32_t)grp, kStreamBG << 24, (uint32_t)nB, (uint32_t)(nB >> 32)), p.rk);
    float4 iou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    float4 rnd_ou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    const bool ou = kOU && kA;
    if (ou) {                          // OU current of the four neurons and their N(0,1) draws (quantile table, top 16 bits of
        iou = ld_cg_f4(p.Iou + i0);    // a Philox word each); gathered here so that the latency hides behind the staged copies
        const uint4 wo = philox4x32_10_rk(make_uint4((uint32_t)grp, kStreamOU << 24, (uint32_t)nA, (uint32_t)(nA >> 32)), p.rk);
        rnd_ou = make_float4(__ldg(p.ntab + (wo.x >> 16)), __ldg(p.ntab + (wo.y >> 16)), __ldg(p.ntab + (wo.z >> 16)),
                             __ldg(p.ntab + (wo.w >> 16)));
    }
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
        spike_bits = neuron_group<kB, kA, false, kOU>(p, s_tc, s_T, sg, tp0, tp0, tp0, tp0, i0, slot, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou);
    else                                // a type boundary inside the group (rare)
        spike_bits = neuron_group<kB, kA, false, kOU>(p, s_tc, s_T, sg, tp0, tp1, tp2, tp3, i0, slot, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou);
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
            len[q] = __ldg(p.row_len + i0 + q);
            rb[q] = __ldg(p.row_begin + i0 + q);
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
            const int i = i0 + q;
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
                    if (lane == 0) bs->heavy_row[nlo & 1u][at] = (task * 32 + src) * 4 + q;
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
            len[q] = __ldg(p.row_len + i0 + q);
            my_events += (unsigned)len[q];
            if (p.near_max > 0)        // deferred mode: only the far part of the row is pushed now
                len[q] -= (int)__ldg(p.seg + (size_t)(i0 + q) * (size_t)(p.near_max + 1) + (size_t)p.near_max);
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
        base = atomicAdd(&p.ctl->step_counts[n & 1ull], tot);
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
            const int i = i0 + q;
            p.spike_ids[spk_pos & p.spike_mask] = i;
            p.spike_tag[spk_pos & p.spike_mask] = (uint32_t)n;
            ++spk_pos;
            const int nch = (len[q] + kChunk - 1) / kChunk;
            for (int c = 0; c < nch; ++c) p.work[work_pos++] = make_int2(i, c);
            const int r = (p.n_regions > 1) ? region_of(p, i) : 0;
            atomicAdd(p.region_counts + (size_t)win * p.n_regions + r, 1u);
        }
}

template <bool kOU>
__global__ void __launch_bounds__(kRunThreads, 1) k_update_stream(const __grid_constant__ SimDev p, const RunCfg cfg) {
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
    const unsigned long long n = p.ctl->step;
    const unsigned long long sb = p.ctl->spike_begin;
    const int first = (int)blockIdx.x * cfg.tasks_per_block;
    const int last = min(first + cfg.tasks_per_block, cfg.n_tasks);
    const int task0 = first + warp;
    if (task0 >= last) return;
    const size_t Np = (size_t)p.Npad;
    int32_t* const slot0 = p.ring + (size_t)(n & (unsigned long long)(p.D - 1)) * 4 * Np;
    const int i00 = (task0 * 32 + (int)lane) * 4;
    const int task_stride = n_warps * 128;
    unsigned bg_acc = 0u;
    request_state(p, sg, i00);
    request_ring(p, sg, slot0 + i00);
    cp_async_commit();
    for (int task = task0; task < last; task += n_warps) {
        const int next_off = (task + n_warps < last) ? task_stride : 0;
        const int grp = task * 32 + (int)lane;
        const int i0 = grp * 4;
        // one Philox block serves the four neurons (word q -> neuron i0 + q); drawn while the copies fly
        uint4 rnd = make_uint4(0u, 0u, 0u, 0u);
        if (!kOU || p.bg_on) rnd = philox4x32_10_rk(make_uint4((uint32_t)grp, kStreamBG << 24, (uint32_t)n, (uint32_t)(n >> 32)), p.rk);
        float4 iou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        float4 rnd_ou = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (kOU) {
            iou = ld_cg_f4(p.Iou + i0);
            const uint4 wo = philox4x32_10_rk(make_uint4((uint32_t)grp, kStreamOU << 24, (uint32_t)n, (uint32_t)(n >> 32)), p.rk);
            rnd_ou = make_float4(__ldg(p.ntab + (wo.x >> 16)), __ldg(p.ntab + (wo.y >> 16)), __ldg(p.ntab + (wo.z >> 16)),
                                 __ldg(p.ntab + (wo.w >> 16)));
        }
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
            spike_bits = neuron_group<true, true, true, kOU>(p, s_tc, s_T, sg, tp0, tp0, tp0, tp0, i0, slot0 + i0, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou);
        else                            // a type boundary inside the group (rare)
            spike_bits = neuron_group<true, true, true, kOU>(p, s_tc, s_T, sg, tp0, tp1, tp2, tp3, i0, slot0 + i0, next_off, v_bits, rt_bits, rnd, bg_acc, &iou, rnd_ou);
        if (kOU) st_cg_f4(p.Iou + i0, iou);
        cp_async_commit();
        if (__ballot_sync(0xffffffffu, spike_bits != 0)) emit_global(p, n, sb, i0, lane, spike_bits);
    }
    const unsigned bg_warp = __reduce_add_sync(0xffffffffu, bg_acc);
    if (lane == 0 && bg_warp)
        atomicAdd(p.bg_parts + ((blockIdx.x * (unsigned)n_warps + (unsigned)warp) & (kBgParts - 1)), (unsigned long long)bg_warp);
}

// ---------------------------------------------------------------------------
// State initialisation: V0 = Vreset + (Vth - Vreset) * U, U = (u >> 8) * 2^-24
// keyed by (dyn_seed, STREAM_V0, i); g = 0, ref = 0.
// ---------------------------------------------------------------------------
__global__ void k_init_state(const __grid_constant__ SimDev p, const uint8_t* __restrict__ ntype) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.Npad) return;
    const int tp = (i < p.N) ? ntype[i] : 0;
    const TypeConst& c = p.tc[tp];
    const uint4 r = philox4x32_10(make_uint4((uint32_t)i, kStreamV0 << 24, 0u, 0u), p.seed_lo, p.seed_hi);
    const float U = __fmul_rn(__uint2float_rn(r.x >> 8), 5.9604644775390625e-08f);
    p.V[i] = (i < p.N) ? __fadd_rn(c.Vreset, __fmul_rn(__fsub_rn(c.Vth, c.Vreset), U)) : 0.0f;
    for (int u = 0; u < 4; ++u) p.g[(size_t)u * p.Npad + i] = 0.0f;
    p.rt[i] = (uint16_t)(tp << 12);
    if (p.ou_on) p.Iou[i] = (i < p.N && c.ou) ? c.ou_mu : 0.0f;   // the OU current starts at its mean
}

// ===========================================================================
// Mode DB_EXEC_KERNELS_DEFERRED.  Pushing a spike's whole row when it fires
// scatters 4-byte reductions over every ring slot the row's delays reach: on
// networks whose ring is far larger than L2 every event misses (measured:
// ~99 B of DRAM sectors per 17-byte event, profiles/).  Here the rows are
// sorted by delay and the push of the synapses with delay d <= near_max is
// DEFERRED: after the update of step n, the kernel walks the spike lists of
// the steps n + 1 - d (d = 1 .. near_max; the raster keeps them) and pushes
// from each of those rows the segment with delay d -- all of it arrives in
// step n + 1, so every reduction hits the ONE ring slot n + 1 (16 B x N, L2
// sized), and DRAM only streams the CSR segments.  Synapses with longer
// delays (the far part of a row) are pushed when the neuron fires, as in the
// other modes.  The sums are the same integers, whatever the order.
// ===========================================================================

// Sort the rows [row0, row1) by delay into scratch arrays (indexed by synapse - s0) and fill their
// segment tables; one warp per row, counting sort over the 256 possible delays.
constexpr int kSortWarps = 8;
template <bool kHalf>
__global__ void __launch_bounds__(kSortWarps * 32) k_sort_rows(const int64_t* __restrict__ row_begin,
        const int32_t* __restrict__ row_len, const uint32_t* __restrict__ tgt_rec, const void* __restrict__ w,
        const uint8_t* __restrict__ delay, const int64_t row0, const int64_t row1, const int64_t s0,
        uint32_t* __restrict__ tgt_out, void* __restrict__ w_out, uint8_t* __restrict__ delay_out,
        uint32_t* __restrict__ seg, const int near_max) {
    __shared__ unsigned s_cnt[kSortWarps][256];
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    unsigned* cnt = s_cnt[warp];
    const long long n_warps = (long long)gridDim.x * kSortWarps;
    for (long long j = row0 + (long long)blockIdx.x * kSortWarps + warp; j < row1; j += n_warps) {
        const int64_t rb = row_begin[j];
        const int len = row_len[j];
        for (int k = (int)lane; k < 256; k += 32) cnt[k] = 0u;
        __syncwarp();
        for (int e = (int)lane; e < len; e += 32) atomicAdd(&cnt[delay[rb + e]], 1u);
        __syncwarp();
        // exclusive scan of the 256 counters: lane l owns the bins 8 l .. 8 l + 7
        unsigned loc[8], sum = 0u;
#pragma unroll
        for (int k = 0; k < 8; ++k) { loc[k] = sum; sum += cnt[lane * 8 + k]; }
        unsigned inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= (unsigned)d) inc += o;
        }
        const unsigned base = inc - sum;
        __syncwarp();
#pragma unroll
        for (int k = 0; k < 8; ++k) cnt[lane * 8 + k] = base + loc[k];      // start of every delay inside the row
        __syncwarp();
        // segment table: first synapse with delay >= d, d = 1 .. near_max + 1 (delays are >= 1)
        for (int d = 1 + (int)lane; d <= near_max + 1; d += 32)
            seg[(size_t)j * (size_t)(near_max + 1) + (size_t)(d - 1)] = (d < 256) ? cnt[d] : (unsigned)len;
        __syncwarp();
        for (int e = (int)lane; e < len; e += 32) {
            const unsigned d = delay[rb + e];
            const int64_t o = rb - s0 + (int64_t)atomicAdd(&cnt[d], 1u);
            tgt_out[o] = tgt_rec[rb + e];
            delay_out[o] = (uint8_t)d;
            if (kHalf) static_cast<__half*>(w_out)[o] = static_cast<const __half*>(w)[rb + e];
            else       static_cast<float*>(w_out)[o] = static_cast<const float*>(w)[rb + e];
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

// Push `len` synapses starting at `rb` (any alignment), one synapse per lane and pass.
// kFixed: all of them land in slot `slot_fixed` (a delay segment); else the slot follows the stored delay.
template <bool kHalf, bool kFixed>
__device__ __forceinline__ void deliver_scalar(const SimDev& p, const unsigned nlo, const unsigned slot_fixed,
                                               const int64_t rb, const int len, const unsigned lane) {
    const size_t Np = (size_t)p.Npad;
    const unsigned Dm = (unsigned)(p.D - 1);
    for (int e = (int)lane; e < len; e += 32) {
        const unsigned t = __ldg(p.tgt_rec + rb + e);
        float wf;
        if (kHalf) wf = __half2float(__ldg(static_cast<const __half*>(p.w) + rb + e));
        else       wf = __ldg(static_cast<const float*>(p.w) + rb + e);
        const unsigned sl = kFixed ? slot_fixed : ((nlo + (unsigned)__ldg(p.delay + rb + e)) & Dm);
        const int wq = __float2int_rn(__fmul_rn(wf, p.wscale));
        red_add_s32(p.ring + ((size_t)sl * 4 + (t >> 30)) * Np + (t & 0x3FFFFFFFu), wq);
    }
}

// Spike list of step m in the two-kernel modes: raster positions [begin, end).  `n` = current step
// (its own entry is not in the step log yet: the count comes from the step counter).
__device__ __forceinline__ void spike_range(const SimDev& p, const unsigned long long n, const unsigned long long counts,
                                            const long long m, unsigned long long& begin, unsigned long long& end) {
    begin = end = 0ull;
    if (m < 0) return;
    if ((unsigned long long)m == n) { begin = p.ctl->spike_begin; end = begin + (counts >> 32); return; }
    begin = (m == 0) ? 0ull : p.step_end[(unsigned long long)(m - 1) & p.step_log_mask];
    end = p.step_end[(unsigned long long)m & p.step_log_mask];
}

template <bool kHalf>
__global__ void __launch_bounds__(256) k_deliver_deferred(const __grid_constant__ SimDev p) {
    __shared__ unsigned long long s_begin[32];
    __shared__ unsigned s_cum[33];                  // s_cum[d] = near items of the delays < d + 1 (exclusive prefix)
    __shared__ unsigned s_pref[8][32];              // per warp: first flat synapse index of each of its 32 items
    __shared__ long long s_rb[8][32];               // per warp: first synapse of each item
    const unsigned long long n = p.ctl->step;
    const unsigned long long counts = p.ctl->step_counts[n & 1ull];
    const unsigned n_work = (unsigned)counts;       // far-part chunks of this step's spikes
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const int S = p.near_max + 1;
    if (threadIdx.x < 32) {
        unsigned long long b = 0ull, e = 0ull;
        if ((int)lane < p.near_max) spike_range(p, n, counts, (long long)n - (long long)lane, b, e);   // d = lane + 1
        const unsigned c = (unsigned)(e - b);
        unsigned inc = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= (unsigned)d) inc += o;
        }
        s_begin[lane] = b;
        s_cum[lane + 1] = inc;
        if (lane == 0) s_cum[0] = 0u;
    }
    __syncthreads();
    // ---- far part of the rows that fired in this step (delay > near_max): pushed now, slot by stored delay
    for (unsigned q = warp; q < n_work; q += n_warps) {
        const int2 wk = p.work[q];
        const int j = wk.x;
        const int near_end = (int)__ldg(p.seg + (size_t)j * S + p.near_max);
        const int off = near_end + wk.y * kChunk;
        const int len = min(kChunk, __ldg(p.row_len + j) - off);
        deliver_scalar<kHalf, false>(p, (unsigned)n, 0u, __ldg(p.row_begin + j) + off, len, lane);
    }
    // ---- near part: segment d of every row that fired in step n + 1 - d arrives in step n + 1.
    // An item = (delay d, one spike of step n + 1 - d).  A warp takes 32 items at a time: every lane
    // fetches the descriptor of one item (spike id -> segment bounds -> row start: all 32 chains in
    // flight together), then the lanes walk the synapses of the 32 segments as ONE flat range, so that
    // the loads of a pass are independent whatever the segment lengths are.
    const unsigned total = s_cum[32];
    const unsigned slot = (unsigned)(n + 1ull) & (unsigned)(p.D - 1);
    const size_t Np = (size_t)p.Npad;
    int32_t* const ring_slot = p.ring + (size_t)slot * 4 * Np;
    unsigned* const w_pref = s_pref[threadIdx.x >> 5];
    long long* const w_rb = s_rb[threadIdx.x >> 5];
    for (unsigned base = warp * 32u; base < total; base += n_warps * 32u) {
        const unsigned q = base + lane;
        int len = 0;
        long long rb = 0;
        if (q < total) {
            unsigned lo = 0u, hi = (unsigned)p.near_max;                     // largest dm1 with s_cum[dm1] <= q
            while (hi - lo > 1u) { const unsigned mid = (lo + hi) >> 1; if (s_cum[mid] <= q) lo = mid; else hi = mid; }
            const unsigned long long pos = s_begin[lo] + (unsigned long long)(q - s_cum[lo]);
            const int j = p.spike_ids[pos & p.spike_mask];
            const uint32_t* sg = p.seg + (size_t)j * S + lo;
            const int o0 = (int)__ldg(sg), o1 = (int)__ldg(sg + 1);
            len = o1 - o0;
            rb = (long long)__ldg(p.row_begin + j) + o0;
        }
        unsigned inc = (unsigned)len;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= (unsigned)d) inc += o;
        }
        const unsigned flat = __shfl_sync(0xffffffffu, inc, 31);
        w_pref[lane] = inc - (unsigned)len;
        w_rb[lane] = rb;
        __syncwarp();
        for (unsigned s0 = 0u; s0 < flat; s0 += 128u) {                      // four independent passes in flight
            unsigned t[4];
            float wf[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const unsigned sx = s0 + (unsigned)u * 32u + lane;
                t[u] = 0u; wf[u] = 0.0f;
                if (sx < flat) {
                    unsigned k = 0u;                                         // largest k with w_pref[k] <= sx
#pragma unroll
                    for (unsigned step = 16u; step; step >>= 1) if (w_pref[k + step] <= sx) k += step;
                    const long long e = w_rb[k] + (long long)(sx - w_pref[k]);
                    t[u] = __ldg(p.tgt_rec + e);
                    if (kHalf) wf[u] = __half2float(__ldg(static_cast<const __half*>(p.w) + e));
                    else       wf[u] = __ldg(static_cast<const float*>(p.w) + e);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (s0 + (unsigned)u * 32u + lane < flat)
                    red_add_s32(ring_slot + (size_t)(t[u] >> 30) * Np + (t[u] & 0x3FFFFFFFu), __float2int_rn(__fmul_rn(wf[u], p.wscale)));
        }
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned ticket = atomicAdd(&p.ctl->done_blocks, 1u);
        if (ticket == gridDim.x - 1) {            // every block has read n / counts / the step log: safe to advance
            p.ctl->done_blocks = 0u;
            finalize_step(p, n, counts);
        }
    }
}

// Read-back of the ring in deferred mode: the arrivals still to come are the ring's content PLUS the
// near segments not pushed yet -- spikes of step m (n - near_max < m < n), delays n - m < d <= near_max,
// arriving in step m + d.  Adds them for the targets [first, first + count) into `out`, which has the
// layout of DB_FIELD_RING: out[(slot * count + i) * 4 + receptor], slot = arrival step mod D_api.
template <bool kHalf>
__global__ void __launch_bounds__(256) k_pending_ring(const __grid_constant__ SimDev p, int32_t* __restrict__ out,
                                                      const int first, const int count, const int D_api) {
    const unsigned long long n = p.ctl->step;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    const int S = p.near_max + 1;
    for (int age = 1; age < p.near_max; ++age) {              // m = n - age: delays age + 1 .. near_max are pending
        const long long m = (long long)n - age;
        unsigned long long b, e;
        spike_range(p, n, 0ull, m, b, e);
        for (unsigned long long pos = b + warp; pos < e; pos += n_warps) {
            const int j = p.spike_ids[pos & p.spike_mask];
            const int64_t rb = __ldg(p.row_begin + j);
            const int o0 = (int)__ldg(p.seg + (size_t)j * S + age);          // first synapse with delay >= age + 1
            const int o1 = (int)__ldg(p.seg + (size_t)j * S + p.near_max);   // start of the far part
            for (int s = o0 + (int)lane; s < o1; s += 32) {
                const unsigned t = __ldg(p.tgt_rec + rb + s);
                const int tg = (int)(t & 0x3FFFFFFFu) - first;
                if (tg < 0 || tg >= count) continue;
                float wf;
                if (kHalf) wf = __half2float(__ldg(static_cast<const __half*>(p.w) + rb + s));
                else       wf = __ldg(static_cast<const float*>(p.w) + rb + s);
                const unsigned long long arrive = (unsigned long long)m + (unsigned long long)__ldg(p.delay + rb + s);
                const size_t slot = (size_t)(arrive % (unsigned long long)D_api);
                atomicAdd(out + (slot * (size_t)count + (size_t)tg) * 4 + (t >> 30), __float2int_rn(__fmul_rn(wf, p.wscale)));
            }
        }
    }
}

// ---------------------------------------------------------------------------
// host-side launchers (called from db_api.cu)
// ---------------------------------------------------------------------------
cudaError_t launch_init_state(const SimDev& p, const uint8_t* ntype_dev, cudaStream_t st) {
    k_init_state<<<(p.Npad + 255) / 256, 256, 0, st>>>(p, ntype_dev);
    return cudaGetLastError();
}

void run_shape(const SimDev& p, int n_sm, int* grid, int* threads, RunCfg* cfg);

// Function attributes belong to the device context: called once per handle (finish_setup), on the handle's device.
cudaError_t prepare_kernels() {
    cudaError_t e = cudaFuncSetAttribute(k_update_stream<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStageBytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_update_stream<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStageBytes);
    return e;
}

cudaError_t launch_update(const SimDev& p, int n_sm, cudaStream_t st) {
    int grid = 0, threads = 0;
    RunCfg cfg{};
    run_shape(p, n_sm, &grid, &threads, &cfg);
    if (p.ou_on) k_update_stream<true><<<grid, threads - 32, (size_t)kStageBytes, st>>>(p, cfg);      // no service warp here
    else         k_update_stream<false><<<grid, threads - 32, (size_t)kStageBytes, st>>>(p, cfg);
    return cudaGetLastError();
}

cudaError_t launch_deliver(const SimDev& p, int grid, cudaStream_t st) {
    if (p.near_max > 0) {
        if (p.w_fp16) k_deliver_deferred<true><<<grid, 256, 0, st>>>(p);
        else          k_deliver_deferred<false><<<grid, 256, 0, st>>>(p);
    } else {
        if (p.w_fp16) k_deliver<true><<<grid, 256, 0, st>>>(p);
        else          k_deliver<false><<<grid, 256, 0, st>>>(p);
    }
    return cudaGetLastError();
}

cudaError_t launch_sort_rows(const SimDev& p, int n_sm, int64_t row0, int64_t row1, int64_t s0, uint32_t* tgt_out, void* w_out,
                             uint8_t* delay_out, uint32_t* seg, int near_max, cudaStream_t st) {
    const int grid = (int)std::min<int64_t>((row1 - row0 + kSortWarps - 1) / kSortWarps, (int64_t)n_sm * 16);
    if (grid <= 0) return cudaSuccess;
    if (p.w_fp16) k_sort_rows<true><<<grid, kSortWarps * 32, 0, st>>>(p.row_begin, p.row_len, p.tgt_rec, p.w, p.delay, row0, row1,
                                                                     s0, tgt_out, w_out, delay_out, seg, near_max);
    else          k_sort_rows<false><<<grid, kSortWarps * 32, 0, st>>>(p.row_begin, p.row_len, p.tgt_rec, p.w, p.delay, row0, row1,
                                                                      s0, tgt_out, w_out, delay_out, seg, near_max);
    return cudaGetLastError();
}

cudaError_t launch_pending_ring(const SimDev& p, int n_sm, int32_t* out, int first, int count, int D_api, cudaStream_t st) {
    if (p.w_fp16) k_pending_ring<true><<<n_sm * 4, 256, 0, st>>>(p, out, first, count, D_api);
    else          k_pending_ring<false><<<n_sm * 4, 256, 0, st>>>(p, out, first, count, D_api);
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
