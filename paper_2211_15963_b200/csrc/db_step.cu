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

__device__ __forceinline__ int region_of(const SimDev& p, int i) {
    int lo = 0, hi = p.n_regions;                 // region_start[lo] <= i < region_start[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(p.region_start + mid) <= i) lo = mid; else hi = mid;
    }
    return lo;
}

// ---------------------------------------------------------------------------
// One neuron, one step.  Returns 1 if it spikes.  `a` holds the four consumed
// ring cells (AMPA already including the background), v / g / ref are updated
// in place.
// ---------------------------------------------------------------------------
__device__ __forceinline__ int neuron_step(const TypeConst& c, float scale, const int a[4],
                                           float& v, float g[4], int& ref) {
    float x[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = __fmul_rn(__int2float_rn(a[u]), scale);
    const float t0 = __fmul_rn(__fmul_rn(c.G[0], g[0]), __fsub_rn(c.E[0], v));
    const float t1 = __fmul_rn(__fmul_rn(c.G[1], g[1]), __fsub_rn(c.E[1], v));
    const float t2 = __fmul_rn(__fmul_rn(c.G[2], g[2]), __fsub_rn(c.E[2], v));
    const float t3 = __fmul_rn(__fmul_rn(c.G[3], g[3]), __fsub_rn(c.E[3], v));
    const float I = __fadd_rn(__fadd_rn(__fadd_rn(__fadd_rn(t0, t1), t2), t3), c.Iext);
    const float leak = __fmul_rn(c.neg_gL, __fsub_rn(v, c.VL));
    float vn = __fadd_rn(v, __fmul_rn(c.kappa, __fadd_rn(leak, I)));
#pragma unroll
    for (int u = 0; u < 4; ++u) g[u] = __fadd_rn(__fmul_rn(g[u], c.alpha[u]), x[u]);
    int spike = 0;
    if (ref > 0) { vn = c.Vreset; ref -= 1; }
    else if (vn >= c.Vth) { spike = 1; vn = c.Vreset; ref = c.R; }
    v = vn;
    return spike;
}

__device__ __forceinline__ int poisson_count(const TypeConst& c, uint32_t u) {
    int k = 0;
    while (k < c.M && u >= c.T[k]) ++k;           // thresholds increase: same as counting all u >= T_m
    return k;
}

// ---------------------------------------------------------------------------
// a1 + a2 + a4 for the four neurons i0..i0+3 owned by this thread.  Called by
// whole warps (Npad is a multiple of 128).
// ---------------------------------------------------------------------------
__device__ __forceinline__ void update_group(const SimDev& p, const unsigned long long n,
                                             const unsigned long long spike_begin, const int grp) {
    const int i0 = grp * 4;
    const size_t Np = (size_t)p.Npad;
    int32_t* slot = p.ring + (size_t)(n & (unsigned long long)(p.D - 1)) * 4 * Np + i0;

    // all loads first: ten independent 128-bit (and one 64-bit) requests in flight
    int4 ar[4];
    float4 gr[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) ar[u] = ld_stream_i4(slot + u * Np);
    const float4 v4 = ld_stream_f4(p.V + i0);
#pragma unroll
    for (int u = 0; u < 4; ++u) gr[u] = ld_stream_f4(p.g + u * Np + i0);
    const ushort4 rt4 = *reinterpret_cast<const ushort4*>(p.rt + i0);

    // one Philox block serves the four neurons (word q -> neuron i0 + q)
    const uint4 rnd = philox4x32_10(make_uint4((uint32_t)grp, kStreamBG << 24,
                                               (uint32_t)n, (uint32_t)(n >> 32)),
                                    p.seed_lo, p.seed_hi);

    float v[4] = {v4.x, v4.y, v4.z, v4.w};
    int a[4][4] = {{ar[0].x, ar[1].x, ar[2].x, ar[3].x}, {ar[0].y, ar[1].y, ar[2].y, ar[3].y},
                   {ar[0].z, ar[1].z, ar[2].z, ar[3].z}, {ar[0].w, ar[1].w, ar[2].w, ar[3].w}};
    float g[4][4] = {{gr[0].x, gr[1].x, gr[2].x, gr[3].x}, {gr[0].y, gr[1].y, gr[2].y, gr[3].y},
                     {gr[0].z, gr[1].z, gr[2].z, gr[3].z}, {gr[0].w, gr[1].w, gr[2].w, gr[3].w}};
    unsigned short rt[4] = {rt4.x, rt4.y, rt4.z, rt4.w};
    const uint32_t rw[4] = {rnd.x, rnd.y, rnd.z, rnd.w};

    unsigned spike_bits = 0;
    unsigned bg = 0, ovf = 0, rt_changed = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int tp = rt[q] >> 12;
        const TypeConst& c = p.tc[tp];
        const bool valid = (i0 + q) < p.N;
#pragma unroll
        for (int u = 0; u < 4; ++u) ovf |= (unsigned)(a[q][u] > (1 << 30) || a[q][u] < -(1 << 30));
        const int k = valid ? poisson_count(c, rw[q]) : 0;
        bg += (unsigned)k;
        a[q][0] = (int)((unsigned)a[q][0] + (unsigned)k * (unsigned)c.wq_bg);
        int ref = rt[q] & kRefMask;
        const int ref_in = ref;
        const int s = neuron_step(c, p.scale, a[q], v[q], g[q], ref);
        rt_changed |= (unsigned)(ref != ref_in);
        rt[q] = (unsigned short)((tp << 12) | ref);
        if (s && valid) spike_bits |= 1u << q;
    }

    // stores: state always, consumed ring cells and rt only where something changed
    st_stream_f4(p.V + i0, make_float4(v[0], v[1], v[2], v[3]));
#pragma unroll
    for (int u = 0; u < 4; ++u)
        st_stream_f4(p.g + u * Np + i0, make_float4(g[0][u], g[1][u], g[2][u], g[3][u]));
#pragma unroll
    for (int u = 0; u < 4; ++u)
        if ((ar[u].x | ar[u].y | ar[u].z | ar[u].w) != 0) st_stream_i4(slot + u * Np, make_int4(0, 0, 0, 0));
    if (rt_changed) *reinterpret_cast<ushort4*>(p.rt + i0) = make_ushort4(rt[0], rt[1], rt[2], rt[3]);
    if (ovf) p.ctl->overflow = 1u;

    // background-event counter: one reduction per warp, spread over many cells
    const unsigned lane = threadIdx.x & 31u;
    const unsigned bg_warp = __reduce_add_sync(0xffffffffu, bg);
    if (lane == 0 && bg_warp)
        atomicAdd(p.bg_parts + ((unsigned)(grp >> 5) & (kBgParts - 1)), (unsigned long long)bg_warp);

    // ---- a2: compaction.  Spikes are rare (rate * dt per neuron-step): whole warps skip this.
    const unsigned any = __ballot_sync(0xffffffffu, spike_bits != 0);
    if (any == 0) return;
    unsigned my_spk = __popc(spike_bits), my_work = 0, my_events = 0;
    int len[4] = {0, 0, 0, 0};
#pragma unroll
    for (int q = 0; q < 4; ++q)
        if (spike_bits & (1u << q)) {
            len[q] = __ldg(p.row_len + i0 + q);
            my_work += (unsigned)((len[q] + kChunk - 1) / kChunk);
            my_events += (unsigned)len[q];
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
            ++spk_pos;
            const int nch = (len[q] + kChunk - 1) / kChunk;
            for (int c = 0; c < nch; ++c) p.work[work_pos++] = make_int2(i, c);
            const int r = (p.n_regions > 1) ? region_of(p, i) : 0;
            atomicAdd(p.region_counts + (size_t)win * p.n_regions + r, 1u);
        }
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
    p.step_end[n & p.step_log_mask] = end;
    c->step_counts[n & 1ull] = 0ull;
    if ((n + 1) % (unsigned long long)p.window_steps == 0) {
        const unsigned w = (unsigned)(((n + 1) / (unsigned long long)p.window_steps + 1) % p.max_windows);
        for (int r = 0; r < p.n_regions; ++r) p.region_counts[(size_t)w * p.n_regions + r] = 0u;
    }
    c->step = n + 1;
}

// ===========================================================================
// Mode DB_EXEC_KERNELS: two kernels per step.
// ===========================================================================
__global__ void __launch_bounds__(256) k_update(const __grid_constant__ SimDev p) {
    const int grp = blockIdx.x * blockDim.x + threadIdx.x;
    if (grp * 4 >= p.Npad) return;
    const unsigned long long n = p.ctl->step;
    const unsigned long long sb = p.ctl->spike_begin;
    update_group(p, n, sb, grp);
}

template <bool kHalf>
__global__ void __launch_bounds__(256) k_deliver(const __grid_constant__ SimDev p) {
    const unsigned long long n = p.ctl->step;
    const unsigned long long counts = p.ctl->step_counts[n & 1ull];
    const unsigned n_work = (unsigned)counts;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned n_warps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned q = warp; q < n_work; q += n_warps) deliver_item<kHalf>(p, n, p.work[q], lane);
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
// Mode DB_EXEC_PERSISTENT: one cooperative kernel runs all the steps; two grid
// barriers per step replace two kernel launches.
// ===========================================================================
__device__ __forceinline__ unsigned long long globaltimer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

template <bool kHalf>
__global__ void __launch_bounds__(256) k_persistent(const __grid_constant__ SimDev p, const unsigned n_steps) {
    cg::grid_group grid = cg::this_grid();
    const unsigned lane = threadIdx.x & 31u;
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned n_thr = gridDim.x * blockDim.x;
    const unsigned n_grp = (unsigned)(p.Npad / 4);
    unsigned long long n = p.ctl->step;
    unsigned long long sb = p.ctl->spike_begin;
    const bool timer = (tid == 0);
    unsigned long long t0 = timer ? globaltimer_ns() : 0ull, t_upd = 0, t_del = 0;
    unsigned long long prev_counts = 0ull;
    for (unsigned s = 0; s < n_steps; ++s, ++n) {
        if (tid == 0 && s > 0) finalize_step(p, n - 1, prev_counts);   // overlaps this step's update
        for (unsigned grp = tid; grp < n_grp; grp += n_thr) update_group(p, n, sb, (int)grp);
        grid.sync();
        if (timer) { const unsigned long long t1 = globaltimer_ns(); t_upd += t1 - t0; t0 = t1; }
        const unsigned long long counts = *(volatile unsigned long long*)&p.ctl->step_counts[n & 1ull];
        const unsigned n_work = (unsigned)counts;
        for (unsigned q = tid >> 5; q < n_work; q += n_thr >> 5) deliver_item<kHalf>(p, n, p.work[q], lane);
        sb += counts >> 32;
        prev_counts = counts;
        grid.sync();
        if (timer) { const unsigned long long t1 = globaltimer_ns(); t_del += t1 - t0; t0 = t1; }
    }
    if (tid == 0) {
        if (n_steps) finalize_step(p, n - 1, prev_counts);
        p.ctl->t_update += t_upd; p.ctl->t_deliver += t_del;
    }
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
}

// ---------------------------------------------------------------------------
// host-side launchers (called from db_api.cu)
// ---------------------------------------------------------------------------
cudaError_t launch_init_state(const SimDev& p, const uint8_t* ntype_dev, cudaStream_t st) {
    k_init_state<<<(p.Npad + 255) / 256, 256, 0, st>>>(p, ntype_dev);
    return cudaGetLastError();
}

int update_grid(const SimDev& p) { return (p.Npad / 4 + 255) / 256; }

cudaError_t launch_update(const SimDev& p, cudaStream_t st) {
    k_update<<<update_grid(p), 256, 0, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_deliver(const SimDev& p, int grid, cudaStream_t st) {
    if (p.w_fp16) k_deliver<true><<<grid, 256, 0, st>>>(p);
    else          k_deliver<false><<<grid, 256, 0, st>>>(p);
    return cudaGetLastError();
}

cudaError_t persistent_max_grid(const SimDev& p, int n_sm, int* grid) {
    int per_sm = 0;
    cudaError_t e = p.w_fp16
        ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_persistent<true>, 256, 0)
        : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_persistent<false>, 256, 0);
    *grid = per_sm * n_sm;
    return e;
}

cudaError_t launch_persistent(const SimDev& p, unsigned n_steps, int grid, cudaStream_t st) {
    void* args[] = {(void*)&p, (void*)&n_steps};
    const void* fn = p.w_fp16 ? (const void*)k_persistent<true> : (const void*)k_persistent<false>;
    return cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(256), args, 0, st);
}

}  // namespace dbk
