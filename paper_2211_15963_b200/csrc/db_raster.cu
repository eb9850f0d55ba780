// a5, read-back of the raster: select the entries of a step range out of the tagged raster ring and sort them by
// (step, id) on the device (the host-side std::sort of ~7e5 entries per 1000 steps of configs[1] took 26-30 ms, three
// times the simulation itself).  One pass builds 64-bit keys (step - step_begin) << 32 | id, all ones for entries of
// other steps; cub's radix sort (a library sort, used as such) orders them; the first n keys are the answer.
#include <cub/device/device_radix_sort.cuh>
#include "db_host.h"

namespace dbk {

__global__ void __launch_bounds__(256) k_raster_keys(const __grid_constant__ SimDev p, const unsigned long long scan_begin,
                                                     const unsigned long long m, const uint32_t lo, const uint32_t span,
                                                     unsigned long long* __restrict__ keys) {
    for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < m;
         k += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long pos = (scan_begin + k) & p.spike_mask;
        const uint32_t rel = p.spike_tag[pos] - lo;
        keys[k] = rel < span ? ((unsigned long long)rel << 32) | (unsigned long long)(uint32_t)p.spike_ids[pos] : ~0ull;
    }
}

// The sorted keys split into the two arrays of the API: step (64-bit) and id, `count` of them.
__global__ void __launch_bounds__(256) k_raster_split(const unsigned long long* __restrict__ keys, const unsigned long long count,
                                                      const unsigned long long step_begin, unsigned long long* __restrict__ steps,
                                                      int32_t* __restrict__ ids) {
    for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < count;
         k += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long key = keys[k];
        if (steps) steps[k] = step_begin + (key >> 32);
        if (ids) ids[k] = (int32_t)(uint32_t)key;
    }
}

// Keep the scratch of the last calls in the device's stream-ordered pool (default: everything goes back to the OS at
// every synchronize).  The pool belongs to the device: set once per handle, on the handle's device.
cudaError_t raster_pool_setup(int device) {
    cudaMemPool_t pool = nullptr;
    unsigned long long keep = 256ull << 20;
    cudaError_t e = cudaDeviceGetDefaultMemPool(&pool, device);
    if (e == cudaSuccess) e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    return e;
}

// The n entries of the step range, sorted by (step, id), straight into the caller's host arrays (either may be NULL;
// at most `cap` entries): the device sorts and splits, two copies bring the result back -- at DMA speed when the
// caller's arrays are pinned.  *consistent = the n-th key is valid and the one after it is not.
cudaError_t raster_sorted_read(const SimDev& p, int n_sm, uint64_t scan_begin, uint64_t m, uint32_t lo, uint32_t span, uint64_t n,
                               uint64_t step_begin, uint64_t* steps_host, int32_t* ids_host, uint64_t cap, bool* consistent,
                               cudaStream_t st) {
    unsigned long long *a = nullptr, *b = nullptr, *steps_dev = nullptr;
    int32_t* ids_dev = nullptr;
    void* tmp = nullptr;
    size_t tmp_bytes = 0;
    *consistent = false;
    if (n == 0 || n > m) return cudaSuccess;
    const uint64_t count = std::min<uint64_t>(n, cap);
    cudaError_t e = cudaMallocAsync(&a, (size_t)m * 8, st);
    if (e == cudaSuccess) e = cudaMallocAsync(&b, (size_t)m * 8, st);
    if (e == cudaSuccess && steps_host) e = cudaMallocAsync(&steps_dev, (size_t)count * 8, st);
    if (e == cudaSuccess && ids_host) e = cudaMallocAsync(&ids_dev, (size_t)count * 4, st);
    int end_bit = 33;                                   // bits of (span - 1) above the id word, + the sentinel's
    while (end_bit < 64 && ((uint64_t)span >> (end_bit - 32)) != 0) ++end_bit;
    end_bit = end_bit < 64 ? end_bit + 1 : 64;          // one more bit tells the all-ones sentinel from any valid key
    if (e == cudaSuccess) e = cub::DeviceRadixSort::SortKeys(nullptr, tmp_bytes, a, b, (int64_t)m, 0, end_bit, st);
    if (e == cudaSuccess) e = cudaMallocAsync(&tmp, tmp_bytes ? tmp_bytes : 16, st);
    if (e == cudaSuccess) {
        const unsigned grid = (unsigned)std::min<uint64_t>((m + 255) / 256, (uint64_t)n_sm * 16);
        k_raster_keys<<<grid, 256, 0, st>>>(p, scan_begin, m, lo, span, a);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cub::DeviceRadixSort::SortKeys(tmp, tmp_bytes, a, b, (int64_t)m, 0, end_bit, st);
    if (e == cudaSuccess && count && (steps_dev || ids_dev)) {
        const unsigned grid = (unsigned)std::min<uint64_t>((count + 255) / 256, (uint64_t)n_sm * 16);
        k_raster_split<<<grid, 256, 0, st>>>(b, count, step_begin, steps_dev, ids_dev);
        e = cudaGetLastError();
    }
    unsigned long long edge[2] = {0ull, ~0ull};         // keys n - 1 and n
    if (e == cudaSuccess) e = cudaMemcpyAsync(edge, b + (n - 1), (n < m ? 2 : 1) * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && steps_dev) e = cudaMemcpyAsync(steps_host, steps_dev, (size_t)count * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && ids_dev) e = cudaMemcpyAsync(ids_host, ids_dev, (size_t)count * 4, cudaMemcpyDeviceToHost, st);
    if (a) cudaFreeAsync(a, st);
    if (b) cudaFreeAsync(b, st);
    if (steps_dev) cudaFreeAsync(steps_dev, st);
    if (ids_dev) cudaFreeAsync(ids_dev, st);
    if (tmp) cudaFreeAsync(tmp, st);
    const cudaError_t e2 = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = e2;
    *consistent = (edge[0] != ~0ull) && (edge[1] == ~0ull);
    return e;
}

}  // namespace dbk
