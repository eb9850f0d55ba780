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

// keys_host gets min(n + 1, m) keys (the one after the last is there for the consistency check of the caller).
// Keep the scratch of the last calls in the device's stream-ordered pool (default: everything goes back to the OS at
// every synchronize).  The pool belongs to the device: set once per handle, on the handle's device.
cudaError_t raster_pool_setup(int device) {
    cudaMemPool_t pool = nullptr;
    unsigned long long keep = 256ull << 20;
    cudaError_t e = cudaDeviceGetDefaultMemPool(&pool, device);
    if (e == cudaSuccess) e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    return e;
}

cudaError_t raster_sorted_keys(const SimDev& p, int n_sm, uint64_t scan_begin, uint64_t m, uint32_t lo, uint32_t span, uint64_t n,
                               std::vector<unsigned long long>* keys_host, cudaStream_t st) {
    unsigned long long *a = nullptr, *b = nullptr;
    void* tmp = nullptr;
    size_t tmp_bytes = 0;
    cudaError_t e = cudaMallocAsync(&a, (size_t)m * 8, st);
    if (e == cudaSuccess) e = cudaMallocAsync(&b, (size_t)m * 8, st);
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
    if (e == cudaSuccess) {
        keys_host->resize((size_t)std::min<uint64_t>(n + 1, m));
        e = cudaMemcpyAsync(keys_host->data(), b, keys_host->size() * 8, cudaMemcpyDeviceToHost, st);
    }
    if (a) cudaFreeAsync(a, st);
    if (b) cudaFreeAsync(b, st);
    if (tmp) cudaFreeAsync(tmp, st);
    const cudaError_t e2 = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = e2;
    return e;
}

}  // namespace dbk
