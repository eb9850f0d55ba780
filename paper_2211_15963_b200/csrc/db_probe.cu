// Measurement aid, not on the step path: the rate at which the device retires 4-byte integer reductions
// (red.global.add.s32, the instruction of a3) to uniformly random cells of a region of a given size.  Spike
// delivery is a scatter of such reductions; when the ring is far larger than L2 every one of them is a random
// 32-byte-sector DRAM access, and the bound that matters is the device's random-access rate, not its streaming
// bandwidth.  bench.py reports the delivery kernels against this number next to the HBM roofline.
//
// Built into its own bench-only helper library (libdb_probe.so), NOT into libdb_b200.so: it is not part of the product ABI.
//   int32_t db_probe_scatter(int32_t device, uint64_t region_bytes, uint64_t n_ops, uint32_t reps, double* ops_per_s)
//   `n_ops` reductions per launch into a scratch region of `region_bytes` (allocated and freed inside; >= 4), `reps` timed
//   launches after one warm-up, CUDA events on the default stream; *ops_per_s: HOST.  Returns 0, or -1 bad argument,
//   -2 out of memory, -3 CUDA error.
#include <cstdint>
#include <cuda_runtime.h>
#define DB_OK 0
#define DB_EINVAL (-1)
#define DB_ENOMEM (-2)
#define DB_ECUDA (-3)

namespace dbk {

__global__ void __launch_bounds__(256) k_probe_scatter(int32_t* __restrict__ region, const uint64_t n_cells,
                                                       const uint64_t ops_per_thread, const uint32_t salt) {
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint64_t x = (t + 1) * 0x9E3779B97F4A7C15ull + salt;           // xorshift64* stream per thread
    for (uint64_t k = 0; k < ops_per_thread; ++k) {
        x ^= x >> 12; x ^= x << 25; x ^= x >> 27;
        const uint64_t r = x * 0x2545F4914F6CDD1Dull;
        const uint64_t cell = (uint64_t)(((unsigned __int128)r * n_cells) >> 64);
        asm volatile("red.global.add.s32 [%0], %1;" :: "l"(region + cell), "r"(1) : "memory");
    }
}

}  // namespace dbk

extern "C" int32_t db_probe_scatter(int32_t device, uint64_t region_bytes, uint64_t n_ops, uint32_t reps, double* ops_per_s) {
    using namespace dbk;
    if (!ops_per_s || region_bytes < 4 || n_ops == 0 || reps == 0) return DB_EINVAL;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return DB_ECUDA;
    if (cudaSetDevice(device) != cudaSuccess) return DB_ECUDA;
    cudaDeviceProp prop{};
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return DB_ECUDA;
    int32_t* region = nullptr;
    if (cudaMalloc(&region, region_bytes) != cudaSuccess) { cudaGetLastError(); return DB_ENOMEM; }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int32_t rc = DB_OK;
    const int grid = prop.multiProcessorCount * 8, threads = 256;
    const uint64_t per_thread = (n_ops + (uint64_t)grid * threads - 1) / ((uint64_t)grid * threads);
    float ms = 0.0f;
    if (cudaMemset(region, 0, region_bytes) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
        cudaEventCreate(&e1) != cudaSuccess) rc = DB_ECUDA;
    if (rc == DB_OK) {
        k_probe_scatter<<<grid, threads>>>(region, region_bytes / 4, per_thread, 0u);      // warm-up
        cudaEventRecord(e0);
        for (uint32_t r = 0; r < reps; ++r) k_probe_scatter<<<grid, threads>>>(region, region_bytes / 4, per_thread, r + 1u);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess || !(ms > 0)) rc = DB_ECUDA;
    }
    if (rc == DB_OK) *ops_per_s = (double)per_thread * grid * threads * reps / (ms * 1e-3);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(region);
    cudaGetLastError();
    return rc;
}
