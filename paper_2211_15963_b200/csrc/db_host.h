// Host-side interfaces between the translation units of the library.
#pragma once
#include <cstdint>
#include <string>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/db_b200.h"
#include "db_device.cuh"

namespace dbk {

// ---- db_step.cu ------------------------------------------------------------
cudaError_t launch_init_state(const SimDev& p, const uint8_t* ntype_dev, const float* iext_tab_dev /*[types][65536] or NULL*/, cudaStream_t st);
cudaError_t prepare_kernels();                                            // per handle, on its device: opt-in shared-memory sizes
cudaError_t launch_update(const SimDev& p, int n_sm, int mode, cudaStream_t st);   // mode: see k_update_stream
cudaError_t launch_deliver(const SimDev& p, int grid, unsigned parity, cudaStream_t st);   // parity = step & 1 (list mode: which work-list half)
// DB_EXEC_KERNELS_DEFERRED: sort the rows [row0, row1) by (delay, target window) into scratch arrays indexed by
// (synapse - s0); add the records waiting in the arrival lists to a DB_FIELD_RING read-out
cudaError_t launch_sort_rows(const SimDev& p, int n_sm, int64_t row0, int64_t row1, int64_t s0, uint32_t* tgt_out, void* w_out,
                             uint8_t* delay_out, uint32_t* seg, cudaStream_t st);
cudaError_t launch_deliver_external(const SimDev& p, int n_sm, const int32_t* ids_dev, unsigned n_ids, unsigned long long step, cudaStream_t st);
cudaError_t launch_delay_hist(const uint8_t* delay, int64_t n, unsigned long long* hist /*[256], zeroed*/, int n_sm, cudaStream_t st);
cudaError_t launch_lists_to_ring(const SimDev& p, int n_sm, int32_t* out, int first, int count, int D_api, cudaStream_t st);
cudaError_t persistent_fits(const SimDev& p, bool heavy, int n_sm, bool* ok);
cudaError_t launch_persistent(const SimDev& p, bool heavy, unsigned n_steps, int n_sm, cudaStream_t st);

// ---- db_raster.cu ----------------------------------------------------------
// the raster entries at positions [scan_begin, scan_begin + m) whose step lies in [lo, lo + span), sorted by (step, id):
// keys (step - step_begin) << 32 | id, entries of other steps sort behind them as ~0
cudaError_t raster_pool_setup(int device);                                 // per handle: keep the read-back scratch in the stream-ordered pool
cudaError_t raster_sorted_read(const SimDev& p, int n_sm, uint64_t scan_begin, uint64_t m, uint32_t lo, uint32_t span, uint64_t n,
                               uint64_t step_begin, uint64_t* steps_host, int32_t* ids_host, uint64_t cap, bool* consistent,
                               cudaStream_t st);

// ---- db_bold.cu ------------------------------------------------------------
cudaError_t launch_bold_init(const BoldDev& b, int n_regions, cudaStream_t st);
cudaError_t launch_bold(const SimDev& p, const BoldDev& b, cudaStream_t st);   // consume the completed windows

// ---- db_gen.cu -------------------------------------------------------------
struct GenHostTables {                 // distribution tables formed on the host in double
    std::vector<int64_t> region_start; // [R + 1]
    std::vector<int32_t> region_nexc;  // [R]
    std::vector<uint32_t> region_cdf;  // [R][R - 1] cumulative thresholds of the inter-region matrix
    std::vector<float> weight_tab;     // [65536] lognormal quantiles
    std::vector<int32_t> outdeg_tab;   // [65536] (mode 1)
    int32_t K_intra = 0, K_inter = 0;
};

double std_normal_quantile(double p);   // inverse normal CDF (Newton on erfc), double precision
double gamma_quantile(double p, double shape, double scale);   // inverse Gamma CDF, double precision

bool gen_host_tables(const db_network_spec& spec, uint64_t seed, GenHostTables* out, std::string* err);

struct GenAlloc { void* user; void* (*alloc)(void* user, size_t bytes); };

struct GenResult {
    int64_t* row_begin = nullptr; int32_t* row_len = nullptr;
    uint32_t* tgt_rec = nullptr; void* w = nullptr; uint8_t* delay = nullptr;
    int64_t E = 0, Epad = 0;
    uint64_t work_cap = 0;
    uint64_t heavy_chunks = 0;      // chunks of the rows longer than kInlineMax
    int32_t max_delay = 0;
    bool oom = false;
};

// Builds the presynaptic-major CSR on the device.  Returns a CUDA error, or
// cudaSuccess with *err non-empty for spec / memory problems.
cudaError_t generate_network(const db_network_spec& spec, uint64_t seed, const GenHostTables& tabs,
                             const GenAlloc& ga, cudaStream_t st, int32_t Npad, uint8_t* ntype_dev,
                             GenResult* out, std::string* err);

}  // namespace dbk
