// Device-side data layout of one simulation (HBM), shared by the step kernels,
// the generator and the C ABI.  See DESIGN.md "Data layout".
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dbk {

constexpr int kMaxTypes = 8;          // neuron types with their own constants (rt keeps the type in 4 bits); 8 = the populations of a micro-column (Ext. Table 3)
constexpr int kPoissonMax = 32;
constexpr int kNeuronPad = 1024;     // Npad is a multiple of this: whole warps, 128-bit accesses
constexpr int kRowAlign = 4;         // CSR rows start on a multiple of 4 synapses (128-bit target loads)
constexpr int kChunk = 512;          // synapses per delivery work item (one warp)
constexpr int kInlineMax = 1024;     // persistent kernel: rows up to this length are delivered by the warp that found the spike
constexpr int kRunThreads = 640;     // persistent kernel: most threads per block (one block per SM); 96 registers per thread (measured: 512 .. 1024 threads, profiles/r1s_threads_per_block.md)
constexpr int kRefMask = 0x0FFF;     // rt = type << 12 | refractory steps left

// Philox streams
constexpr uint32_t kStreamV0 = 1, kStreamBG = 2, kStreamSRC = 3, kStreamSYN = 4,
                   kStreamREGION = 5, kStreamINTER = 6, kStreamDEG = 7, kStreamOU = 8, kStreamIEXT = 9;

struct TypeConst {                   // per neuron type, rounded once on the host
    float neg_gL, VL, Vth, Vreset, kappa, Iext;
    float G[4], E[4], alpha[4];
    int32_t R;                       // refractory steps
    int32_t wq_bg;                   // fixed-point background weight
    int32_t M;                       // number of Poisson thresholds
    uint32_t T[kPoissonMax];
    float ou_mu, ou_a, ou_s;         // OU background: mean, dt / tau, sigma sqrt(2 dt / tau) (0 when off)
    int32_t ou;                      // OU background on for this type
    int32_t ix_on;                   // external current of the type's neurons has a Gamma part (R31)
};

struct alignas(128) Ctl {            // device-resident control block
    unsigned long long step;         // current time step n
    unsigned long long spike_begin;  // spikes emitted before step n
    unsigned long long step_counts[4];  // [n & 3] of step n: high 32 = spikes, low 32 = work items (one atomic); cleared when step n + 1 closes
    unsigned long long events;       // synaptic events delivered so far
    unsigned long long spike_cursor; // persistent kernel: next free raster position (= spike_begin between steps)
    unsigned int overflow;           // sticky ring overflow flag
    unsigned int done_blocks;        // delivery kernel: finished-block ticket
    unsigned long long ev_spilled;   // list mode: records that found their list full and went into the ring instead
    unsigned long long work_step[2]; // [n & 1]: the step whose work list sits in half n & 1 (left by the update kernel for kernel C)
    unsigned int done_lists;         // kernel C: finished-block ticket
    unsigned int pad0[7];
    // persistent kernel (see db_step.cu), on a 128-byte line of their own (every block polls it):
    // arrivals of the blocks that closed unit j go to the monotonic counter [j & 3] (blocks are at most
    // two units apart), the spike count of the step produced by unit j to unit_spikes[j & 3]
    unsigned int bar[4];
    unsigned int unit_spikes[4];
    unsigned int pad1[24];
};
static_assert(sizeof(Ctl) == 256, "Ctl layout");

constexpr int kBgParts = 1024;       // background-event counter is spread over this many cells

struct SimDev {                      // passed by value to every kernel
    int32_t N, Npad;                 // neurons this handle owns (state, ring, targets are indexed 0 .. N - 1)
    int32_t id0, n_rows;             // global id of its first neuron (a multiple of 1024), neurons of the whole network = CSR rows
    int32_t D, S;
    float scale;                     // 2^-S
    float wscale;                    // 2^S
    uint32_t seed_lo, seed_hi;
    uint32_t rk[20];                 // Philox round keys of the dynamics seed: (k0, k1) + r * (0x9E3779B9, 0xBB67AE85), r = 0..9
    // neuron state, structure of arrays
    float* V;                        // [Npad]
    float* g;                        // [4][Npad]
    uint16_t* rt;                    // [Npad] type << 12 | ref
    float* Iou;                      // [Npad] OU background current (allocated only if some type uses it)
    const float* ntab;               // [65536] standard-normal quantiles (same condition)
    int32_t ou_on;
    float* iext;                     // [Npad] external current per neuron (R31; allocated only if some type draws it from a Gamma law)
    int32_t bg_on;                   // some type has a Poisson background (else its Philox draw is skipped)
    int32_t bin_steps;               // time bin b_t for transferring spikes, in steps (>= 1; R29)
    int32_t* ring;                   // [D][4][Npad] fixed-point arrivals
    // presynaptic-major CSR
    const int64_t* row_begin;        // [N] first synapse of row j (multiple of kRowAlign)
    const int32_t* row_len;          // [N]
    const uint32_t* tgt_rec;         // [Epad] receptor << 30 | target
    const void* w;                   // [Epad] float or __half
    const uint8_t* delay;            // [Epad]
    int32_t w_fp16;
    // DB_EXEC_KERNELS_DEFERRED: arrival lists (db_step.cu).  8-byte records (receptor << 30 | target, fixed-point weight)
    // waiting for their arrival step.  Lists are private to the blocks of the delivery kernel: block b owns one list per
    // cursor index c = slot * ev_W + window (near family: slot = arrival & (ev_Dn - 1); far family after it: slot = arrival
    // & (ev_D - 1)); its records start at ev_rec[(c * ev_P + b) * capacity] and its cursor is ev_cnt[b * ev_n_cur + c]
    // between launches (shared memory during one)
    int32_t ev_on;                   // 0: every synapse is pushed into the ring when its neuron fires
    int32_t ev_direct;               // arrivals <= this many steps ahead (1) go straight into the ring
    int32_t ev_near_lim;             // arrivals <= this many steps ahead go to the near family (ring of ev_Dn slots)
    int32_t ev_near_d;               // delays <= this are near whatever the position in the time bin: ev_near_lim - (b_t - 1)
    const uint32_t* seg;             // [N][ev_near_d * ev_W + 1] rows sorted by (delay, window): first synapse (relative to the row) of every
                                     // (delay, window) run of the near part; the last entry starts the far part
    int32_t ev_Dn, ev_D;             // slots of the near / far family (powers of two; ev_D = D)
    int32_t ev_W, ev_P;              // target windows per slot (1, 2 or 4), blocks of the delivery kernel (= lists per cursor index)
    int32_t ev_n_cur, ev_n_far;      // cursor indices per block (both families); ev_n_far = 0: no delay beyond ev_near_lim
    uint32_t ev_cap_near, ev_cap_far;// records per list
    uint32_t ev_wb[3];               // first neuron of the windows 1, 2, 3 (0xFFFFFFFF when unused)
    uint2* ev_rec;                   // near lists, then far lists
    unsigned* ev_cnt;
    // spike list = raster ring; per-step work list
    int32_t* spike_ids;              // [spike_cap] circular
    uint32_t* spike_tag;             // [spike_cap] low 32 bits of the step of each entry (steps may interleave by one)
    unsigned long long spike_mask;
    int2* work;                      // [2][work_half] (neuron, chunk) of the steps n & 1 = 0 / 1 (kernel B of step n may run beside the update of n + 1)
    unsigned long long work_half;
    unsigned long long* step_end;    // [step_log_cap] circular: spikes emitted up to and including step n
    uint32_t step_log_mask;
    // regions
    const int32_t* region_start;     // [n_regions + 1]
    int32_t n_regions;
    uint32_t* region_counts;         // [max_windows][n_regions] circular
    int32_t window_steps;
    uint32_t max_windows;
    unsigned long long* bg_parts;    // [kBgParts]
    Ctl* ctl;
    TypeConst tc[kMaxTypes];
};

struct BoldDev {                     // Balloon-Windkessel read-out (db_bold.cu); kept out of SimDev: not on the step path
    double* state;                   // [n_regions][4] s, f, v, q
    double* y;                       // [n_regions]
    const double* scale;             // [n_regions] z_scale / (region size * window seconds)
    unsigned long long* cursor;      // next window to consume
    double kappa, gamma, tau, alpha, rho, V0, k1, k2, k3;
    double h;                        // Euler step = window seconds
};

}  // namespace dbk
