/* ============================================================================
 * db_b200.h -- C ABI of the B200-native single-GPU step loop of the Digital
 * Brain spiking-network simulator (arXiv 2211.15963).
 *
 * "P:L<n>" = line n of PAPER.md; "R<n>" = reading n in DESIGN.md.
 *
 * One iteration (SI "Numerical method" P:L469-490, Supp. Alg. 2
 * P:L869-884):
 *   neuron update   conductances  J_u(t+dt) = exp(-dt/tau_u) J_u(t) + arrivals   (SI Eq.(3))
 *                   membrane      C dV/dt = -g_L (V - V_L) + sum_u g_u (V_u - V) J_u + I_bg + I_ext
 *                                 stepped with first-order Euler (SI Eq.(5), R1)
 *                   threshold / reset / refractory clamp
 *   spike list      stack the spiking neurons                                    (Alg. 2 line 2)
 *   delivery        push each spike along its destination list into the delayed,
 *                   fixed-point per-receptor ring buffer with integer atomics    (Alg. 2 l.3-4)
 *   region rates    firing rate of neuron groups
 *
 * Conventions
 *   - Every function returns int32_t: DB_OK (0) or a negative DB_E* code; text
 *     is available from db_last_error().  Nothing throws or aborts across the ABI.
 *   - `db_sim` is opaque and owned by the library; db_destroy() frees it and all
 *     device memory it obtained (through db_runtime.alloc/free when given, else
 *     cudaMalloc/cudaFree).
 *   - All pointer arguments are HOST pointers unless the name ends in `_dev`.
 *     Output buffers are caller-allocated with a capacity in elements; the call
 *     writes at most that many and reports the total available.
 *   - All device work is enqueued on db_runtime.stream (a cudaStream_t; NULL =
 *     the legacy default stream).  db_step() is asynchronous; every db_read_* /
 *     db_get_* / db_export_* call synchronises that stream first.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - There is no CPU fallback: without a CUDA device every create call fails
 *     with DB_ECUDA.
 * ==========================================================================*/
#ifndef DB_B200_H
#define DB_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DB_OK       0
#define DB_EINVAL  (-1)   /* bad argument / spec out of the supported range */
#define DB_ENOMEM  (-2)   /* host or device allocation failed */
#define DB_ECUDA   (-3)   /* CUDA runtime error (no device, launch failure, ...) */
#define DB_ERANGE  (-4)   /* requested steps / elements are not (or no longer) available */
#define DB_ESTATE  (-5)   /* call not valid in the current state of the handle */

#define DB_MAX_TYPES 8    /* neuron types, each with its own constants (property table P:L816-832 held per type, R-D1): the generator
                             uses 0 = excitatory, 1 = inhibitory; a CSR may use all eight (e.g. the populations of a micro-column,
                             Ext. Table 3, or (region group, type) pairs) */
#define DB_N_RECEPTORS 4  /* 0 AMPA, 1 NMDA, 2 GABA_A, 3 GABA_B */

typedef struct db_sim db_sim;

/* Per neuron type constants: the paper's property table (Supp. Table 5,
 * P:L816-832), held per type instead of per neuron (R-D1).  Units ms / mV;
 * with C = 1, g_L = 1/tau_m. */
typedef struct db_type_params {
    double C, gL, VL, Vth, Vreset, Tref_ms, Iext;
    double G[DB_N_RECEPTORS];       /* g_u, maximal conductance */
    double E[DB_N_RECEPTORS];       /* V_u, reversal potential */
    double tau_ms[DB_N_RECEPTORS];  /* tau_u */
    double bg_rate_hz;              /* Poisson background rate per neuron (R14) */
    double bg_weight;               /* its weight; delivered to AMPA */
    /* OU background current (main Eq.(1), SI Eq.(4); Ext. Table 2: mu 0.66, sigma
     * 0.12, tau 10), read per R3: I += (mu - I) dt/tau + sigma sqrt(2 dt/tau) xi, xi ~ N(0,1) from a
     * 65536-point quantile table; enters the membrane equation as a current.  ou_tau_ms = 0: off. */
    double ou_mu, ou_sigma, ou_tau_ms;
    /* External current per neuron ("I_ext,i are parameters, independently sampled following a Gamma
     * distribution"; property table; reading R31): I_ext,i = Iext + Gamma(shape, scale), drawn once per neuron at
     * creation through a 65,536-point quantile table (top 16 bits of a Philox word keyed by dyn_seed, stream 9, neuron).
     * iext_gamma_shape = 0: every neuron of the type gets Iext.  When any type uses it the currents are an extra fp32
     * plane the update streams (+4 B per neuron-step); readable and writable as DB_FIELD_IEXT. */
    double iext_gamma_shape, iext_gamma_scale;
} db_type_params;

/* Balloon-Windkessel BOLD read-out per region (Extended Data Table 4; reading R30): one explicit Euler
 * step per completed region-rate window (step length = window_steps * dt), z = z_scale * region rate in Hz, state
 * (s, f, v, q) starts at rest (0, 1, 1, 1).  The paper prints no constants; the usual ones of its reference 19
 * are kappa 0.65 /s, gamma 0.41 /s, tau 0.98 s, alpha 0.32, rho 0.34, V0 0.02, k1 7 rho, k2 2, k3 2 rho - 0.2. */
typedef struct db_bold_params {
    int32_t enabled;                /* 0: no BOLD read-out (db_read_bold returns DB_ESTATE) */
    int32_t reserved;
    double kappa, gamma, tau, alpha, rho, V0, k1, k2, k3, z_scale;
} db_bold_params;

/* Execution mode of db_step(). */
#define DB_EXEC_AUTO       0   /* library picks */
#define DB_EXEC_KERNELS    1   /* two kernels per step (update+compaction, delivery), CUDA-graph replayed */
#define DB_EXEC_PERSISTENT 2   /* one cooperative persistent kernel looping over the steps */
#define DB_EXEC_KERNELS_DEFERRED 3 /* two kernels per step with ARRIVAL LISTS: a row is read once, when its neuron fires, and every
                                      synapse becomes an 8-byte record in the list of its arrival step (rows sorted by delay, one
                                      atomic per run); the kernel of step n streams the list of step n + 1 into ring slot n + 1, the
                                      only slot that takes reductions, so they stay in L2 and DRAM only streams.  Same results.
                                      Falls back to DB_EXEC_KERNELS when no delay exceeds 1 step or memory is short */

typedef struct db_sim_params {
    uint32_t struct_size;     /* = sizeof(db_sim_params) */
    double   dt_ms;           /* 0.1 or 1 */
    int32_t  S;               /* fixed-point shift of the ring: increment = lrintf(w * 2^S) (R28) */
    int32_t  D;               /* ring depth in steps: power of two, > largest delay */
    int32_t  window_steps;    /* region-rate window in steps (R24) */
    int32_t  n_types;         /* 1..DB_MAX_TYPES */
    db_type_params type[DB_MAX_TYPES];
    uint64_t dyn_seed;        /* keys V0 and the Poisson background */
    uint64_t raster_capacity; /* spikes kept for db_read_spikes (0 = default); older ones are overwritten */
    uint32_t max_windows;     /* region-rate windows kept (0 = default 4096) */
    int32_t  exec_mode;       /* DB_EXEC_* */
    int32_t  spike_bin_steps; /* time bin b_t for transferring spikes, in steps (SI "Numerical method" P:L471-490:
                                 b_t = 1 ms even at dt = 0.1 ms; reading R29): a neuron that fires in step n is
                                 transferred at the end of its bin, step n_k = b_t floor(n / b_t) + b_t - 1, and a
                                 synapse of delay d is read in step n_k + d.  0 or 1: every step is a boundary.
                                 Needs b_t <= R + 1 of every type (A_j is 0 or 1) and largest delay + b_t - 1 < D;
                                                                  DB_FIELD_RING already holds the pushes of the spikes of the open bin. */
    db_bold_params bold;      /* BOLD read-out per region, fed by the region-rate windows (off by default) */
} db_sim_params;

/* Device memory and stream plumbing supplied by the caller (the Python binding
 * backs alloc/free with torch tensors and passes torch's current stream). */
typedef struct db_runtime {
    void* (*alloc)(size_t bytes, void* user);   /* returns a DEVICE pointer, 256-byte aligned, or NULL */
    void  (*free)(void* dev_ptr, void* user);
    void*  user;
    void*  stream;                               /* cudaStream_t */
    int32_t device;                              /* CUDA device ordinal */
} db_runtime;

/* Synthetic network (stand-in for the paper's HRGCME generator, P:L408-439,
 * P:L322-331; recipe in DESIGN.md "Generator"). */
#define DB_MODE_FIXED_INDEGREE  0
#define DB_MODE_OUTDEG_LOGNORMAL 1
typedef struct db_network_spec {
    uint32_t struct_size;        /* = sizeof(db_network_spec) */
    int64_t  N;                  /* neurons, 2 <= N < 2^30 */
    int32_t  n_regions;          /* contiguous id ranges; excitatory neurons first in each */
    double   region_size_sigma;  /* sizes ~ lognormal(0, sigma), normalised to N */
    double   exc_frac;           /* 0.8 */
    int32_t  mode;               /* DB_MODE_* */
    int32_t  K;                  /* in-degree per neuron (mode 0) */
    double   intra_frac;         /* share of K drawn inside the own region (n_regions > 1) */
    double   region_matrix_sigma;/* inter-region matrix ~ lognormal(0, sigma), zero diagonal, row-normalised */
    double   outdeg_mean, outdeg_sigma; int32_t outdeg_cap;   /* mode 1 (R27) */
    double   w_mu, w_sigma, w_scale, inh_mult, slow_frac;     /* weights (R11), NMDA / GABA_B share (R12) */
    int32_t  delay_intra_min, delay_intra_max, delay_inter_min, delay_inter_max;  /* steps, 1..255 */
    int32_t  weight_fp16;        /* store weights as binary16 (config 3) instead of fp32 */
    int64_t  own_first, own_count; /* region-sharded simulation (SI Eq.(6); layout P:L494): the handle owns
                                    the neurons [own_first, own_first + own_count) of the N-neuron network -- their state, their
                                    ring, and the synapses ONTO them from every source; own_first a multiple of 1024;
                                    own_count = 0: the whole network.  DB_MODE_FIXED_INDEGREE only.  Ids in the raster, in
                                    db_read_state / db_write_state and in db_deliver_external are global */
    db_sim_params sim;
    const db_runtime* runtime;   /* may be NULL */
} db_network_spec;

/* A presynaptic-major CSR on the HOST: row j = destination list of neuron j. */
typedef struct db_csr_view {
    int64_t N, E;
    int32_t n_regions;
    const int64_t* region_start; /* [n_regions + 1] */
    const uint8_t* ntype;        /* [N] neuron type index */
    const int64_t* row_ptr;      /* [N + 1] */
    const int32_t* tgt;          /* [E] target neuron */
    const float*   w;            /* [E] weight */
    const uint8_t* delay;        /* [E] delay in steps, 1 <= delay < D */
    const uint8_t* rec;          /* [E] receptor 0..3 */
    int32_t weight_fp16;         /* store on the device as binary16 (w must already be representable) */
    int64_t own_first, own_count; /* as in db_network_spec: keep only the synapses onto [own_first, own_first + own_count); 0, 0 = all */
} db_csr_view;

/* Library-allocated host copy of the network (db_export_csr); release with db_free_csr. */
typedef struct db_csr_host {
    int64_t N, E;
    int32_t n_regions;
    int64_t* region_start; uint8_t* ntype; int64_t* row_ptr;
    int32_t* tgt; float* w; uint8_t* delay; uint8_t* rec;   /* rows sorted by (target, receptor) */
} db_csr_host;

typedef struct db_counters {
    uint64_t steps;        /* time steps done */
    uint64_t spikes;       /* spikes emitted */
    uint64_t events;       /* synaptic events delivered = sum of out-degrees of spiking neurons */
    uint64_t bg_events;    /* background Poisson events drawn */
    uint32_t ring_overflow;/* sticky: some consumed ring cell exceeded 2^30 in magnitude (R28) */
    uint32_t exec_mode;    /* DB_EXEC_* actually in use */
    uint64_t launches;     /* kernels launched by db_step / db_step_profiled on this handle */
    uint64_t list_spilled; /* DB_EXEC_KERNELS_DEFERRED: records that found their arrival list full and were reduced into
                              the ring directly (exact either way; a capacity diagnostic) */
} db_counters;

/* Per-phase device time of the last db_step_profiled() call, in milliseconds. */
typedef struct db_phase_times {
    double update_ms;      /* neuron update + compaction (a1 + a2 + a4) */
    double deliver_ms;     /* spike delivery (a3) */
    double total_ms;       /* whole call on the stream */
    uint64_t steps, spikes, events;   /* work done inside the call */
} db_phase_times;

#define DB_FIELD_V      0  /* float  [count] */
#define DB_FIELD_G_AMPA 1  /* float  [count] */
#define DB_FIELD_G_NMDA 2
#define DB_FIELD_G_GABAA 3
#define DB_FIELD_G_GABAB 4
#define DB_FIELD_REF    5  /* int32  [count], refractory steps left */
#define DB_FIELD_TYPE   6  /* uint8  [count] */
#define DB_FIELD_RING   7  /* int32  [D][count][4] fixed-point arrivals, slot = step mod D */
#define DB_FIELD_OUTDEG 8  /* int32  [count], out-degree = length of the neuron's destination list (read only) */
#define DB_FIELD_IOU    9  /* float  [count], OU background current (zeros when no type uses it) */
#define DB_FIELD_IEXT  10  /* float  [count], external current of every neuron (R31); writable only when the plane exists */

/* a0: generate the network on the device from `spec` (seed keys every draw of
 * the generator), build the CSR and initialise the state (V0 keyed by
 * spec->sim.dyn_seed). */
int32_t db_create(const db_network_spec* spec, uint64_t seed, db_sim** out);

/* Same, from a host CSR (tests, tiny networks, externally built networks). */
int32_t db_create_from_csr(const db_sim_params* sim, const db_csr_view* csr,
                           const db_runtime* runtime, db_sim** out);

int32_t db_destroy(db_sim* sim);

/* a1-a4 (one iteration per time step: SI "Numerical method" P:L469-490, Supp. Alg. 2) for n_steps consecutive
 * time steps; asynchronous on the stream. */
int32_t db_step(db_sim* sim, uint32_t n_steps);

/* Region-sharded simulation, second sum of SI Eq.(6): the neurons `ids` [n] (global ids, HOST pointer; neurons
 * this handle does NOT own) fired in time step `step`; their synapses onto the handle's neurons are pushed into its ring
 * (arrival = end of the spike's time bin + delay).  To be called before the handle steps past `step` + the smallest
 * delay of the network: DB_ERANGE otherwise (the arrival step would already be consumed), DB_EINVAL for an id out of
 * range or owned by the handle.  Two handles that exchange their db_read_spikes output every d_min steps reproduce the
 * single-handle simulation bit for bit (tests).  Asynchronous on the stream like db_step. */
int32_t db_deliver_external(db_sim* sim, uint64_t step, const int32_t* ids, uint64_t n);

/* The lists of n_steps (1..4096) consecutive time steps in one call and one kernel launch: ids[offsets[s] .. offsets[s + 1])
 * (HOST pointers; offsets[0] = 0, non-decreasing, offsets[n_steps] = number of ids) fired in step step_begin + s -- the
 * layout db_read_spikes returns a step range in.  Same checks as db_deliver_external, applied to the first and the last
 * step of the window that carry spikes; same result as one db_deliver_external call per step.  This is the call of the
 * exchange step of a sharded run (every d_min steps, SI Eq.(6)). */
int32_t db_deliver_external_window(db_sim* sim, uint64_t step_begin, uint32_t n_steps, const uint64_t* offsets, const int32_t* ids);

/* The exchange step without the host in the data path, for shards held by ONE process (several handles on one GPU, or on
 * GPUs with peer access: NVLink / NVSwitch): `sim` pushes the rows of the spikes that `src` -- another shard of the same
 * network -- fired in the steps [step_begin, step_end), reading them straight out of src's raster ring in device memory
 * (peer-mapped when src lives on another GPU; DB_ESTATE when the devices have no peer access).  One kernel on sim's
 * stream, ordered after the steps src has launched so far; no sort, no list, no copy (the reductions commute), and the call
 * itself neither waits nor reads back unless src's raster ring is so small that the range might have been overwritten
 * (then it checks, which waits for src's stream).  src may step on, but must not be destroyed, and must not log more than
 * its raster capacity of new spikes, until sim's stream has passed this point.  Errors as db_deliver_external, applied to
 * the first and the last step of the range (DB_ERANGE: too late / too early for sim's ring, steps src has not simulated
 * or no longer holds); same result as db_read_spikes on src followed by db_deliver_external_window on sim (tests).
 * Between processes (one per GPU under torchrun) the lists travel by all-gather instead:
 * paper_2211_15963_b200/sharded.py. */
int32_t db_exchange_peer(db_sim* sim, db_sim* src, uint64_t step_begin, uint64_t step_end);

/* The same operation for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): identical arguments, checks and result (the ring cells and the event counter get the
 * same integers), but the device copy of `ids` lives in a static device array of DB_EXTERNAL_STATIC_MAX ids (256 KB that
 * every GPU which loads the library holds until the process exits) instead of a buffer db_deliver_external grows on
 * demand.  Calls no cudaMalloc / cudaFree and no allocating library routine.  n > DB_EXTERNAL_STATIC_MAX: DB_EINVAL
 * (db_last_error says so); split the list, or use db_deliver_external.  All handles on one device share the array and it
 * keeps the last call's list: a call overwrites the entries it reads (nothing needs clearing), and two calls that overlap
 * on the GPU (handles on different streams of the same device) race -- serialise them. */
#define DB_EXTERNAL_STATIC_MAX 65536
int32_t db_deliver_external_static(db_sim* sim, uint64_t step, const int32_t* ids, uint64_t n);

/* Same in DB_EXEC_KERNELS mode with CUDA events around every kernel; blocks
 * until done.  For per-kernel roofline measurement. */
int32_t db_step_profiled(db_sim* sim, uint32_t n_steps, db_phase_times* out);

/* a5, the simulator's first output (Supp. Alg. 2 "Output: spike trains"; recorded per ms in the paper).
 * Spikes with step_begin <= step < step_end, sorted by (step, id).  Writes at
 * most `cap` pairs, *n_out = number available.  DB_ERANGE if part of the range
 * was already overwritten in the raster ring or lies in the future. */
int32_t db_read_spikes(db_sim* sim, uint64_t step_begin, uint64_t step_end,
                       uint64_t* steps, int32_t* ids, uint64_t cap, uint64_t* n_out);

/* a5, the second output (Alg. 2 "Output: ... membrane potentials"; "state variables of neurons"): state of
 * the neurons [first, first + count) -- GLOBAL ids, inside the range the handle owns -- into dst (layout per DB_FIELD_*).
 * DB_FIELD_RING = the arrivals still to come, in every execution mode (ring content plus records waiting in arrival lists). */
int32_t db_read_state(db_sim* sim, uint32_t field, int64_t first, int64_t count, void* dst);
/* Overwrite state: the test hook of the identical-state one-step parity case, and how an outer loop (the paper's
 * assimilation, out of scope here) replaces parameters such as DB_FIELD_IEXT.  DB_FIELD_RING only before the
 * first step when arrival lists are in use (DB_ESTATE otherwise). */
int32_t db_write_state(db_sim* sim, uint32_t field, int64_t first, int64_t count, const void* src);

/* a4 (K7 "firing rates of neuron groups"; "over a sliding window").
 * Firing rate in Hz per (window, region) for the completed windows still kept:
 * spikes / (region size * window seconds) (R24).  rates_hz[w * n_regions + r];
 * *first_window = index of the first window returned. */
int32_t db_region_rates(db_sim* sim, float* rates_hz, uint64_t cap_windows,
                        uint64_t* n_windows, uint64_t* first_window);
/* The integer counts behind them (same indexing). */
int32_t db_region_counts(db_sim* sim, uint32_t* counts, uint64_t cap_windows,
                         uint64_t* n_windows, uint64_t* first_window);

/* BOLD signal of every region after the last completed region-rate window: y [n_regions] and, if `state` is not
 * NULL, the model state [n_regions][4] = (s, f, v, q); HOST buffers owned by the caller, fp64.  *n_windows (may be
 * NULL) = windows consumed so far.  Synchronises the stream.  DB_ESTATE when the read-out was not enabled. */
int32_t db_read_bold(db_sim* sim, double* y, double* state, uint64_t* n_windows);

int32_t db_export_csr(db_sim* sim, db_csr_host* out);
int32_t db_free_csr(db_csr_host* csr);

int32_t db_get_counters(db_sim* sim, db_counters* out);
int32_t db_synchronize(db_sim* sim);

/* Text of the last error on this handle (sim == NULL: last create error of this thread). */
const char* db_last_error(const db_sim* sim);

#ifdef __cplusplus
}
#endif
#endif /* DB_B200_H */
