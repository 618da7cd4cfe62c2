/*
 * dies.h -- C ABI of libdies: the data-parallel hot path of DIES (arXiv 2408.13807) on one B200.
 *
 * Monte Carlo propagation of photon packages through a 1D spherically symmetric dust cloud of
 * concentric shells with the immediate re-emission (IRE) method (section 2.1),
 * with the weighted sampling schemes of the paper's Table 1 -- initial direction k_bg (Eq. 5),
 * re-emission and scattering directions g_E, g_S (Eq. 6-7), absorption and scattering free paths k_A,
 * k_S, also density dependent (Eq. 8) -- and forced first interaction (Eq. 9-12).  Citations are lines of /root/reference/PAPER.md; "R<n>" are the readings of
 * DESIGN.md.  Every step of the path runs in hand-written sm_100a CUDA kernels; there is no CPU
 * fallback: every entry point that needs the device returns DIES_ECUDA when it is missing.
 *
 * Conventions
 *  - All array arguments are caller-owned HOST pointers unless marked "device"; they are copied
 *    during the call and never kept.  Getters write into caller-owned host buffers.
 *  - The caller allocates the device workspace (dies_workspace_bytes) and keeps it alive until
 *    dies_destroy; the library never allocates device memory for a model.
 *  - All functions return DIES_OK (0) or a negative error code; dies_last_error() gives a
 *    thread-local message.  Nothing is printed, nothing aborts.
 *  - Units are the caller's; only consistency is required: kappa * rho * length dimensionless,
 *    emis and L / (rho * volume) in the same power-per-dust-mass unit.
 *  - A handle is not thread-safe; different handles are independent.
 *  - Shells are numbered 0 (innermost) .. n_shells-1; frequency bins 0 .. n_freq-1.
 *
 * Random numbers (part of the parity contract): Philox4x32-10 with
 * key = (seed lo32, seed hi32), counter = (package_id lo32, package_id hi32, block, model_index);
 * block counts the 4-word blocks consumed by the package from 0; a 32-bit word x gives the
 * uniform u = ((x >> 9) + 0.5) * 2^-23 in (0,1).
 */
#ifndef DIES_H
#define DIES_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dies_model dies_model;   /* opaque; owned by the library, freed by dies_destroy */

enum {
    DIES_OK = 0,
    DIES_EINVAL = -1,      /* bad argument (sizes, ordering, sign, NULL) */
    DIES_ENOMEM = -2,      /* workspace too small or host allocation failed */
    DIES_ECUDA = -3,       /* CUDA runtime error or no sm_100 device */
    DIES_ESTATE = -4,      /* call out of order (e.g. run before set_sources) */
    DIES_EOVERFLOW = -5    /* a 64-bit tally exceeded 2^62 */
};

/* modes of dies_run */
enum { DIES_MODE_IRE = 0, DIES_MODE_FIXED_T = 1,
       /* One iteration of the traditional Monte Carlo (R22): every active source and the
        * dust send n_packages packages each, absorption is tallied continuously along the paths, scatterings are
        * discrete events.  The dust emits, uniformly over every cell (L251), the power per mass the cell absorbed in the
        * PREVIOUS run of the handle (whatever its mode; nothing before the first run), with the cell's emission spectrum.
        * Calling dies_run with this mode repeatedly is the TMC iteration; dies_get_temperature after each run gives the
        * temperatures to watch for convergence (L31).  Plain runs only: k_bg = 0.5, no ffi, no weighting, no accumulate,
        * fixed_shift <= 24 (DIES_EINVAL otherwise; a rejected call leaves the handle, a pending dies_seek included, as
        * it was).  The tallies of a TMC run are in an energy unit that includes the dust luminosity: a later run in
        * another mode cannot accumulate onto them and an IRE-mode trace cannot replay against them (DIES_ESTATE);
        * traces themselves are IRE or fixed-temperature only (DIES_EINVAL for this mode). */
       DIES_MODE_TMC = 2 };

/* event types of dies_trace_* (quadruples: type, shell, freq_bin, crossings so far) */
enum { DIES_EV_LAUNCH = 0, DIES_EV_SCATTER = 1, DIES_EV_ABSORB = 2, DIES_EV_ESCAPE = 3,
       DIES_EV_TERMINATE = 4, DIES_EV_UNINTERACTED = 5 };

/* indices into the array filled by dies_get_counters */
enum { DIES_C_PACKAGES = 0, DIES_C_CROSSINGS, DIES_C_FFI_CROSSINGS, DIES_C_SCATTERINGS, DIES_C_ABSORPTIONS,
       DIES_C_ESCAPED, DIES_C_UNINTERACTED, DIES_C_TERMINATED, DIES_C_EXTRA_BLOCKS, DIES_C_CLAMP_HI_SAMPLES,
       DIES_C_INJECTED_RAW, DIES_C_TERMINATED_RAW, DIES_C_REWEIGHT_RAW, DIES_C_ESCAPED_RAW, DIES_C_T_CLAMP_LO,
       DIES_C_T_CLAMP_HI, DIES_C_KERNEL_LAUNCHES, DIES_N_COUNTERS };
/* Raw (fixed-point) bookkeeping, exact in integers: INJECTED_RAW + REWEIGHT_RAW = ESCAPED_RAW + TERMINATED_RAW.
 * REWEIGHT_RAW is the signed sum (two's complement) of the changes the free-path weights made to package quanta. */

typedef struct {
    double   k_bg;        /* Eq. 5: mu = u^k_bg, W = 2 k_bg mu^(2-1/k_bg); 0.5 = unweighted (Eq. 2)          */
    int32_t  ffi;         /* Eq. 9-12: forced first interaction on the launch flight (R11)                  */
    int32_t  mode;        /* DIES_MODE_IRE, DIES_MODE_FIXED_T (rows from dies_set_fixed_temperature) or _TMC */
    int32_t  accumulate;  /* 0: zero tallies and counters first; 1: continue (package ids continue too)     */
    int32_t  fixed_shift; /* S: a package of weight W adds round(W 2^S) to the 64-bit tallies; 0 -> 24      */
    uint64_t n_total;     /* packages per source over the whole (possibly split) run; package energy is
                             L_source / n_total (L51).  0 -> n_packages of this call                        */
    /* Free-path weighting (section 2.2.2, Eq. 8; R17): the absorption and scattering clocks run
     * k_A and k_S times faster than the true optical depths, p'(tau) = k e^{-k tau}; the package weight follows
     * W = e^{tau (k-1)} / k.  0 means 1 (unweighted).  Not combined with ffi (DIES_EINVAL).                        */
    double   k_A;         /* absorption: everywhere, or at the highest density of the model if k_A_dilute > 0     */
    double   k_A_dilute;  /* > 0: k_A depends on density (L130, L211): this value at the lowest density, k_A at the
                             highest, linear in log(rho) between                                                  */
    double   k_S;         /* scattering                                                                           */
    /* Directional weighting (section 2.2.1, Eq. 6-7; R19).  Angles are measured from the direction
     * towards the model centre for packages of the external field and away from it for those of the central source.
     * Not combined with ffi (DIES_EINVAL).                                                                          */
    double   g_E;         /* re-emission directions from a Henyey-Greenstein function HG(g_E) instead of isotropic,
                             weight (1/2) / p_HG; 0 = isotropic (the plain method), |g_E| < 1                      */
    double   g_S;         /* scattering directions from HG(g_S) about that radial direction, weight = dust HG density
                             at the true scattering angle / p_HG(g_S); only if use_g_S != 0, |g_S| < 1             */
    int32_t  use_g_S;     /* g_S = 0 is a weighting too (isotropic sampling, L207), hence the switch               */
    int32_t  reemit_in_cell; /* L253 (R20): re-emit from a random position of the cell volume (radius uniform in volume
                             between the shell boundaries) instead of the absorption site; 0 = the IRE method proper */
} dies_run_opts;

/* Bytes of device workspace a model (n_models = 1) or a batch needs. */
int dies_workspace_bytes(int n_shells, int n_freq, int n_T, int n_models, size_t* bytes);

/* The model of PAPER.md L49 / L67-71 / L87: shells, dust, and the emission table behind the two lookup
 * tables (absorbed energy -> temperature; (T_old, T_new, u) -> re-emitted frequency).
 *   r_bounds  n_shells+1 strictly ascending, r_bounds[0] >= 0; r_bounds[0] > 0 is an empty cavity (R10)
 *   rho       n_shells, >= 0, dust mass per volume
 *   freq      n_freq ascending; labels only (frequencies are discrete bins, R3)
 *   kappa_abs, kappa_sca  n_freq, >= 0, per dust mass; g_hg n_freq, |g| < 1 (Henyey-Greenstein, L167)
 *   T_grid    n_T strictly ascending
 *   emis      n_T x n_freq row-major, >= 0, power emitted per dust mass in bin k at T_t; rows must not
 *             decrease with t in any bin and their sums must strictly increase
 *   workspace_dev  DEVICE pointer, 256-byte aligned, workspace_bytes >= dies_workspace_bytes(...)
 * Tables are built on the device during the call (which synchronises before returning). */
int dies_create_model(int n_shells, const double* r_bounds, const double* rho,
                      int n_freq, const double* freq,
                      const double* kappa_abs, const double* kappa_sca, const double* g_hg,
                      int n_T, const double* T_grid, const double* emis,
                      void* workspace_dev, size_t workspace_bytes, dies_model** out);

/* Config 5: n_models spheres of n_shells shells each sharing dust and emission tables.
 *   r_bounds n_models x (n_shells+1), rho n_models x n_shells, row-major. */
int dies_create_batch(int n_models, int n_shells, const double* r_bounds, const double* rho,
                      int n_freq, const double* freq,
                      const double* kappa_abs, const double* kappa_sca, const double* g_hg,
                      int n_T, const double* T_grid, const double* emis,
                      void* workspace_dev, size_t workspace_bytes, dies_model** out);

/* Sources (L49-55).  ext_bin_intensity: n_freq bin-integrated mean intensities of the isotropic external
 * field (luminosity 4 pi R^2 * pi * sum_k J_k), or NULL.  L_point > 0 with point_bin_weights (n_freq
 * relative spectrum) is the central point source, else pass 0 / NULL.  Each active source gets n_total
 * packages of equal energy (L51, R2): ids [0, n_total) external, then the point source. */
int dies_set_sources(dies_model*, const double* ext_bin_intensity, double L_point, const double* point_bin_weights);
/* Batch form: ext n_models x n_freq or NULL; L_point n_models or NULL; point weights n_models x n_freq or NULL. */
int dies_set_sources_batch(dies_model*, const double* ext_bin_intensity, const double* L_point,
                           const double* point_bin_weights);

/* Follow n_packages packages per active source (per model) on `cuda_stream` (a cudaStream_t; NULL = default
 * stream).  Asynchronous: returns after the launches.  opts == NULL means {0.5, 0, IRE, 0, 24, n_packages, 1, 0, 1, 0, 0, 0, 0}. */
int dies_run(dies_model*, uint64_t n_packages, uint64_t seed, const dies_run_opts* opts, void* cuda_stream);
/* Sharding of fixed-temperature runs over processes / GPUs: the next dies_run that does not
 * accumulate follows the package ids first_id .. first_id + n_packages - 1 (per source) of a run of opts->n_total
 * packages instead of starting at 0.  Integer tallies of disjoint id ranges add up to the tallies of the whole run. */
int dies_seek(dies_model*, uint64_t first_id);
int dies_run_batch(dies_model*, uint64_t n_packages_per_model, uint64_t seed, const dies_run_opts* opts,
                   void* cuda_stream);
/* Sharding of a batch over processes / GPUs (config 5): the models of this handle are the models
 * first_model .. first_model + n_models - 1 of a larger batch.  The model index is word 3 of the Philox counter (RNG
 * contract), so a shard created from a slice of the batch's arrays follows exactly the packages the whole batch would
 * follow for these models: the results of the shards, concatenated, are those of the one-GPU batch (bit for bit in
 * fixed-temperature mode).  No exchange between shards is needed.  Default 0. */
int dies_set_model_offset(dies_model*, uint32_t first_model);

/* Dust temperatures from the absorbed-energy tallies (L87 lookup table; log-log interpolation, R6):
 * T[n_models x n_shells]; n must equal that size.  Synchronises the stream of the last run. */
int dies_get_temperature(dies_model*, double* T, int n);
/* Escaping luminosity per frequency bin, n_models x n_freq (L87 last sentence; un-interacted FFI share included). */
int dies_get_escape_spectrum(dies_model*, double* L_esc, int n);

/* Parity-test support ---------------------------------------------------------------------------------- */
/* Fixed-temperature tracking mode: shell i re-emits with the table row of T[i] (#{t: T_grid[t] <= T[i]}). */
int dies_set_fixed_temperature(dies_model*, const double* T, int n);
/* Raw 64-bit tallies (n_models x n_shells) and the energy per raw unit of each model (n_models). */
int dies_get_absorbed(dies_model*, int64_t* raw, double* energy_per_raw_unit, int n);
/* DIES_N_COUNTERS counters summed over models (see enum); n must be DIES_N_COUNTERS. */
int dies_get_counters(dies_model*, uint64_t* c, int n);
/* Replay packages first_id .. first_id+count-1 of model model_index against the current tallies (read only)
 * and list their events: events[p][e] = (type, shell, freq_bin, crossings so far), at most max_events each;
 * n_events[p] is the true number.  Runs the same device code as dies_run. */
int dies_trace_packages(dies_model*, int model_index, uint64_t first_id, int count, uint64_t n_total, uint64_t seed,
                        const dies_run_opts* opts, int32_t* events, int max_events, int32_t* n_events);
int dies_trace_package(dies_model*, uint64_t package_id, uint64_t n_total, uint64_t seed, const dies_run_opts* opts,
                       int32_t* events, int max_events, int32_t* n_events);
/* dies_trace_packages for callers that must not allocate device memory.
 *
 * Who needs it: a process in which a framework's caching allocator (PyTorch's, for one) has already taken nearly all of
 * the GPU, so that a raw cudaMalloc from this library fails although the framework still has room to hand out; and a
 * service that replays packages while other streams run trackers, where cudaMalloc / cudaFree would stall the whole
 * device (cudaFree waits for all work on it).  dies_trace_packages does both per call; this entry point does neither.
 *
 * How: the event lists, the event counts and the package counter live in one fixed array inside the library image
 * (1 MiB + 16 KiB + 256 B).  Every GPU on which libdies.so is loaded holds that array until the process exits, used or
 * not.  Inputs (the handle and its caller-owned workspace) and outputs (the host buffers events / n_events) are passed
 * exactly as for dies_trace_packages, and the results are the same, with one difference: entries of events[p] past
 * n_events[p] are zero here and undefined there.
 *
 * Limits: count <= DIES_TRACE_STATIC_MAX_PACKAGES and count * max_events <= DIES_TRACE_STATIC_MAX_EVENTS, else
 * DIES_EINVAL with a message that names the limit (nothing is launched); split a longer id range over several calls.
 *
 * Set-up: the first call on each GPU looks up the array's device address (once per device, under a lock, with the
 * calling thread's current device, which must be the one the handle's workspace lives on).  Make that first call
 * before any stream capture begins.
 *
 * Sharing: all calls, of all handles and threads, use the same array on a GPU.  It keeps the contents of the last
 * call; this entry point clears the part it uses before launching.  Two calls whose device work overlaps (two threads,
 * two handles) race on it and corrupt each other's lists: serialise them.  The call synchronises the device before it
 * returns, so calls made one after the other from one thread never overlap.
 *
 * No cudaMalloc, cudaFree or allocating library routine is called. */
#define DIES_TRACE_STATIC_MAX_PACKAGES 4096
#define DIES_TRACE_STATIC_MAX_EVENTS   65536
int dies_trace_packages_static(dies_model*, int model_index, uint64_t first_id, int count, uint64_t n_total,
                               uint64_t seed, const dies_run_opts* opts, int32_t* events, int max_events,
                               int32_t* n_events);
/* The device Philox and uniform of the RNG contract: out[4*j..] = words of block `block` of package first_id+j. */
int dies_test_philox(uint64_t seed, uint64_t first_id, uint32_t block, uint32_t model_index, int n,
                     uint32_t* words, float* uniforms);
/* Device tables as built (for table parity): eps n_T (double), F n_T x n_freq (float). Either may be NULL. */
int dies_get_tables(dies_model*, double* eps, float* F);

/* Measurement support (the atomic side of the roofline): throughput of the absorption
 * step's memory operation alone -- every lane of every resident warp draws one of n_addr (<= 65535) 64-bit tallies,
 * uniformly (weights == NULL) or with the probabilities weights[n_addr] (host, >= 0: the workload's per-shell
 * absorption histogram); equal draws of a warp are merged when aggregate != 0 (as the tracker does when all quanta
 * are equal), and one RETURNING 64-bit atomicAdd per distinct tally per warp is issued and consumed; iters rounds
 * per lane.  lane_ops_per_s = absorptions/s this pattern sustains, atomics_per_s = atomic instructions/s issued. */
int dies_bench_atomics(int n_addr, const double* weights, int aggregate, int iters, double* lane_ops_per_s,
                       double* atomics_per_s);

/* Launch tuning of the trackers (process-wide; the defaults are the measured optimum on config 2).
 * It is not part of the method: integer tallies of fixed-temperature runs do not depend on it at all, full-IRE results
 * only through the order of absorptions (within noise).  Fields that are 0 keep their current value;
 * dies_set_tuning(NULL) restores the defaults; out-of-range values give DIES_EINVAL and change nothing. */
typedef struct {
    int32_t slots_uniform;  /* dies_fly: pool slots per lane when all packages carry one quantum, 1..8 (default 5)   */
    int32_t slots;          /* dies_fly: the same with per-package quanta (k_bg, FFI, two sources), 1..8 (4)         */
    int32_t visit;          /* dies_fly: crossing blocks between two event phases, 1..64 (default: chosen per model,
                               2..8, so that a crossing phase lasts about two mean flights as counted by the model's
                               last read-out; 8 before the first read-out).  Because the automatic value follows the
                               read-outs, the ORDER in which a full-IRE run makes its absorptions -- and so its result,
                               within the Monte Carlo noise -- depends on whether a getter was called between two runs
                               of the handle.  Set visit explicitly for results that repeat bit for bit whatever the
                               getter calls; fixed-temperature tallies never depend on it                            */
    int32_t min_ready;      /* dies_fly: partial event batches only while fewer packages are ready, 1..256 (32)      */
    int32_t chunk;          /* package ids a warp takes from the global counter at a time, 32..4096 (128)            */
    int32_t pkg_per_block;  /* grid sizing of small runs: packages per block, 32..2^20 (256)                         */
    int32_t w_pool;         /* dies_track (weighted runs): pool slots per warp, 32..248 (96)                         */
    int32_t w_thr_hi;       /* dies_track: swap stopped lanes for ready packages when fewer fly, 1..32 (20)          */
    int32_t w_thr_lo;       /* dies_track: with no ready package left, leave when fewer fly, 1..32 (16)              */
    int32_t w_min_ready;    /* dies_track: mixed event batches only while fewer packages are ready, 1..248 (32)      */
    int32_t atom_stride;    /* dies_bench_atomics: 64-bit words between two tallies, 1..64 (32)                      */
} dies_tuning;
int dies_set_tuning(const dies_tuning* t);
int dies_get_tuning(dies_tuning* t);

int dies_destroy(dies_model*);
const char* dies_last_error(void);
/* "sm_100a" build tag, number of SMs and resident blocks per SM of the tracker (for the bench log). */
int dies_device_info(int* n_sms, int* blocks_per_sm, int* threads_per_block);

#ifdef __cplusplus
}
#endif
#endif /* DIES_H */
