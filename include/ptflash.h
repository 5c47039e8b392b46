/* ptflash.h -- C ABI of libptflash: batched isothermal two-phase (vapour-liquid) flash of N independent
 * mixtures at given (P, T, z) under the Soave-Redlich-Kwong equation of state, on one NVIDIA B200 (sm_100a).
 *
 * The operation is the one PTFlash (arXiv 2205.03090) defines in section 2.1: for every
 * mixture decide "single phase" or "two phases"; in the latter case return the vapour mole fraction
 * beta (= theta_V), the liquid composition x and the vapour composition y satisfying the mass balance
 * (1a), (1b) and the iso-fugacity condition (2).  The method is the paper's (section 2.2, Fig. 2,
 * PAPER.md:51-111; App. A-C): Wilson K-values (eq. 6) -> 3 successive-substitution
 * probes -> Michelsen's two-sided tangent-plane stability test (eq. 3-5, SS then trust-region Newton,
 * App. B.1) -> Rachford-Rice (eq. 7, App. C) + successive substitution + trust-region Newton on the
 * Gibbs energy (eq. 8, App. B.2).  Every iteration rebuilds the SRK mixture parameters (A.2), solves the
 * cubic (A.3) choosing the root of minimum Gibbs energy, and evaluates ln-fugacity coefficients (A.6).
 * Every step runs in hand-written fp64 CUDA kernels; there is no CPU fallback.
 *
 * Layout: all per-mixture arrays are structure-of-arrays, fp64, component-major: element (i, n) of z, x,
 * y, lnK lives at [i * N + n] (i = component 0..nc-1, n = mixture 0..N-1).  P, T, beta, phase, ... are [N].
 * Units: T and Tc in K; P in the same unit as Pc (bar in the benchmark configs); the gas constant cancels.
 *
 * Threading: a handle may be used by one thread at a time; calls on one handle are serialised on the
 * stream given.  Use one handle per stream for concurrency.
 */
#ifndef PTFLASH_H
#define PTFLASH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ptflash_handle_s* ptflash_handle_t;

#define PTFLASH_OK 0
#define PTFLASH_EINVAL (-1) /* null handle / null required pointer / N < 0 or > PTFLASH_MAX_N / unknown option or value out of range */
#define PTFLASH_ECUDA (-2)  /* CUDA allocation, copy or launch failure; text in ptflash_last_error() */

#define PTFLASH_MAX_NC 16
#define PTFLASH_MAX_N 1073741823LL /* 2^30 - 1 mixtures per call (work queues hold 32-bit ids); larger N -> PTFLASH_EINVAL */

/* out_phase values */
#define PTFLASH_PHASE_INVALID (-1) /* non-finite input, P <= 0, T <= 0, z_i < 0 or |sum z - 1| > 1e-9: beta, x, y = NaN */
#define PTFLASH_PHASE_SINGLE 1
#define PTFLASH_PHASE_TWO 2

/* out_status bits (per mixture; problems are data, never call failures -- cf. Alg. 1 PAPER.md:550-552,
 * which returns the indices of unconverged samples) */
#define PTFLASH_ST_STAB_CAP 1      /* a stability trial hit its iteration cap */
#define PTFLASH_ST_SPLIT_CAP 2     /* the phase split hit its iteration cap */
#define PTFLASH_ST_BAND 4          /* 0 < |tpd_min| < band (1e-9): label decided inside the near-zero TPD band */
#define PTFLASH_ST_SPLIT_FAILED 8  /* "unstable" verdict but the split ended trivial or with beta outside (0,1): reported as single phase */
#define PTFLASH_ST_LNK0_REJECTED 32 /* caller-supplied lnK0 non-finite or |lnK0| > 700: Wilson used instead */
#define PTFLASH_ST_WARM_RESTART 64  /* PTFLASH_FLAG_SKIP_STABILITY split did not reach two phases: hint dropped, mixture re-flashed from Wilson with the full stability analysis */

/* flags[n] bits for ptflash_flash_ex (interface effect of the paper's classifier/initializer, section 4.3
 * caller-supplied K estimates and a "known unstable" verdict) */
#define PTFLASH_FLAG_SKIP_STABILITY 1 /* go straight to the phase split from lnK0 */
#define PTFLASH_FLAG_USE_LNK0 2       /* use lnK0 instead of Wilson for the probe and the stability starts */

/* ptflash_create: bind a component system to the current CUDA device.
 *   nc      number of components, 2..PTFLASH_MAX_NC
 *   Tc, Pc, omega   HOST arrays [nc]: critical temperature (K), critical pressure, acentric factor (Table 1)
 *   kij     HOST array [nc*nc] row-major, symmetric, zero diagonal (A.2b PAPER.md:415); NULL = all zero
 * Everything is copied; the caller keeps its arrays.  Returns NULL on failure (bad nc, null pointer,
 * non-finite or non-positive Tc/Pc, asymmetric kij, CUDA error); reason in ptflash_last_error(). */
ptflash_handle_t ptflash_create(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij);

/* ptflash_flash: flash N mixtures.  All pointers are DEVICE pointers on the handle's device.
 *   z [nc][N], P [N], T [N]          inputs (section 2.1); z is normalised once internally (z / sum z)
 *   out_beta [N]                      two-phase: vapour fraction in (0,1); single phase: 1 if Z_feed > 1/3 else 0
 *   out_x, out_y [nc][N]              two-phase: liquid / vapour mole fractions (each sums to 1); single phase: both = z
 *   out_phase [N]                     number of phases: 1, 2, or -1 (invalid input)
 *   out_iters [N] (may be NULL)       number of K-value updates performed (probe + split SS + split Newton)
 *   stream                            cudaStream_t (NULL = legacy default stream)
 * Asynchronous: enqueues work on `stream` and returns; outputs are valid once the stream reaches that point.
 * The caller owns every buffer; inputs and outputs must not alias.  The handle owns a workspace that
 * grows on first use (a growth synchronises the stream) and a second, internal stream: after the stability stages the two
 * parts of the phase split run concurrently, forked from and joined back into `stream` by events, so the ordering
 * guarantees above hold for `stream` alone.  One call in flight per handle (use one handle per stream for concurrency).
 * The call makes the handle's device current while it runs and restores the caller's.  N == 0 is a no-op.
 * Returns PTFLASH_OK / EINVAL / ECUDA. */
int ptflash_flash(ptflash_handle_t h, int64_t N, const double* z, const double* P, const double* T,
                  double* out_beta, double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters,
                  void* stream);

/* Extended call: same nine arrays plus optional ones (NULL = absent). */
typedef struct ptflash_io {
  int64_t N;
  const double* z;           /* [nc][N] */
  const double* P;           /* [N] */
  const double* T;           /* [N] */
  const double* lnK0;        /* optional in  [nc][N]: initial ln K (warm start, BASELINE config 5) */
  const uint8_t* flags;      /* optional in  [N]: PTFLASH_FLAG_* (ignored where lnK0 is NULL) */
  double* out_beta;          /* [N] */
  double* out_x;             /* [nc][N] */
  double* out_y;             /* [nc][N] */
  int32_t* out_phase;        /* [N] */
  int32_t* out_iters;        /* optional out [N] */
  double* out_tpd_min;       /* optional out [N]: minimum reduced TPD found (eq. 3; probe value for probe-proved mixtures; NaN when stability was skipped) */
  double* out_lnK;           /* optional out [nc][N]: converged ln K (0 for single phase) */
  int32_t* out_status;       /* optional out [N]: PTFLASH_ST_* bits */
  int32_t* out_stab_iters;   /* optional out [N]: stability iterations (SS + Newton, both starts) */
  double* out_dbeta_dK;      /* optional out [nc][N]: d beta / d K_i at the reported solution (K = y / x), by the implicit-function
                                formula of eq. 13: -[d f_RR / d beta]^-1 d f_RR / d K_i; 0 for a z_i = 0
                                component; NaN unless out_phase == 2 */
} ptflash_io_t;
int ptflash_flash_ex(ptflash_handle_t h, const ptflash_io_t* io, void* stream);

/* End-to-end variant with HOST buffers (same meaning and layout as ptflash_flash; pinned memory needed for the copies to be
 * asynchronous): the batch is cut into PTFLASH_OPT_HOST_CHUNKS chunks of consecutive mixtures, each copied host->device,
 * flashed and copied back device->host on an internal stream of its own (strided slices of the SoA arrays), so that the
 * transfers of one chunk overlap the kernels of the others; all of it starts after the work already queued on `stream`,
 * and the call returns after everything has completed (it synchronises).  Staging buffers, the chunks' workspaces and
 * streams belong to the handle; ptflash_get_stats then reports the sums over the chunks. */
int ptflash_flash_host(ptflash_handle_t h, int64_t N, const double* z, const double* P, const double* T,
                       double* out_beta, double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters,
                       void* stream);

/* Pipelined host-buffer variant for a stream of batches (what a simulator or a data-generation loop submits): the call
 * enqueues the H2D copies of the inputs, the flash kernels and the D2H copies of the results of ONE batch on an internal
 * stream and returns without waiting.  Up to PTFLASH_HOST_DEPTH batches are in flight, each on a stream and a workspace of
 * its own, so the copies of one batch run under the kernels of its neighbours (PCIe is full duplex); a call first waits for
 * the batch submitted PTFLASH_HOST_DEPTH calls earlier.  The host buffers of a batch (pinned memory needed) must stay
 * valid, and its outputs are defined, only after ptflash_host_wait -- or after PTFLASH_HOST_DEPTH later submissions.  Use
 * distinct output buffers for batches that can be in flight together.  ptflash_get_stats reports the most recent batch.
 * Returns PTFLASH_OK / EINVAL / ECUDA. */
#define PTFLASH_HOST_DEPTH 3
int ptflash_flash_host_async(ptflash_handle_t h, int64_t N, const double* z, const double* P, const double* T,
                             double* out_beta, double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters);
/* Blocks until every batch submitted with ptflash_flash_host_async has completed (its results are in the host buffers). */
int ptflash_host_wait(ptflash_handle_t h);

/* Synchronises the handle's last stream, frees constants and workspace.  NULL is a no-op. */
int ptflash_destroy(ptflash_handle_t h);

/* ptflash_flash_static: the same flash as ptflash_flash, for callers that must not allocate.
 *
 * Why it exists.  ptflash_flash keeps its work queues and the per-mixture state handed from stage kernel to stage kernel in
 * a workspace (~0.66 KB per mixture at nc = 10) that the handle cudaMallocs on first use and replaces -- stream
 * synchronise, cudaFree, cudaMalloc -- whenever a larger batch arrives; ptflash_create itself allocates pinned host memory.
 * Some users of a flash library cannot accept that inside the call:
 *   - a reservoir or process simulator that has already handed nearly all device memory to its own arena (or runs inside a
 *     framework whose caching allocator has): a raw cudaMalloc from a library can then fail although the pool has room;
 *   - a time-step loop with a latency budget: cudaMalloc and cudaFree serialise against the whole device, so a workspace
 *     growth stalls every other stream of the process at an unpredictable step;
 *   - a process held to a fixed memory budget (several jobs sharing one GPU), where a library must state its footprint up
 *     front and never grow it.
 * This entry point needs no handle and calls no cudaMalloc, cudaMallocHost, cudaFree, stream or event creation, nor any
 * library routine that allocates.  Its workspace is an array of PTFLASH_STATIC_SCRATCH_BYTES (32 MiB) that is part of the
 * library's device code: every GPU on which the library's code gets loaded holds those 32 MiB until the process exits,
 * whether or not this function is ever called.  That fixed size is the price and the limit: N <= PTFLASH_STATIC_MAX_N.
 *
 *   nc, Tc, Pc, omega, kij   the component system, HOST arrays exactly as for ptflash_create (kij may be NULL); it is
 *                            validated and folded into constants on every call (a few hundred flops on the host)
 *   N                        0..PTFLASH_STATIC_MAX_N mixtures; N == 0 is a no-op; a larger N is refused with PTFLASH_EINVAL
 *                            and a message naming the limit (nothing is launched) -- cut the batch, or use ptflash_flash
 *   z, P, T, out_*           DEVICE pointers on the CURRENT device, meaning and layout as for ptflash_flash; the caller owns
 *                            them; out_iters may be NULL; inputs and outputs must not alias
 *   stream                   cudaStream_t of the current device (NULL = legacy default stream)
 * Results are those of ptflash_flash on a fresh handle with default options: the same stage kernels run in the same order,
 * all on `stream` (there is no internal second or third stream here, so on big batches it is somewhat slower; at these
 * sizes a call is launch-latency bound anyway).  Asynchronous: returns once the kernels are queued.  No statistics, no
 * options, no warm start: use a handle for those.
 *
 * Set-up.  The first call on a device looks up the device address of the workspace (cudaGetSymbolAddress) and, the first
 * time it meets a given (nc, all-zero-kij or not) there, raises the shared-memory limit of the two Newton kernels and asks
 * the occupancy calculator how many CTAs fit.  Both may make the CUDA runtime load the library's device code.  Make one
 * call per device and per component system during start-up, before the region that must not allocate and before any stream
 * capture begins.
 *
 * Sharing.  All calls on one device use the same array, whatever the thread or stream, and the array keeps whatever the
 * previous call left in it.  The function clears the part that must start at zero (stage counters and queue lengths) on
 * `stream` at the head of every call; nothing else is read before this call has written it.  Two calls that can run on the GPU
 * at the same time (different streams without an ordering between them, or two host threads) corrupt each other's queues:
 * order them yourself, e.g. keep to one stream per device.  Calls on different devices are independent.
 * Returns PTFLASH_OK / PTFLASH_EINVAL (bad system, N out of range, null pointer) / PTFLASH_ECUDA. */
#define PTFLASH_STATIC_MAX_N 32768
#define PTFLASH_STATIC_SCRATCH_BYTES 33554432 /* 32 MiB: holds the workspace of 32768 mixtures of 16 components (29.6 MiB) */
int ptflash_flash_static(int nc, const double* Tc, const double* Pc, const double* omega, const double* kij,
                         int64_t N, const double* z, const double* P, const double* T,
                         double* out_beta, double* out_x, double* out_y, int32_t* out_phase, int32_t* out_iters,
                         void* stream);

/* Options (tolerances and caps); defaults in brackets follow DESIGN.md section 3 / PAPER.md:79,90,97,105,558 */
enum {
  PTFLASH_OPT_TOL_SS = 0,          /* SS residual target, stability and split [1e-10] */
  PTFLASH_OPT_TOL_NEWTON_G = 1,    /* Newton gradient target [1e-12] */
  PTFLASH_OPT_TOL_NEWTON_STEP = 2, /* phase-split Newton: a full (eta = 0) step with max_i |s_i| / min(n^V_i, n^L_i) below this is
                                      applied and the iteration stops; the error left behind is second order [1e-7, relative:
                                      next to a phase boundary the mole numbers of the incipient phase are themselves ~1e-9,
                                      so an absolute threshold would stop on an unconverged point] */
  PTFLASH_OPT_PROBE_MARGIN = 3,    /* probe: "negative" means < -margin [1e-8] */
  PTFLASH_OPT_TRIVIAL_TOL = 4,     /* trivial stability solution: max|lnW - lnz| < tol [1e-6] */
  PTFLASH_OPT_BAND = 5,            /* near-zero TPD band [1e-9] */
  PTFLASH_OPT_PROBE_ITERS = 6,     /* [3] */
  PTFLASH_OPT_STAB_SS_ITERS = 7,   /* [9] */
  PTFLASH_OPT_STAB_TR_ITERS = 8,   /* [60] */
  PTFLASH_OPT_SPLIT_SS_ITERS = 9,  /* [9]: SS iterations before switching to Newton */
  PTFLASH_OPT_SPLIT_TR_ITERS = 10, /* [60] */
  PTFLASH_OPT_USE_NEWTON = 11,     /* [1]; 0 = pure successive substitution */
  PTFLASH_OPT_SS_CAP = 12,         /* [100000]: SS cap when Newton is off or theta stays outside (0,1) */
  PTFLASH_OPT_ENGINE = 13,         /* [1] 1 = staged persistent kernels with work queues; 0 = single run-to-completion kernel */
  PTFLASH_OPT_STAGE_PROFILE = 14,  /* [0] 1 = record a CUDA event between the stage kernels (engine 1), see ptflash_get_stage_ms */
  PTFLASH_OPT_TOL_NEWTON_STEP_STAB = 15, /* the same for the stability Newton, whose result enters only through tm (itself
                                            second order in the error of W) and the K seed [1e-6] */
  PTFLASH_OPT_HINT_SS_CAP = 16,    /* [12] a PTFLASH_FLAG_SKIP_STABILITY split whose successive substitution is still outside
                                      0 < theta < 1 after this many iterations is dropped and the mixture re-flashed from
                                      Wilson (PTFLASH_ST_WARM_RESTART; reading C21) */
  PTFLASH_OPT_SPLIT_TRIVIAL_TOL = 17, /* [1e-5] the phase split has collapsed into the trivial solution x = y when max_i |ln K_i| < tol
                                      (-> PTFLASH_ST_SPLIT_FAILED, or a warm restart); reading C22 */
  PTFLASH_OPT_STABILITY_ONLY = 18, /* [0] 1 = stop after the label: probe + stability analysis, no phase split -- the mode the paper
                                      uses to label 10^6 samples for its classifier.  out_phase = 1 stable / 2
                                      unstable; x = y = z; out_beta = the single-phase convention for a stable feed, NaN for an
                                      unstable one; out_lnK = the K that would seed the split; out_tpd_min as usual;
                                      a PTFLASH_FLAG_SKIP_STABILITY mixture is reported unstable without any work */
  PTFLASH_OPT_HOST_CHUNKS = 19,    /* [8] ptflash_flash_host cuts the batch into at most this many chunks (1..8, none below 32768
                                      mixtures), each on a stream of its own, so that the PCIe copies of one chunk overlap the
                                      kernels of the others */
  PTFLASH_OPT_HINT_ETA_SEARCH = 20, /* [0] 0 = a split entered through PTFLASH_FLAG_SKIP_STABILITY takes the truncated
                                      modified-Cholesky step of every other split (one factorisation per trust-region iteration);
                                      1 = it takes the restricted step of B.4a by the eta search, the oracle's path, so that the
                                      SAME hints fail and PTFLASH_ST_WARM_RESTART agrees with the oracle mixture by mixture (with
                                      0 the answers are the same, but ~2 hints per 1000 mixtures next to the phase boundary fail
                                      or survive differently: which hints fail is a property of the iteration path); costs
                                      1.4x on the warm-start workload */
  PTFLASH_OPT_HINT_TR_CAP = 21,    /* [15] a PTFLASH_FLAG_SKIP_STABILITY split that has not converged after this many trust-region
                                      iterations is dropped and the mixture re-flashed from Wilson (PTFLASH_ST_WARM_RESTART;
                                      DESIGN.md reading C21): converging hinted splits of the warm-start workload need <= 11, failing
                                      ones wander until the cap */
  PTFLASH_OPT_EARLY_SPLIT_SS = 22, /* [0] 1 = the successive-substitution stage of the phase split of the mixtures the probe found
                                      unstable starts right after the probe, next to the stability analysis of the others, instead
                                      of after it.  Scheduling only, same results.  It pays on workloads with "crawlers" -- splits
                                      still outside 0 < theta < 1 after split_ss_iters iterations, which continue the substitution
                                      (reading C13) for hundreds of iterations on a stream of their own: started early,
                                      that serial chain ends under the rest of the call (paper's 9-component workload: 4.8 -> 4.0 ms
                                      per 1e6); without crawlers it costs ~5 % (the early stage no longer fills the machine next to
                                      the latency-bound tail of the stability-found splits) */
  PTFLASH_OPT_HOST_ROW_COPIES = 23, /* [0] 1 = ptflash_flash_host moves the strided slices of z, x, y with one plain copy per component row
                                      instead of one 2D copy per array.  The call does that by itself when N * 8 bytes exceeds the
                                      pitch a 2D copy accepts (2^31 - 1 bytes, i.e. N >= 2^28 mixtures); the option exists to
                                      exercise that path at ordinary sizes.  Same results */
  PTFLASH_NUM_OPTS = 24
};
int ptflash_set_option(ptflash_handle_t h, int key, double value);
int ptflash_get_option(ptflash_handle_t h, int key, double* value);

/* Counters of the last completed call, shaped like the paper's profiler (Table 4).
 * Synchronises the handle's last stream. */
typedef struct ptflash_stats {
  int64_t n_total, n_invalid;
  int64_t n_probe_case1, n_probe_case2, n_probe_case3; /* section 2.2.3 */
  int64_t n_stability;      /* mixtures sent to the stability analysis */
  int64_t n_stab_newton;    /* stability trials that needed the trust-region stage */
  int64_t n_split;          /* mixtures sent to the phase split */
  int64_t n_split_newton;   /* phase splits that needed the trust-region stage */
  int64_t n_two_phase;
  int64_t kernel_launches;  /* kernels launched by the last call */
  /* The remaining columns of Table 4; index [0] = vapour-like start, [1] = liquid-like start.
   * "# of samples": ss stages n_stability (each start) and n_split, tr stages n_stab_tr[] and n_split_newton.
   * "Convergence": a stability trial / phase split that does not go on to the trust-region stage ended within the SS
   * cap (n_stability - n_stab_tr[k], n_split - n_split_newton); a trust-region stage converged unless it hit its cap
   * (n_stab_capped[k], n_split_capped); the probe's figure is n_probe_case3 / n_total (footnote 1 of Table 4).
   * "Max number of iterations": the max_* fields. */
  int64_t n_stab_tr[2];      /* stability trials that went on to the trust-region stage, per start (sum = n_stab_newton) */
  int64_t n_stab_capped[2];  /* stability trials that hit an iteration cap, per start */
  int64_t n_split_capped;    /* phase splits that hit an iteration cap */
  int64_t n_warm_restarts;   /* PTFLASH_FLAG_SKIP_STABILITY hints that failed and were re-flashed cold (PTFLASH_ST_WARM_RESTART) */
  int32_t max_probe_iters, max_stab_ss_iters[2], max_stab_tr_iters[2], max_split_ss_iters, max_split_tr_iters;
  int32_t reserved_;
} ptflash_stats_t;
/* Returns PTFLASH_ECUDA (reason in ptflash_last_error) also if the last call left an internal work queue longer than its
 * array.  By construction that cannot happen (every queue holds at most N, or 2 N, ids; the argument is written out above
 * carve_workspace in csrc/ptflash_staged.cuh), and the appends are not clamped; the last kernel of every call compares the
 * final queue lengths with their capacities, so a violation is seen AFTER the fact -- memory behind the queue has then been
 * overwritten and the call's results are not to be trusted -- and only here, since the flash calls return before the
 * kernels have run. */
int ptflash_get_stats(ptflash_handle_t h, ptflash_stats_t* out);

/* Batched Rachford-Rice solve with its derivative -- what the paper's initializer training evaluates for every sample
 * (PAPER.md:279-286): theta from (K, z) by eq. 7 (solver of App. C: Newton on h_RR inside a
 * shrinking sign bracket on (alpha_l, alpha_r), negative flash allowed), x_i = z_i / (1 + (K_i - 1) theta), y_i = K_i x_i
 * (normalised), and d theta / d K_i = -[d f_RR / d theta]^-1 d f_RR / d K_i (eq. 13) at the solution.
 *   lnK, z [nc][N]      DEVICE inputs (ln K so that the caller's network output is used as is; z is normalised internally)
 *   out_theta [N]       DEVICE; NaN where there is no window (all K_i >= 1 or all <= 1 over the z_i > 0 components) or the
 *                       input is invalid (non-finite, z_i < 0, |ln K_i| > 700 -- cf. the overflow reported at PAPER.md:363)
 *   out_x, out_y, out_dtheta_dK [nc][N]   DEVICE, each may be NULL; NaN where out_theta is NaN; 0 derivative for z_i = 0
 * Asynchronous on `stream`; the caller owns all buffers.  Returns PTFLASH_OK / EINVAL / ECUDA. */
int ptflash_rachford_rice(ptflash_handle_t h, int64_t N, const double* lnK, const double* z, double* out_theta,
                          double* out_x, double* out_y, double* out_dtheta_dK, void* stream);

/* Stage times of the last call made with PTFLASH_OPT_STAGE_PROFILE = 1 (engine 1), measured with CUDA events recorded
 * on the call's stream between the stage kernels -- the per-stage "time" row of the paper's profiler (Table 4
 * PAPER.md:332-345).  Order: init, probe, stab_ss, stab_newton, stab_decide, split_ss, split_newton; a call with
 * PTFLASH_FLAG_* flags inserts three stages after init -- split_ss and split_newton of the hinted mixtures, and the re-queueing
 * of the failed hints -- so that the hints that fail take the cold path in the same pass.  Writes up to `cap` values (milliseconds) to HOST array `ms`,
 * returns the number written (0 if profiling was off), or PTFLASH_EINVAL / PTFLASH_ECUDA.  Synchronises the stream. */
#define PTFLASH_NUM_STAGES 7
int ptflash_get_stage_ms(ptflash_handle_t h, float* ms, int cap);

/* FP64 roofline probe: runs an unrolled independent-DFMA kernel on every SM for `iters` iterations and returns
 * the achieved FP64 FLOP/s (used by bench.py as the measured denominator of the ALU roofline). */
int ptflash_fp64_peak(int iters, double* flops_per_s, double* elapsed_ms, void* stream);

/* Diagnostic: evaluates ONE of the library's own fp64 math routines (csrc/ptflash_math.cuh: the branch-free exp / log /
 * reciprocal sequences every kernel uses instead of the CUDA math library) element-wise, y[i] = fn(x[i]), on DEVICE arrays
 * x, y [n], asynchronously on `stream`.  It exists so that the accuracy claims of those routines (<= 2 ulp on their stated
 * ranges, the clamps at their edges) can be tested directly against libm instead of only through the flash results.
 *   fn  0 exp_fast   (x <= 709; clamped below at -708)      1 exp_tab  (x <= 709; clamped below at -700)
 *       2 log_fast   (normal x > 0)                           3 log1p_fast (0 <= x < 1)
 *       4 rcp_fast   (normal x, 1/x normal)                   5 rsqrt_fast (normal x > 0)
 *       6 sqrt_fast  (x >= 0)                                 7 div_fast(1, x)          8 rcp_nr1 (~2^-40 relative)
 * Returns PTFLASH_OK / EINVAL / ECUDA. */
#define PTFLASH_NUM_MATH_FN 9
int ptflash_math_probe(int fn, int64_t n, const double* x, double* y, void* stream);

/* Text of the last error on the calling thread ("" if none). */
const char* ptflash_last_error(void);

/* Library version string, e.g. "ptflash-b200 0.1 (sm_100a)". */
const char* ptflash_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PTFLASH_H */
