/* nsgw.h -- C-ABI of libnsgw.so: the batched acceptance-walk nested-sampling hot path of arXiv 2509.04336
 * (Prathaban et al.) as hand-written sm_100a CUDA.
 *
 * Citations: "P:NNN" = line NNN of the paper text; "R:Lnn" = reading Lnn in DESIGN.md section 3 (adopted where
 * the paper is silent).  The hot path is: delete the k lowest-logL live points, accumulate logX/logZ with the
 * saw-tooth live count (eq. 3-5), start k independent walkers, each doing a fixed number of
 * differential-evolution proposals in the unit hypercube (footnote P:120) with periodic wrap for ra/psi/phase
 * (P:196), a prior transform (Table 1), a frequency-domain GW log-likelihood ratio (P:153, P:174,
 * use_ratio P:196) and accept iff logL > logL* (P:96); then adapt the walk length at batch level.
 *
 * Conventions
 *  - All *_dev pointers are CUDA device pointers, fp64 (or int32 where typed), row-major, caller-owned.  The library copies
 *    strain / PSD / live points into handle-owned device memory in ns_init and never keeps a caller pointer afterwards.
 *  - *_host pointers are host memory.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *  - Calls enqueue work on `stream` and return without synchronising unless the comment says "synchronises".
 *  - Return value: 0 OK, -1 invalid argument, -2 CUDA error, -3 bad state/handle, -4 out of memory, -5 unsupported
 *    configuration.  ns_last_error() returns a static/handle-owned message.  No exceptions cross the ABI.
 *    A handle is not thread-safe.  There is no CPU fallback: without a CUDA device every compute call returns -2.
 *  - theta columns (Table 1 order): 0 Mc[Msun] 1 q 2 chi1 3 chi2 4 dL[Mpc] 5 theta_jn 6 psi 7 phase 8 tc[s]
 *    9 ra 10 dec.  Unit-cube rows u use the same order.  Unphysical theta (q not in (0,1], |chi|>1, dL<=0, Mc<=0,
 *    non-finite) gives logL = -inf for that row, never an error.
 */
#ifndef NSGW_H
#define NSGW_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NSGW_MAX_DIM 16
#define NSGW_MAX_DET 4
#define NSGW_STRUCT_VERSION 1

enum { NSGW_LIKE_GAUSSIAN_TOY = 0, NSGW_LIKE_GW_TAYLORF2 = 1, NSGW_LIKE_GW_PHENOMD_FORM = 2, NSGW_LIKE_CUBE_SHELL = 3 };
enum { NSGW_PRIOR_UNIFORM = 0, NSGW_PRIOR_POWERLAW2 = 1, NSGW_PRIOR_SINE = 2, NSGW_PRIOR_COSINE = 3, NSGW_PRIOR_FIXED = 4 };

typedef struct ns_handle ns_handle;

/* Problem + sampler description (plain data, copied by ns_init). */
typedef struct {
  int32_t struct_version;              /* NSGW_STRUCT_VERSION */
  int32_t like_kind;                   /* NSGW_LIKE_* ; GW kinds need ndim = 11 */
  int32_t ndim;                        /* 1..16 */
  int32_t n_live, n_delete;            /* k = n_delete (num_delete); 1 <= k <= n_live - 2 */
  int32_t naccept, maxmcmc;            /* 60, 5000 */
  double walks0;                       /* initial walk length (R:L13), e.g. 100 */
  double delay;                        /* walk-length smoothing; < 0 -> max(n_live/(10 k) - 1, 0) (R:L14) */
  int32_t prior_kind[NSGW_MAX_DIM];    /* NSGW_PRIOR_* per dimension; FIXED dims take the value prior_lo */
  double prior_lo[NSGW_MAX_DIM], prior_hi[NSGW_MAX_DIM];
  int32_t periodic[NSGW_MAX_DIM];      /* 1 = wrap the unit-cube coordinate instead of rejecting */
  int32_t n_det, n_freq;               /* GW: detectors (kernels are built for 1..3; 4 returns -5) and bins per detector */
  double f_min, df;                    /* f_k = f_min + k df, k = 0..n_freq-1 (both ends inclusive, R:L1) */
  double det_vertex[NSGW_MAX_DET][3];  /* Earth-fixed vertex position [m] */
  double det_xarm[NSGW_MAX_DET][3], det_yarm[NSGW_MAX_DET][3]; /* arm unit vectors */
  double gmst;                         /* Greenwich mean sidereal time at the reference epoch [rad] */
  double toy_mean[NSGW_MAX_DIM];       /* GAUSSIAN_TOY: logL = toy_lognorm - (theta-mean)^T P (theta-mean) / 2 */
  double toy_prec[NSGW_MAX_DIM * NSGW_MAX_DIM]; /* row-major [ndim][ndim] in the leading ndim*ndim entries */
  double toy_lognorm;
  const double* phenom_table_host;     /* [19][11] fit table (DESIGN.md A.2); NULL -> built-in surrogate default */
} ns_config;

/* Per-step report written by ns_step / ns_run. */
typedef struct {
  int64_t iteration;                   /* index of the step just done (0-based) */
  double logl_star;                    /* threshold = largest logL of the deleted batch */
  double logx, logz, h;                /* accumulators after the step (dead points only) */
  double dlogz;                        /* logaddexp(logZ, max logL_live + logX) - logZ            (R:L18 kind 0) */
  double live_frac_log;                /* logsumexp(logL_live) - ln n_live + logX - logZ          (R:L18 kind 1) */
  int32_t walk_len;                    /* W used by this step (R:L12) */
  int32_t pad0;
  double walks_next;                   /* real-valued walk length after adaptation (R:L13) */
  double accept_mean;                  /* mean accepted proposals per walker */
  int32_t accept_min, accept_max;
  int64_t n_eval, n_oob, n_stuck;      /* likelihood evaluations, out-of-bounds proposals, zero-accept walkers (R:L15) */
  int64_t n_eval_total;                /* since ns_init, including the initial live points */
} ns_stats;

/* Creates a sampler/likelihood context.  live_u_dev: [n_live, ndim] unit-cube points (NULL -> drawn from `seed`,
 * Philox tag 2).  strain_dev: [n_det, n_freq, 2] (re, im), time origin at the reference epoch (R:L4); psd_dev: [n_det, n_freq]
 * one-sided PSD; both NULL for non-GW kinds.  Precomputes the noise-weighted tables and evaluates logL of every live point.
 * n_live may be 0 (likelihood-only context: only gw_* and ns_prior_transform_batch / ns_walk_batch are then valid).
 * Synchronises. */
int ns_init(ns_handle** out, const ns_config* cfg, const double* live_u_dev, const double* strain_dev, const double* psd_dev,
            uint64_t seed, void* stream);
void ns_free(ns_handle* h);
const char* ns_last_error(const ns_handle* h); /* h may be NULL: message of the last failed ns_init */

/* logL of B physical parameter rows (R:L1: sum_det <d,h> - <h,h>/2).  parts_dev (optional) [B, 2 n_det] receives
 * <d,h>_det, <h,h>_det interleaved. */
int gw_loglike_batch(ns_handle* h, const double* theta_dev, int64_t B, double* logl_dev, double* parts_dev, void* stream);

/* Same with HOST buffers (the end-to-end entry point bench.py's `e2e` leg times).  Pinned (device-accessible) buffers are used in
 * place: the set-up kernel fetches theta_host [B, 11] over the host link while it computes, the finishing code stores into
 * logl_host [B].  Pageable buffers go H2D into handle-owned scratch -> the same kernels -> D2H.  Synchronises before returning. */
int gw_loglike_batch_host(ns_handle* h, const double* theta_host, int64_t B, double* logl_host, void* stream);

/* gw_loglike_batch for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc):
 * the same kernels (k_setup -> k_bins_lp + k_finish for TaylorF2, k_setup -> k_pd_lp for PhenomD-form; R:L1) with their scratch
 * -- coefficient blocks, per-range partial sums, tickets -- in ONE file-scope device array of NSGW_NOALLOC_SCRATCH_BYTES
 * (16.1 MiB) that every GPU loading the library holds until exit.  Calls no cudaMalloc / cudaFree and no allocating library
 * routine; enqueues on `stream` and does not synchronise.  theta_dev [B, 11] and logl_dev [B] are the caller's device buffers.
 * Limits: B <= NSGW_NOALLOC_MAX_ROWS and the handle's n_freq <= NSGW_NOALLOC_MAX_BINS; beyond either the call returns -5 with
 * the limit in ns_last_error and launches nothing (split the batch, or use gw_loglike_batch).  Every call on a device shares
 * the array: calls that overlap on the GPU (two streams, two handles, two host threads) race -- keep them on one stream or order
 * them with events.  The array keeps the last call's contents; the call clears what must start at zero itself.  Ranges are
 * 256 bins whatever B is, so logl_dev agrees with gw_loglike_batch to rounding order (1e-10 relative), not bit for bit.
 * Errors as gw_loglike_batch; the current device must be the handle's. */
#define NSGW_NOALLOC_MAX_ROWS 4096
#define NSGW_NOALLOC_MAX_BINS 16384
#define NSGW_NOALLOC_SCRATCH_BYTES 16908544
int gw_loglike_batch_noalloc(ns_handle* h, const double* theta_dev, int64_t B, double* logl_dev, void* stream);

/* Detector-frame signal of ONE parameter row on the handle's grid: out_dev [n_det, n_freq, 2] (R:L3). Used to build injections. */
int gw_waveform(ns_handle* h, const double* theta_dev, double* out_dev, void* stream);

/* Unit cube -> physical parameters (Table 1 kinds). */
int ns_prior_transform_batch(ns_handle* h, const double* u_dev, int64_t B, double* theta_dev, void* stream);

/* logL of B unit-cube rows under the handle's likelihood (transform + likelihood). */
int ns_loglike_u_batch(ns_handle* h, const double* u_dev, int64_t B, double* logl_dev, void* stream);

/* Lock-step acceptance walk of B walkers, walk_len proposals each, all against the frozen donor set
 * donors_u_dev [m, ndim] (m >= 2).  u_dev [B, ndim] / logl_dev [B]: start state in, end state out.  Walker row r uses Philox
 * counter (block, step, slot0 + r, stream_id), key = seed.  Counters (optional, may be NULL): accepted,
 * evaluated, out-of-bounds proposals per walker.  trace_flags_dev [B, walk_len] u8 (bit0 oob, bit1 accepted, bit2 evaluated)
 * and trace_logl_dev [B, walk_len] (NaN when not evaluated) are optional. */
int ns_walk_batch(ns_handle* h, const double* donors_u_dev, int32_t m, double* u_dev, double* logl_dev, int64_t B,
                  double logl_star, int32_t walk_len, uint64_t seed, uint32_t stream_id, int64_t slot0,
                  int32_t* n_accept_dev, int32_t* n_eval_dev, int32_t* n_oob_dev, uint8_t* trace_flags_dev,
                  double* trace_logl_dev, void* stream);

/* One nested-sampling iteration: select the k lowest, evidence scan, start points, walks, write-back, adapt.
 * stats_host (optional) is filled after a stream synchronise (synchronises iff non-NULL).  dead_dev (optional) [k, ndim+3]
 * receives (u.., logL, log w, n_i) of the deleted points in ascending logL. */
int ns_step(ns_handle* h, ns_stats* stats_host, double* dead_dev, void* stream);

/* Steps until the termination rule fires (term_kind 0: dlogz < tol; 1: live evidence fraction < tol) or
 * max_iter.  dead_dev (optional) [max_iter * k, ndim+3].  Returns the number of steps done (>= 0) or an error (< 0).
 * Synchronises once per step (one 128-byte read-back). */
int64_t ns_run(ns_handle* h, int32_t term_kind, double term_tol, int64_t max_iter, ns_stats* last_host, double* dead_dev,
               void* stream);

/* Runs n_runs independent samplers concurrently on one GPU (the paper's population studies, are many
 * independent runs).  Each handle steps on a stream of its own, so the walk kernels of different runs share the SMs: one run with
 * k = n_live/2 walkers leaves SM slots empty (3.4 walkers per SM at k = 500) and its kernels have tails; several runs fill them.
 * Every run is bit-identical to the same handle driven by ns_run.  All runs use the same termination rule; a finished run stops
 * stepping.  last_host[n_runs], iters_host[n_runs] (either may be NULL) receive each run's last statistics and iteration count;
 * dead_dev (may be NULL, and so may its entries) holds one [max_iter * k, ndim+3] device buffer per run.  Synchronises once per
 * round.  Returns the total number of iterations performed, or a negative error code. */
int64_t ns_run_many(ns_handle** hs, int32_t n_runs, int32_t term_kind, double term_tol, int64_t max_iter, ns_stats* last_host,
                    int64_t* iters_host, double** dead_dev);

/* Hit-and-run slice-sampling inner kernel (the blackjax-ns default the paper builds on, and names as a future
 * comparison; reading R:L25), as a batch call with the same shape as ns_walk_batch: every row of u_dev [B, ndim]
 * (in: start, out: end; logl_dev [B] likewise) does n_steps slice steps under "inside the unit cube (periodic dims wrap) and
 * logL > logl_star".  One step: direction Lc z / |z| with z ~ N(0, I) over the non-FIXED dims and lc_dev [ndim, ndim] a
 * lower-triangular factor (row-major; e.g. the Cholesky factor of the live points' covariance in unit-cube coordinates); bracket of
 * width 1 placed uniformly about the point, stepped out while its ends are inside (at most 32 times per end); shrinkage with
 * uniform candidates (at most 64).  Philox counter (block, step, slot0 + row, stream_id) as in ns_walk_batch.  Counters (each
 * may be NULL): likelihood evaluations, out-of-cube candidates, bracket expansions, rejected shrink candidates, steps that gave up.
 * trace_evals_dev / trace_logl_dev (optional, [B, n_steps]): evaluations of each step and logL after it.  The number of
 * evaluations per step varies from walker to walker (this is the divergence the acceptance walk avoids).  Exact likelihood only
 * (-5 when NSGW_OPT_LIKELIHOOD selects relative binning). */
int ns_slice_batch(ns_handle* h, const double* lc_dev, double* u_dev, double* logl_dev, int64_t B, double logl_star, int32_t n_steps,
                   uint64_t seed, uint32_t stream_id, int64_t slot0, int32_t* n_eval_dev, int32_t* n_oob_dev, int32_t* n_expand_dev,
                   int32_t* n_shrink_dev, int32_t* n_stuck_dev, int32_t* trace_evals_dev, double* trace_logl_dev, void* stream);

/* ---- Relative binning ("heterodyned likelihood"; the paper names it as the remedy for the bins x samples cost,
 * P:172, and gives no formula: DESIGN.md reading R:L24 restates the published scheme). ----
 * ns_relbin_setup builds, on the device, the summary data about the fiducial parameters theta0_host[11] (physical, Table-1 order):
 * bin edges equally spaced in Delta(f) = 2 pi chi sum_gamma sgn(gamma) (f/f*_gamma)^gamma with floor(Delta_tot/eps) bins (or the
 * caller's edges_host[n_edges]: strictly increasing grid indices from 0 to n_freq-1; pass NULL, 0 for the default), and per
 * detector and bin A0, A1 (complex), B0, B1.  Replaces any earlier set-up of the handle.  Synchronises.  *n_bins_host (may be
 * NULL) receives the number of bins.  Errors: -1 bad chi/eps/edges or unphysical theta0, -3 no GW likelihood.
 * ns_relbin_get copies out the edges [n_bins+1] and/or the summary data laid out A0[n_det][n_bins][2], A1[n_det][n_bins][2],
 * B0[n_det][n_bins], B1[n_det][n_bins] (host pointers, either may be NULL).  Synchronises.
 * gw_loglike_relbin_batch: as gw_loglike_batch, with <d,h> ~ Re sum_b [A0 conj(r0) + A1 conj(r1)] and
 * <h,h> ~ sum_b [B0 |r0|^2 + 2 B1 Re(r0 conj(r1))], r = h(theta)/h(theta0) at the bin edges: the waveform is evaluated at
 * n_bins+1 frequencies per row instead of n_freq.  An approximation of gw_loglike_batch: exact when r is constant (distance,
 * phase), second order in the bin width otherwise.  parts_dev as in gw_loglike_batch. */
int ns_relbin_setup(ns_handle* h, const double* theta0_host, double chi, double eps, const int32_t* edges_host, int32_t n_edges,
                    int32_t* n_bins_host, void* stream);
int ns_relbin_get(ns_handle* h, int32_t* edges_host, double* summary_host, void* stream);
int gw_loglike_relbin_batch(ns_handle* h, const double* theta_dev, int64_t B, double* logl_dev, double* parts_dev, void* stream);

/* Copies the live set out: u_dev [n_live, ndim], logl_dev [n_live] (either may be NULL). */
int ns_get_live(ns_handle* h, double* u_dev, double* logl_dev, void* stream);

/* Adds the remaining live points (n_i = n, n-1, .., 1; R:L17) to a copy of the accumulators.  Synchronises. */
int ns_finalize_evidence(ns_handle* h, double* logz_host, double* logz_err_host, double* h_host, void* stream);

/* Weighted posterior sample of a run ("posterior samples as a natural by-product"; "weights ... calculated using the
 * prior volumes enclosed between successive dead points and the likelihoods"; DESIGN reading R:L26).  Rows: the n_dead rows of
 * dead_dev ([n_dead, ndim+3] device, as ns_step / ns_run wrote them; may be NULL when n_dead = 0) followed by the handle's
 * n_live live points in ascending logL, whose widths continue the shrinkage with n_i = n, n-1, .., 1 (R:L17).  N = n_dead + n_live.
 * theta_dev [N, ndim] (device, optional) receives the prior transform of every row; logp_dev [N] (device, required) the
 * normalised log posterior weight logL_i + log w_i - logZ, logZ = log sum_i L_i w_i over the rows.  summary_host (optional,
 * [2 + ndim] host doubles; the call synchronises iff it is given): logZ, Kish's effective sample size 1 / sum p_i^2, and per
 * parameter the credible level sum_i p_i [theta_i,d < theta_ref_host[d]] of a reference point (host, [ndim], physical
 * parameters; optional, needs theta_dev; NaN when absent) -- the statistic a PP test histograms.  The handle's sampler
 * state is not changed.  Errors: -1 bad arguments, -3 no live set. */
int ns_posterior(ns_handle* h, const double* dead_dev, int64_t n_dead, double* theta_dev, double* logp_dev,
                 const double* theta_ref_host, double* summary_host, void* stream);

/* Equal-weight posterior sample by systematic resampling of the rows ns_posterior produced (DESIGN reading R:L27): one uniform
 * U from the Philox block with counter (0, 0, 0, 4 << 24) under key = seed; draw j = 0..n_out-1 sits at (j + U) / n_out of the
 * cumulative weights C_i = p_0 + .. + p_i (row order) and takes the first row with C_i > (j + U) / n_out * C_{N-1}; row i is
 * drawn floor(n_out p_i) or ceil(n_out p_i) times.  logp_dev [N] (device); cum_dev [N] (device scratch, receives C);
 * idx_dev [n_out] int64 (device, optional) the drawn rows, ascending; theta_out_dev [n_out, ndim] (device, optional) the rows of
 * theta_dev [N, ndim] gathered.  At least one output.  Asynchronous on `stream`.  Errors: -1 bad arguments. */
int ns_posterior_resample(ns_handle* h, const double* logp_dev, const double* theta_dev, int64_t N, int64_t n_out, uint64_t seed,
                          double* cum_dev, int64_t* idx_dev, double* theta_out_dev, void* stream);

/* Checkpoint / resume (the paper stores the dead points).  The sampler's whole state is the live set, the
 * evidence accumulators, the real-valued walk length, the iteration counter and the seed: every random number is a function of
 * (seed, iteration, walker slot, step), so a handle created from the same configuration and data and given this state continues
 * bit-for-bit as the original would have.  ns_get_state copies the scalars to *state_host and the live set to live_u_dev
 * [n_live, ndim] / live_logl_dev [n_live] (device; either may be NULL); ns_set_state installs them (all three required).  Both
 * synchronise.  Errors: -1 bad arguments / state, -3 no live set. */
typedef struct {
  int32_t struct_version;              /* NSGW_STRUCT_VERSION */
  int32_t pad0;
  int64_t iteration;                   /* steps done so far */
  int64_t n_eval_total;
  double logx, logz, h;                /* accumulators over the dead points */
  double walks;                        /* real-valued walk length (R:L13) */
  uint64_t seed;
} ns_state;
int ns_get_state(ns_handle* h, ns_state* state_host, double* live_u_dev, double* live_logl_dev, void* stream);
int ns_set_state(ns_handle* h, const ns_state* state_host, const double* live_u_dev, const double* live_logl_dev, void* stream);

/* Theoretical occupancy of the kernel that evaluates the likelihood of `rows` proposals in one round of the worklist walk
 * (NSGW_OPT_WALK_KERNEL): resident warps per SM as a fraction of 64 (occupancy API x the share of the SMs' CTA slots the launch
 * fills) in *warps_active_host, CTAs per SM in *ctas_per_sm_host (either may be NULL).  For the config-5 sweep's report. */
int nsgw_sweep_occupancy(ns_handle* h, int64_t rows, double* warps_active_host, int32_t* ctas_per_sm_host);

/* Device FP64 FMA throughput probe used for the roofline denominator: runs `iters` dependent-chain DFMAs x 8 chains per
 * thread on a full grid and returns achieved TFLOP/s in *tflops_host (synchronises; timed with CUDA events). */
int nsgw_measure_fp64_peak(int64_t iters, double* tflops_host, void* stream);

/* Optional timing of the dominant kernel (the bin sweep of gw_loglike_batch): while enabled, every launch is bracketed by a
 * CUDA event pair on the launching stream (at most 4096 pairs are kept).  nsgw_profile_read synchronises on those events,
 * returns their summed duration and count, and clears them. */
int nsgw_profile_enable(ns_handle* h, int32_t on);
int nsgw_profile_read(ns_handle* h, double* total_ms_host, int64_t* launches_host);

/* Tuning / test options of a handle.  key NSGW_OPT_BINS_KERNEL selects the kernel behind gw_loglike_batch (and the initial
 * live-set evaluation): 0 = automatic (by model and batch size), 1 = CTA per particle (pair), bins strided over threads
 * (k_bins; both models), 2 = lane per particle, bin tiles staged in shared memory (k_bins_lp for TaylorF2, k_pd_lp for
 * PhenomD-form).  Both compute the same sums in a different, fixed order.
 * Returns -1 for an unknown key or value. */
#define NSGW_OPT_BINS_KERNEL 0
/* key NSGW_OPT_WALK_SPEC: speculative chunk size of the GW walk kernel.  k_walk_gw proposes consecutive steps of a walker from
 * its current point until that many of them are in bounds (at most 128 steps), sets those up and evaluates them together, and
 * discards the steps after the first acceptance; results are identical for every value.  0 = automatic (every walker adapts
 * its own size between 1 and 32 from its chain: halved after a chunk with an acceptance, doubled after one without),
 * 1..32 = fixed (1 = one likelihood evaluation at a time, the sequential algorithm). */
#define NSGW_OPT_WALK_SPEC 1
/* key NSGW_OPT_LIKELIHOOD: 0 = exact likelihood (default), 1 = relative binning (needs ns_relbin_setup): used by ns_step / ns_run
 * / ns_walk_batch / ns_loglike_u_batch.  Setting it re-evaluates the live points' logL with the chosen likelihood (default
 * stream, synchronises); do so again after a new ns_relbin_setup. */
#define NSGW_OPT_LIKELIHOOD 2
/* key NSGW_OPT_INNER_KERNEL: what ns_step / ns_run replace the deleted points with: 0 = the acceptance walk (default; the paper's
 * kernel), 1 = hit-and-run slice sampling (R:L25): direction factor = Cholesky factor of the covariance of the surviving live
 * points (recomputed on the device every iteration), NSGW_OPT_SLICE_STEPS steps per replacement (key 4; 0 = 5 per non-FIXED
 * dimension), no walk-length adaptation; ns_stats then reports walk_len = the number of slice steps and accept_* = the steps that
 * moved the point.  Exact likelihood only. */
#define NSGW_OPT_INNER_KERNEL 3
#define NSGW_OPT_SLICE_STEPS 4
/* key NSGW_OPT_WALK_STAGE: 1 = the PhenomD-form walk kernel stages the table values of each thread's next bin in shared memory
 * with asynchronous copies (same arithmetic, bit-identical results; costs chunk slots, measured 10 % slower on config 3);
 * 0 (default) = plain loads.  A tuning switch. */
#define NSGW_OPT_WALK_STAGE 5
/* key NSGW_OPT_WALK_KERNEL: how ns_step / ns_run / ns_walk_batch run the acceptance walk on a GW likelihood.  0 = automatic
 * (exact likelihood: 3 when walkers x expected chunk length -- from the walk length and naccept -- reaches 12000 rows per round, else 2;
 * relative binning: 1); 1 = one CTA per walker, all steps in one launch (k_walk_gw); 2 and 3 =
 * batch-wide rounds: every walker proposes a chunk of steps, the likelihood of all the batch's in-bounds proposals is evaluated in one
 * launch, every walker resolves its chunk (first acceptance discards the later steps), repeat; the host follows the device two rounds
 * behind, so these calls synchronise with the stream while they run.  2 sweeps the rows with the CTA-per-row-pair kernel (k_bins),
 * 3 with the lane-per-row kernels (k_pd_lp for PhenomD-form, k_bins_lp for TaylorF2).  For a given value, decisions, counters,
 * traces and end points are identical for every chunk length and batch composition; between values the kernels sum a row's bins
 * in different fixed orders, so logL agrees to rounding (1e-12) and a decision can differ only where logL is that close to logL*. */
#define NSGW_OPT_WALK_KERNEL 6
/* key NSGW_OPT_HOST_ZERO_COPY: 1 (default) = gw_loglike_batch_host reads theta and writes logL in place when both buffers are pinned
 * (device-accessible) host memory, with no copy in the stream; 0 = always copy through handle-owned device scratch.  Same results. */
#define NSGW_OPT_HOST_ZERO_COPY 7
int nsgw_set_option(ns_handle* h, int32_t key, int32_t value);

/* Number of kernels launched by this library since process start (for bench.py's gpu_launches). */
int64_t nsgw_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* NSGW_H */
