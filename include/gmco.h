/* gmco.h -- C ABI of libgmco: the gL-BFGS hot path of gMCO (arXiv 1904.01567) on one B200.
 *
 * The library optimises K HDR-brachytherapy plans in parallel.  Every plan shares the
 * dose-rate matrix D and the structure table and has its own hidden weights
 * (Eq. 4).  One "round" on the device is
 *     dose  d = D t, t = x o x            PAPER.md:55-59  (Eq. 1, dwell weights x = sqrt(t))
 *     penalty f, derivative r = dF/dd     PAPER.md:61-66  (Eq. 2)
 *     objective F = sum_j w_j mean_i f    PAPER.md:71-74  (Eq. 4)
 *     gradient g = 2 x o (D^T r)          PAPER.md:66-69  (Eq. 3 summed over points)
 *     L-BFGS two-loop + Armijo step       PAPER.md:115-119 (Liu & Nocedal; reading DESIGN.md 2.2)
 * and nothing crosses the host/device boundary inside the loop.
 *
 * Conventions for EVERY entry point
 *   - Pointers marked "host or device" may be either: copies use cudaMemcpyDefault (UVA).
 *     All arrays are fp32 (int32 where stated), dense, C order, no aliasing between arguments.
 *   - The caller owns every argument buffer; the handle owns only what it allocates itself
 *     and gmco_destroy frees it.  Input buffers may be freed as soon as the call returns
 *     (host inputs) or as soon as the stream has passed the call (device inputs).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *     gmco_create / gmco_optimize / gmco_evaluate only ENQUEUE work on it;
 *     gmco_result synchronises it.
 *   - Return value: GMCO_OK (0) or a negative gmco_status; never throws, aborts or prints.
 *     gmco_last_error(h) gives a message for the last failure on that handle
 *     (gmco_last_error(NULL) for a failed gmco_create).
 *   - Requires an sm_100 device (B200).  There is no CPU fallback: without a usable GPU
 *     every compute entry point returns GMCO_E_UNSUPPORTED or GMCO_E_CUDA.
 */
#ifndef GMCO_H_
#define GMCO_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define GMCO_API __attribute__((visibility("default")))
#else
#define GMCO_API
#endif

#define GMCO_VERSION 140          /* 0.1.4: gmco_tc_info.grad_pair, gmco_options.dose_kernel = 2 */
#define GMCO_MAX_STRUCTS 8
#define GMCO_MAX_HISTORY 16
#define GMCO_MAX_CRITERIA 8
#define GMCO_MAX_OBJECTIVES 16
#define GMCO_MAX_RADIAL_COEF 8

typedef enum gmco_status {
  GMCO_OK = 0,
  GMCO_E_INVALID = -1,      /* NULL pointer, bad size, NaN/negative input, sizes do not add up   */
  GMCO_E_UNSUPPORTED = -2,  /* no sm_100 device, or a size outside the supported range            */
  GMCO_E_CUDA = -3,         /* a CUDA call failed (message holds cudaGetErrorString), or a kernel reported a
                               protocol error through the device error word (message names kernel and site) */
  GMCO_E_NOMEM = -4,        /* device allocation failed                                           */
  GMCO_E_STATE = -5         /* call out of order (e.g. gmco_result before gmco_optimize)          */
} gmco_status;

/* Precision / pipe of the two contractions D t and D^T r. */
typedef enum gmco_precision {
  GMCO_PREC_TF32X3 = 0,     /* tcgen05 kind::tf32, 3-product split (fp32-equivalent); cases with more than
                               384 dwell positions do not fit the tensor layout and run as SIMT_FP32  */
  GMCO_PREC_SIMT_FP32 = 1   /* plain fp32 FMA kernels (reference datum and debug route)            */
} gmco_precision;

/* Arithmetic of gmco_sa_run. */
typedef enum gmco_sa_precision {
  GMCO_SA_FP64 = 0,         /* dose, penalty differences and the accept test in fp64: the parity route   */
  GMCO_SA_FP32 = 1          /* everything in fp32: the speed route                                       */
} gmco_sa_precision;

/* Per-plan exit status written by gmco_result. */
typedef enum gmco_plan_status {
  GMCO_PLAN_ITERS = 0,      /* ran the full iteration budget                                       */
  GMCO_PLAN_CONVERGED = 1,  /* eps rule met or gradient exactly zero                */
  GMCO_PLAN_STALLED = 2     /* max_trials step halvings without an Armijo decrease                 */
} gmco_plan_status;

/* One penalised point group ("structure": an organ, or one point class of it; Table 1,
 * PAPER.md:80-88).  Rows of D belong to structures contiguously, in table order. */
typedef struct gmco_structure {
  int32_t n_points;   /* > 0                                                                      */
  float d_lo, d_hi;   /* D_min, D_max of Eq. 2 in Gy; -INFINITY / +INFINITY disables a side       */
  float w_lo, w_hi;   /* class-solution weights w_min, w_max (>= 0)                               */
  int32_t dvh_kind;   /* 0 none | 1 V_level: % of points with d >= level% of Rx
                                | 2 D_level: dose of the ceil(level% * n)-th hottest point, % of Rx */
  float dvh_level;    /* percent, e.g. 100 (V100), 75 (V75), 10 (D10)         */
} gmco_structure;

typedef struct gmco_options {
  int32_t m;          /* L-BFGS history length, 1..GMCO_MAX_HISTORY           default 10          */
  float eps;          /* stop a plan when |F - F+| <= eps max(F, 1e-30); 0 = off      default 0   */
  float c1;           /* Armijo constant                                      default 1e-4        */
  int32_t max_trials; /* step halvings before a plan is declared stalled      default 20          */
  int32_t precision;  /* gmco_precision                                       default TF32X3      */
  float eps_f;        /* objective-noise allowance of the approximate line-search test: a trial
                         step that fails Armijo is still accepted when F+ <= F + eps_f |F| and
                         g+.p <= (2 c1 - 1) g.p (Hager & Zhang 2005; reading A5b).
                         0 = Armijo only                                      default 1e-6        */
  int32_t compaction; /* 1: the tensor route packs the plans that are still running into the leading
                         128-plan tiles every round, so a round costs what the RUNNING plans cost
                         (plans stop at different rounds: eps > 0, or unequal numbers of
                         step halvings); 0: every plan keeps its tile            default 1        */
  int32_t dose_kernel;/* 0: automatic -- the DOSE contraction runs on CTA pairs (tcgen05 cta_group::2) where the shape
                         allows, else on one CTA per plan tile;
                         1: round 1's kernel choice -- always one CTA per plan tile.  The choices compute the same
                         products; they differ in partial-sum order (low-order bits).  gmco_stats.dose_kernel
                         says which one ran.
                         2: as 0, and the GRADIENT contraction runs on CTA pairs as well (k_grad_tc_pair: each CTA
                         loads half of every D slab) where the shape allows -- at most 256 dwell positions, even
                         numbers of plan tiles and of 32-dwell groups; else as 0.  Not the default: it has run
                         on the CPU emulation of the kernels only.     default 0        */
  int32_t wide_accum; /* above 256 dwell positions (streamed T_lo layout) only.  1: the main product T_hi D_hi is
                         accumulated in TWO TMEM accumulators (first / second half of the dwell groups) that the
                         epilogue sums in fp32, which halves the tensor core's truncation error at
                         the price of a shallower operand ring (4 instead of 8 dwell groups of T_hi stay in TMEM);
                         0: one main accumulator.  Not yet validated on hardware.        default 0        */
  int32_t line_search;/* 0: a rejected trial step is halved and evaluated in the next round's batched contraction
                         (the plan rides along: one extra column per halving).  1: polynomial line search of
                         north_star item (4): when the first trial step (alpha = 1) of an iteration is rejected, the
                         dose columns d = D(x o x), a = D(x o p), b = D(p o p) of that plan are formed once and every
                         further candidate alpha = 1/2, 1/4, ... is valued from d + 2 alpha a + alpha^2 b without a
                         contraction; the first candidate that meets the acceptance rule becomes the next trial
                         point, which is then evaluated afresh (an iteration with h rejected steps costs 2 rounds
                         instead of 1 + h).  Same algorithm, same iteration counts.  On the stand-in cases no
                         iteration has more than two rejected steps, so it saves 0.5 % of plan-rounds and costs
                         two more launches per round: off by default.  Not yet validated on
                         hardware.                                                default 0        */
} gmco_options;

/* Counters of the last gmco_optimize + gmco_result pair (host side, filled by gmco_result). */
typedef struct gmco_stats {
  int64_t device_bytes;     /* bytes currently allocated by the handle                            */
  int32_t rounds;           /* evaluation rounds that had a running plan (1 + iterations + backtracks of the slowest plan) */
  int32_t kernel_launches;  /* kernels launched by the library since gmco_optimize was called     */
  int32_t plans_iters, plans_converged, plans_stalled;
  int32_t eval_launches;    /* profiling only: contraction launches that had work (see gmco_set_profiling) */
  float eval_ms;            /* profiling only: summed device time of those launches, CUDA events  */
  int32_t eval_plans;       /* profiling only: plan-evaluations those launches did (running plans, summed over rounds) */
  float dose_ms, grad_ms, step_ms; /* profiling only: eval_ms split into the dose kernel and the gradient kernel, and the
                               summed device time of the per-plan step kernel of the same rounds                */
  int32_t dose_kernel;      /* gmco_tc_info.dose_kernel of the dose kernel that ran (-1 on the SIMT route)        */
} gmco_stats;

/* Launch schedule and on-chip layout of the tensor route for one shape: what gmco_optimize would launch.  Host
 * arithmetic only (no GPU needed): used by the tests to prove on the CPU that every shape's shared-memory carve-up,
 * TMEM columns and TMA boxes fit, and by bench.py to record which kernels ran. */
typedef struct gmco_tc_info {
  int32_t ok;               /* 0: the shape does not run on the tensor route (n_dwell > 384)                      */
  int32_t a_pad, n_pad, n_alloc, k_pad;   /* padded sizes: dwell columns (32), points (64 per structure), rows allocated (256), plans (128) */
  int32_t n_tiles, segs, n_chunks, n_slabs, compact_cap;
  int32_t dose_kernel;      /* 0 k_dose_tc<resident T_lo>, 1 k_dose_tc<streamed T_lo>, 2 k_dose_tc_pair<static schedule>,
                               3 k_dose_tc_pair<run-time ring>                                                    */
  int32_t dose_threads, dose_stages, dose_stage_bytes, dose_smem_bytes, dose_smem_end, dose_scr_slot, dose_tmem_cols;
  int32_t dose_tmem_groups, dose_n_main; /* dwell groups of T_hi kept in TMEM; main accumulators (2 with wide_accum) */
  int32_t grad_threads, grad_ps, grad_stages, grad_stage_bytes, grad_smem_bytes, grad_smem_end, grad_staging_bytes,
      grad_tmem_cols;
  int32_t smem_limit, tmem_limit;        /* 232448 B opt-in dynamic shared memory per CTA, 512 TMEM columns       */
  int32_t grad_pair;        /* 1: the gradient kernel is k_grad_tc_pair (dose_kernel = 2 and the shape allows it); the
                               grad_* fields above then describe that kernel                                       */
} gmco_tc_info;


typedef struct gmco_handle gmco_handle;

GMCO_API int gmco_version(void);                       /* GMCO_VERSION of the loaded library               */
GMCO_API void gmco_default_options(gmco_options* opt); /* fills the defaults listed above                  */

/* a0 -- case setup (PAPER.md:97 step (i) hands over the dose-rate matrix; PAPER.md:113 first
 * transfer).  Copies D (host or device, [n_points][ldD] with ldD >= n_dwell, point-major as
 * in Eq. 1) into the handle's padded, pre-split device layout; the caller may free D afterwards.
 * structs: HOST array of n_structs (1..GMCO_MAX_STRUCTS) entries, sum n_points == n_points.
 * rx_dose: prescription in Gy (> 0), used by the DVH indices only.  opt may be NULL.
 * Limits: 1 <= n_dwell <= 480.  On failure *out is NULL. */
GMCO_API int gmco_create(gmco_handle** out, const float* D, int64_t n_points, int64_t n_dwell, int64_t ldD,
                const gmco_structure* structs, int32_t n_structs, float rx_dose,
                const gmco_options* opt, void* cuda_stream);

/* a1-a7 -- optimise K plans for `iters` L-BFGS iterations each.
 * T0: start dwell times in seconds, >= 0, [K][n_dwell] or, if t0_broadcast != 0, [n_dwell]
 * shared by all plans (host or device).  weights: hidden weights [K][n_structs][2] = (lo, hi)
 * per structure, >= 0 (host or device); the effective weight of a term is
 * weights[k][s][side] * structs[s].w_side / structs[s].n_points (Eq. 4 x Table 1; the
 * library does NOT normalise hidden weights to sum 1).  K = 0 and iters = 0 are valid
 * (iters = 0 evaluates the start point only).  Enqueues on cuda_stream and returns. */
GMCO_API int gmco_optimize(gmco_handle* h, const float* T0, int32_t t0_broadcast, const float* weights,
                  int32_t K, int32_t iters, void* cuda_stream);

/* a8 -- results of the last gmco_optimize (PAPER.md:113 second transfer; DVH indices
 * PAPER.md:132-140).  Finishes any plan that still has backtracking rounds outstanding,
 * evaluates dose once more at the final dwell times, and writes (host or device, any may be NULL):
 *   T [K][n_dwell] seconds; objective [K]; dvh [K][n_structs] (0 where dvh_kind = 0);
 *   objective_terms [K][n_structs][2]; iters_done [K]; plan_status [K] (gmco_plan_status).
 * Synchronises the stream given to gmco_optimize.  GMCO_E_STATE if no optimisation ran. */
GMCO_API int gmco_result(gmco_handle* h, float* T, float* objective, float* dvh, float* objective_terms,
                int32_t* iters_done, int32_t* plan_status);

/* Test / debug hook -- one evaluation (Eqs. 1-4) of K plans at dwell times T ([K][n_dwell],
 * or [n_dwell] if t_broadcast) through the SAME kernels the optimiser uses.  Outputs (host or
 * device, any may be NULL): dose [n_points][K] (plan fastest) -- the fused path never stores
 * dose otherwise; F [K]; grad_x [K][n_dwell] = dF/dx with x = sqrt(T).  Enqueues, then
 * synchronises the stream (it is a test hook: the input check and the device error word are
 * read back before it returns).  Discards any optimisation state. */
GMCO_API int gmco_evaluate(gmco_handle* h, const float* T, int32_t t_broadcast, const float* weights,
                  int32_t K, float* dose, float* F, float* grad_x, void* cuda_stream);

/* gSA -- K simulated-annealing chains on the case of `h`, the comparison method of the paper
 * (PAPER.md:96-113 steps (ii)-(v); move / cooling / acceptance rule from
 * BASELINE.json configs[4]).  Chain k starts at T0 and, at step n = 0..steps-1,
 *   j = jdx[n];  sigma = max(0.1 t_j, 0.01 tau);  t' = max(t_j + sigma z[n], 0);
 *   d' = d + (t' - t_j) D[:, j]  (incremental Eq. 1);  dF = F(d') - F(d)  (Eqs. 2, 4);
 *   accept if dF <= 0, else if u[n] < exp(-dF / T_n),  T_n = temp0 * exp(n ln cooling).
 * The random draws are INPUTS (the library owns no generator): jdx int32 in [0, n_dwell),
 * z ~ N(0,1) and u ~ U[0,1) as fp64, each [K][steps] or, if draws_broadcast != 0, [steps] shared
 * by all chains (host or device).  T0 / weights as in gmco_optimize.  tau: the scale of the move
 * floor in seconds (>= 0).  precision: gmco_sa_precision.
 * Outputs (host or device, any may be NULL): T [K][n_dwell] fp64 seconds; objective [K] fp64, summed
 * afresh from the final dose; n_accepted [K] int64 accepted moves (dF = 0 counts as accepted).
 * Enqueues on cuda_stream and synchronises it before returning.  Does not touch the state of
 * gmco_optimize / gmco_result.  GMCO_E_UNSUPPORTED if the chain state does not fit one CTA
 * (more than 12800 padded points in fp64, 25600 in fp32); GMCO_E_INVALID for an index outside
 * [0, n_dwell) or negative / non-finite T0, weights. */
GMCO_API int gmco_sa_run(gmco_handle* h, const float* T0, int32_t t0_broadcast, const float* weights, int32_t K,
                int64_t steps, const int32_t* jdx, const double* z, const double* u, int32_t draws_broadcast,
                double tau, double temp0, double cooling, int32_t precision, double* T, double* objective,
                int64_t* n_accepted, void* cuda_stream);

/* Step (i) -- the dose-rate matrix ("dose rate matrix calculation (repeated for N_pnt dose calculation
 * points x N_act dwell positions)"; the model is BASELINE.json configs[0]'s TG-43 point-source approximation):
 *   D[i][l] = sk_lambda * g(r) / r^2,   r = |points[i] - dwell[l]| / 10 (mm -> cm), r = max(r, r_floor_cm),
 *   g(r) = sum_c g_coef[c] r^c  (radial dose function as a polynomial in r [cm]; coefficients are inputs).
 * points [n_points][3], dwell [n_dwell][3]: fp32 millimetres (host or device); g_coef: HOST array of n_coef
 * (1..GMCO_MAX_RADIAL_COEF) doubles, lowest power first; D: [n_points][ldD] fp32, ldD >= n_dwell (host or device),
 * Gy/s per unit dwell weight.  fp64 arithmetic, rounded once to fp32.  Needs no handle; errors are reported through
 * gmco_last_error(NULL).  Enqueues on cuda_stream; synchronises it if any argument is a host pointer. */
GMCO_API int gmco_dose_rate_matrix(const float* points, int64_t n_points, const float* dwell, int64_t n_dwell,
                          const double* g_coef, int32_t n_coef, double sk_lambda, double r_floor_cm, float* D,
                          int64_t ldD, void* cuda_stream);

/* One DVH acceptance criterion (RTOG 0924 and the stricter RTOG+ set). */
typedef struct gmco_criterion {
  int32_t structure;      /* index into the structure table: the criterion reads dvh[k][structure]               */
  int32_t sense;          /* +1: index >= limit (target coverage, V100 >= 90 %);  -1: index < limit (D10 < 118 %) */
  float limit_rtog;       /* in the units of that DVH index (the caller turns "1 cc" into % of the organ's points) */
  float limit_rtog_plus;  /* RTOG+ differs from RTOG only in the target coverage (95 %)                           */
  int32_t role;           /* 0 target: its index ranks the valid plans (highest wins)
                             1 must hold for a fallback plan (urethra)
                             2 organ at risk whose indices are summed to rank the fallback plans (bladder, rectum) */
} gmco_criterion;

/* Plan evaluation and selection from a pool (readings A22-A23).
 * dvh: [K][n_structs] as written by gmco_result (host or device).  Class of a plan: 2 = meets every RTOG+ limit,
 * 1 = meets every RTOG limit, 0 = violates at least one.  Selected plan, in descending priority: the RTOG+ plan
 * with the highest target index; else the RTOG plan with the highest target index; else, among the plans that meet
 * the RTOG limits of roles 0 and 1 (all plans if there is none), the one with the lowest sum of the role-2 indices
 * (fp32, summed in criterion order).  Ties go to the lowest plan index.
 * Outputs (host or device, any may be NULL): plan_class [K]; selected [1] (-1 if K = 0);
 * class_counts [3] = plans of class 0, 1, 2.  Enqueues on cuda_stream and synchronises it. */
GMCO_API int gmco_select_plan(gmco_handle* h, const float* dvh, int32_t K, const gmco_criterion* criteria,
                     int32_t n_criteria, int32_t* plan_class, int32_t* selected, int32_t* class_counts,
                     void* cuda_stream);

/* Pareto filter: plan a dominates plan b if objectives[a][m] <= objectives[b][m] for every m and
 * < for at least one m; a plan is non-dominated if no plan dominates it (equal plans do not dominate each other).
 * objectives: [K][M] fp32, every column minimised, 1 <= M <= GMCO_MAX_OBJECTIVES (host or device) -- e.g.
 * gmco_result's objective_terms viewed as [K][2 n_structs].  Outputs (host or device, any may be NULL):
 * nondominated [K] bytes (1 / 0); n_nondominated [1].  NaN compares false both ways: a plan with a NaN objective
 * neither dominates nor is dominated.  Enqueues on cuda_stream and synchronises it. */
GMCO_API int gmco_pareto_front(gmco_handle* h, const float* objectives, int32_t K, int32_t M,
                      uint8_t* nondominated, int32_t* n_nondominated, void* cuda_stream);

/* Counters of the last optimise/result pair.  GMCO_E_STATE before the first gmco_result. */
GMCO_API int gmco_get_stats(const gmco_handle* h, gmco_stats* out);

/* Schedule of the tensor route for a case of n_dwell dwell positions, structures of
 * struct_points[0..n_structs) points (HOST array) and K plans on a device with num_sms multiprocessors (148 on
 * B200); dose_kernel and wide_accum as in gmco_options.  Pure host arithmetic: needs no GPU and no handle.
 * GMCO_E_INVALID for NULL / non-positive arguments; out->ok = 0 (and GMCO_OK) when the shape is outside the tensor
 * route. */
GMCO_API int gmco_tc_schedule(int64_t n_dwell, const int32_t* struct_points, int32_t n_structs, int32_t K,
                     int32_t num_sms, int32_t dose_kernel, int32_t wide_accum, gmco_tc_info* out);

/* Measurement aid (bench.py's roofline leg).  With enable != 0 every kernel of a round of the
 * following gmco_optimize / gmco_result (the dose kernel: D t, penalty, objective; the gradient
 * kernel: D^T r; the per-plan step kernel) is bracketed by CUDA events on the caller's stream;
 * gmco_result sums their elapsed times over the rounds in which at least one plan was running and
 * reports them in gmco_stats (eval_ms = dose_ms + grad_ms, step_ms, eval_launches).  Off by
 * default; results are identical either way. */
GMCO_API int gmco_set_profiling(gmco_handle* h, int32_t enable);

/* Frees everything the handle owns (synchronises its stream first).  NULL is a no-op. */
GMCO_API void gmco_destroy(gmco_handle* h);

/* Message of the last error on h (or of the last failed gmco_create if h is NULL).
 * Valid until the next call on that handle from the same thread. */
GMCO_API const char* gmco_last_error(const gmco_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* GMCO_H_ */
