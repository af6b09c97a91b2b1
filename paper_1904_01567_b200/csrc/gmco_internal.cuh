// gmco_internal.cuh -- device layout, handle and kernel launch prototypes of libgmco.
// Product code: shares nothing with oracle/.  See DESIGN.md section 4 for the HBM layout.
#pragma once

#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>

#include "gmco.h"

namespace gmco {

constexpr int kChunk = 32;        // points per chunk: K-step granule of the gradient MMA, penalty granule
constexpr int kStructAlign = 64;  // every structure is padded to a multiple of this many rows
constexpr int kRowAlloc = 256;    // D rows are allocated up to a multiple of this (tile over-reads stay in bounds)
constexpr int kPlanTile = 128;    // plans per tensor tile = TMEM lanes
constexpr int kMaxApad = 480;     // 512 TMEM columns - at least one 32-point chunk of dose accumulator
constexpr int kMaxApadTensor = 384; // tensor route: T_hi (A_pad TMEM columns) + one 128-column accumulator pair
constexpr int kMaxNpl = kMaxApad / 32;  // dwell elements per lane in the warp-per-plan kernels
constexpr int kRoundLogCap = 8192;      // rounds whose running-plan count is logged (profiling aid)
constexpr int kLsCap = 128;             // polynomial line search (option): plans queued per round at most (kernels_ls.cu)

// per-plan status codes on the device
enum : int { PLAN_RUNNING = -1 };

// Device error word (PlanDev::dev_err, 4 ints): [0] DevErr code (0 = none; the first error wins), [1] site =
// DevErrKernel << 8 | DevErrWait, [2] blockIdx.x | blockIdx.y << 16, [3] detail.  Kernels never trap and never spin
// without a bound: a wait that does not complete, or a shared-memory / TMEM carve-up that does not fit, is written here,
// the kernel runs through its normal teardown, and the host turns the word into GMCO_E_CUDA after its next synchronise.
enum DevErr : int { DEVERR_NONE = 0, DEVERR_WAIT_TIMEOUT = 1, DEVERR_SMEM_LAYOUT = 2, DEVERR_TMEM_LAYOUT = 3 };
enum DevErrKernel : int { DEVERR_K_DOSE_RESIDENT = 1, DEVERR_K_DOSE_STREAMED = 2, DEVERR_K_DOSE_PAIR = 3, DEVERR_K_GRAD = 4, DEVERR_K_STEP = 5, DEVERR_K_GRAD_PAIR = 6 };
enum DevErrWait : int {
  DEVERR_W_EMPTY = 1, DEVERR_W_FULL = 2, DEVERR_W_TG_READY = 3, DEVERR_W_TIN_FULL = 4, DEVERR_W_ACC_FULL = 5,
  DEVERR_W_ACC_EMPTY = 6, DEVERR_W_CONV = 7, DEVERR_W_HISTORY = 8
};

// Static description of the case (gmco_create), all device pointers.
struct CaseDev {
  int N = 0, A = 0, S = 0;          // user sizes
  int N_pad = 0;                    // sum of structure sizes rounded up to kStructAlign
  int N_alloc = 0;                  // N_pad rounded up to kRowAlloc (rows that exist in memory)
  int A_pad = 0;                    // A rounded up to 32
  float rx = 0.f;
  float* D = nullptr;               // [N_alloc][A_pad] fp32, padded rows/cols are 0
  float* D_hi = nullptr;            // [N_alloc][A_pad] tf32 hi part   (tensor path: B operand of both contractions)
  float* D_lo = nullptr;            // [N_alloc][A_pad] tf32 lo part
  float* pt_lo = nullptr;           // [N_alloc] D_min of the point's structure (-inf on padding rows)
  float* pt_hi = nullptr;           // [N_alloc] D_max (+inf on padding rows)
  int* tile_struct = nullptr;       // [N_alloc / 64] structure id of each 64-row tile (uniform by construction)
  int* tile_valid = nullptr;        // [N_alloc / 64] leading rows of the tile that are real points (rest is padding)
  int* row_src = nullptr;           // [N_alloc] original row index, -1 on padding rows
  int* sel_pos = nullptr;           // [N_alloc] position inside the D_level selection buffer, -1 if unused
  int n_sel = 0;                    // total points of dvh_kind == 2 structures
};

struct StructHost {
  int n_points, row_begin /*padded*/, n_rows_pad, sel_begin;
  float d_lo, d_hi, w_lo, w_hi;
  int dvh_kind; float dvh_level;
};

// Per-K workspace (gmco_optimize / gmco_evaluate), all [K_pad] or [K_pad][A_pad].
struct PlanDev {
  int K = 0, K_pad = 0, m = 0;
  float *x = nullptr, *g = nullptr, *p = nullptr, *xt = nullptr;   // [K_pad][A_pad]
  float *T = nullptr;                                              // trial dwell times (GEMM operand), fp32; the dose kernel splits them
  float *T_lo = nullptr;                                           // tf32 lo part of T: only with more than 256 dwell positions (streamed layout)
  float *Sh = nullptr, *Yh = nullptr;                              // [m][K_pad][A_pad] history
  float *rho = nullptr, *gam = nullptr;                            // [m][K_pad] 1/(s.y) and (s.y)/(y.y)
  float *Weff = nullptr;                                           // [K_pad][2*S] weights * base / n_s
  float *WeffC = nullptr;                                          // [K_pad][2*S] the same by tile SLOT (compaction)
  int *slot = nullptr;                                             // [K_pad] row of the plan in T / R / the partials
  float *F = nullptr, *gp = nullptr, *alpha = nullptr;             // [K_pad]
  int *it_done = nullptr, *trials = nullptr, *hcount = nullptr, *hhead = nullptr, *status = nullptr;
  int *n_running = nullptr;                                        // [2] ping-pong counter of RUNNING plans
  int *tile_seg = nullptr;                                         // [K_pad / 128 + 1] partial-slot range of each plan tile (tensor route)
  int *round_log = nullptr;                                        // [kRoundLogCap] running plans at the start of round r
  int *rounds_done = nullptr;                                      // [2] rounds the device-driven loop has gone through (its bound) | rounds that had a running plan
  int *bad_input = nullptr;                                        // [1] set when T0 / weights hold NaN, inf or negatives
  int *dev_err = nullptr;                                          // [4] device error word (DevErr above)
  // polynomial line search (gmco_options.line_search = 1; all null otherwise)
  int *ls_list = nullptr;                                          // [kLsCap] plans whose first trial step was rejected this round
  int *ls_count = nullptr;                                         // [2] how many | finished CTAs of k_ls_pick
  float *ls_cols = nullptr;                                        // [3][kLsCap][N_alloc] dose columns d, a, b of the queued plans
  // partial results of one evaluation round
  float *Fpart = nullptr; float *Gpart = nullptr;
  float *R = nullptr;               // SIMT route: dF/dd [K_pad][N_alloc]; tensor route: dF/dd / 2 [N_alloc][K_pad]
  int nF = 0, nFcomp = 1, nG = 0;                                  // SIMT: slot counts (uniform over plans)
  // result staging
  float *res_terms = nullptr;                                      // [K_pad][2*S]
  int *res_cnt = nullptr;                                          // [K_pad][S]
  float *res_sel = nullptr;                                        // [K_pad][n_sel]
  float *res_dvh = nullptr;                                        // [K_pad][S]
};

struct StepParams {
  int K, A_pad, m, iters, max_trials;
  float c1, eps, eps_f;
  // partial layout
  const float* Fpart; int nF, nFcomp; long long f_slot_stride;
  const float* Gpart; int nG; long long g_slot_stride;
  int tile_local;                     // 1: partial rows are indexed by plan % 128 and slots come from tile_seg
  const int* tile_seg;                // [n_tiles + 1] slot range of each plan tile (tensor path)
  int compact_cap, total_ctas;        // compaction (tensor path): segment cap per tile and CTAs per grid; 0 = off
  int dose_pair;                      // the objective partials follow the CTA-pair split (kernels_tc.cu compact_remap_pair)
  int grad_pair;                      // so do the gradient partials (k_grad_tc_pair, gmco_options.dose_kernel = 2)
  int S;
  int ls_cap;                         // > 0: a plan whose FIRST trial step is rejected is queued for the polynomial line search
};

// ---- kernel launchers (each returns the number of kernels it launched, or < 0 on CUDA error) ----
int launch_setup_case(const CaseDev& c, const float* D_user, long long ldD, const int* row_src_dev,
                      bool want_split, cudaStream_t st);
int launch_init_plans(const CaseDev& c, const PlanDev& p, const float* T0, int t0_bcast, const float* w_user,
                      const float* struct_scale /*[2S] base/n*/, cudaStream_t st);
// gate: device int; the kernel returns at once when *gate == 0 (no plan is running); nullptr = always run
int launch_simt_eval(const CaseDev& c, const PlanDev& p, bool write_R, float* dose_out /*[N][K] or null*/,
                     bool dvh_mode, const float* dvh_thr /*[S] device*/, const int* gate, cudaStream_t st);
int launch_simt_grad(const CaseDev& c, const PlanDev& p, const int* gate, cudaStream_t st);
int launch_round_begin(int* zero_ctr, const int* gate, int* log_slot, int* round_ctr, cudaStream_t st);
int launch_loop_cond(cudaGraphConditionalHandle cond, const PlanDev& p, int max_rounds, cudaStream_t st);
int launch_step_parity(const CaseDev& c, const PlanDev& p, const StepParams& sp, int parity, float g_scale,
                       cudaStream_t st);
int launch_eval_finish_scaled(const CaseDev& c, const PlanDev& p, const StepParams& sp, float g_scale, float* F_out,
                              float* grad_out, cudaStream_t st);
int launch_result(const CaseDev& c, const PlanDev& p, const StructHost* sh, float* T_out, float* F_out,
                  float* dvh_out, float* terms_out, int* iters_out, int* status_out, cudaStream_t st);
int launch_prepare_final(const CaseDev& c, const PlanDev& p, cudaStream_t st);
// polynomial line search (kernels_ls.cu): dose columns of the queued plans, then the choice of their next trial step
int launch_ls(const CaseDev& c, const PlanDev& p, int max_trials, float c1, float eps_f, bool use_slot, cudaStream_t st);

// gSA (kernels_sa.cu): one CTA of kSaThreads per chain, draws staged kSaBlock steps at a time
constexpr int kSaThreads = 512;
constexpr int kSaBlock = 128;
struct SaArgs {
  const float* Dt; long long ldt;             // transposed dose-rate matrix [A][ldt], ldt = N_alloc
  const float *pt_lo, *pt_hi; const int* tile_struct;
  int N_pad, A, A_pad, S;
  double wscale[2 * GMCO_MAX_STRUCTS];        // base weight / n_points per (structure, side), fp64
  const float* T0; int t0_bcast; const float* w_user;
  long long steps; const int* jdx; const double *z, *u; int draws_bcast;
  double tau, temp0, log_cooling;
  double *T_out, *F_out, *F_tracked; long long* n_accepted; int* bad_input;
};
int launch_sa_transpose(const CaseDev& c, float* Dt, cudaStream_t st);
size_t sa_smem_bytes(const CaseDev& c, int precision, int ppt);
int sa_points_per_thread(const CaseDev& c);
int launch_sa_chains(const CaseDev& c, const SaArgs& a, int K, int precision, cudaStream_t st);

// dose-rate matrix (kernels_doserate.cu)
struct DoseRateArgs { double coef[GMCO_MAX_RADIAL_COEF]; int n_coef; double sk_lambda, r_floor_cm; };
int launch_dose_rate(const float* pts, long long N, const float* dwell, int A, const DoseRateArgs& m, float* D,
                     long long ldD, cudaStream_t st);

// plan-pool post-processing (kernels_pool.cu)
struct SelectArgs {
  int n;
  int structure[GMCO_MAX_CRITERIA], sense[GMCO_MAX_CRITERIA], role[GMCO_MAX_CRITERIA];
  float limit_rtog[GMCO_MAX_CRITERIA], limit_plus[GMCO_MAX_CRITERIA];
};
int launch_pareto(const float* obj, int K, int M, unsigned char* nondom, int* count, cudaStream_t st);
int launch_select(const float* dvh, int K, int S, const SelectArgs& c, int* plan_class, int* out, cudaStream_t st);

// tensor path (kernels_tc.cu)
struct TcPlan;                                   // host-side schedule + tensor maps
TcPlan* tc_plan_create(const CaseDev& c, const PlanDev& p, const StructHost* sh, int num_sms, int force_single,
                       int wide_accum, int want_grad_pair, cudaStream_t st, char* err, int errlen);
void tc_plan_destroy(TcPlan*);
int tc_num_segments(const TcPlan*);
int tc_dose_pair(const TcPlan*);           // 1: the dose kernel runs as CTA pairs (its compaction split is per tile PAIR)
int tc_grad_pair(const TcPlan*);           // 1: the gradient kernel runs as CTA pairs as well
int tc_dose_kernel(const TcPlan*);         // tcl::DoseKernelId of the dose kernel that is dispatched
int tc_choose_segs(int n_tiles, int n_pad_points, int num_sms);
const int* tc_tile_seg_dev(const TcPlan*);
int tc_compact_cap(const TcPlan*);
// which < 0: both contractions; 0: the dose kernel only; 1: the gradient kernel only
int launch_tc_eval(const TcPlan* tp, const CaseDev& c, const PlanDev& p, float* dose_dbg, const int* gate,
                   int* zero_ctr, int* log_slot, bool compact, int which, cudaStream_t st);

}  // namespace gmco
