// gmco_api.cu -- the C ABI of include/gmco.h: argument checks, device layout, round driver.
// Host logic only; every arithmetic step of the path runs in the kernels.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <string>
#include <vector>

#include "gmco_internal.cuh"
#include "tc_layout.h"

using namespace gmco;

namespace {

thread_local char g_create_error[512] = "";

struct Arena {              // one stream-ordered allocation, carved into 256 B aligned pieces
  char* base = nullptr; size_t size = 0, used = 0; cudaStream_t st = nullptr;
  template <class T> T* take(size_t n) {
    const size_t bytes = (n * sizeof(T) + 255) & ~size_t(255);
    T* p = reinterpret_cast<T*>(base ? base + used : nullptr);
    used += bytes;
    return p;
  }
};

enum HandleState { ST_CREATED = 0, ST_OPTIMIZED = 1, ST_RESULT = 2, ST_EVALUATED = 3 };

}  // namespace

struct gmco_handle {
  gmco_options opt{};
  CaseDev c{};
  PlanDev p{};
  std::vector<StructHost> sh;
  std::vector<gmco_structure> structs;
  Arena case_arena, plan_arena;
  int plan_capacity_K = -1;
  float* struct_scale = nullptr;     // [2S] device: base weight / n_points
  float* dvh_thr = nullptr;          // [S] device
  // staging
  float* stage_D = nullptr;
  float *in_T0 = nullptr, *in_w = nullptr;
  float *out_T = nullptr, *out_F = nullptr, *out_dvh = nullptr, *out_terms = nullptr;
  int *out_iters = nullptr, *out_status = nullptr;
  int host_flags[4] = {0, 0, 0, 0};  // pageable: the copies into it are followed by a stream synchronise
  int host_err[4] = {0, 0, 0, 0};    // copy of the device error word
  TcPlan* tc = nullptr;
  float* sa_Dt = nullptr;            // gSA: transposed copy of D [A][N_alloc], built by the first gmco_sa_run
  // device-driven round loop: a CUDA graph whose only node is a WHILE conditional; its body is two rounds
  // (parity 0, parity 1) and a kernel that keeps the loop going while a plan is still running
  cudaGraph_t loop_graph = nullptr;
  cudaGraphExec_t loop_exec = nullptr;
  cudaStream_t cap_stream = nullptr;  // capture only (the caller's stream may be the legacy stream, which cannot capture)
  int loop_K = -1, loop_iters = -1, loop_launches_per_pair = 0;
  bool used_graph = false;
  cudaStream_t stream = nullptr;
  int device = 0, num_sms = 0;
  HandleState state = ST_CREATED;
  int iters = 0, rounds_enqueued = 0, rounds_with_work = 0, launches = 0;
  gmco_stats stats{};
  bool have_stats = false;
  bool profile = false;              // gmco_set_profiling
  std::vector<cudaEvent_t> ev;       // 4 per profiled round: | dose | gradient | step |
  int ev_used = 0;
  char err[512] = "";
};

namespace {

int fail(gmco_handle* h, int code, const char* fmt, const char* a = "") {
  char* dst = h ? h->err : g_create_error;
  snprintf(dst, 512, fmt, a);
  return code;
}

#define CK(h, call)                                                              \
  do {                                                                           \
    cudaError_t e_ = (call);                                                     \
    if (e_ != cudaSuccess) {                                                     \
      const int code_ = e_ == cudaErrorMemoryAllocation ? GMCO_E_NOMEM : GMCO_E_CUDA; \
      return fail(h, code_, #call ": %s", cudaGetErrorString(e_));               \
    }                                                                            \
  } while (0)

#define LN(h, expr)                                                              \
  do {                                                                           \
    int n_ = (expr);                                                             \
    if (n_ < 0) return fail(h, GMCO_E_CUDA, #expr ": %s", cudaGetErrorString(cudaGetLastError())); \
    (h)->launches += n_;                                                         \
  } while (0)

// the device error word (gmco_internal.cuh DevErr) as a GMCO_E_CUDA message; GMCO_OK when it is clear
int check_dev_err(gmco_handle* h, const int* e) {
  if (e[0] == DEVERR_NONE) return GMCO_OK;
  static const char* const kern[] = {"?", "k_dose_tc<resident>", "k_dose_tc<streamed>", "k_dose_tc_pair", "k_grad_tc", "k_step", "k_grad_tc_pair"};
  static const char* const wait[] = {"-", "ring slot free", "ring slot filled", "T group ready", "T tile landed", "accumulator full",
                                     "accumulator free", "R tile split", "history copies"};
  static const char* const what[] = {"?", "a barrier wait did not complete", "the shared-memory carve-up does not fit the launch",
                                     "the TMEM columns do not fit"};
  const int k = (e[1] >> 8) & 0xff, wsite = e[1] & 0xff;
  snprintf(h->err, sizeof(h->err), "device error word: %s in %s (wait: %s), block (%d, %d), detail %d; results are invalid",
           what[e[0] >= 1 && e[0] <= 3 ? e[0] : 0], kern[k >= 1 && k <= 6 ? k : 0], wait[wsite >= 1 && wsite <= 8 ? wsite : 0],
           e[2] & 0xffff, (e[2] >> 16) & 0xffff, e[3]);
  return GMCO_E_CUDA;
}

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at{};
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int round_up(long long v, int a) { return (int)(((v + a - 1) / a) * a); }

int arena_alloc(gmco_handle* h, Arena& a, cudaStream_t st) {
  a.size = a.used ? a.used : 256;
  a.used = 0;
  a.st = st;
  cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&a.base), a.size, st);
  if (e != cudaSuccess) { a.base = nullptr; return fail(h, GMCO_E_NOMEM, "cudaMallocAsync: %s", cudaGetErrorString(e)); }
  return GMCO_OK;
}

void arena_free(Arena& a, cudaStream_t st) {
  if (a.base) cudaFreeAsync(a.base, st);
  a = Arena{};
}

// carve (or, with base == nullptr, just measure) the case arena
void carve_case(gmco_handle* h, bool want_split, bool need_stage) {
  Arena& a = h->case_arena;
  CaseDev& c = h->c;
  const size_t nd = (size_t)c.N_alloc * c.A_pad;
  c.D = a.take<float>(nd);
  if (want_split) {
    c.D_hi = a.take<float>(nd); c.D_lo = a.take<float>(nd);
  }
  c.pt_lo = a.take<float>(c.N_alloc); c.pt_hi = a.take<float>(c.N_alloc);
  c.tile_struct = a.take<int>(c.N_alloc / 64); c.tile_valid = a.take<int>(c.N_alloc / 64);
  c.row_src = a.take<int>(c.N_alloc); c.sel_pos = a.take<int>(c.N_alloc);
  h->struct_scale = a.take<float>(2 * GMCO_MAX_STRUCTS);
  h->dvh_thr = a.take<float>(GMCO_MAX_STRUCTS);
  h->stage_D = need_stage ? a.take<float>((size_t)c.N * c.A) : nullptr;
}

void carve_plans(gmco_handle* h, int K, long long dose_stage_elems) {
  Arena& a = h->plan_arena;
  const CaseDev& c = h->c;
  PlanDev& p = h->p;
  p.K = K; p.K_pad = round_up(K, kPlanTile); p.m = h->opt.m;
  const size_t ka = (size_t)p.K_pad * c.A_pad, kp = (size_t)p.K_pad;
  p.x = a.take<float>(ka); p.g = a.take<float>(ka); p.p = a.take<float>(ka); p.xt = a.take<float>(ka);
  p.T = a.take<float>(ka);
  // tf32 lo part of T: read (by TMA) only by the streamed dose layout, i.e. above 256 dwell positions on the tensor route
  p.T_lo = (h->opt.precision == GMCO_PREC_TF32X3 && c.A_pad > 32 * tcl::kTmemGroups) ? a.take<float>(ka) : nullptr;
  p.Sh = a.take<float>(ka * p.m); p.Yh = a.take<float>(ka * p.m);
  p.rho = a.take<float>(kp * p.m); p.gam = a.take<float>(kp * p.m);
  p.Weff = a.take<float>(kp * 2 * c.S); p.WeffC = a.take<float>(kp * 2 * c.S); p.slot = a.take<int>(kp);
  p.F = a.take<float>(kp); p.gp = a.take<float>(kp); p.alpha = a.take<float>(kp);
  p.it_done = a.take<int>(kp); p.trials = a.take<int>(kp); p.hcount = a.take<int>(kp); p.hhead = a.take<int>(kp);
  p.status = a.take<int>(kp);
  p.n_running = a.take<int>(2); p.bad_input = a.take<int>(1); p.rounds_done = a.take<int>(2); p.dev_err = a.take<int>(4);
  p.round_log = a.take<int>(kRoundLogCap);
  if (h->opt.line_search == 1) {
    p.ls_list = a.take<int>(kLsCap); p.ls_count = a.take<int>(2); p.ls_cols = a.take<float>((size_t)3 * kLsCap * c.N_alloc);
  } else {
    p.ls_list = nullptr; p.ls_count = nullptr; p.ls_cols = nullptr;
  }
  p.tile_seg = a.take<int>(p.K_pad / kPlanTile + 1);
  // partials: the SIMT dose pass (also the final pass of gmco_result) needs [tiles][K_pad][2]
  const size_t f_simt = (size_t)(c.N_alloc / 64) * kp * 2;
  p.nFcomp = 2; p.nF = c.N_alloc / 64;
  const bool simt = h->opt.precision == GMCO_PREC_SIMT_FP32;
  size_t f_elems = f_simt, g_elems = 0;
  if (simt) {
    // split count depends on the point count only, so a plan's summation order does not depend on K
    int ns = c.N_alloc / 256;
    if (ns < 1) ns = 1;
    if (ns > 32) ns = 32;
    p.nG = ns;
    g_elems = (size_t)ns * ka;
    p.R = a.take<float>(kp * c.N_alloc);
  } else {
    // one partial slot per CTA of the tensor kernels' grid (plan tiles x point segments)
    const int n_tiles = p.K_pad / kPlanTile;
    const size_t nseg = n_tiles > 0 ? (size_t)n_tiles * tc_choose_segs(n_tiles, c.N_pad, h->num_sms) : 1;
    g_elems = nseg * kPlanTile * c.A_pad;
    if (nseg * kPlanTile * 2 > f_elems) f_elems = nseg * kPlanTile * 2;
    p.nG = 0;
    p.R = a.take<float>(kp * c.N_alloc);             // [N_alloc][K_pad] on this route
  }
  p.Fpart = a.take<float>(f_elems); p.Gpart = a.take<float>(g_elems);
  p.res_terms = a.take<float>(kp * 2 * c.S); p.res_cnt = a.take<int>(kp * c.S);
  p.res_sel = a.take<float>(kp * (size_t)(c.n_sel > 0 ? c.n_sel : 1)); p.res_dvh = a.take<float>(kp * c.S);
  h->in_T0 = a.take<float>((size_t)(K > 0 ? K : 1) * c.A); h->in_w = a.take<float>((size_t)(K > 0 ? K : 1) * 2 * c.S);
  h->out_T = a.take<float>((size_t)(K > 0 ? K : 1) * c.A); h->out_F = a.take<float>(kp + 1);
  h->out_dvh = a.take<float>(kp * c.S + 1); h->out_terms = a.take<float>(kp * 2 * c.S + 1);
  h->out_iters = a.take<int>(kp + 1); h->out_status = a.take<int>(kp + 1);
  (void)dose_stage_elems;
}

void destroy_loop_graph(gmco_handle* h);

int ensure_plans(gmco_handle* h, int K, cudaStream_t st) {
  if (h->plan_capacity_K == K && h->plan_arena.base && h->stream == st) {
    return GMCO_OK;
  }
  if (h->tc) { tc_plan_destroy(h->tc); h->tc = nullptr; }
  destroy_loop_graph(h);
  arena_free(h->plan_arena, h->stream);
  carve_plans(h, K, 0);                       // measuring pass
  int rc = arena_alloc(h, h->plan_arena, st);
  if (rc) return rc;
  carve_plans(h, K, 0);
  h->plan_capacity_K = K;
  if (h->opt.precision == GMCO_PREC_TF32X3 && K > 0) {
    h->tc = tc_plan_create(h->c, h->p, h->sh.data(), h->num_sms, h->opt.dose_kernel == 1, h->opt.wide_accum == 1, h->opt.dose_kernel == 2, st, h->err,
                           sizeof(h->err));
    if (!h->tc) return GMCO_E_UNSUPPORTED;
  }
  return GMCO_OK;
}

StepParams make_step_params(const gmco_handle* h, int iters) {
  StepParams sp{};
  const PlanDev& p = h->p; const CaseDev& c = h->c;
  sp.K = p.K; sp.A_pad = c.A_pad; sp.m = p.m; sp.iters = iters; sp.max_trials = h->opt.max_trials;
  sp.c1 = h->opt.c1; sp.eps = h->opt.eps; sp.eps_f = h->opt.eps_f;
  sp.Fpart = p.Fpart; sp.Gpart = p.Gpart;
  if (h->opt.precision == GMCO_PREC_SIMT_FP32) {
    sp.nF = p.nF; sp.nFcomp = 2; sp.f_slot_stride = (long long)p.K_pad * 2;
    sp.nG = p.nG; sp.g_slot_stride = (long long)p.K_pad * c.A_pad;
    sp.tile_local = 0; sp.tile_seg = nullptr;
  } else {
    sp.nF = 0; sp.nFcomp = 2; sp.f_slot_stride = 2 * kPlanTile;
    sp.nG = 0; sp.g_slot_stride = (long long)kPlanTile * c.A_pad;
    sp.tile_local = 1; sp.tile_seg = tc_tile_seg_dev(h->tc);
    if (h->opt.compaction) { sp.compact_cap = tc_compact_cap(h->tc); sp.total_ctas = tc_num_segments(h->tc); }
    sp.dose_pair = tc_dose_pair(h->tc); sp.grad_pair = tc_grad_pair(h->tc);
  }
  sp.S = c.S;
  sp.ls_cap = h->opt.line_search == 1 ? kLsCap : 0;
  return sp;
}

// SIMT kernels emit r = 2 w (d - D_lim) / n, the tensor kernel emits r / 2 (one multiply less per element)
float g_scale_of(const gmco_handle* h) { return h->opt.precision == GMCO_PREC_SIMT_FP32 ? 2.f : 4.f; }

// zero_ctr / log_slot: start-of-round bookkeeping (reset the other parity's running-plan counter, log this round's,
// count the round if a plan is running).  The tensor route does it in its first kernel; the SIMT route launches
// k_round_begin.  mid: event recorded between the dose kernel and the gradient kernel (profiling), or null.
int enqueue_eval(gmco_handle* h, float* dose_dbg, const int* gate, int* zero_ctr, int* log_slot, cudaEvent_t mid,
                 cudaStream_t st) {
  if (h->opt.precision == GMCO_PREC_SIMT_FP32) {
    if (zero_ctr) LN(h, launch_round_begin(zero_ctr, gate, log_slot, h->p.rounds_done + 1, st));
    LN(h, launch_simt_eval(h->c, h->p, true, dose_dbg, false, nullptr, gate, st));
    if (mid) CK(h, cudaEventRecord(mid, st));
    LN(h, launch_simt_grad(h->c, h->p, gate, st));
  } else if (!mid) {
    LN(h, launch_tc_eval(h->tc, h->c, h->p, dose_dbg, gate, zero_ctr, log_slot, gate && h->opt.compaction, -1, st));
  } else {
    LN(h, launch_tc_eval(h->tc, h->c, h->p, dose_dbg, gate, zero_ctr, log_slot, gate && h->opt.compaction, 0, st));
    CK(h, cudaEventRecord(mid, st));
    LN(h, launch_tc_eval(h->tc, h->c, h->p, dose_dbg, gate, zero_ctr, log_slot, gate && h->opt.compaction, 1, st));
  }
  return GMCO_OK;
}

// one round: every running plan has its trial point evaluated, then accepted or its step halved
int enqueue_round(gmco_handle* h, int parity, int log_idx, bool prof, const StepParams& sp, cudaStream_t st) {
  if (prof) {
    while ((int)h->ev.size() < h->ev_used + 4) {
      cudaEvent_t e;
      CK(h, cudaEventCreate(&e));
      h->ev.push_back(e);
    }
    CK(h, cudaEventRecord(h->ev[h->ev_used], st));
  }
  int rc = enqueue_eval(h, nullptr, h->p.n_running + parity, h->p.n_running + (parity ^ 1),
                        log_idx < kRoundLogCap ? h->p.round_log + log_idx : nullptr, prof ? h->ev[h->ev_used + 1] : nullptr, st);
  if (rc) return rc;
  if (prof) CK(h, cudaEventRecord(h->ev[h->ev_used + 2], st));
  LN(h, launch_step_parity(h->c, h->p, sp, parity, g_scale_of(h), st));
  if (sp.ls_cap) LN(h, launch_ls(h->c, h->p, sp.max_trials, sp.c1, sp.eps_f, sp.compact_cap > 0, st));
  if (prof) { CK(h, cudaEventRecord(h->ev[h->ev_used + 3], st)); h->ev_used += 4; }
  return GMCO_OK;
}

// host-driven rounds (profiling mode: per-round events need one launch per round)
int enqueue_rounds(gmco_handle* h, int n, cudaStream_t st) {
  const StepParams sp = make_step_params(h, h->iters);
  for (int i = 0; i < n; ++i) {
    const bool prof = h->profile && h->rounds_enqueued < kRoundLogCap;
    int rc = enqueue_round(h, h->rounds_enqueued & 1, h->rounds_enqueued, prof, sp, st);
    if (rc) return rc;
    h->rounds_enqueued++;
  }
  return GMCO_OK;
}

void destroy_loop_graph(gmco_handle* h) {
  if (h->loop_exec) cudaGraphExecDestroy(h->loop_exec);
  if (h->loop_graph) cudaGraphDestroy(h->loop_graph);
  h->loop_exec = nullptr; h->loop_graph = nullptr; h->loop_K = -1; h->loop_iters = -1;
}

long long max_rounds_of(const gmco_handle* h) { return 1 + (long long)h->iters * ((long long)h->opt.max_trials + 1); }

// device-driven rounds: WHILE(conditional) { round(parity 0); round(parity 1); keep going while n_running[0] > 0 }
int build_loop_graph(gmco_handle* h) {
  if (h->loop_exec && h->loop_K == h->p.K && h->loop_iters == h->iters) return GMCO_OK;
  destroy_loop_graph(h);
  if (!h->cap_stream) CK(h, cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
  CK(h, cudaGraphCreate(&h->loop_graph, 0));
  cudaGraphConditionalHandle cond;
  CK(h, cudaGraphConditionalHandleCreate(&cond, h->loop_graph, 1, cudaGraphCondAssignDefault));
  cudaGraphNodeParams np{};
  np.type = cudaGraphNodeTypeConditional;
  np.conditional.handle = cond; np.conditional.type = cudaGraphCondTypeWhile; np.conditional.size = 1;
  cudaGraphNode_t node;
  CK(h, cudaGraphAddNode(&node, h->loop_graph, nullptr, 0, &np));
  cudaGraph_t body = np.conditional.phGraph_out[0];
  CK(h, cudaStreamBeginCaptureToGraph(h->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
  const StepParams sp = make_step_params(h, h->iters);
  const int before = h->launches;
  const long long mr = max_rounds_of(h);
  int rc = enqueue_round(h, 0, kRoundLogCap, false, sp, h->cap_stream);
  if (!rc) rc = enqueue_round(h, 1, kRoundLogCap, false, sp, h->cap_stream);
  if (!rc && launch_loop_cond(cond, h->p, (int)(mr > 0x7fffffff ? 0x7fffffff : mr), h->cap_stream) < 0)
    rc = fail(h, GMCO_E_CUDA, "loop condition kernel: %s", cudaGetErrorString(cudaGetLastError()));
  h->loop_launches_per_pair = h->launches - before + 1;
  h->launches = before;
  cudaError_t e = cudaStreamEndCapture(h->cap_stream, nullptr);
  if (rc) { destroy_loop_graph(h); return rc; }
  if (e != cudaSuccess) { destroy_loop_graph(h); return fail(h, GMCO_E_CUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e)); }
  e = cudaGraphInstantiate(&h->loop_exec, h->loop_graph, 0);
  if (e != cudaSuccess) { destroy_loop_graph(h); return fail(h, GMCO_E_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e)); }
  h->loop_K = h->p.K; h->loop_iters = h->iters;
  return GMCO_OK;
}

int copy_inputs(gmco_handle* h, const float* T0, int bcast, const float* w, int K, cudaStream_t st,
                const float** T0_dev, const float** w_dev) {
  const CaseDev& c = h->c;
  const size_t nT = (size_t)(bcast ? 1 : K) * c.A, nW = (size_t)K * 2 * c.S;
  if (is_device_ptr(T0)) *T0_dev = T0;
  else {
    for (size_t i = 0; i < nT; ++i)
      if (!(T0[i] >= 0.f) || isinf(T0[i])) return fail(h, GMCO_E_INVALID, "T0 holds a negative, NaN or infinite dwell time%s");
    CK(h, cudaMemcpyAsync(h->in_T0, T0, nT * sizeof(float), cudaMemcpyHostToDevice, st));
    *T0_dev = h->in_T0;
  }
  if (is_device_ptr(w)) *w_dev = w;
  else {
    for (size_t i = 0; i < nW; ++i)
      if (!(w[i] >= 0.f) || isinf(w[i])) return fail(h, GMCO_E_INVALID, "weights hold a negative, NaN or infinite value%s");
    CK(h, cudaMemcpyAsync(h->in_w, w, nW * sizeof(float), cudaMemcpyHostToDevice, st));
    *w_dev = h->in_w;
  }
  return GMCO_OK;
}

}  // namespace

namespace {
// stage a host array on the device (stream-ordered scratch), or pass a device pointer through
template <class T>
int stage_in(gmco_handle* h, const T* src, size_t n, T** scratch, const T** dev, cudaStream_t st) {
  *scratch = nullptr;
  if (is_device_ptr(src)) { *dev = src; return GMCO_OK; }
  CK(h, cudaMallocAsync(reinterpret_cast<void**>(scratch), n * sizeof(T), st));
  CK(h, cudaMemcpyAsync(*scratch, src, n * sizeof(T), cudaMemcpyHostToDevice, st));
  *dev = *scratch;
  return GMCO_OK;
}
}  // namespace

extern "C" {

int gmco_version(void) { return GMCO_VERSION; }

void gmco_default_options(gmco_options* o) {
  if (!o) return;
  memset(o, 0, sizeof(*o));
  o->m = 10; o->eps = 0.f; o->c1 = 1e-4f; o->max_trials = 20; o->precision = GMCO_PREC_TF32X3; o->eps_f = 1e-6f; o->compaction = 1;
  o->dose_kernel = 0; o->wide_accum = 0; o->line_search = 0;
}

const char* gmco_last_error(const gmco_handle* h) { return h ? h->err : g_create_error; }

int gmco_create(gmco_handle** out, const float* D, int64_t n_points, int64_t n_dwell, int64_t ldD,
                const gmco_structure* structs, int32_t n_structs, float rx_dose, const gmco_options* opt,
                void* cuda_stream) {
  if (!out) return fail(nullptr, GMCO_E_INVALID, "out is NULL%s");
  *out = nullptr;
  if (!D || !structs) return fail(nullptr, GMCO_E_INVALID, "D or structs is NULL%s");
  if (n_points <= 0 || n_dwell <= 0 || ldD < n_dwell || n_points > (1 << 28))
    return fail(nullptr, GMCO_E_INVALID, "bad n_points / n_dwell / ldD%s");
  if (n_structs < 1 || n_structs > GMCO_MAX_STRUCTS) return fail(nullptr, GMCO_E_INVALID, "n_structs outside 1..8%s");
  if (!(rx_dose > 0.f) || isinf(rx_dose)) return fail(nullptr, GMCO_E_INVALID, "rx_dose must be positive and finite%s");
  if (n_dwell > kMaxApad) return fail(nullptr, GMCO_E_UNSUPPORTED, "n_dwell above 480 is not supported%s");
  gmco_options o;
  gmco_default_options(&o);
  if (opt) o = *opt;
  if (o.m < 1 || o.m > GMCO_MAX_HISTORY || o.max_trials < 1 || !(o.c1 > 0.f) || !(o.c1 < 1.f) || !(o.eps >= 0.f) ||
      !(o.eps_f >= 0.f) || !(o.eps_f < 1.f) ||
      (o.precision != GMCO_PREC_TF32X3 && o.precision != GMCO_PREC_SIMT_FP32) || (o.compaction != 0 && o.compaction != 1) ||
      o.dose_kernel < 0 || o.dose_kernel > 2 || (o.wide_accum != 0 && o.wide_accum != 1) ||
      (o.line_search != 0 && o.line_search != 1))
    return fail(nullptr, GMCO_E_INVALID, "bad gmco_options%s");
  // the tensor layout holds T_hi (A_pad columns) plus an accumulator pair in 512 TMEM columns: wider cases take
  // the plain-fp32 kernels (the paper's largest N_act is 385)
  if (o.precision == GMCO_PREC_TF32X3 && round_up(n_dwell, 32) > kMaxApadTensor) o.precision = GMCO_PREC_SIMT_FP32;
  long long tot = 0;
  for (int s = 0; s < n_structs; ++s) {
    const gmco_structure& g = structs[s];
    if (g.n_points <= 0 || !(g.w_lo >= 0.f) || !(g.w_hi >= 0.f) || isinf(g.w_lo) || isinf(g.w_hi) || isnan(g.d_lo) ||
        isnan(g.d_hi) || g.dvh_kind < 0 || g.dvh_kind > 2 || (g.dvh_kind && !(g.dvh_level > 0.f)))
      return fail(nullptr, GMCO_E_INVALID, "bad gmco_structure entry%s");
    tot += g.n_points;
  }
  if (tot != n_points) return fail(nullptr, GMCO_E_INVALID, "structure sizes do not add up to n_points%s");

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(nullptr, GMCO_E_UNSUPPORTED, "no CUDA device: %s", cudaGetErrorString(e));
  // cudaDeviceGetAttribute, not cudaGetDeviceProperties: the latter takes about a millisecond per call
  int cc_major = 0, n_sms = 0;
  e = cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return fail(nullptr, GMCO_E_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
  if (cc_major != 10) return fail(nullptr, GMCO_E_UNSUPPORTED, "libgmco needs an sm_100 device (B200)%s");

  gmco_handle* h = new (std::nothrow) gmco_handle();
  if (!h) return fail(nullptr, GMCO_E_NOMEM, "host allocation failed%s");
  h->opt = o; h->device = dev; h->num_sms = n_sms;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  h->structs.assign(structs, structs + n_structs);
  cudaStream_t st = h->stream;

  // keep freed blocks in the pool so that create/destroy cycles do not hit the OS allocator
  cudaMemPool_t pool;
  if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
    uint64_t thr = UINT64_MAX;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
  }

  // ---- row layout: every structure padded to a multiple of 64 rows ----
  CaseDev& c = h->c;
  c.N = (int)n_points; c.A = (int)n_dwell; c.S = n_structs; c.rx = rx_dose;
  c.A_pad = round_up(n_dwell, 32);
  int row = 0, src = 0, sel = 0;
  h->sh.resize(n_structs);
  for (int s = 0; s < n_structs; ++s) {
    StructHost& q = h->sh[s];
    q.n_points = structs[s].n_points; q.row_begin = row; q.n_rows_pad = round_up(q.n_points, kStructAlign);
    q.d_lo = structs[s].d_lo; q.d_hi = structs[s].d_hi; q.w_lo = structs[s].w_lo; q.w_hi = structs[s].w_hi;
    q.dvh_kind = structs[s].dvh_kind; q.dvh_level = structs[s].dvh_level;
    q.sel_begin = q.dvh_kind == 2 ? sel : -1;
    if (q.dvh_kind == 2) sel += q.n_points;
    row += q.n_rows_pad; src += q.n_points;
  }
  c.N_pad = row; c.N_alloc = round_up(row, kRowAlloc); c.n_sel = sel;

  const bool want_split = o.precision == GMCO_PREC_TF32X3;
  const bool dev_D = is_device_ptr(D);
  carve_case(h, want_split, !dev_D);
  int rc = arena_alloc(h, h->case_arena, st);
  if (rc) { snprintf(g_create_error, 512, "%s", h->err); delete h; return rc; }
  carve_case(h, want_split, !dev_D);

#define CKC(call)                                                                                   \
  do {                                                                                              \
    cudaError_t e2_ = (call);                                                                       \
    if (e2_ != cudaSuccess) {                                                                       \
      fail(nullptr, GMCO_E_CUDA, #call ": %s", cudaGetErrorString(e2_));                            \
      arena_free(h->case_arena, st); delete h; return GMCO_E_CUDA;                                  \
    }                                                                                               \
  } while (0)

  std::vector<float> pt_lo(c.N_alloc, -INFINITY), pt_hi(c.N_alloc, INFINITY), scale(2 * GMCO_MAX_STRUCTS, 0.f),
      thr(GMCO_MAX_STRUCTS, -1.f);
  std::vector<int> tile_struct(c.N_alloc / 64, 0), tile_valid(c.N_alloc / 64, 0), row_src(c.N_alloc, -1),
      sel_pos(c.N_alloc, -1);
  src = 0;
  for (int s = 0; s < n_structs; ++s) {
    const StructHost& q = h->sh[s];
    for (int i = 0; i < q.n_points; ++i) {
      pt_lo[q.row_begin + i] = q.d_lo; pt_hi[q.row_begin + i] = q.d_hi;
      row_src[q.row_begin + i] = src + i;
      if (q.dvh_kind == 2) sel_pos[q.row_begin + i] = q.sel_begin + i;
    }
    for (int t = q.row_begin / 64; t < (q.row_begin + q.n_rows_pad) / 64; ++t) {
      tile_struct[t] = s;
      const int left = q.n_points - (t * 64 - q.row_begin);
      tile_valid[t] = left >= 64 ? 64 : left;
    }
    scale[2 * s] = q.w_lo / (float)q.n_points; scale[2 * s + 1] = q.w_hi / (float)q.n_points;
    if (q.dvh_kind == 1) thr[s] = q.dvh_level / 100.f * rx_dose;
    src += q.n_points;
  }
  // tiles past N_pad keep structure 0 with infinite thresholds: zero contribution
  CKC(cudaMemcpyAsync(c.pt_lo, pt_lo.data(), c.N_alloc * sizeof(float), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(c.pt_hi, pt_hi.data(), c.N_alloc * sizeof(float), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(c.tile_struct, tile_struct.data(), tile_struct.size() * sizeof(int), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(c.tile_valid, tile_valid.data(), tile_valid.size() * sizeof(int), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(c.row_src, row_src.data(), c.N_alloc * sizeof(int), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(c.sel_pos, sel_pos.data(), c.N_alloc * sizeof(int), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(h->struct_scale, scale.data(), scale.size() * sizeof(float), cudaMemcpyHostToDevice, st));
  CKC(cudaMemcpyAsync(h->dvh_thr, thr.data(), thr.size() * sizeof(float), cudaMemcpyHostToDevice, st));
  const float* D_dev = D;
  long long ld = ldD;
  if (!dev_D) {
    CKC(cudaMemcpy2DAsync(h->stage_D, (size_t)c.A * sizeof(float), D, (size_t)ldD * sizeof(float),
                          (size_t)c.A * sizeof(float), (size_t)c.N, cudaMemcpyHostToDevice, st));
    D_dev = h->stage_D; ld = c.A;
  }
  // the host vectors above are pageable: the async copies have completed their staging on return
  CKC(cudaStreamSynchronize(st));
  if (launch_setup_case(c, D_dev, ld, c.row_src, want_split, st) < 0) {
    fail(nullptr, GMCO_E_CUDA, "case setup kernels: %s", cudaGetErrorString(cudaGetLastError()));
    arena_free(h->case_arena, st); delete h; return GMCO_E_CUDA;
  }
#undef CKC
  *out = h;
  return GMCO_OK;
}

int gmco_set_profiling(gmco_handle* h, int32_t enable) {
  if (!h) return GMCO_E_INVALID;
  h->profile = enable != 0;
  return GMCO_OK;
}

void gmco_destroy(gmco_handle* h) {
  if (!h) return;
  cudaStreamSynchronize(h->stream);
  for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
  if (h->tc) tc_plan_destroy(h->tc);
  destroy_loop_graph(h);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->sa_Dt) cudaFreeAsync(h->sa_Dt, h->stream);
  arena_free(h->plan_arena, h->stream);
  arena_free(h->case_arena, h->stream);
  delete h;
}

int gmco_optimize(gmco_handle* h, const float* T0, int32_t t0_broadcast, const float* weights, int32_t K,
                  int32_t iters, void* cuda_stream) {
  if (!h) return GMCO_E_INVALID;
  if (K < 0 || iters < 0) return fail(h, GMCO_E_INVALID, "K and iters must be >= 0%s");
  if (K > 0 && (!T0 || !weights)) return fail(h, GMCO_E_INVALID, "T0 or weights is NULL%s");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int rc = ensure_plans(h, K, st);
  if (rc) return rc;
  h->stream = st; h->iters = iters; h->rounds_enqueued = 0; h->launches = 0; h->have_stats = false;
  h->state = ST_CREATED; h->ev_used = 0;
  if (K == 0) { h->state = ST_OPTIMIZED; return GMCO_OK; }
  const float *T0d = nullptr, *wd = nullptr;
  rc = copy_inputs(h, T0, t0_broadcast, weights, K, st, &T0d, &wd);
  if (rc) return rc;
  LN(h, launch_init_plans(h->c, h->p, T0d, t0_broadcast ? 1 : 0, wd, h->struct_scale, st));
  // round 0 evaluates the start point; every further round is one trial step of every running plan.
  // Profiling mode drives the rounds from the host; backtracking plans need extra rounds, so it enqueues some
  // slack now (rounds with nothing running return at once) and gmco_result adds more if a plan is still running.
  h->used_graph = !h->profile;
  if (h->used_graph) {
    // the loop runs on the device until no plan is running: no slack rounds, no host polling
    rc = build_loop_graph(h);
    if (rc) return rc;
    CK(h, cudaGraphLaunch(h->loop_exec, st));
  } else {
    const int slack = iters > 0 ? (iters / 6 > 4 ? iters / 6 : 4) : 0;
    rc = enqueue_rounds(h, 1 + iters + slack, st);
    if (rc) return rc;
  }
  h->state = ST_OPTIMIZED;
  return GMCO_OK;
}

int gmco_result(gmco_handle* h, float* T, float* objective, float* dvh, float* objective_terms, int32_t* iters_done,
                int32_t* plan_status) {
  if (!h) return GMCO_E_INVALID;
  if (h->state != ST_OPTIMIZED && h->state != ST_RESULT) return fail(h, GMCO_E_STATE, "gmco_result needs a prior gmco_optimize%s");
  cudaStream_t st = h->stream;
  const PlanDev& p = h->p; const CaseDev& c = h->c;
  const int K = p.K;
  if (K == 0) {
    memset(&h->stats, 0, sizeof(h->stats));
    h->stats.device_bytes = (int64_t)(h->case_arena.size + h->plan_arena.size);
    h->stats.dose_kernel = -1;
    h->have_stats = true; h->state = ST_RESULT;
    return GMCO_OK;
  }
  if (h->state == ST_OPTIMIZED) {
    const long long max_rounds = max_rounds_of(h);
    int rounds_with_work = 0;
    for (;;) {
      const int parity = h->used_graph ? 0 : h->rounds_enqueued & 1;   // counter the NEXT round would read
      CK(h, cudaMemcpyAsync(h->host_flags, p.n_running + parity, sizeof(int), cudaMemcpyDeviceToHost, st));
      CK(h, cudaMemcpyAsync(h->host_flags + 1, p.bad_input, sizeof(int), cudaMemcpyDeviceToHost, st));
      CK(h, cudaMemcpyAsync(h->host_flags + 2, p.rounds_done, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
      CK(h, cudaMemcpyAsync(h->host_err, p.dev_err, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
      CK(h, cudaStreamSynchronize(st));
      // a failed optimisation leaves nothing to return: a second gmco_result is a state error, not the same failure again
      if (h->host_err[0]) { h->state = ST_CREATED; return check_dev_err(h, h->host_err); }
      if (h->host_flags[1]) { h->state = ST_CREATED; return fail(h, GMCO_E_INVALID, "T0 or weights hold a negative, NaN or infinite value%s"); }
      rounds_with_work = h->host_flags[3];
      if (h->used_graph) {
        h->rounds_enqueued = h->host_flags[2];
        h->launches += (h->host_flags[2] / 2) * h->loop_launches_per_pair;
        break;
      }
      if (h->host_flags[0] == 0 || h->rounds_enqueued >= max_rounds) break;
      int rc = enqueue_rounds(h, 8, st);
      if (rc) return rc;
    }
    h->rounds_with_work = rounds_with_work;
    // final dose pass at the accepted dwell times: objective terms, V_level counts, D_level doses
    LN(h, launch_prepare_final(c, p, st));
    LN(h, launch_simt_eval(c, p, false, nullptr, true, h->dvh_thr, nullptr, st));
    LN(h, launch_result(c, p, h->sh.data(), h->out_T, h->out_F, h->out_dvh, h->out_terms, h->out_iters,
                        h->out_status, st));
  }
  if (T) CK(h, cudaMemcpyAsync(T, h->out_T, (size_t)K * c.A * sizeof(float), cudaMemcpyDefault, st));
  if (objective) CK(h, cudaMemcpyAsync(objective, h->out_F, (size_t)K * sizeof(float), cudaMemcpyDefault, st));
  if (dvh) CK(h, cudaMemcpyAsync(dvh, h->out_dvh, (size_t)K * c.S * sizeof(float), cudaMemcpyDefault, st));
  if (objective_terms)
    CK(h, cudaMemcpyAsync(objective_terms, h->out_terms, (size_t)K * 2 * c.S * sizeof(float), cudaMemcpyDefault, st));
  if (iters_done) CK(h, cudaMemcpyAsync(iters_done, h->out_iters, (size_t)K * sizeof(int), cudaMemcpyDefault, st));
  if (plan_status) CK(h, cudaMemcpyAsync(plan_status, h->out_status, (size_t)K * sizeof(int), cudaMemcpyDefault, st));
  CK(h, cudaStreamSynchronize(st));
  if (h->state == ST_OPTIMIZED) {
    std::vector<int> stv(K);
    CK(h, cudaMemcpy(stv.data(), h->out_status, (size_t)K * sizeof(int), cudaMemcpyDeviceToHost));
    gmco_stats s{};
    s.device_bytes = (int64_t)(h->case_arena.size + h->plan_arena.size);
    s.rounds = h->rounds_with_work; s.kernel_launches = h->launches;
    s.dose_kernel = h->tc ? tc_dose_kernel(h->tc) : -1;
    for (int k = 0; k < K; ++k) {
      if (stv[k] == GMCO_PLAN_ITERS) s.plans_iters++;
      else if (stv[k] == GMCO_PLAN_CONVERGED) s.plans_converged++;
      else s.plans_stalled++;
    }
    if (h->profile && h->ev_used > 0) {
      const int nr = h->ev_used / 4;
      std::vector<int> log(nr);
      CK(h, cudaMemcpy(log.data(), p.round_log, (size_t)nr * sizeof(int), cudaMemcpyDeviceToHost));
      double ms_dose = 0.0, ms_grad = 0.0, ms_step = 0.0;
      for (int r = 0; r < nr; ++r) {
        if (log[r] <= 0) continue;                         // nothing was running: the launches returned at once
        float t = 0.f;
        CK(h, cudaEventElapsedTime(&t, h->ev[4 * r], h->ev[4 * r + 1])); ms_dose += t;
        CK(h, cudaEventElapsedTime(&t, h->ev[4 * r + 1], h->ev[4 * r + 2])); ms_grad += t;
        CK(h, cudaEventElapsedTime(&t, h->ev[4 * r + 2], h->ev[4 * r + 3])); ms_step += t;
        s.eval_launches++; s.eval_plans += log[r];
      }
      s.dose_ms = (float)ms_dose; s.grad_ms = (float)ms_grad; s.step_ms = (float)ms_step;
      s.eval_ms = (float)(ms_dose + ms_grad);
    }
    h->stats = s; h->have_stats = true;
  }
  h->state = ST_RESULT;
  return GMCO_OK;
}

int gmco_evaluate(gmco_handle* h, const float* T, int32_t t_broadcast, const float* weights, int32_t K, float* dose,
                  float* F, float* grad_x, void* cuda_stream) {
  if (!h) return GMCO_E_INVALID;
  if (K < 0) return fail(h, GMCO_E_INVALID, "K must be >= 0%s");
  if (K == 0) return GMCO_OK;
  if (!T || !weights) return fail(h, GMCO_E_INVALID, "T or weights is NULL%s");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int rc = ensure_plans(h, K, st);
  if (rc) return rc;
  h->stream = st; h->state = ST_EVALUATED; h->launches = 0;
  const CaseDev& c = h->c; const PlanDev& p = h->p;
  float* dose_dev = dose;
  const bool dose_host = dose && !is_device_ptr(dose);
  auto body = [&]() -> int {                             // one cleanup point for the scratch below
    const float *Td = nullptr, *wd = nullptr;
    int r = copy_inputs(h, T, t_broadcast, weights, K, st, &Td, &wd);
    if (r) return r;
    LN(h, launch_init_plans(c, p, Td, t_broadcast ? 1 : 0, wd, h->struct_scale, st));
    if (dose_host) CK(h, cudaMallocAsync(reinterpret_cast<void**>(&dose_dev), (size_t)c.N * K * sizeof(float), st));
    r = enqueue_eval(h, dose_dev, nullptr, nullptr, nullptr, nullptr, st);
    if (r) return r;
    StepParams sp = make_step_params(h, 0);
    sp.compact_cap = 0;                                    // one evaluation of every plan in place: no slots
    float* Fd = F ? h->out_F : nullptr;
    float* gd = grad_x ? h->out_T : nullptr;
    LN(h, launch_eval_finish_scaled(c, p, sp, g_scale_of(h), Fd, gd, st));
    if (F) CK(h, cudaMemcpyAsync(F, Fd, (size_t)K * sizeof(float), cudaMemcpyDefault, st));
    if (grad_x) CK(h, cudaMemcpyAsync(grad_x, gd, (size_t)K * c.A * sizeof(float), cudaMemcpyDefault, st));
    if (dose_host) CK(h, cudaMemcpyAsync(dose, dose_dev, (size_t)c.N * K * sizeof(float), cudaMemcpyDeviceToHost, st));
    CK(h, cudaMemcpyAsync(h->host_flags + 1, p.bad_input, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(h, cudaMemcpyAsync(h->host_err, p.dev_err, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
    return GMCO_OK;
  };
  rc = body();
  if (dose_host && dose_dev && dose_dev != dose) cudaFreeAsync(dose_dev, st);
  if (rc) return rc;
  CK(h, cudaStreamSynchronize(st));
  if (h->host_err[0]) return check_dev_err(h, h->host_err);
  if (h->host_flags[1]) return fail(h, GMCO_E_INVALID, "T or weights hold a negative, NaN or infinite value%s");
  return GMCO_OK;
}

int gmco_sa_run(gmco_handle* h, const float* T0, int32_t t0_broadcast, const float* weights, int32_t K, int64_t steps,
                const int32_t* jdx, const double* z, const double* u, int32_t draws_broadcast, double tau,
                double temp0, double cooling, int32_t precision, double* T, double* objective, int64_t* n_accepted,
                void* cuda_stream) {
  if (!h) return GMCO_E_INVALID;
  if (K < 0 || steps < 0) return fail(h, GMCO_E_INVALID, "K and steps must be >= 0%s");
  if (K == 0) return GMCO_OK;
  if (!T0 || !weights) return fail(h, GMCO_E_INVALID, "T0 or weights is NULL%s");
  if (steps > 0 && (!jdx || !z || !u)) return fail(h, GMCO_E_INVALID, "jdx, z or u is NULL%s");
  if (precision != GMCO_SA_FP64 && precision != GMCO_SA_FP32) return fail(h, GMCO_E_INVALID, "unknown gmco_sa_precision%s");
  if (!(tau >= 0.0) || !(temp0 >= 0.0) || !(cooling > 0.0) || isinf(tau) || isinf(temp0) || isinf(cooling))
    return fail(h, GMCO_E_INVALID, "tau, temp0 must be finite and >= 0, cooling finite and > 0%s");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const CaseDev& c = h->c;
  const int ppt = sa_points_per_thread(c);
  const size_t smem = sa_smem_bytes(c, precision, ppt);
  if (smem > 227 * 1024) return fail(h, GMCO_E_UNSUPPORTED, "gSA: the case has too many points for one CTA's shared memory%s");
  h->launches = 0;
  if (!h->sa_Dt) {
    CK(h, cudaMallocAsync(reinterpret_cast<void**>(&h->sa_Dt), (size_t)c.A * c.N_alloc * sizeof(float), st));
    LN(h, launch_sa_transpose(c, h->sa_Dt, st));
  }
  // one stream-ordered block for this call: staged host inputs and the outputs
  const size_t nd = (size_t)(draws_broadcast ? 1 : K) * (size_t)steps;
  const size_t nT0 = (size_t)(t0_broadcast ? 1 : K) * c.A, nw = (size_t)K * 2 * c.S;
  const bool T0_host = !is_device_ptr(T0), w_host = !is_device_ptr(weights);
  const bool j_host = steps > 0 && !is_device_ptr(jdx), z_host = steps > 0 && !is_device_ptr(z),
             u_host = steps > 0 && !is_device_ptr(u);
  Arena a;
  char* blk = nullptr;
  double *dT = nullptr, *dF = nullptr, *dFt = nullptr, *dz = nullptr, *du = nullptr;
  long long* dn = nullptr; int *dbad = nullptr, *dj = nullptr; float *dT0 = nullptr, *dw = nullptr;
  for (int pass = 0; pass < 2; ++pass) {
    a.base = blk; a.used = 0;
    dT = a.take<double>((size_t)K * c.A); dF = a.take<double>(K); dFt = a.take<double>(K);
    dn = a.take<long long>(K); dbad = a.take<int>(1);
    if (z_host) dz = a.take<double>(nd);
    if (u_host) du = a.take<double>(nd);
    if (j_host) dj = a.take<int>(nd);
    if (T0_host) dT0 = a.take<float>(nT0);
    if (w_host) dw = a.take<float>(nw);
    if (pass == 0) CK(h, cudaMallocAsync(reinterpret_cast<void**>(&blk), a.used, st));
  }
  int rc = GMCO_OK;
  auto body = [&]() -> int {
    CK(h, cudaMemsetAsync(dbad, 0, sizeof(int), st));
    if (z_host) CK(h, cudaMemcpyAsync(dz, z, nd * sizeof(double), cudaMemcpyHostToDevice, st));
    if (u_host) CK(h, cudaMemcpyAsync(du, u, nd * sizeof(double), cudaMemcpyHostToDevice, st));
    if (j_host) CK(h, cudaMemcpyAsync(dj, jdx, nd * sizeof(int), cudaMemcpyHostToDevice, st));
    if (T0_host) CK(h, cudaMemcpyAsync(dT0, T0, nT0 * sizeof(float), cudaMemcpyHostToDevice, st));
    if (w_host) CK(h, cudaMemcpyAsync(dw, weights, nw * sizeof(float), cudaMemcpyHostToDevice, st));
    SaArgs sa{};
    sa.Dt = h->sa_Dt; sa.ldt = c.N_alloc; sa.pt_lo = c.pt_lo; sa.pt_hi = c.pt_hi; sa.tile_struct = c.tile_struct;
    sa.N_pad = c.N_pad; sa.A = c.A; sa.A_pad = c.A_pad; sa.S = c.S;
    for (int s = 0; s < c.S; ++s) {
      sa.wscale[2 * s] = (double)h->sh[s].w_lo / (double)h->sh[s].n_points;
      sa.wscale[2 * s + 1] = (double)h->sh[s].w_hi / (double)h->sh[s].n_points;
    }
    sa.T0 = T0_host ? dT0 : T0; sa.t0_bcast = t0_broadcast ? 1 : 0; sa.w_user = w_host ? dw : weights;
    sa.steps = steps; sa.jdx = j_host ? dj : jdx; sa.z = z_host ? dz : z; sa.u = u_host ? du : u;
    sa.draws_bcast = draws_broadcast ? 1 : 0;
    sa.tau = tau; sa.temp0 = temp0; sa.log_cooling = log(cooling);
    sa.T_out = dT; sa.F_out = dF; sa.F_tracked = dFt; sa.n_accepted = dn; sa.bad_input = dbad;
    LN(h, launch_sa_chains(c, sa, K, precision, st));
    if (T) CK(h, cudaMemcpyAsync(T, dT, (size_t)K * c.A * sizeof(double), cudaMemcpyDefault, st));
    if (objective) CK(h, cudaMemcpyAsync(objective, dF, (size_t)K * sizeof(double), cudaMemcpyDefault, st));
    if (n_accepted) CK(h, cudaMemcpyAsync(n_accepted, dn, (size_t)K * sizeof(long long), cudaMemcpyDefault, st));
    CK(h, cudaMemcpyAsync(h->host_flags + 3, dbad, sizeof(int), cudaMemcpyDeviceToHost, st));
    return GMCO_OK;
  };
  rc = body();
  cudaFreeAsync(blk, st);
  if (rc) return rc;
  CK(h, cudaStreamSynchronize(st));
  if (h->host_flags[3] & 1) return fail(h, GMCO_E_INVALID, "T0 or weights hold a negative, NaN or infinite value%s");
  if (h->host_flags[3] & 2) return fail(h, GMCO_E_INVALID, "jdx holds an index outside [0, n_dwell)%s");
  return GMCO_OK;
}

int gmco_dose_rate_matrix(const float* points, int64_t n_points, const float* dwell, int64_t n_dwell,
                          const double* g_coef, int32_t n_coef, double sk_lambda, double r_floor_cm, float* D, int64_t ldD,
                          void* cuda_stream) {
  gmco_handle* h = nullptr;                           // errors go to the create-error slot
  if (n_points < 0 || n_dwell < 0 || n_dwell > (1 << 20) || ldD < n_dwell || n_coef < 1 || n_coef > GMCO_MAX_RADIAL_COEF ||
      !g_coef || !(sk_lambda >= 0.0) || !(r_floor_cm > 0.0) || isinf(sk_lambda) || isinf(r_floor_cm))
    return fail(h, GMCO_E_INVALID, "bad sizes, ldD < n_dwell, n_coef outside 1..GMCO_MAX_RADIAL_COEF, or r_floor_cm <= 0%s");
  if (n_points == 0 || n_dwell == 0) return GMCO_OK;
  if (!points || !dwell || !D) return fail(h, GMCO_E_INVALID, "points, dwell or D is NULL%s");
  DoseRateArgs m{};
  for (int c = 0; c < n_coef; ++c) { if (isnan(g_coef[c]) || isinf(g_coef[c])) return fail(h, GMCO_E_INVALID, "g_coef not finite%s"); m.coef[c] = g_coef[c]; }
  m.n_coef = n_coef; m.sk_lambda = sk_lambda; m.r_floor_cm = r_floor_cm;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  float *sp = nullptr, *sq = nullptr, *dD = D;
  const float *dp = nullptr, *dq = nullptr;
  const bool D_host = !is_device_ptr(D);
  auto body = [&]() -> int {
    int rc = stage_in(h, points, (size_t)n_points * 3, &sp, &dp, st);
    if (!rc) rc = stage_in(h, dwell, (size_t)n_dwell * 3, &sq, &dq, st);
    if (rc) return rc;
    long long ld = ldD;
    if (D_host) { CK(h, cudaMallocAsync(reinterpret_cast<void**>(&dD), (size_t)n_points * n_dwell * sizeof(float), st)); ld = n_dwell; }
    if (launch_dose_rate(dp, n_points, dq, (int)n_dwell, m, dD, ld, st) < 0)
      return fail(h, GMCO_E_CUDA, "k_dose_rate: %s", cudaGetErrorString(cudaGetLastError()));
    if (D_host)
      CK(h, cudaMemcpy2DAsync(D, (size_t)ldD * sizeof(float), dD, (size_t)n_dwell * sizeof(float),
                              (size_t)n_dwell * sizeof(float), (size_t)n_points, cudaMemcpyDeviceToHost, st));
    return GMCO_OK;
  };
  const int rc = body();
  if (sp) cudaFreeAsync(sp, st);
  if (sq) cudaFreeAsync(sq, st);
  if (D_host && dD != D && dD) cudaFreeAsync(dD, st);
  if (rc) return rc;
  if (D_host || sp || sq) CK(h, cudaStreamSynchronize(st));
  return GMCO_OK;
}

int gmco_select_plan(gmco_handle* h, const float* dvh, int32_t K, const gmco_criterion* criteria, int32_t n_criteria,
                     int32_t* plan_class, int32_t* selected, int32_t* class_counts, void* cuda_stream) {
  if (!h) return GMCO_E_INVALID;
  if (K < 0 || n_criteria < 1 || n_criteria > GMCO_MAX_CRITERIA || !criteria)
    return fail(h, GMCO_E_INVALID, "K < 0, or n_criteria outside 1..GMCO_MAX_CRITERIA, or criteria is NULL%s");
  SelectArgs sa{};
  sa.n = n_criteria;
  int n_target = 0;
  for (int i = 0; i < n_criteria; ++i) {
    const gmco_criterion& q = criteria[i];
    if (q.structure < 0 || q.structure >= h->c.S || (q.sense != 1 && q.sense != -1) || q.role < 0 || q.role > 2 ||
        isnan(q.limit_rtog) || isnan(q.limit_rtog_plus))
      return fail(h, GMCO_E_INVALID, "criterion with a bad structure index, sense, role or limit%s");
    n_target += q.role == 0;
    sa.structure[i] = q.structure; sa.sense[i] = q.sense; sa.role[i] = q.role;
    sa.limit_rtog[i] = q.limit_rtog; sa.limit_plus[i] = q.limit_rtog_plus;
  }
  if (n_target != 1) return fail(h, GMCO_E_INVALID, "exactly one criterion must have role 0 (target)%s");
  int host_out[4] = {-1, 0, 0, 0};
  if (K > 0) {
    if (!dvh) return fail(h, GMCO_E_INVALID, "dvh is NULL%s");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    float* scr = nullptr; const float* ddvh = nullptr;
    int rc = stage_in(h, dvh, (size_t)K * h->c.S, &scr, &ddvh, st);
    if (rc) return rc;
    int* dout = nullptr;
    CK(h, cudaMallocAsync(reinterpret_cast<void**>(&dout), ((size_t)K + 4) * sizeof(int), st));
    h->launches = 0;
    LN(h, launch_select(ddvh, K, h->c.S, sa, plan_class ? dout + 4 : nullptr, dout, st));
    CK(h, cudaMemcpyAsync(host_out, dout, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
    if (plan_class) CK(h, cudaMemcpyAsync(plan_class, dout + 4, (size_t)K * sizeof(int), cudaMemcpyDefault, st));
    cudaFreeAsync(dout, st);
    if (scr) cudaFreeAsync(scr, st);
    CK(h, cudaStreamSynchronize(st));
  }
  if (selected) CK(h, cudaMemcpy(selected, host_out, sizeof(int), cudaMemcpyDefault));
  if (class_counts) CK(h, cudaMemcpy(class_counts, host_out + 1, 3 * sizeof(int), cudaMemcpyDefault));
  return GMCO_OK;
}

int gmco_pareto_front(gmco_handle* h, const float* objectives, int32_t K, int32_t M, uint8_t* nondominated,
                      int32_t* n_nondominated, void* cuda_stream) {
  if (!h) return GMCO_E_INVALID;
  if (K < 0 || M < 1 || M > GMCO_MAX_OBJECTIVES) return fail(h, GMCO_E_INVALID, "K < 0 or M outside 1..GMCO_MAX_OBJECTIVES%s");
  int host_n = 0;
  if (K > 0) {
    if (!objectives) return fail(h, GMCO_E_INVALID, "objectives is NULL%s");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    float* scr = nullptr; const float* dobj = nullptr;
    int rc = stage_in(h, objectives, (size_t)K * M, &scr, &dobj, st);
    if (rc) return rc;
    unsigned char* dmask = nullptr;
    CK(h, cudaMallocAsync(reinterpret_cast<void**>(&dmask), (size_t)K + 16, st));
    int* dcount = reinterpret_cast<int*>(dmask + (((size_t)K + 3) & ~size_t(3)));
    h->launches = 0;
    LN(h, launch_pareto(dobj, K, M, dmask, dcount, st));
    CK(h, cudaMemcpyAsync(&host_n, dcount, sizeof(int), cudaMemcpyDeviceToHost, st));
    if (nondominated) CK(h, cudaMemcpyAsync(nondominated, dmask, (size_t)K, cudaMemcpyDefault, st));
    cudaFreeAsync(dmask, st);
    if (scr) cudaFreeAsync(scr, st);
    CK(h, cudaStreamSynchronize(st));
  }
  if (n_nondominated) CK(h, cudaMemcpy(n_nondominated, &host_n, sizeof(int), cudaMemcpyDefault));
  return GMCO_OK;
}

int gmco_tc_schedule(int64_t n_dwell, const int32_t* struct_points, int32_t n_structs, int32_t K, int32_t num_sms,
                     int32_t dose_kernel, int32_t wide_accum, gmco_tc_info* out) {
  if (!out || !struct_points || n_dwell < 1 || n_structs < 1 || n_structs > GMCO_MAX_STRUCTS || K < 1 || num_sms < 1 ||
      dose_kernel < 0 || dose_kernel > 2 || (wide_accum != 0 && wide_accum != 1))
    return fail(nullptr, GMCO_E_INVALID, "gmco_tc_schedule: NULL or non-positive argument%s");
  memset(out, 0, sizeof(*out));
  long long n_pad = 0;
  for (int s = 0; s < n_structs; ++s) {
    if (struct_points[s] < 1) return fail(nullptr, GMCO_E_INVALID, "gmco_tc_schedule: structure without points%s");
    n_pad += round_up(struct_points[s], kStructAlign);
  }
  if (n_pad > (1 << 28)) return fail(nullptr, GMCO_E_INVALID, "gmco_tc_schedule: too many points%s");
  out->smem_limit = tcl::kSmemMax; out->tmem_limit = tcl::kTmemCols;
  out->a_pad = round_up(n_dwell, 32); out->n_pad = (int)n_pad; out->n_alloc = round_up(n_pad, kRowAlloc);
  out->k_pad = round_up(K, kPlanTile);
  if (out->a_pad > kMaxApadTensor) return GMCO_OK;   // ok = 0: the SIMT route takes the case
  const tcl::Schedule q = tcl::choose_schedule(out->a_pad, out->n_pad, out->k_pad, num_sms, dose_kernel == 1, wide_accum == 1, dose_kernel == 2);
  if (!q.ok) return GMCO_OK;
  out->ok = 1;
  out->n_tiles = q.n_tiles; out->segs = q.segs; out->n_chunks = q.n_chunks; out->n_slabs = q.n_slabs;
  out->compact_cap = q.segs > 36 ? q.segs : 36;
  out->dose_kernel = q.dose_kernel; out->dose_threads = 320; out->grad_threads = 192;
  if (q.dose_pair) {
    const tcl::PairSmem l = tcl::pair_smem(q.G, q.pair_stages);
    out->dose_stages = q.pair_stages; out->dose_stage_bytes = tcl::kPairEntry; out->dose_smem_bytes = q.pair_smem;
    out->dose_smem_end = l.end; out->dose_scr_slot = -1; out->dose_tmem_cols = tcl::pair_tmem_cols(q.G);
  } else {
    const tcl::DoseSmem l = tcl::dose_smem(q.tlo_resident != 0, q.G, q.dose_stages, q.dose_tmem_groups);
    out->dose_stages = q.dose_stages; out->dose_stage_bytes = l.stage_bytes; out->dose_smem_bytes = q.dose_smem;
    out->dose_smem_end = l.end; out->dose_scr_slot = q.tlo_resident ? -1 : l.scr_slot;
    out->dose_tmem_cols = tcl::dose_tmem_cols(q.G, q.dose_tmem_groups, q.dose_n_main);
  }
  out->dose_tmem_groups = q.dose_pair ? tcl::kTmemGroups : q.dose_tmem_groups; out->dose_n_main = q.dose_pair ? 1 : q.dose_n_main;
  const tcl::GradSmem gl = tcl::grad_smem(q.grad_ps, q.G, q.grad_stages);
  out->grad_ps = q.grad_ps; out->grad_stages = q.grad_stages; out->grad_stage_bytes = gl.stage_bytes;
  out->grad_smem_bytes = q.grad_smem; out->grad_smem_end = gl.end; out->grad_staging_bytes = gl.staging_bytes;
  out->grad_tmem_cols = tcl::grad_tmem_cols(out->a_pad);
  if (q.grad_pair) {                                 // the gradient kernel that would launch is k_grad_tc_pair
    const tcl::GradSmem gp = tcl::grad_pair_smem(q.grad_ps, q.G, q.gpair_stages);
    out->grad_stages = q.gpair_stages; out->grad_stage_bytes = gp.stage_bytes; out->grad_smem_bytes = q.gpair_smem;
    out->grad_smem_end = gp.end; out->grad_staging_bytes = gp.staging_bytes;
  }
  out->grad_pair = q.grad_pair;
  return GMCO_OK;
}

int gmco_get_stats(const gmco_handle* h, gmco_stats* out) {
  if (!h || !out) return GMCO_E_INVALID;
  if (!h->have_stats) return GMCO_E_STATE;
  *out = h->stats;
  return GMCO_OK;
}

}  // extern "C"
