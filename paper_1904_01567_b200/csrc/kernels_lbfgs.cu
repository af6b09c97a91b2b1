// kernels_lbfgs.cu -- per-plan state kernels: start point (a1), L-BFGS two-loop recursion (a6),
// Armijo accept / backtrack, history update and stop test (a7).  One warp per plan; a dwell
// vector of A_pad <= 480 floats lives in registers (A_pad / 32 per lane), dot products are
// butterfly reductions in a fixed order, so a plan's trajectory does not depend on K.
//
// Algorithm = DESIGN.md section 2.2 (reading A5 of the paper's "description omitted" L-BFGS,
// PAPER.md:115-119, after Liu & Nocedal 1989).  The batch advances in ROUNDS: in every round each
// running plan has exactly one trial point x + alpha p evaluated by the contraction kernels; this
// kernel then either accepts it (history push, new direction, alpha = 1) or halves alpha.
#include "gmco_internal.cuh"
#include "gmco_ptx.cuh"

namespace gmco {

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int off = 16; off; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

struct PlanPtrs {
  float *x, *g, *p, *xt, *T, *T_lo, *Sh, *Yh, *rho, *gam, *F, *gp, *alpha;
  int *it_done, *trials, *hcount, *hhead, *status, *n_running, *bad_input, *dev_err, *ls_list, *ls_count;
  int K_pad;
  float *Weff, *WeffC;        // [K_pad][2S] effective weights by plan / by slot
  int* slot;                  // [K_pad] row of plan k in T, R and the partials (= k without compaction)
};

static PlanPtrs make_ptrs(const PlanDev& p) {
  PlanPtrs q;
  q.x = p.x; q.g = p.g; q.p = p.p; q.xt = p.xt; q.T = p.T; q.T_lo = p.T_lo;
  q.Sh = p.Sh; q.Yh = p.Yh; q.rho = p.rho; q.gam = p.gam; q.F = p.F; q.gp = p.gp; q.alpha = p.alpha;
  q.it_done = p.it_done; q.trials = p.trials; q.hcount = p.hcount; q.hhead = p.hhead; q.status = p.status;
  q.n_running = p.n_running; q.bad_input = p.bad_input; q.dev_err = p.dev_err; q.K_pad = p.K_pad;
  q.ls_list = p.ls_list; q.ls_count = p.ls_count;
  q.Weff = p.Weff; q.WeffC = p.WeffC; q.slot = p.slot;
  return q;
}

// ---------------------------------------------------------------------------------------------
// a1: x = sqrt(T0), trial point = start point, effective weights, per-plan scalars.
__global__ void k_init_plans(PlanPtrs pp, int K, int A, int A_pad, int S, const float* __restrict__ T0, int bcast,
                             const float* __restrict__ w_user, const float* __restrict__ scale, float* __restrict__ Weff) {
  const int k = blockIdx.x;
  int bad = 0;
  for (int a = threadIdx.x; a < A_pad; a += blockDim.x) {
    float t0 = 0.f;
    if (k < K && a < A) {
      t0 = bcast ? T0[a] : T0[(long long)k * A + a];
      if (!(t0 >= 0.f) || isinf(t0)) { bad = 1; t0 = 0.f; }
    }
    const float x = sqrtf(t0), t = x * x;
    const long long i = (long long)k * A_pad + a;
    pp.x[i] = x; pp.xt[i] = x; pp.g[i] = 0.f; pp.p[i] = 0.f;
    pp.T[i] = t;
    if (pp.T_lo) pp.T_lo[i] = tf32_rn(t - tf32_rn(t));   // only the streamed dose layout (more than 256 dwell positions) reads it
  }
  for (int j = threadIdx.x; j < 2 * S; j += blockDim.x) {
    float w = 0.f;
    if (k < K) { w = w_user[(long long)k * 2 * S + j]; if (!(w >= 0.f) || isinf(w)) { bad = 1; w = 0.f; } }
    Weff[(long long)k * 2 * S + j] = w * scale[j];
    pp.WeffC[(long long)k * 2 * S + j] = w * scale[j];
  }
  if (bad) atomicExch(pp.bad_input, 1);
  if (threadIdx.x == 0) {
    pp.F[k] = 0.f; pp.gp[k] = 0.f; pp.alpha[k] = 1.f;
    pp.it_done[k] = 0; pp.trials[k] = -1;                 // -1: the start point itself is being evaluated
    pp.hcount[k] = 0; pp.hhead[k] = 0; pp.slot[k] = k;
    pp.status[k] = k < K ? PLAN_RUNNING : GMCO_PLAN_ITERS;
    if (k == 0) { pp.n_running[0] = K; pp.n_running[1] = 0; }
  }
}

int launch_init_plans(const CaseDev& c, const PlanDev& p, const float* T0, int t0_bcast, const float* w_user,
                      const float* struct_scale, cudaStream_t st) {
  if (p.K_pad == 0) return 0;
  cudaMemsetAsync(p.bad_input, 0, sizeof(int), st);
  cudaMemsetAsync(p.rounds_done, 0, 2 * sizeof(int), st);
  cudaMemsetAsync(p.dev_err, 0, 4 * sizeof(int), st);
  if (p.ls_count) cudaMemsetAsync(p.ls_count, 0, 2 * sizeof(int), st);
  k_init_plans<<<p.K_pad, 128, 0, st>>>(make_ptrs(p), p.K, c.A, c.A_pad, c.S, T0, t0_bcast, w_user, struct_scale,
                                        p.Weff);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
// Fixed-order reduction of the contraction kernels' partial results for plan k.
// The loads are what costs time (one L2/HBM round trip per dependent batch), so they are issued in as few batches as
// the registers allow -- the objective partials and up to 18 gradient slots (all of C3's) before the first add; the
// adds keep slot order, so the result does not depend on scheduling.
template <int NPL, int B>
__device__ __forceinline__ void add_slots(const float*& gp, int& s, int g1, long long stride, int npl, float (&G)[NPL]) {
  for (; s + B <= g1; s += B, gp += B * stride) {
    float v[B][NPL];
#pragma unroll
    for (int u = 0; u < B; ++u)
#pragma unroll
      for (int j = 0; j < NPL; ++j) v[u][j] = j < npl ? __ldcs(gp + u * stride + 32 * j) : 0.f;
#pragma unroll
    for (int u = 0; u < B; ++u)
#pragma unroll
      for (int j = 0; j < NPL; ++j) G[j] += v[u][j];
  }
}

template <int NPL>
__device__ __forceinline__ float reduce_partials(const StepParams& sp, int k, int lane, int npl, float (&G)[NPL],
                                                 int row = -1, int n_running = 0) {
  int f0 = 0, f1 = sp.nF, g0 = 0, g1 = sp.nG;
  long long prow = k;
  if (row >= 0) {                                          // compaction: the split the tensor kernels derived (compact_remap)
    const int ta = (n_running + 127) >> 7;
    int sa = sp.total_ctas / ta;
    if (sa > sp.compact_cap) sa = sp.compact_cap;
    g0 = (row >> 7) * sa; g1 = g0 + sa; prow = row & 127;
    if (sp.dose_pair) {                                    // compact_remap_pair: CTA pairs over tile pairs
      sa = (sp.total_ctas >> 1) / ((ta + 1) >> 1);
      if (sa > sp.compact_cap) sa = sp.compact_cap;
    }
    f0 = (row >> 7) * sa; f1 = f0 + sa;
    if (sp.grad_pair) { g0 = f0; g1 = f1; }                // k_grad_tc_pair deals its CTA pairs the same way
  } else if (sp.tile_local) { f0 = g0 = sp.tile_seg[k >> 7]; f1 = g1 = sp.tile_seg[(k >> 7) + 1]; prow = k & 127; }
  const int nfe = (f1 - f0) * sp.nFcomp;                   // SIMT: (lo, hi) pairs per slot
  auto f_at = [&](int i) {
    const int slot = f0 + i / sp.nFcomp, comp = i % sp.nFcomp;
    return sp.Fpart[(long long)slot * sp.f_slot_stride + prow * sp.nFcomp + comp];
  };
  // objective partials: the first two per lane are in flight together with the first gradient batch
  const float fa = lane < nfe ? f_at(lane) : 0.f, fb = lane + 32 < nfe ? f_at(lane + 32) : 0.f;
#pragma unroll
  for (int j = 0; j < NPL; ++j) G[j] = 0.f;
  const float* gp = sp.Gpart + (long long)g0 * sp.g_slot_stride + prow * sp.A_pad + lane;
  int s = g0;
  add_slots<NPL, (NPL <= 8 ? 18 : 6)>(gp, s, g1, sp.g_slot_stride, npl, G);
  add_slots<NPL, 6>(gp, s, g1, sp.g_slot_stride, npl, G);
  add_slots<NPL, 1>(gp, s, g1, sp.g_slot_stride, npl, G);
  float f = fa + fb;
  for (int i = lane + 64; i < nfe; i += 32) f += f_at(i);
  return warp_sum(f);
}

// ---------------------------------------------------------------------------------------------
// The history of a plan (m pairs, 2 m A_pad floats) is staged in shared memory by bulk asynchronous copies issued
// at the very start, so the 2 m dependent dot products of the two-loop recursion read shared memory instead of
// paying one HBM/L2 latency each.  wpb warps (= plans) per CTA; dynamic smem = wpb * 2 m A_pad floats.
template <int NPL>
__global__ void __launch_bounds__(128) k_step(StepParams sp, PlanPtrs pp, int parity, float g_scale, int wpb) {
  extern __shared__ __align__(128) float s_hist[];
  __shared__ float s_a[4][GMCO_MAX_HISTORY];
  __shared__ __align__(8) uint64_t s_bar[4];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int k = blockIdx.x * wpb + warp;
  if (k >= sp.K) return;
  // three independent loads, issued together: tested one after the other they were three dependent memory round trips
  // before the first useful load (36 % of the kernel's stall samples)
  const int n_run = pp.n_running[parity];
  const int status0 = pp.status[k];
  const int cur = sp.compact_cap ? pp.slot[k] : -1;            // where this round's partials of the plan are
  const int npl = sp.A_pad >> 5;
  const long long row = (long long)k * sp.A_pad + lane;
  // Every global read of the plan's state is issued here as well, before the status is known (all rows exist for
  // k < K; a plan that has stopped just discards them): the whole kernel then pays about one memory round trip plus the
  // batches of the gradient partials (it is latency-bound, not bandwidth-bound).  rho / gamma of the m history pairs
  // live in lanes 0..m-1 and are broadcast by shuffle in the two-loop recursion: a global load per recursion step
  // would put 2 m dependent L2 latencies on the critical path.
  float G[NPL], xt[NPL], gt[NPL], x[NPL], g[NPL];
#pragma unroll
  for (int j = 0; j < NPL; ++j) {
    xt[j] = j < npl ? pp.xt[row + 32 * j] : 0.f;
    x[j] = j < npl ? pp.x[row + 32 * j] : 0.f;
    g[j] = j < npl ? pp.g[row + 32 * j] : 0.f;
  }
  float rho_l = lane < sp.m ? pp.rho[(long long)lane * pp.K_pad + k] : 0.f;
  float gam_l = lane < sp.m ? pp.gam[(long long)lane * pp.K_pad + k] : 0.f;
  int tr = pp.trials[k];
  float F = pp.F[k];
  int it = pp.it_done[k];
  int hc = pp.hcount[k], hh = pp.hhead[k];
  const float alpha = pp.alpha[k], gp = pp.gp[k];
  if (n_run == 0 || status0 != PLAN_RUNNING) return;
  const long long hstride = (long long)pp.K_pad * sp.A_pad;
  float* hS = s_hist + (size_t)warp * 2 * sp.m * sp.A_pad;     // [m][A_pad] s vectors, by ring slot
  float* hY = hS + (size_t)sp.m * sp.A_pad;                    // [m][A_pad] y vectors
  {
    uint64_t* bar = &s_bar[warp];
    const uint32_t bytes = (uint32_t)sp.A_pad * 4u;
    if (lane == 0) {
      mbar_init(bar, 1);
      fence_barrier_init();
      mbar_expect_tx(bar, bytes * 2u * (uint32_t)sp.m);
    }
    __syncwarp();
    for (int i = lane; i < 2 * sp.m; i += 32) {                // one 4 A_pad byte row per lane
      const int slot = i < sp.m ? i : i - sp.m;
      const float* src = (i < sp.m ? pp.Sh : pp.Yh) + slot * hstride + (long long)k * sp.A_pad;
      bulk_load(hS + (size_t)i * sp.A_pad, src, bytes, bar);
    }
  }
  // Every path below waits for the copies before the warp may leave (the CTA's shared memory must outlive them).
  // The wait is bounded: copies that have not landed after seconds are a fault of the machine, not a state to spin
  // in -- the device error word is set (the host reports GMCO_E_CUDA) and the warp goes on.
  auto hist_wait = [&]() {
    const uint32_t bar = smem_u32(&s_bar[warp]);
    bool ok = false;
    unsigned long long t0 = 0;
    for (uint32_t spins = 1; !ok; ++spins) {
      ok = mbar_try_wait_addr(bar, 0);
      if (!ok && (spins & 4095u) == 0u) {        // the clock is read rarely: this wait is on the kernel's critical path
        const unsigned long long now = global_ns();
        if (t0 == 0) t0 = now;
        else if (now - t0 > 4000000000ull) {
          if (lane == 0 && atomicCAS(pp.dev_err, 0, (int)DEVERR_WAIT_TIMEOUT) == 0) {
            pp.dev_err[1] = (DEVERR_K_STEP << 8) | DEVERR_W_HISTORY; pp.dev_err[2] = (int)blockIdx.x; pp.dev_err[3] = k;
          }
          break;
        }
      }
    }
  };

  const float Ft = reduce_partials<NPL>(sp, k, lane, npl, G, cur, n_run);
#pragma unroll
  for (int j = 0; j < NPL; ++j) gt[j] = g_scale * xt[j] * G[j];   // Eq. 3 summed: g = 2 x o (D^T r)
  int status = PLAN_RUNNING;
  bool new_dir = false;
  // A plan that goes on to another round counts itself and, with compaction, takes the count as its slot: the running
  // plans fill rows [0, n_running) of T, and the contraction kernels touch the leading tiles only.  Which slot a plan
  // gets depends on scheduling; its numbers do not (every row of a tile is summed the same way).
  auto claim_row = [&]() -> long long {
    int s = 0;
    if (lane == 0) s = atomicAdd(&pp.n_running[parity ^ 1], 1);
    if (!sp.compact_cap) return row;
    s = __shfl_sync(0xffffffffu, s, 0);
    if (lane == 0) pp.slot[k] = s;
    if (lane < 2 * sp.S) pp.WeffC[(long long)s * 2 * sp.S + lane] = pp.Weff[(long long)k * 2 * sp.S + lane];
    return (long long)s * sp.A_pad + lane;
  };

  if (tr < 0) {                                              // start point: nothing to compare against
#pragma unroll
    for (int j = 0; j < NPL; ++j) { x[j] = xt[j]; g[j] = gt[j]; }
    F = Ft;
    new_dir = true;
    if (it >= sp.iters) status = GMCO_PLAN_ITERS;
  } else {
    bool accept = Ft <= F + sp.c1 * alpha * gp;              // Armijo
    if (!accept && sp.eps_f > 0.f && Ft <= F + sp.eps_f * fabsf(F)) {
      // approximate test (reading A5b): F within its noise allowance and slope condition
      // phi'(alpha) <= (2 c1 - 1) phi'(0), with alpha phi'(alpha) = g+ . (x+ - x)
      float gts = 0.f;
#pragma unroll
      for (int j = 0; j < NPL; ++j) gts = fmaf(gt[j], xt[j] - x[j], gts);
      gts = warp_sum(gts);
      accept = gts <= (2.f * sp.c1 - 1.f) * alpha * gp;
    }
    if (accept) {                                            // accept x+ = x + alpha p
      float sy = 0.f, ss = 0.f, yy = 0.f;
      float sv[NPL], yv[NPL];
#pragma unroll
      for (int j = 0; j < NPL; ++j) {
        sv[j] = xt[j] - x[j]; yv[j] = gt[j] - g[j];
        sy = fmaf(sv[j], yv[j], sy); ss = fmaf(sv[j], sv[j], ss); yy = fmaf(yv[j], yv[j], yy);
      }
      sy = warp_sum(sy); ss = warp_sum(ss); yy = warp_sum(yy);
      hist_wait();                                           // the staged copy of slot hh is about to be replaced
      if (sy > 1e-10f * sqrtf(ss) * sqrtf(yy)) {             // curvature guard
        float* Sd = pp.Sh + hh * hstride + row;
        float* Yd = pp.Yh + hh * hstride + row;
#pragma unroll
        for (int j = 0; j < NPL; ++j)
          if (j < npl) {
            Sd[32 * j] = sv[j]; Yd[32 * j] = yv[j];
            hS[hh * sp.A_pad + lane + 32 * j] = sv[j]; hY[hh * sp.A_pad + lane + 32 * j] = yv[j];
          }
        if (lane == hh) {
          rho_l = 1.f / sy; gam_l = sy / yy;
          pp.rho[(long long)hh * pp.K_pad + k] = rho_l; pp.gam[(long long)hh * pp.K_pad + k] = gam_l;
        }
        hh = hh + 1 == sp.m ? 0 : hh + 1;
        hc = min(hc + 1, sp.m);
      }
      const float Fold = F;
#pragma unroll
      for (int j = 0; j < NPL; ++j) { x[j] = xt[j]; g[j] = gt[j]; }
      F = Ft;
      it += 1;
      new_dir = true;
      if (sp.eps > 0.f && fabsf(Fold - F) <= sp.eps * fmaxf(Fold, 1e-30f)) status = GMCO_PLAN_CONVERGED;
      else if (it >= sp.iters) status = GMCO_PLAN_ITERS;
    } else {                                                 // reject: halve the step along the same p
      tr += 1;
      if (tr >= sp.max_trials) {
        status = GMCO_PLAN_STALLED;
      } else {
        const float a2 = alpha * 0.5f;
        const long long trow = claim_row();
#pragma unroll
        for (int j = 0; j < NPL; ++j)
          if (j < npl) {
            const float pv = pp.p[row + 32 * j];
            const float xn = fmaf(a2, pv, x[j]), t = xn * xn;
            pp.xt[row + 32 * j] = xn; pp.T[trow + 32 * j] = t;
            if (pp.T_lo) pp.T_lo[trow + 32 * j] = tf32_rn(t - tf32_rn(t));
          }
        if (lane == 0) { pp.alpha[k] = a2; pp.trials[k] = tr; }
        // option: the first rejection of an iteration queues the plan for the polynomial line search (kernels_ls.cu),
        // which may replace the halved trial point written above by a later candidate before the next round
        if (sp.ls_cap && tr == 1 && lane == 0) {
          const int e = atomicAdd(pp.ls_count, 1);
          if (e < sp.ls_cap) pp.ls_list[e] = k;
        }
      }
    }
  }

  if (new_dir) {
#pragma unroll
    for (int j = 0; j < NPL; ++j)
      if (j < npl) { pp.x[row + 32 * j] = x[j]; pp.g[row + 32 * j] = g[j]; }
    float gg = 0.f;
#pragma unroll
    for (int j = 0; j < NPL; ++j) gg = fmaf(g[j], g[j], gg);
    const float gnorm = sqrtf(warp_sum(gg));
    if (status == PLAN_RUNNING && gnorm == 0.f) status = GMCO_PLAN_CONVERGED;
    if (status == PLAN_RUNNING) {
      // two-loop recursion (Liu & Nocedal 1989): q = g; newest -> oldest; scale; oldest -> newest
      float q[NPL];
#pragma unroll
      for (int j = 0; j < NPL; ++j) q[j] = g[j];
      hist_wait();
      __syncwarp();
      for (int i = 0; i < hc; ++i) {
        int slot = hh - 1 - i; if (slot < 0) slot += sp.m;
        const float* Sd = hS + slot * sp.A_pad + lane;
        const float* Yd = hY + slot * sp.A_pad + lane;
        float sv[NPL], yv[NPL], d = 0.f;
#pragma unroll
        for (int j = 0; j < NPL; ++j) { sv[j] = j < npl ? Sd[32 * j] : 0.f; yv[j] = j < npl ? Yd[32 * j] : 0.f; }
#pragma unroll
        for (int j = 0; j < NPL; ++j) d = fmaf(sv[j], q[j], d);
        const float a = __shfl_sync(0xffffffffu, rho_l, slot) * warp_sum(d);
#pragma unroll
        for (int j = 0; j < NPL; ++j) q[j] = fmaf(-a, yv[j], q[j]);
        if (lane == 0) s_a[warp][i] = a;
      }
      __syncwarp();
      int newest = hh - 1; if (newest < 0) newest += sp.m;
      const float gam_n = __shfl_sync(0xffffffffu, gam_l, newest);
      const float gamma = hc > 0 ? gam_n : 1.f / gnorm;
#pragma unroll
      for (int j = 0; j < NPL; ++j) q[j] *= gamma;
      for (int i = hc - 1; i >= 0; --i) {
        int slot = hh - 1 - i; if (slot < 0) slot += sp.m;
        const float* Sd = hS + slot * sp.A_pad + lane;
        const float* Yd = hY + slot * sp.A_pad + lane;
        float sv[NPL], yv[NPL], d = 0.f;
#pragma unroll
        for (int j = 0; j < NPL; ++j) { sv[j] = j < npl ? Sd[32 * j] : 0.f; yv[j] = j < npl ? Yd[32 * j] : 0.f; }
#pragma unroll
        for (int j = 0; j < NPL; ++j) d = fmaf(yv[j], q[j], d);
        const float b = __shfl_sync(0xffffffffu, rho_l, slot) * warp_sum(d);
        const float coef = s_a[warp][i] - b;
#pragma unroll
        for (int j = 0; j < NPL; ++j) q[j] = fmaf(sv[j], coef, q[j]);
      }
      float gpn = 0.f;
#pragma unroll
      for (int j = 0; j < NPL; ++j) gpn = fmaf(g[j], -q[j], gpn);
      gpn = warp_sum(gpn);
      if (!(gpn < 0.f)) {                                    // not a descent direction: restart from -g/|g|
        hc = 0;
        const float inv = 1.f / gnorm;
        gpn = 0.f;
#pragma unroll
        for (int j = 0; j < NPL; ++j) { q[j] = g[j] * inv; gpn = fmaf(g[j], -q[j], gpn); }
        gpn = warp_sum(gpn);
      }
      const long long trow = claim_row();
#pragma unroll
      for (int j = 0; j < NPL; ++j)
        if (j < npl) {
          const float pv = -q[j];
          const float xn = x[j] + pv, t = xn * xn;
          pp.p[row + 32 * j] = pv; pp.xt[row + 32 * j] = xn;
          pp.T[trow + 32 * j] = t;
          if (pp.T_lo) pp.T_lo[trow + 32 * j] = tf32_rn(t - tf32_rn(t));
        }
      if (lane == 0) { pp.gp[k] = gpn; pp.alpha[k] = 1.f; pp.trials[k] = 0; }
    }
    if (lane == 0) { pp.F[k] = F; pp.it_done[k] = it; pp.hcount[k] = hc; pp.hhead[k] = hh; }
  }
  if (lane == 0 && status != PLAN_RUNNING) pp.status[k] = status;
  hist_wait();
}

template <int NPL>
static void step_launch(const PlanDev& p, const StepParams& sp, int parity, float g_scale, cudaStream_t st) {
  const size_t per_plan = (size_t)2 * sp.m * sp.A_pad * sizeof(float);     // <= 2 * 16 * 480 * 4 = 61 KB
  int wpb = (int)((200u << 10) / per_plan);
  if (wpb > 4) wpb = 4;
  const size_t smem = per_plan * wpb;
  static size_t allowed = 0;                                               // per instantiation
  if (smem > allowed) {
    if (cudaFuncSetAttribute(k_step<NPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(200u << 10)) != cudaSuccess) return;
    allowed = 200u << 10;
  }
  k_step<NPL><<<(p.K + wpb - 1) / wpb, 32 * wpb, smem, st>>>(sp, make_ptrs(p), parity, g_scale, wpb);
}

int launch_step_parity(const CaseDev& c, const PlanDev& p, const StepParams& sp, int parity, float g_scale,
                       cudaStream_t st) {
  if (p.K == 0) return 0;
  const int npl = c.A_pad / 32;
  if (npl <= 2) step_launch<2>(p, sp, parity, g_scale, st);
  else if (npl <= 4) step_launch<4>(p, sp, parity, g_scale, st);
  else if (npl <= 6) step_launch<6>(p, sp, parity, g_scale, st);
  else if (npl <= 8) step_launch<8>(p, sp, parity, g_scale, st);
  else if (npl <= 10) step_launch<10>(p, sp, parity, g_scale, st);
  else if (npl <= 12) step_launch<12>(p, sp, parity, g_scale, st);
  else step_launch<kMaxNpl>(p, sp, parity, g_scale, st);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// zero the "next round" counter; runs before the contraction kernels of a round
__global__ void k_round_begin(int* zero_ctr, const int* gate, int* log_slot, int* round_ctr) {
  *zero_ctr = 0;
  if (log_slot) *log_slot = *gate;
  if (round_ctr && *gate > 0) *round_ctr += 1;
}

// tail of the WHILE body (two rounds): loop again while a plan is running, the round budget lasts and no kernel has
// reported a protocol error
__global__ void k_loop_cond(cudaGraphConditionalHandle cond, const int* __restrict__ n_running, int* rounds_done,
                            const int* __restrict__ dev_err, int max_rounds) {
  const int r = *rounds_done + 2;
  *rounds_done = r;
  cudaGraphSetConditional(cond, (n_running[0] > 0 && r < max_rounds && dev_err[0] == 0) ? 1u : 0u);
}

int launch_loop_cond(cudaGraphConditionalHandle cond, const PlanDev& p, int max_rounds, cudaStream_t st) {
  k_loop_cond<<<1, 1, 0, st>>>(cond, p.n_running, p.rounds_done, p.dev_err, max_rounds);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_round_begin(int* zero_ctr, const int* gate, int* log_slot, int* round_ctr, cudaStream_t st) {
  k_round_begin<<<1, 1, 0, st>>>(zero_ctr, gate, log_slot, round_ctr);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
// gmco_evaluate: F and dF/dx of the trial point from the partials.
template <int NPL>
__global__ void __launch_bounds__(128) k_eval_finish(StepParams sp, const float* __restrict__ xt, int A, float g_scale,
                                                     float* __restrict__ F_out, float* __restrict__ grad_out) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int k = blockIdx.x * 4 + warp;
  if (k >= sp.K) return;
  const int npl = sp.A_pad >> 5;
  float G[NPL];
  const float F = reduce_partials<NPL>(sp, k, lane, npl, G);
  if (lane == 0 && F_out) F_out[k] = F;
  if (grad_out) {
#pragma unroll
    for (int j = 0; j < NPL; ++j) {
      const int a = lane + 32 * j;
      if (j < npl && a < A) grad_out[(long long)k * A + a] = g_scale * xt[(long long)k * sp.A_pad + a] * G[j];
    }
  }
}

int launch_eval_finish_scaled(const CaseDev& c, const PlanDev& p, const StepParams& sp, float g_scale, float* F_out,
                              float* grad_out, cudaStream_t st) {
  if (p.K == 0) return 0;
  const int npl = c.A_pad / 32;
  const int grid = (p.K + 3) / 4;
  if (npl <= 4) k_eval_finish<4><<<grid, 128, 0, st>>>(sp, p.xt, c.A, g_scale, F_out, grad_out);
  else if (npl <= 8) k_eval_finish<8><<<grid, 128, 0, st>>>(sp, p.xt, c.A, g_scale, F_out, grad_out);
  else if (npl <= 12) k_eval_finish<12><<<grid, 128, 0, st>>>(sp, p.xt, c.A, g_scale, F_out, grad_out);
  else k_eval_finish<kMaxNpl><<<grid, 128, 0, st>>>(sp, p.xt, c.A, g_scale, F_out, grad_out);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
// a8 prologue: dwell times of the ACCEPTED point (not the last trial) for the final dose pass.
__global__ void k_prepare_final(const float* __restrict__ x, float* __restrict__ T, long long n, int* __restrict__ cnt,
                                long long ncnt) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { const float v = x[i]; T[i] = v * v; }
  if (i < ncnt) cnt[i] = 0;
}

int launch_prepare_final(const CaseDev& c, const PlanDev& p, cudaStream_t st) {
  if (p.K_pad == 0) return 0;
  const long long n = (long long)p.K_pad * c.A_pad, ncnt = (long long)p.K_pad * c.S;
  k_prepare_final<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p.x, p.T, n, p.res_cnt, ncnt);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace gmco
