// kernels_ls.cu -- the polynomial line search of north_star item (4) / SURVEY 8(c.2), as an option
// (gmco_options.line_search = 1; off by default, DESIGN.md 2.2 says why).
//
// Dose is linear in t and t = x o x, so along a direction p
//     d(alpha) = D (x + alpha p)^2 = d + 2 alpha a + alpha^2 b,   d = D(x o x), a = D(x o p), b = D(p o p)
// (Eq. 1) and every trial step of an iteration can be valued from three dose columns without a further
// contraction.  The round loop keeps its speculative alpha = 1 trial (the trial evaluation IS the fresh evaluation when
// it is accepted, which it is in 19 iterations of 20).  When k_step rejects that first trial it halves the step as it
// always does AND queues the plan (at most kLsCap plans per round; the others simply go on halving).  Then, in the same
// round:
//   k_ls_cols : the three columns of every queued plan, one SIMT contraction over D (64 points x 16 plans per CTA)
//   k_ls_pick : one CTA per queued plan values phi(alpha_j) and phi'(alpha_j) for alpha_j = 2^-j, j = 1 .. max_trials - 1,
//               with the Eq. 2 code of penalty.cuh, takes the FIRST j that meets the Armijo test or the approximate
//               test (reading A5b) -- the rule of DESIGN.md 2.2, against phi(0) formed the same way -- and, if that is
//               not j = 1, replaces the plan's trial point by x + alpha_j p.
// The next round evaluates that point afresh with the tensor kernels and k_step applies its usual tests to the true
// values: the polynomial only chooses which point is tried next, it never decides an acceptance, so the algorithm
// (and the oracle's iteration count) is unchanged; an iteration with h rejected steps costs 2 rounds instead of 1 + h.
// Plain fp32 FMA kernels: a few dozen plans per round at most.  Product code; shares nothing with oracle/.
#include "gmco_internal.cuh"
#include "gmco_ptx.cuh"
#include "penalty.cuh"

namespace gmco {

namespace {

constexpr int kLsMaxCand = 19;      // candidates alpha_j = 2^-j, j = 1 .. min(max_trials - 1, kLsMaxCand)

// cols [3][cap][N_alloc]: d, a, b of queued plan e at cols[(c * cap + e) * N_alloc + point]
__global__ void __launch_bounds__(256)
k_ls_cols(const float* __restrict__ D, int A_pad, int N_alloc, const float* __restrict__ x, const float* __restrict__ p,
          const int* __restrict__ ls_list, const int* __restrict__ ls_count, int cap, float* __restrict__ cols) {
  const int n = min(*ls_count, cap);
  const int e0 = blockIdx.y * 16;
  if (e0 >= n) return;
  __shared__ float Ds[16][68];
  __shared__ float Us[3][16][17];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  const int p0 = blockIdx.x * 64;
  float acc[3][4];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int i = 0; i < 4; ++i) acc[c][i] = 0.f;
  const int lr = tid >> 2, lc = (tid & 3) * 4;        // D loader: row 0..63, 4 consecutive dwell positions
  const int uk = tid >> 4, up = tid & 15;             // column loader: dwell position a0 + uk of queued plan e0 + up
  const int plan_u = e0 + up < n ? ls_list[e0 + up] : -1;
  for (int a0 = 0; a0 < A_pad; a0 += 16) {
    const float4 dv = *reinterpret_cast<const float4*>(D + (long long)(p0 + lr) * A_pad + a0 + lc);
    Ds[lc + 0][lr] = dv.x; Ds[lc + 1][lr] = dv.y; Ds[lc + 2][lr] = dv.z; Ds[lc + 3][lr] = dv.w;
    float xv = 0.f, pv = 0.f;
    if (plan_u >= 0) { xv = x[(long long)plan_u * A_pad + a0 + uk]; pv = p[(long long)plan_u * A_pad + a0 + uk]; }
    Us[0][uk][up] = xv * xv; Us[1][uk][up] = xv * pv; Us[2][uk][up] = pv * pv;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      const float4 dp = *reinterpret_cast<const float4*>(&Ds[kk][ty * 4]);
      const float dd[4] = {dp.x, dp.y, dp.z, dp.w};
      const float u0 = Us[0][kk][tx], u1 = Us[1][kk][tx], u2 = Us[2][kk][tx];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        acc[0][i] = fmaf(dd[i], u0, acc[0][i]); acc[1][i] = fmaf(dd[i], u1, acc[1][i]); acc[2][i] = fmaf(dd[i], u2, acc[2][i]);
      }
    }
    __syncthreads();
  }
  if (e0 + tx < n) {
#pragma unroll
    for (int c = 0; c < 3; ++c)
      *reinterpret_cast<float4*>(cols + ((long long)c * cap + e0 + tx) * N_alloc + p0 + ty * 4) =
          make_float4(acc[c][0], acc[c][1], acc[c][2], acc[c][3]);
  }
}

struct LsPickArgs {
  const float *cols, *pt_lo, *pt_hi, *Weff, *x, *p, *gp;
  const int *tile_struct, *ls_list, *slot;
  int *ls_count;              // [2]: queued plans of this round | CTAs of k_ls_pick that have finished
  float *xt, *T, *T_lo, *alpha;
  int* trials;
  int cap, N_alloc, N_pad, A_pad, S, n_cand, use_slot;
  float c1, eps_f;
};

__global__ void __launch_bounds__(256) k_ls_pick(LsPickArgs a) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n = min(a.ls_count[0], a.cap);
  const int e = blockIdx.x;
  __shared__ float s_red[8][2 * kLsMaxCand + 1];
  __shared__ int s_pick;
  if (e < n) {
    const int k = a.ls_list[e];
    const float* cd = a.cols + ((long long)0 * a.cap + e) * a.N_alloc;
    const float* ca = a.cols + ((long long)1 * a.cap + e) * a.N_alloc;
    const float* cb = a.cols + ((long long)2 * a.cap + e) * a.N_alloc;
    float phi[kLsMaxCand + 1], slope[kLsMaxCand];
#pragma unroll
    for (int j = 0; j <= kLsMaxCand; ++j) phi[j] = 0.f;
#pragma unroll
    for (int j = 0; j < kLsMaxCand; ++j) slope[j] = 0.f;
    for (int i = tid; i < a.N_pad; i += 256) {
      const int s = a.tile_struct[i >> 6];
      const float dlo = a.pt_lo[i], dhi = a.pt_hi[i];           // padding rows: -inf / +inf, and their columns are 0
      const float wlo = a.Weff[(long long)k * 2 * a.S + 2 * s], whi = a.Weff[(long long)k * 2 * a.S + 2 * s + 1];
      const float d = cd[i], va = ca[i], vb = cb[i];
      phi[0] += eq2_value<float>(d, dlo, dhi, wlo, whi);
      float al = 1.f;
#pragma unroll
      for (int j = 1; j <= kLsMaxCand; ++j) {
        al *= 0.5f;
        if (j <= a.n_cand) {
          const float dj = fmaf(al * al, vb, fmaf(2.f * al, va, d));
          float f_lo = 0.f, f_hi = 0.f;
          const float r_half = eq2_accumulate<float>(dj, dlo, dhi, wlo, whi, f_lo, f_hi);     // dF/dd / 2
          phi[j] += f_lo + f_hi;
          slope[j - 1] = fmaf(2.f * r_half, 2.f * fmaf(al, vb, va), slope[j - 1]);            // dF/dd . dd/dalpha
        }
      }
    }
    // fixed-order reduction: butterfly inside the warp, then warp 0..7 in order
#pragma unroll
    for (int j = 0; j <= kLsMaxCand; ++j) {
      float v = phi[j];
#pragma unroll
      for (int off = 16; off; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      if (lane == 0) s_red[warp][j] = v;
    }
#pragma unroll
    for (int j = 0; j < kLsMaxCand; ++j) {
      float v = slope[j];
#pragma unroll
      for (int off = 16; off; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      if (lane == 0) s_red[warp][kLsMaxCand + 1 + j] = v;
    }
    __syncthreads();
    if (tid == 0) {
      float tot[2 * kLsMaxCand + 1];
      for (int j = 0; j < 2 * kLsMaxCand + 1; ++j) {
        float v = 0.f;
        for (int w = 0; w < 8; ++w) v += s_red[w][j];
        tot[j] = v;
      }
      const float F0 = tot[0], gp = a.gp[k];
      int pick = 0;
      float al = 1.f;
      for (int j = 1; j <= a.n_cand && !pick; ++j) {
        al *= 0.5f;
        const float Fj = tot[j], sj = tot[kLsMaxCand + j];
        if (Fj <= F0 + a.c1 * al * gp) pick = j;                                                  // Armijo
        else if (a.eps_f > 0.f && Fj <= F0 + a.eps_f * fabsf(F0) && sj <= (2.f * a.c1 - 1.f) * gp) pick = j;   // A5b
      }
      s_pick = pick;
    }
    __syncthreads();
    const int pick = s_pick;
    if (pick > 1) {                                   // j = 1 is the trial k_step has already written
      const float al = exp2f(-(float)pick);
      const long long row = (long long)k * a.A_pad;
      const long long trow = (long long)(a.use_slot ? a.slot[k] : k) * a.A_pad;
      for (int q = tid; q < a.A_pad; q += 256) {
        const float xn = fmaf(al, a.p[row + q], a.x[row + q]), t = xn * xn;
        a.xt[row + q] = xn; a.T[trow + q] = t;
        if (a.T_lo) a.T_lo[trow + q] = tf32_rn(t - tf32_rn(t));
      }
      if (tid == 0) { a.alpha[k] = al; a.trials[k] = pick; }
    }
  }
  // the last CTA to finish clears the queue for the next round (every CTA has read the count by then)
  if (tid == 0) {
    __threadfence();
    const int t = atomicAdd(&a.ls_count[1], 1);
    if (t == (int)gridDim.x - 1) { a.ls_count[0] = 0; a.ls_count[1] = 0; }
  }
}

}  // namespace

int launch_ls(const CaseDev& c, const PlanDev& p, int max_trials, float c1, float eps_f, bool use_slot, cudaStream_t st) {
  if (p.K == 0 || !p.ls_cols) return 0;
  dim3 grid(c.N_alloc / 64, kLsCap / 16);
  k_ls_cols<<<grid, 256, 0, st>>>(c.D, c.A_pad, c.N_alloc, p.x, p.p, p.ls_list, p.ls_count, kLsCap, p.ls_cols);
  if (cudaPeekAtLastError() != cudaSuccess) return -1;
  LsPickArgs a{};
  a.cols = p.ls_cols; a.pt_lo = c.pt_lo; a.pt_hi = c.pt_hi; a.Weff = p.Weff; a.x = p.x; a.p = p.p; a.gp = p.gp;
  a.tile_struct = c.tile_struct; a.ls_list = p.ls_list; a.slot = p.slot; a.ls_count = p.ls_count;
  a.xt = p.xt; a.T = p.T; a.T_lo = p.T_lo; a.alpha = p.alpha; a.trials = p.trials;
  a.cap = kLsCap; a.N_alloc = c.N_alloc; a.N_pad = c.N_pad; a.A_pad = c.A_pad; a.S = c.S;
  a.n_cand = max_trials - 1 < kLsMaxCand ? max_trials - 1 : kLsMaxCand;
  a.use_slot = use_slot ? 1 : 0; a.c1 = c1; a.eps_f = eps_f;
  k_ls_pick<<<kLsCap, 256, 0, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? 2 : -1;
}

}  // namespace gmco
