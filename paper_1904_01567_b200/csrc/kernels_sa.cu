// kernels_sa.cu -- gSA: K simulated-annealing chains in parallel, one CTA per chain
// (PAPER.md:96-113 steps (ii)-(v); the move, cooling and acceptance rule are BASELINE.json configs[4],
// DESIGN.md 2.5).  Each step changes ONE dwell time, so dose is updated incrementally,
//   d' = d + (t' - t_j) D[:, j]      (Eq. 1 is linear in t),
// and the change of the objective is the sum over points of f(d'_i) - f(d_i) with the SAME Eq. 2 code as the
// gL-BFGS dose epilogues (penalty.cuh).  The chain's dose vector, the cached per-point penalties and the
// per-point thresholds/weights live in registers (PPT points per thread) or, for large cases, in shared memory;
// the column D[:, j] comes from a transposed copy Dt[A][N_alloc] so that the read is coalesced, and the column of
// the NEXT step is fetched while the current step reduces.  Random draws are inputs (no generator on either side).
//
// Template parameter R: double = decisions taken in the oracle's precision (the parity route),
//                       float  = everything in fp32 (the speed route).
#include "gmco_internal.cuh"
#include "penalty.cuh"

namespace gmco {

namespace {

constexpr int kSaWarps = kSaThreads / 32;

template <class R> __device__ __forceinline__ R warp_sum_all(R v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ double block_sum_double(double v, double* scratch /*[kSaWarps]*/) {
  v = warp_sum_all<double>(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
#pragma unroll
  for (int w = 0; w < kSaWarps; ++w) s += scratch[w];
  return s;
}

}  // namespace

// Dt[a][r] = D[r][a]
__global__ void k_sa_transpose(const float* __restrict__ D, int N_alloc, int A_pad, int A, float* __restrict__ Dt) {
  __shared__ float tile[32][33];
  const int r0 = blockIdx.x * 32, a0 = blockIdx.y * 32;
  for (int i = threadIdx.y; i < 32; i += blockDim.y) tile[i][threadIdx.x] = D[(size_t)(r0 + i) * A_pad + a0 + threadIdx.x];
  __syncthreads();
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    const int a = a0 + i;
    if (a < A) Dt[(size_t)a * N_alloc + r0 + threadIdx.x] = tile[threadIdx.x][i];
  }
}

int launch_sa_transpose(const CaseDev& c, float* Dt, cudaStream_t st) {
  dim3 grid(c.N_alloc / 32, c.A_pad / 32), block(32, 8);
  k_sa_transpose<<<grid, block, 0, st>>>(c.D, c.N_alloc, c.A_pad, c.A, Dt);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// PPT > 0: points per thread, state in registers.  PPT == 0: state in shared memory, any N_pad that fits.
template <class R, int PPT>
__global__ void __launch_bounds__(kSaThreads) k_sa_chain(const SaArgs a) {
  extern __shared__ __align__(16) unsigned char sa_smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int chain = blockIdx.x;
  const int A = a.A, S2 = 2 * a.S, N_pad = a.N_pad;

  // ---- shared memory carve-up (doubles first) ----
  double* Tn_s = reinterpret_cast<double*>(sa_smem);           // [kSaBlock] temperature of each staged step
  double* z_s = Tn_s + kSaBlock;                                // [kSaBlock]
  double* u_s = z_s + kSaBlock;                                 // [kSaBlock]
  double* scratch = u_s + kSaBlock;                             // [kSaWarps]
  double* weff_s = scratch + kSaWarps;                          // [2 * GMCO_MAX_STRUCTS]
  R* red = reinterpret_cast<R*>(weff_s + 2 * GMCO_MAX_STRUCTS); // [2][kSaWarps]
  R* t_s = red + 2 * kSaWarps;                                  // [A_pad]
  int* j_s = reinterpret_cast<int*>(t_s + a.A_pad);             // [kSaBlock]
  R* d_s = reinterpret_cast<R*>(j_s + kSaBlock);                // PPT == 0: [N_pad] dose, then [N_pad] cached penalty
  R* f_s = d_s + N_pad;
  __shared__ int bad_s;

  // ---- inputs: weights, start dwell times, validation ----
  if (tid == 0) bad_s = 0;
  __syncthreads();
  if (tid < S2) {
    const float w = a.w_user[(size_t)chain * S2 + tid];
    if (!(w >= 0.f) || isinf(w)) bad_s = 1;
    weff_s[tid] = (double)w * a.wscale[tid];
  }
  for (int l = tid; l < A; l += kSaThreads) {
    const float v = a.T0[a.t0_bcast ? l : (size_t)chain * A + l];
    if (!(v >= 0.f) || isinf(v)) bad_s = 1;
    t_s[l] = (R)v;
  }
  __syncthreads();
  if (bad_s) {
    if (tid == 0) atomicOr(a.bad_input, 1);
    return;
  }

  // ---- per-point constants and the start dose d = D t0 (Eq. 1), in dwell order ----
  R d[PPT > 0 ? PPT : 1], fo[PPT > 0 ? PPT : 1], lo[PPT > 0 ? PPT : 1], hi[PPT > 0 ? PPT : 1], wl[PPT > 0 ? PPT : 1],
      wh[PPT > 0 ? PPT : 1];
  double Fpart = 0.0;
  if constexpr (PPT > 0) {
#pragma unroll
    for (int p = 0; p < PPT; ++p) {
      const int i = tid + p * kSaThreads;
      d[p] = R(0); fo[p] = R(0); lo[p] = R(0); hi[p] = R(0); wl[p] = R(0); wh[p] = R(0);
      if (i < N_pad) {
        const int s = a.tile_struct[i >> 6];
        lo[p] = (R)a.pt_lo[i]; hi[p] = (R)a.pt_hi[i];
        wl[p] = (R)weff_s[2 * s]; wh[p] = (R)weff_s[2 * s + 1];
        R acc = R(0);
        for (int l = 0; l < A; ++l) acc += (R)a.Dt[(size_t)l * a.ldt + i] * t_s[l];
        d[p] = acc;
        fo[p] = eq2_value<R>(acc, lo[p], hi[p], wl[p], wh[p]);
        Fpart += (double)fo[p];
      }
    }
  } else {
    for (int i = tid; i < N_pad; i += kSaThreads) {
      const int s = a.tile_struct[i >> 6];
      R acc = R(0);
      for (int l = 0; l < A; ++l) acc += (R)a.Dt[(size_t)l * a.ldt + i] * t_s[l];
      d_s[i] = acc;
      const R f = eq2_value<R>(acc, (R)a.pt_lo[i], (R)a.pt_hi[i], (R)weff_s[2 * s], (R)weff_s[2 * s + 1]);
      f_s[i] = f;
      Fpart += (double)f;
    }
  }
  R F = (R)block_sum_double(Fpart, scratch);

  const int64_t steps = a.steps;
  const size_t draw_base = a.draws_bcast ? 0 : (size_t)chain * (size_t)steps;
  const R tau001 = (R)(0.01 * a.tau);
  long long n_acc = 0;
  int prev_j = -1, prev_acc = 0;
  R prev_tn = R(0);
  int par = 0;

  for (int64_t n0 = 0; n0 < steps; n0 += kSaBlock) {
    const int nb = (int)((steps - n0) < (int64_t)kSaBlock ? (steps - n0) : (int64_t)kSaBlock);
    __syncthreads();                      // the previous block's staged draws are no longer read
    if (tid < nb) {
      const int64_t n = n0 + tid;
      int j = a.jdx[draw_base + n];
      if (j < 0 || j >= A) { atomicOr(a.bad_input, 2); j = 0; }
      j_s[tid] = j;
      z_s[tid] = a.z[draw_base + n];
      u_s[tid] = a.u[draw_base + n];
      Tn_s[tid] = a.temp0 * exp((double)n * a.log_cooling);
    }
    __syncthreads();

    float cn[PPT > 0 ? PPT : 1];          // column of the next step, fetched one step ahead
    if constexpr (PPT > 0) {
      const float* col = a.Dt + (size_t)j_s[0] * a.ldt;
#pragma unroll
      for (int p = 0; p < PPT; ++p) { const int i = tid + p * kSaThreads; cn[p] = i < N_pad ? col[i] : 0.f; }
    }

    for (int s = 0; s < nb; ++s) {
      const int j = j_s[s];
      // t_j: the write of the previous step's accepted value may not be visible yet; every thread knows it
      const R tj = (prev_acc && j == prev_j) ? prev_tn : t_s[j];
      const R sigma = max((R)0.1 * tj, tau001);
      const R tn = max(tj + sigma * (R)z_s[s], R(0));
      const R dt = tn - tj;
      R part = R(0);
      R dn[PPT > 0 ? PPT : 1], fn[PPT > 0 ? PPT : 1];
      if constexpr (PPT > 0) {
        float cc[PPT];
#pragma unroll
        for (int p = 0; p < PPT; ++p) cc[p] = cn[p];
        if (s + 1 < nb) {
          const float* col = a.Dt + (size_t)j_s[s + 1] * a.ldt;
#pragma unroll
          for (int p = 0; p < PPT; ++p) { const int i = tid + p * kSaThreads; cn[p] = i < N_pad ? col[i] : 0.f; }
        }
#pragma unroll
        for (int p = 0; p < PPT; ++p) {
          dn[p] = d[p] + dt * (R)cc[p];
          fn[p] = eq2_value<R>(dn[p], lo[p], hi[p], wl[p], wh[p]);
          part += fn[p] - fo[p];
        }
      } else {
        const float* col = a.Dt + (size_t)j * a.ldt;
        for (int i = tid; i < N_pad; i += kSaThreads) {
          const int st = a.tile_struct[i >> 6];
          const R dnew = d_s[i] + dt * (R)col[i];
          part += eq2_value<R>(dnew, (R)a.pt_lo[i], (R)a.pt_hi[i], (R)weff_s[2 * st], (R)weff_s[2 * st + 1]) - f_s[i];
        }
      }
      part = warp_sum_all<R>(part);
      if (lane == 0) red[par * kSaWarps + warp] = part;
      __syncthreads();
      R dF = R(0);
#pragma unroll
      for (int w = 0; w < kSaWarps; ++w) dF += red[par * kSaWarps + w];
      par ^= 1;

      // Metropolis rule; every thread takes the same decision from the same numbers
      bool accept = dF <= R(0);
      if (!accept) {
        const R Tn = (R)Tn_s[s];
        accept = (Tn > R(0)) && ((R)u_s[s] < exp(-dF / Tn));
      }
      if (accept) {
        if constexpr (PPT > 0) {
#pragma unroll
          for (int p = 0; p < PPT; ++p) { d[p] = dn[p]; fo[p] = fn[p]; }
        } else {
          const float* col = a.Dt + (size_t)j * a.ldt;
          for (int i = tid; i < N_pad; i += kSaThreads) {
            const int st = a.tile_struct[i >> 6];
            const R dnew = d_s[i] + dt * (R)col[i];
            d_s[i] = dnew;
            f_s[i] = eq2_value<R>(dnew, (R)a.pt_lo[i], (R)a.pt_hi[i], (R)weff_s[2 * st], (R)weff_s[2 * st + 1]);
          }
        }
        F += dF;
        ++n_acc;
        if (tid == 0) t_s[j] = tn;
      }
      prev_j = j; prev_tn = tn; prev_acc = accept ? 1 : 0;
    }
  }

  // ---- outputs: dwell times, the objective summed afresh from the cached penalties, acceptance count ----
  __syncthreads();
  for (int l = tid; l < A; l += kSaThreads) a.T_out[(size_t)chain * A + l] = (double)t_s[l];
  double Fend = 0.0;
  if constexpr (PPT > 0) {
#pragma unroll
    for (int p = 0; p < PPT; ++p) Fend += (double)fo[p];
  } else {
    for (int i = tid; i < N_pad; i += kSaThreads) Fend += (double)f_s[i];
  }
  Fend = block_sum_double(Fend, scratch);
  if (tid == 0) {
    a.F_out[chain] = Fend;
    a.F_tracked[chain] = (double)F;
    a.n_accepted[chain] = n_acc;
  }
}

size_t sa_smem_bytes(const CaseDev& c, int precision, int ppt) {
  const size_t R = precision == GMCO_SA_FP64 ? 8 : 4;
  size_t b = sizeof(double) * (3 * kSaBlock + kSaWarps + 2 * GMCO_MAX_STRUCTS) + R * (2 * kSaWarps + c.A_pad) +
             sizeof(int) * kSaBlock;
  if (ppt == 0) b += 2 * R * (size_t)c.N_pad;
  return (b + 15) & ~size_t(15);
}

int sa_points_per_thread(const CaseDev& c) {
  const int need = (c.N_pad + kSaThreads - 1) / kSaThreads;
  for (int ppt : {1, 2, 3, 4, 6, 8}) if (need <= ppt) return ppt;
  return 0;
}

template <class R, int PPT>
static int launch_one(const SaArgs& a, int K, size_t smem, cudaStream_t st) {
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_sa_chain<R, PPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return -1;
  k_sa_chain<R, PPT><<<K, kSaThreads, smem, st>>>(a);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

template <class R>
static int launch_prec(const SaArgs& a, int K, int ppt, size_t smem, cudaStream_t st) {
  switch (ppt) {
    case 1: return launch_one<R, 1>(a, K, smem, st);
    case 2: return launch_one<R, 2>(a, K, smem, st);
    case 3: return launch_one<R, 3>(a, K, smem, st);
    case 4: return launch_one<R, 4>(a, K, smem, st);
    case 6: return launch_one<R, 6>(a, K, smem, st);
    case 8: return launch_one<R, 8>(a, K, smem, st);
    default: return launch_one<R, 0>(a, K, smem, st);
  }
}

int launch_sa_chains(const CaseDev& c, const SaArgs& a, int K, int precision, cudaStream_t st) {
  const int ppt = sa_points_per_thread(c);
  const size_t smem = sa_smem_bytes(c, precision, ppt);
  return precision == GMCO_SA_FP64 ? launch_prec<double>(a, K, ppt, smem, st) : launch_prec<float>(a, K, ppt, smem, st);
}

}  // namespace gmco
