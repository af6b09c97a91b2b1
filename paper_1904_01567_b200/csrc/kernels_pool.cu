// kernels_pool.cu -- what gMCO does with the plan pool after the optimisation (NEXT rows 3-4 of SURVEY.md 8(f)):
//   k_pareto : non-dominated plans over the per-organ objective values
//   k_select : RTOG / RTOG+ classification and the selection rule of PAPER.md:147-151
// Comparisons only (plus one fp32 sum of at most GMCO_MAX_CRITERIA indices in criterion order): integer results,
// bit-exact against the oracle.
#include "gmco_internal.cuh"

namespace gmco {

constexpr int kParetoThreads = 256;

// Plan a dominates plan b if a_m <= b_m for every m and a_m < b_m for at least one m (all objectives are minimised).
__global__ void __launch_bounds__(kParetoThreads) k_pareto(const float* __restrict__ obj, int K, int M,
                                                           unsigned char* __restrict__ nondom, int* __restrict__ count) {
  extern __shared__ float tile[];                    // [kParetoThreads][M]
  const int b = blockIdx.x * kParetoThreads + threadIdx.x;
  float vb[GMCO_MAX_OBJECTIVES];
#pragma unroll
  for (int m = 0; m < GMCO_MAX_OBJECTIVES; ++m) vb[m] = (b < K && m < M) ? obj[(size_t)b * M + m] : 0.f;
  bool dominated = false;
  for (int a0 = 0; a0 < K; a0 += kParetoThreads) {
    const int na = min(kParetoThreads, K - a0);
    __syncthreads();
    for (int i = threadIdx.x; i < na * M; i += kParetoThreads) tile[i] = obj[(size_t)a0 * M + i];
    __syncthreads();
    for (int a = 0; a < na; ++a) {
      bool all_le = true, any_lt = false;
#pragma unroll
      for (int m = 0; m < GMCO_MAX_OBJECTIVES; ++m)
        if (m < M) { const float va = tile[a * M + m]; all_le &= va <= vb[m]; any_lt |= va < vb[m]; }
      dominated |= all_le && any_lt;
    }
  }
  if (b < K) {
    nondom[b] = dominated ? 0 : 1;
    if (!dominated) atomicAdd(count, 1);               // integer count: order-independent
  }
}

int launch_pareto(const float* obj, int K, int M, unsigned char* nondom, int* count, cudaStream_t st) {
  if (cudaMemsetAsync(count, 0, sizeof(int), st) != cudaSuccess) return -1;
  k_pareto<<<(K + kParetoThreads - 1) / kParetoThreads, kParetoThreads, kParetoThreads * M * sizeof(float), st>>>(
      obj, K, M, nondom, count);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------
constexpr int kSelThreads = 1024;

struct Best { float key; int idx; };                   // larger key wins, then the lower index
__device__ __forceinline__ Best better(Best a, Best b) {
  if (b.idx < 0) return a;
  if (a.idx < 0) return b;
  if (b.key > a.key || (b.key == a.key && b.idx < a.idx)) return b;
  return a;
}

// out[0] = selected plan, out[1..3] = number of plans of class 0 (invalid), 1 (RTOG only), 2 (RTOG+)
__global__ void __launch_bounds__(kSelThreads) k_select(const float* __restrict__ dvh, int K, int S, SelectArgs c,
                                                        int* __restrict__ plan_class, int* __restrict__ out) {
  __shared__ Best s_best[4][kSelThreads / 32];
  __shared__ int s_cnt[3];
  if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  // candidates: [0] RTOG+ valid, max target index; [1] RTOG valid, max target index;
  //             [2] target and must-hold criteria met, min OAR sum; [3] any plan, min OAR sum
  Best best[4] = {{0.f, -1}, {0.f, -1}, {0.f, -1}, {0.f, -1}};
  for (int k = threadIdx.x; k < K; k += kSelThreads) {
    bool rtog = true, plus = true, core = true;
    float target = 0.f, oar = 0.f;
    for (int i = 0; i < c.n; ++i) {
      const float v = dvh[(size_t)k * S + c.structure[i]];
      const bool ok = c.sense[i] > 0 ? v >= c.limit_rtog[i] : v < c.limit_rtog[i];
      const bool okp = c.sense[i] > 0 ? v >= c.limit_plus[i] : v < c.limit_plus[i];
      rtog &= ok; plus &= okp;
      if (c.role[i] == 0) target = v;
      if (c.role[i] != 2) core &= ok;
      if (c.role[i] == 2) oar += v;
    }
    plus &= rtog;
    const int cls = plus ? 2 : (rtog ? 1 : 0);
    if (plan_class) plan_class[k] = cls;
    atomicAdd(&s_cnt[cls], 1);
    if (plus) best[0] = better(best[0], Best{target, k});
    if (rtog) best[1] = better(best[1], Best{target, k});
    if (core) best[2] = better(best[2], Best{-oar, k});
    best[3] = better(best[3], Best{-oar, k});
  }
  for (int q = 0; q < 4; ++q) {
    Best b = best[q];
    for (int o = 16; o > 0; o >>= 1) {
      Best t{__shfl_xor_sync(0xffffffffu, b.key, o), __shfl_xor_sync(0xffffffffu, b.idx, o)};
      b = better(b, t);
    }
    if ((threadIdx.x & 31) == 0) s_best[q][threadIdx.x >> 5] = b;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int sel = -1;
    for (int q = 0; q < 4 && sel < 0; ++q) {
      Best b{0.f, -1};
      for (int w = 0; w < kSelThreads / 32; ++w) b = better(b, s_best[q][w]);
      sel = b.idx;
    }
    out[0] = sel; out[1] = s_cnt[0]; out[2] = s_cnt[1]; out[3] = s_cnt[2];
  }
}

int launch_select(const float* dvh, int K, int S, const SelectArgs& c, int* plan_class, int* out, cudaStream_t st) {
  k_select<<<1, kSelThreads, 0, st>>>(dvh, K, S, c, plan_class, out);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace gmco
