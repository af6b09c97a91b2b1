// kernels_doserate.cu -- step (i) of the paper's loop: the dose-rate matrix, N_pnt x N_act evaluations.
// The paper does not print its dose-rate model; BASELINE.json configs[0] fixes the TG-43 point-source approximation
//   D_il = S_K Lambda g(r) / r^2,  r = |p_i - q_l| in cm, floored at r_floor,  g a polynomial in r
// whose coefficients are INPUTS (the library owns no source data).  fp64 arithmetic, one rounding to fp32 at the end:
// N x A is a few million elements, the fp64 pipe does them in microseconds, and D then agrees with the fp64 oracle to
// the last fp32 bit almost everywhere.
#include "gmco_internal.cuh"

namespace gmco {

__global__ void __launch_bounds__(256) k_dose_rate(const float* __restrict__ pts, long long N,
                                                   const float* __restrict__ dwell, int A, DoseRateArgs m,
                                                   float* __restrict__ D, long long ldD) {
  extern __shared__ double s_q[];                     // [A][3] dwell positions in cm
  for (int i = threadIdx.x; i < 3 * A; i += blockDim.x) s_q[i] = (double)dwell[i] / 10.0;
  __syncthreads();
  const long long i = blockIdx.x;
  if (i >= N) return;
  const double px = (double)pts[3 * i] / 10.0, py = (double)pts[3 * i + 1] / 10.0, pz = (double)pts[3 * i + 2] / 10.0;
  for (int l = threadIdx.x; l < A; l += blockDim.x) {
    const double dx = px - s_q[3 * l], dy = py - s_q[3 * l + 1], dz = pz - s_q[3 * l + 2];
    const double r = fmax(sqrt(dx * dx + dy * dy + dz * dz), m.r_floor_cm);
    double g = 0.0;
    for (int c = m.n_coef - 1; c >= 0; --c) g = g * r + m.coef[c];     // Horner, highest power first
    D[i * ldD + l] = (float)(m.sk_lambda * g / (r * r));
  }
}

int launch_dose_rate(const float* pts, long long N, const float* dwell, int A, const DoseRateArgs& m, float* D,
                     long long ldD, cudaStream_t st) {
  const size_t smem = (size_t)3 * A * sizeof(double);
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(k_dose_rate, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return -1;
  k_dose_rate<<<(unsigned)N, 256, smem, st>>>(pts, N, dwell, A, m, D, ldD);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace gmco
