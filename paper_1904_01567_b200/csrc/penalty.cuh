// penalty.cuh -- the one place Eq. 2 is written on the device.
// Used by the dose epilogues of the tensor and SIMT routes and by the gSA kernel (north_star item 5:
// "the shared objective and gradient code reused by a batched gSA kernel").  Product code, no oracle.
#pragma once

namespace gmco {

// f = w_lo min(d - D_lo, 0)^2 + w_hi max(d - D_hi, 0)^2, accumulated into f_lo / f_hi (the two terms are kept
// apart: they are separate objective terms of Eq. 4).  Returns dF/dd / 2 = w_lo min(.) + w_hi max(.).
// D_lo = -inf / D_hi = +inf switch a side off (min(+inf, 0) = 0, max(-inf, 0) = 0).
template <class R>
__device__ __forceinline__ R eq2_accumulate(R d, R d_lo, R d_hi, R w_lo, R w_hi, R& f_lo, R& f_hi) {
  if constexpr (sizeof(R) == 4) {
    const float lo = fminf(d - d_lo, 0.f), hi = fmaxf(d - d_hi, 0.f);
    const float u = w_lo * lo, v = w_hi * hi;
    f_lo = fmaf(u, lo, f_lo);
    f_hi = fmaf(v, hi, f_hi);
    return u + v;
  } else {
    const double lo = fmin(d - d_lo, 0.0), hi = fmax(d - d_hi, 0.0);
    const double u = w_lo * lo, v = w_hi * hi;
    f_lo = fma(u, lo, f_lo);
    f_hi = fma(v, hi, f_hi);
    return u + v;
  }
}

// value only: f(d)
template <class R>
__device__ __forceinline__ R eq2_value(R d, R d_lo, R d_hi, R w_lo, R w_hi) {
  R a = R(0), b = R(0);
  eq2_accumulate<R>(d, d_lo, d_hi, w_lo, w_hi, a, b);
  return a + b;
}

}  // namespace gmco
