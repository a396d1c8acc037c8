// Device helpers shared by the PSWF-LR kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>

#include "plan.hpp"

namespace pswf {

// Stencil rule (reading R4): u = frac(x/L) * M, i0 = ceil(u - w/2), the atom touches grid
// points i0 .. i0+w-1 (mod M); delta = i0 - (u - w/2) in [0,1) is the in-panel coordinate and the
// window argument of point t is z_t = 2 (t + delta) / w - 1.  Done in double for both precisions
// so that no bits of the in-cell offset are lost at u ~ M (a handful of DP ops per atom).
__device__ __forceinline__ void stencil_1d(double x, double invL, int M, int w, int& i0, double& delta) {
  // explicit _rn intrinsics: no FMA contraction, so the integer decision i0 = ceil(u) is taken
  // with exactly the roundings DESIGN.md reading R4 states (and the oracle reproduces)
  double s = __dmul_rn(x, invL);
  s = __dsub_rn(s, floor(s));
  if (s >= 1.0) s = 0.0;
  double u = __dsub_rn(__dmul_rn(s, (double)M), 0.5 * (double)w);
  double cu = ceil(u);
  i0 = (int)cu;
  delta = __dsub_rn(cu, u);
}

__device__ __forceinline__ int wrap_index(int i, int M) {
  i %= M;
  return i < 0 ? i + M : i;
}

template <class T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Horner evaluation of panel polynomial t at xi: sum_m coef[m*w + t] xi^m  (PAPER.md (S81)).
template <class T>
__device__ __forceinline__ T horner_panel(const T* __restrict__ coef, int w, int t, int degree, T xi) {
  T v = coef[degree * w + t];
  for (int m = degree - 1; m >= 0; --m) v = fma(v, xi, coef[m * w + t]);
  return v;
}

}  // namespace pswf
