// Device helpers shared by the PSWF-LR kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>

#include "plan.hpp"

namespace pswf {

// Stencil rule (reading R4): u = frac(s) * M with s the fractional coordinate (x/L when orthorhombic), i0 = ceil(u - w/2), the atom touches grid
// points i0 .. i0+w-1 (mod M); delta = i0 - (u - w/2) in [0,1) is the in-panel coordinate and the
// window argument of point t is z_t = 2 (t + delta) / w - 1.  Done in double for both precisions
// so that no bits of the in-cell offset are lost at u ~ M (a handful of DP ops per atom).
// Fractional coordinate d of a Cartesian position in the cell h (rows = lattice vectors; hinv = h^-1,
// s = r h^-1): s_d = (x hinv[0][d] + y hinv[1][d]) + z hinv[2][d], products and sums rounded separately in
// this order.  For an orthorhombic box the two zero terms leave s = x * (1/L) bit for bit.
__device__ __forceinline__ double frac_coord(double x, double y, double z, const double* hinv, int d) {
  return __dadd_rn(__dadd_rn(__dmul_rn(x, hinv[d]), __dmul_rn(y, hinv[3 + d])), __dmul_rn(z, hinv[6 + d]));
}

__device__ __forceinline__ void stencil_1d(double s, int M, int w, int& i0, double& delta) {
  // explicit _rn intrinsics: no FMA contraction, so the integer decision i0 = ceil(u) is taken
  // with exactly the roundings DESIGN.md reading R4 states (and the oracle reproduces)
  s = __dsub_rn(s, floor(s));
  if (s >= 1.0) s = 0.0;
  double u = __dsub_rn(__dmul_rn(s, (double)M), 0.5 * (double)w);
  double cu = ceil(u);
  i0 = (int)cu;
  delta = __dsub_rn(cu, u);
}

// the three stencils of one atom
template <class T>
__device__ __forceinline__ void stencil_3d(const T* pos3, const double* hinv, const int* M, int w, int (&i0)[3],
                                           double (&delta)[3]) {
  const double x = (double)pos3[0], y = (double)pos3[1], z = (double)pos3[2];
#pragma unroll
  for (int d = 0; d < 3; ++d) stencil_1d(frac_coord(x, y, z, hinv, d), M[d], w, i0[d], delta[d]);
}

// Cartesian gradient / force from its components along the fractional coordinates:
// d/dr_e = sum_d (ds_d/dr_e) d/ds_d = sum_d hinv[e][d] d/ds_d
template <class T>
__device__ __forceinline__ void frac_to_cart(const T* hinv, T& a, T& b, T& c) {
  const T x = hinv[0] * a + hinv[1] * b + hinv[2] * c;
  const T y = hinv[3] * a + hinv[4] * b + hinv[5] * c;
  const T z = hinv[6] * a + hinv[7] * b + hinv[8] * c;
  a = x; b = y; c = z;
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
