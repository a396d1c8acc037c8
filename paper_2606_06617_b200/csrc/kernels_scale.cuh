// Device evaluation of the Green multiplier Phi^_p(k) from the fitted panel polynomials (shared by the
// scale kernel over the full half spectrum, kernels_generic.cu, and the band-limited transform kernel,
// kernels_fft.cu).  Theorem 1 (S47)-(S52), "bare transform + smooth correction".
#pragma once
#include "kernels_common.cuh"

namespace pswf {

template <class T>
struct Cplx { T x, y; };

template <class T>
__device__ __forceinline__ T kernel_value(const ScaleParams<T>& P, int slot, T x, T kappa) {
  // x = kappa / c in (0,1)
  int j = min((int)(x * (T)P.panels), P.panels - 1);
  T xi = (T)2 * (x * (T)P.panels - (T)j) - (T)1;
  const T* cf = P.kcoef + ((size_t)slot * P.panels + j) * (P.degree + 1);
  T t = cf[P.degree];
  for (int m = P.degree - 1; m >= 0; --m) t = fma(t, xi, cf[m]);
  T s;
  switch (P.slot_p[slot]) {
    case 1: s = t / (kappa * kappa); break;            // x 4 pi r_c^2      (S47)
    case 2: s = t / kappa; break;                      // x 2 pi^2 r_c      (S48)
    case 3: s = t - log(x); break;                     // x 4 pi            (S49)
    case 4: s = t; break;                              // x pi^2 c / r_c    (S50)
    case 5: s = t + x * x * log(x); break;             // x 2 pi c^2/(3 r_c^2)  (S51)
    default: s = t; break;                             // x pi^2 c^3/(12 r_c^3) (S52)
  }
  return s * P.slot_pre[slot];
}

// d Phi^_p / dk by the derivative of the SAME panel polynomial plus the derivative of the bare factor
// (virial).  x = kappa / c, kappa = k r_c, dx/dk = x_per_k, dkappa/dk = c x_per_k.
template <class T>
__device__ __forceinline__ T kernel_dvalue(const ScaleParams<T>& P, int slot, T x, T kappa) {
  int j = min((int)(x * (T)P.panels), P.panels - 1);
  T xi = (T)2 * (x * (T)P.panels - (T)j) - (T)1;
  const T* cf = P.kcoef + ((size_t)slot * P.panels + j) * (P.degree + 1);
  T t = cf[P.degree], dt = (T)P.degree * cf[P.degree];
  for (int m = P.degree - 1; m >= 1; --m) {
    t = fma(t, xi, cf[m]);
    dt = fma(dt, xi, (T)m * cf[m]);
  }
  t = fma(t, xi, cf[0]);
  dt *= (T)2 * (T)P.panels;            // dT/dx
  const T rc = P.c * P.x_per_k;
  T ds;
  switch (P.slot_p[slot]) {
    case 1: ds = dt * P.x_per_k / (kappa * kappa) - (T)2 * t * rc / (kappa * kappa * kappa); break;
    case 2: ds = dt * P.x_per_k / kappa - t * rc / (kappa * kappa); break;
    case 3: ds = (dt - (T)1 / x) * P.x_per_k; break;
    case 5: ds = (dt + (T)2 * x * log(x) + x) * P.x_per_k; break;
    default: ds = dt * P.x_per_k; break;
  }
  return ds * P.slot_pre[slot];
}

}  // namespace pswf
