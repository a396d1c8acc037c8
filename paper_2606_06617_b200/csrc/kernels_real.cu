// Real-space complement and self term of the PSWF-mollified inverse-power channels (SURVEY.md
// §8(f) row 1): the part of (S65), that the reciprocal path does not contain,
//     E_real = 1/2 sum_a sum_{i != j, images} q_i^a q_j^a L_{p_a,r_c}(|r_ij|),
//     E_self = sum_a S_{p_a}(0) sum_i (q_i^a)^2 / (2 r_c^p_a)                 (S66),
// with L_{p,r_c}(r) = r_c^-p N_p(x) / x^p for x = r / r_c < 1 and 0 beyond (the complement is
// compactly supported).  N_p and dN_p/dx are Horner piecewise polynomials
// (real_tables.hpp).  The kernel returns E_real - E_self, the per-atom potentials
// phi_i^a = dE/dq_i^a and the forces F_i = -dE/dr_i, optionally ADDED to the reciprocal results.
//
// It reuses the reciprocal path's cell sort: atoms are ordered by stencil cell (z fastest), so the
// neighbours of an atom within r_c are, for every (dx, dy) cell-row offset, one contiguous run of
// the sorted arrays (two when the z range wraps).  One thread per sorted atom, all channels; each
// distinct exponent's polynomial is evaluated once per pair and shared by its channels.
// Requirement (host-checked): r_c < L_d / 2 (minimum image).  Cell search radius
// R_d = floor(r_c / h_d) + 1; a dimension with 2 R_d + 1 >= M_d is searched whole.
#include "kernels_common.cuh"
#include "launch.hpp"

namespace pswf {

namespace {

// wrapped position of sorted atom j (float or double), SoA [3][cap]
template <class T>
__global__ void __launch_bounds__(256) k_sorted_pos(int n, int cap, const T* __restrict__ pos,
                                                     const int* __restrict__ perm, RealGeom<T> g,
                                                     T* __restrict__ spos) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const int i = perm[j];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double s = (double)pos[3 * (size_t)i + d] * g.invL[d];
    s -= floor(s);
    if (s >= 1.0) s = 0.0;
    spos[(size_t)d * cap + j] = (T)(s * g.L[d]);
  }
}

template <class T, int CT, int LPA>   // CT = channel capacity (register arrays); LPA = lanes per atom, 32 or 1
__global__ void __launch_bounds__(128) k_real_pairs(int n, int C, int cap, RealGeom<T> g, RealParams<T> P,
                                                     const int* __restrict__ start, const int* __restrict__ si0,
                                                     const T* __restrict__ spos, const T* __restrict__ sq,
                                                     const int* __restrict__ perm, double* __restrict__ Eacc,
                                                     T* __restrict__ phi, T* __restrict__ F, int accumulate) {
  __shared__ double s_E;
  extern __shared__ __align__(16) unsigned char s_raw[];   // numerator tables: [slot][panel][degree+1] | [..][degree]
  T* s_cf = reinterpret_cast<T*>(s_raw);
  T* s_df = s_cf + P.nslots * P.panels * (P.degree + 1);
  for (int t = threadIdx.x; t < P.nslots * P.panels * (P.degree + 1); t += blockDim.x) s_cf[t] = P.coef[t];
  for (int t = threadIdx.x; t < P.nslots * P.panels * P.degree; t += blockDim.x) s_df[t] = P.dcoef[t];
  if (threadIdx.x == 0) s_E = 0.0;
  __syncthreads();
  // LPA = 32 (small systems: more parallelism): one WARP per sorted atom j, the lanes stride over each
  // contiguous run of neighbour candidates and the warp reduces their contributions at the end;
  // LPA = 1 (large systems, short runs): one thread per atom
  const int lane = LPA == 32 ? (threadIdx.x & 31) : 0;
  const int j = LPA == 32 ? blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5) : blockIdx.x * blockDim.x + threadIdx.x;
  double e_thread = 0.0;
  if (j < n) {
    const int Mx = g.M[0], My = g.M[1], Mz = g.M[2];
    const int cx = wrap_index(si0[j], Mx), cy = wrap_index(si0[(size_t)cap + j], My),
              cz = wrap_index(si0[2 * (size_t)cap + j], Mz);
    const T xj = spos[j], yj = spos[(size_t)cap + j], zj = spos[2 * (size_t)cap + j];
    T qj[CT], ph[CT];
#pragma unroll
    for (int a = 0; a < CT; ++a) { qj[a] = a < C ? sq[(size_t)a * cap + j] : (T)0; ph[a] = (T)0; }
    T fx = 0, fy = 0, fz = 0;
    const T rc2 = P.r_c * P.r_c;
    // cells within R_d of the atom's own, every cell once: when 2 R_d + 1 >= M_d the whole dimension
    const int nx = min(2 * g.R[0] + 1, Mx), ny = min(2 * g.R[1] + 1, My);
    const int x0 = nx == Mx ? 0 : cx - g.R[0], y0 = ny == My ? 0 : cy - g.R[1];
    const bool allz = 2 * g.R[2] + 1 >= Mz;
    for (int dx = 0; dx < nx; ++dx) {
      const int ix = wrap_index(x0 + dx, Mx);
      // prune rows and z ranges that cannot reach r_c: cells k offsets apart are at least (k - 1) h apart
      const T ax = nx == Mx ? (T)0 : (T)max(abs(dx - g.R[0]) - 1, 0) * g.h[0];
      for (int dy = 0; dy < ny; ++dy) {
        const int iy = wrap_index(y0 + dy, My);
        const T ay = ny == My ? (T)0 : (T)max(abs(dy - g.R[1]) - 1, 0) * g.h[1];
        const T rem2 = rc2 - ax * ax - ay * ay;
        if (rem2 <= (T)0) continue;
        const int Rz = min(g.R[2], (int)(sqrt(rem2) * g.inv_hz) + 1);
        const int* row = start + ((size_t)ix * My + iy) * Mz;
        // cells cz - Rz .. cz + Rz (mod Mz): one run, or two when the range wraps
        int z0 = allz ? 0 : cz - Rz, z1 = allz ? Mz : cz + Rz + 1;   // [z0, z1)
        int runs[2][2];
        int nr = 0;
        if (z0 < 0) { runs[nr][0] = row[z0 + Mz]; runs[nr][1] = row[Mz]; ++nr; z0 = 0; }
        if (z1 > Mz) { runs[nr][0] = row[0]; runs[nr][1] = row[z1 - Mz]; ++nr; z1 = Mz; }
        runs[nr][0] = row[z0]; runs[nr][1] = row[z1]; ++nr;
        for (int r = 0; r < nr; ++r)
          for (int k = runs[r][0] + lane; k < runs[r][1]; k += LPA) {
            if (k == j) continue;
            T ddx = spos[k] - xj, ddy = spos[(size_t)cap + k] - yj, ddz = spos[2 * (size_t)cap + k] - zj;
            ddx -= g.L[0] * rint(ddx * (T)g.invL[0]);   // minimum image (r_c < L/2)
            ddy -= g.L[1] * rint(ddy * (T)g.invL[1]);
            ddz -= g.L[2] * rint(ddz * (T)g.invL[2]);
            const T r2 = ddx * ddx + ddy * ddy + ddz * ddz;
            if (!(r2 < rc2) || r2 <= (T)0) continue;
            const T rr = sqrt(r2);
            const T x = rr * P.inv_rc;
            int pj = min((int)(x * (T)P.panels), P.panels - 1);
            const T xi = (T)2 * (x * (T)P.panels - (T)pj) - (T)1;
            const T invx = (T)1 / x;
            T Lval[6], dL[6];   // per distinct exponent: L(r) and dL/dr
#pragma unroll
            for (int s = 0; s < 6; ++s) {
              if (s >= P.nslots) break;
              const T* cf = s_cf + (s * P.panels + pj) * (P.degree + 1);
              const T* df = s_df + (s * P.panels + pj) * P.degree;
              T N = cf[P.degree], dN = df[P.degree - 1];
              for (int m = P.degree - 1; m >= 1; --m) { N = fma(N, xi, cf[m]); dN = fma(dN, xi, df[m - 1]); }
              N = fma(N, xi, cf[0]);
              T ip = invx;                       // x^-p
              for (int e = 1; e < P.slot_p[s]; ++e) ip *= invx;
              Lval[s] = P.slot_pre[s] * N * ip;                                          // r_c^-p N x^-p
              dL[s] = P.slot_pre[s] * P.inv_rc * (dN * ip - (T)P.slot_p[s] * N * ip * invx);
            }
            T fs = 0;   // sum_a q_j^a q_k^a dL/dr
#pragma unroll
            for (int a = 0; a < CT; ++a) {
              if (a < C) {
                const T qk = sq[(size_t)a * cap + k];
                const int s = P.chan_slot[a];
                ph[a] = fma(qk, Lval[s], ph[a]);
                fs = fma(qj[a] * qk, dL[s], fs);
              }
            }
            const T sc = fs / rr;   // F_j = + sum qq L'(r) (r_k - r_j) / r
            fx = fma(sc, ddx, fx);
            fy = fma(sc, ddy, fy);
            fz = fma(sc, ddz, fz);
          }
      }
    }
    if (LPA == 32) {
      fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
#pragma unroll
      for (int a = 0; a < CT; ++a) ph[a] = warp_sum(ph[a]);
    }
    if (lane == 0) {
      const int dst = perm[j];
#pragma unroll
      for (int a = 0; a < CT; ++a) {
        if (a < C) {
          const T pa = ph[a] - P.self_pre[a] * qj[a];   // self term: phi_self = -S_p(0) q / r_c^p
          e_thread += 0.5 * (double)qj[a] * (double)pa;
          if (phi) {
            T* o = phi + (size_t)a * n + dst;
            *o = accumulate ? *o + pa : pa;
          }
        }
      }
      if (F) {
        T* o = F + 3 * (size_t)dst;
        if (accumulate) { o[0] += fx; o[1] += fy; o[2] += fz; }
        else { o[0] = fx; o[1] = fy; o[2] = fz; }
      }
    }
  }
  e_thread = warp_sum(e_thread);
  if ((threadIdx.x & 31) == 0 && e_thread != 0.0) atomicAdd(&s_E, e_thread);
  __syncthreads();
  if (threadIdx.x == 0 && s_E != 0.0) atomicAdd(Eacc, s_E);
}

__global__ void k_real_finalize(const double* __restrict__ Eacc, double* __restrict__ E, int accumulate) {
  if (threadIdx.x == 0 && blockIdx.x == 0) *E = accumulate ? *E + *Eacc : *Eacc;
}

}  // namespace

template <class T>
void launch_real_space(pswf_lr_plan* p, int n, const T* pos, const RealGeom<T>& g, const RealParams<T>& P, double* E,
                       T* phi, T* F, int accumulate, cudaStream_t st) {
  cudaMemsetAsync(p->d_Ereal, 0, sizeof(double), st);
  if (n > 0) {
    k_sorted_pos<T><<<(n + 255) / 256, 256, 0, st>>>(n, p->cap_atoms, pos, p->d_perm, g, (T*)p->d_spos);
    const size_t tb = sizeof(T) * (size_t)P.nslots * P.panels * (2 * P.degree + 1);   // <= 6 * 32 * 49 * 8 = 75 KB
#define PSWF_REAL_L(CTV, LPAV, NB)                                                                              \
  cudaFuncSetAttribute(k_real_pairs<T, CTV, LPAV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tb);       \
  k_real_pairs<T, CTV, LPAV><<<NB, 128, tb, st>>>(n, p->C, p->cap_atoms, g, P, p->d_count, p->d_si0,            \
                                                  (const T*)p->d_spos, (const T*)p->d_sq, p->d_perm,            \
                                                  p->d_Ereal, phi, F, accumulate)
#define PSWF_REAL(CTV)                                        \
  if (n < 65536) { PSWF_REAL_L(CTV, 32, (n + 3) / 4); }       \
  else { PSWF_REAL_L(CTV, 1, (n + 127) / 128); }
    if (p->C <= 4) { PSWF_REAL(4); }
    else if (p->C <= 8) { PSWF_REAL(8); }
    else { PSWF_REAL(kMaxChannels); }
#undef PSWF_REAL
#undef PSWF_REAL_L
  }
  if (E) k_real_finalize<<<1, 32, 0, st>>>(p->d_Ereal, E, accumulate);
}

template void launch_real_space<float>(pswf_lr_plan*, int, const float*, const RealGeom<float>&,
                                       const RealParams<float>&, double*, float*, float*, int, cudaStream_t);
template void launch_real_space<double>(pswf_lr_plan*, int, const double*, const RealGeom<double>&,
                                        const RealParams<double>&, double*, double*, double*, int, cudaStream_t);

}  // namespace pswf
