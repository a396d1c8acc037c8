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
// the sorted arrays (two when the z range wraps).  One warp per sorted atom, all channels; each
// distinct exponent's polynomial is evaluated once per pair and shared by its channels.
// Requirement (host-checked): r_c < half the distance between opposite cell faces (minimum image; L_d / 2 in
// an orthorhombic box).  Cell search radius R_d = floor(r_c / h_d) + 1 with h_d the distance between
// neighbouring grid planes; a dimension with 2 R_d + 1 >= M_d is searched whole.  General cells (R-cell,
// DESIGN.md §2): fractional coordinates, minimum image there, converted with the lattice vectors.
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
  if (g.tri) {   // wrapped fractional coordinates
    const double r[3] = {(double)pos[3 * (size_t)i], (double)pos[3 * (size_t)i + 1], (double)pos[3 * (size_t)i + 2]};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double s = r[0] * g.hinv[d] + r[1] * g.hinv[3 + d] + r[2] * g.hinv[6 + d];
      s -= floor(s);
      if (s >= 1.0) s = 0.0;
      spos[(size_t)d * cap + j] = (T)s;
    }
    return;
  }
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double s = (double)pos[3 * (size_t)i + d] * g.invL[d];
    s -= floor(s);
    if (s >= 1.0) s = 0.0;
    spos[(size_t)d * cap + j] = (T)(s * g.L[d]);
  }
}

// One warp per sorted atom, lanes <-> candidate cell rows, accepted pairs COMPACTED.
// The (dx, dy) cell rows around the atom are dealt to the lanes 32 at a time; every lane tests the
// atoms of its row's z run against r_c (a cheap step at full lane occupancy), accepted neighbours go
// to a per-warp queue in shared memory (ballot + popc), and whenever 32 are queued all lanes evaluate
// one pair each -- the polynomial work runs with full warps instead of the ~38% of the lanes that a
// test-and-evaluate loop keeps busy.
template <class T, int CT>
__global__ void __launch_bounds__(128) k_real_pairs_q(int n, int C, int cap, RealGeom<T> g, RealParams<T> P,
                                                       const int* __restrict__ start, const int* __restrict__ si0,
                                                       const T* __restrict__ spos, const T* __restrict__ sq,
                                                       const int* __restrict__ perm, double* __restrict__ Eacc,
                                                       T* __restrict__ phi, T* __restrict__ F, int accumulate,
                                                       double* __restrict__ Wacc) {
  __shared__ double s_E;
  __shared__ double s_W[6];
  __shared__ int s_qk[4][64];        // queue of accepted neighbour indices, one ring per warp
  __shared__ T s_qd[4][64][4];       // their minimum-image displacement and r^2
  extern __shared__ __align__(16) unsigned char s_raw[];
  T* s_cf = reinterpret_cast<T*>(s_raw);
  T* s_df = s_cf + P.nslots * P.panels * (P.degree + 1);
  for (int t = threadIdx.x; t < P.nslots * P.panels * (P.degree + 1); t += blockDim.x) s_cf[t] = P.coef[t];
  for (int t = threadIdx.x; t < P.nslots * P.panels * P.degree; t += blockDim.x) s_df[t] = P.dcoef[t];
  if (threadIdx.x == 0) s_E = 0.0;
  if (threadIdx.x < 6) s_W[threadIdx.x] = 0.0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int j = blockIdx.x * 4 + wid;
  double e_thread = 0.0;
  T wv[6] = {0, 0, 0, 0, 0, 0};   // virial of this lane's pairs: -1/2 sum qq L'(r) d_a d_b / r (each pair is visited twice)
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
    const int nx = min(2 * g.R[0] + 1, Mx), ny = min(2 * g.R[1] + 1, My);
    const int x0 = nx == Mx ? 0 : cx - g.R[0], y0 = ny == My ? 0 : cy - g.R[1];
    const bool allz = 2 * g.R[2] + 1 >= Mz;
    int qhead = 0, qcount = 0;   // warp-uniform
    int* qk = s_qk[wid];
    T (*qd)[4] = s_qd[wid];

    // one accepted pair per lane: polynomial evaluation and accumulation
    auto evaluate = [&](int k, T ddx, T ddy, T ddz, T r2) {
      const T rr = sqrt(r2);
      const T x = rr * P.inv_rc;
      const int pj = min((int)(x * (T)P.panels), P.panels - 1);
      const T xi = (T)2 * (x * (T)P.panels - (T)pj) - (T)1;
      const T invx = (T)1 / x;
      T Lval[kMaxSlots], dL[kMaxSlots];
#pragma unroll
      for (int s = 0; s < kMaxSlots; ++s) {
        if (s >= P.nslots) break;
        const T* cf = s_cf + (s * P.panels + pj) * (P.degree + 1);
        const T* df = s_df + (s * P.panels + pj) * P.degree;
        T N = cf[P.degree], dN = df[P.degree - 1];
        for (int m = P.degree - 1; m >= 1; --m) { N = fma(N, xi, cf[m]); dN = fma(dN, xi, df[m - 1]); }
        N = fma(N, xi, cf[0]);
        T ip = invx;
        for (int e = 1; e < P.slot_p[s]; ++e) ip *= invx;
        Lval[s] = P.slot_pre[s] * N * ip;
        dL[s] = P.slot_pre[s] * P.inv_rc * (dN * ip - (T)P.slot_p[s] * N * ip * invx);
      }
      T fs = 0;
#pragma unroll
      for (int a = 0; a < CT; ++a) {
        if (a < C) {
          const T qk_ = sq[(size_t)a * cap + k];
          const int s = P.chan_slot[a];
          ph[a] = fma(qk_, Lval[s], ph[a]);
          fs = fma(qj[a] * qk_, dL[s], fs);
        }
      }
      const T sc = fs / rr;
      fx = fma(sc, ddx, fx);
      fy = fma(sc, ddy, fy);
      fz = fma(sc, ddz, fz);
      if (Wacc) {
        const T hs = (T)-0.5 * sc;
        wv[0] = fma(hs * ddx, ddx, wv[0]); wv[1] = fma(hs * ddy, ddy, wv[1]); wv[2] = fma(hs * ddz, ddz, wv[2]);
        wv[3] = fma(hs * ddx, ddy, wv[3]); wv[4] = fma(hs * ddx, ddz, wv[4]); wv[5] = fma(hs * ddy, ddz, wv[5]);
      }
    };
    auto drain = [&](int m) {   // the first m (<= 32) queued pairs, one per lane
      __syncwarp();
      if (lane < m) {
        const int e = (qhead + lane) & 63;
        evaluate(qk[e], qd[e][0], qd[e][1], qd[e][2], qd[e][3]);
      }
      __syncwarp();
      qhead = (qhead + m) & 63;
      qcount -= m;
    };

    const int nrows = nx * ny;
    for (int rb = 0; rb < nrows; rb += 32) {
      // this lane's row and its (up to two) z runs
      int k0 = 0, k1 = 0, k2 = 0, k3 = 0;
      const int ri = rb + lane;
      if (ri < nrows) {
        const int dx = ri / ny, dy = ri - dx * ny;
        const T ax = nx == Mx ? (T)0 : (T)max(abs(dx - g.R[0]) - 1, 0) * g.h[0];
        const T ay = ny == My ? (T)0 : (T)max(abs(dy - g.R[1]) - 1, 0) * g.h[1];
        // orthorhombic: the per-axis lower bounds add in quadrature; general cell: each bounds |r| on its own
        // (|r| >= |ds_d| x plane distance), so a row is dropped only when one of them reaches r_c
        const T rem2 = g.tri ? (ax < P.r_c && ay < P.r_c ? rc2 : (T)0) : rc2 - ax * ax - ay * ay;
        if (rem2 > (T)0) {
          const int Rz = g.tri ? g.R[2] : min(g.R[2], (int)(sqrt(rem2) * g.inv_hz) + 1);
          const int* row = start + ((size_t)wrap_index(x0 + dx, Mx) * My + wrap_index(y0 + dy, My)) * Mz;
          int z0 = allz ? 0 : cz - Rz, z1 = allz ? Mz : cz + Rz + 1;
          if (z0 < 0) { k2 = row[z0 + Mz]; k3 = row[Mz]; z0 = 0; }
          if (z1 > Mz) { k2 = row[0]; k3 = row[z1 - Mz]; z1 = Mz; }
          k0 = row[z0]; k1 = row[z1];
        }
      }
      // lockstep over the run positions: test, compact, evaluate when a warp's worth is queued
      for (int seg = 0; seg < 2; ++seg) {
        int k = seg == 0 ? k0 : k2;
        const int kend = seg == 0 ? k1 : k3;
        while (__any_sync(0xffffffffu, k < kend)) {
          bool acc = false;
          T ddx = 0, ddy = 0, ddz = 0, r2 = 0;
          if (k < kend && k != j) {
            ddx = spos[k] - xj; ddy = spos[(size_t)cap + k] - yj; ddz = spos[2 * (size_t)cap + k] - zj;
            if (g.tri) {
              const T sx = ddx - rint(ddx), sy = ddy - rint(ddy), sz = ddz - rint(ddz);
              ddx = sx * g.hm[0] + sy * g.hm[3] + sz * g.hm[6];
              ddy = sx * g.hm[1] + sy * g.hm[4] + sz * g.hm[7];
              ddz = sx * g.hm[2] + sy * g.hm[5] + sz * g.hm[8];
            } else {
              ddx -= g.L[0] * rint(ddx * (T)g.invL[0]);
              ddy -= g.L[1] * rint(ddy * (T)g.invL[1]);
              ddz -= g.L[2] * rint(ddz * (T)g.invL[2]);
            }
            r2 = ddx * ddx + ddy * ddy + ddz * ddz;
            acc = r2 < rc2 && r2 > (T)0;
          }
          const unsigned m = __ballot_sync(0xffffffffu, acc);
          if (acc) {
            const int e = (qhead + qcount + __popc(m & ((1u << lane) - 1u))) & 63;
            qk[e] = k;
            qd[e][0] = ddx; qd[e][1] = ddy; qd[e][2] = ddz; qd[e][3] = r2;
          }
          qcount += __popc(m);
          if (qcount >= 32) drain(32);
          ++k;
        }
      }
    }
    if (qcount > 0) drain(qcount);
    fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
#pragma unroll
    for (int a = 0; a < CT; ++a) ph[a] = warp_sum(ph[a]);
    if (lane == 0) {
      const int dst = perm[j];
#pragma unroll
      for (int a = 0; a < CT; ++a) {
        if (a < C) {
          const T pa = ph[a] - P.self_pre[a] * qj[a];
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
  if (Wacc) {
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      const double t = warp_sum((double)wv[i]);
      if ((threadIdx.x & 31) == 0 && t != 0.0) atomicAdd(&s_W[i], t);
    }
  }
  __syncthreads();
  if (threadIdx.x == 0 && s_E != 0.0) atomicAdd(Eacc, s_E);
  if (Wacc && threadIdx.x < 6 && s_W[threadIdx.x] != 0.0) atomicAdd(&Wacc[threadIdx.x], s_W[threadIdx.x]);
}

__global__ void k_real_finalize(const double* __restrict__ Eacc, double* __restrict__ E, int accumulate) {
  if (threadIdx.x == 0 && blockIdx.x == 0) *E = accumulate ? *E + *Eacc : *Eacc;
}

}  // namespace

template <class T>
void launch_real_space(pswf_lr_plan* p, int n, const T* pos, const RealGeom<T>& g, const RealParams<T>& P, double* E,
                       T* phi, T* F, int accumulate, cudaStream_t st) {
  cudaMemsetAsync(p->d_Ereal, 0, sizeof(double), st);
  p->n_memsets += 1;
  p->n_kernels += (n > 0 ? 2 : 0) + (E ? 1 : 0);
  // virial: added to the plan's accumulator when accumulate is set (after pswf_lr_execute), else restarted
  double* wacc = p->virial ? p->d_virial : nullptr;
  if (wacc && !accumulate) cudaMemsetAsync(wacc, 0, sizeof(double) * 6, st);
  if (n > 0) {
    k_sorted_pos<T><<<(n + 255) / 256, 256, 0, st>>>(n, p->cap_atoms, pos, p->d_perm, g, (T*)p->d_spos);
    const size_t tb = sizeof(T) * (size_t)P.nslots * P.panels * (2 * P.degree + 1);   // <= 6 * 32 * 49 * 8 = 75 KB
#define PSWF_REAL(CTV)                                                                                          \
  cudaFuncSetAttribute(k_real_pairs_q<T, CTV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tb);            \
  k_real_pairs_q<T, CTV><<<(n + 3) / 4, 128, tb, st>>>(n, p->C, p->cap_atoms, g, P, p->d_count, p->d_si0,        \
                                                        (const T*)p->d_spos, (const T*)p->d_sq, p->d_perm,        \
                                                        p->d_Ereal, phi, F, accumulate, wacc)
    if (p->C <= 4) { PSWF_REAL(4); }
    else if (p->C <= 8) { PSWF_REAL(8); }
    else { PSWF_REAL(kMaxChannels); }
#undef PSWF_REAL
  }
  if (E) k_real_finalize<<<1, 32, 0, st>>>(p->d_Ereal, E, accumulate);
}

template void launch_real_space<float>(pswf_lr_plan*, int, const float*, const RealGeom<float>&,
                                       const RealParams<float>&, double*, float*, float*, int, cudaStream_t);
template void launch_real_space<double>(pswf_lr_plan*, int, const double*, const RealGeom<double>&,
                                        const RealParams<double>&, double*, double*, double*, int, cudaStream_t);

}  // namespace pswf
