// Tiled fp32 spread / gather kernels for sm_100a (default path, w = 8).
//
// Design.  Shared-memory float atomics are CAS loops on sm_100a (ATOMS.CAST.SPIN) and
// a w^3 = 512-point scatter per atom-channel is FMA/issue bound, not HBM bound, so both kernels keep
// the accumulation in REGISTERS and sweep the x dimension with a sliding window:
//
//  * spread ("output-stationary"): a warp owns a 4 x 8 patch of (y,z) grid columns, one column per
//    lane, and walks x; its window acc[8][CB] holds the 8 x-planes an atom in the current stencil
//    plane can touch.  Every atom whose 8 x 8 (y,z) footprint meets the patch is visited (atoms are
//    cell-sorted, so they are 4+7 contiguous runs per plane); a lane multiplies its (wy, wz) by the
//    atom's q and adds wx[a] * that into the window: 8*CB FMAs per lane per atom.  When the window
//    leaves a plane the finished values are stored once, coalesced, with plain stores: no atomics,
//    no zero-fill of the grid, deterministic summation order.
//  * gather ("input-stationary"): a warp owns one stencil-cell column (s_y, s_z) and walks s_x; its
//    window g[8][2][CB] holds the 8 x 8 x 8 grid values an atom of the current cell needs (64 (y,z)
//    offsets = 2 per lane), refreshed by one coalesced plane load per step.  Per atom: Horner weights
//    and derivative weights once (lanes 0..23), x-contraction with value and derivative weights in
//    one pass over the window, then a 9-shuffle transpose-reduce of (phi_a, F) across the warp.
//
// The per-atom panel polynomials are evaluated once per evaluation into 128-byte records
// (wx[8], wy[8], wz[8], s_z, q[C]) that the spread warps read through L1/L2.
#include "kernels_common.cuh"
#include "launch.hpp"

namespace pswf {

namespace {

constexpr int FW = 8;     // window width handled by the fast path
constexpr int PY = 4;     // patch rows (y) per warp
constexpr int PZ = 8;     // patch columns (z) per warp, contiguous in memory
constexpr int GATHER_TX = 32;


// occupancy of each (s_y, s_z) column of stencil cells, from the cell starts (gather skips vacuum)
__global__ void k_colcount(int Mx, int My, int Mz, const int* __restrict__ start, int* __restrict__ colcount) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= My * Mz) return;
  int cnt = 0;
  for (int x = 0; x < Mx; ++x) {
    const size_t k = (size_t)x * My * Mz + col;
    cnt += __ldg(start + k + 1) - __ldg(start + k);
  }
  colcount[col] = cnt;
}

// ------------------------------------------------------------------------------------------------
// gather
// ------------------------------------------------------------------------------------------------
// 9-shuffle transpose-reduce of 8 values over the 32 lanes; on return lane l holds in v[0] the full
// sum of input index  ((l >> 4) & 1) * 4 + ((l >> 3) & 1) * 2 + ((l >> 2) & 1).
__device__ __forceinline__ float reduce8(float (&v)[8], int lane) {
  const bool hi16 = lane & 16;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float send = hi16 ? v[i] : v[i + 4];
    float keep = hi16 ? v[i + 4] : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
  const bool hi8 = lane & 8;
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    float send = hi8 ? v[i] : v[i + 2];
    float keep = hi8 ? v[i + 2] : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
  }
  const bool hi4 = lane & 4;
  {
    float send = hi4 ? v[0] : v[1];
    float keep = hi4 ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2);
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  return v[0];
}

template <int CB>
__global__ void __launch_bounds__(256) k_gather_tiled(int n, int C, int cap, int cb0, int nseg, GridGeom<float> g,
                                                      const int* __restrict__ start,
                                                      const int* __restrict__ colcount,
                                                      const float* __restrict__ sdelta, const float* __restrict__ sq,
                                                      const int* __restrict__ perm, const float* __restrict__ grid,
                                                      float* __restrict__ phi, float* __restrict__ Facc,
                                                      int accumulate_F) {
  __shared__ float s_coef[(kMaxWindowDegree + 1) * FW];
  __shared__ float s_dcoef[kMaxWindowDegree * FW];
  __shared__ __align__(16) float s_w[8][6 * FW];   // per warp: wx, wy, wz, dwx, dwy, dwz of the current atom
  const int Mx = g.M[0], My = g.M[1], Mz = g.M[2];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < (g.wdeg + 1) * FW; i += blockDim.x) s_coef[i] = g.wcoef[i];
  for (int i = threadIdx.x; i < g.wdeg * FW; i += blockDim.x) s_dcoef[i] = g.wdcoef[i];
  __syncthreads();
  // block -> 8 adjacent z columns of one (segment, s_y); warp -> column
  int bid = blockIdx.x;
  const int seg = bid % nseg; bid /= nseg;
  const int nzb = (Mz + 7) / 8;
  const int zb = bid % nzb;
  const int sy = bid / nzb;
  const int sz = zb * 8 + wid;
  if (sz >= Mz || sy >= My) return;
  if (__ldg(colcount + sy * Mz + sz) == 0) return;        // vacuum column: nothing to gather
  const int X0 = seg * GATHER_TX, X1 = min(X0 + GATHER_TX, Mx);
  const size_t Mtot = (size_t)Mx * My * Mz;
  // lane -> 2 (b, c) offsets of the 8 x 8 (y,z) footprint: c = lane & 7, b = (lane >> 3) + 4k
  const int c_off = lane & 7, b0 = lane >> 3;
  int iz = sz + c_off; if (iz >= Mz) iz -= Mz;
  int iy0 = sy + b0;      if (iy0 >= My) iy0 -= My;
  int iy1 = sy + b0 + 4;  if (iy1 >= My) iy1 -= My;
  const size_t col0 = (size_t)iy0 * Mz + iz, col1 = (size_t)iy1 * Mz + iz;
  const size_t plane = (size_t)My * Mz;

  float win[FW][2][CB];
  auto load_plane = [&](int xs, float (&dst)[2][CB]) {
    int x = xs; if (x >= Mx) x -= Mx;
    const float* p0 = grid + (size_t)cb0 * Mtot + (size_t)x * plane;
#pragma unroll
    for (int c = 0; c < CB; ++c) {
      dst[0][c] = __ldg(p0 + (size_t)c * Mtot + col0);
      dst[1][c] = __ldg(p0 + (size_t)c * Mtot + col1);
    }
  };
  // warm-up: planes X0 .. X0+6 go to slots (X0 + a) % 8 = a (X0 is a multiple of 8)
#pragma unroll
  for (int a = 0; a < FW - 1; ++a) load_plane(X0 + a, win[a]);

  for (int s0 = X0; s0 < X1; s0 += FW) {
#pragma unroll
    for (int u = 0; u < FW; ++u) {
      const int sx = s0 + u;
      if (sx < X1) {
        load_plane(sx + FW - 1, win[(u + FW - 1) % FW]);
        const int key = (sx * My + sy) * Mz + sz;
        const int jlo = __ldg(start + key), jhi = __ldg(start + key + 1);
        for (int j = jlo; j < jhi; ++j) {
          // weights and derivative weights of atom j: lanes 0..23, one panel each
          if (lane < 3 * FW) {
            const int d = lane >> 3, tt = lane & 7;
            const float xi = 2.f * __ldg(sdelta + (size_t)d * cap + j) - 1.f;
            float v = s_coef[g.wdeg * FW + tt];
            float dv = s_dcoef[(g.wdeg - 1) * FW + tt];
            for (int m = g.wdeg - 1; m >= 1; --m) {
              v = fmaf(v, xi, s_coef[m * FW + tt]);
              dv = fmaf(dv, xi, s_dcoef[(m - 1) * FW + tt]);
            }
            v = fmaf(v, xi, s_coef[tt]);
            s_w[wid][lane] = v;
            s_w[wid][3 * FW + lane] = dv * g.dxi_dr[d];
          }
          __syncwarp();
          const float4 xa = *reinterpret_cast<const float4*>(&s_w[wid][0]);
          const float4 xb = *reinterpret_cast<const float4*>(&s_w[wid][4]);
          const float4 da = *reinterpret_cast<const float4*>(&s_w[wid][3 * FW]);
          const float4 db = *reinterpret_cast<const float4*>(&s_w[wid][3 * FW + 4]);
          const float wx[FW] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
          const float dx[FW] = {da.x, da.y, da.z, da.w, db.x, db.y, db.z, db.w};
          const float wz = s_w[wid][2 * FW + c_off], dz = s_w[wid][5 * FW + c_off];
          const float wy0 = s_w[wid][FW + b0], wy1 = s_w[wid][FW + b0 + 4];
          const float dy0 = s_w[wid][4 * FW + b0], dy1 = s_w[wid][4 * FW + b0 + 4];
          __syncwarp();
          const float yz[2] = {wy0 * wz, wy1 * wz};
          const float dyz[2] = {dy0 * wz, dy1 * wz};
          const float ydz[2] = {wy0 * dz, wy1 * dz};
          float red[8];
          float fx = 0.f, fy = 0.f, fz = 0.f;
#pragma unroll
          for (int c = 0; c < CB; ++c) {
            float val = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
#pragma unroll
            for (int k = 0; k < 2; ++k) {
              float S0 = 0.f, S1 = 0.f;
#pragma unroll
              for (int a = 0; a < FW; ++a) {
                const float gv = win[(u + a) % FW][k][c];
                S0 = fmaf(wx[a], gv, S0);
                S1 = fmaf(dx[a], gv, S1);
              }
              val = fmaf(yz[k], S0, val);
              gx = fmaf(yz[k], S1, gx);
              gy = fmaf(dyz[k], S0, gy);
              gz = fmaf(ydz[k], S0, gz);
            }
            const float qc = (cb0 + c < C) ? __ldg(sq + (size_t)(cb0 + c) * cap + j) : 0.f;
            fx = fmaf(-qc, gx, fx);
            fy = fmaf(-qc, gy, fy);
            fz = fmaf(-qc, gz, fz);
            red[c] = val;
          }
#pragma unroll
          for (int c = CB; c < 4; ++c) red[c] = 0.f;
          red[4] = fx; red[5] = fy; red[6] = fz; red[7] = 0.f;
          const float tot = reduce8(red, lane);
          // lane l (with (l & 3) == 0) holds output index (l>>4)*4 + ((l>>3)&1)*2 + ((l>>2)&1)
          if ((lane & 3) == 0) {
            const int idx = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
            const int dst = __ldg(perm + j);
            if (idx < CB) {
              if (phi && cb0 + idx < C) phi[(size_t)(cb0 + idx) * n + dst] = tot;
            } else if (idx >= 4 && idx < 7 && Facc) {
              float* fp = Facc + 3 * (size_t)dst + (idx - 4);
              *fp = accumulate_F ? (*fp + tot) : tot;
            }
          }
        }
      }
    }
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
bool fast_path_supported(const pswf_lr_plan* p) {
  if (p->precision != PSWF_LR_F32 || p->w != FW) return false;
  for (int d = 0; d < 3; ++d)
    if (p->M[d] < 2 * FW + 8) return false;     // unambiguous periodic offsets inside a patch
  if (p->M[0] % FW != 0) return false;          // x segments start on multiples of 8
  return true;
}

void launch_fast_prepare(pswf_lr_plan* p, int n, const float*, const float*, const GridGeom<float>&,
                         cudaStream_t st) {
  (void)n;
  const int ncol = p->M[1] * p->M[2];
  k_colcount<<<(ncol + 255) / 256, 256, 0, st>>>(p->M[0], p->M[1], p->M[2], p->d_count, p->d_colcount);
}

void launch_fast_gather(pswf_lr_plan* p, int n, const GridGeom<float>& g, float* phi, float* F, cudaStream_t st) {
  if (n <= 0) return;
  const int Mx = p->M[0], My = p->M[1], Mz = p->M[2];
  const int nseg = (Mx + GATHER_TX - 1) / GATHER_TX;
  const unsigned blocks = (unsigned)(nseg * ((Mz + 7) / 8) * My);
  int cb0 = 0;
  int pass = 0;
  while (cb0 < p->C) {
    const int left = p->C - cb0;
    const int acc = pass > 0 ? 1 : 0;
#define PSWF_GATHER(CBV)                                                                                      \
  k_gather_tiled<CBV><<<blocks, 256, 0, st>>>(n, p->C, p->cap_atoms, cb0, nseg, g, p->d_count, p->d_colcount, \
                                              (const float*)p->d_sdelta, (const float*)p->d_sq, p->d_perm,    \
                                              (const float*)p->d_grid, phi, F, acc)
    if (left >= 4) { PSWF_GATHER(4); cb0 += 4; }
    else if (left == 3) { PSWF_GATHER(3); cb0 += 3; }
    else if (left == 2) { PSWF_GATHER(2); cb0 += 2; }
    else { PSWF_GATHER(1); cb0 += 1; }
#undef PSWF_GATHER
    ++pass;
  }
}

}  // namespace pswf
