// Fast fp32 gather + force kernel for sm_100a (a5; default path, w <= 8).
//
// phi_i^a = sum_g W(x_g - r_i) phi_g^a,  grad phi_i^a = sum_g grad_{r_i} W(x_g - r_i) phi_g^a  (the
// derivative of the SAME panel polynomials),  F_i = - sum_a q_i^a grad phi_i^a.
// 4 w^3 C flops per atom and ~0.5 atoms per grid cell: bound by FP32 issue, not by HBM.
//
// Design: INPUT-STATIONARY IN REGISTERS, one warp per column of stencil cells.
//  * a warp owns the cells (s_x, s_y, s_z), s_x in one x segment, of one (s_y, s_z) column.  Every
//    atom of those cells reads the same 8 x 8 (y,z) footprint, two points per lane, so all 32 lanes
//    work on every atom and the per-atom sums are a warp shuffle reduction (no atomics);
//  * the 8 x-planes an atom can touch live in a register window win[8][2][CB]; slot k holds the plane
//    x == k (mod 8).  The per-atom weight records written by k_scatter_records hold wx and dwx/dx
//    ROTATED by the atom's cell index mod 8, so the x contraction is sum_k wxr[k] * win[k] with static
//    register indices: one copy of the atom code, no unrolled window rotation (the first tiled
//    kernel's 118 KB of SASS thrashed the instruction cache, profiles/r1a);
//  * the potential grid is first copied from cuFFT's planar layout [C][M] into a channel-interleaved
//    one [M][CB] (k_interleave, L2-resident, ~10 us), so that one 16-byte load per footprint point
//    refreshes the slot that left the window for all channels (with planar loads the address
//    arithmetic of 8 scalar loads per x step was a third of all instructions, profiles/r1c);
//    the loads are served by L1: neighbouring columns of the CTA share 7/8 of their footprint;
//  * the lanes of a segment fetch the cell boundaries of its 32 cells at once, prefetch the
//    records of the non-empty cells to L2, skip leading / trailing empty cells and return at once
//    when the segment holds no atoms (vacuum of configuration 5);
//  * per atom: x contraction with value and derivative weights in one pass (2 x 8 x 2 FFMA per
//    channel per lane), combination with the (y,z) weights, 9-shuffle transpose-reduce of
//    (phi_a, F_x, F_y, F_z), scattered store to the caller's atom order.
#include "kernels_common.cuh"
#include "launch.hpp"

namespace pswf {

namespace {

constexpr int SW = 8;        // stencil slots per dimension
constexpr int XSEG = 32;     // cells per x segment: one lane per cell boundary pair
constexpr int GBY = 2, GBZ = 4;   // cell columns per CTA (y x z): 8 warps

template <int CB> struct VecOf;
template <> struct VecOf<1> { using type = float; };
template <> struct VecOf<2> { using type = float2; };
template <> struct VecOf<4> { using type = float4; };

template <int CB>
__device__ __forceinline__ void unpack(const typename VecOf<CB>::type& v, float (&o)[CB]) {
  if constexpr (CB == 1) { o[0] = v; }
  else if constexpr (CB == 2) { o[0] = v.x; o[1] = v.y; }
  else { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
}

// planar [C][M] -> interleaved [M][CB] for the channels cb0 .. cb0+CB-1 (missing channels read as 0)
template <int CB>
__global__ void __launch_bounds__(256) k_interleave(size_t Mtot, int nch, const float* __restrict__ planar,
                                                    typename VecOf<CB>::type* __restrict__ out) {
  const size_t m = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= Mtot) return;
  float v[CB];
#pragma unroll
  for (int c = 0; c < CB; ++c) v[c] = c < nch ? __ldg(planar + (size_t)c * Mtot + m) : 0.f;
  if constexpr (CB == 1) out[m] = v[0];
  else if constexpr (CB == 2) out[m] = make_float2(v[0], v[1]);
  else out[m] = make_float4(v[0], v[1], v[2], v[3]);
}

// 9-shuffle transpose-reduce of 8 values over the 32 lanes; on return lane l holds in v[0] the full
// sum of input index  ((l >> 4) & 1) * 4 + ((l >> 3) & 1) * 2 + ((l >> 2) & 1).
__device__ __forceinline__ float reduce8(float (&v)[8], int lane) {
  const bool hi16 = lane & 16;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float send = hi16 ? v[i] : v[i + 4];
    const float keep = hi16 ? v[i + 4] : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
  const bool hi8 = lane & 8;
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const float send = hi8 ? v[i] : v[i + 2];
    const float keep = hi8 ? v[i + 2] : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
  }
  const bool hi4 = lane & 4;
  {
    const float send = hi4 ? v[0] : v[1];
    const float keep = hi4 ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2);
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  return v[0];
}

__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

template <int CB>
__global__ void __launch_bounds__(32 * GBY * GBZ, 2)
    k_gather_cols(int n, int C, int cb0, int Mx, int My, int Mz, int nseg, int nby, int nbz, int recf,
                  const int* __restrict__ start, const float* __restrict__ rec, const float* __restrict__ drec,
                  const int* __restrict__ perm, const typename VecOf<CB>::type* __restrict__ gridi,
                  float* __restrict__ phi, float* __restrict__ Facc, int accumulate_F) {
  using V = typename VecOf<CB>::type;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // block -> (segment, y block, z block); consecutive blocks walk z, then y: CTAs resident on an SM
  // at the same time share most of their footprints in L1
  int bid = blockIdx.x;
  const int bz = bid % nbz; bid /= nbz;
  const int by = bid % nby; bid /= nby;
  const int seg = bid;
  const int sy = by * GBY + wid / GBZ, sz = bz * GBZ + wid % GBZ;
  if (sy >= My || sz >= Mz) return;
  const int X0 = seg * XSEG, X1 = min(X0 + XSEG, Mx);

  // cell boundaries of the segment: lane l <-> cell X0 + l
  int jlo_l = 0, jhi_l = 0;
  if (X0 + lane < X1) {
    const size_t key = ((size_t)(X0 + lane) * My + sy) * Mz + sz;
    jlo_l = __ldg(start + key);
    jhi_l = __ldg(start + key + 1);
  }
  const unsigned mask = __ballot_sync(0xffffffffu, jhi_l > jlo_l);
  if (mask == 0u) return;   // no atoms in this segment of the column (vacuum)
  if (jhi_l > jlo_l) {
    const float* r = rec + (size_t)jlo_l * recf;
    prefetch_l2(r);
    prefetch_l2(r + 32);
    prefetch_l2(drec + (size_t)jlo_l * (3 * SW));
  }
  const int first = __ffs(mask) - 1, last = 31 - __clz(mask);

  // lane -> 2 (b, c) points of the 8 x 8 (y,z) footprint: c = lane & 7, b = (lane >> 3) + 4u
  const int c_off = lane & 7, b0 = lane >> 3;
  int iz = sz + c_off; if (iz >= Mz) iz -= Mz;
  int iy0 = sy + b0;      if (iy0 >= My) iy0 -= My;
  int iy1 = sy + b0 + 4;  if (iy1 >= My) iy1 -= My;
  const unsigned plane = (unsigned)My * Mz;
  const V* g0 = gridi + (size_t)iy0 * Mz + iz;
  const V* g1 = gridi + (size_t)iy1 * Mz + iz;
  // record offsets of this lane's (y,z) weights (records are rotated by the cell index mod 8)
  const int oy0 = SW + ((sy + b0) & 7), oy1 = SW + ((sy + b0 + 4) & 7), oz = 2 * SW + ((sz + c_off) & 7);

  float win[SW][2][CB];
  auto load_plane = [&](int xs) {
    int x = xs; if (x >= Mx) x -= Mx;
    const unsigned off = (unsigned)x * plane;
    switch (xs & 7) {     // the loads sit inside the cases so that they write the slot registers directly
#define PSWF_LOAD(K)                         \
  case K:                                    \
    unpack<CB>(__ldg(g0 + off), win[K][0]);  \
    unpack<CB>(__ldg(g1 + off), win[K][1]);  \
    break;
      PSWF_LOAD(0) PSWF_LOAD(1) PSWF_LOAD(2) PSWF_LOAD(3)
      PSWF_LOAD(4) PSWF_LOAD(5) PSWF_LOAD(6) PSWF_LOAD(7)
#undef PSWF_LOAD
    }
  };
#pragma unroll
  for (int k = 0; k < SW; ++k)
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int c = 0; c < CB; ++c) win[k][u][c] = 0.f;

  // warm-up: planes sx0 .. sx0+6 of the first non-empty cell
  const int sx0 = X0 + first, sx1 = X0 + last;
  for (int a = 0; a < SW - 1; ++a) load_plane(sx0 + a);

  for (int sx = sx0; sx <= sx1; ++sx) {
    load_plane(sx + SW - 1);
    if (!((mask >> (sx - X0)) & 1u)) continue;
    const int jlo = __shfl_sync(0xffffffffu, jlo_l, sx - X0);
    const int jhi = __shfl_sync(0xffffffffu, jhi_l, sx - X0);
    for (int j = jlo; j < jhi; ++j) {
      const float* r = rec + (size_t)j * recf;
      const float* dr = drec + (size_t)j * (3 * SW);
      const float4 xa = __ldg(reinterpret_cast<const float4*>(r));
      const float4 xb = __ldg(reinterpret_cast<const float4*>(r) + 1);
      const float4 da = __ldg(reinterpret_cast<const float4*>(dr));
      const float4 db = __ldg(reinterpret_cast<const float4*>(dr) + 1);
      const float4 q4 = __ldg(reinterpret_cast<const float4*>(r + 3 * SW) + (cb0 >> 2));
      const float wy0 = __ldg(r + oy0), wy1 = __ldg(r + oy1), wz = __ldg(r + oz);
      const float dy0 = __ldg(dr + oy0), dy1 = __ldg(dr + oy1), dz = __ldg(dr + oz);
      const float wx[SW] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
      const float dx[SW] = {da.x, da.y, da.z, da.w, db.x, db.y, db.z, db.w};
      const float qv[4] = {q4.x, q4.y, q4.z, q4.w};
      const float yz[2] = {wy0 * wz, wy1 * wz};
      const float dyz[2] = {dy0 * wz, dy1 * wz};
      const float ydz[2] = {wy0 * dz, wy1 * dz};
      float red[8];
      float fx = 0.f, fy = 0.f, fz = 0.f;
#pragma unroll
      for (int c = 0; c < CB; ++c) {
        float val = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          float S0 = 0.f, S1 = 0.f;
#pragma unroll
          for (int k = 0; k < SW; ++k) {
            S0 = fmaf(wx[k], win[k][u][c], S0);
            S1 = fmaf(dx[k], win[k][u][c], S1);
          }
          val = fmaf(yz[u], S0, val);
          gx = fmaf(yz[u], S1, gx);
          gy = fmaf(dyz[u], S0, gy);
          gz = fmaf(ydz[u], S0, gz);
        }
        const float qc = qv[c];
        fx = fmaf(-qc, gx, fx);
        fy = fmaf(-qc, gy, fy);
        fz = fmaf(-qc, gz, fz);
        red[c] = val;
      }
#pragma unroll
      for (int c = CB; c < 4; ++c) red[c] = 0.f;
      red[4] = fx; red[5] = fy; red[6] = fz; red[7] = 0.f;
      const float tot = reduce8(red, lane);
      // lane l with (l & 3) == 0 holds output index (l>>4)*4 + ((l>>3)&1)*2 + ((l>>2)&1)
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

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
size_t gather_grid_bytes(const pswf_lr_plan* p) {
  // interleaved copy of the potential grid: channel groups of 4 (last group 1, 2 or 4 wide)
  const size_t Mtot = (size_t)p->M[0] * p->M[1] * p->M[2];
  size_t fl = 0;
  for (int cb0 = 0; cb0 < p->C; cb0 += 4) {
    const int left = p->C - cb0;
    fl += Mtot * (left >= 3 ? 4 : left);
  }
  return fl * sizeof(float);
}

void launch_fast_gather(pswf_lr_plan* p, int n, float* phi, float* F, cudaStream_t st) {
  if (n <= 0) return;
  const int Mx = p->M[0], My = p->M[1], Mz = p->M[2];
  const size_t Mtot = (size_t)Mx * My * Mz;
  const int nseg = (Mx + XSEG - 1) / XSEG;
  const int nby = (My + GBY - 1) / GBY, nbz = (Mz + GBZ - 1) / GBZ;
  const unsigned blocks = (unsigned)(nseg * nby * nbz);
  const unsigned iblocks = (unsigned)((Mtot + 255) / 256);
  const int recf = stencil_rec_floats(p->C);
  float* gi = (float*)p->d_gridi;
  int pass = 0;
  for (int cb0 = 0; cb0 < p->C; cb0 += 4, ++pass) {
    const int left = p->C - cb0;
    const int acc = pass > 0 ? 1 : 0;
    const float* planar = (const float*)p->d_grid + (size_t)cb0 * Mtot;
#define PSWF_GATHER(CBV, NCH)                                                                               \
  do {                                                                                                      \
    using V = typename VecOf<CBV>::type;                                                                    \
    k_interleave<CBV><<<iblocks, 256, 0, st>>>(Mtot, NCH, planar, (V*)gi);                                  \
    k_gather_cols<CBV><<<blocks, 32 * GBY * GBZ, 0, st>>>(n, p->C, cb0, Mx, My, Mz, nseg, nby, nbz, recf,   \
                                                          p->d_count, (const float*)p->d_rec,               \
                                                          (const float*)p->d_drec, p->d_perm,               \
                                                          (const V*)gi, phi, F, acc);                       \
    gi += Mtot * CBV;                                                                                       \
  } while (0)
    if (left >= 4) PSWF_GATHER(4, 4);
    else if (left == 3) PSWF_GATHER(4, 3);
    else if (left == 2) PSWF_GATHER(2, 2);
    else PSWF_GATHER(1, 1);
#undef PSWF_GATHER
  }
}

}  // namespace pswf
