// Fast fp32 gather + force kernel for sm_100a (a5; default path, w <= 8).
//
// phi_i^a = sum_g W(x_g - r_i) phi_g^a,  grad phi_i^a = sum_g grad_{r_i} W(x_g - r_i) phi_g^a  (the
// derivative of the SAME panel polynomials),  F_i = - sum_a q_i^a grad phi_i^a.
// 4 w^3 C flops per atom and ~0.5 atoms per grid cell: bound by FP32 issue, not by HBM.
//
// Design: INPUT-STATIONARY IN REGISTERS, one warp per ROW of stencil cells, swept
// along z -- the direction in which the cell-sorted atoms are contiguous.
//  * a warp owns the cell row (s_x, s_y, .) and walks it in 32-cell segments.  A segment's atoms are ONE
//    contiguous run of the sorted arrays, so records and permutation entries stream through L1
//    (prefetched a few atoms ahead) instead of costing an L2 round trip per atom (v2, profiles/r1b:
//    a quarter of the kernel time was spent waiting for per-atom record loads);
//  * every atom of those cells reads the same 8 x 8 (x,y) footprint, two points per lane, so all 32
//    lanes work on every atom and the per-atom sums are a warp shuffle reduction (no atomics);
//  * the 8 z-planes an atom can touch live in a register window win[8][2][CB]; slot k holds the plane
//    z == k (mod 8).  The weight records hold wz and dwz/dz ROTATED by the atom's cell index mod 8,
//    so the z contraction is sum_k wzr[k] * win[k] with static register indices: one copy of the
//    atom code, no unrolled window rotation;
//  * the potential grid is read in a transposed, channel-interleaved layout [z][x][y][CB], so that a
//    z-plane is contiguous and one 16-byte load per footprint point refreshes the slot that left the
//    window for all channels.  The band-limited transform path writes that layout directly
//    (k_z_inverse_il, kernels_fft.cu); after the dense path k_interleave_t copies it from cuFFT's planar
//    [C][x][y][z] (L2-resident).  Neighbouring rows of the CTA share 7/8 of their footprint in L1;
//  * the lanes of a segment fetch the cell boundaries of its 32 cells at once, skip leading /
//    trailing empty cells and return at once when the segment holds no atoms (vacuum of
//    configuration 5);
//  * per atom: z contraction with value and derivative weights in one pass (2 x 8 x 2 FFMA per
//    channel per lane), combination with the (x,y) weights, 9-shuffle transpose-reduce of
//    (phi_a, F_x, F_y, F_z), scattered store to the caller's atom order.
#include <algorithm>
#include <cstdint>
#include <type_traits>

#include "kernels_common.cuh"
#include "launch.hpp"

namespace pswf {

namespace {

constexpr int SW = 8;        // stencil slots per dimension

struct HinvF { float m[9]; };   // h^-1 (row e, column d = ds_d/dr_e), kernel parameter
constexpr int ZSEG = 32;     // cells per z segment: one lane per cell boundary pair

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

// planar [C][x][y][z] -> transposed + interleaved [z][x][y][CB] for the channels cb0 .. cb0+CB-1
// (missing channels read as 0).  One CTA per (x, 32 x 32 tile of (y,z)); reads coalesced along z,
// writes coalesced along y.
template <int CB>
__global__ void __launch_bounds__(256) k_interleave_t(int Mx, int My, int Mz, int nch, const float* __restrict__ planar,
                                                      typename VecOf<CB>::type* __restrict__ out) {
  __shared__ float tile[CB][32][33];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int z0 = blockIdx.x * 32, y0 = blockIdx.y * 32, x = blockIdx.z;
  const size_t Mtot = (size_t)Mx * My * Mz;
#pragma unroll
  for (int c = 0; c < CB; ++c)
#pragma unroll
    for (int yy = ty; yy < 32; yy += 8) {
      float v = 0.f;
      if (c < nch && y0 + yy < My && z0 + tx < Mz)
        v = __ldg(planar + (size_t)c * Mtot + ((size_t)x * My + (y0 + yy)) * Mz + z0 + tx);
      tile[c][yy][tx] = v;
    }
  __syncthreads();
#pragma unroll
  for (int zz = ty; zz < 32; zz += 8) {
    if (y0 + tx < My && z0 + zz < Mz) {
      float v[CB];
#pragma unroll
      for (int c = 0; c < CB; ++c) v[c] = tile[c][tx][zz];
      const size_t o = ((size_t)(z0 + zz) * Mx + x) * My + y0 + tx;
      if constexpr (CB == 1) out[o] = v[0];
      else if constexpr (CB == 2) out[o] = make_float2(v[0], v[1]);
      else out[o] = make_float4(v[0], v[1], v[2], v[3]);
    }
  }
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

// The same for 4 values (forces only: the potentials were not asked for): 6 shuffles; on return lane l holds
// in v[0] the full sum of input index ((l >> 4) & 1) * 2 + ((l >> 3) & 1).
__device__ __forceinline__ float reduce4(float (&v)[8], int lane) {
  const bool hi16 = lane & 16;
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const float send = hi16 ? v[i] : v[i + 2];
    const float keep = hi16 ? v[i + 2] : v[i];
    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
  const bool hi8 = lane & 8;
  {
    const float send = hi8 ? v[0] : v[1];
    const float keep = hi8 ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
  }
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 4);
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2);
  v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
  return v[0];
}

// Packed FP32 pairs (sm_100a FFMA2: one instruction, two IEEE fused multiply-adds per lane; ptxas
// uses its broadcast-scalar operand form for pack2(w, w)).  The gather is issue-bound, not
// FMA-pipe-bound: pairing adjacent channels halves the FMA instruction count of the contraction.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
  return d;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}

__device__ __forceinline__ f32x2 ffma2v(f32x2 a, f32x2 b, f32x2 c) {   // program order kept
  f32x2 d;
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}

// shared-memory accesses by 32-bit shared-space address
__device__ __forceinline__ float4 lds_f32x4(uint32_t a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ float lds_f32(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts_f32(uint32_t a, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory");
}

constexpr int kStage = 32;       // atoms staged per warp at a time (one lane per atom for the output pass)

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)),
               "l"(gsrc)
               : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// floats of shared memory per warp: kStage records, kStage derivative records, kStage x 8 results
// (+ one spare result row: the sink of the software-pipelined reduction when nothing is pending)
__host__ __device__ constexpr int gather_warp_floats(int recf) { return kStage * (recf + 3 * SW + 8) + 8; }

// PHI = false: the caller passed phi == NULL (an MD step needs E and F only): no potential sums, a 4-value
// reduction instead of the 8-value one.
template <int CB, int GBX, int GBY, int NCTA, bool PHI>   // GBX x GBY cell rows (warps) per CTA, NCTA resident CTAs per SM
__global__ void __launch_bounds__(32 * GBX * GBY, NCTA)
    k_gather_rows(int n, int C, int cb0, int Mx, int My, int Mz, int nseg, int nbx, int nby, int recf,
                  const int* __restrict__ start, const float* __restrict__ rec, const float* __restrict__ drec,
                  const int* __restrict__ perm, const typename VecOf<CB>::type* __restrict__ gridt,
                  float* __restrict__ phi, float* __restrict__ Facc, int accumulate_F,
                  const __grid_constant__ HinvF Hi) {
  using V = typename VecOf<CB>::type;
  extern __shared__ __align__(16) float s_all[];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  float* s_rec = s_all + (size_t)wid * gather_warp_floats(recf);   // [kStage][recf]
  float* s_drec = s_rec + kStage * recf;                            // [kStage][24]
  float* s_out = s_drec + kStage * 3 * SW;                          // [kStage + 1][8]
  // block -> (z segment, x block, y block); consecutive blocks walk y, then x: CTAs resident on an SM
  // at the same time share most of their footprints in L1
  int bid = blockIdx.x;
  const int by = bid % nby; bid /= nby;
  const int bx = bid % nbx;
  const int sx = bx * GBX + wid / GBY, sy = by * GBY + wid % GBY;
  if (sx >= Mx || sy >= My) return;
  // lane -> 2 points of the 8 x 8 (x,y) footprint: y offset c = lane & 7, x offsets b and b + 4
  const int c_off = lane & 7, b0 = lane >> 3;
  int iy = sy + c_off;      if (iy >= My) iy -= My;
  // the lane's two x points are sx + b0 and sx + b0 + 4; "point 0" is the one whose rotated weight index
  // (x mod 8) has bit 2 clear, so that point 1's weight sits 4 floats further in every record (an immediate)
  const int xa = sx + b0, xb = sx + b0 + 4;
  const bool swp = (xa & 4) != 0;
  int ix0 = swp ? xb : xa;  if (ix0 >= Mx) ix0 -= Mx;
  int ix1 = swp ? xa : xb;  if (ix1 >= Mx) ix1 -= Mx;
  // loop invariants as shuffle results: ptxas cannot rematerialise those from the constant bank (it
  // re-read Mx, My and cb0 with LDC in every advance / atom otherwise)
  const unsigned plane = __shfl_sync(0xffffffffu, (unsigned)Mx * My, 0), wrap = plane * (unsigned)Mz;
  const int cb0r = __shfl_sync(0xffffffffu, cb0, 0);
  const V* g0 = gridt + (size_t)ix0 * My + iy;
  const V* g1 = gridt + (size_t)ix1 * My + iy;
  // keep the two lane pointers in registers: left to itself ptxas re-derives them from the kernel
  // parameter with a uniform constant load in front of every refill load (70% of the refill's stall
  // samples in profiles/r1c)
  asm volatile("" : "+l"(g0), "+l"(g1));
  // record offsets of this lane's (x,y) weights (records are rotated by the cell index mod 8)
  const int ox0 = (sx + b0) & 3, oy = SW + ((sy + c_off) & 7);   // x weights of the lane: ox0 and ox0 + 4

  // window registers: channel pairs are held PACKED (one 64-bit register pair = {c, c+1}, exactly as
  // the 16-byte plane loads deliver them), ready to be FFMA2 operands
  constexpr int NE = (CB % 2 == 0) ? CB / 2 : CB;
  using WE = typename std::conditional<CB % 2 == 0, f32x2, float>::type;
  WE win[SW][2][NE];
  auto ldw = [&](const V* p, WE (&d)[NE]) {
    if constexpr (CB == 4) {
      const ulonglong2 t = __ldg(reinterpret_cast<const ulonglong2*>(p));
      d[0] = t.x; d[1] = t.y;
    } else if constexpr (CB == 2) {
      d[0] = __ldg(reinterpret_cast<const unsigned long long*>(p));
    } else {
      d[0] = __ldg(p);
    }
  };
  // The window survives from one segment to the next: curA is the cell whose 8 planes it holds.
  int curA = -4 * SW;
  // the warp walks the z segments of its row one after the other (a CTA per segment spent a tenth
  // of its short life being launched)
  // cell boundaries of a segment: lane l <-> cell Z0 + l (the atoms of the row are one run); those of
  // the NEXT segment are fetched while the current one is processed
  const int* rowstart = start + ((size_t)sx * My + sy) * Mz;
  auto fetch_bounds = [&](int sg, int& lo, int& hi) {
    const int z = sg * ZSEG + lane;
    lo = 0; hi = 0;
    if (sg < nseg && z < Mz) { lo = __ldg(rowstart + z); hi = __ldg(rowstart + z + 1); }
  };
  int nlo, nhi;
  fetch_bounds(0, nlo, nhi);
  for (int seg = 0; seg < nseg; ++seg) {
  const int Z0 = seg * ZSEG;
  const int jlo_l = nlo, jhi_l = nhi;
  fetch_bounds(seg + 1, nlo, nhi);
  const unsigned mask = __ballot_sync(0xffffffffu, jhi_l > jlo_l);
  if (mask == 0u) continue;   // no atoms in this segment of the row (vacuum)
  const int first = __ffs(mask) - 1, last = 31 - __clz(mask);
  const int jbeg = __shfl_sync(0xffffffffu, jlo_l, first), jend = __shfl_sync(0xffffffffu, jhi_l, last);

  // stage the records of atoms [js, js + kStage) of the run: asynchronous 16-byte copies, one
  // contiguous stream for rec and one for drec; lane l keeps the permutation entry of atom js + l
  int js = jbeg, perm_l = 0;
  auto stage = [&]() {
    const int cnt = min(kStage, jend - js);
    const float4* gr = reinterpret_cast<const float4*>(rec + (size_t)js * recf);
    const float4* gd = reinterpret_cast<const float4*>(drec + (size_t)js * (3 * SW));
    const int nr = cnt * (recf >> 2), nd = cnt * 6;
    for (int t = lane; t < nr; t += 32) cp_async16(reinterpret_cast<float4*>(s_rec) + t, gr + t);
    for (int t = lane; t < nd; t += 32) cp_async16(reinterpret_cast<float4*>(s_drec) + t, gd + t);
    perm_l = lane < cnt ? __ldg(perm + js + lane) : 0;
  };
  // write the results of the staged atoms: lane l <-> atom js + l, scattered to the caller's order
  auto flush = [&](int cnt) {
    __syncwarp();
    if (lane < cnt) {
      const float4 a = *reinterpret_cast<const float4*>(s_out + 8 * (lane + 1));
      const float4 f = *reinterpret_cast<const float4*>(s_out + 8 * (lane + 1) + 4);
      const float pv[4] = {a.x, a.y, a.z, a.w};
      if constexpr (PHI) {
#pragma unroll
        for (int c = 0; c < CB; ++c)
          if (cb0 + c < C) phi[(size_t)(cb0 + c) * n + perm_l] = pv[c];
      }
      if (Facc) {
        // the derivative records are along the fractional coordinates: F_e = sum_d hinv[e][d] F^s_d
        float fx = -f.x, fy = -f.y, fz = -f.z;   // F = -sum_a q_a grad phi_a
        frac_to_cart(Hi.m, fx, fy, fz);
        float* fp = Facc + 3 * (size_t)perm_l;
        if (accumulate_F) { fp[0] += fx; fp[1] += fy; fp[2] += fz; }
        else { fp[0] = fx; fp[1] = fy; fp[2] = fz; }
      }
    }
    __syncwarp();
  };
  stage();

  // The lane sums of an atom are reduced across the warp one atom LATE, inside the next atom's
  // contraction, so that the five dependent shuffle levels (~150 cycles) overlap its FFMAs.
  float pend[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) pend[i] = 0.f;
  // lane l with (l & 3) == 0 ends up with output index (l>>4)*4 + ((l>>3)&1)*2 + ((l>>2)&1)
  const int out_idx = PHI ? ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1)
                          : 4 + ((lane >> 4) & 1) * 2 + ((lane >> 3) & 1);   // forces live in floats 4..6 of a result row
  // result slot of the pending atom for this lane; the spare row (kStage) when nothing is pending.  Running
  // pointers (records, derivative records, result slot) replace a per-atom multiply-and-add chain each.
  // Result rows: row 0 is a spare, atom t of the staging buffer owns row t + 1; the pending atom's slot is
  // always the row BEFORE out_cur (the spare when nothing is pending).  Records are read by 32-bit shared
  // address: two running bases plus lane-constant byte offsets, one add per scalar pair.
  const uint32_t rec0 = (uint32_t)__cvta_generic_to_shared(s_rec), drec0 = (uint32_t)__cvta_generic_to_shared(s_drec);
  const uint32_t out0 = (uint32_t)__cvta_generic_to_shared(s_out + 8 + out_idx);
  // Loop invariants that ptxas otherwise re-creates inside the atom loop (the record stride from the kernel
  // parameters: LDC + LEA per atom; the lane index from SR_TID: an S2R at the head of every atom's shuffle
  // chain): passed through a volatile shared-memory word, which cannot be rematerialised.
  __shared__ int s_pin[2][32 * GBX * GBY];
  s_pin[0][threadIdx.x] = 4 * recf;
  s_pin[1][threadIdx.x] = lane;
  const uint32_t recB = (uint32_t) * reinterpret_cast<volatile int*>(&s_pin[0][threadIdx.x]);
  const int lane_p = *reinterpret_cast<volatile int*>(&s_pin[1][threadIdx.x]);
  const uint32_t cx = 4u * ox0, cy = 4u * oy, cq = 4u * (3 * SW + cb0r);
  uint32_t ra = rec0, da = drec0;          // record / derivative record of the next atom (one contiguous run per segment)
  uint32_t out_cur = out0;
  int staged_left = kStage;                // atoms left in the staging buffer
  auto retire = [&]() {
    if constexpr (PHI) {
      const float tot = reduce8(pend, lane_p);
      if ((lane_p & 3) == 0) sts_f32(out_cur - 32u, tot);
    } else {
      const float tot = reduce4(pend, lane_p);
      if ((lane_p & 7) == 0) sts_f32(out_cur - 32u, tot);
    }
  };

  // walk the non-empty cells of the segment; the window advances to each of them in one go
  auto advance_to = [&](const int an) {
      const int first_new = max(curA + SW, an);
      const int cnt = an + SW - first_new;      // 1 .. 8 new planes
      if (cnt <= 2) {
        const int z = first_new >= Mz ? first_new - Mz : first_new;
        const unsigned off = (unsigned)z * plane;
        unsigned off2 = off + plane; if (off2 == wrap) off2 = 0u;
        const bool two = cnt == 2;
        switch (first_new & 7) {
#define PSWF_SLOT(K)                                     \
  case K:                                                \
    ldw(g0 + off, win[K][0]);                            \
    ldw(g1 + off, win[K][1]);                            \
    if (two) {                                           \
      ldw(g0 + off2, win[(K + 1) & 7][0]);               \
      ldw(g1 + off2, win[(K + 1) & 7][1]);               \
    }                                                    \
    break;
          PSWF_SLOT(0) PSWF_SLOT(1) PSWF_SLOT(2) PSWF_SLOT(3)
          PSWF_SLOT(4) PSWF_SLOT(5) PSWF_SLOT(6) PSWF_SLOT(7)
#undef PSWF_SLOT
        }
      } else {
        // slot k holds plane pk = base + k (k >= an mod 8) or base + 8 + k (k < an mod 8), base = an rounded
        // down to a multiple of 8; M_z is a multiple of 8, so the wrap past M_z hits the second group as a whole.
        // One copy of the eight predicated slot loads per value of an mod 8: which group a slot belongs to is
        // then static (one compare and one multiply-add per slot; 92 -> ~60 instructions per refill).
        auto refill = [&](auto A7c) {
          constexpr int A7 = decltype(A7c)::value;
          const int base = an - A7;
          const unsigned offA = (unsigned)base * plane;
          const int baseB = base + SW;
          const unsigned offB = (unsigned)(baseB >= Mz ? baseB - Mz : baseB) * plane;
          const int lim = first_new - base;           // load slot k iff k + (k < A7 ? 8 : 0) >= lim
#pragma unroll
          for (int k = 0; k < SW; ++k) {
            if (k + (k < A7 ? SW : 0) >= lim) {
              const unsigned off = (k < A7 ? offB : offA) + (unsigned)k * plane;
              ldw(g0 + off, win[k][0]);
              ldw(g1 + off, win[k][1]);
            }
          }
        };
        switch (an & 7) {
          case 0: refill(std::integral_constant<int, 0>()); break;
          case 1: refill(std::integral_constant<int, 1>()); break;
          case 2: refill(std::integral_constant<int, 2>()); break;
          case 3: refill(std::integral_constant<int, 3>()); break;
          case 4: refill(std::integral_constant<int, 4>()); break;
          case 5: refill(std::integral_constant<int, 5>()); break;
          case 6: refill(std::integral_constant<int, 6>()); break;
          default: refill(std::integral_constant<int, 7>()); break;
        }
      }
      curA = an;
  };
  // one atom: S = slot of the NEWEST plane of the window; the z contraction visits it last
  auto atom = [&](const int j, auto Sc) {
      constexpr int S = decltype(Sc)::value;
        if (staged_left == 0) {   // staging buffer exhausted (dense rows): write results, stage the next atoms
          retire();
          flush(kStage);
          js += kStage;
          stage();
          cp_async_wait_all();
          __syncwarp();
          ra = rec0; da = drec0; out_cur = out0; staged_left = kStage;
        }
        --staged_left;
        const float4 za = lds_f32x4(ra + 4u * 2 * SW);
        const float4 zb = lds_f32x4(ra + 4u * (2 * SW + 4));
        const float4 dza = lds_f32x4(da + 4u * 2 * SW);
        const float4 dzb = lds_f32x4(da + 4u * (2 * SW + 4));
        const float4 q4 = lds_f32x4(ra + cq);
        const uint32_t rx = ra + cx, dx = da + cx;
        const float wx0 = lds_f32(rx), wx1 = lds_f32(rx + 16u), wy = lds_f32(ra + cy);
        const float dx0 = lds_f32(dx), dx1 = lds_f32(dx + 16u), dy = lds_f32(da + cy);
        ra += recB; da += 4u * 3 * SW;
        const float wz[SW] = {za.x, za.y, za.z, za.w, zb.x, zb.y, zb.z, zb.w};
        const float dz[SW] = {dza.x, dza.y, dza.z, dza.w, dzb.x, dzb.y, dzb.z, dzb.w};
        const float qv[4] = {q4.x, q4.y, q4.z, q4.w};
        const float xy[2] = {wx0 * wy, wx1 * wy};      // value and d/dz
        const float dxy[2] = {dx0 * wy, dx1 * wy};     // d/dx
        const float xdy[2] = {wx0 * dy, wx1 * dy};     // d/dy
        retire();   // the previous atom's reduction: independent of everything below (placing its shuffle levels
                    // between the FFMA2 blocks by hand was measured: no gain)
        float fx = 0.f, fy = 0.f, fz = 0.f;
        if constexpr (CB % 2 == 0) {
          // channel pairs (c, c+1): {S_c, S_c+1} += w * {win_c, win_c+1}, one FFMA2 each.  The force needs
          // only sum_c q_c S_c: the charge-weighted sums T are formed BEFORE the (x,y) weights are applied
          // (4 FFMA2 per pair + 6 scalar FMAs instead of 9 FFMA2 per pair + unpacking)
          f32x2 T00 = 0ull, T01 = 0ull, T10 = 0ull, T11 = 0ull;
          // all channel pairs in one pass over the 8 planes: 4 (CB = 2) or 8 (CB = 4) independent FFMA2 chains
          // in round-robin order, so that a chain's next link issues 8 or 16 cycles after the previous one
          constexpr int NP = CB / 2;
          f32x2 S00[NP], S10[NP], S01[NP], S11[NP];
#pragma unroll
          for (int h = 0; h < NP; ++h) { S00[h] = 0ull; S10[h] = 0ull; S01[h] = 0ull; S11[h] = 0ull; }
#pragma unroll
          for (int kk = 0; kk < SW; ++kk) {
            constexpr int k0 = (S + 1) & 7;
            const int k = (k0 + kk) & 7;
            const f32x2 wk = pack2(wz[k], wz[k]), dk = pack2(dz[k], dz[k]);
#pragma unroll
            for (int h = 0; h < NP; ++h) {
              const f32x2 ga = win[k][0][h], gb = win[k][1][h];
              S00[h] = ffma2v(ga, wk, S00[h]);
              S10[h] = ffma2v(ga, dk, S10[h]);
              S01[h] = ffma2v(gb, wk, S01[h]);
              S11[h] = ffma2v(gb, dk, S11[h]);
            }
          }
          const f32x2 xy0 = pack2(xy[0], xy[0]), xy1 = pack2(xy[1], xy[1]);
#pragma unroll
          for (int h = 0; h < NP; ++h) {
            const f32x2 q2 = pack2(qv[2 * h], qv[2 * h + 1]);
            T00 = ffma2(q2, S00[h], T00);
            T01 = ffma2(q2, S01[h], T01);
            T10 = ffma2(q2, S10[h], T10);
            T11 = ffma2(q2, S11[h], T11);
            if constexpr (PHI) {
              const f32x2 val = ffma2(S01[h], xy1, ffma2(S00[h], xy0, 0ull));
              unpack2(val, pend[2 * h], pend[2 * h + 1]);
            }
          }
          float a, b;
          unpack2(T00, a, b); const float t00 = a + b;
          unpack2(T01, a, b); const float t01 = a + b;
          unpack2(T10, a, b); const float t10 = a + b;
          unpack2(T11, a, b); const float t11 = a + b;
          // (minus sign: applied once per atom in flush())
          fx = wy * fmaf(dx1, t01, dx0 * t00);
          fy = dy * fmaf(wx1, t01, wx0 * t00);
          fz = fmaf(xy[1], t11, xy[0] * t10);
        } else {
#pragma unroll
        for (int c = 0; c < CB; ++c) {
          float val = 0.f, gx = 0.f, gy = 0.f, gz = 0.f;
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            float S0 = 0.f, S1 = 0.f;
#pragma unroll
            for (int k = 0; k < SW; ++k) {
              S0 = fmaf(wz[k], win[k][u][c], S0);
              S1 = fmaf(dz[k], win[k][u][c], S1);
            }
            val = fmaf(xy[u], S0, val);
            gz = fmaf(xy[u], S1, gz);
            gx = fmaf(dxy[u], S0, gx);
            gy = fmaf(xdy[u], S0, gy);
          }
          const float qc = qv[c];
          fx = fmaf(qc, gx, fx);
          fy = fmaf(qc, gy, fy);
          fz = fmaf(qc, gz, fz);
          if constexpr (PHI) pend[c] = val;
        }
        }
        if constexpr (PHI) {
#pragma unroll
          for (int c = CB; c < 4; ++c) pend[c] = 0.f;
          pend[4] = fx; pend[5] = fy; pend[6] = fz; pend[7] = 0.f;
        } else {
          pend[0] = fx; pend[1] = fy; pend[2] = fz; pend[3] = 0.f;
        }
        out_cur += 32u;   // this atom's row becomes the pending one
  };
  {
  unsigned rem = mask;        // non-empty cells not yet visited
  bool first_cell = true;
  while (rem != 0u) {
    const int cur = __ffs(rem) - 1;   // current cell, relative to Z0
    rem &= rem - 1u;
    advance_to(Z0 + cur);
    if (first_cell) {   // this segment's records were staged before the window loads were issued
      cp_async_wait_all();
      __syncwarp();
      first_cell = false;
    }
    const int jlo = __shfl_sync(0xffffffffu, jlo_l, cur);
    const int jhi = __shfl_sync(0xffffffffu, jhi_l, cur);
    for (int j = jlo; j < jhi; ++j) atom(j, std::integral_constant<int, 7>());
  }
  }
  retire();
  flush(jend - js);
  }   // segments
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
size_t gather_grid_bytes(const pswf_lr_plan* p) {
  // interleaved copy of the potential grid: channel groups of 4 (last group 1, 2 or 4 wide)
  const size_t Mtot = (size_t)p->M[0] * p->M[1] * p->M[2];
  size_t fl = 0;
  const int G = p->gather_group;
  for (int cb0 = 0; cb0 < p->C; cb0 += G) {
    const int left = std::min(G, p->C - cb0);
    fl += Mtot * (left >= 3 ? 4 : left);
  }
  return fl * sizeof(float);
}

template <int GBX, int GBY, int NCTA>
void launch_fast_gather_t(pswf_lr_plan* p, int n, float* phi, float* F, bool have_il, cudaStream_t st) {
  const int Mx = p->M[0], My = p->M[1], Mz = p->M[2];
  const size_t Mtot = (size_t)Mx * My * Mz;
  const int nseg = (Mz + ZSEG - 1) / ZSEG;
  const int nbx = (Mx + GBX - 1) / GBX, nby = (My + GBY - 1) / GBY;
  const unsigned blocks = (unsigned)(nbx * nby);
  const dim3 iblocks((unsigned)((Mz + 31) / 32), (unsigned)((My + 31) / 32), (unsigned)Mx);
  const int recf = stencil_rec_floats(p->C);
  const size_t smem = sizeof(float) * GBX * GBY * (size_t)gather_warp_floats(recf);
  float* gi = (float*)p->d_gridi;
  HinvF Hi;
  for (int i = 0; i < 9; ++i) Hi.m[i] = (float)p->hinv[i];
  int pass = 0;
  const int G = p->gather_group;
  for (int cb0 = 0; cb0 < p->C; cb0 += G, ++pass) {
    const int left = std::min(G, p->C - cb0);
    const int acc = pass > 0 ? 1 : 0;
    const float* planar = (const float*)p->d_grid + (size_t)cb0 * Mtot;
#define PSWF_GATHER(CBV, NCH, NCTAV)                                                                        \
  do {                                                                                                      \
    using V = typename VecOf<CBV>::type;                                                                    \
    p->n_kernels += have_il ? 1 : 2;                                                                        \
    if (!have_il) k_interleave_t<CBV><<<iblocks, 256, 0, st>>>(Mx, My, Mz, NCH, planar, (V*)gi);            \
    auto kern = phi ? k_gather_rows<CBV, GBX, GBY, NCTAV, true> : k_gather_rows<CBV, GBX, GBY, NCTAV, false>; \
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                     \
    kern<<<blocks, 32 * GBX * GBY, smem, st>>>(n, p->C, cb0, Mx, My, Mz, nseg, nbx, nby, recf, p->d_count,        \
                                               (const float*)p->d_rec, (const float*)p->d_drec, p->d_perm,  \
                                               (const V*)gi, phi, F, acc, Hi);                              \
    gi += Mtot * CBV;                                                                                       \
  } while (0)
    if (left >= 4) PSWF_GATHER(4, 4, NCTA);
    else if (left == 3) PSWF_GATHER(4, 3, NCTA);
    else if (left == 2) PSWF_GATHER(2, 2, 6);
    else PSWF_GATHER(1, 1, 6);
#undef PSWF_GATHER
  }
}

void launch_fast_gather(pswf_lr_plan* p, int n, float* phi, float* F, bool grid_is_interleaved, cudaStream_t st) {
  if (n <= 0) return;
  // 2 x 2 cell rows (4 warps) per CTA, 4 CTAs per SM: short-lived CTAs lose fewer warp slots to the
  // longest row than 8-warp ones (489 -> 474 us), and the 128-register budget is the same
  launch_fast_gather_t<2, 2, 4>(p, n, phi, F, grid_is_interleaved, st);
}

}  // namespace pswf
