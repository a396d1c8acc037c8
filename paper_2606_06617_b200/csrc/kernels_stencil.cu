// Fast fp32 stencil kernels for sm_100a: spread (a1) and the per-atom weight records it consumes.
//
// Spread, Eq. (20)-(21),(24), is rho_g^a = sum_j q_j^a wx_j(g_x) wy_j(g_y) wz_j(g_z):
// w^3 C FMAs per atom and ~0.5 atoms per grid cell, i.e. bound by FP32 issue, not by HBM.  Shared-
// memory float atomics are CAS loops on sm_100a, so the kernel is OUTPUT-STATIONARY AT THREAD LEVEL
// and atomic-free:
//
//  * a thread owns two adjacent grid columns (y, z0) and (y, z0+1) and sweeps x; its accumulators
//    acc[8][2][CB] live in registers, slot k holding the plane x == k (mod 8);
//  * atoms are cell-sorted; for every cell plane s_x the CTA stages the weight records of the cells
//    (s_y, s_z) that can touch its 8WY x 8WZ patch into shared memory with TMA bulk copies
//    (cp.async.bulk + mbarrier, double buffered, one contiguous run per cell row);
//  * every thread then walks ITS OWN list of atoms -- the 8 x 9 cells whose footprint covers its
//    two columns, read through a per-plane table of cell boundaries -- so nearly all lanes do
//    useful FMAs (a warp-wide broadcast of each atom would keep only 64/165 of them busy);
//  * the record holds the three weight vectors ROTATED by the atom's cell index mod 8, so a thread
//    reads wy at offset (y & 7), wz at (z0 & 7) and multiplies slot k by wxr[k]: no per-atom index
//    arithmetic, no register rotation, no unrolled plane loop;
//  * the x range is cut into segments that form one wave of CTAs; when a plane leaves the window its slot
//    is stored once with plain coalesced stores, except the 7 planes a segment shares with each
//    neighbour, which are merged with red.global.add.v2.f32 into the grid (zero-filled by a memset before
//    the launch).  No shared-memory atomics.  In-cell atom order comes from atomicAdd ranks and the seam
//    planes from RED, so results are NOT bitwise reproducible from run to run (differences ~1e-7).
//
// Requirements of this path (host-checked): fp32, even w <= 8 (narrower windows are zero padded to 8
// slots), M_d a multiple of 8 and >= 16.
#include <algorithm>
#include <climits>
#include <cstdint>

#include "kernels_common.cuh"
#include "launch.hpp"

namespace pswf {

namespace {

constexpr int SW = 8;  // stencil slots per dimension

// ------------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + TMA bulk copy (global -> shared)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ------------------------------------------------------------------------------------------------
// scatter into cell-sorted order + per-atom weight records
// record (recf floats): wxr[8] | wyc[8] | wzc[8] | q[C padded to 4]; wxr[k] = wx[(k - s_x) & 7] etc.
// derivative record (24 floats, gather only): dxr[8] | dyc[8] | dzc[8], d/dr_d of the same weights
// (derivative of the SAME panel polynomials), rotated the same way.
// ------------------------------------------------------------------------------------------------
// rotate right by s: out[k] = v[(k - s) & 7], three conditional stages (24 selects)
__device__ __forceinline__ void rotate8(float (&v)[SW], int s) {
  float t[SW];
  const bool r4 = s & 4, r2 = s & 2, r1 = s & 1;
#pragma unroll
  for (int k = 0; k < SW; ++k) t[k] = r4 ? v[(k + 4) & 7] : v[k];
#pragma unroll
  for (int k = 0; k < SW; ++k) v[k] = r2 ? t[(k + 6) & 7] : t[k];
#pragma unroll
  for (int k = 0; k < SW; ++k) t[k] = r1 ? v[(k + 7) & 7] : v[k];
#pragma unroll
  for (int k = 0; k < SW; ++k) v[k] = t[k];
}

// perm[sorted slot] = atom: the only scattered write of the sort (4 bytes per atom).
__global__ void __launch_bounds__(256) k_perm(int n, const int* __restrict__ start, const int* __restrict__ key,
                                              const int* __restrict__ rank, int* __restrict__ perm) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) perm[__ldg(start + __ldg(key + i)) + __ldg(rank + i)] = i;
}

// One thread per SORTED slot j: gathers pos / q of atom perm[j] (random 32-byte reads out of L2; the
// inputs fit it) and builds the records.  The 112-byte weight records straddle 32-byte sectors, so
// they leave through shared memory and the CTA writes 128 consecutive records with fully coalesced
// 16-byte stores; the 96-byte derivative records are three whole sectors each and are stored
// directly (staging them too halved the resident CTAs: 100 us instead of 58 us).  (Scattering
// finished records from atom order cost 300 us: 17 partially written sectors per atom; profiles/r1b.)
//
// The panel polynomials arrive BY VALUE (kernel parameter space = constant bank): with the panel
// index and the power static, every Horner step is one FFMA with a constant-bank operand and no
// coefficient load.  The rotation by the cell index is done on the finished weights in registers.
constexpr int kRecThreads = 128;

template <int DEG>   // polynomial degree actually evaluated (the tables are zero beyond the plan's degree)
__global__ void __launch_bounds__(kRecThreads) k_records(int n, int C, int recf, const float* __restrict__ pos,
                                                         const float* __restrict__ q, GridGeom<float> g,
                                                         const __grid_constant__ WindowPoly P,
                                                         const int* __restrict__ perm, float* __restrict__ rec,
                                                         float* __restrict__ drec) {
  extern __shared__ __align__(16) float s_rec[];   // [kRecThreads][recf]
  const int j0 = blockIdx.x * kRecThreads;
  const int j = j0 + threadIdx.x;
  if (j < n) {
    const int i = __ldg(perm + j);
    float* r = s_rec + threadIdx.x * recf;
    float* dr = drec + (size_t)j * (3 * SW);   // 96 bytes = three whole 32-byte sectors: stored directly
    const float px[3] = {__ldg(pos + 3 * (size_t)i), __ldg(pos + 3 * (size_t)i + 1), __ldg(pos + 3 * (size_t)i + 2)};
    for (int c0 = 0; c0 < recf - 3 * SW; c0 += 4) {
      float qq[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) qq[u] = c0 + u < C ? __ldg(q + (size_t)(c0 + u) * n + i) : 0.f;
      reinterpret_cast<float4*>(r + 3 * SW)[c0 >> 2] = make_float4(qq[0], qq[1], qq[2], qq[3]);
    }
    int i0v[3];
    double deltav[3];
    stencil_3d(px, g.hinv, g.M, g.w, i0v, deltav);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int i0 = i0v[d];
      const double delta = deltav[d];
      const int s = wrap_index(i0, g.M[d]);
      const float xi = 2.f * (float)delta - 1.f;
      float v[SW], dv[SW];
#pragma unroll
      for (int t = 0; t < SW; ++t) {
        float a = P.c[DEG][t], b = P.d[DEG - 1][t];
#pragma unroll
        for (int m = DEG - 1; m >= 1; --m) {
          a = fmaf(a, xi, P.c[m][t]);
          b = fmaf(b, xi, P.d[m - 1][t]);
        }
        a = fmaf(a, xi, P.c[0][t]);
        v[t] = a;
        dv[t] = b * g.dxi_ds[d];   // derivative along the fractional coordinate; the gather converts
      }
      rotate8(v, s);
      rotate8(dv, s);
      reinterpret_cast<float4*>(r)[2 * d] = make_float4(v[0], v[1], v[2], v[3]);
      reinterpret_cast<float4*>(r)[2 * d + 1] = make_float4(v[4], v[5], v[6], v[7]);
      reinterpret_cast<float4*>(dr)[2 * d] = make_float4(dv[0], dv[1], dv[2], dv[3]);
      reinterpret_cast<float4*>(dr)[2 * d + 1] = make_float4(dv[4], dv[5], dv[6], dv[7]);
    }
  }
  __syncthreads();
  const int nrec = min(kRecThreads, n - j0);
  const int rq = recf >> 2;
  float4* grec = reinterpret_cast<float4*>(rec + (size_t)j0 * recf);
  for (int t = threadIdx.x; t < nrec * rq; t += kRecThreads) grec[t] = reinterpret_cast<const float4*>(s_rec)[t];
}

// ------------------------------------------------------------------------------------------------
// spread
// ------------------------------------------------------------------------------------------------
// A round = the atoms of one cell plane that are staged at once: whole cell rows [r0, r1) of the
// plane, or -- when a single row holds more atoms than the staging buffer -- the atoms [a0, a1) of
// the one row r0 (indices local to the row).
struct RoundDesc {
  int p;          // cell plane, counted through the CTA's segments (a segment's planes are pb .. pe-1)
  int r0, r1;     // rows of the plane handled by this round
  int a0, a1;     // atom sub-range of a single-row round (0, INT_MAX otherwise)
  int total;      // atoms staged
  int flush;      // 1: the plane is complete after this round
  int np, nr, na; // where the next round starts (plane, row, atom)
};

template <int WY, int WZ>
struct SpreadShape {
  static constexpr int TY = 8 * WY, TZ = 8 * WZ;
  static constexpr int NROW = TY + 7, NCELL = TZ + 7, NB = TZ + 8;
  static constexpr int NT = 32 * WY * WZ;
  // Staging buffers in flight: two, each as large as shared memory allows -- a cell plane whose atoms do
  // not fit one buffer is split into two rounds, and every round costs the consumers a run-descriptor pass
  // and a barrier (three smaller buffers split every plane: 329 -> 405 us, round 1).  Cell-boundary tables:
  // two, handed back to the producer by the consumers (tabfree barriers) as soon as they have built the run
  // descriptors of a plane's last round; a third table cost 11 records of each buffer.
  static constexpr int kStages = 2;
  static constexpr int kTabs = 2;
  static constexpr int kOffDesc = 64, kOffRowoff = 192, kOffRow = kOffRowoff + kStages * 32 * 4;
  static constexpr int kHeader = kOffRow + kTabs * 32 * 16;   // mbar | desc | rowoff | rowinfo
  static constexpr int kTables = kTabs * NROW * NB * 4;
  static constexpr int kRuns = SW * NT * 8;   // per thread: 8 packed run descriptors of the current round (the prefetch past the
                                               // last one reads the first staged records: in bounds, never used)
  static_assert(NROW <= 32, "one lane per row in the round builder");
  static_assert(kOffDesc + kStages * sizeof(RoundDesc) <= kOffRowoff && (2 * kStages + kTabs) * 8 <= kOffDesc, "header");
};

// Packed FP32 pairs (sm_100a FFMA2: one instruction, two IEEE fused multiply-adds per lane -- the FLOP
// rate of FFMA at half the issue slots; the stencil kernels are issue-bound, not FMA-pipe-bound).
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
__device__ __forceinline__ void ffma2_acc(f32x2& c, f32x2 a, f32x2 b) {   // c += a * b, in place
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));
}

// zero one half of a packed pair in place (the same register keeps holding the accumulator: a fresh
// pack2() in each arm of the flush switch left ptxas with 16 register moves per atom visit)
__device__ __forceinline__ void zero_lo(f32x2& v) {
  asm("{\n.reg .b32 lo, hi;\nmov.b64 {lo, hi}, %0;\nmov.b64 %0, {0f00000000, hi};\n}" : "+l"(v));
}
__device__ __forceinline__ void zero_hi(f32x2& v) {
  asm("{\n.reg .b32 lo, hi;\nmov.b64 {lo, hi}, %0;\nmov.b64 %0, {lo, 0f00000000};\n}" : "+l"(v));
}

__device__ __forceinline__ void red_add_v2(float* p, float a, float b) {
  asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

__device__ __forceinline__ f32x2 fmul2(f32x2 a, f32x2 b) {
  f32x2 d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// One thread's atoms of a round are (at most) 8 runs of staged records, one per cell row s_y = y-7 .. y:
// the cells s_z = z0-7 .. z0+1 of the row, clipped to the round's atom range [a0, a1).  Atoms of the
// first cell miss column z0+1 (j < ja) and atoms of the last cell miss column z0 (j >= jb).
// The runs are computed once per round in a uniform, fully unrolled pass (all lanes busy, shared-
// memory latencies overlapped) and left in shared memory as packed descriptors {j | jend << 16,
// ja | jb << 16} in staged-record units; EMPTY RUNS ARE DROPPED, so the atom loop can switch runs
// with a handful of predicated instructions instead of a divergent search for the next non-empty
// one (v4 spent a third of its warp instructions there; profiles/r1f).  Returns the thread's atom
// count of the round.
__device__ __forceinline__ int build_runs(uint2* runs, const int NT, const int r_beg, const int r_hi, const int* Lp,
                                          const int NB, const int NROWS, const int* ro, const int a0, const int a1) {
  int total = 0;
  uint2* out = runs;
  // branch-free: every lane handles 8 row slots; a row outside [r_beg, r_hi) or without atoms for this
  // thread stores its descriptor too, but does not advance `out`, so the next one overwrites it
#pragma unroll
  for (int i = 0; i < SW; ++i) {
    const int rr = r_beg + i;
    const int rc = min(rr, NROWS - 1);   // (clamped: stays inside the table; masked below)
    const int2 a = *reinterpret_cast<const int2*>(Lp + rc * NB);
    const int2 b = *reinterpret_cast<const int2*>(Lp + rc * NB + SW);
    const int off = ro[rc] - a0;      // staged position of the row's atom 0
    const int j = off + max(a.x, a0);
    const int jend = off + min(b.y, a1);
    const int ja = min(max(off + a.y, 0), 0xffff);
    const int jb = min(max(off + b.x, 0), 0xffff);
    const bool ne = rr < r_hi && jend > j;
    *out = make_uint2((unsigned)j | ((unsigned)jend << 16), (unsigned)ja | ((unsigned)jb << 16));
    out += ne ? NT : 0;
    total += ne ? jend - j : 0;
  }
  return total;
}

// shared-memory loads by 32-bit shared-space address (keeps the address arithmetic of the atom loop at
// one IMAD and three adds per visit)
__device__ __forceinline__ ulonglong2 lds_u64x2(uint32_t a) {
  ulonglong2 v;
  asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ f32x2 lds_u64(uint32_t a) {
  f32x2 v;
  asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ float lds_f32(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ uint2 lds_u32x2(uint32_t a) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
  return v;
}

// The atom loop: one trip per (atom, thread) visit, `total` trips, all bookkeeping branch-free.
//  * p[u] = wy * wz[u] by one FMUL2, v[u][c] = p[u] * q[c], the 32 accumulations as FFMA2
//    {plane k, plane k+1} += {wx[k], wx[k+1]} * v (broadcast operand form);
//  * the next run's descriptor is fetched a run ahead; the switch is a few predicated instructions;
//  * SOFTWARE PIPELINED: the thread-specific words of the NEXT visit (wy, wz pair, charges) are
//    requested before the current visit's FFMA2 block, so the LDS -> FMUL2 -> FSEL -> FMUL chain that
//    feeds the first FFMA2 no longer waits for shared memory (30% of the loop's stall samples in
//    profiles/r2a).
template <int CB>
__device__ __forceinline__ void walk_atoms(f32x2 (&acc)[SW / 2][2][CB], const uint2* runs, const int NT, const int total,
                                           const float* rbase, const int recf, const int cb0, const int oy,
                                           const int oz) {
  // loop invariants pinned to registers (ptxas otherwise reloads the kernel parameters from the
  // constant bank inside the atom loop; a shuffle result cannot be rematerialised from there)
  const uint32_t recB = 4u * (uint32_t)__shfl_sync(0xffffffffu, recf, 0);
  const uint32_t sb = smem_u32(rbase);
  const uint32_t qB = 4u * (3 * SW + (uint32_t)__shfl_sync(0xffffffffu, cb0, 0)), yB = 4u * oy, zB = 4u * oz;
  if (total <= 0) return;
  uint32_t nrun = smem_u32(runs);
  const uint32_t runB = 8u * NT;
  uint2 nd = lds_u32x2(nrun);
  int j = (int)(nd.x & 0xffffu), jend = (int)(nd.x >> 16), ja = (int)(nd.y & 0xffffu), jb = (int)(nd.y >> 16);
  nrun += runB;
  nd = lds_u32x2(nrun);          // (past the thread's last run: stale but in-bounds, never used)
  uint32_t a = sb + (uint32_t)j * recB;
  float wyv = lds_f32(a + yB);
  f32x2 wz2 = lds_u64(a + zB);
  f32x2 q01 = 0ull, q23 = 0ull;
  auto load_q = [&](uint32_t at) {
    if constexpr (CB >= 3) {
      const ulonglong2 tq = lds_u64x2(at + qB);
      q01 = tq.x; q23 = tq.y;
    } else if constexpr (CB == 2) {
      q01 = lds_u64(at + qB);
    } else {
      q01 = pack2(lds_f32(at + qB), 0.f);
    }
  };
  load_q(a);
  int t = total;
  bool more;
#pragma unroll 1
  do {
    const ulonglong2 wa = lds_u64x2(a);        // {wx0,wx1}, {wx2,wx3}
    const ulonglong2 wb = lds_u64x2(a + 16);   // {wx4,wx5}, {wx6,wx7}
    float qv[4];
    unpack2(q01, qv[0], qv[1]);
    unpack2(q23, qv[2], qv[3]);
    float p0, p1;
    unpack2(fmul2(wz2, pack2(wyv, wyv)), p0, p1);
    p0 = j < jb ? p0 : 0.f;
    p1 = j >= ja ? p1 : 0.f;
    float v0[CB], v1[CB];
    // scalar products on purpose: with FMUL2 pairs here ptxas overlays eight accumulator pairs on the
    // dying 64-bit temporaries and copies them back every visit (16 IMAD.MOV per trip)
#pragma unroll
    for (int c = 0; c < CB; ++c) { v0[c] = p0 * qv[c]; v1[c] = p1 * qv[c]; }
    ++j;
    if (j == jend) {             // next run (if-converted: no divergence)
      j = (int)(nd.x & 0xffffu); jend = (int)(nd.x >> 16);
      ja = (int)(nd.y & 0xffffu); jb = (int)(nd.y >> 16);
      nrun += runB;
      nd = lds_u32x2(nrun);
    }
    more = --t > 0;
    if (more) {                  // the next visit's words (after the last visit j is stale: no load)
      a = sb + (uint32_t)j * recB;
      wyv = lds_f32(a + yB);
      wz2 = lds_u64(a + zB);
      load_q(a);
    }
    const f32x2 wx[SW / 2] = {wa.x, wa.y, wb.x, wb.y};
#pragma unroll
    for (int c = 0; c < CB; ++c) {
      const f32x2 d0 = pack2(v0[c], v0[c]), d1 = pack2(v1[c], v1[c]);
#pragma unroll
      for (int k2 = 0; k2 < SW / 2; ++k2) {
        ffma2_acc(acc[k2][0][c], wx[k2], d0);
        ffma2_acc(acc[k2][1][c], wx[k2], d1);
      }
    }
  } while (more);
}

template <int WY, int WZ, int CB, int NCTA>
// WY x WZ consumer warps + one producer warp.  (Stating the cap as __maxnreg__(136) removes ptxas's
// register-saving copies in the atom loop, but 136 registers x 160 threads run as TWO CTAs per SM:
// 353 us against 300 us.)
__global__ void __launch_bounds__(32 * WY * WZ + 32, NCTA)
    k_spread_os(int Mx, int My, int Mz, int npy, int npz, int cap, int recf, int cb0,
                const int* __restrict__ start, const float* __restrict__ rec, float* __restrict__ grid) {
  using S = SpreadShape<WY, WZ>;
  constexpr int NROW = S::NROW, NB = S::NB, NT = S::NT;
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr int NS = S::kStages, NTAB = S::kTabs;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);                 // [NS] records of a round have landed
  uint64_t* empty = full + NS;                                        // [NS] all consumer warps are done with them
  uint64_t* tabfree = empty + NS;                                     // [NTAB] ... with a plane's cell-boundary table
  RoundDesc* s_desc = reinterpret_cast<RoundDesc*>(smem + S::kOffDesc);   // [NS]
  int* s_rowoff = reinterpret_cast<int*>(smem + S::kOffRowoff);       // [NS][32]
  int4* s_row = reinterpret_cast<int4*>(smem + S::kOffRow);            // [NTAB][32]  {gA0, nA, gB0, nB}
  int* s_L = reinterpret_cast<int*>(smem + S::kHeader);               // [NTAB][NROW][NB]
  uint2* s_run = reinterpret_cast<uint2*>(smem + S::kHeader + S::kTables) + threadIdx.x;   // [8][NT], this thread's
  float* s_rec = reinterpret_cast<float*>(smem + S::kHeader + S::kTables + S::kRuns);     // [2][cap * recf]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // This CTA's share of the work: the npy * npz patches x Mx cell planes, patch-major, are cut into
  // gridDim.x equal ranges (one wave: every SM holds NCTA CTAs of the same length -- with whole segments
  // per patch, 64 patches x 6 segments left 60 of 148 SMs a CTA short).  A range that crosses a patch
  // boundary is one segment per patch, worked off one after the other.  The atoms are PARTITIONED over the segments
  // (no halo is re-read); the 7 output planes a segment shares with each neighbour are merged in global
  // memory by RED.
  const int gtot = npy * npz * Mx;
  const int g0 = (int)((long long)blockIdx.x * gtot / gridDim.x), g1 = (int)((long long)(blockIdx.x + 1) * gtot / gridDim.x);
  const int nsg = (g1 - 1) / Mx - g0 / Mx + 1;   // 1, or 2 across a patch boundary (more only when patches outnumber CTAs)
  int X0, NP, pb, pe, Y0, Z0, nAc, zb0, nBc, ncell;
  // cells of a row: sz_u = Z0-7 .. Z0+TZ-1; those below 0 wrap to the end of the row (run A)
  auto set_segment = [&](int sg) {
    const int patch = g0 / Mx + sg;
    const int lo = max(g0, patch * Mx), hi = min(g1, (patch + 1) * Mx);
    X0 = lo - patch * Mx; NP = hi - lo;
    pb = lo - g0; pe = pb + NP;          // running plane indices: table slots and barrier phases carry over
    Y0 = (patch / npz) * S::TY; Z0 = (patch % npz) * S::TZ;
    nAc = Z0 < SW - 1 ? SW - 1 - Z0 : 0;
    zb0 = Z0 - (SW - 1) + nAc;
    nBc = min(S::NCELL - nAc, Mz - zb0);
    ncell = nAc + nBc;
  };
  set_segment(0);

  // this thread's two columns
  const int wy_ = warp / WZ, wz_ = warp % WZ;
  const int ly = lane >> 2, lzp = lane & 3;
  int y, z0;
  bool lane_ok;
  auto set_columns = [&] {
    y = Y0 + wy_ * 8 + ly; z0 = Z0 + wz_ * 8 + 2 * lzp;
    lane_ok = y < My && z0 < Mz;
  };
  set_columns();
  const int rlo = wy_ * 8 + ly;          // first of the 8 rows (s_y = y-7 .. y) this thread reads
  const int clo = wz_ * 8 + 2 * lzp;     // boundary index of cell s_z = z0-7
  const int oy = SW + ly, oz = 2 * SW + 2 * lzp;   // patch origins are multiples of 8
  const size_t Mtot = (size_t)Mx * My * Mz;

  // Cell-boundary table of plane pl (producer warp): lane r fetches row r's run bases (4 loads), every
  // lane its share of the 23 x 24 table entries (one load each).
  auto build_plane = [&](int pl) {
    const int tb = pl % NTAB;
    const int sx = X0 + (pl - pb);
    // every load of the plane -- the lane's row bases and its table entries -- is requested before the
    // first result is used: ONE L2 round trip per plane (the producer's time per plane adds to the
    // consumers': spread = 140 us + 161 us x N / 1e6 at the config-4 grid with three round trips)
    const int syu_l = Y0 - (SW - 1) + lane;
    const bool row_ok = lane < NROW && syu_l < My;
    int gA0 = 0, eA = 0, gB0 = 0, eB = 0;
    if (row_ok) {
      const int sy = syu_l < 0 ? syu_l + My : syu_l;
      const int* rs = start + ((size_t)sx * My + sy) * Mz;
      if (nAc) { gA0 = __ldg(rs + Mz - nAc); eA = __ldg(rs + Mz); }
      gB0 = __ldg(rs + zb0);
      eB = __ldg(rs + zb0 + nBc);
    }
    constexpr int kEnt = (NROW * NB + 31) / 32;
    int got[kEnt];
#pragma unroll
    for (int k = 0; k < kEnt; ++k) {
      const int t = lane + 32 * k;
      const int r = t / NB, b = t - r * NB;
      const int syu = Y0 - (SW - 1) + r;
      got[k] = 0;
      if (t < NROW * NB && syu < My) {
        const int sy = syu < 0 ? syu + My : syu;
        const int* rs = start + ((size_t)sx * My + sy) * Mz;
        got[k] = b < nAc ? __ldg(rs + Mz - nAc + b) : __ldg(rs + zb0 + min(b, ncell) - nAc);
      }
    }
    if (lane < NROW) s_row[tb * 32 + lane] = row_ok ? make_int4(gA0, eA - gA0, gB0, eB - gB0) : make_int4(0, 0, 0, 0);
    if (pl >= NTAB) mbar_wait(&tabfree[tb], ((pl / NTAB) - 1) & 1);   // plane pl-NTAB's table has been read
    __syncwarp();
#pragma unroll
    for (int k = 0; k < kEnt; ++k) {
      const int t = lane + 32 * k;
      const int r = t / NB, b = t - r * NB;
      const int syu = Y0 - (SW - 1) + r;
      if (t < NROW * NB) {
        int val = 0;
        if (syu < My) {
          const int4 ri = s_row[tb * 32 + r];
          val = b < nAc ? got[k] - ri.x : ri.y + got[k] - ri.z;
        }
        s_L[(tb * NROW + r) * NB + b] = val;
      }
    }
  };

  // round builder (warp 0): the next round starts at (plane pn, row rn0, atom an0 of that row)
  auto build_round = [&](int pn, int rn0, int an0, int nb) -> RoundDesc {
    RoundDesc nd;
    nd.p = pn; nd.r0 = rn0; nd.r1 = NROW; nd.a0 = 0; nd.a1 = INT_MAX; nd.total = 0; nd.flush = 1;
    nd.np = pn + 1; nd.nr = 0; nd.na = 0;
    if (pn < pe) {
      const int tb = pn % NTAB;
      const bool mine = lane >= rn0 && lane < NROW;
      int tot = mine ? s_L[(tb * NROW + lane) * NB + NB - 1] : 0;
      if (lane == rn0) tot -= an0;
      int cum = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, cum, o);
        if (lane >= o) cum += t;
      }
      const int nfit = __popc(__ballot_sync(0xffffffffu, mine && cum <= cap));
      const int t0 = __shfl_sync(0xffffffffu, tot, rn0);
      const bool single = an0 > 0 || nfit == 0;
      int so, cnt;   // this lane's row: staged position of its first atom, atoms staged
      if (single) {  // (the rest of) one row, at most a buffer full
        const int take = min(cap, t0);
        nd.r1 = rn0 + 1; nd.a0 = an0; nd.a1 = an0 + take; nd.total = take;
        if (t0 > take) { nd.flush = 0; nd.np = pn; nd.nr = rn0; nd.na = an0 + take; }
        else if (rn0 + 1 < NROW) { nd.flush = 0; nd.np = pn; nd.nr = rn0 + 1; }
        so = 0; cnt = take;
      } else {       // whole rows
        nd.r1 = rn0 + nfit;
        nd.total = __shfl_sync(0xffffffffu, cum, nd.r1 - 1);
        if (nd.r1 < NROW) { nd.flush = 0; nd.np = pn; nd.nr = nd.r1; }
        so = cum - tot; cnt = tot;
      }
      const bool in_round = lane >= rn0 && lane < nd.r1;
      if (in_round) s_rowoff[nb * 32 + lane] = so;
      if (lane == 0) s_desc[nb] = nd;
      __syncwarp();   // descriptor and row offsets are written before the barrier can complete
      if (lane == 0) {
        if (nd.total > 0) mbar_arrive_expect_tx(&full[nb], (uint32_t)nd.total * recf * 4u);
        else mbar_arrive(&full[nb]);
      }
      __syncwarp();
      if (in_round && cnt > 0) {
        const int4 ri = s_row[tb * 32 + lane];   // the row = run A (ri.y atoms at ri.x) then run B
        const int lo = nd.a0, hi = nd.a0 + cnt;
        const int a_lo = min(lo, ri.y), a_hi = min(hi, ri.y);
        const int b_lo = max(lo, ri.y) - ri.y, b_hi = max(hi, ri.y) - ri.y;
        float* dst = s_rec + (size_t)nb * cap * recf + (size_t)so * recf;
        if (a_hi > a_lo)
          bulk_g2s(dst, rec + (size_t)(ri.x + a_lo) * recf, (uint32_t)(a_hi - a_lo) * recf * 4u, &full[nb]);
        if (b_hi > b_lo)
          bulk_g2s(dst + (size_t)(a_hi - a_lo) * recf, rec + (size_t)(ri.z + b_lo) * recf,
                   (uint32_t)(b_hi - b_lo) * recf * 4u, &full[nb]);
      }
    }
    return nd;
  };

  if (tid == 0) {
    for (int i = 0; i < NS; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], WY * WZ); }
    for (int i = 0; i < NTAB; ++i) mbar_init(&tabfree[i], WY * WZ);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == WY * WZ) {
    // ---- producer warp: cell-boundary tables one plane ahead, rounds two ahead of the consumers.
    //      Table slot (p+1) % NTAB last served plane p+1-NTAB; build_plane waits for the consumers to
    //      hand it back (tabfree) after its loads are in flight.
    //      The round counter n and the plane counter run on through the CTA's segments; a segment's
    //      last round is the one that completes plane pe-1 (every plane has at least one round), so no
    //      terminal descriptor is needed.
    int n = 0;
    for (int sg = 0; sg < nsg; ++sg) {
      if (sg) set_segment(sg);
      build_plane(pb);
      __syncwarp();
      int pn = pb, rn = 0, an = 0;
      for (;; ++n) {
        const int nb = n % NS;
        if (n >= NS) mbar_wait(&empty[nb], ((n / NS) - 1) & 1);
        const RoundDesc nd = build_round(pn, rn, an, nb);
        if (nd.r0 == 0 && nd.a0 == 0 && nd.p + 1 < pe) { build_plane(nd.p + 1); __syncwarp(); }
        pn = nd.np; rn = nd.nr; an = nd.na;
        if (pn >= pe) { ++n; break; }
      }
    }
    return;
  }

  f32x2 acc[SW / 2][2][CB];   // register window: acc[k/2][column][channel] = {plane k, plane k+1}, k = x mod 8
#pragma unroll
  for (int k = 0; k < SW / 2; ++k)
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int c = 0; c < CB; ++c) acc[k][u][c] = 0ull;

  // ---- consumer warps: free-running, coupled to the producer (and to nothing else) by the barriers
  int sg = 0;
  for (int n = 0;; ++n) {
    const int cur = n % NS;
    mbar_wait(&full[cur], (n / NS) & 1);
    const RoundDesc d = s_desc[cur];
    // ---- this thread's atoms of the round ----
    {
      const int tb = d.p % NTAB;
      const int r_beg = max(rlo, d.r0);
      const int r_hi = lane_ok ? min(rlo + SW, d.r1) : r_beg;
      const int total =
          build_runs(s_run, NT, r_beg, r_hi, s_L + (size_t)tb * NROW * NB + clo, NB, NROW, s_rowoff + cur * 32, d.a0, d.a1);
      if (d.flush) {   // the plane's last round: its cell-boundary table goes back to the producer
        __syncwarp();
        if (lane == 0) mbar_arrive(&tabfree[tb]);
      }
      walk_atoms<CB>(acc, s_run, NT, total, s_rec + (size_t)cur * cap * recf, recf, cb0, oy, oz);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[cur]);   // this warp is done with the staged records and the round's offsets
    // ---- plane complete: its slot leaves the window; after the last cell plane so do the 7 planes
    //      beyond it.  Planes shared with a neighbouring segment are added (RED), the others stored.
    if (d.flush && lane_ok) {
      const int nfl = d.p == pe - 1 ? SW : 1;
      for (int i = 0; i < nfl; ++i) {
        const int pl = d.p - pb + i;
        int P = X0 + pl; if (P >= Mx) P -= Mx;
        const bool shared = pl < SW - 1 || pl >= NP;
        float* gp = grid + (size_t)cb0 * Mtot + ((size_t)P * My + y) * Mz + z0;
        switch (P & 7) {
#define PSWF_FLUSH(K)                                                                          \
  case K:                                                                                      \
    _Pragma("unroll") for (int c = 0; c < CB; ++c) {                                           \
      float a0, a1, b0, b1;                                                                    \
      unpack2(acc[K / 2][0][c], a0, a1);                                                       \
      unpack2(acc[K / 2][1][c], b0, b1);                                                       \
      const float s0 = (K & 1) ? a1 : a0, s1 = (K & 1) ? b1 : b0;                              \
      if (shared) red_add_v2(gp + (size_t)c * Mtot, s0, s1);                                   \
      else *reinterpret_cast<float2*>(gp + (size_t)c * Mtot) = make_float2(s0, s1);            \
      if (K & 1) { zero_hi(acc[K / 2][0][c]); zero_hi(acc[K / 2][1][c]); }                     \
      else { zero_lo(acc[K / 2][0][c]); zero_lo(acc[K / 2][1][c]); }                           \
    }                                                                                          \
    break;
          PSWF_FLUSH(0) PSWF_FLUSH(1) PSWF_FLUSH(2) PSWF_FLUSH(3)
          PSWF_FLUSH(4) PSWF_FLUSH(5) PSWF_FLUSH(6) PSWF_FLUSH(7)
#undef PSWF_FLUSH
        }
      }
    }
    if (d.flush && d.p == pe - 1) {   // the segment's last round: on to the CTA's second segment, if any
      if (++sg == nsg) break;
      set_segment(sg);
      set_columns();
    }
  }
}

template <int WY, int WZ, int NCTA>
struct SpreadLaunch {
  using S = SpreadShape<WY, WZ>;
  static size_t smem_bytes(int cap, int recf) { return S::kHeader + S::kTables + S::kRuns + S::kStages * (size_t)cap * recf * 4; }

  template <int CB>
  static void run(pswf_lr_plan* p, int ncta, int cap, int recf, int cb0, cudaStream_t st) {
    const int Mx = p->M[0], My = p->M[1], Mz = p->M[2];
    const int npy = (My + S::TY - 1) / S::TY, npz = (Mz + S::TZ - 1) / S::TZ;
    const size_t sm = smem_bytes(cap, recf);
    auto kern = k_spread_os<WY, WZ, CB, NCTA>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    p->n_kernels += 1;
    kern<<<(unsigned)ncta, S::NT + 32, sm, st>>>(Mx, My, Mz, npy, npz, cap, recf, cb0, p->d_count,
                                                         (const float*)p->d_rec, (float*)p->d_grid);
  }

  static void all_channels(pswf_lr_plan* p, cudaStream_t st) {
    const int recf = stencil_rec_floats(p->C);
    // staging capacity: NCTA CTAs per SM
    const size_t budget = (size_t)(228 * 1024) / NCTA - 1024;   // 228 KB per SM, 1 KB of it reserved per CTA
    int cap = (int)((budget - S::kHeader - S::kTables - S::kRuns) / (S::kStages * (size_t)recf * 4));
    cap &= ~7;
    // ONE full wave of CTAs, each with the same number of (patch, cell plane) pairs.  The atoms are
    // partitioned over the segments, so short segments cost no extra arithmetic, only RED traffic for the
    // 7 shared planes; a second, partly filled wave would cost a full segment time (512 CTAs on 444 slots;
    // profiles/r1b).  On small grids down to one cell plane per CTA: the planes of a CTA are a latency
    // chain of ~2.5 us each (42 -> 15 us at configuration 2 against 8 planes per CTA).
    const int npatch = ((p->M[1] + S::TY - 1) / S::TY) * ((p->M[2] + S::TZ - 1) / S::TZ);
    const int nseg = std::max(1, std::min(NCTA * p->sm_count, npatch * p->M[0]));
    // (the RED-merged planes start from zero: the grid is zeroed with the sort's buffers at the start of the
    // evaluation, launch_bin_sort)
    int cb0 = 0;
    while (cb0 < p->C) {
      const int left = p->C - cb0;
      if (left >= 4) { run<4>(p, nseg, cap, recf, cb0, st); cb0 += 4; }
      else if (left == 3) { run<3>(p, nseg, cap, recf, cb0, st); cb0 += 3; }
      else if (left == 2) { run<2>(p, nseg, cap, recf, cb0, st); cb0 += 2; }
      else { run<1>(p, nseg, cap, recf, cb0, st); cb0 += 1; }
    }
  }
};

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int stencil_rec_floats(int C) {
  int f = 3 * SW + ((C + 3) / 4) * 4;
  if (((f / 4) & 1) == 0) f += 4;   // odd number of 16-byte quads: consecutive records hit distinct banks
  return f;
}

bool stencil_path_supported(const pswf_lr_plan* p) {
  if (p->precision != PSWF_LR_F32 || p->w > SW || p->wt.degree > kFastWindowDegree) return false;
  for (int d = 0; d < 3; ++d)
    if (p->M[d] % SW != 0 || p->M[d] < 2 * SW) return false;
  return true;
}

size_t stencil_record_bytes(const pswf_lr_plan* p) { return sizeof(float) * stencil_rec_floats(p->C); }
size_t stencil_drecord_bytes(const pswf_lr_plan*) { return sizeof(float) * 3 * SW; }

void launch_scatter_records(pswf_lr_plan* p, int n, const float* pos, const float* q, const GridGeom<float>& g,
                            cudaStream_t st) {
  if (n <= 0) return;
  const int recf = stencil_rec_floats(p->C);
  p->n_kernels += 2;
  k_perm<<<(n + 255) / 256, 256, 0, st>>>(n, p->d_count, p->d_key, p->d_rank, p->d_perm);
  const size_t sm = sizeof(float) * kRecThreads * (size_t)recf;
  const unsigned nb = (unsigned)((n + kRecThreads - 1) / kRecThreads);
#define PSWF_REC(D)                                                                                              \
  case D:                                                                                                        \
    k_records<D><<<nb, kRecThreads, sm, st>>>(n, p->C, recf, pos, q, g, p->wpoly, p->d_perm, (float*)p->d_rec,   \
                                              (float*)p->d_drec);                                                \
    break;
  switch (std::max(p->wt.degree, 6)) {   // Horner steps beyond the plan's degree would multiply zeros
    PSWF_REC(6) PSWF_REC(7) PSWF_REC(8) PSWF_REC(9) PSWF_REC(10) PSWF_REC(11)
    default:
      k_records<kFastWindowDegree><<<nb, kRecThreads, sm, st>>>(n, p->C, recf, pos, q, g, p->wpoly, p->d_perm,
                                                                (float*)p->d_rec, (float*)p->d_drec);
  }
#undef PSWF_REC
}

void launch_stencil_spread(pswf_lr_plan* p, int n, cudaStream_t st) {
  (void)n;
  // 16 x 16 column patches: 4 consumer warps + 1 producer warp, three CTAs per SM (<= 128 registers).
  // Measured at configuration 4 (end of round 2): 244 us.  Rejected: 16 x 32 patches x 2 CTAs (113-register cap:
  // spills), 16 x 16 x 4 CTAs, 136 registers x 2 CTAs.
  SpreadLaunch<2, 2, 3>::all_channels(p, st);
}

}  // namespace pswf
