// Reference-quality CUDA kernels of the PSWF-LR path: binning/counting sort, warp-per-atom
// spread with global atomics, the fused scale+reduce kernel over the half spectrum, and a
// warp-per-atom gather.  They run every configuration in both precisions (any even w <= 16,
// any channel count); the fp64 path and kernel_path = 1 always use them.  The tiled fp32
// kernels in kernels_stencil.cu / kernels_gather.cu replace sort-scatter, spread and gather on the
// default path.
#include <atomic>

#include "kernels_common.cuh"
#include "kernels_scale.cuh"
#include "launch.hpp"

namespace pswf {

// ------------------------------------------------------------------------------------------------
// a0. bin + counting sort (not in the paper, required by tiled kernels).
// Key = stencil cell (s_x, s_y, s_z), s_d = i0_d mod M_d, z fastest.
// ------------------------------------------------------------------------------------------------
template <class T>
__global__ void k_bin_count(int n, const T* __restrict__ pos, GridGeom<T> g, int* __restrict__ count,
                            int* __restrict__ key, int* __restrict__ rank) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int s[3], i0[3];
  double delta[3];
  stencil_3d(pos + 3 * (size_t)i, g.hinv, g.M, g.w, i0, delta);
#pragma unroll
  for (int d = 0; d < 3; ++d) s[d] = wrap_index(i0[d], g.M[d]);
  int k = (s[0] * g.M[1] + s[1]) * g.M[2] + s[2];
  key[i] = k;
  rank[i] = atomicAdd(&count[k], 1);
}

// Exclusive scan of count[0..n) in place in ONE pass (decoupled look-back): a tile of 16384 counts per
// CTA; tiles are handed out by a ticket counter, so every tile a CTA waits for is already running.
// state[0] = ticket counter, state[1 + t] = (status << 32) | value of tile t with status 1 = the
// tile's own sum, 2 = inclusive prefix up to and including the tile; zeroed before each launch.
constexpr int kScanThreads = 1024;
constexpr int kScanItems = 16;   // 16384 counts per tile: 128 tiles at 128^3, one wave, a 4x shorter look-back chain than 4096
int scan_tile_size() { return kScanThreads * kScanItems; }

__global__ void __launch_bounds__(kScanThreads) k_scan_lookback(int n, int* __restrict__ data,
                                                                unsigned long long* __restrict__ state,
                                                                int total_slot, int total) {
  __shared__ int warp_tot[kScanThreads / 32];
  __shared__ int s_tile, s_prefix;
  if (threadIdx.x == 0) s_tile = (int)atomicAdd(reinterpret_cast<unsigned int*>(state), 1u);
  __syncthreads();
  const int tile = s_tile;
  const int base = (tile * kScanThreads + threadIdx.x) * kScanItems;
  int v[kScanItems];
  int sum = 0;
  if (base + kScanItems <= n) {
#pragma unroll
    for (int j = 0; j < kScanItems; j += 4) {
      const int4 a = *reinterpret_cast<const int4*>(data + base + j);
      v[j] = a.x; v[j + 1] = a.y; v[j + 2] = a.z; v[j + 3] = a.w;
    }
  } else {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) v[j] = (base + j < n) ? data[base + j] : 0;
  }
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) sum += v[j];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    int t = (lane < kScanThreads / 32) ? warp_tot[lane] : 0;
    int inc = t;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    if (lane < kScanThreads / 32) warp_tot[lane] = inc - t;  // exclusive warp offsets
    const int tile_sum = __shfl_sync(0xffffffffu, inc, 31);
    volatile unsigned long long* st = state + 1;
    int prefix = 0;
    if (tile == 0) {
      if (lane == 0) st[0] = (2ull << 32) | (unsigned int)tile_sum;
    } else {
      if (lane == 0) st[tile] = (1ull << 32) | (unsigned int)tile_sum;
      // warp-wide look-back: lane l inspects tile (p - l); the window moves back 32 tiles at a time
      for (int p = tile - 1;; p -= 32) {
        unsigned long long sv = 2ull << 32;            // tiles before 0: an inclusive prefix of 0
        unsigned ready;
        do {
          if (p - lane >= 0) sv = st[p - lane];
          ready = __ballot_sync(0xffffffffu, (sv >> 32) != 0ull);
          // only the lanes up to the first inclusive prefix have to be valid
          const unsigned incl_mask = __ballot_sync(0xffffffffu, (sv >> 32) == 2ull);
          const unsigned need = incl_mask ? ((incl_mask & (0u - incl_mask)) << 1) - 1u : 0xffffffffu;
          if ((ready & need) == need) {
            int pv = ((need >> lane) & 1u) ? (int)(unsigned int)sv : 0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) pv += __shfl_xor_sync(0xffffffffu, pv, o);
            prefix += pv;
            ready = incl_mask ? 0xffffffffu : 0xfffffffeu;   // all-ones: done; else: next window
            break;
          }
        } while (true);
        if (ready == 0xffffffffu) break;
      }
      if (lane == 0) st[tile] = (2ull << 32) | (unsigned int)(prefix + tile_sum);
    }
    if (lane == 0) s_prefix = prefix;
  }
  __syncthreads();
  int run = s_prefix + warp_tot[wid] + incl - sum;
  if (base + kScanItems <= n) {
    int o[kScanItems];
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) { o[j] = run; run += v[j]; }
#pragma unroll
    for (int j = 0; j < kScanItems; j += 4)
      *reinterpret_cast<int4*>(data + base + j) = make_int4(o[j], o[j + 1], o[j + 2], o[j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
      if (base + j < n) data[base + j] = run;
      run += v[j];
    }
  }
  if (tile == 0 && threadIdx.x == 0) data[total_slot] = total;
}

// ------------------------------------------------------------------------------------------------
// No-allocation variant of the scan (pswf_lr_exclusive_scan_static, include/pswf_lr.h): the tile state
// lives in a file-scope device array instead of the plan's cudaMalloc'd d_scan_state.  8200 bytes, held by
// every GPU that loads the library until the process exits.  All calls share it: calls that overlap on
// the GPU (two streams) race.
// ------------------------------------------------------------------------------------------------
constexpr int kScanStaticTiles = PSWF_LR_SCAN_STATIC_MAX / (kScanThreads * kScanItems);   // 1024 tiles of 16384 counts
static_assert(kScanStaticTiles * kScanThreads * kScanItems == PSWF_LR_SCAN_STATIC_MAX, "whole tiles");
static __device__ __align__(256) unsigned long long g_scan_state_static[kScanStaticTiles + 1];

// the inclusive prefix of the last tile is the total
__global__ void k_scan_total(const unsigned long long* __restrict__ state, int ntiles, int* __restrict__ out) {
  if (blockIdx.x == 0 && threadIdx.x == 0) *out = (int)(unsigned int)state[ntiles];
}

// In host code g_scan_state_static is a host-side stand-in, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, looked up once per device with that device current (no allocation).
int launch_scan_static(int* data, int n, cudaStream_t st) {
  constexpr int kDevs = 64;
  static std::atomic<unsigned long long*> cache[kDevs];
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return PSWF_LR_ERR_CUDA; }
  unsigned long long* state = (dev >= 0 && dev < kDevs) ? cache[dev].load() : nullptr;
  if (!state) {
    if (cudaGetSymbolAddress((void**)&state, g_scan_state_static) != cudaSuccess || !state) {
      cudaGetLastError();
      return PSWF_LR_ERR_CUDA;
    }
    if (dev >= 0 && dev < kDevs) cache[dev].store(state);
  }
  const int ntiles = (n + kScanThreads * kScanItems - 1) / (kScanThreads * kScanItems);
  // the array keeps the previous call's ticket counter and tile states: all of what this call uses restarts at zero
  if (cudaMemsetAsync(state, 0, sizeof(unsigned long long) * ((size_t)ntiles + 1), st) != cudaSuccess) {
    cudaGetLastError();
    return PSWF_LR_ERR_CUDA;
  }
  k_scan_lookback<<<ntiles, kScanThreads, 0, st>>>(n, data, state, n, 0);
  k_scan_total<<<1, 32, 0, st>>>(state, ntiles, data + n);
  if (cudaGetLastError() != cudaSuccess) return PSWF_LR_ERR_CUDA;
  return 0;
}

template <class T>
__global__ void k_scatter(int n, int C, int cap, const T* __restrict__ pos, const T* __restrict__ q,
                          GridGeom<T> g, const int* __restrict__ start, const int* __restrict__ key,
                          const int* __restrict__ rank, int* __restrict__ perm, int* __restrict__ si0,
                          T* __restrict__ sdelta, T* __restrict__ sq) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int dst = start[key[i]] + rank[i];
  perm[dst] = i;
  int i0[3];
  double delta[3];
  stencil_3d(pos + 3 * (size_t)i, g.hinv, g.M, g.w, i0, delta);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    si0[(size_t)d * cap + dst] = i0[d];
    sdelta[(size_t)d * cap + dst] = (T)delta[d];
  }
  for (int c = 0; c < C; ++c) sq[(size_t)c * cap + dst] = q[(size_t)c * n + i];
}

// ------------------------------------------------------------------------------------------------
// a1. spread, reference kernel: one warp per atom, w^3 global atomic adds per channel.
// rho_g^a = sum_j q_j^a prod_d psi((x_{g,d} - r_{j,d}) / omega_d)     Eq. (20)-(21),(24)
// ------------------------------------------------------------------------------------------------
template <class T>
__global__ void k_spread_ref(int n, int C, int cap, GridGeom<T> g, const int* __restrict__ si0,
                             const T* __restrict__ sdelta, const T* __restrict__ sq, T* __restrict__ grid) {
  __shared__ T wts[8][3 * kMaxW];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int j = blockIdx.x * 8 + wid;
  if (j >= n) return;
  const int w = g.w;
  for (int t = lane; t < 3 * w; t += 32) {
    int d = t / w, tt = t - d * w;
    T xi = (T)2 * sdelta[(size_t)d * cap + j] - (T)1;
    wts[wid][d * kMaxW + tt] = horner_panel(g.wcoef, w, tt, g.wdeg, xi);
  }
  __syncwarp();
  const int i0x = si0[j], i0y = si0[(size_t)cap + j], i0z = si0[2 * (size_t)cap + j];
  const size_t Mtot = (size_t)g.M[0] * g.M[1] * g.M[2];
  const int w3 = w * w * w;
  for (int idx = lane; idx < w3; idx += 32) {
    int a = idx / (w * w), r = idx - a * w * w, b = r / w, cc = r - b * w;
    T wt = wts[wid][a] * wts[wid][kMaxW + b] * wts[wid][2 * kMaxW + cc];
    size_t gi = ((size_t)wrap_index(i0x + a, g.M[0]) * g.M[1] + wrap_index(i0y + b, g.M[1])) * g.M[2] +
                wrap_index(i0z + cc, g.M[2]);
    for (int c = 0; c < C; ++c) atomicAdd(&grid[(size_t)c * Mtot + gi], sq[(size_t)c * cap + j] * wt);
  }
}

// ------------------------------------------------------------------------------------------------
// a3. scale (deconvolve x Green) + Fourier-space energy reduction, fused over channels.
// phi^_a(m) = D_{p_a}(m) rho^_a(m),  D_p(m) = (h_x h_y h_z / M_tot) Phi^_p(|k_m|) / W^(k_m)^2
// (Eq. (22),(25); reading R10), zero for |k| r_c >= c and on Nyquist planes (R11);
// E_a = 1/2 sum_m D |rho^_a(m)|^2 (Eq. (26)) with Hermitian weights over the half spectrum.
// Phi^_p is evaluated once per distinct exponent per mode by Horner on the smooth part
// and reused by every channel with that exponent.
// ------------------------------------------------------------------------------------------------
// (Cplx, kernel_value, kernel_dvalue: kernels_scale.cuh)
// VIR: also accumulate the virial W_ab = 1/2 sum_m' |rho^|^2 [D delta_ab + (dD/dk) k_a k_b / |k|] of the
// discrete energy (its exact strain derivative: the window transform depends on k h only, which a
// homogeneous strain leaves unchanged) into Wacc[6] = xx, yy, zz, xy, xz, yz.
template <class T, bool VIR>
__global__ void k_scale(ScaleParams<T> P, Cplx<T>* __restrict__ spec, double* __restrict__ Ech, int want_E,
                        double* __restrict__ Wacc) {
  const size_t Mhalf = (size_t)P.M[0] * P.M[1] * P.Mzh;
  const size_t m = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  __shared__ double red[kMaxChannels];
  __shared__ double redw[6];
  if (threadIdx.x < kMaxChannels) red[threadIdx.x] = 0.0;
  if (VIR && threadIdx.x < 6) redw[threadIdx.x] = 0.0;
  __syncthreads();
  bool active = m < Mhalf;
  bool inside = false;
  T D[kMaxSlots];
  T dDk[kMaxSlots];    // (dD/dk) / |k| per slot
  T kv[3] = {(T)0, (T)0, (T)0};
  double wloc[6] = {0, 0, 0, 0, 0, 0};
  T herm = (T)0;
  int iz = 0;
  bool is_zero_mode = false;
  if (active) {
    iz = (int)(m % P.Mzh);
    size_t r = m / P.Mzh;
    int iy = (int)(r % P.M[1]);
    int ix = (int)(r / P.M[1]);
    int fx = ix <= P.M[0] / 2 ? ix : ix - P.M[0];
    int fy = iy <= P.M[1] / 2 ? iy : iy - P.M[1];
    int fz = iz;
    bool nyq = ((P.M[0] % 2 == 0) && ix == P.M[0] / 2) || ((P.M[1] % 2 == 0) && iy == P.M[1] / 2) ||
               ((P.M[2] % 2 == 0) && iz == P.M[2] / 2);
    const T kx = P.recip[0] * (T)fx + P.recip[3] * (T)fy + P.recip[6] * (T)fz;
    const T ky = P.recip[1] * (T)fx + P.recip[4] * (T)fy + P.recip[7] * (T)fz;
    const T kz = P.recip[2] * (T)fx + P.recip[5] * (T)fy + P.recip[8] * (T)fz;
    T kn = sqrt(kx * kx + ky * ky + kz * kz);
    T x = kn * P.x_per_k;
    is_zero_mode = (ix == 0 && iy == 0 && iz == 0);
    inside = !nyq && !is_zero_mode && x < (T)1;
    herm = (iz == 0 || ((P.M[2] % 2 == 0) && iz == P.M[2] / 2)) ? (T)1 : (T)2;
    if (inside) {
      T base = P.base * P.invW2[0][ix] * P.invW2[1][iy] * P.invW2[2][iz];
      T kappa = x * P.c;
      for (int s = 0; s < P.nslots; ++s) D[s] = base * kernel_value(P, s, x, kappa);
      if (VIR) {
        kv[0] = kx; kv[1] = ky; kv[2] = kz;
        for (int s = 0; s < P.nslots; ++s) dDk[s] = base * kernel_dvalue(P, s, x, kappa) / kn;
      }
    }
  }
  for (int c = 0; c < P.C; ++c) {
    double e = 0.0;
    if (active) {
      Cplx<T>* ptr = spec + (size_t)c * Mhalf + m;
      if (inside || is_zero_mode) {
        T d = is_zero_mode ? P.chan_D0[c] : D[P.chan_slot[c]];
        Cplx<T> v = *ptr;
        const T a2 = herm * (v.x * v.x + v.y * v.y);
        e = (double)(a2 * d);
        if (VIR) {
          wloc[0] += e; wloc[1] += e; wloc[2] += e;
          if (!is_zero_mode) {
            const double g = (double)(a2 * dDk[P.chan_slot[c]]);
            wloc[0] += g * kv[0] * kv[0]; wloc[1] += g * kv[1] * kv[1]; wloc[2] += g * kv[2] * kv[2];
            wloc[3] += g * kv[0] * kv[1]; wloc[4] += g * kv[0] * kv[2]; wloc[5] += g * kv[1] * kv[2];
          }
        }
        v.x *= d;
        v.y *= d;
        *ptr = v;
      } else {
        Cplx<T> z;
        z.x = (T)0;
        z.y = (T)0;
        *ptr = z;  // outside the band: no read, just clear
      }
    }
    if (want_E) {
      e = warp_sum(e);
      if ((threadIdx.x & 31) == 0 && e != 0.0) atomicAdd(&red[c], e);
    }
  }
  if (want_E) {
    __syncthreads();
    if (threadIdx.x < P.C && red[threadIdx.x] != 0.0) atomicAdd(&Ech[threadIdx.x], 0.5 * red[threadIdx.x]);
  }
  if (VIR) {
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      const double t = warp_sum(wloc[i]);
      if ((threadIdx.x & 31) == 0 && t != 0.0) atomicAdd(&redw[i], t);
    }
    __syncthreads();
    if (threadIdx.x < 6 && redw[threadIdx.x] != 0.0) atomicAdd(&Wacc[threadIdx.x], 0.5 * redw[threadIdx.x]);
  }
}

__global__ void k_finalize_energy(int C, const double* __restrict__ Ech, double* __restrict__ E) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double s = 0.0;
    for (int c = 0; c < C; ++c) s += Ech[c];
    *E = s;
  }
}

// ------------------------------------------------------------------------------------------------
// a5. gather + force, reference kernel: one warp per atom.
// phi_i^a = sum_g W(x_g - r_i) phi_g^a;  grad = sum_g grad_{r_i} W phi_g^a (derivative of the SAME
// panel polynomials);  F_i = - sum_a q_i^a grad phi_i^a.
// ------------------------------------------------------------------------------------------------
template <class T>
__global__ void k_gather_ref(int n, int C, int cap, GridGeom<T> g, const int* __restrict__ si0,
                             const T* __restrict__ sdelta, const T* __restrict__ sq,
                             const int* __restrict__ perm, const T* __restrict__ grid, T* __restrict__ phi,
                             T* __restrict__ F) {
  __shared__ T wts[8][6 * kMaxW];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int j = blockIdx.x * 8 + wid;
  if (j >= n) return;
  const int w = g.w;
  for (int t = lane; t < 3 * w; t += 32) {
    int d = t / w, tt = t - d * w;
    T xi = (T)2 * sdelta[(size_t)d * cap + j] - (T)1;
    wts[wid][d * kMaxW + tt] = horner_panel(g.wcoef, w, tt, g.wdeg, xi);
    wts[wid][(3 + d) * kMaxW + tt] = horner_panel(g.wdcoef, w, tt, g.wdeg - 1, xi) * g.dxi_ds[d];
  }
  __syncwarp();
  const int i0x = si0[j], i0y = si0[(size_t)cap + j], i0z = si0[2 * (size_t)cap + j];
  const size_t Mtot = (size_t)g.M[0] * g.M[1] * g.M[2];
  const int w3 = w * w * w;
  const int dst = perm[j];
  T fx = 0, fy = 0, fz = 0;
  for (int c = 0; c < C; ++c) {
    T v = 0, gx = 0, gy = 0, gz = 0;
    const T* gc = grid + (size_t)c * Mtot;
    for (int idx = lane; idx < w3; idx += 32) {
      int a = idx / (w * w), r = idx - a * w * w, b = r / w, cc = r - b * w;
      size_t gi = ((size_t)wrap_index(i0x + a, g.M[0]) * g.M[1] + wrap_index(i0y + b, g.M[1])) * g.M[2] +
                  wrap_index(i0z + cc, g.M[2]);
      T val = gc[gi];
      T wx = wts[wid][a], wy = wts[wid][kMaxW + b], wz = wts[wid][2 * kMaxW + cc];
      T dx = wts[wid][3 * kMaxW + a], dy = wts[wid][4 * kMaxW + b], dz = wts[wid][5 * kMaxW + cc];
      T yz = wy * wz * val;
      v += wx * yz;
      gx += dx * yz;
      gy += wx * dy * wz * val;
      gz += wx * wy * dz * val;
    }
    v = warp_sum(v);
    gx = warp_sum(gx);
    gy = warp_sum(gy);
    gz = warp_sum(gz);
    T qc = sq[(size_t)c * cap + j];
    fx -= qc * gx;
    fy -= qc * gy;
    fz -= qc * gz;
    if (lane == 0 && phi) phi[(size_t)c * n + dst] = v;
  }
  if (lane == 0 && F) {
    frac_to_cart(g.hinv_t, fx, fy, fz);   // the derivative weights are along the fractional coordinates
    F[3 * (size_t)dst + 0] = fx;
    F[3 * (size_t)dst + 1] = fy;
    F[3 * (size_t)dst + 2] = fz;
  }
}

// ------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------
template <class T>
void launch_bin_sort(pswf_lr_plan* p, int n, const T* pos, const T* q, const GridGeom<T>& g, bool scatter,
                     bool zero_energy, cudaStream_t st) {
  const int Mtot = p->M[0] * p->M[1] * p->M[2];
  // one memset: cell counts + scan state (an evaluation: also the energy / virial accumulators in front of them
  // and the charge grid behind them, plan.hpp)
  if (zero_energy) cudaMemsetAsync(p->d_zero_block, 0, p->zero_block_bytes, st);
  else cudaMemsetAsync((char*)p->d_zero_block + p->zero_sort_offset, 0, p->zero_sort_bytes, st);
  p->n_memsets += 1;
  p->n_kernels += (n > 0 ? 1 : 0) + 1 + ((n > 0 && scatter) ? 1 : 0);
  if (n > 0)
    k_bin_count<T><<<(n + 255) / 256, 256, 0, st>>>(n, pos, g, p->d_count, p->d_key, p->d_rank);
  k_scan_lookback<<<p->n_scan_blocks, kScanThreads, 0, st>>>(Mtot, p->d_count, p->d_scan_state, Mtot, n);
  if (n > 0 && scatter)
    k_scatter<T><<<(n + 255) / 256, 256, 0, st>>>(n, p->C, p->cap_atoms, pos, q, g, p->d_count, p->d_key,
                                                   p->d_rank, p->d_perm, p->d_si0, (T*)p->d_sdelta,
                                                   (T*)p->d_sq);
}

template <class T>
void launch_spread_ref(pswf_lr_plan* p, int n, const GridGeom<T>& g, cudaStream_t st) {
  // (the grid was zeroed with the sort's buffers at the start of the evaluation, launch_bin_sort)
  p->n_kernels += n > 0 ? 1 : 0;
  if (n > 0)
    k_spread_ref<T><<<(n + 7) / 8, 256, 0, st>>>(n, p->C, p->cap_atoms, g, p->d_si0, (const T*)p->d_sdelta,
                                                  (const T*)p->d_sq, (T*)p->d_grid);
}

template <class T>
void launch_scale(pswf_lr_plan* p, const ScaleParams<T>& P, bool want_E, cudaStream_t st) {
  const size_t Mhalf = (size_t)P.M[0] * P.M[1] * P.Mzh;
  const int threads = 256;
  const unsigned nb = (unsigned)((Mhalf + threads - 1) / threads);
  p->n_kernels += 1;
  if (p->virial)
    k_scale<T, true><<<nb, threads, 0, st>>>(P, (Cplx<T>*)p->d_spec, p->d_Ech, want_E ? 1 : 0, p->d_virial);
  else
    k_scale<T, false><<<nb, threads, 0, st>>>(P, (Cplx<T>*)p->d_spec, p->d_Ech, want_E ? 1 : 0, nullptr);
}

void launch_finalize_energy(pswf_lr_plan* p, double* E, cudaStream_t st) {
  p->n_kernels += 1;
  k_finalize_energy<<<1, 32, 0, st>>>(p->C, p->d_Ech, E);
}

template <class T>
void launch_gather_ref(pswf_lr_plan* p, int n, const GridGeom<T>& g, T* phi, T* F, cudaStream_t st) {
  p->n_kernels += n > 0 ? 1 : 0;
  if (n > 0)
    k_gather_ref<T><<<(n + 7) / 8, 256, 0, st>>>(n, p->C, p->cap_atoms, g, p->d_si0, (const T*)p->d_sdelta,
                                                  (const T*)p->d_sq, p->d_perm, (const T*)p->d_grid, phi, F);
}

#define PSWF_INSTANTIATE(T)                                                                               \
  template void launch_bin_sort<T>(pswf_lr_plan*, int, const T*, const T*, const GridGeom<T>&, bool, bool, cudaStream_t); \
  template void launch_spread_ref<T>(pswf_lr_plan*, int, const GridGeom<T>&, cudaStream_t);              \
  template void launch_scale<T>(pswf_lr_plan*, const ScaleParams<T>&, bool, cudaStream_t);               \
  template void launch_gather_ref<T>(pswf_lr_plan*, int, const GridGeom<T>&, T*, T*, cudaStream_t);
PSWF_INSTANTIATE(float)
PSWF_INSTANTIATE(double)

}  // namespace pswf
