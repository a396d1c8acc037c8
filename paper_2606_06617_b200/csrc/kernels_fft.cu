// Band-limited transform path of the fast fp32 pipeline (a2-a4): z transforms by cuFFT, and ONE
// kernel that does, per kept k_z plane and channel, the forward (x,y) transform, the deconvolve x
// Green multiply with the Fourier-space energy reduction (Eq. (22),(25),(26)) and the
// inverse (x,y) transform, entirely in shared memory.
//
// Why: Phi^_p(k) == 0 for |k| r_c >= c, and with eta = h c / (pi r_c) = 0.5 that ball
// reaches only |m_d| < M_d / 4: 6.4% of the half spectrum.  The dense path (3-D cuFFT, k_scale over
// the whole half spectrum, 3-D cuFFT back) moves ~480 MB per evaluation at config 4 for a result
// that lives in 63 x 63 x 32 modes per channel.  Here
//   * cuFFT R2C along z writes the spectrum PLANE-MAJOR, [k_z][c][x][y] (output stride C Mx My), so a
//     (k_z, c) plane is one contiguous Mx x My block and the planes beyond the band are never read;
//   * k_xy_scale loads one plane into shared memory (Mx x (My+1) complex, 132 KB at 128 x 128), runs
//     decimation-in-frequency passes along x for every y, along y only for the kept k_x, multiplies
//     by D_p(m) in the resulting digit-reversed order (no reordering pass: a position -> frequency table
//     does it), zeroes what lies outside the band, and runs the decimation-in-time inverse passes;
//   * cuFFT C2R along z reads a second plane-major buffer whose planes beyond the band are zero from
//     plan creation on and are never written.
// Requirements (host-checked; otherwise the dense path runs): fp32, Mx and My powers of two in
// 8..256 with the padded plane fitting shared memory.  With pswf_lr_set_virial the same pass accumulates the
// virial of the reciprocal energy (VIR variants).
#include <algorithm>
#include <cmath>

#include "kernels_common.cuh"
#include "kernels_scale.cuh"
#include "launch.hpp"

namespace pswf {

namespace {

constexpr int kXYThreads = 1024;

struct XYParams {
  int Mx, My, pitch, C;
  int nrx, rx[4], nry, ry[4];   // radices of the forward passes along x / y (product = Mx / My)
  int kmaxx, kmaxy;             // kept signed frequencies: |f| <= kmax
  int Mzh;                      // Mz/2 + 1 (stride of the dump layout)
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// multiply by -i (forward, e^{-i...}) or +i (inverse)
template <bool INV>
__device__ __forceinline__ float2 rot90(float2 a) {
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

template <int R, bool INV>
struct Dft;
template <bool INV>
struct Dft<2, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[2]) {
    const float2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};
template <bool INV>
struct Dft<4, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[4]) {
    const float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
    const float2 t2 = cadd(v[1], v[3]), t3 = rot90<INV>(csub(v[1], v[3]));
    v[0] = cadd(t0, t2);
    v[2] = csub(t0, t2);
    v[1] = cadd(t1, t3);
    v[3] = csub(t1, t3);
  }
};
template <bool INV>
struct Dft<8, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[8]) {
    float2 e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
    Dft<4, INV>::run(e);
    Dft<4, INV>::run(o);
    const float h = 0.70710678118654752f;
    // W8^1 = (1 -+ i)/sqrt2, W8^2 = -+ i, W8^3 = (-1 -+ i)/sqrt2   (upper sign: forward)
    const float2 w1 = INV ? make_float2(h, h) : make_float2(h, -h);
    const float2 w3 = INV ? make_float2(-h, h) : make_float2(-h, -h);
    o[1] = cmul(o[1], w1);
    o[2] = rot90<INV>(o[2]);
    o[3] = cmul(o[3], w3);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      v[k] = cadd(e[k], o[k]);
      v[k + 4] = csub(e[k], o[k]);
    }
  }
};

template <bool INV>
struct Dft<16, INV> {
  static __device__ __forceinline__ void run(float2 (&v)[16]) {
    float2 e[8] = {v[0], v[2], v[4], v[6], v[8], v[10], v[12], v[14]};
    float2 o[8] = {v[1], v[3], v[5], v[7], v[9], v[11], v[13], v[15]};
    Dft<8, INV>::run(e);
    Dft<8, INV>::run(o);
    // W16^k = exp(-+ 2 pi i k / 16), k = 1 .. 7 (upper sign: forward)
    const float h = 0.70710678118654752f, c1 = 0.92387953251128674f, s1 = 0.38268343236508977f;
    const float sg = INV ? 1.f : -1.f;
    o[1] = cmul(o[1], make_float2(c1, sg * s1));
    o[2] = cmul(o[2], make_float2(h, sg * h));
    o[3] = cmul(o[3], make_float2(s1, sg * c1));
    o[4] = rot90<INV>(o[4]);
    o[5] = cmul(o[5], make_float2(-s1, sg * c1));
    o[6] = cmul(o[6], make_float2(-h, sg * h));
    o[7] = cmul(o[7], make_float2(-c1, sg * s1));
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      v[k] = cadd(e[k], o[k]);
      v[k + 8] = csub(e[k], o[k]);
    }
  }
};

// One radix-R pass over `npen` pencils of length N.  Element n of pencil p is s[pen(p) * sp + n * sn];
// consecutive threads take consecutive pencils (conflict-free for sp = 1, and for sp = pitch = My + 1).
// Forward (decimation in frequency): the block of length L splits into R sub-blocks of length L / R,
//   out[j + r L/R] = W_L^{j r} sum_m in[j + m L/R] W_R^{m r};  the inverse pass is its exact adjoint.
template <int R, bool INV>
__device__ __forceinline__ void fft_pass(float2* s, int npen, const short* pen, int sp, int sn, int N, int L,
                                         const float2* tw) {
  const int Lr = L / R, per = N / R, tws = N / L;
  for (int it = threadIdx.x; it < npen * per; it += kXYThreads) {
    const int g = it / npen, pi = it - g * npen;
    const int p = pen ? pen[pi] : pi;
    const int b = g / Lr, j = g - b * Lr;
    float2* base = s + p * sp + (b * L + j) * sn;
    const int step = Lr * sn;
    float2 v[R];
#pragma unroll
    for (int m = 0; m < R; ++m) v[m] = base[m * step];
    if (INV) {
#pragma unroll
      for (int r = 1; r < R; ++r) {
        const float2 w = tw[j * r * tws];
        v[r] = cmul(v[r], make_float2(w.x, -w.y));
      }
    }
    Dft<R, INV>::run(v);
    if (!INV) {
#pragma unroll
      for (int r = 1; r < R; ++r) v[r] = cmul(v[r], tw[j * r * tws]);
    }
#pragma unroll
    for (int m = 0; m < R; ++m) base[m * step] = v[m];
  }
}

template <bool INV>
__device__ __forceinline__ void fft_axis(float2* s, int npen, const short* pen, int sp, int sn, int N, int nr,
                                         const int* rad, const float2* tw) {
  // forward: L = N, N/r0, N/(r0 r1), ...; inverse: the same passes in reverse order
  int Ls[4];
  int L = N;
  for (int i = 0; i < nr; ++i) { Ls[i] = L; L /= rad[i]; }
  for (int ii = 0; ii < nr; ++ii) {
    const int i = INV ? nr - 1 - ii : ii;
    switch (rad[i]) {
      case 8: fft_pass<8, INV>(s, npen, pen, sp, sn, N, Ls[i], tw); break;
      case 4: fft_pass<4, INV>(s, npen, pen, sp, sn, N, Ls[i], tw); break;
      default: fft_pass<2, INV>(s, npen, pen, sp, sn, N, Ls[i], tw); break;
    }
    __syncthreads();
  }
}

// position -> DFT index after the forward passes (mixed-radix digit reversal)
__device__ __forceinline__ int freq_of_pos(int pos, int N, int nr, const int* rad) {
  int k = 0, mul = 1, L = N;
  for (int i = 0; i < nr; ++i) {
    L /= rad[i];
    const int d = pos / L;
    pos -= d * L;
    k += d * mul;
    mul *= rad[i];
  }
  return k;
}

// grid = (kept k_z planes, channels).  spec_in / spec_out: plane-major [kz][c][x][y] complex.
// DUMP: also write the scaled modes in the dense layout [c][kx][ky][kz] (test hook).
// Virial of one mode, as in k_scale: W_ab += e delta_ab + herm |rho^|^2 (dD/dk / |k|) k_a k_b
// with e = herm D |rho^|^2 (the factor 1/2 is applied with the final reduction).
__device__ __forceinline__ void virial_of_mode(double (&w)[6], double e, double g, float kx, float ky, float kz,
                                               bool zero_mode) {
  w[0] += e; w[1] += e; w[2] += e;
  if (!zero_mode) {
    w[0] += g * kx * kx; w[1] += g * ky * ky; w[2] += g * kz * kz;
    w[3] += g * kx * ky; w[4] += g * kx * kz; w[5] += g * ky * kz;
  }
}
// The CTA that finishes last adds the channel energies up (E = sum_c E_c): no separate one-warp kernel between
// the multiply and the inverse z transform.  `done` counts finished CTAs; it is zeroed with the evaluation's
// other accumulators.  Called by thread 0 after its atomicAdd into Ech.
__device__ __forceinline__ void finish_energy(double* Ech, int C, double* E_out, unsigned int* done) {
  if (E_out == nullptr) return;
  __threadfence();
  const unsigned int t = atomicAdd(done, 1u);
  if (t == gridDim.x * gridDim.y - 1u) {
    __threadfence();
    double e = 0.0;
    for (int c = 0; c < C; ++c) e += atomicAdd(&Ech[c], 0.0);   // (read at L2, where the other CTAs' atomics landed)
    *E_out = e;
  }
}

// block sums of the six components -> Wacc (one atomicAdd per component and CTA); s_red: one double per warp
__device__ __forceinline__ void virial_reduce(const double (&w)[6], double* s_red, double* Wacc) {
  const int tid = threadIdx.x;
#pragma unroll 1
  for (int i = 0; i < 6; ++i) {
    __syncthreads();
    const double t = warp_sum(w[i]);
    if ((tid & 31) == 0) s_red[tid >> 5] = t;
    __syncthreads();
    if (tid < 32) {
      double u = tid < (int)(blockDim.x >> 5) ? s_red[tid] : 0.0;
      u = warp_sum(u);
      if (tid == 0 && u != 0.0) atomicAdd(&Wacc[i], 0.5 * u);
    }
  }
}

template <bool DUMP, bool VIR>
__global__ void __launch_bounds__(kXYThreads, 1)
    k_xy_scale(const XYParams X, const ScaleParams<float> P, const float2* __restrict__ spec_in,
               float2* __restrict__ spec_out, double* __restrict__ Ech, float2* __restrict__ dump,
               double* __restrict__ Wacc, double* __restrict__ E_out, unsigned int* __restrict__ done) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* s = reinterpret_cast<float2*>(smem_raw);                 // [Mx][pitch]
  float2* twx = s + (size_t)X.Mx * X.pitch;                        // [Mx]  exp(-2 pi i k / Mx)
  float2* twy = twx + X.Mx;                                        // [My]
  short* fx_of = reinterpret_cast<short*>(twy + X.My);             // [Mx]  position -> DFT index
  short* fy_of = fx_of + X.Mx;                                     // [My]
  short* keptx = fy_of + X.My;                                     // [Mx]  kept x positions (first nkx)
  __shared__ int s_nkx;
  __shared__ double s_red[kXYThreads / 32];
  const int kz = blockIdx.x, c = blockIdx.y;
  const int Mx = X.Mx, My = X.My, pitch = X.pitch;
  const int tid = threadIdx.x;

  // tables
  for (int i = tid; i < Mx; i += kXYThreads) {
    float sn, cs;
    sincospif(-2.f * (float)i / (float)Mx, &sn, &cs);
    twx[i] = make_float2(cs, sn);
    fx_of[i] = (short)freq_of_pos(i, Mx, X.nrx, X.rx);
  }
  for (int i = tid; i < My; i += kXYThreads) {
    float sn, cs;
    sincospif(-2.f * (float)i / (float)My, &sn, &cs);
    twy[i] = make_float2(cs, sn);
    fy_of[i] = (short)freq_of_pos(i, My, X.nry, X.ry);
  }
  // the plane
  const size_t plane = ((size_t)kz * X.C + c) * Mx * My;
  {
    const float2* src = spec_in + plane;
    for (int i = tid; i < Mx * My; i += kXYThreads) {
      const int x = i / My, y = i - x * My;
      s[x * pitch + y] = __ldg(src + i);
    }
  }
  __syncthreads();
  if (tid == 0) {   // kept x positions, in position order
    int n = 0;
    for (int i = 0; i < Mx; ++i) {
      const int f = fx_of[i] <= Mx / 2 ? fx_of[i] : fx_of[i] - Mx;
      if (abs(f) <= X.kmaxx) keptx[n++] = (short)i;
    }
    s_nkx = n;
  }
  // forward: along x for every y, then along y for the kept k_x only
  fft_axis<false>(s, My, nullptr, 1, pitch, Mx, X.nrx, X.rx, twx);   // (ends with a barrier: s_nkx visible)
  const int nkx = s_nkx;
  fft_axis<false>(s, nkx, keptx, pitch, 1, My, X.nry, X.ry, twy);

  // scale by D_p(m) = (h^3 / Mtot) Phi^_p(|k|) / W^(k)^2 inside the ball, zero elsewhere; E_c
  const int slot = P.chan_slot[c];
  const float fzf = (float)kz;
  const float wz = P.invW2[2][kz];
  const float herm = kz == 0 ? 1.f : 2.f;
  double e = 0.0;
  double wloc[6] = {0, 0, 0, 0, 0, 0};
  for (int it = tid; it < nkx * My; it += kXYThreads) {
    const int a = it / My, py = it - a * My;
    const int px = keptx[a];
    const int ix = fx_of[px], iy = fy_of[py];
    const int fx = ix <= Mx / 2 ? ix : ix - Mx, fy = iy <= My / 2 ? iy : iy - My;
    float2 v = make_float2(0.f, 0.f);
    if (abs(fy) <= X.kmaxy) {
      const float kx = P.recip[0] * (float)fx + P.recip[3] * (float)fy + P.recip[6] * fzf;
      const float ky = P.recip[1] * (float)fx + P.recip[4] * (float)fy + P.recip[7] * fzf;
      const float kzv = P.recip[2] * (float)fx + P.recip[5] * (float)fy + P.recip[8] * fzf;
      const float kn = sqrtf(kx * kx + ky * ky + kzv * kzv);
      const float x = kn * P.x_per_k;
      const bool zero_mode = (ix | iy | kz) == 0;
      if (zero_mode || x < 1.f) {
        float d;
        const float wgt = P.base * P.invW2[0][ix] * P.invW2[1][iy] * wz;
        if (zero_mode) d = P.chan_D0[c];
        else d = wgt * kernel_value(P, slot, x, x * P.c);
        v = s[px * pitch + py];
        const float a2 = herm * (v.x * v.x + v.y * v.y);
        e += (double)(a2 * d);
        if (VIR) {
          const double g = zero_mode ? 0.0 : (double)(a2 * (wgt * kernel_dvalue(P, slot, x, x * P.c) / kn));
          virial_of_mode(wloc, (double)(a2 * d), g, kx, ky, kzv, zero_mode);
        }
        v.x *= d;
        v.y *= d;
        if (DUMP) dump[(((size_t)c * Mx + ix) * My + iy) * X.Mzh + kz] = v;
      }
    }
    s[px * pitch + py] = v;
  }
  // rows of the dropped k_x hold forward-pass leftovers: clear them for the inverse x passes
  for (int it = tid; it < Mx * My; it += kXYThreads) {
    const int px = it / My, py = it - px * My;
    const int f = fx_of[px] <= Mx / 2 ? fx_of[px] : fx_of[px] - Mx;
    if (abs(f) > X.kmaxx) s[px * pitch + py] = make_float2(0.f, 0.f);
  }
  __syncthreads();
  // inverse: along y for the kept k_x, then along x for every y
  fft_axis<true>(s, nkx, keptx, pitch, 1, My, X.nry, X.ry, twy);
  fft_axis<true>(s, My, nullptr, 1, pitch, Mx, X.nrx, X.rx, twx);
  {
    float2* dst = spec_out + plane;
    for (int i = tid; i < Mx * My; i += kXYThreads) {
      const int x = i / My, y = i - x * My;
      dst[i] = s[x * pitch + y];
    }
  }
  // E_c += 1/2 sum_m herm D |rho^|^2 over this plane (double)
  e = warp_sum(e);
  if ((tid & 31) == 0) s_red[tid >> 5] = e;
  __syncthreads();
  if (tid < 32) {
    double t = tid < kXYThreads / 32 ? s_red[tid] : 0.0;
    t = warp_sum(t);
    if (tid == 0) {
      if (t != 0.0) atomicAdd(&Ech[c], 0.5 * t);
      finish_energy(Ech, X.C, E_out, done);
    }
  }
  if (VIR) virial_reduce(wloc, s_red, Wacc);
}

// ------------------------------------------------------------------------------------------------
// Compile-time variants for the common sizes: radices, strides and pass lengths are constants, the
// pencil index comes from shifts (pencil counts are padded to a power of two), the last pass of an
// axis (L == R: all twiddles are 1) multiplies nothing.  34 M -> ~9 M warp instructions per launch at
// 128 x 128 (profiles/r2b, r2c).
// ------------------------------------------------------------------------------------------------
template <int N> struct Rad;
template <> struct Rad<8>   { static constexpr int n = 1, r0 = 8, r1 = 1, r2 = 1; };
template <> struct Rad<16>  { static constexpr int n = 2, r0 = 4, r1 = 4, r2 = 1; };
template <> struct Rad<32>  { static constexpr int n = 2, r0 = 8, r1 = 4, r2 = 1; };
template <> struct Rad<64>  { static constexpr int n = 2, r0 = 8, r1 = 8, r2 = 1; };
template <> struct Rad<128> { static constexpr int n = 2, r0 = 16, r1 = 8, r2 = 1; };   // two shared-memory passes instead of three (8, 4, 4)
template <> struct Rad<256> { static constexpr int n = 2, r0 = 16, r1 = 16, r2 = 1; };

__host__ __device__ constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }

template <int NT, int N, int R, int L, bool INV, int SP, int SN>
__device__ __forceinline__ void fft_pass_t(float2* s, const int npen, const int lgpad, const short* pen,
                                           const float2* tw) {
  constexpr int Lr = L / R, per = N / R, tws = N / L, step = Lr * SN;
  const int padmask = (1 << lgpad) - 1;
  for (int it = threadIdx.x; it < (per << lgpad); it += NT) {
    const int pi = it & padmask, g = it >> lgpad;
    if (pi >= npen) continue;
    const int p = pen ? pen[pi] : pi;
    const int b = g / Lr, j = g % Lr;     // compile-time powers of two
    float2* base = s + p * SP + (b * L + j) * SN;
    float2 v[R];
#pragma unroll
    for (int m = 0; m < R; ++m) v[m] = base[m * step];
    if (INV && L > R) {
#pragma unroll
      for (int r = 1; r < R; ++r) {
        const float2 w = tw[j * (r * tws)];
        v[r] = cmul(v[r], make_float2(w.x, -w.y));
      }
    }
    Dft<R, INV>::run(v);
    if (!INV && L > R) {
#pragma unroll
      for (int r = 1; r < R; ++r) v[r] = cmul(v[r], tw[j * (r * tws)]);
    }
#pragma unroll
    for (int m = 0; m < R; ++m) base[m * step] = v[m];
  }
}

template <int NT, int N, bool INV, int SP, int SN>
__device__ __forceinline__ void fft_axis_t(float2* s, const int npen, const int lgpad, const short* pen,
                                           const float2* tw) {
  using Rd = Rad<N>;
  constexpr int L0 = N, L1 = N / Rd::r0, L2 = L1 / Rd::r1;
  if (!INV) {
    fft_pass_t<NT, N, Rd::r0, L0, INV, SP, SN>(s, npen, lgpad, pen, tw);
    __syncthreads();
    if constexpr (Rd::n >= 2) { fft_pass_t<NT, N, Rd::r1, L1, INV, SP, SN>(s, npen, lgpad, pen, tw); __syncthreads(); }
    if constexpr (Rd::n >= 3) { fft_pass_t<NT, N, Rd::r2, L2, INV, SP, SN>(s, npen, lgpad, pen, tw); __syncthreads(); }
  } else {
    if constexpr (Rd::n >= 3) { fft_pass_t<NT, N, Rd::r2, L2, INV, SP, SN>(s, npen, lgpad, pen, tw); __syncthreads(); }
    if constexpr (Rd::n >= 2) { fft_pass_t<NT, N, Rd::r1, L1, INV, SP, SN>(s, npen, lgpad, pen, tw); __syncthreads(); }
    fft_pass_t<NT, N, Rd::r0, L0, INV, SP, SN>(s, npen, lgpad, pen, tw);
    __syncthreads();
  }
}

template <int N>
__device__ __forceinline__ int freq_of_pos_t(int pos) {
  using Rd = Rad<N>;
  constexpr int L1 = N / Rd::r0, L2 = L1 / Rd::r1;
  const int d0 = pos / L1, r = pos % L1;
  int k = d0;
  if constexpr (Rd::n >= 2) {
    const int d1 = r / L2, r2 = r % L2;
    k += d1 * Rd::r0;
    if constexpr (Rd::n >= 3) k += r2 * (Rd::r0 * Rd::r1);
  }
  return k;
}

// Same kernel as k_xy_scale with Mx = My = M fixed at compile time.
template <int M, bool DUMP, bool VIR>
__global__ void __launch_bounds__(kXYThreads, 1)
    k_xy_scale_t(const XYParams X, const ScaleParams<float> P, const float2* __restrict__ spec_in,
                 float2* __restrict__ spec_out, double* __restrict__ Ech, float2* __restrict__ dump,
                 double* __restrict__ Wacc, double* __restrict__ E_out, unsigned int* __restrict__ done) {
  constexpr int pitch = M + 1, NT = kXYThreads, LG = ilog2(M);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* s = reinterpret_cast<float2*>(smem_raw);                 // [M][pitch]
  float2* tw = s + (size_t)M * pitch;                              // [M]  exp(-2 pi i k / M)
  short* f_of = reinterpret_cast<short*>(tw + M);                  // [M]  position -> DFT index
  short* keptx = f_of + M;                                         // [M]  kept x positions (first nkx)
  __shared__ int s_nkx;
  __shared__ double s_red[NT / 32];
  const int kz = blockIdx.x, c = blockIdx.y;
  const int tid = threadIdx.x;
  if (tid < 32) {   // kept x positions, in position order (one warp: ballot + prefix popcount)
    int n = 0;
    for (int i0 = 0; i0 < M; i0 += 32) {
      const int i = i0 + tid;
      const int k = freq_of_pos_t<M>(i);
      const int f = k <= M / 2 ? k : k - M;
      const bool keep = i < M && abs(f) <= X.kmaxx;
      const unsigned m = __ballot_sync(0xffffffffu, keep);
      if (keep) keptx[n + __popc(m & ((1u << tid) - 1u))] = (short)i;
      n += __popc(m);
    }
    if (tid == 0) s_nkx = n;
  }
  for (int i = tid; i < M; i += NT) {
    float sn, cs;
    sincospif(-2.f * (float)i / (float)M, &sn, &cs);
    tw[i] = make_float2(cs, sn);
    f_of[i] = (short)freq_of_pos_t<M>(i);
  }
  const size_t plane = ((size_t)kz * X.C + c) * M * M;
  {
    const float4* src = reinterpret_cast<const float4*>(spec_in + plane);   // two complex per load
    // all of a thread's loads in flight before the first store (the plane comes from L2 / HBM: one round trip
    // instead of one per element pair)
    constexpr int kPer = (M * M / 2 + NT - 1) / NT, kBatch = kPer < 8 ? kPer : 8;
    for (int i0 = tid; i0 < M * M / 2; i0 += NT * kBatch) {
      float4 t[kBatch];
#pragma unroll
      for (int u = 0; u < kBatch; ++u) {
        const int i = i0 + u * NT;
        t[u] = i < M * M / 2 ? __ldg(src + i) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int u = 0; u < kBatch; ++u) {
        const int i = i0 + u * NT;
        if (i < M * M / 2) {
          const int x = i >> (LG - 1), y = (i & (M / 2 - 1)) * 2;
          s[x * pitch + y] = make_float2(t[u].x, t[u].y);
          s[x * pitch + y + 1] = make_float2(t[u].z, t[u].w);
        }
      }
    }
  }
  __syncthreads();
  const int nkx = s_nkx;
  int lgk = 0;
  while ((1 << lgk) < nkx) ++lgk;
  // forward: along x for every y, then along y for the kept k_x only
  fft_axis_t<NT, M, false, 1, pitch>(s, M, LG, nullptr, tw);
  fft_axis_t<NT, M, false, pitch, 1>(s, nkx, lgk, keptx, tw);

  const int slot = P.chan_slot[c];
  const float fzf = (float)kz;
  const float wz = P.invW2[2][kz];
  const float herm = kz == 0 ? 1.f : 2.f;
  double e = 0.0;
  double wloc[6] = {0, 0, 0, 0, 0, 0};
  for (int it = tid; it < (nkx << LG); it += NT) {
    const int a = it >> LG, py = it & (M - 1);
    const int px = keptx[a];
    const int ix = f_of[px], iy = f_of[py];
    const int fx = ix <= M / 2 ? ix : ix - M, fy = iy <= M / 2 ? iy : iy - M;
    float2 v = make_float2(0.f, 0.f);
    if (abs(fy) <= X.kmaxy) {
      const float kx = P.recip[0] * (float)fx + P.recip[3] * (float)fy + P.recip[6] * fzf;
      const float ky = P.recip[1] * (float)fx + P.recip[4] * (float)fy + P.recip[7] * fzf;
      const float kzv = P.recip[2] * (float)fx + P.recip[5] * (float)fy + P.recip[8] * fzf;
      const float kn = sqrtf(kx * kx + ky * ky + kzv * kzv);
      const float x = kn * P.x_per_k;
      const bool zero_mode = (ix | iy | kz) == 0;
      if (zero_mode || x < 1.f) {
        float d;
        const float wgt = P.base * P.invW2[0][ix] * P.invW2[1][iy] * wz;
        if (zero_mode) d = P.chan_D0[c];
        else d = wgt * kernel_value(P, slot, x, x * P.c);
        v = s[px * pitch + py];
        const float a2 = herm * (v.x * v.x + v.y * v.y);
        e += (double)(a2 * d);
        if (VIR) {
          const double g = zero_mode ? 0.0 : (double)(a2 * (wgt * kernel_dvalue(P, slot, x, x * P.c) / kn));
          virial_of_mode(wloc, (double)(a2 * d), g, kx, ky, kzv, zero_mode);
        }
        v.x *= d;
        v.y *= d;
        if (DUMP) dump[(((size_t)c * M + ix) * M + iy) * X.Mzh + kz] = v;
      }
    }
    s[px * pitch + py] = v;
  }
  for (int it = tid; it < M * M; it += NT) {
    const int px = it >> LG, py = it & (M - 1);
    const int k = f_of[px];
    const int f = k <= M / 2 ? k : k - M;
    if (abs(f) > X.kmaxx) s[px * pitch + py] = make_float2(0.f, 0.f);
  }
  __syncthreads();
  fft_axis_t<NT, M, true, pitch, 1>(s, nkx, lgk, keptx, tw);
  fft_axis_t<NT, M, true, 1, pitch>(s, M, LG, nullptr, tw);
  {
    float4* dst = reinterpret_cast<float4*>(spec_out + plane);
    for (int i = tid; i < M * M / 2; i += NT) {
      const int x = i >> (LG - 1), y = (i & (M / 2 - 1)) * 2;
      const float2 a = s[x * pitch + y], b = s[x * pitch + y + 1];
      dst[i] = make_float4(a.x, a.y, b.x, b.y);
    }
  }
  e = warp_sum(e);
  if ((tid & 31) == 0) s_red[tid >> 5] = e;
  __syncthreads();
  if (tid < 32) {
    double t = tid < NT / 32 ? s_red[tid] : 0.0;
    t = warp_sum(t);
    if (tid == 0) {
      if (t != 0.0) atomicAdd(&Ech[c], 0.5 * t);
      finish_energy(Ech, X.C, E_out, done);
    }
  }
  if (VIR) virial_reduce(wloc, s_red, Wacc);
}

// ------------------------------------------------------------------------------------------------
// z transforms for power-of-two Mz, band-limited on the complex side: forward R2C keeps k_z <= kmaxz
// only (half the cuFFT output is never written), inverse C2R reads only those planes.  A CTA takes the
// YT pencils (c, x, y0 .. y0+YT-1); two real pencils ride in one complex transform,
//   z[n] = a[n] + i b[n]  <->  A[k] = (Z[k] + conj Z[N-k]) / 2,  B[k] = (Z[k] - conj Z[N-k]) / (2i),
// so the plane-major spectrum [kz][c][x][y] is written / read as runs of YT consecutive y.
// ------------------------------------------------------------------------------------------------
constexpr int kZThreads = 256;
constexpr int kZTile = 32;   // real pencils per CTA

// real pencils per CTA of the forward transform: 64 (32 complex pencils: the radix-16 pass then has one butterfly
// per thread) while the tile fits 48 KB of static shared memory
__host__ __device__ constexpr int z_tile_fwd(int NZ) { return NZ > 128 ? 32 : 64; }

template <int NZ>
__global__ void __launch_bounds__(kZThreads)
    k_z_forward(int C, int Mx, int My, int YT, int kmaxz, const float* __restrict__ grid, float2* __restrict__ spec) {
  constexpr int pitch = NZ + 1, NT = kZThreads;
  __shared__ __align__(16) float2 s[(z_tile_fwd(NZ) / 2) * pitch];
  __shared__ float2 tw[NZ];
  __shared__ short pos_of[NZ];
  const int tid = threadIdx.x;
  const int ytiles = My / YT;
  int b = blockIdx.x;
  const int yt = b % ytiles; b /= ytiles;
  const int x = b % Mx;
  const int c = b / Mx;
  const int y0 = yt * YT, npen = YT / 2;
  int lgp = 0;
  while ((1 << lgp) < npen) ++lgp;
  for (int i = tid; i < NZ; i += NT) {
    float sn, cs;
    sincospif(-2.f * (float)i / (float)NZ, &sn, &cs);
    tw[i] = make_float2(cs, sn);
    pos_of[freq_of_pos_t<NZ>(i)] = (short)i;
  }
  {
    const float* src = grid + (((size_t)c * Mx + x) * My + y0) * NZ;   // YT contiguous pencils
    // pencils 2q (real part) and 2q+1 (imaginary part), four z at a time: two 16-byte loads, four complex stores
    for (int i = tid; i < npen * (NZ / 4); i += NT) {
      const int q = i / (NZ / 4), n = (i % (NZ / 4)) * 4;
      const float4 a = __ldg(reinterpret_cast<const float4*>(src + (size_t)(2 * q) * NZ + n));
      const float4 b = __ldg(reinterpret_cast<const float4*>(src + (size_t)(2 * q + 1) * NZ + n));
      float2* d = s + q * pitch + n;
      d[0] = make_float2(a.x, b.x);
      d[1] = make_float2(a.y, b.y);
      d[2] = make_float2(a.z, b.z);
      d[3] = make_float2(a.w, b.w);
    }
  }
  __syncthreads();
  fft_axis_t<NT, NZ, false, pitch, 1>(s, npen, lgp, nullptr, tw);
  const size_t pl = (size_t)C * Mx * My;
  float2* dst = spec + ((size_t)c * Mx + x) * My + y0;
  for (int i = tid; i < (kmaxz + 1) * npen; i += NT) {
    const int k = i / npen, q = i - k * npen;
    const float2 zk = s[q * pitch + pos_of[k]];
    const float2 zm = s[q * pitch + pos_of[(NZ - k) & (NZ - 1)]];
    const float4 o = make_float4(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y), 0.5f * (zk.y + zm.y),
                                 -0.5f * (zk.x - zm.x));
    *reinterpret_cast<float4*>(dst + (size_t)k * pl + 2 * q) = o;
  }
}

// INTERLEAVE = false: real grid [C][Mx][My][Mz].
template <int NZ>
__global__ void __launch_bounds__(kZThreads)
    k_z_inverse(int C, int Mx, int My, int YT, int kmaxz, const float2* __restrict__ spec, float* __restrict__ grid) {
  constexpr int pitch = NZ + 1, NT = kZThreads;
  __shared__ __align__(16) float2 s[(kZTile / 2) * pitch];
  __shared__ float2 tw[NZ];
  __shared__ short pos_of[NZ];
  const int tid = threadIdx.x;
  const int ytiles = My / YT;
  int b = blockIdx.x;
  const int yt = b % ytiles; b /= ytiles;
  const int x = b % Mx;
  const int c = b / Mx;
  const int y0 = yt * YT, npen = YT / 2;
  int lgp = 0;
  while ((1 << lgp) < npen) ++lgp;
  for (int i = tid; i < NZ; i += NT) {
    float sn, cs;
    sincospif(-2.f * (float)i / (float)NZ, &sn, &cs);
    tw[i] = make_float2(cs, sn);
    pos_of[freq_of_pos_t<NZ>(i)] = (short)i;
  }
  for (int i = tid; i < npen * pitch; i += NT) s[i] = make_float2(0.f, 0.f);
  __syncthreads();
  const size_t pl = (size_t)C * Mx * My;
  const float2* src = spec + ((size_t)c * Mx + x) * My + y0;
  for (int i = tid; i < (kmaxz + 1) * npen; i += NT) {
    const int k = i / npen, q = i - k * npen;
    const float4 ab = __ldg(reinterpret_cast<const float4*>(src + (size_t)k * pl + 2 * q));   // A[k], B[k]
    s[q * pitch + pos_of[k]] = make_float2(ab.x - ab.w, ab.y + ab.z);                         // A + i B
    if (k > 0) s[q * pitch + pos_of[NZ - k]] = make_float2(ab.x + ab.w, ab.z - ab.y);         // conj A + i conj B
  }
  __syncthreads();
  fft_axis_t<NT, NZ, true, pitch, 1>(s, npen, lgp, nullptr, tw);
  float* dstg = grid + (((size_t)c * Mx + x) * My + y0) * NZ;
  for (int i = tid; i < YT * NZ; i += NT) {
    const int y = i / NZ, n = i % NZ;
    const float* d = reinterpret_cast<const float*>(s + (y >> 1) * pitch + n);
    dstg[i] = d[y & 1];
  }
}

// Inverse z transform that writes the potential grid directly in the layout the fast gather reads,
// transposed and channel-interleaved [z][x][y][CBV] (kernels_gather.cu), for the channels cb0 ..
// cb0+nch-1: the separate transposing copy (k_interleave_t, 12 us at config 4) and the planar real
// grid it read are gone.  A CTA takes (x, YT = 16 pencils in y) for all channels of the group.
__host__ __device__ constexpr int z_tile_il(int NZ) { return NZ > 128 ? 8 : 16; }   // static shared memory <= 48 KB

template <int CBV> struct ZVec;
template <> struct ZVec<1> { using type = float; };
template <> struct ZVec<2> { using type = float2; };
template <> struct ZVec<4> { using type = float4; };

template <int NZ, int CBV>
__global__ void __launch_bounds__(kZThreads)
    k_z_inverse_il(int C, int cb0, int nch, int Mx, int My, int YT, int kmaxz, const float2* __restrict__ spec,
                   typename ZVec<CBV>::type* __restrict__ out) {
  constexpr int pitch = NZ + 1, NT = kZThreads;
  __shared__ __align__(16) float2 s[CBV * (z_tile_il(NZ) / 2) * pitch];
  __shared__ float2 tw[NZ];
  __shared__ short pos_of[NZ];
  const int tid = threadIdx.x;
  const int ytiles = My / YT;
  const int yt = blockIdx.x % ytiles, x = blockIdx.x / ytiles;
  const int y0 = yt * YT, npc = YT / 2, npen = CBV * npc;   // pencil index = ch * npc + q
  int lgp = 0;
  while ((1 << lgp) < npen) ++lgp;
  for (int i = tid; i < NZ; i += NT) {
    float sn, cs;
    sincospif(-2.f * (float)i / (float)NZ, &sn, &cs);
    tw[i] = make_float2(cs, sn);
    pos_of[freq_of_pos_t<NZ>(i)] = (short)i;
  }
  for (int i = tid; i < npen * pitch; i += NT) s[i] = make_float2(0.f, 0.f);
  __syncthreads();
  const size_t pl = (size_t)C * Mx * My;
  for (int i = tid; i < (kmaxz + 1) * nch * npc; i += NT) {
    const int q = i % npc, r = i / npc, ch = r % nch, k = r / nch;
    const float2* src = spec + (size_t)k * pl + ((size_t)(cb0 + ch) * Mx + x) * My + y0 + 2 * q;
    const float4 ab = __ldg(reinterpret_cast<const float4*>(src));                              // A[k], B[k]
    float2* sp = s + (ch * npc + q) * pitch;
    sp[pos_of[k]] = make_float2(ab.x - ab.w, ab.y + ab.z);                                      // A + i B
    if (k > 0) sp[pos_of[NZ - k]] = make_float2(ab.x + ab.w, ab.z - ab.y);                      // conj A + i conj B
  }
  __syncthreads();
  fft_axis_t<NT, NZ, true, pitch, 1>(s, npen, lgp, nullptr, tw);
  // out[z][x][y][CBV]: for every z a run of YT * CBV floats
  using V = typename ZVec<CBV>::type;
  for (int i = tid; i < NZ * YT; i += NT) {
    const int y = i % YT, z = i / YT;
    float v[CBV];
#pragma unroll
    for (int ch = 0; ch < CBV; ++ch)
      v[ch] = reinterpret_cast<const float*>(s + (ch * npc + (y >> 1)) * pitch + z)[y & 1];
    V o;
    if constexpr (CBV == 1) o = v[0];
    else if constexpr (CBV == 2) o = make_float2(v[0], v[1]);
    else o = make_float4(v[0], v[1], v[2], v[3]);
    out[((size_t)z * Mx + x) * My + y0 + y] = o;
  }
}

int factor_radices(int N, int* rad) {
  int n = 0;
  while (N >= 8 && N != 16) { rad[n++] = 8; N /= 8; }   // 16 = 4 x 4
  while (N >= 4) { rad[n++] = 4; N /= 4; }
  if (N == 2) rad[n++] = 2;
  return n;
}

size_t xy_smem_bytes(int Mx, int My) {
  return sizeof(float2) * ((size_t)Mx * (My + 1) + Mx + My) + sizeof(short) * (2 * (size_t)Mx + My) + 16;
}

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

}  // namespace

bool fused_fft_supported(const pswf_lr_plan* p) {
  if (p->precision != PSWF_LR_F32) return false;
  const int Mx = p->M[0], My = p->M[1];
  if (!is_pow2(Mx) || !is_pow2(My) || Mx < 8 || My < 8 || Mx > 256 || My > 256) return false;
  return xy_smem_bytes(Mx, My) <= 227 * 1024;
}

void fused_fft_limits(const pswf_lr_plan* p, int kmax[3]) {
  const double kc = p->c / p->r_c;
  for (int d = 0; d < 3; ++d) {
    int f = (int)std::floor(kc * p->L[d] / (2 * kPi) + 1e-9);
    kmax[d] = std::max(0, std::min(f, (p->M[d] - 1) / 2));   // never the Nyquist index
  }
}

// forward z transform (cuFFT, plane-major output) must already be in p->d_spec; writes p->d_spec2
void launch_xy_scale(pswf_lr_plan* p, const ScaleParams<float>& P, double* E, cudaStream_t st) {
  XYParams X;
  X.Mx = p->M[0]; X.My = p->M[1]; X.pitch = p->M[1] + 1; X.C = p->C;
  X.nrx = factor_radices(X.Mx, X.rx);
  X.nry = factor_radices(X.My, X.ry);
  X.kmaxx = p->fused_kmax[0]; X.kmaxy = p->fused_kmax[1];
  X.Mzh = p->M[2] / 2 + 1;
  const size_t sm = xy_smem_bytes(X.Mx, X.My);
  const dim3 grid((unsigned)(p->fused_kmax[2] + 1), (unsigned)p->C);
  p->n_kernels += 1;
  double* wacc = p->virial ? p->d_virial : nullptr;   // zeroed by the caller before the launch
  float2* dump = nullptr;
  if (p->debug_dump_spectrum) {
    const size_t Mhalf = (size_t)p->M[0] * p->M[1] * X.Mzh;
    cudaMemsetAsync(p->d_spec_dump, 0, sizeof(float2) * Mhalf * p->C, st);
    dump = (float2*)p->d_spec_dump;
  }
#define PSWF_XY(KERN)                                                                                        \
  do {                                                                                                       \
    cudaFuncSetAttribute(KERN, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);                        \
    KERN<<<grid, kXYThreads, sm, st>>>(X, P, (const float2*)p->d_spec, (float2*)p->d_spec2, p->d_Ech, dump, \
                                       wacc, E, p->d_done);                                                  \
  } while (0)
#define PSWF_XY_SQ(MV)                                                  \
  case MV:                                                              \
    if (wacc) {  /* virial: accumulated in the same pass */             \
      if (dump) PSWF_XY((k_xy_scale_t<MV, true, true>));                \
      else PSWF_XY((k_xy_scale_t<MV, false, true>));                    \
    } else if (dump) PSWF_XY((k_xy_scale_t<MV, true, false>));          \
    else PSWF_XY((k_xy_scale_t<MV, false, false>));                     \
    return;
  if (X.Mx == X.My) {
    switch (X.Mx) {
      PSWF_XY_SQ(16) PSWF_XY_SQ(32) PSWF_XY_SQ(64) PSWF_XY_SQ(128)
      default: break;
    }
  }
  if (wacc) {
    if (dump) PSWF_XY((k_xy_scale<true, true>));
    else PSWF_XY((k_xy_scale<false, true>));
  } else if (dump) PSWF_XY((k_xy_scale<true, false>));
  else PSWF_XY((k_xy_scale<false, false>));
#undef PSWF_XY_SQ
#undef PSWF_XY
}


bool fused_z_supported(const pswf_lr_plan* p) {
  const int Mz = p->M[2];
  return is_pow2(Mz) && Mz >= 8 && Mz <= 256 && (p->M[1] % 2) == 0;
}

namespace {
int z_tile(int My) {
  int yt = std::min(kZTile, My);
  while (My % yt) yt >>= 1;
  return yt;
}
}  // namespace

void launch_z_forward(pswf_lr_plan* p, cudaStream_t st) {
  const int C = p->C, Mx = p->M[0], My = p->M[1];
  int YT = std::min(z_tile_fwd(p->M[2]), My);
  while (My % YT) YT >>= 1;
  const unsigned nb = (unsigned)(C * Mx * (My / YT));
  p->n_kernels += 1;
#define PSWF_ZF(NZ) \
  case NZ: k_z_forward<NZ><<<nb, kZThreads, 0, st>>>(C, Mx, My, YT, p->fused_kmax[2], (const float*)p->d_grid, (float2*)p->d_spec); break;
  switch (p->M[2]) { PSWF_ZF(8) PSWF_ZF(16) PSWF_ZF(32) PSWF_ZF(64) PSWF_ZF(128) PSWF_ZF(256) default: break; }
#undef PSWF_ZF
}

// the fast gather's layout, channel groups of 4 as in launch_fast_gather (last group 1, 2 or 4 wide)
void launch_z_inverse_interleaved(pswf_lr_plan* p, cudaStream_t st) {
  const int C = p->C, Mx = p->M[0], My = p->M[1];
  int YT = std::min(z_tile_il(p->M[2]), My);
  while (My % YT) YT >>= 1;
  const unsigned nb = (unsigned)(Mx * (My / YT));
  const size_t Mtot = (size_t)Mx * My * p->M[2];
  float* gi = (float*)p->d_gridi;
  const int G = p->gather_group;
  for (int cb0 = 0; cb0 < C; cb0 += G) {
    const int left = std::min(G, C - cb0);
    const int cbv = left >= 3 ? 4 : left, nch = left;
    p->n_kernels += 1;
#define PSWF_ZIL(NZ, CBV)                                                                                         \
  k_z_inverse_il<NZ, CBV><<<nb, kZThreads, 0, st>>>(C, cb0, nch, Mx, My, YT, p->fused_kmax[2], (const float2*)p->d_spec2, \
                                                    (typename ZVec<CBV>::type*)gi)
#define PSWF_ZIL_N(NZ)                     \
  case NZ:                                 \
    if (cbv == 4) PSWF_ZIL(NZ, 4);         \
    else if (cbv == 2) PSWF_ZIL(NZ, 2);    \
    else PSWF_ZIL(NZ, 1);                  \
    break;
    switch (p->M[2]) { PSWF_ZIL_N(16) PSWF_ZIL_N(32) PSWF_ZIL_N(64) PSWF_ZIL_N(128) PSWF_ZIL_N(256) default: break; }
#undef PSWF_ZIL_N
#undef PSWF_ZIL
    gi += Mtot * cbv;
  }
}

void launch_z_inverse(pswf_lr_plan* p, cudaStream_t st) {
  const int C = p->C, Mx = p->M[0], My = p->M[1], YT = z_tile(My);
  const unsigned nb = (unsigned)(C * Mx * (My / YT));
  p->n_kernels += 1;
#define PSWF_ZI(NZ) \
  case NZ: k_z_inverse<NZ><<<nb, kZThreads, 0, st>>>(C, Mx, My, YT, p->fused_kmax[2], (const float2*)p->d_spec2, (float*)p->d_grid); break;
  switch (p->M[2]) { PSWF_ZI(8) PSWF_ZI(16) PSWF_ZI(32) PSWF_ZI(64) PSWF_ZI(128) PSWF_ZI(256) default: break; }
#undef PSWF_ZI
}

}  // namespace pswf
