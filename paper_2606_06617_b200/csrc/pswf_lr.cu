// C ABI of libpswf_lr: plan creation (host-side PSWF solve + Horner tables + cuFFT plans),
// execute (bin/sort -> spread -> FFT -> scale+reduce -> inverse FFT -> gather), destroy.
// See include/pswf_lr.h for the contract and the PAPER.md passages behind each step.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <type_traits>

#include "launch.hpp"

using namespace pswf;

#define CUDA_TRY(expr)                                   \
  do {                                                   \
    cudaError_t _e = (expr);                             \
    if (_e != cudaSuccess) return PSWF_LR_ERR_CUDA;      \
  } while (0)
#define CUFFT_TRY(expr)                                  \
  do {                                                   \
    cufftResult _r = (expr);                             \
    if (_r != CUFFT_SUCCESS) return PSWF_LR_ERR_CUFFT;   \
  } while (0)

namespace {

// A plan is bound to the device current at its creation: every entry point that touches the device
// switches to it for the call and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  bool ok = true, switched = false;
  explicit DeviceGuard(const pswf_lr_plan* p) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != p->device) {
      ok = cudaSetDevice(p->device) == cudaSuccess;
      switched = ok;
    }
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

template <class T>
int upload(void** dst, const std::vector<double>& src, long long* bytes) {
  std::vector<T> tmp(src.begin(), src.end());
  size_t nb = sizeof(T) * std::max<size_t>(tmp.size(), 1);
  if (cudaMalloc(dst, nb) != cudaSuccess) return PSWF_LR_ERR_ALLOC;
  if (!tmp.empty() && cudaMemcpy(*dst, tmp.data(), sizeof(T) * tmp.size(), cudaMemcpyHostToDevice) != cudaSuccess)
    return PSWF_LR_ERR_CUDA;
  *bytes += (long long)nb;
  return 0;
}

inline size_t real_size(const pswf_lr_plan* p) { return p->precision == PSWF_LR_F64 ? 8 : 4; }

int dev_alloc(void** ptr, size_t bytes, long long* total) {
  if (cudaMalloc(ptr, std::max<size_t>(bytes, 16)) != cudaSuccess) {
    *ptr = nullptr;
    return PSWF_LR_ERR_ALLOC;
  }
  *total += (long long)bytes;
  return 0;
}

void free_atoms(pswf_lr_plan* p) {
  void** ptrs[] = {&p->d_spos, (void**)&p->d_key, (void**)&p->d_rank, (void**)&p->d_perm, (void**)&p->d_si0, &p->d_sdelta,
                   &p->d_sq,          &p->d_rec,          &p->d_drec,         &p->d_pos_in[0],    &p->d_q_in[0],     &p->d_phi_out[0],
                   &p->d_F_out[0],    &p->d_pos_in[1],    &p->d_q_in[1],      &p->d_phi_out[1],   &p->d_F_out[1],
                   &p->d_pos_in[2],   &p->d_q_in[2],      &p->d_phi_out[2],   &p->d_F_out[2]};
  for (void** q : ptrs) {
    if (*q) cudaFree(*q);
    *q = nullptr;
  }
}

int ensure_capacity(pswf_lr_plan* p, int n) {
  if (n <= p->cap_atoms) return 0;
  // growing: wait for everything in flight, then reallocate (documented in the header)
  if (cudaDeviceSynchronize() != cudaSuccess) return PSWF_LR_ERR_CUDA;
  free_atoms(p);
  p->workspace_bytes -= p->atom_bytes;   // everything per-atom (staging slots included) was just released
  p->atom_bytes = 0;
  int cap = std::max(n, std::max(p->cap_atoms * 2, 1024));
  const size_t rs = real_size(p);
  long long b = 0;
  int rc = 0;
  rc |= dev_alloc((void**)&p->d_key, sizeof(int) * (size_t)cap, &b);
  rc |= dev_alloc((void**)&p->d_rank, sizeof(int) * (size_t)cap, &b);
  rc |= dev_alloc((void**)&p->d_perm, sizeof(int) * (size_t)cap, &b);
  rc |= dev_alloc((void**)&p->d_si0, sizeof(int) * 3 * (size_t)cap, &b);
  rc |= dev_alloc(&p->d_sdelta, rs * 3 * (size_t)cap, &b);
  rc |= dev_alloc(&p->d_sq, rs * (size_t)p->C * cap, &b);
  rc |= dev_alloc(&p->d_spos, rs * 3 * (size_t)cap, &b);
  p->cap_atoms = cap;
  size_t recb = stencil_path_supported(p) ? stencil_record_bytes(p) * (size_t)cap : 0;
  if (recb) rc |= dev_alloc(&p->d_rec, recb, &b);
  if (recb) rc |= dev_alloc(&p->d_drec, stencil_drecord_bytes(p) * (size_t)cap, &b);
  if (rc) {
    free_atoms(p);
    p->cap_atoms = 0;
    return PSWF_LR_ERR_ALLOC;
  }
  p->workspace_bytes += b;
  p->atom_bytes += b;
  return 0;
}

int ensure_host_staging(pswf_lr_plan* p, int slots) {
  const size_t rs = real_size(p);
  long long b = 0;
  int rc = 0;
  for (int s = 0; s < slots; ++s) {
    if (p->d_pos_in[s]) continue;
    rc |= dev_alloc(&p->d_pos_in[s], rs * 3 * (size_t)p->cap_atoms, &b);
    rc |= dev_alloc(&p->d_q_in[s], rs * (size_t)p->C * p->cap_atoms, &b);
    rc |= dev_alloc(&p->d_phi_out[s], rs * (size_t)p->C * p->cap_atoms, &b);
    rc |= dev_alloc(&p->d_F_out[s], rs * 3 * (size_t)p->cap_atoms, &b);
    if (!p->d_E_out[s]) rc |= dev_alloc((void**)&p->d_E_out[s], sizeof(double), &b);
  }
  p->workspace_bytes += b;
  p->atom_bytes += b;
  return rc ? PSWF_LR_ERR_ALLOC : 0;
}

template <class T>
GridGeom<T> make_geom(const pswf_lr_plan* p) {
  GridGeom<T> g;
  for (int d = 0; d < 3; ++d) {
    g.M[d] = p->M[d];
    g.dxi_ds[d] = (T)(-2.0 * p->M[d]);
  }
  for (int i = 0; i < 9; ++i) {
    g.hinv[i] = p->hinv[i];
    g.hinv_t[i] = (T)p->hinv[i];
  }
  g.w = p->w;
  g.wdeg = p->wt.degree;
  g.wcoef = (const T*)p->d_wcoef;
  g.wdcoef = (const T*)p->d_wdcoef;
  return g;
}

bool exponent_supported(int p) { return (p >= 1 && p <= 6) || p == 8 || p == 10; }

double slot_prefactor(int p, double c, double r_c) {
  // Phi^_p = r_c^(3-p) S^_p, constants of Theorem 1 folded in (see host_tables.hpp / k_scale)
  switch (p) {
    case 1: return 4 * kPi * r_c * r_c;
    case 2: return 2 * kPi * kPi * r_c;
    case 3: return 4 * kPi;
    case 4: return kPi * kPi * c / r_c;
    case 5: return 2 * kPi * c * c / (3 * r_c * r_c);
    case 6: return kPi * kPi * c * c * c / (12 * r_c * r_c * r_c);
    case 8: return kPi * kPi * std::pow(c / r_c, 5) / 72;      // SI Section 6, (S56) applied to (S52)
    default: return kPi * kPi * std::pow(c / r_c, 7) / 576;    // p = 10
  }
}

template <class T>
ScaleParams<T> make_scale(const pswf_lr_plan* p) {
  ScaleParams<T> P;
  memset(&P, 0, sizeof(P));
  double mt = 1, ltab = 1;
  for (int d = 0; d < 3; ++d) {
    P.M[d] = p->M[d];
    P.invW2[d] = (const T*)p->d_invW2[d];
    mt *= p->M[d];
    ltab *= p->L[d];
  }
  // reciprocal basis 2 pi h^-T: k_e = sum_d m_d recip[3 d + e], recip[3 d + e] = 2 pi hinv[e][d]
  for (int d = 0; d < 3; ++d)
    for (int e = 0; e < 3; ++e) P.recip[3 * d + e] = (T)(2 * kPi * p->hinv[3 * e + d]);
  // D_p(m) = (V / Mtot^2) Phi^ / W^2 with W^ = prod_d omega_d lambda_0 psi(.), prod_d omega_d = (w/2)^3 V / Mtot.
  // The 1-D tables carry omega_d = w |a_d| / (2 M_d); in a skewed cell prod |a_d| > V, corrected here.
  const double vcorr = (ltab / p->volume) * (ltab / p->volume);
  const double hv = p->volume / mt * vcorr;
  P.Mzh = p->M[2] / 2 + 1;
  P.C = p->C;
  P.nslots = (int)p->distinct_p.size();
  for (int s = 0; s < P.nslots; ++s) {
    P.slot_p[s] = p->distinct_p[s];
    P.slot_pre[s] = (T)slot_prefactor(p->distinct_p[s], p->c, p->r_c);
  }
  for (int a = 0; a < p->C; ++a) {
    P.chan_slot[a] = p->chan_slot[a];
    double d0 = p->zero_mode == 0 ? (hv / mt) * p->Phi0[p->chan_slot[a]] / (p->What0 * p->What0) : 0.0;
    P.chan_D0[a] = (T)d0;
  }
  P.x_per_k = (T)(p->r_c / p->c);
  P.c = (T)p->c;
  P.base = (T)(hv / mt);
  P.panels = p->kt.panels;
  P.degree = p->kt.degree;
  P.kcoef = (const T*)p->d_kcoef;
  return P;
}

template <class T>
int execute_t(pswf_lr_plan* p, int n, const T* pos, const T* q, double* E, T* phi, T* F, cudaStream_t st) {
  constexpr bool kIsF32 = std::is_same<T, float>::value;
  const bool stencil = kIsF32 && (p->kernel_path == 0) && stencil_path_supported(p);
  GridGeom<T> g = make_geom<T>(p);
  ScaleParams<T> P = make_scale<T>(p);
  cudaEvent_t* ev = nullptr;
  if (p->profiling && p->prof_count < kProfileRing)
    ev = p->events.data() + (size_t)p->prof_count * (PSWF_LR_N_STAGES + 1);
  if (ev) cudaEventRecord(ev[0], st);
  // a0
  launch_bin_sort<T>(p, n, pos, q, g, !stencil, true, st);   // (zeroes the energy / virial accumulators too)
  if constexpr (kIsF32) {
    if (stencil) launch_scatter_records(p, n, pos, q, g, st);
  }
  if (ev) cudaEventRecord(ev[1], st);
  // a1
  if constexpr (kIsF32) {
    if (stencil) launch_stencil_spread(p, n, st);
  }
  if (!stencil) launch_spread_ref<T>(p, n, g, st);
  if (ev) cudaEventRecord(ev[2], st);
  // a2-a4.  Band-limited path: R2C along z (plane-major spectrum), then per kept (k_z, channel) plane
  // forward (x,y) transform, multiply + energy, inverse (x,y) transform in one kernel, then C2R along z.
  const bool fused = kIsF32 && p->fused_fft;
  if (fused) {
    if (p->fused_z) {
      launch_z_forward(p, st);
    } else {
      CUFFT_TRY(cufftSetStream(p->fft_zf, st));
      p->n_cufft++;
      CUFFT_TRY(cufftExecR2C(p->fft_zf, (cufftReal*)p->d_grid, (cufftComplex*)p->d_spec));
    }
  } else {
    p->n_cufft++;
    CUFFT_TRY(cufftSetStream(p->fft_fwd, st));
    if (sizeof(T) == 4)
      CUFFT_TRY(cufftExecR2C(p->fft_fwd, (cufftReal*)p->d_grid, (cufftComplex*)p->d_spec));
    else
      CUFFT_TRY(cufftExecD2Z(p->fft_fwd, (cufftDoubleReal*)p->d_grid, (cufftDoubleComplex*)p->d_spec));
  }
  if (ev) cudaEventRecord(ev[3], st);
  // a3
  // (d_Ech and d_virial were zeroed with the sort's buffers at the start of the evaluation)
  if constexpr (kIsF32) {
    if (fused) launch_xy_scale(p, P, E, st);   // (its last CTA writes E)
  }
  if (!fused) {
    launch_scale<T>(p, P, true, st);
    if (E) launch_finalize_energy(p, E, st);
  }
  if (ev) cudaEventRecord(ev[4], st);
  if (phi || F) {
    // a4
    bool il = false;
    if (fused) {
      // own z transform: straight into the gather's interleaved layout when the fast gather follows
      // (the planar grid is then written only on request, for pswf_lr_debug_copy(what = 2))
      il = p->fused_z && stencil && p->M[2] >= 16;
      if (il) launch_z_inverse_interleaved(p, st);
      if (p->fused_z && (!il || p->debug_dump_spectrum)) {
        launch_z_inverse(p, st);
      } else if (!p->fused_z) {
        p->n_cufft++;
        CUFFT_TRY(cufftSetStream(p->fft_zi, st));
        CUFFT_TRY(cufftExecC2R(p->fft_zi, (cufftComplex*)p->d_spec2, (cufftReal*)p->d_grid));
      }
    } else {
      p->n_cufft++;
      CUFFT_TRY(cufftSetStream(p->fft_inv, st));
      if (sizeof(T) == 4)
        CUFFT_TRY(cufftExecC2R(p->fft_inv, (cufftComplex*)p->d_spec, (cufftReal*)p->d_grid));
      else
        CUFFT_TRY(cufftExecZ2D(p->fft_inv, (cufftDoubleComplex*)p->d_spec, (cufftDoubleReal*)p->d_grid));
    }
    if (ev) cudaEventRecord(ev[5], st);
    // a5
    if constexpr (kIsF32) {
      if (stencil) launch_fast_gather(p, n, phi, F, il, st);
    }
    if (!stencil) launch_gather_ref<T>(p, n, g, phi, F, st);
    if (ev) cudaEventRecord(ev[6], st);
  } else if (ev) {
    cudaEventRecord(ev[5], st);
    cudaEventRecord(ev[6], st);
  }
  if (ev) p->prof_count++;
  p->last_n_atoms = n;
  CUDA_TRY(cudaGetLastError());
  return 0;
}

}  // namespace

namespace {
template <class T>
int execute_real_t(pswf_lr_plan* p, int n, const T* pos, const T* q, double* E, T* phi, T* F, int accumulate,
                   cudaStream_t st) {
  GridGeom<T> g = make_geom<T>(p);
  launch_bin_sort<T>(p, n, pos, q, g, true, false, st);   // generic sort: perm, si0, sq
  RealGeom<T> rg;
  RealParams<T> P;
  memset(&P, 0, sizeof(P));
  for (int d = 0; d < 3; ++d) {
    rg.M[d] = p->M[d];
    rg.R[d] = p->real_R[d];
    rg.invL[d] = 1.0 / p->L[d];
    rg.L[d] = (T)p->L[d];
    rg.h[d] = (T)p->real_h[d];
  }
  rg.inv_hz = (T)(1.0 / p->real_h[2]);
  rg.tri = p->triclinic ? 1 : 0;
  for (int i = 0; i < 9; ++i) {
    rg.hinv[i] = p->hinv[i];
    rg.hm[i] = (T)p->cell[i];
  }
  P.C = p->C;
  P.nslots = (int)p->distinct_p.size();
  P.panels = p->rt.panels;
  P.degree = p->rt.degree;
  for (int s = 0; s < P.nslots; ++s) {
    P.slot_p[s] = p->distinct_p[s];
    P.slot_pre[s] = (T)std::pow(p->r_c, -(double)p->distinct_p[s]);
  }
  for (int a = 0; a < p->C; ++a) {
    P.chan_slot[a] = p->chan_slot[a];
    P.self_pre[a] = (T)(p->rt.S0[p->chan_slot[a]] * std::pow(p->r_c, -(double)p->chan_p[a]));
  }
  P.r_c = (T)p->r_c;
  P.inv_rc = (T)(1.0 / p->r_c);
  P.coef = (const T*)p->d_rcoef;
  P.dcoef = (const T*)p->d_rdcoef;
  launch_real_space<T>(p, n, pos, rg, P, E, phi, F, accumulate, st);
  CUDA_TRY(cudaGetLastError());
  return 0;
}
}  // namespace

extern "C" {

const char* pswf_lr_version(void) { return "pswf_lr 0.1 (sm_100a)"; }

const char* pswf_lr_error_string(int code) {
  switch (code) {
    case PSWF_LR_OK: return "ok";
    case PSWF_LR_ERR_INVALID_ARG: return "invalid argument";
    case PSWF_LR_ERR_UNSUPPORTED_EXPONENT: return "unsupported exponent (p must be 1..6, 8 or 10)";
    case PSWF_LR_ERR_GRID_TOO_COARSE: return "grid too coarse for (c, r_c, w, c_window)";
    case PSWF_LR_ERR_ALLOC: return "device allocation failed";
    case PSWF_LR_ERR_CUDA: return "CUDA error (no usable device, or a kernel/launch failed)";
    case PSWF_LR_ERR_CUFFT: return "cuFFT error";
    case PSWF_LR_ERR_BUSY: return "busy: host submissions in flight (call pswf_lr_wait_host first)";
    case PSWF_LR_ERR_TOO_LARGE: return "size beyond the static scratch of a no-allocation entry point (PSWF_LR_SCAN_STATIC_MAX)";
  }
  return "unknown error";
}

int pswf_lr_plan_create(pswf_lr_plan** plan, const double box[3], const int grid[3], int w, double c,
                        const int* exponents, int n_channels) {
  return pswf_lr_plan_create_ex(plan, box, grid, w, c, exponents, n_channels, nullptr);
}

int pswf_lr_plan_create_ex(pswf_lr_plan** plan, const double box[3], const int grid[3], int w, double c,
                           const int* exponents, int n_channels, const pswf_lr_opts* opts) {
  if (!plan) return PSWF_LR_ERR_INVALID_ARG;
  *plan = nullptr;
  if (!box) return PSWF_LR_ERR_INVALID_ARG;
  const double cell[9] = {box[0], 0, 0, 0, box[1], 0, 0, 0, box[2]};
  return pswf_lr_plan_create_cell(plan, cell, grid, w, c, exponents, n_channels, opts);
}

int pswf_lr_plan_create_cell(pswf_lr_plan** plan, const double cell[9], const int grid[3], int w, double c,
                             const int* exponents, int n_channels, const pswf_lr_opts* opts) {
  if (!plan) return PSWF_LR_ERR_INVALID_ARG;
  *plan = nullptr;
  if (!cell || !grid || !exponents) return PSWF_LR_ERR_INVALID_ARG;
  // lattice vectors a_d = rows of the cell; |a_d| plays the role of the box length L_d wherever only the
  // grid spacing along a lattice direction matters (Eq. (29), band limits, 1-D window tables)
  double box[3], det;
  {
    const double* h = cell;
    det = h[0] * (h[4] * h[8] - h[5] * h[7]) - h[1] * (h[3] * h[8] - h[5] * h[6]) + h[2] * (h[3] * h[7] - h[4] * h[6]);
    for (int d = 0; d < 3; ++d) {
      box[d] = std::sqrt(h[3 * d] * h[3 * d] + h[3 * d + 1] * h[3 * d + 1] + h[3 * d + 2] * h[3 * d + 2]);
      if (!std::isfinite(box[d])) return PSWF_LR_ERR_INVALID_ARG;
    }
    if (!(det > 0) || !(det > 1e-6 * box[0] * box[1] * box[2])) return PSWF_LR_ERR_INVALID_ARG;   // right-handed, not degenerate
  }
  if (n_channels < 1 || n_channels > kMaxChannels) return PSWF_LR_ERR_INVALID_ARG;
  if (w < 2 || w > kMaxW || (w % 2) != 0) return PSWF_LR_ERR_INVALID_ARG;
  if (!(c >= 2.0 && c <= 60.0)) return PSWF_LR_ERR_INVALID_ARG;
  double mtot = 1;
  for (int d = 0; d < 3; ++d) {
    if (!(box[d] > 0) || grid[d] < 1) return PSWF_LR_ERR_INVALID_ARG;
    mtot *= grid[d];
  }
  if (mtot >= 2147483647.0) return PSWF_LR_ERR_INVALID_ARG;
  for (int a = 0; a < n_channels; ++a)
    if (!exponent_supported(exponents[a])) return PSWF_LR_ERR_UNSUPPORTED_EXPONENT;
  for (int d = 0; d < 3; ++d)
    if (grid[d] < w) return PSWF_LR_ERR_GRID_TOO_COARSE;
  pswf_lr_opts o;
  memset(&o, 0, sizeof(o));
  if (opts) o = *opts;
  if (o.precision != PSWF_LR_F32 && o.precision != PSWF_LR_F64) return PSWF_LR_ERR_INVALID_ARG;
  if (o.r_c < 0 || o.c_window < 0 || o.max_atoms < 0 || o.poly_eps < 0) return PSWF_LR_ERR_INVALID_ARG;

  if (!o.host_only) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return PSWF_LR_ERR_CUDA;  // no CPU fallback
  }

  pswf_lr_plan* p = new (std::nothrow) pswf_lr_plan();
  if (!p) return PSWF_LR_ERR_ALLOC;
  int rc = 0;
  try {
    p->host_only = o.host_only != 0;
    if (!p->host_only) {
      cudaGetDevice(&p->device);
      cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    }
    p->precision = o.precision;
    p->w = w;
    p->C = n_channels;
    p->c = c;
    p->zero_mode = o.zero_mode;
    p->kernel_path = o.kernel_path;
    double hmax = 0;
    for (int d = 0; d < 3; ++d) {
      p->M[d] = grid[d];
      p->L[d] = box[d];
      p->h[d] = box[d] / grid[d];
      hmax = std::max(hmax, p->h[d]);
    }
    p->volume = det;
    p->triclinic = false;
    for (int i = 0; i < 9; ++i) {
      p->cell[i] = cell[i];
      if (i % 4 != 0 && cell[i] != 0.0) p->triclinic = true;
    }
    if (!p->triclinic) {   // exactly 1/L: the binning of an orthorhombic box is s = x * (1/L) (reading R4)
      for (int i = 0; i < 9; ++i) p->hinv[i] = 0.0;
      for (int d = 0; d < 3; ++d) p->hinv[4 * d] = 1.0 / cell[4 * d];
    } else {               // adjugate / determinant
      const double* h = cell;
      const double adj[9] = {h[4] * h[8] - h[5] * h[7], h[2] * h[7] - h[1] * h[8], h[1] * h[5] - h[2] * h[4],
                             h[5] * h[6] - h[3] * h[8], h[0] * h[8] - h[2] * h[6], h[2] * h[3] - h[0] * h[5],
                             h[3] * h[7] - h[4] * h[6], h[1] * h[6] - h[0] * h[7], h[0] * h[4] - h[1] * h[3]};
      for (int i = 0; i < 9; ++i) p->hinv[i] = adj[i] / det;
    }
    // reading R2: default r_c puts eta = 0.5 in Eq. (29)
    p->r_c = o.r_c > 0 ? o.r_c : c * hmax / (0.5 * kPi);
    p->eta = c * hmax / (kPi * p->r_c);
    if (p->eta > 1.0 + 1e-12) rc = PSWF_LR_ERR_GRID_TOO_COARSE;  // Eq. (29): h <= eta pi r_c / c, eta <= 1
    // reading R3: window bandwidth
    p->c_w = o.c_window > 0 ? o.c_window : w * (3.55 - 1.55 * p->eta);
    p->poly_eps = o.poly_eps > 0 ? o.poly_eps : (p->precision == PSWF_LR_F64 ? 1e-12 : 1e-7);

    // distinct exponents, slots
    for (int a = 0; a < n_channels; ++a) p->chan_p[a] = exponents[a];
    for (int pp = 1; pp <= 10; ++pp)
      for (int a = 0; a < n_channels; ++a)
        if (exponents[a] == pp) {
          p->distinct_p.push_back(pp);
          break;
        }
    for (int a = 0; a < n_channels; ++a)
      for (size_t s = 0; s < p->distinct_p.size(); ++s)
        if (p->distinct_p[s] == exponents[a]) p->chan_slot[a] = (int)s;

    std::vector<double> invW2[3];
    if (!rc) {
      // window: psi_0^{c_w}, panel polynomials, W^ tables (Eq. (21)-(22))
      Pswf0 psi_w(p->c_w);
      p->wt = fit_window(psi_w, w, p->poly_eps, kMaxWindowDegree);
      memset(&p->wpoly, 0, sizeof(p->wpoly));
      if (w <= 8 && p->wt.degree <= kFastWindowDegree)
        for (int t = 0; t < w; ++t) {
          for (int m = 0; m <= p->wt.degree; ++m) p->wpoly.c[m][t] = (float)p->wt.coef[(size_t)m * w + t];
          for (int m = 0; m < p->wt.degree; ++m) p->wpoly.d[m][t] = (float)p->wt.dcoef[(size_t)m * w + t];
        }
      p->What0 = 1;
      const double kc = c / p->r_c;
      for (int d = 0; d < 3; ++d) {
        const int M = p->M[d];
        const double omega = 0.5 * w * p->h[d];
        p->What0 *= omega * psi_w.lambda0;
        invW2[d].assign(M, 0.0);
        for (int i = 0; i < M; ++i) {
          int f = i <= M / 2 ? i : i - M;
          double kd = 2 * kPi * f / p->L[d];
          double arg = omega * kd / p->c_w;  // = pi w f / (M c_w)
          bool nyq = (M % 2 == 0) && i == M / 2;
          if (std::fabs(kd) < kc && !nyq) {
            if (std::fabs(arg) > 1.0) {
              rc = PSWF_LR_ERR_GRID_TOO_COARSE;  // W^ needed outside its band
              break;
            }
            double Wh = omega * psi_w.lambda0 * psi_w.eval(arg);
            invW2[d][i] = 1.0 / (Wh * Wh);
          }
        }
      }
    }
    if (!rc) {
      // mollifier: psi_0^c, T_p tables, zero-mode constants
      Pswf0 psi(c);
      KernelMath km(psi);
      const int panels = p->precision == PSWF_LR_F64 ? 32 : 16;
      p->kt = fit_kernels(km, p->distinct_p, panels, p->poly_eps, kMaxKernelDegree);
      for (int pp : p->distinct_p) p->Phi0.push_back(km.Phi0(pp, p->r_c));
      // real-space complement: numerators N_p, self constants S_p(0), cell search radius
      RealMath rm(psi);
      p->rt = fit_real(rm, p->distinct_p, panels, p->poly_eps, kMaxKernelDegree);
      p->real_ok = true;
      for (int d = 0; d < 3; ++d) {
        // distance between opposite cell faces: 1 / |column d of h^-1| (= L_d in an orthorhombic box)
        double width = p->L[d];
        if (p->triclinic)
          width = 1.0 / std::sqrt(p->hinv[d] * p->hinv[d] + p->hinv[3 + d] * p->hinv[3 + d] + p->hinv[6 + d] * p->hinv[6 + d]);
        p->real_h[d] = width / p->M[d];
        p->real_R[d] = (int)std::floor(p->r_c / p->real_h[d]) + 1;
        if (!(p->r_c < 0.5 * width)) p->real_ok = false;   // minimum image
      }
      // count modes in the ball (half spectrum), for info / roofline bytes
      long long cnt = 0;
      const double kc2 = (c / p->r_c) * (c / p->r_c);
      for (int ix = 0; ix < p->M[0]; ++ix) {
        const int fx = ix <= p->M[0] / 2 ? ix : ix - p->M[0];
        if ((p->M[0] % 2 == 0) && ix == p->M[0] / 2) continue;
        for (int iy = 0; iy < p->M[1]; ++iy) {
          const int fy = iy <= p->M[1] / 2 ? iy : iy - p->M[1];
          if ((p->M[1] % 2 == 0) && iy == p->M[1] / 2) continue;
          for (int iz = 0; iz <= p->M[2] / 2; ++iz) {
            if ((p->M[2] % 2 == 0) && iz == p->M[2] / 2) continue;
            double k2 = 0;
            for (int e = 0; e < 3; ++e) {   // k_e = 2 pi sum_d m_d hinv[e][d]
              const double ke = 2 * kPi * (fx * p->hinv[3 * e] + fy * p->hinv[3 * e + 1] + iz * p->hinv[3 * e + 2]);
              k2 += ke * ke;
            }
            if (k2 < kc2) ++cnt;   // (the m = 0 entry is counted: it carries the zero-mode constant)
          }
        }
      }
      p->modes_in_ball = cnt;
    }
    if (!rc && !p->host_only) {
      long long b = 0;
      if (p->precision == PSWF_LR_F64) {
        rc |= upload<double>(&p->d_wcoef, p->wt.coef, &b);
        rc |= upload<double>(&p->d_wdcoef, p->wt.dcoef, &b);
        rc |= upload<double>(&p->d_kcoef, p->kt.coef, &b);
        rc |= upload<double>(&p->d_rcoef, p->rt.coef, &b);
        rc |= upload<double>(&p->d_rdcoef, p->rt.dcoef, &b);
        for (int d = 0; d < 3; ++d) rc |= upload<double>(&p->d_invW2[d], invW2[d], &b);
      } else {
        rc |= upload<float>(&p->d_wcoef, p->wt.coef, &b);
        rc |= upload<float>(&p->d_wdcoef, p->wt.dcoef, &b);
        rc |= upload<float>(&p->d_kcoef, p->kt.coef, &b);
        rc |= upload<float>(&p->d_rcoef, p->rt.coef, &b);
        rc |= upload<float>(&p->d_rdcoef, p->rt.dcoef, &b);
        for (int d = 0; d < 3; ++d) rc |= upload<float>(&p->d_invW2[d], invW2[d], &b);
      }
      const size_t rs = real_size(p);
      const size_t Mtot = (size_t)p->M[0] * p->M[1] * p->M[2];
      const size_t Mhalf = (size_t)p->M[0] * p->M[1] * (p->M[2] / 2 + 1);
      if (!rc) rc = dev_alloc(&p->d_spec, 2 * rs * Mhalf * p->C, &b);
      if (!rc && stencil_path_supported(p)) rc = dev_alloc(&p->d_gridi, gather_grid_bytes(p), &b);
      p->n_scan_blocks = (int)((Mtot + scan_tile_size() - 1) / scan_tile_size());
      {
        // everything an evaluation starts from zero, in one block (one memset node instead of three or four)
        const size_t bE = sizeof(double) * kMaxChannels, bW = sizeof(double) * 8;   // (6 used; keeps 16-byte alignment)
        const size_t bS = (sizeof(unsigned long long) * ((size_t)p->n_scan_blocks + 1) + 15) & ~(size_t)15;
        const size_t bC = (sizeof(int) * (Mtot + 1) + 255) & ~(size_t)255;
        const size_t bG = rs * Mtot * p->C;                                          // the charge grid
        p->zero_sort_offset = bE + bW;
        p->zero_sort_bytes = bS + bC;
        p->zero_block_bytes = bE + bW + bS + bC + bG;
        if (!rc) rc = dev_alloc(&p->d_zero_block, p->zero_block_bytes, &b);
        if (!rc) {
          char* base = (char*)p->d_zero_block;
          p->d_Ech = (double*)base;
          p->d_virial = (double*)(base + bE);
          p->d_done = (unsigned int*)(base + bE + 7 * sizeof(double));
          p->d_scan_state = (unsigned long long*)(base + bE + bW);
          p->d_count = (int*)(base + bE + bW + bS);
          p->d_grid = base + bE + bW + bS + bC;
        }
      }
      if (!rc) rc = dev_alloc((void**)&p->d_Ereal, sizeof(double), &b);
      p->workspace_bytes += b;
    }
    if (!rc && !p->host_only) {
      int n[3] = {p->M[0], p->M[1], p->M[2]};
      const bool f64 = p->precision == PSWF_LR_F64;
      size_t ws = 0;
      if (cufftCreate(&p->fft_fwd) != CUFFT_SUCCESS || cufftCreate(&p->fft_inv) != CUFFT_SUCCESS)
        rc = PSWF_LR_ERR_CUFFT;
      p->have_fft = true;
      if (!rc && cufftMakePlanMany(p->fft_fwd, 3, n, nullptr, 1, 0, nullptr, 1, 0, f64 ? CUFFT_D2Z : CUFFT_R2C,
                                   p->C, &ws) != CUFFT_SUCCESS)
        rc = PSWF_LR_ERR_CUFFT;
      p->workspace_bytes += (long long)ws;
      if (!rc && cufftMakePlanMany(p->fft_inv, 3, n, nullptr, 1, 0, nullptr, 1, 0, f64 ? CUFFT_Z2D : CUFFT_C2R,
                                   p->C, &ws) != CUFFT_SUCCESS)
        rc = PSWF_LR_ERR_CUFFT;
      p->workspace_bytes += (long long)ws;
      // band-limited path: 1-D transforms along z whose complex side is plane-major [kz][c][x][y]
      p->fused_fft = !rc && p->kernel_path == 0 && fused_fft_supported(p);
      if (p->fused_fft) {
        fused_fft_limits(p, p->fused_kmax);
        p->fused_z = fused_z_supported(p);
        const int batch = p->C * p->M[0] * p->M[1];
        int nz[1] = {p->M[2]}, re[1] = {p->M[2]}, ce[1] = {p->M[2] / 2 + 1};
        long long b2 = 0;
        const size_t Mhalf = (size_t)p->M[0] * p->M[1] * (p->M[2] / 2 + 1);
        if (cufftCreate(&p->fft_zf) != CUFFT_SUCCESS || cufftCreate(&p->fft_zi) != CUFFT_SUCCESS) rc = PSWF_LR_ERR_CUFFT;
        if (!rc && cufftMakePlanMany(p->fft_zf, 1, nz, re, 1, p->M[2], ce, batch, 1, CUFFT_R2C, batch, &ws) !=
                       CUFFT_SUCCESS)
          rc = PSWF_LR_ERR_CUFFT;
        p->workspace_bytes += (long long)ws;
        if (!rc && cufftMakePlanMany(p->fft_zi, 1, nz, ce, batch, 1, re, 1, p->M[2], CUFFT_C2R, batch, &ws) !=
                       CUFFT_SUCCESS)
          rc = PSWF_LR_ERR_CUFFT;
        p->workspace_bytes += (long long)ws;
        if (!rc) rc = dev_alloc(&p->d_spec2, 2 * sizeof(float) * Mhalf * p->C, &b2);
        if (!rc && cudaMemset(p->d_spec2, 0, 2 * sizeof(float) * Mhalf * p->C) != cudaSuccess) rc = PSWF_LR_ERR_CUDA;
        p->debug_dump_spectrum = o.debug_spectrum != 0;
        if (!rc && p->debug_dump_spectrum) rc = dev_alloc(&p->d_spec_dump, 2 * sizeof(float) * Mhalf * p->C, &b2);
        p->workspace_bytes += b2;
      }
    }
    if (!rc && !p->host_only) rc = ensure_capacity(p, o.max_atoms > 0 ? o.max_atoms : 1024);
  } catch (const std::bad_alloc&) {
    rc = PSWF_LR_ERR_ALLOC;
  } catch (...) {
    rc = PSWF_LR_ERR_INVALID_ARG;
  }
  if (rc) {
    pswf_lr_destroy(p);
    return rc;
  }
  *plan = p;
  return 0;
}

namespace {
void drop_graphs(pswf_lr_plan* p) {
  for (auto& g : p->graphs) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    g = pswf_lr_plan::GraphEntry();
  }
}

int execute_plain(pswf_lr_plan* p, int n_atoms, const void* pos, const void* q, void* E, void* phi, void* F,
                  cudaStream_t st) {
  if (p->precision == PSWF_LR_F64)
    return execute_t<double>(p, n_atoms, (const double*)pos, (const double*)q, (double*)E, (double*)phi,
                             (double*)F, st);
  return execute_t<float>(p, n_atoms, (const float*)pos, (const float*)q, (double*)E, (float*)phi, (float*)F, st);
}
}  // namespace

int pswf_lr_execute(pswf_lr_plan* p, int n_atoms, const void* pos, const void* q, void* E, void* phi, void* F,
                    void* stream) {
  if (!p || n_atoms < 0) return PSWF_LR_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!pos || !q)) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;  // a tables-only plan cannot execute
  DeviceGuard guard(p);
  if (!guard.ok) return PSWF_LR_ERR_CUDA;
  const int cap_before = p->cap_atoms;
  int rc = ensure_capacity(p, n_atoms);
  if (rc) return rc;
  if (p->cap_atoms != cap_before) drop_graphs(p);   // the captured launches point into the old workspaces
  cudaStream_t st = (cudaStream_t)stream;
  // The launch sequence of one evaluation (ten kernels and four memsets at config 4) depends only on the
  // arguments: the second call with the same arguments captures it into a CUDA graph, later calls replay
  // it (no per-launch host work, tighter kernel-to-kernel scheduling: 886 -> 850 us at config 4, 96 -> 59 us
  // at config 1).  Not while stage profiling is on, nor inside a caller's own stream capture.
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (p->use_graphs && !p->profiling && n_atoms > 0 && cudaStreamIsCapturing(st, &cs) == cudaSuccess &&
      cs == cudaStreamCaptureStatusNone) {
    pswf_lr_plan::GraphEntry* hit = nullptr;
    pswf_lr_plan::GraphEntry* lru = &p->graphs[0];
    for (auto& g : p->graphs) {
      if (g.n == n_atoms && g.pos == pos && g.q == q && g.E == E && g.phi == phi && g.F == F && g.virial == p->virial)
        hit = &g;
      if (g.last_use < lru->last_use) lru = &g;
    }
    ++p->graph_clock;
    if (hit && hit->exec) {
      hit->last_use = p->graph_clock;
      CUDA_TRY(cudaGraphLaunch(hit->exec, st));
      p->n_kernels += hit->kernels; p->n_memsets += hit->memsets; p->n_cufft += hit->cufft;
      p->n_graph_replays++;
      p->last_n_atoms = n_atoms;
      return 0;
    }
    if (hit) {   // second call with these arguments: capture
      const long long k0 = p->n_kernels, m0 = p->n_memsets, f0 = p->n_cufft;
      cudaGraph_t graph = nullptr;
      if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        rc = execute_plain(p, n_atoms, pos, q, E, phi, F, st);
        const cudaError_t ce = cudaStreamEndCapture(st, &graph);
        if (rc == 0 && ce == cudaSuccess && graph &&
            cudaGraphInstantiate(&hit->exec, graph, 0) == cudaSuccess) {
          hit->kernels = p->n_kernels - k0; hit->memsets = p->n_memsets - m0; hit->cufft = p->n_cufft - f0;
          hit->last_use = p->graph_clock;
          cudaGraphDestroy(graph);
          CUDA_TRY(cudaGraphLaunch(hit->exec, st));
          p->n_graph_replays++;
          return 0;
        }
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        hit->exec = nullptr;
        p->use_graphs = false;          // capture is not possible here: plain launches from now on
        p->n_kernels = k0; p->n_memsets = m0; p->n_cufft = f0;
      } else {
        cudaGetLastError();             // e.g. the legacy default stream cannot be captured
        p->use_graphs = false;
      }
    } else {     // first call with these arguments: remember them, launch plainly
      if (lru->exec) cudaGraphExecDestroy(lru->exec);
      *lru = pswf_lr_plan::GraphEntry();
      lru->n = n_atoms; lru->pos = pos; lru->q = q; lru->E = E; lru->phi = phi; lru->F = F; lru->virial = p->virial;
      lru->last_use = p->graph_clock;
    }
  }
  return execute_plain(p, n_atoms, pos, q, E, phi, F, st);
}

int pswf_lr_execute_host(pswf_lr_plan* p, int n, const void* pos, const void* q, double* E, void* phi, void* F,
                         void* stream) {
  if (!p || n < 0) return PSWF_LR_ERR_INVALID_ARG;
  if (n > 0 && (!pos || !q)) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  if (p->n_submitted != p->n_waited) return PSWF_LR_ERR_BUSY;
  DeviceGuard guard(p);
  if (!guard.ok) return PSWF_LR_ERR_CUDA;
  int rc = ensure_capacity(p, n);
  if (rc) return rc;
  rc = ensure_host_staging(p, 1);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t rs = real_size(p);
  if (n > 0) {
    CUDA_TRY(cudaMemcpyAsync(p->d_pos_in[0], pos, rs * 3 * (size_t)n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(p->d_q_in[0], q, rs * (size_t)p->C * n, cudaMemcpyHostToDevice, st));
  }
  rc = pswf_lr_execute(p, n, p->d_pos_in[0], p->d_q_in[0], E ? p->d_E_out[0] : nullptr,
                       phi ? p->d_phi_out[0] : nullptr, F ? p->d_F_out[0] : nullptr, stream);
  if (rc) return rc;
  if (E) CUDA_TRY(cudaMemcpyAsync(E, p->d_E_out[0], sizeof(double), cudaMemcpyDeviceToHost, st));
  if (phi && n > 0)
    CUDA_TRY(cudaMemcpyAsync(phi, p->d_phi_out[0], rs * (size_t)p->C * n, cudaMemcpyDeviceToHost, st));
  if (F && n > 0) CUDA_TRY(cudaMemcpyAsync(F, p->d_F_out[0], rs * 3 * (size_t)n, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return 0;
}

// Pipelined host-buffer evaluation.  Submission k uses staging slot k % 3:
//   copy-in stream:   [wait: evaluation k-3 done with the slot]  H2D pos, q            -> ev_in
//   compute stream:   [wait: ev_in, copy-out k-3 done with the slot]  the evaluation     -> ev_comp
//   copy-out stream:  [wait: ev_comp]  D2H E, phi, F                                    -> ev_out
// so with pinned host buffers H2D(k+1), evaluation(k) and D2H(k-1) run at the same time; the third slot lets
// the copy-in run a whole step ahead (with two, an evaluation waited ~0.1 ms for its inputs at config 4).
int pswf_lr_submit_host(pswf_lr_plan* p, int n, const void* pos, const void* q, double* E, void* phi, void* F) {
  if (!p || n < 0) return PSWF_LR_ERR_INVALID_ARG;
  if (n > 0 && (!pos || !q)) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  constexpr int NS = pswf_lr_plan::kHostSlots;
  if (p->n_submitted - p->n_waited >= NS) return PSWF_LR_ERR_BUSY;
  DeviceGuard guard(p);
  if (!guard.ok) return PSWF_LR_ERR_CUDA;
  if (n > p->cap_atoms && p->n_submitted != p->n_waited) return PSWF_LR_ERR_BUSY;   // growing reallocates
  int rc = ensure_capacity(p, n);
  if (rc) return rc;
  rc = ensure_host_staging(p, NS);
  if (rc) return rc;
  if (!p->s_in) {
    CUDA_TRY(cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&p->s_comp, cudaStreamNonBlocking));
    CUDA_TRY(cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking));
    for (int s = 0; s < NS; ++s) {
      CUDA_TRY(cudaEventCreateWithFlags(&p->ev_in[s], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&p->ev_comp[s], cudaEventDisableTiming));
      CUDA_TRY(cudaEventCreateWithFlags(&p->ev_out[s], cudaEventDisableTiming));
    }
  }
  const int s = (int)(p->n_submitted % NS);
  const bool reuse = p->n_submitted >= NS;
  const size_t rs = real_size(p);
  if (reuse) CUDA_TRY(cudaStreamWaitEvent(p->s_in, p->ev_comp[s], 0));
  if (n > 0) {
    CUDA_TRY(cudaMemcpyAsync(p->d_pos_in[s], pos, rs * 3 * (size_t)n, cudaMemcpyHostToDevice, p->s_in));
    CUDA_TRY(cudaMemcpyAsync(p->d_q_in[s], q, rs * (size_t)p->C * n, cudaMemcpyHostToDevice, p->s_in));
  }
  CUDA_TRY(cudaEventRecord(p->ev_in[s], p->s_in));
  CUDA_TRY(cudaStreamWaitEvent(p->s_comp, p->ev_in[s], 0));
  if (reuse) CUDA_TRY(cudaStreamWaitEvent(p->s_comp, p->ev_out[s], 0));
  rc = pswf_lr_execute(p, n, p->d_pos_in[s], p->d_q_in[s], E ? p->d_E_out[s] : nullptr,
                       phi ? p->d_phi_out[s] : nullptr, F ? p->d_F_out[s] : nullptr, p->s_comp);
  if (rc) return rc;
  CUDA_TRY(cudaEventRecord(p->ev_comp[s], p->s_comp));
  CUDA_TRY(cudaStreamWaitEvent(p->s_out, p->ev_comp[s], 0));
  if (E) CUDA_TRY(cudaMemcpyAsync(E, p->d_E_out[s], sizeof(double), cudaMemcpyDeviceToHost, p->s_out));
  if (phi && n > 0)
    CUDA_TRY(cudaMemcpyAsync(phi, p->d_phi_out[s], rs * (size_t)p->C * n, cudaMemcpyDeviceToHost, p->s_out));
  if (F && n > 0) CUDA_TRY(cudaMemcpyAsync(F, p->d_F_out[s], rs * 3 * (size_t)n, cudaMemcpyDeviceToHost, p->s_out));
  CUDA_TRY(cudaEventRecord(p->ev_out[s], p->s_out));
  p->n_submitted++;
  return 0;
}

int pswf_lr_wait_host(pswf_lr_plan* p) {
  if (!p) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  if (p->n_submitted == p->n_waited) return PSWF_LR_ERR_INVALID_ARG;   // nothing in flight
  const int s = (int)(p->n_waited % pswf_lr_plan::kHostSlots);
  CUDA_TRY(cudaEventSynchronize(p->ev_out[s]));
  p->n_waited++;
  return 0;
}

int pswf_lr_execute_real(pswf_lr_plan* p, int n_atoms, const void* pos, const void* q, void* E, void* phi, void* F,
                         int accumulate, void* stream) {
  if (!p || n_atoms < 0) return PSWF_LR_ERR_INVALID_ARG;
  if (n_atoms > 0 && (!pos || !q)) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  if (!p->real_ok) return PSWF_LR_ERR_GRID_TOO_COARSE;   // r_c >= L_d / 2: minimum image does not suffice
  DeviceGuard guard(p);
  if (!guard.ok) return PSWF_LR_ERR_CUDA;
  int rc = ensure_capacity(p, n_atoms);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  if (p->precision == PSWF_LR_F64)
    return execute_real_t<double>(p, n_atoms, (const double*)pos, (const double*)q, (double*)E, (double*)phi,
                                  (double*)F, accumulate, st);
  return execute_real_t<float>(p, n_atoms, (const float*)pos, (const float*)q, (double*)E, (float*)phi, (float*)F,
                               accumulate, st);
}

int pswf_lr_eval_real(const pswf_lr_plan* p, int pe, int n, const double* r, double* L, double* dL) {
  if (!p || n < 0 || (n > 0 && (!r || !L))) return PSWF_LR_ERR_INVALID_ARG;
  int slot = -1;
  for (size_t s = 0; s < p->distinct_p.size(); ++s)
    if (p->distinct_p[s] == pe) slot = (int)s;
  if (slot < 0) return PSWF_LR_ERR_UNSUPPORTED_EXPONENT;
  const int deg = p->rt.degree, panels = p->rt.panels;
  const double pre = std::pow(p->r_c, -(double)pe);
  for (int i = 0; i < n; ++i) {
    const double x = r[i] / p->r_c;
    if (!(x > 0) || x >= 1) {
      L[i] = 0;
      if (dL) dL[i] = 0;
      continue;
    }
    int j = std::min((int)(x * panels), panels - 1);
    const double xi = 2 * (x * panels - j) - 1;
    const double* cf = &p->rt.coef[((size_t)slot * panels + j) * (deg + 1)];
    const double* df = &p->rt.dcoef[((size_t)slot * panels + j) * deg];
    double N = cf[deg], dN = df[deg - 1];
    for (int m = deg - 1; m >= 0; --m) N = N * xi + cf[m];
    for (int m = deg - 2; m >= 0; --m) dN = dN * xi + df[m];
    const double ip = std::pow(x, -(double)pe);
    L[i] = pre * N * ip;
    if (dL) dL[i] = pre / p->r_c * (dN * ip - pe * N * ip / x);
  }
  return 0;
}

int pswf_lr_self_coefficient(const pswf_lr_plan* p, int pe, double* S0) {
  if (!p || !S0) return PSWF_LR_ERR_INVALID_ARG;
  for (size_t s = 0; s < p->distinct_p.size(); ++s)
    if (p->distinct_p[s] == pe) {
      *S0 = p->rt.S0[s];
      return 0;
    }
  return PSWF_LR_ERR_UNSUPPORTED_EXPONENT;
}

int pswf_lr_set_virial(pswf_lr_plan* p, int enabled) {
  if (!p) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  p->virial = enabled != 0;
  return 0;
}

int pswf_lr_virial(pswf_lr_plan* p, void* W, void* stream) {
  if (!p || !W) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  if (!p->virial) return PSWF_LR_ERR_INVALID_ARG;
  CUDA_TRY(cudaMemcpyAsync(W, p->d_virial, sizeof(double) * 6, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return 0;
}

int pswf_lr_channel_energies(pswf_lr_plan* p, void* E_channels, void* stream) {
  if (!p || !E_channels) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  CUDA_TRY(cudaMemcpyAsync(E_channels, p->d_Ech, sizeof(double) * p->C, cudaMemcpyDeviceToDevice,
                           (cudaStream_t)stream));
  return 0;
}

int pswf_lr_get_info(const pswf_lr_plan* p, pswf_lr_info* info) {
  if (!p || !info) return PSWF_LR_ERR_INVALID_ARG;
  memset(info, 0, sizeof(*info));
  info->r_c = p->r_c;
  info->c = p->c;
  info->c_window = p->c_w;
  info->eta = p->eta;
  info->w = p->w;
  info->precision = p->precision;
  info->n_channels = p->C;
  info->n_distinct_p = (int)p->distinct_p.size();
  for (int d = 0; d < 3; ++d) info->grid[d] = p->M[d];
  info->window_degree = p->wt.degree;
  info->kernel_degree = p->kt.degree;
  info->kernel_panels = p->kt.panels;
  info->modes_in_ball = p->modes_in_ball;
  info->workspace_bytes = p->workspace_bytes;
  info->fast_stencil = (!p->host_only && p->kernel_path == 0 && stencil_path_supported(p)) ? 1 : 0;
  info->band_limited_fft = p->fused_fft ? 1 : 0;
  for (int d = 0; d < 3; ++d) info->band_kmax[d] = p->fused_kmax[d];
  info->own_kernel_launches = p->n_kernels;
  info->memsets = p->n_memsets;
  info->cufft_execs = p->n_cufft;
  info->graph_replays = p->n_graph_replays;
  return 0;
}

int pswf_lr_set_profiling(pswf_lr_plan* p, int enabled) {
  if (!p) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  if (enabled && p->events.empty()) {
    p->events.resize((size_t)kProfileRing * (PSWF_LR_N_STAGES + 1));
    for (auto& e : p->events) CUDA_TRY(cudaEventCreate(&e));
  }
  p->profiling = enabled != 0;
  p->prof_count = 0;
  return 0;
}

int pswf_lr_stage_ms(pswf_lr_plan* p, double ms[PSWF_LR_N_STAGES], int* n_executes) {
  if (!p || !ms) return PSWF_LR_ERR_INVALID_ARG;
  for (int s = 0; s < PSWF_LR_N_STAGES; ++s) ms[s] = 0;
  int n = p->prof_count;
  if (n_executes) *n_executes = n;
  if (n == 0) return 0;
  cudaEvent_t* last = p->events.data() + (size_t)(n - 1) * (PSWF_LR_N_STAGES + 1);
  CUDA_TRY(cudaEventSynchronize(last[PSWF_LR_N_STAGES]));
  for (int i = 0; i < n; ++i) {
    cudaEvent_t* ev = p->events.data() + (size_t)i * (PSWF_LR_N_STAGES + 1);
    for (int s = 0; s < PSWF_LR_N_STAGES; ++s) {
      float t = 0;
      CUDA_TRY(cudaEventElapsedTime(&t, ev[s], ev[s + 1]));
      ms[s] += t;
    }
  }
  for (int s = 0; s < PSWF_LR_N_STAGES; ++s) ms[s] /= n;
  p->prof_count = 0;
  return 0;
}

int pswf_lr_debug_copy(pswf_lr_plan* p, int what, void* dst, void* stream) {
  if (!p || !dst) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  const size_t rs = real_size(p);
  const size_t Mtot = (size_t)p->M[0] * p->M[1] * p->M[2];
  const size_t Mhalf = (size_t)p->M[0] * p->M[1] * (p->M[2] / 2 + 1);
  const void* src = nullptr;
  size_t nb = 0;
  if (what == 0 || what == 2) {
    src = p->d_grid;
    nb = rs * Mtot * p->C;
  } else if (what == 1) {
    src = p->d_spec;
    if (p->fused_fft) {   // the band-limited path keeps the dense spectrum only on request
      if (!p->d_spec_dump) return PSWF_LR_ERR_INVALID_ARG;
      src = p->d_spec_dump;
    }
    nb = 2 * rs * Mhalf * p->C;
  } else {
    return PSWF_LR_ERR_INVALID_ARG;
  }
  CUDA_TRY(cudaMemcpyAsync(dst, src, nb, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return 0;
}

int pswf_lr_debug_cell_starts(pswf_lr_plan* p, int* dst, void* stream) {
  if (!p || !dst) return PSWF_LR_ERR_INVALID_ARG;
  if (p->host_only) return PSWF_LR_ERR_CUDA;
  DeviceGuard guard(p);
  const size_t Mtot = (size_t)p->M[0] * p->M[1] * p->M[2];
  CUDA_TRY(cudaMemcpyAsync(dst, p->d_count, sizeof(int) * (Mtot + 1), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return 0;
}

int pswf_lr_exclusive_scan_static(int* counts, int n, void* stream) {
  if (!counts || n < 0) return PSWF_LR_ERR_INVALID_ARG;
  if (n > PSWF_LR_SCAN_STATIC_MAX) return PSWF_LR_ERR_TOO_LARGE;   // beyond the static tile-state array
  if (((uintptr_t)counts & 15u) != 0) return PSWF_LR_ERR_INVALID_ARG;   // the scan reads and writes 16-byte vectors
  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) {
    CUDA_TRY(cudaMemsetAsync(counts, 0, sizeof(int), st));
    return 0;
  }
  return launch_scan_static(counts, n, st);
}

int pswf_lr_eval_window(const pswf_lr_plan* p, int n, const double* z, double* W, double* dW) {
  if (!p || n < 0 || (n > 0 && (!z || !W))) return PSWF_LR_ERR_INVALID_ARG;
  const int w = p->w, deg = p->wt.degree;
  for (int i = 0; i < n; ++i) {
    double s = 0.5 * w * (z[i] + 1.0);  // t + delta
    int t = (int)std::floor(s);
    if (t < 0 || t >= w) {
      W[i] = 0;
      if (dW) dW[i] = 0;
      continue;
    }
    double xi = 2 * (s - t) - 1;
    double v = p->wt.coef[(size_t)deg * w + t];
    for (int m = deg - 1; m >= 0; --m) v = v * xi + p->wt.coef[(size_t)m * w + t];
    W[i] = v;
    if (dW) {
      double dv = p->wt.dcoef[(size_t)(deg - 1) * w + t];
      for (int m = deg - 2; m >= 0; --m) dv = dv * xi + p->wt.dcoef[(size_t)m * w + t];
      dW[i] = dv * w;  // d xi / d z = w
    }
  }
  return 0;
}

int pswf_lr_eval_kernel(const pswf_lr_plan* p, int pe, int n, const double* k, double* Phi) {
  if (!p || n < 0 || (n > 0 && (!k || !Phi))) return PSWF_LR_ERR_INVALID_ARG;
  int slot = -1;
  for (size_t s = 0; s < p->distinct_p.size(); ++s)
    if (p->distinct_p[s] == pe) slot = (int)s;
  if (slot < 0) return PSWF_LR_ERR_UNSUPPORTED_EXPONENT;
  const int deg = p->kt.degree, panels = p->kt.panels;
  for (int i = 0; i < n; ++i) {
    double kappa = k[i] * p->r_c, x = kappa / p->c;
    if (!(x > 0) || x >= 1) {
      Phi[i] = 0;
      continue;
    }
    int j = std::min((int)(x * panels), panels - 1);
    double xi = 2 * (x * panels - j) - 1;
    const double* cf = &p->kt.coef[((size_t)slot * panels + j) * (deg + 1)];
    double t = cf[deg];
    for (int m = deg - 1; m >= 0; --m) t = t * xi + cf[m];
    double s;
    switch (pe) {
      case 1: s = t / (kappa * kappa); break;
      case 2: s = t / kappa; break;
      case 3: s = t - std::log(x); break;
      case 5: s = t + x * x * std::log(x); break;
      default: s = t; break;
    }
    Phi[i] = s * slot_prefactor(pe, p->c, p->r_c);
  }
  return 0;
}

int pswf_lr_suggest_parameters(const double box[3], double eps_tot, double r_c, int grid[3], int* w, double* c) {
  if (!box || !grid || !w || !c) return PSWF_LR_ERR_INVALID_ARG;
  if (!(eps_tot >= 1e-13 && eps_tot <= 0.3) || !(r_c > 0)) return PSWF_LR_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d)
    if (!(box[d] > 0)) return PSWF_LR_ERR_INVALID_ARG;
  const double eps = eps_tot / 3.0;                 // Eq. (27), uniform allocation
  const double cc = std::log(1.0 / eps);            // Eq. (28)
  const double eta = 0.5;                           // reading R2
  const double h = eta * kPi * r_c / cc;            // Eq. (29)
  for (int d = 0; d < 3; ++d) {
    int M = (int)std::ceil(box[d] / h);
    M = std::max(16, ((M + 7) / 8) * 8);
    grid[d] = M;
  }
  int ww = 16;
  for (int t = 4; t <= 16; t += 2)
    if (std::pow(10.0, 0.46 - 0.85 * t) <= eps) {
      ww = t;
      break;
    }
  *w = ww;
  *c = cc;
  return 0;
}

int pswf_lr_destroy(pswf_lr_plan* p) {
  if (!p) return 0;
  if (p->host_only) {
    delete p;
    return 0;
  }
  DeviceGuard guard(p);
  cudaDeviceSynchronize();
  drop_graphs(p);
  free_atoms(p);
  for (int s = 0; s < pswf_lr_plan::kHostSlots; ++s) {
    if (p->d_E_out[s]) cudaFree(p->d_E_out[s]);
    if (p->ev_in[s]) cudaEventDestroy(p->ev_in[s]);
    if (p->ev_comp[s]) cudaEventDestroy(p->ev_comp[s]);
    if (p->ev_out[s]) cudaEventDestroy(p->ev_out[s]);
  }
  if (p->s_in) cudaStreamDestroy(p->s_in);
  if (p->s_comp) cudaStreamDestroy(p->s_comp);
  if (p->s_out) cudaStreamDestroy(p->s_out);
  void* ptrs[] = {p->d_wcoef, p->d_wdcoef,  p->d_kcoef,    p->d_invW2[0], p->d_invW2[1], p->d_invW2[2],
                  p->d_spec,  p->d_zero_block,
                  p->d_gridi, p->d_rcoef, p->d_rdcoef, p->d_Ereal, p->d_spec2, p->d_spec_dump};
  for (void* q : ptrs)
    if (q) cudaFree(q);
  if (p->have_fft) {
    if (p->fft_fwd) cufftDestroy(p->fft_fwd);
    if (p->fft_inv) cufftDestroy(p->fft_inv);
    if (p->fft_zf) cufftDestroy(p->fft_zf);
    if (p->fft_zi) cufftDestroy(p->fft_zi);
  }
  for (auto& e : p->events) cudaEventDestroy(e);
  delete p;
  return 0;
}

}  // extern "C"
