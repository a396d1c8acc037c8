// Plan object shared by the translation units of libpswf_lr (product code, sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>

#include <vector>

#include "../../include/pswf_lr.h"
#include "host_tables.hpp"
#include "real_tables.hpp"

namespace pswf {

constexpr int kMaxChannels = 32;
constexpr int kMaxSlots = 8;       // distinct exponents: 1..6, 8, 10
constexpr int kMaxW = 16;
constexpr int kMaxWindowDegree = 30;
constexpr int kMaxKernelDegree = 24;
constexpr int kProfileRing = 512;
constexpr int kFastWindowDegree = 12;   // fast fp32 path: panel polynomials zero-padded to this degree

// Window panel polynomials of the fast fp32 path, passed to kernels by value (constant bank):
// c[m][t] = coefficient of xi^m of panel t (zero for t >= w or m > degree); d = d/dxi of the same.
struct WindowPoly {
  float c[kFastWindowDegree + 1][8];
  float d[kFastWindowDegree][8];
};

// Parameters of the scale (deconvolve x Green) kernel, passed by value.
template <class T>
struct ScaleParams {
  int M[3];
  int Mzh;             // Mz/2 + 1
  int C;               // channels
  int nslots;          // distinct exponents
  int slot_p[kMaxSlots];   // exponent of each slot
  int chan_slot[kMaxChannels];
  T chan_D0[kMaxChannels];   // multiplier of the m = 0 mode per channel (0 when dropped)
  T slot_pre[kMaxSlots];   // r_c^(3-p) * constant prefactor of each slot
  T recip[9];          // reciprocal basis 2 pi h^-T: k_e = sum_d m_d recip[3 d + e] (diagonal 2 pi / L_d when orthorhombic)
  T x_per_k;           // r_c / c
  T c;                 // mollifier bandwidth
  T base;              // h_x h_y h_z / M_tot
  int panels, degree;
  const T* kcoef;      // [slot][panel][degree+1]
  const T* invW2[3];   // 1 / W^_d(m)^2 per signed DFT index
};

// Geometry used by bin/spread/gather kernels.
template <class T>
struct GridGeom {
  int M[3];
  int w;
  double hinv[9];      // h^-1, s = r h^-1 (binning is done in double, reading R4); diag(1/L_d) when orthorhombic
  T hinv_t[9];         // the same in plan precision: Cartesian gradient from fractional components
  T dxi_ds[3];         // d xi / d s_d = -2 M_d
  int wdeg;            // window polynomial degree
  const T* wcoef;      // [(wdeg+1)][w]
  const T* wdcoef;     // [wdeg][w]
};

// Geometry and tables of the real-space complement kernel (kernels_real.cu), passed by value.
template <class T>
struct RealGeom {
  int M[3];
  int R[3];            // cell search radius per dimension: floor(r_c / h_d) + 1
  double invL[3];
  T L[3];
  T h[3];              // cell size of the sort: distance between neighbouring grid planes (h_d in an orthorhombic box)
  T inv_hz;
  // general cells (tri != 0): positions are kept as wrapped FRACTIONAL coordinates, the minimum image is taken
  // there (valid for r_c < half the smallest distance between opposite cell faces, host-checked) and
  // converted with the lattice vectors hm[3 d + e] (row d = vector a_d)
  int tri;
  double hinv[9];      // h^-1: s_d = sum_e r_e hinv[3 e + d]
  T hm[9];
};
template <class T>
struct RealParams {
  int C, nslots, panels, degree;
  int slot_p[kMaxSlots];
  int chan_slot[kMaxChannels];
  T slot_pre[kMaxSlots];       // r_c^-p per slot
  T self_pre[kMaxChannels];    // S_p(0) / r_c^p per channel
  T r_c, inv_rc;
  const T* coef;               // [slot][panel][degree+1]  N_p
  const T* dcoef;              // [slot][panel][degree]    dN_p/dx
};

}  // namespace pswf

struct pswf_lr_plan {
  // resolved parameters
  int precision = 0, w = 0, C = 0, zero_mode = 0, kernel_path = 0;
  int M[3] = {0, 0, 0};
  double L[3] = {0, 0, 0}, h[3] = {0, 0, 0};   // |a_d| (edge lengths) and |a_d| / M_d
  double cell[9] = {0}, hinv[9] = {0};         // lattice vectors (rows) and h^-1; diagonal when orthorhombic
  double volume = 0;                           // |det h|
  bool triclinic = false;
  double c = 0, r_c = 0, c_w = 0, eta = 0, poly_eps = 0;
  int chan_p[pswf::kMaxChannels] = {0};
  int chan_slot[pswf::kMaxChannels] = {0};
  std::vector<int> distinct_p;
  std::vector<double> Phi0;       // per distinct p
  double What0 = 0;               // W^(0) = prod_d omega_d lambda_0
  long long modes_in_ball = 0;
  long long workspace_bytes = 0;
  long long atom_bytes = 0;       // part of workspace_bytes that scales with the atom capacity
  // host tables
  pswf::WindowTable wt;
  pswf::KernelTable kt;
  pswf::WindowPoly wpoly;         // fast path copy of wt (float, zero padded)
  pswf::RealTable rt;             // real-space complement numerators N_p, S_p(0)
  int real_R[3] = {0, 0, 0};      // cell search radius of the pair kernel
  double real_h[3] = {0, 0, 0};   // distance between neighbouring grid planes (h_d in an orthorhombic box)
  bool real_ok = false;           // r_c < L_d / 2 and 2 R_d + 1 <= M_d in every dimension
  void* d_rcoef = nullptr;
  void* d_rdcoef = nullptr;
  void* d_spos = nullptr;         // real [3][cap] wrapped positions in sorted order
  double* d_Ereal = nullptr;      // [1]
  double* d_virial = nullptr;     // [6] xx, yy, zz, xy, xz, yz (when virial accumulation is enabled)
  bool virial = false;
  // device tables (plan precision)
  void* d_wcoef = nullptr;
  void* d_wdcoef = nullptr;
  void* d_kcoef = nullptr;
  void* d_invW2[3] = {nullptr, nullptr, nullptr};
  // device workspaces
  void* d_grid = nullptr;         // real  [C][Mx][My][Mz]
  void* d_gridi = nullptr;        // real  [M][CB] channel-interleaved copy of the potential grid (fast gather)
  void* d_spec = nullptr;         // cplx  [C][Mx][My][Mz/2+1]
  int* d_count = nullptr;         // [Mtot + 1] cell counts -> exclusive starts
  unsigned long long* d_scan_state = nullptr;   // [1 + n_scan_blocks] ticket counter + tile states of the scan
  int n_scan_blocks = 0;
  // One allocation, zero-filled by ONE memset per evaluation: [d_Ech | d_virial | d_scan_state | d_count | d_grid]
  // (the sort of pswf_lr_execute_real zeroes d_scan_state and d_count only: the energies and the potential grid
  // of the preceding execute stay readable)
  void* d_zero_block = nullptr;
  unsigned int* d_done = nullptr;   // finished CTAs of the fused multiply kernel (last one sums the energies)
  size_t zero_block_bytes = 0, zero_sort_offset = 0, zero_sort_bytes = 0;
  double* d_Ech = nullptr;        // [C]
  // per-atom workspaces (capacity cap_atoms)
  int cap_atoms = 0;
  int* d_key = nullptr;
  int* d_rank = nullptr;
  int* d_perm = nullptr;
  int* d_si0 = nullptr;           // [3][cap] unwrapped first grid index
  void* d_sdelta = nullptr;       // real [3][cap]
  void* d_sq = nullptr;           // real [C][cap]
  void* d_rec = nullptr;          // fast path: per-atom weight records
  void* d_drec = nullptr;         // fast path: per-atom derivative-weight records (gather)
  // host-buffer entry points: three staging slots (slot 0 serves pswf_lr_execute_host; submit / wait
  // cycle through them so that copy-in, evaluation and copy-out of consecutive submissions overlap)
  static constexpr int kHostSlots = 3;
  void* d_pos_in[kHostSlots] = {};
  void* d_q_in[kHostSlots] = {};
  void* d_phi_out[kHostSlots] = {};
  void* d_F_out[kHostSlots] = {};
  double* d_E_out[kHostSlots] = {};
  cudaStream_t s_in = nullptr, s_comp = nullptr, s_out = nullptr;
  cudaEvent_t ev_in[kHostSlots] = {}, ev_comp[kHostSlots] = {}, ev_out[kHostSlots] = {};
  long long n_submitted = 0, n_waited = 0;
  int last_n_atoms = 0;
  // launch accounting (pswf_lr_info): this library's own kernels, memsets, cuFFT executions since creation
  long long n_kernels = 0, n_memsets = 0, n_cufft = 0;
  // launch sequences of pswf_lr_execute cached as CUDA graphs, keyed by the call's arguments (an MD loop
  // passes the same device buffers every step); invalidated when workspaces are reallocated
  struct GraphEntry {
    int n = -1;
    const void *pos = nullptr, *q = nullptr;
    void *E = nullptr, *phi = nullptr, *F = nullptr;
    bool virial = false;
    cudaGraphExec_t exec = nullptr;
    long long kernels = 0, memsets = 0, cufft = 0;   // launches one replay stands for
    long long last_use = 0;
  };
  static constexpr int kGraphEntries = 4;
  GraphEntry graphs[kGraphEntries];
  bool use_graphs = true;
  long long graph_clock = 0, n_graph_replays = 0;
  // cuFFT
  cufftHandle fft_fwd = 0, fft_inv = 0;
  bool have_fft = false;
  // band-limited transform path (kernels_fft.cu): z transforms with plane-major spectra + k_xy_scale
  bool fused_fft = false;
  bool fused_z = false;           // z transforms by k_z_forward / k_z_inverse instead of cuFFT
  int fused_kmax[3] = {0, 0, 0};  // kept signed DFT indices per dimension: |f| <= kmax (never Nyquist)
  cufftHandle fft_zf = 0, fft_zi = 0;
  void* d_spec2 = nullptr;        // cplx [Mz/2+1][C][Mx][My]; planes beyond the band stay zero
  int gather_group = 4;           // channels per gather pass / interleaved grid group (4, or 2: narrower register window)
  bool debug_dump_spectrum = false;
  void* d_spec_dump = nullptr;    // cplx [C][Mx][My][Mz/2+1] dense copy of the scaled modes (test hook)
  // profiling
  bool profiling = false;
  std::vector<cudaEvent_t> events;  // kProfileRing * (N_STAGES + 1)
  int prof_count = 0;
  int device = 0;
  bool host_only = false;
  int sm_count = 148;
};
