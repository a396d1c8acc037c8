// Host-side launchers of the PSWF-LR kernels (declarations).
#pragma once
#include "plan.hpp"

namespace pswf {

template <class T>
void launch_bin_sort(pswf_lr_plan* p, int n, const T* pos, const T* q, const GridGeom<T>& g, bool scatter,
                     bool zero_energy, cudaStream_t st);
int scan_tile_size();   // counts per tile of the single-pass scan (sizes its state array)
int launch_scan_static(int* data, int n, cudaStream_t st);   // 1 <= n <= PSWF_LR_SCAN_STATIC_MAX; no allocation
template <class T>
void launch_spread_ref(pswf_lr_plan* p, int n, const GridGeom<T>& g, cudaStream_t st);
template <class T>
void launch_scale(pswf_lr_plan* p, const ScaleParams<T>& P, bool want_E, cudaStream_t st);
void launch_finalize_energy(pswf_lr_plan* p, double* E, cudaStream_t st);
template <class T>
void launch_gather_ref(pswf_lr_plan* p, int n, const GridGeom<T>& g, T* phi, T* F, cudaStream_t st);

// fast fp32 path: per-atom weight records + output-stationary spread (kernels_stencil.cu),
// register-window gather (kernels_gather.cu)
bool stencil_path_supported(const pswf_lr_plan* p);
int stencil_rec_floats(int C);
size_t stencil_record_bytes(const pswf_lr_plan* p);
size_t stencil_drecord_bytes(const pswf_lr_plan* p);
size_t gather_grid_bytes(const pswf_lr_plan* p);
void launch_fast_gather(pswf_lr_plan* p, int n, float* phi, float* F, bool grid_is_interleaved, cudaStream_t st);
void launch_scatter_records(pswf_lr_plan* p, int n, const float* pos, const float* q, const GridGeom<float>& g,
                            cudaStream_t st);
void launch_stencil_spread(pswf_lr_plan* p, int n, cudaStream_t st);

// band-limited transform path (kernels_fft.cu)
bool fused_fft_supported(const pswf_lr_plan* p);
void fused_fft_limits(const pswf_lr_plan* p, int kmax[3]);
void launch_xy_scale(pswf_lr_plan* p, const ScaleParams<float>& P, double* E, cudaStream_t st);   // E (device, may be NULL): total energy
bool fused_z_supported(const pswf_lr_plan* p);   // own z transforms (power-of-two Mz); else cuFFT along z
void launch_z_forward(pswf_lr_plan* p, cudaStream_t st);
void launch_z_inverse(pswf_lr_plan* p, cudaStream_t st);
void launch_z_inverse_interleaved(pswf_lr_plan* p, cudaStream_t st);   // writes p->d_gridi (fast gather layout)

// real-space complement + self term (kernels_real.cu); uses the sort left by launch_bin_sort(scatter = true)
template <class T>
void launch_real_space(pswf_lr_plan* p, int n, const T* pos, const RealGeom<T>& g, const RealParams<T>& P, double* E,
                       T* phi, T* F, int accumulate, cudaStream_t st);

}  // namespace pswf
