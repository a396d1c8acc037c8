// Stand-alone microbenchmarks behind two design decisions of the stencil kernels:
//   1. the FP32 peak the "alu" roofline uses: FFMA and packed FFMA2 issue rates per SM;
//   2. why the spread is output-stationary in REGISTERS instead of accumulating in shared-memory tiles:
//      atomicAdd(float) on shared memory compiles to a compare-and-swap loop (SASS ATOMS.CAST.SPIN), and
//      even a conflict-free, non-atomic read-modify-write of shared memory moves 8 bytes per FMA.
// Not part of libpswf_lr.so.  Build and run on a B200:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/microbench_peaks \
//        paper_2606_06617_b200/csrc/microbench_peaks.cu && /tmp/microbench_peaks
//   cuobjdump -sass /tmp/microbench_peaks | grep -E "ATOMS|FFMA2" | sort | uniq -c
#include <cstdio>
#include <cuda_runtime.h>

typedef unsigned long long f32x2;

__global__ void k_ffma(float* out, float a, float b, int iters) {
  float v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = threadIdx.x * 1e-3f + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = fmaf(v[i], a, b);
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += v[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_ffma2(float* out, float a, float b, int iters) {
  f32x2 v[16], A, B;
  asm("mov.b64 %0, {%1, %1};" : "=l"(A) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(B) : "f"(b));
#pragma unroll
  for (int i = 0; i < 16; ++i) asm("mov.b64 %0, {%1, %2};" : "=l"(v[i]) : "f"(threadIdx.x * 1e-3f + i), "f"(1.f * i));
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v[i]) : "l"(A), "l"(B));
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v[i]));
    s += lo + hi;
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// every thread adds into its own word of a 32 KB shared tile (no two lanes share a bank or an address)
__global__ void k_smem_atomic(float* out, int iters) {
  __shared__ float tile[8192];
  for (int i = threadIdx.x; i < 8192; i += blockDim.x) tile[i] = 0.f;
  __syncthreads();
  float w = 1.0f + threadIdx.x * 1e-6f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) atomicAdd(&tile[(threadIdx.x + 1024 * k) & 8191], w);
  }
  __syncthreads();
  out[blockIdx.x * blockDim.x + threadIdx.x] = tile[threadIdx.x];
}

__global__ void k_smem_rmw(float* out, int iters) {
  __shared__ float tile[8192];
  for (int i = threadIdx.x; i < 8192; i += blockDim.x) tile[i] = 0.f;
  __syncthreads();
  float w = 1.0f + threadIdx.x * 1e-6f;
  volatile float* t = tile;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int idx = (threadIdx.x + 1024 * k) & 8191;
      t[idx] = fmaf(w, 1.0001f, t[idx]);
    }
  }
  __syncthreads();
  out[blockIdx.x * blockDim.x + threadIdx.x] = tile[threadIdx.x];
}

template <class F>
float time_ms(F launch) {
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  launch();
  cudaDeviceSynchronize();
  cudaEventRecord(a);
  launch();
  cudaEventRecord(b);
  cudaEventSynchronize(b);
  float ms = 0;
  cudaEventElapsedTime(&ms, a, b);
  return ms;
}

int main() {
  cudaDeviceProp pr;
  cudaGetDeviceProperties(&pr, 0);
  const int sms = pr.multiProcessorCount;
  int khz = 0;
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
  const double clk = khz * 1e3;
  printf("device %s, %d SMs, max SM clock %.0f MHz\n", pr.name, sms, clk / 1e6);
  float* out;
  cudaMalloc(&out, sizeof(float) * sms * 8 * 1024);
  const int iters = 4096, blocks = sms * 8, threads = 1024 / 4;   // 8 CTAs of 256 threads per SM: 64 warps
  {
    float ms = time_ms([&] { k_ffma<<<blocks, threads>>>(out, 1.0001f, 0.5f, iters); });
    double fma = (double)blocks * threads * 16.0 * iters;
    printf("FFMA : %.2f TFLOP/s  = %.1f FMA/clk/SM at max clock\n", 2 * fma / ms / 1e9, fma / (ms * 1e-3) / sms / clk);
  }
  {
    float ms = time_ms([&] { k_ffma2<<<blocks, threads>>>(out, 1.0001f, 0.5f, iters); });
    double fma = (double)blocks * threads * 32.0 * iters;
    printf("FFMA2: %.2f TFLOP/s  = %.1f FMA/clk/SM at max clock (two FMAs per lane per instruction)\n",
           2 * fma / ms / 1e9, fma / (ms * 1e-3) / sms / clk);
  }
  {
    const int it2 = 512;
    float ms = time_ms([&] { k_smem_atomic<<<sms, 1024>>>(out, it2); });
    double ops = (double)sms * 1024 * 8.0 * it2;
    printf("shared atomicAdd(float), conflict-free: %.1f G adds/s = %.2f adds/clk/SM\n", ops / ms / 1e6,
           ops / (ms * 1e-3) / sms / clk);
    ms = time_ms([&] { k_smem_rmw<<<sms, 1024>>>(out, it2); });
    printf("shared LDS + FFMA + STS (no atomicity), conflict-free: %.1f G adds/s = %.2f adds/clk/SM\n", ops / ms / 1e6,
           ops / (ms * 1e-3) / sms / clk);
    printf("for comparison, the register-accumulating spread needs 128 FMA/clk/SM to reach the FP32 peak\n");
  }
  cudaFree(out);
  return 0;
}
