// peak.cu - register-only FP64 issue-rate loops: the denominator of "% of FP64 peak".
// Not part of the method.  afqmc_measure_fp64_peak (include/afqmc.h).
#include <cuda_runtime.h>

#include "../../include/afqmc.h"
#include "dmma.cuh"

namespace {

constexpr int kIters = 4096;

__global__ void __launch_bounds__(256) dmma_loop(double* out, int reps, long long* cyc) {
  double c[16][2];
#pragma unroll
  for (int i = 0; i < 16; ++i) { c[i][0] = threadIdx.x * 1e-9; c[i][1] = i * 1e-9; }
  double a = 1.0 + threadIdx.x * 1e-12, b = 1.0 - threadIdx.x * 1e-12;
  long long t0 = clock64();
  for (int r = 0; r < reps; ++r)
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
      for (int i = 0; i < 16; ++i) afq::dmma884(c[i][0], c[i][1], a, b);
    }
  long long t1 = clock64();
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) cyc[0] = t1 - t0;
}

__global__ void __launch_bounds__(256) dfma_loop(double* out, int reps, long long* cyc) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = threadIdx.x * 1e-9 + i;
  double a = 1.0 + threadIdx.x * 1e-12, b = 1e-9;
  long long t0 = clock64();
  for (int r = 0; r < reps; ++r)
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
      for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
    }
  long long t1 = clock64();
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 12345.678) out[0] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) cyc[0] = t1 - t0;
}

}  // namespace

extern "C" int32_t afqmc_measure_fp64_peak(double ms, double* out3) {
  if (!out3) return AFQMC_ERR_INVALID;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return AFQMC_ERR_CUDA;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  double* d = nullptr;
  long long* cyc = nullptr;
  if (cudaMalloc(&d, 64) != cudaSuccess || cudaMalloc(&cyc, 16) != cudaSuccess) return AFQMC_ERR_ALLOC;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int ctas = sms * 2;  // 2 CTAs x 8 warps per SM = 4 warps per SM sub-partition
  for (int which = 0; which < 2; ++which) {
    int reps = 1;
    float el = 0.f;
    long long hc = 0;
    for (int pass = 0; pass < 3; ++pass) {   // calibrate, then the timed run
      cudaEventRecord(e0);
      if (which == 0) dmma_loop<<<ctas, 256>>>(d, reps, cyc); else dfma_loop<<<ctas, 256>>>(d, reps, cyc);
      cudaEventRecord(e1);
      if (cudaEventSynchronize(e1) != cudaSuccess) return AFQMC_ERR_CUDA;
      cudaEventElapsedTime(&el, e0, e1);
      if (pass < 2) {
        double want = (pass == 0 ? 20.0 : ms);
        reps = (int)(reps * want / (el > 1e-3 ? el : 1e-3)) + 1;
      }
    }
    cudaMemcpy(&hc, cyc, 8, cudaMemcpyDeviceToHost);
    const double per_thread = (double)reps * kIters * 16;
    const double flops = which == 0 ? per_thread * (ctas * 8.0) * 512.0          // 8x8x4 MACs x 2 per warp
                                    : per_thread * (ctas * 256.0) * 2.0;
    out3[which] = flops / (el * 1e-3) / 1e12;
    if (which == 0) out3[2] = (double)hc / (el * 1e-3) / 1e6;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  cudaFree(cyc);
  return AFQMC_OK;
}
