// Roofline denominator for the per-cell contraction: the FP64 rate of this GPU measured with register-resident
// loops of mma.sync.m8n8k4.f64 (DMMA, the tensor pipe the contraction kernel uses) and of plain DFMA.
// MEASURED_PEAKS.json carries only HBM and bf16 figures, so the FP64 peak is measured by the library itself
// (chfsi_measure_fp64_peak, include/chfsi.h); bench.py calls it in the same run it reports against.
#include <cuda_runtime.h>

#include "../../include/chfsi.h"

namespace {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

constexpr int kAcc = 16;

__global__ void __launch_bounds__(512) k_peak_dmma(double* out, int iters, double a0, double b0) {
  double acc[kAcc][2];
#pragma unroll
  for (int i = 0; i < kAcc; ++i) acc[i][0] = acc[i][1] = 0.0;
  const double a = a0 + threadIdx.x, b = b0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < kAcc; ++i) dmma884(acc[i][0], acc[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kAcc; ++i) s += acc[i][0] + acc[i][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(512) k_peak_dfma(double* out, int iters, double a0, double b0) {
  double acc[kAcc];
#pragma unroll
  for (int i = 0; i < kAcc; ++i) acc[i] = i;
  const double a = a0, b = b0 + threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < kAcc; ++i) acc[i] = fma(acc[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kAcc; ++i) s += acc[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" int chfsi_measure_fp64_peak(double* dmma_tflops, double* dfma_tflops, void* cuda_stream) {
  if (!dmma_tflops || !dfma_tflops) return CHFSI_ERR_BAD_ARGUMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return CHFSI_ERR_CUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return CHFSI_ERR_CUDA;
  const int threads = 512, grid = sms * 2, iters = 8192;
  double* out = nullptr;
  if (cudaMalloc((void**)&out, (size_t)grid * threads * sizeof(double)) != cudaSuccess) return CHFSI_ERR_OUT_OF_MEMORY;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
    if (e0) cudaEventDestroy(e0);
    cudaFree(out);
    return CHFSI_ERR_CUDA;
  }
  double best[2] = {0.0, 0.0};
  for (int which = 0; which < 2; ++which) {
    for (int rep = 0; rep < 6; ++rep) {   // rep 0 is the warm-up
      cudaEventRecord(e0, st);
      if (which == 0) k_peak_dmma<<<grid, threads, 0, st>>>(out, iters, 1.0, 1e-3);
      else k_peak_dfma<<<grid, threads, 0, st>>>(out, iters * 8, 1.0000001, 1e-3);
      cudaEventRecord(e1, st);
      if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out); return CHFSI_ERR_CUDA; }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      const double flops = which == 0 ? (double)grid * (threads / 32) * iters * kAcc * 512.0
                                      : (double)grid * threads * (double)iters * 8 * kAcc * 2.0;
      const double tf = flops / (ms * 1e-3) * 1e-12;
      if (rep > 0 && tf > best[which]) best[which] = tf;
    }
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  *dmma_tflops = best[0]; *dfma_tflops = best[1];
  return cudaGetLastError() == cudaSuccess ? CHFSI_OK : CHFSI_ERR_CUDA;
}
