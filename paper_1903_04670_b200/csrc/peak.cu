// peak.cu -- dgfs_measure_fp64_peak: the denominator of the roofline line.
//
// MEASURED_PEAKS.json carries HBM and bf16 numbers only, and the collision operator is bound by the
// plain FP64 pipe (an FFT is not a dense contraction), so the library measures that pipe itself:
// every thread runs 8 independent DFMA chains (no memory traffic), 4 CTAs of 256 threads per SM.
#include <cuda_runtime.h>
#include "../../include/dgfs.h"

namespace {
__global__ void __launch_bounds__(256) k_dfma_chains(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 123.456) out[0] = s;     // never true: keeps the chains alive
}
}  // namespace

extern "C" int dgfs_measure_fp64_peak(int device, double seconds, double* tflops_burst, double* tflops_sustained) {
  if (seconds <= 0 || seconds > 30) return DGFS_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return DGFS_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return DGFS_ECUDA;
  double* d = nullptr;
  if (cudaMalloc(&d, 8) != cudaSuccess) return DGFS_ENOMEM;
  const int blocks = prop.multiProcessorCount * 4, iters = 4096;
  const double flops = 2.0 * 8 * 16 * (double)iters * 256.0 * blocks;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  k_dfma_chains<<<blocks, 256>>>(d, iters, 0.999999, 1e-9);     // warm-up
  cudaDeviceSynchronize();
  double best = 0, total_ms = 0, total_fl = 0;
  while (total_ms < seconds * 1e3) {
    cudaEventRecord(e0);
    k_dfma_chains<<<blocks, 256>>>(d, iters, 0.999999, 1e-9);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return DGFS_ECUDA; }
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    double tf = flops / (ms * 1e-3) / 1e12;
    if (tf > best) best = tf;
    total_ms += ms; total_fl += flops;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (tflops_burst) *tflops_burst = best;
  if (tflops_sustained) *tflops_sustained = total_fl / (total_ms * 1e-3) / 1e12;
  return DGFS_OK;
}
