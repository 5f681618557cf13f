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

// ------------------------------------------------------------------------------------------------------------------
// dgfs_measure_dft: the two ways BASELINE.json's north_star names for the small 1-D transforms, timed on chip (no
// global traffic inside the timed loop), so that the choice between them is a measurement:
//   method 0: the register FFT of fft_reg.cuh, one transform per thread (what every pass of the pipeline uses);
//   method 1: the same DFT as a dense contraction on the FP64 tensor path, mma.sync.m8n8k4.f64 (tcgen05 has no FP64
//             type): [Yr; Yi] = [Wr -Wi; Wi Wr] [Xr; Xi], a (2N x 2N) x (2N x 8) product per warp = 8 transforms,
//             (2N/8)(2N/4) MMAs; W fragments in registers (N <= 16) or read from shared memory per MMA (conflict-free
//             pitch), X fragments and accumulators in registers.
#include <cmath>
#include <vector>
#include "fft_reg.cuh"

namespace {
using dgfs::cplx;

template <int N>
__global__ void __launch_bounds__(128) k_dft_fft(cplx* out, int reps, int write) {
  cplx x[N];
  const int gid = blockIdx.x * blockDim.x + threadIdx.x;
#pragma unroll
  for (int i = 0; i < N; ++i) x[i] = make_double2(cos(0.37 * i + 0.01 * (gid % 97)), sin(0.11 * i * i + 0.02 * (gid % 89)));
  if (write) {                                  // one forward transform, written out for the self-check
    dgfs::fft_reg<N, -1>(x);
    if (gid == 0) for (int i = 0; i < N; ++i) out[i] = x[i];
    return;
  }
  for (int r = 0; r < reps; ++r) {              // forward, inverse, 1/N: two transforms per iteration
    dgfs::fft_reg<N, -1>(x);
    dgfs::fft_reg<N, +1>(x);
#pragma unroll
    for (int i = 0; i < N; ++i) { x[i].x *= 1.0 / N; x[i].y *= 1.0 / N; }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) s += x[i].x + x[i].y;
  if (s == 123.456) out[0] = make_double2(s, s);
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// One warp = 8 transforms (the 8 columns of the B operand).  wreal: [2N][2N] real form of the forward DFT matrix.
template <int N, bool AREG>
__global__ void __launch_bounds__(128) k_dft_mma(const double* __restrict__ wreal, cplx* out, int reps, int write) {
  constexpr int D = 2 * N, MT = D / 8, KT = D / 4, PITCH = D + 2;
  extern __shared__ double sw[];                // [D][PITCH]
  for (int i = threadIdx.x; i < D * D; i += blockDim.x) sw[(i / D) * PITCH + i % D] = wreal[i];
  __syncthreads();
  const int lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int arow = lane >> 2, acol = lane & 3;  // A: row = lane / 4, col = lane % 4;  B: row = lane % 4, col = lane / 4
  double b[KT];                                 // X fragments: row kt * 4 + lane % 4 of [Xr; Xi], transform lane / 4
#pragma unroll
  for (int kt = 0; kt < KT; ++kt) {
    const int row = kt * 4 + acol, i = row % N, tr = (gw * 8 + arow) % 97, tq = (gw * 8 + arow) % 89;
    b[kt] = row < N ? cos(0.37 * i + 0.01 * tr) : sin(0.11 * i * i + 0.02 * tq);
  }
  double areg[AREG ? MT * KT : 1];
  if (AREG) {
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int kt = 0; kt < KT; ++kt) areg[AREG ? mt * KT + kt : 0] = sw[(mt * 8 + arow) * PITCH + kt * 4 + acol];
  }
  double c[MT][2];
#pragma unroll
  for (int mt = 0; mt < MT; ++mt) c[mt][0] = c[mt][1] = 0.0;
  const int nrep = write ? 1 : reps;
  for (int r = 0; r < nrep; ++r) {
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int kt = 0; kt < KT; ++kt) {
        const double a = AREG ? areg[AREG ? mt * KT + kt : 0] : sw[(mt * 8 + arow) * PITCH + kt * 4 + acol];
        dmma884(c[mt][0], c[mt][1], a, b[kt]);
      }
  }
  if (write) {                                  // C: row = lane / 4, columns 2 (lane % 4) and + 1; transform 0 = column 0
    if (gw == 0 && acol == 0)
      for (int mt = 0; mt < MT; ++mt) {
        const int row = mt * 8 + arow;          // row of [Yr; Yi]
        if (row < N) out[row].x = c[mt][0]; else out[row - N].y = c[mt][0];
      }
    return;
  }
  double s = 0;
#pragma unroll
  for (int mt = 0; mt < MT; ++mt) s += c[mt][0] + c[mt][1];
  if (s == 123.456) out[0] = make_double2(s, s);
}

template <int N>
int measure_dft(int method, double seconds, double* dfts_per_s, double* max_err, int nsm) {
  constexpr int D = 2 * N;
  cplx* d_out = nullptr;
  double* d_w = nullptr;
  if (cudaMalloc(&d_out, sizeof(cplx) * N) != cudaSuccess) return DGFS_ENOMEM;
  std::vector<double> w((size_t)D * D);
  const double pi = 3.14159265358979323846;
  for (int k = 0; k < N; ++k)
    for (int j = 0; j < N; ++j) {
      const int kj = (k * j) % N;                       // forward kernel e^{-2 pi i kj / N}
      const double wr = cos(2 * pi * kj / N), wi = -sin(2 * pi * kj / N);
      w[(size_t)k * D + j] = wr; w[(size_t)k * D + N + j] = -wi;
      w[(size_t)(N + k) * D + j] = wi; w[(size_t)(N + k) * D + N + j] = wr;
    }
  if (cudaMalloc(&d_w, sizeof(double) * D * D) != cudaSuccess) { cudaFree(d_out); return DGFS_ENOMEM; }
  cudaMemcpy(d_w, w.data(), sizeof(double) * D * D, cudaMemcpyHostToDevice);
  constexpr bool AREG = N <= 16;
  const size_t smem = sizeof(double) * D * (D + 2);
  cudaFuncSetAttribute(k_dft_mma<N, AREG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  const int threads = 128;
  int bps = 0;
  if (method == 0) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_dft_fft<N>, threads, 0);
  else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_dft_mma<N, AREG>, threads, smem);
  if (bps < 1) bps = 1;
  const int blocks = nsm * bps;
  auto launch = [&](int reps, int write) {
    if (method == 0) k_dft_fft<N><<<write ? 1 : blocks, threads>>>(d_out, reps, write);
    else k_dft_mma<N, AREG><<<write ? 1 : blocks, threads, smem>>>(d_w, d_out, reps, write);
  };
  // self-check: transform 0 against the direct sum on the host
  launch(1, 1);
  std::vector<cplx> got(N);
  if (cudaMemcpy(got.data(), d_out, sizeof(cplx) * N, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaFree(d_out); cudaFree(d_w); return DGFS_ECUDA; }
  double err = 0, mx = 0;
  for (int k = 0; k < N; ++k) {
    double re = 0, im = 0;
    for (int j = 0; j < N; ++j) {
      const double xr = cos(0.37 * j), xi = sin(0.11 * j * j);
      const int kj = (k * j) % N;
      const double wr = cos(2 * pi * kj / N), wi = -sin(2 * pi * kj / N);
      re += wr * xr - wi * xi; im += wr * xi + wi * xr;
    }
    err = fmax(err, fmax(fabs(re - got[k].x), fabs(im - got[k].y)));
    mx = fmax(mx, fmax(fabs(re), fabs(im)));
  }
  if (max_err) *max_err = err / mx;
  const int reps = 2000;
  const double per_launch = method == 0 ? 2.0 * reps * threads * (double)blocks : (double)reps * (threads / 32) * 8.0 * blocks;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  launch(reps, 0);
  cudaDeviceSynchronize();
  double total_ms = 0, total = 0;
  while (total_ms < seconds * 1e3) {
    cudaEventRecord(e0);
    launch(reps, 0);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d_out); cudaFree(d_w); return DGFS_ECUDA; }
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    total_ms += ms; total += per_launch;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out); cudaFree(d_w);
  if (dfts_per_s) *dfts_per_s = total / (total_ms * 1e-3);
  return DGFS_OK;
}
}  // namespace

extern "C" int dgfs_measure_dft(int device, int N, int method, double seconds, double* dfts_per_second, double* rel_err) {
  if (seconds <= 0 || seconds > 30 || (method != 0 && method != 1)) return DGFS_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return DGFS_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return DGFS_ECUDA;
  switch (N) {
    case 8: return measure_dft<8>(method, seconds, dfts_per_second, rel_err, prop.multiProcessorCount);
    case 16: return measure_dft<16>(method, seconds, dfts_per_second, rel_err, prop.multiProcessorCount);
    case 24: return measure_dft<24>(method, seconds, dfts_per_second, rel_err, prop.multiProcessorCount);
    case 32: return measure_dft<32>(method, seconds, dfts_per_second, rel_err, prop.multiProcessorCount);
    case 48: return measure_dft<48>(method, seconds, dfts_per_second, rel_err, prop.multiProcessorCount);
  }
  return DGFS_EINVAL;
}

// ------------------------------------------------------------------------------------------------------------------
// dgfs_measure_fp64_mix: do the plain FP64 pipe (DFMA) and the FP64 tensor path (mma.sync.m8n8k4.f64, SASS DMMA) run
// side by side, or is it one unit?  Every thread carries n_dfma independent DFMA chains and every warp n_dmma independent
// MMA chains in the same unrolled loop; no memory traffic.  If the two were separate pipes a mixed kernel would take the
// longer of the two pure times; on B200 the times ADD (profiles/r02_dft_probe.md): a plane job cannot hand part of its
// arithmetic to the tensor path to get past the DFMA rate.
namespace {
__device__ __forceinline__ void dmma_884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
template <int NF, int NM>
__global__ void __launch_bounds__(256) k_fp64_mix(double* out, int iters, double a, double b) {
  double x[8], c[8][2];
#pragma unroll
  for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x * 1e-3 + i; c[i][0] = i; c[i][1] = -i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
#pragma unroll
      for (int j = 0; j < NF; ++j) x[j] = fma(x[j], a, b);
#pragma unroll
      for (int j = 0; j < NM; ++j) dmma_884(c[j][0], c[j][1], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i] + c[i][0] + c[i][1];
  if (s == 123.456) out[0] = s;     // never true: keeps the chains alive
}
template <int NF, int NM>
int run_mix(int device, double seconds, double* tf_dfma, double* tf_dmma) {
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return DGFS_ECUDA;
  double* d = nullptr;
  if (cudaMalloc(&d, 8) != cudaSuccess) return DGFS_ENOMEM;
  const int blocks = prop.multiProcessorCount * 4, iters = 2000;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  k_fp64_mix<NF, NM><<<blocks, 256>>>(d, iters, 0.999999, 1e-9);
  cudaDeviceSynchronize();
  double best = 1e30, total = 0.0;
  while (total < seconds * 1e3) {
    cudaEventRecord(e0);
    k_fp64_mix<NF, NM><<<blocks, 256>>>(d, iters, 0.999999, 1e-9);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return DGFS_ECUDA; }
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
    total += ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  // thread-level DFMAs (2 flop) and warp-level m8n8k4 MMAs (512 flop) of the best launch
  const double nf = (double)NF * 8 * iters * 256.0 * blocks, nm = (double)NM * 8 * iters * 8.0 * blocks;
  if (tf_dfma) *tf_dfma = 2.0 * nf / (best * 1e-3) / 1e12;
  if (tf_dmma) *tf_dmma = 512.0 * nm / (best * 1e-3) / 1e12;
  return DGFS_OK;
}
}  // namespace

extern "C" int dgfs_measure_fp64_mix(int device, int n_dfma, int n_dmma, double seconds, double* tflops_dfma, double* tflops_dmma) {
  if (seconds <= 0 || seconds > 30) return DGFS_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return DGFS_ECUDA;
  if (n_dfma == 8 && n_dmma == 0) return run_mix<8, 0>(device, seconds, tflops_dfma, tflops_dmma);
  if (n_dfma == 0 && n_dmma == 8) return run_mix<0, 8>(device, seconds, tflops_dfma, tflops_dmma);
  if (n_dfma == 8 && n_dmma == 8) return run_mix<8, 8>(device, seconds, tflops_dfma, tflops_dmma);
  if (n_dfma == 8 && n_dmma == 2) return run_mix<8, 2>(device, seconds, tflops_dfma, tflops_dmma);
  if (n_dfma == 4 && n_dmma == 4) return run_mix<4, 4>(device, seconds, tflops_dfma, tflops_dmma);
  return DGFS_EINVAL;      // chains per thread / per warp: (8,0), (0,8), (8,8), (8,2), (4,4)
}

