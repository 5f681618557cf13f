// fft_reg.cuh -- fully unrolled complex FFTs of length N | 96 held in one thread's registers.
//
// Used for every 1-D pass of the 3-D transforms of Algorithm 2.  Convention
// (reading C-3): DIR = -1 is the forward transform with kernel e^{-2 pi i jk/N}, DIR = +1 the
// inverse kernel e^{+2 pi i jk/N}; both UNNORMALISED (the 1/N^3 factors are folded into the tables).
//
// Decimation in time, radix 4 / 2 / 3 chosen at compile time; all indices are compile-time constants
// after unrolling, so arrays live in registers and twiddles become literal operands.
#pragma once
#include <cuda_runtime.h>
#include "twiddle96.h"

namespace dgfs {

typedef double2 cplx;

__host__ __device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__host__ __device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
// a + b * c
__host__ __device__ __forceinline__ cplx cfma(cplx b, cplx c, cplx a) {
  return make_double2(fma(b.x, c.x, fma(-b.y, c.y, a.x)), fma(b.x, c.y, fma(b.y, c.x, a.y)));
}

// cos / sin of 2 pi k / 96 for any integer k, from the quarter-wave table (exact symmetries).
__host__ __device__ constexpr double cos96(int k) {
  k = ((k % 96) + 96) % 96;
  if (k > 48) k = 96 - k;                    // cos(2pi - x) = cos x
  return (k <= 24) ? cos96_quarter(k) : -cos96_quarter(48 - k);
}
__host__ __device__ constexpr double sin96(int k) { return cos96(k - 24); }

// x * e^{DIR * 2 pi i k / N}, k known at compile time after unrolling; trivial cases cost nothing.
template <int N, int DIR>
__host__ __device__ __forceinline__ cplx twiddle_mul(cplx x, int k) {
  static_assert(96 % N == 0, "N must divide 96");
  const int k96 = ((k * (96 / N)) % 96 + 96) % 96;
  if (k96 == 0) return x;
  if (k96 == 48) return make_double2(-x.x, -x.y);
  if (k96 == 24) return (DIR > 0) ? make_double2(-x.y, x.x) : make_double2(x.y, -x.x);   // * (+-i)
  if (k96 == 72) return (DIR > 0) ? make_double2(x.y, -x.x) : make_double2(-x.y, x.x);   // * (-+i)
  const double c = cos96(k96);
  const double s = (DIR > 0) ? sin96(k96) : -sin96(k96);
  if (k96 % 24 == 12) {                      // |c| == |s| == sqrt(1/2): 2 add + 2 mul
    const double h = 0.70710678118654752440;
    const double sc = (c > 0) ? 1.0 : -1.0, ss = (s > 0) ? 1.0 : -1.0;
    // (x + iy)(sc + i ss) h = h[(sc x - ss y) + i(ss x + sc y)]
    return make_double2(h * (sc * x.x - ss * x.y), h * (ss * x.x + sc * x.y));
  }
  return make_double2(x.x * c - x.y * s, x.x * s + x.y * c);
}

// out[0..N) = DFT_N of in[0], in[IS], ..., in[(N-1) IS]
template <int N, int DIR, int IS>
struct RegFFT {
  static constexpr int R = (N % 4 == 0) ? 4 : ((N % 2 == 0) ? 2 : 3);
  static constexpr int M = N / R;
  static_assert(N % R == 0, "unsupported length");
  __host__ __device__ static __forceinline__ void run(const cplx* __restrict__ in, cplx* __restrict__ out) {
    cplx t[R][M];
#pragma unroll
    for (int j = 0; j < R; ++j) RegFFT<M, DIR, IS * R>::run(in + j * IS, t[j]);
#pragma unroll
    for (int k = 0; k < M; ++k) {
      if (R == 2) {
        cplx a = t[0][k], b = twiddle_mul<N, DIR>(t[1][k], k);
        out[k] = cadd(a, b);
        out[k + M] = csub(a, b);
      } else if (R == 4) {
        cplx a = t[0][k];
        cplx b = twiddle_mul<N, DIR>(t[1][k], k);
        cplx c = twiddle_mul<N, DIR>(t[2][k], 2 * k);
        cplx d = twiddle_mul<N, DIR>(t[3][k], 3 * k);
        cplx ac0 = cadd(a, c), ac1 = csub(a, c), bd0 = cadd(b, d), bd1 = csub(b, d);
        // multiply bd1 by DIR * i
        cplx ibd1 = (DIR > 0) ? make_double2(-bd1.y, bd1.x) : make_double2(bd1.y, -bd1.x);
        out[k] = cadd(ac0, bd0);
        out[k + M] = cadd(ac1, ibd1);
        out[k + 2 * M] = csub(ac0, bd0);
        out[k + 3 * M] = csub(ac1, ibd1);
      } else {  // R == 3
        cplx a = t[0][k];
        cplx b = twiddle_mul<N, DIR>(t[1][k], k);
        cplx c = twiddle_mul<N, DIR>(t[2][k], 2 * k);
        const double s3 = (DIR > 0) ? 0.86602540378443864676 : -0.86602540378443864676;
        cplx bc = cadd(b, c), d = csub(b, c);
        cplx m = make_double2(fma(-0.5, bc.x, a.x), fma(-0.5, bc.y, a.y));
        out[k] = cadd(a, bc);
        // w = e^{DIR 2 pi i/3} = -1/2 + i s3:  X1 = a + w b + conj(w) c = m + i s3 (b - c)
        out[k + M] = make_double2(fma(-s3, d.y, m.x), fma(s3, d.x, m.y));
        out[k + 2 * M] = make_double2(fma(s3, d.y, m.x), fma(-s3, d.x, m.y));
      }
    }
  }
};
template <int DIR, int IS>
struct RegFFT<1, DIR, IS> {
  __host__ __device__ static __forceinline__ void run(const cplx* __restrict__ in, cplx* __restrict__ out) {
    out[0] = in[0];
  }
};

// In-place convenience wrapper: x[0..N) -> DFT_N(x), natural order in and out.
template <int N, int DIR>
__host__ __device__ __forceinline__ void fft_reg(cplx (&x)[N]) {
  cplx y[N];
  RegFFT<N, DIR, 1>::run(x, y);
#pragma unroll
  for (int i = 0; i < N; ++i) x[i] = y[i];
}

}  // namespace dgfs
