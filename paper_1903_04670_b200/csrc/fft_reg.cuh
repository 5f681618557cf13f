// fft_reg.cuh -- fully unrolled complex FFTs of length N | 96 held in one thread's registers.
//
// Used for every 1-D pass of the 3-D transforms of Algorithm 2.  Convention
// (reading C-3): DIR = -1 is the forward transform with kernel e^{-2 pi i jk/N}, DIR = +1 the
// inverse kernel e^{+2 pi i jk/N}; both UNNORMALISED (the 1/N^3 factors are folded into the tables).
//
// Decimation in time, radix 4 / 2 / 3 chosen at compile time; all indices are compile-time constants
// after unrolling, so arrays live in registers and twiddles become literal operands.  Radix-2 and radix-4
// butterflies are in multiply-add form (twiddle_pm): 24 instead of 28 FP64 instructions per general radix-4
// butterfly, 392 instead of 432 per 32-point transform.
// Every routine is a template on the complex type (double2, or float2 for dgfs_params::precision = 1); the twiddles
// are the same correctly rounded double constants, converted at compile time.
#pragma once
#include <cuda_runtime.h>
#include "twiddle96.h"

namespace dgfs {

typedef double2 cplx;

typedef float2 cplxf;
template <class C> struct real_of;
template <> struct real_of<double2> { typedef double type; };
template <> struct real_of<float2> { typedef float type; };
template <class C> __host__ __device__ __forceinline__ C mkc(typename real_of<C>::type x, typename real_of<C>::type y) { C c; c.x = x; c.y = y; return c; }
__host__ __device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__host__ __device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

template <class C> __host__ __device__ __forceinline__ C cmul(C a, C b) {
  return mkc<C>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <class C> __host__ __device__ __forceinline__ C cadd(C a, C b) { return mkc<C>(a.x + b.x, a.y + b.y); }
template <class C> __host__ __device__ __forceinline__ C csub(C a, C b) { return mkc<C>(a.x - b.x, a.y - b.y); }
// a + b * c
template <class C> __host__ __device__ __forceinline__ C cfma(C b, C c, C a) {
  return mkc<C>(fma_(b.x, c.x, fma_(-b.y, c.y, a.x)), fma_(b.x, c.y, fma_(b.y, c.x, a.y)));
}

// cos / sin of 2 pi k / 96 for any integer k, from the quarter-wave table (exact symmetries).
__host__ __device__ constexpr double cos96(int k) {
  k = ((k % 96) + 96) % 96;
  if (k > 48) k = 96 - k;                    // cos(2pi - x) = cos x
  return (k <= 24) ? cos96_quarter(k) : -cos96_quarter(48 - k);
}
__host__ __device__ constexpr double sin96(int k) { return cos96(k - 24); }

// x * e^{DIR * 2 pi i k / N}, k known at compile time after unrolling; trivial cases cost nothing.
template <int N, int DIR, class C>
__host__ __device__ __forceinline__ C twiddle_mul(C x, int k) {
  typedef typename real_of<C>::type R;
  static_assert(96 % N == 0, "N must divide 96");
  const int k96 = ((k * (96 / N)) % 96 + 96) % 96;
  if (k96 == 0) return x;
  if (k96 == 48) return mkc<C>(-x.x, -x.y);
  if (k96 == 24) return (DIR > 0) ? mkc<C>(-x.y, x.x) : mkc<C>(x.y, -x.x);   // * (+-i)
  if (k96 == 72) return (DIR > 0) ? mkc<C>(x.y, -x.x) : mkc<C>(-x.y, x.x);   // * (-+i)
  const R c = (R)cos96(k96);
  const R s = (R)((DIR > 0) ? sin96(k96) : -sin96(k96));
  if (k96 % 24 == 12) {                      // |c| == |s| == sqrt(1/2): 2 add + 2 mul
    const R h = (R)0.70710678118654752440;
    const R sc = (c > 0) ? (R)1 : (R)-1, ss = (s > 0) ? (R)1 : (R)-1;
    // (x + iy)(sc + i ss) h = h[(sc x - ss y) + i(ss x + sc y)]
    return mkc<C>(h * (sc * x.x - ss * x.y), h * (ss * x.x + sc * x.y));
  }
  return mkc<C>(x.x * c - x.y * s, x.x * s + x.y * c);
}

// p = a + w x, m = a - w x with w = e^{DIR * 2 pi i k / N}, k known at compile time.  The product is never formed:
// with t = Im w / Re w (or its inverse when |Re w| < |Im w|, so that |t| <= 1),
//   w x = Re w * (x.re - t x.im, x.im + t x.re),
// which takes two FMAs, and each of the four outputs one more: 6 instructions instead of 4 (product) + 4 (sums).
template <int N, int DIR, class C>
__host__ __device__ __forceinline__ void twiddle_pm(C a, C x, int k, C& p, C& m) {
  typedef typename real_of<C>::type R;
  static_assert(96 % N == 0, "N must divide 96");
  const int k96 = ((k * (96 / N)) % 96 + 96) % 96;
  if (k96 == 0) { p = cadd(a, x); m = csub(a, x); return; }
  if (k96 == 48) { p = csub(a, x); m = cadd(a, x); return; }
  if (k96 == 24 || k96 == 72) {                          // w = +-i
    const bool plus = (k96 == 24) == (DIR > 0);          // w = +i
    const C u = mkc<C>(a.x - x.y, a.y + x.x), v = mkc<C>(a.x + x.y, a.y - x.x);
    p = plus ? u : v;
    m = plus ? v : u;
    return;
  }
  const double cd = cos96(k96);
  const double sd = (DIR > 0) ? sin96(k96) : -sin96(k96);
  const bool big_c = (cd < 0 ? -cd : cd) >= (sd < 0 ? -sd : sd);
  if (big_c) {
    const R t = (R)(sd / cd), c = (R)cd;
    const C xt = mkc<C>(fma_(-t, x.y, x.x), fma_(t, x.x, x.y));
    p = mkc<C>(fma_(c, xt.x, a.x), fma_(c, xt.y, a.y));
    m = mkc<C>(fma_(-c, xt.x, a.x), fma_(-c, xt.y, a.y));
  } else {
    const R t = (R)(cd / sd), s = (R)sd;
    const C xt = mkc<C>(fma_(t, x.x, -x.y), fma_(t, x.y, x.x));
    p = mkc<C>(fma_(s, xt.x, a.x), fma_(s, xt.y, a.y));
    m = mkc<C>(fma_(-s, xt.x, a.x), fma_(-s, xt.y, a.y));
  }
}

// out[0..N) = DFT_N of in[0], in[IS], ..., in[(N-1) IS]
template <int N, int DIR, int IS>
struct RegFFT {
  static constexpr int R = (N % 4 == 0) ? 4 : ((N % 2 == 0) ? 2 : 3);
  static constexpr int M = N / R;
  static_assert(N % R == 0, "unsupported length");
  template <class C>
  __host__ __device__ static __forceinline__ void run(const C* __restrict__ in, C* __restrict__ out) {
    typedef typename real_of<C>::type T;
    C t[R][M];
#pragma unroll
    for (int j = 0; j < R; ++j) RegFFT<M, DIR, IS * R>::run(in + j * IS, t[j]);
#pragma unroll
    for (int k = 0; k < M; ++k) {
      if (R == 2) {
        twiddle_pm<N, DIR>(t[0][k], t[1][k], k, out[k], out[k + M]);
      } else if (R == 4) {
        // w^{3k} d = w^k (w^{2k} d): both pairs take the twiddle w^{2k} first, then w^k (and w^k times DIR * i,
        // i.e. w^{k + N/4}, for the odd outputs); every product is folded into the sums (twiddle_pm)
        C ac0, ac1, e0, e1;
        twiddle_pm<N, DIR>(t[0][k], t[2][k], 2 * k, ac0, ac1);         // a +- w^{2k} c
        twiddle_pm<N, DIR>(t[1][k], t[3][k], 2 * k, e0, e1);           // b +- w^{2k} d
        twiddle_pm<N, DIR>(ac0, e0, k, out[k], out[k + 2 * M]);
        twiddle_pm<N, DIR>(ac1, e1, k + N / 4, out[k + M], out[k + 3 * M]);
      } else {  // R == 3
        C a = t[0][k];
        C b = twiddle_mul<N, DIR>(t[1][k], k);
        C c = twiddle_mul<N, DIR>(t[2][k], 2 * k);
        const T s3 = (T)((DIR > 0) ? 0.86602540378443864676 : -0.86602540378443864676);
        C bc = cadd(b, c), d = csub(b, c);
        C m = mkc<C>(fma_((T)-0.5, bc.x, a.x), fma_((T)-0.5, bc.y, a.y));
        out[k] = cadd(a, bc);
        // w = e^{DIR 2 pi i/3} = -1/2 + i s3:  X1 = a + w b + conj(w) c = m + i s3 (b - c)
        out[k + M] = mkc<C>(fma_(-s3, d.y, m.x), fma_(s3, d.x, m.y));
        out[k + 2 * M] = mkc<C>(fma_(s3, d.y, m.x), fma_(-s3, d.x, m.y));
      }
    }
  }
};
template <int DIR, int IS>
struct RegFFT<1, DIR, IS> {
  template <class C>
  __host__ __device__ static __forceinline__ void run(const C* __restrict__ in, C* __restrict__ out) {
    out[0] = in[0];
  }
};

// In-place convenience wrapper: x[0..N) -> DFT_N(x), natural order in and out.
template <int N, int DIR, class C>
__host__ __device__ __forceinline__ void fft_reg(C (&x)[N]) {
  C y[N];
  RegFFT<N, DIR, 1>::run(x, y);
#pragma unroll
  for (int i = 0; i < N; ++i) x[i] = y[i];
}

}  // namespace dgfs
