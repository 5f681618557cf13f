// kernels_v0.cuh -- device code of the stage-per-kernel (v0) pipeline of Algorithm 2.
// Shared by collide.cu (v0 orchestration: VSS / table_mode-1 pairs, N = 48) and collide_v1.cu (which
// reuses the step-1 and step-10 kernels).  See collide.cu for the organisation.
#pragma once
#include "ctx.h"

namespace dgfs {

__device__ __forceinline__ int sfreq(int j, int N) { return j - (j >= N / 2 ? N : 0); }

// One warp transforms one N x N plane: pass 1 over the slow index (pencil per lane), transposition
// through `buf` (row pitch N+1: conflict-free for 16-byte accesses), pass 2 over the other index.
//   ld(i, a)      : input element i of pencil a (pass 1)
//   mid(x, j)     : optional factor applied to element j on the way into pass 2
//   st(j, b, val) : output element j of pass-2 pencil b
template <int N, int DIR, class Ld, class Mid, class St>
__device__ __forceinline__ void warp_plane_fft(cplx* buf, int lane, Ld ld, Mid mid, St st) {
  constexpr int P = N + 1;
  for (int a = lane; a < N; a += 32) {
    cplx v[N];
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = ld(i, a);
    fft_reg<N, DIR>(v);
#pragma unroll
    for (int i = 0; i < N; ++i) buf[i * P + a] = v[i];
  }
  __syncwarp();
  for (int b = lane; b < N; b += 32) {
    cplx v[N];
#pragma unroll
    for (int j = 0; j < N; ++j) v[j] = mid(buf[b * P + j], j);
    fft_reg<N, DIR>(v);
#pragma unroll
    for (int j = 0; j < N; ++j) st(j, b, v[j]);
  }
  __syncwarp();
}

template <int N>
constexpr size_t plane_smem_per_warp() { return sizeof(cplx) * (size_t)(N * (N + 1) + N); }

// ---- S1: f -> f^.  z pass: thread per (cy,cx) pencil; real input.  out[kz][cy][cx].
template <int N>
__global__ void __launch_bounds__(128) k_zfwd_real(const double* __restrict__ f, cplx* __restrict__ T) {
  constexpr int N2 = N * N, N3 = N2 * N;
  const int pid = blockIdx.x * 128 + threadIdx.x;
  if (pid >= N2) return;
  const int cy = pid / N, cx = pid % N;
  const double2* src = reinterpret_cast<const double2*>(f + (size_t)blockIdx.y * N3 + ((size_t)cx * N + cy) * N);
  cplx v[N];
#pragma unroll
  for (int i = 0; i < N / 2; ++i) {
    double2 t = src[i];
    v[2 * i] = make_double2(t.x, 0.0);
    v[2 * i + 1] = make_double2(t.y, 0.0);
  }
  fft_reg<N, -1>(v);
  cplx* dst = T + (size_t)blockIdx.y * N3 + pid;
#pragma unroll
  for (int k = 0; k < N; ++k) dst[(size_t)k * N2] = v[k];
}

// ---- forward x,y passes of one kz plane per warp.  MODE 0: store (f^);  MODE 1: QG += w_r b t3
// (steps 7-8).  in: T[item][slice][kz][cy][cx];  out (SPEC layout): [kz][kx][ky].
template <int N, int W, int MODE>
__global__ void __launch_bounds__(32 * W) k_plane_fwd(DevTables tab, const cplx* __restrict__ T, int Tslices,
                                                      cplx* __restrict__ out, int r) {
  constexpr int N2 = N * N, N3 = N2 * N;
  extern __shared__ cplx sm[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int kz = blockIdx.x * W + warp;
  if (kz >= N) return;
  cplx* buf = sm + (size_t)warp * (N * (N + 1) + N);
  const int item = blockIdx.y;
  int pair = 0, nsl = 1;
  bool full = false;
  double scale = 1.0;
  if (MODE == 1) {
    pair = item % tab.npairs;
    full = tab.full[pair];
    nsl = full ? tab.M : 1;
    scale = tab.w_rho[r];
  }
  cplx* o = out + (size_t)item * N3 + (size_t)kz * N2;
  const int kzs = sfreq(kz, N);
  for (int sl = 0; sl < nsl; ++sl) {
    // R-11: the transposed VHS pair (q,p) reads the summed products of (p,q)
    const int sitem = (MODE == 1 && !full) ? item - pair + tab.tsrc[pair] : item;
    const cplx* in = T + ((size_t)sitem * Tslices + sl) * N3 + (size_t)kz * N2;
    const double* bv = tab.bvhs + ((size_t)pair * tab.N_rho + r) * tab.K2n;
    warp_plane_fft<N, -1>(
        buf, lane, [&](int cy, int cx) { return in[cy * N + cx]; }, [](cplx x, int) { return x; },
        [&](int kx, int ky, cplx val) {
          const int idx = kx * N + ky;
          if (MODE == 0) {
            o[idx] = val;
          } else {
            cplx acc = o[idx];
            if (full) {
              cplx b = bfull_at(tab, pair, r, sl, sfreq(kx, N), sfreq(ky, N), kzs);
              acc.x += scale * (b.x * val.x - b.y * val.y);
              acc.y += scale * (b.x * val.y + b.y * val.x);
            } else {
              const int kxs = sfreq(kx, N), kys = sfreq(ky, N);
              const double b = scale * bv[kxs * kxs + kys * kys + kzs * kzs];
              acc.x = fma(b, val.x, acc.x);
              acc.y = fma(b, val.y, acc.y);
            }
            o[idx] = acc;
          }
        });
  }
}

// ---- steps 4-6a: phases + inverse x,y passes of one lz plane, for every (s, side).
// in: f^[xl][species][lz][lx][ly];  out: G[item][s][side][lz][cy][cx].
template <int N, int W>
__global__ void __launch_bounds__(32 * W) k_shift_xy(DevTables tab, const cplx* __restrict__ fhat, cplx* __restrict__ G, int r) {
  constexpr int N2 = N * N, N3 = N2 * N;
  extern __shared__ cplx sm[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* buf = sm + (size_t)warp * (N * (N + 1) + N);
  cplx* qv = buf + N * (N + 1);
  const int lz = blockIdx.x, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  const int p = pair / tab.ns, q = pair % tab.ns;
  for (int job = warp; job < 2 * tab.M; job += W) {
    const int s = job >> 1, side = job & 1;
    if (tab.sskip[(size_t)pair * tab.M + s]) continue;       // R-10 / R-11: the antipode (or the transposed pair) carries it
    const cplx* in = fhat + ((size_t)xl * tab.ns + (side ? q : p)) * N3 + (size_t)lz * N2;
    const cplx* ph = tab.phase + ((((size_t)pair * tab.N_rho + r) * tab.M + s) * 2 + side) * 3 * N;
    for (int j = lane; j < N; j += 32) qv[j] = cmul(ph[N + j], ph[2 * N + lz]);
    cplx* o = G + (((size_t)item * tab.M + s) * 2 + side) * N3 + (size_t)lz * N2;
    warp_plane_fft<N, +1>(
        buf, lane, [&](int lx, int ly) { return cmul(in[lx * N + ly], ph[lx]); },
        [&](cplx x, int ly) { return cmul(x, qv[ly]); }, [&](int cy, int cx, cplx val) { o[cy * N + cx] = val; });
  }
}

// ---- step 10, spectral part: inverse x,y passes of QG (job 0) and of c^(pq) f^_q (job 1),
// both scaled by 1/N^3 (unnormalised transforms, reading C-3).  out: G2[item][job][lz][cy][cx].
template <int N>
__global__ void __launch_bounds__(64) k_final_xy(DevTables tab, const cplx* __restrict__ fhat, const cplx* __restrict__ QG,
                                                 cplx* __restrict__ G2) {
  constexpr int N2 = N * N, N3 = N2 * N;
  extern __shared__ cplx sm[];
  const int job = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* buf = sm + (size_t)job * (N * (N + 1) + N);
  const int lz = blockIdx.x, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  const int q = pair % tab.ns;
  const double inv = 1.0 / ((double)N3);
  const cplx* in = (job == 0 ? QG + (size_t)item * N3 : fhat + ((size_t)xl * tab.ns + q) * N3) + (size_t)lz * N2;
  const cplx* cl = tab.closs + (size_t)pair * N3 + (size_t)lz * N2;
  cplx* o = G2 + ((size_t)item * 2 + job) * N3 + (size_t)lz * N2;
  warp_plane_fft<N, +1>(
      buf, lane,
      [&](int lx, int ly) {
        cplx v = in[lx * N + ly];
        if (job == 1) v = cmul(v, cl[lx * N + ly]);
        return make_double2(v.x * inv, v.y * inv);
      },
      [](cplx x, int) { return x; }, [&](int cy, int cx, cplx val) { o[cy * N + cx] = val; });
}

// ---- steps 6b-6c: inverse z pass of A and B (thread pair per pencil: even / odd outputs), product,
// sum over s (VHS) and forward z pass.  in: G[item][s][side][lz][pid];  out: T[item][slice][kz][pid].
template <int N, int PAR>
__device__ __forceinline__ void half_inverse_z(const cplx* __restrict__ in, cplx (&u)[N / 2]) {
  constexpr int H = N / 2, N2 = N * N;
#pragma unroll
  for (int j = 0; j < H; ++j) {
    cplx x0 = in[(size_t)j * N2], x1 = in[(size_t)(j + H) * N2];
    u[j] = (PAR == 0) ? cadd(x0, x1) : twiddle_mul<N, +1>(csub(x0, x1), j);
  }
  fft_reg<H, +1>(u);
}

template <int N, int PAR>
__device__ __forceinline__ void z_prod_body(const DevTables& tab, const cplx* __restrict__ G, cplx* __restrict__ T,
                                            int Tslices, cplx* S, int item, int pid, bool act, bool full) {
  constexpr int H = N / 2, N2 = N * N, N3 = N2 * N;
  const int tid = threadIdx.x;
  const int M = tab.M;
  bool fresh = true;
  const unsigned char* skip = tab.sskip + (size_t)(item % tab.npairs) * M;
  int last = M - 1;                                        // last sphere point this pair runs (R-10 / R-11)
  while (last >= 0 && skip[last]) --last;
  for (int s = 0; s <= last; ++s) {
    if (skip[s]) continue;
    const cplx* ga = G + (((size_t)item * M + s) * 2) * N3 + pid;
    cplx a[H], b[H];
    half_inverse_z<N, PAR>(ga, a);
    half_inverse_z<N, PAR>(ga + N3, b);
#pragma unroll
    for (int k = 0; k < H; ++k) {
      cplx pr = cmul(a[k], b[k]);
      if (!fresh) pr = cadd(pr, S[k * 256 + tid]);
      S[k * 256 + tid] = pr;
    }
    fresh = false;
    if (full || s == last) {
      // forward z transform of the accumulated samples (decimation in time over the thread pair)
      cplx y[H];
#pragma unroll
      for (int k = 0; k < H; ++k) y[k] = S[k * 256 + tid];
      fft_reg<H, -1>(y);
      if (PAR == 1) {
#pragma unroll
        for (int k = 0; k < H; ++k) y[k] = twiddle_mul<N, -1>(y[k], k);
      }
#pragma unroll
      for (int k = 0; k < H; ++k) S[k * 256 + tid] = y[k];
      __syncthreads();
      cplx* t = T + ((size_t)item * Tslices + (full ? s : 0)) * N3 + pid;
#pragma unroll
      for (int k = 0; k < H; ++k) {
        cplx o = S[k * 256 + (tid ^ 128)];
        cplx x = (PAR == 0) ? cadd(y[k], o) : csub(o, y[k]);
        if (act) t[(size_t)(k + PAR * H) * N2] = x;
      }
      __syncthreads();
      fresh = true;
    }
  }
}

template <int N>
__global__ void __launch_bounds__(256) k_z_prod(DevTables tab, const cplx* __restrict__ G, cplx* __restrict__ T, int Tslices) {
  constexpr int N2 = N * N;
  extern __shared__ cplx S[];   // [N/2][256]
  const int tid = threadIdx.x;
  int pid = blockIdx.x * 128 + (tid & 127);
  const bool act = pid < N2;
  if (!act) pid = N2 - 1;
  const int item = blockIdx.y;
  const bool full = tab.full[item % tab.npairs];
  if ((tid >> 7) == 0) z_prod_body<N, 0>(tab, G, T, Tslices, S, item, pid, act, full);
  else z_prod_body<N, 1>(tab, G, T, Tslices, S, item, pid, act, full);
}

// ---- step 10, physical part: inverse z pass of both arrays, Q = beta Re(gain - f_p loss).
// SUM = true: out[x][p][:] = sum_q (Eq. 1), blockIdx.y = xl*ns + p.  SUM = false: out[item][:].
template <int N, bool SUM>
__global__ void __launch_bounds__(128) k_z_final(DevTables tab, const cplx* __restrict__ G2, const double* __restrict__ f,
                                                 double* __restrict__ out) {
  constexpr int N2 = N * N, N3 = N2 * N;
  const int pid = blockIdx.x * 128 + threadIdx.x;
  if (pid >= N2) return;
  const int cy = pid / N, cx = pid % N;
  const int ns = tab.ns;
  int xl, p, q0, q1;
  if (SUM) { xl = blockIdx.y / ns; p = blockIdx.y % ns; q0 = 0; q1 = ns; }
  else { int item = blockIdx.y; xl = item / tab.npairs; int pair = item % tab.npairs; p = pair / ns; q0 = pair % ns; q1 = q0 + 1; }
  const size_t voff = ((size_t)cx * N + cy) * N;
  const double2* fp = reinterpret_cast<const double2*>(f + ((size_t)xl * ns + p) * N3 + voff);
  double acc[N];
#pragma unroll
  for (int i = 0; i < N; ++i) acc[i] = 0.0;
  for (int q = q0; q < q1; ++q) {
    const int item = xl * tab.npairs + p * ns + q;
    const double beta = tab.beta[p * ns + q];
    const cplx* g = G2 + (size_t)item * 2 * N3 + pid;
    double gain[N];
    {
      cplx v[N];
#pragma unroll
      for (int i = 0; i < N; ++i) v[i] = g[(size_t)i * N2];
      fft_reg<N, +1>(v);
#pragma unroll
      for (int i = 0; i < N; ++i) gain[i] = v[i].x;
    }
    cplx v[N];
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = g[N3 + (size_t)i * N2];
    fft_reg<N, +1>(v);
#pragma unroll
    for (int i = 0; i < N / 2; ++i) {
      double2 fv = fp[i];
      acc[2 * i] += beta * (gain[2 * i] - fv.x * v[2 * i].x);
      acc[2 * i + 1] += beta * (gain[2 * i + 1] - fv.y * v[2 * i + 1].x);
    }
  }
  double2* o = reinterpret_cast<double2*>(out + (size_t)blockIdx.y * N3 + voff);
#pragma unroll
  for (int i = 0; i < N / 2; ++i) o[i] = make_double2(acc[2 * i], acc[2 * i + 1]);
}

}  // namespace dgfs
