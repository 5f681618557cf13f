// collide.cu -- dgfs_collide / dgfs_collide_pairs: Algorithm 2 of PAPER.md on sm_100a.
//
// Per pair (p,q), spatial point x, radial node r, sphere point s (steps 2-8):
//   A = ifft3(e^{+i mu_q a_rs} f^_p),  B = ifft3(e^{-i mu_p a_rs} f^_q),  QG += w_r w_s b_rs fft3(A.B),
// then  Q = beta Re( ifft3(QG) - f_p . ifft3(c f^_q) )  (step 10).
//
// Organisation: every 3-D transform is split into a 2-D transform of one
// spectral plane done by ONE WARP (lane = pencil, 1-D FFTs in registers, one transposition through
// that warp's shared-memory tile) and a 1-D transform along z done by thread pairs (even / odd
// outputs, registers only).  The phases e^{+-i mu a_rs} are separable (a_rs is linear in l) and
// are applied as 1-D factors on the way into the x and y passes.  For VHS pairs b_rs does not
// depend on s, so sum_s w_s A.B is formed before the forward transform (exact rearrangement R-1).
#include <cmath>
#include <cstdio>
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
    const cplx* in = T + ((size_t)item * Tslices + sl) * N3 + (size_t)kz * N2;
    const double* bv = tab.bvhs + ((size_t)pair * tab.N_rho + r) * tab.K2n;
    const cplx* bf = (MODE == 1 && full) ? tab.bfull[pair] + ((size_t)r * tab.M + sl) * N3 + (size_t)kz * N2 : nullptr;
    warp_plane_fft<N, -1>(
        buf, lane, [&](int cy, int cx) { return in[cy * N + cx]; }, [](cplx x, int) { return x; },
        [&](int kx, int ky, cplx val) {
          const int idx = kx * N + ky;
          if (MODE == 0) {
            o[idx] = val;
          } else {
            cplx acc = o[idx];
            if (full) {
              cplx b = bf[idx];
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
  for (int s = 0; s < M; ++s) {
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
    if (full || s == M - 1) {
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

// ------------------------------------------------------------------ host orchestration ---------
int ensure_workspace(dgfs_ctx* c, size_t bytes) {
  if (bytes <= c->ws_bytes) return DGFS_OK;
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) return check_cuda(c, e, "workspace sync");
  cudaFree(c->ws);
  c->ws = nullptr; c->ws_bytes = 0;
  int rc = check_cuda(c, cudaMalloc(&c->ws, bytes), "workspace allocation");
  if (rc) return rc;
  c->ws_bytes = bytes;
  return DGFS_OK;
}

ChunkPlan plan_chunks(const dgfs_ctx* c, int nx) {
  ChunkPlan pl{};
  const size_t arr = (size_t)c->N3 * sizeof(cplx);
  const size_t g_per_point = (size_t)c->npairs * c->M * 2 * arr;
  size_t nbx = c->scratch_budget / g_per_point;
  if (nbx < 1) nbx = 1;
  if (nbx > (size_t)nx) nbx = nx;
  if (nbx * c->npairs > 65535) nbx = 65535 / c->npairs;      // gridDim.y limit
  if (nbx < 1) nbx = 1;
  pl.nbx = (int)nbx;
  const size_t items = nbx * c->npairs;
  const size_t tsl = c->any_full ? c->M : 1;
  size_t off = 0;
  pl.off_fhat = off; off += nbx * c->ns * arr;
  pl.off_qg = off;   off += items * arr;
  pl.off_g = off;    off += nbx * g_per_point;
  pl.off_t = off;    off += items * tsl * arr;
  pl.total = off;
  return pl;
}

template <int N>
static int collide_impl(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  constexpr int N2 = N * N, N3 = N2 * N;
  constexpr int W = (N <= 32) ? 4 : 2;
  const ChunkPlan pl = plan_chunks(c, nx);
  int rc = ensure_workspace(c, pl.total);
  if (rc) return rc;
  char* ws = (char*)c->ws;
  cplx* fhat = (cplx*)(ws + pl.off_fhat);
  cplx* QG = (cplx*)(ws + pl.off_qg);
  cplx* G = (cplx*)(ws + pl.off_g);
  cplx* T = (cplx*)(ws + pl.off_t);
  const int ns = c->ns, np = c->npairs;
  const int tsl = c->any_full ? c->M : 1;
  const size_t smem_plane = plane_smem_per_warp<N>() * W;
  const size_t smem_final = plane_smem_per_warp<N>() * 2;
  const size_t smem_z = sizeof(cplx) * (N / 2) * 256;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(k_plane_fwd<N, W, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_plane_fwd<N, W, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_shift_xy<N, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_final_xy<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_final);
    cudaFuncSetAttribute(k_z_prod<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_z);
    attr_done = true;
  }
  const int pen_blocks = (N2 + 127) / 128;
  const int plane_blocks = (N + W - 1) / W;
  // algorithmic FLOPs per spatial point of each r-loop kernel (FFT3 = 15 N^3 log2 N,
  // a 1-D pass is a third of it): phases 12 N^3, product 6 N^3, accumulate 8 N^3 (complex b) / 4 N^3 (real b)
  const double fft3 = 15.0 * N3 * log2((double)N);
  double fl_shift = 0, fl_zprod = 0, fl_acc = 0;
  for (int pr = 0; pr < np; ++pr) {
    const double M = c->M;
    fl_shift += M * (2.0 * fft3 * 2.0 / 3.0 + 12.0 * N3);
    fl_zprod += M * (2.0 * fft3 / 3.0 + 6.0 * N3) + (c->full[pr] ? M : 1.0) * fft3 / 3.0;
    fl_acc += (c->full[pr] ? M * (fft3 * 2.0 / 3.0 + 8.0 * N3) : (fft3 * 2.0 / 3.0 + 4.0 * N3));
  }
  for (int x0 = 0; x0 < nx; x0 += pl.nbx) {
    const int nb = (nx - x0 < pl.nbx) ? nx - x0 : pl.nbx;
    const int items = nb * np;
    const double* fc = f + (size_t)x0 * ns * N3;
    // S1: f^ for every species of every point of the chunk (R-2: once per species, not per pair)
    { ProfScope ps(c->prof, st, "k_zfwd_real", nb * ns * fft3 / 3.0);
      k_zfwd_real<N><<<dim3(pen_blocks, nb * ns), 128, 0, st>>>(fc, T); }
    { ProfScope ps(c->prof, st, "k_plane_fwd<store>", nb * ns * fft3 * 2.0 / 3.0);
      k_plane_fwd<N, W, 0><<<dim3(plane_blocks, nb * ns), 32 * W, smem_plane, st>>>(c->tab, T, 1, fhat, 0); }
    cudaMemsetAsync(QG, 0, (size_t)items * N3 * sizeof(cplx), st);
    for (int r = 0; r < c->N_rho; ++r) {
      { ProfScope ps(c->prof, st, "k_shift_xy", nb * fl_shift);
        k_shift_xy<N, W><<<dim3(N, items), 32 * W, smem_plane, st>>>(c->tab, fhat, G, r); }
      { ProfScope ps(c->prof, st, "k_z_prod", nb * fl_zprod);
        k_z_prod<N><<<dim3(pen_blocks, items), 256, smem_z, st>>>(c->tab, G, T, tsl); }
      { ProfScope ps(c->prof, st, "k_plane_fwd<accumulate>", nb * fl_acc);
        k_plane_fwd<N, W, 1><<<dim3(plane_blocks, items), 32 * W, smem_plane, st>>>(c->tab, T, tsl, QG, r); }
    }
    { ProfScope ps(c->prof, st, "k_final_xy", items * (2.0 * fft3 * 2.0 / 3.0 + 6.0 * N3));
      k_final_xy<N><<<dim3(N, items), 64, smem_final, st>>>(c->tab, fhat, QG, G); }
    { ProfScope ps(c->prof, st, "k_z_final", items * (2.0 * fft3 / 3.0 + 5.0 * N3));
      if (pairs_out)
        k_z_final<N, false><<<dim3(pen_blocks, items), 128, 0, st>>>(c->tab, G, fc, out + (size_t)x0 * np * N3);
      else
        k_z_final<N, true><<<dim3(pen_blocks, nb * ns), 128, 0, st>>>(c->tab, G, fc, out + (size_t)x0 * ns * N3); }
  }
  return check_cuda(c, cudaGetLastError(), "collide launch");
}

int run_collide(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  switch (c->N) {
    case 8: return collide_impl<8>(c, f, out, nx, pairs_out, st);
    case 16: return collide_impl<16>(c, f, out, nx, pairs_out, st);
    case 24: return collide_impl<24>(c, f, out, nx, pairs_out, st);
    case 32: return collide_impl<32>(c, f, out, nx, pairs_out, st);
    case 48: return collide_impl<48>(c, f, out, nx, pairs_out, st);
  }
  return set_error(c, DGFS_ENOSUP, "unsupported N");
}

}  // namespace dgfs

using namespace dgfs;

static int collide_common(dgfs_ctx* c, const double* f, double* out, int nx, void* stream, bool pairs, const char* who) {
  if (!c) return DGFS_EINVAL;
  if (nx < 0) return set_error(c, DGFS_EINVAL, std::string(who) + ": nx must be >= 0");
  if (nx == 0) return DGFS_OK;
  if (!f || !out) return set_error(c, DGFS_EINVAL, std::string(who) + ": f and output must not be NULL");
  if ((const void*)f == (const void*)out) return set_error(c, DGFS_EINVAL, std::string(who) + ": output must not alias f");
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) return check_cuda(c, e, "cudaSetDevice");
  return run_collide(c, f, out, nx, pairs, (cudaStream_t)stream);
}

extern "C" int dgfs_collide(dgfs_ctx* c, const double* f, double* Q, int nx, void* stream) {
  return collide_common(c, f, Q, nx, stream, false, "dgfs_collide");
}
extern "C" int dgfs_collide_pairs(dgfs_ctx* c, const double* f, double* Qpq, int nx, void* stream) {
  return collide_common(c, f, Qpq, nx, stream, true, "dgfs_collide_pairs");
}
// Host-buffer form: slabs of `hp_pts` points go host -> device -> kernels -> host on three streams,
// double buffered, so that the copies of slab i+1 / i-1 overlap the kernels of slab i.
extern "C" int dgfs_collide_host(dgfs_ctx* c, const double* f_host, double* Q_host, int nx) {
  if (!c) return DGFS_EINVAL;
  if (nx < 0) return set_error(c, DGFS_EINVAL, "dgfs_collide_host: nx must be >= 0");
  if (nx == 0) return DGFS_OK;
  if (!f_host || !Q_host) return set_error(c, DGFS_EINVAL, "dgfs_collide_host: f_host and Q_host must not be NULL");
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) return check_cuda(c, e, "cudaSetDevice");
  const size_t per_pt = (size_t)c->ns * c->N3;
  int slab = (int)((size_t)(128u << 20) / (per_pt * sizeof(double)));      // ~128 MiB per slab buffer
  if (slab < 1) slab = 1;
  if (slab > nx) slab = nx;
  int rc;
  if (!c->hp_stream[0]) {
    for (int i = 0; i < 3; ++i) {
      if ((rc = check_cuda(c, cudaStreamCreateWithFlags(&c->hp_stream[i], cudaStreamNonBlocking), "stream create"))) return rc;
      for (int b = 0; b < 2; ++b)
        if ((rc = check_cuda(c, cudaEventCreateWithFlags(&c->hp_ev[i][b], cudaEventDisableTiming), "event create"))) return rc;
    }
  }
  if (slab > c->hp_pts) {
    cudaDeviceSynchronize();
    for (int b = 0; b < 2; ++b) {
      cudaFree(c->hp_f[b]); cudaFree(c->hp_q[b]); c->hp_f[b] = c->hp_q[b] = nullptr;
    }
    c->hp_pts = 0;
    for (int b = 0; b < 2; ++b) {
      if ((rc = check_cuda(c, cudaMalloc((void**)&c->hp_f[b], slab * per_pt * sizeof(double)), "host-pipe slab allocation"))) return rc;
      if ((rc = check_cuda(c, cudaMalloc((void**)&c->hp_q[b], slab * per_pt * sizeof(double)), "host-pipe slab allocation"))) return rc;
    }
    c->hp_pts = slab;
  }
  if ((rc = ensure_workspace(c, plan_chunks(c, slab).total))) return rc;
  cudaStream_t s_in = c->hp_stream[0], s_k = c->hp_stream[1], s_out = c->hp_stream[2];
  int i = 0;
  for (int x0 = 0; x0 < nx; x0 += slab, ++i) {
    const int n = (nx - x0 < slab) ? nx - x0 : slab, b = i & 1;
    const size_t bytes = (size_t)n * per_pt * sizeof(double);
    if (i >= 2) cudaStreamWaitEvent(s_in, c->hp_ev[1][b], 0);             // kernels of slab i-2 have read hp_f[b]
    cudaMemcpyAsync(c->hp_f[b], f_host + (size_t)x0 * per_pt, bytes, cudaMemcpyHostToDevice, s_in);
    cudaEventRecord(c->hp_ev[0][b], s_in);
    cudaStreamWaitEvent(s_k, c->hp_ev[0][b], 0);
    if (i >= 2) cudaStreamWaitEvent(s_k, c->hp_ev[2][b], 0);              // download of slab i-2 has read hp_q[b]
    if ((rc = run_collide(c, c->hp_f[b], c->hp_q[b], n, false, s_k))) return rc;
    cudaEventRecord(c->hp_ev[1][b], s_k);
    cudaStreamWaitEvent(s_out, c->hp_ev[1][b], 0);
    cudaMemcpyAsync(Q_host + (size_t)x0 * per_pt, c->hp_q[b], bytes, cudaMemcpyDeviceToHost, s_out);
    cudaEventRecord(c->hp_ev[2][b], s_out);
  }
  for (int k = 0; k < 3; ++k)
    if ((rc = check_cuda(c, cudaStreamSynchronize(c->hp_stream[k]), "dgfs_collide_host"))) return rc;
  return DGFS_OK;
}

extern "C" size_t dgfs_workspace_bytes(const dgfs_ctx* c, int nx) {
  if (!c || nx <= 0) return 0;
  return plan_chunks(c, nx).total;
}
extern "C" int dgfs_reserve(dgfs_ctx* c, int nx) {
  if (!c) return DGFS_EINVAL;
  if (nx < 0) return set_error(c, DGFS_EINVAL, "dgfs_reserve: nx must be >= 0");
  if (nx == 0) return DGFS_OK;
  cudaSetDevice(c->device);
  return ensure_workspace(c, plan_chunks(c, nx).total);
}
extern "C" long long dgfs_launch_count(const dgfs_ctx* c) { return c ? c->prof.total_launches : 0; }
extern "C" int dgfs_profile_enable(dgfs_ctx* c, int on) {
  if (!c) return DGFS_EINVAL;
  c->prof.on = on != 0;
  return DGFS_OK;
}
extern "C" int dgfs_profile_count(const dgfs_ctx* c) { return c ? (int)c->prof.entries.size() : 0; }
extern "C" int dgfs_profile_get(dgfs_ctx* c, int i, const char** name, long long* launches, double* ms, double* flops) {
  if (!c) return DGFS_EINVAL;
  if (i < 0 || i >= (int)c->prof.entries.size()) return set_error(c, DGFS_EINVAL, "dgfs_profile_get: index out of range");
  cudaSetDevice(c->device);
  c->prof.drain();
  const ProfEntry& e = c->prof.entries[i];
  if (name) *name = e.name.c_str();
  if (launches) *launches = e.launches;
  if (ms) *ms = e.ms;
  if (flops) *flops = e.flops;
  return DGFS_OK;
}
extern "C" int dgfs_profile_reset(dgfs_ctx* c) {
  if (!c) return DGFS_EINVAL;
  cudaSetDevice(c->device);
  c->prof.drain();
  for (auto& e : c->prof.entries) { e.launches = 0; e.ms = 0; e.flops = 0; }
  return DGFS_OK;
}
extern "C" double dgfs_flops_per_pair_eval(const dgfs_ctx* c, int p, int q) {
  if (!c || p < 0 || q < 0 || p >= c->ns || q >= c->ns) return 0.0;
  const double N3 = c->N3, fft3 = 15.0 * N3 * log2((double)c->N);
  const double tail = 2.0 * fft3 + 11.0 * N3 + fft3 / c->ns;
  const double rs = (double)c->N_rho * c->M;
  if (c->full[p * c->ns + q]) return rs * (3.0 * fft3 + 26.0 * N3) + tail;             // verbatim Algo 2
  return rs * (2.0 * fft3 + 22.0 * N3) + c->N_rho * (fft3 + 4.0 * N3) + tail;           // with R-1
}
