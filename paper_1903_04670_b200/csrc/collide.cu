// collide.cu -- dgfs_collide / dgfs_collide_pairs: Algorithm 2 of PAPER.md on sm_100a.
// This file holds the C ABI entry points and the stage-per-kernel (v0) pipeline, which serves N = 48 configurations
// with full-table pairs (VSS, table_mode 1) and DGFS_PIPELINE=v0; everything else runs collide_v1.cu.
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
#include "kernels_v0.cuh"

namespace dgfs {

// dgfs_params::nyquist_filter: P f = prod_d (1 - E_d) f, (E_d f)(c) = (-1)^{c_d} (1/N) sum_{c_d'} (-1)^{c_d'} f:
// removes the spectral planes l_d = -N/2 without a transform.  One pass per axis; thread per pencil of that axis.
// AXIS 0: stride N^2 (cx), 1: stride N (cy), 2: stride 1 (cz).
template <int N, int AXIS>
__global__ void __launch_bounds__(128) k_nyq_filter(const double* src, double* dst) {
  constexpr int N2 = N * N, N3 = N2 * N;
  const int pid = blockIdx.x * 128 + threadIdx.x;
  if (pid >= N2) return;
  const int a = pid / N, b = pid % N;
  const size_t base = (size_t)blockIdx.y * N3 + (AXIS == 0 ? (size_t)a * N + b : AXIS == 1 ? (size_t)a * N2 + b : (size_t)a * N2 + (size_t)b * N);
  constexpr size_t stride = AXIS == 0 ? N2 : AXIS == 1 ? N : 1;
  double v[N], m = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i) { v[i] = src[base + i * stride]; m += (i & 1) ? -v[i] : v[i]; }
  m *= 1.0 / N;
#pragma unroll
  for (int i = 0; i < N; ++i) dst[base + i * stride] = (i & 1) ? v[i] + m : v[i] - m;
}

template <int N>
static void nyquist_filter_impl(const double* src, double* dst, int narr, cudaStream_t st) {
  const dim3 grid((N * N + 127) / 128, narr);
  k_nyq_filter<N, 2><<<grid, 128, 0, st>>>(src, dst);
  k_nyq_filter<N, 1><<<grid, 128, 0, st>>>(dst, dst);
  k_nyq_filter<N, 0><<<grid, 128, 0, st>>>(dst, dst);
}

int launch_nyquist_filter(dgfs_ctx* c, const double* src, double* dst, int narr, cudaStream_t st) {
  switch (c->N) {
    case 8: nyquist_filter_impl<8>(src, dst, narr, st); break;
    case 16: nyquist_filter_impl<16>(src, dst, narr, st); break;
    case 24: nyquist_filter_impl<24>(src, dst, narr, st); break;
    case 32: nyquist_filter_impl<32>(src, dst, narr, st); break;
    case 48: nyquist_filter_impl<48>(src, dst, narr, st); break;
    default: return set_error(c, DGFS_ENOSUP, "unsupported N");
  }
  return DGFS_OK;
}

// ------------------------------------------------------------------ host orchestration ---------
// Workspace growth is ordered on the caller's stream (stream-ordered allocator): the old block is released after
// everything enqueued so far, the new one exists before anything enqueued later; no device-wide synchronisation.
// Not possible while `st` is being captured into a CUDA graph: dgfs_reserve first (include/dgfs.h).
int ensure_workspace(dgfs_ctx* c, size_t bytes, cudaStream_t st) {
  if (bytes <= c->ws_bytes) return DGFS_OK;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cap);
  if (cap != cudaStreamCaptureStatusNone)
    return set_error(c, DGFS_EINVAL, "workspace too small during stream capture: call dgfs_reserve before capturing");
  if (!c->pool_set) {
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, c->device) == cudaSuccess) {
      unsigned long long keep = ~0ull;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    c->pool_set = true;
  }
  if (c->ev_last_set) cudaStreamWaitEvent(st, c->ev_last, 0);      // earlier calls on other streams still use the old block
  drop_graphs_v1(c);                                               // captured graphs point into the old block
  if (c->ws) cudaFreeAsync(c->ws, st);
  c->ws = nullptr; c->ws_bytes = 0;
  int rc = check_cuda(c, cudaMallocAsync(&c->ws, bytes, st), "workspace allocation");
  if (rc) { c->ws = nullptr; return rc; }
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
  pl.off_fp = off;   off += c->nyq_filter ? nbx * c->ns * (arr / 2) : 0;      // filtered inputs (real)
  pl.total = off;
  return pl;
}

template <int N>
static int collide_impl(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  constexpr int N2 = N * N, N3 = N2 * N;
  constexpr int W = (N <= 32) ? 4 : 2;
  const ChunkPlan pl = plan_chunks(c, nx);
  int rc = ensure_workspace(c, pl.total, st);
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
  if (!c->v0_attr_done) {                 // per context, hence per device
    cudaFuncSetAttribute(k_plane_fwd<N, W, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_plane_fwd<N, W, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_shift_xy<N, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_final_xy<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_final);
    cudaFuncSetAttribute(k_z_prod<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_z);
    c->v0_attr_done = true;
  }
  const int pen_blocks = (N2 + 127) / 128;
  const int plane_blocks = (N + W - 1) / W;
  // algorithmic FLOPs per spatial point of each r-loop kernel (FFT3 = 15 N^3 log2 N,
  // a 1-D pass is a third of it): phases 12 N^3, product 6 N^3, accumulate 8 N^3 (complex b) / 4 N^3 (real b)
  const double fft3 = 15.0 * N3 * log2((double)N);
  double fl_shift = 0, fl_zprod = 0, fl_acc = 0;
  for (int pr = 0; pr < np; ++pr) {
    const double M = c->M;
    double run = 0;
    for (int s = 0; s < c->M; ++s) run += !c->v0_sskip[(size_t)pr * c->M + s];
    fl_shift += run * (2.0 * fft3 * 2.0 / 3.0 + 12.0 * N3);
    fl_zprod += run * (2.0 * fft3 / 3.0 + 6.0 * N3) + (c->full[pr] ? M : (run > 0 ? 1.0 : 0.0)) * fft3 / 3.0;
    fl_acc += (c->full[pr] ? M * (fft3 * 2.0 / 3.0 + 8.0 * N3) : (fft3 * 2.0 / 3.0 + 4.0 * N3));
  }
  for (int x0 = 0; x0 < nx; x0 += pl.nbx) {
    const int nb = (nx - x0 < pl.nbx) ? nx - x0 : pl.nbx;
    const int items = nb * np;
    const double* fc = f + (size_t)x0 * ns * N3;
    if (c->nyq_filter) {         // the operator acts on P f (dgfs_params::nyquist_filter)
      double* fp = (double*)(ws + pl.off_fp);
      if ((rc = launch_nyquist_filter(c, fc, fp, nb * ns, st))) return rc;
      fc = fp;
    }
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

// One call at a time owns the context's workspace (and, for v1, its auxiliary streams): a call first waits, on its
// stream, for the last launch of the previous call, whichever stream that was issued on.
int run_collide(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cap);
  const bool capturing = cap != cudaStreamCaptureStatusNone;      // a captured graph orders its own nodes
  if (!capturing && c->ev_last_set) cudaStreamWaitEvent(st, c->ev_last, 0);
  int rc;
  if (c->use_v1) rc = run_collide_v1(c, f, out, nx, pairs_out, st);
  else switch (c->N) {
    case 8: rc = collide_impl<8>(c, f, out, nx, pairs_out, st); break;
    case 16: rc = collide_impl<16>(c, f, out, nx, pairs_out, st); break;
    case 24: rc = collide_impl<24>(c, f, out, nx, pairs_out, st); break;
    case 32: rc = collide_impl<32>(c, f, out, nx, pairs_out, st); break;
    case 48: rc = collide_impl<48>(c, f, out, nx, pairs_out, st); break;
    default: rc = set_error(c, DGFS_ENOSUP, "unsupported N");
  }
  if (!capturing && c->ev_last) { cudaEventRecord(c->ev_last, st); c->ev_last_set = true; }
  return rc;
}

static size_t workspace_for(const dgfs_ctx* c, int nx) {
  return c->use_v1 ? workspace_bytes_v1(c, nx) : plan_chunks(c, nx).total;
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
  int slab = (int)((size_t)(256u << 20) / (per_pt * sizeof(double)));      // ~256 MiB per slab buffer
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
  if ((rc = ensure_workspace(c, workspace_for(c, slab), c->hp_stream[1]))) return rc;
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
  return workspace_for(c, nx);
}
extern "C" int dgfs_reserve(dgfs_ctx* c, int nx) {
  if (!c) return DGFS_EINVAL;
  if (nx < 0) return set_error(c, DGFS_EINVAL, "dgfs_reserve: nx must be >= 0");
  if (nx == 0) return DGFS_OK;
  cudaSetDevice(c->device);
  int rc = ensure_workspace(c, workspace_for(c, nx), nullptr);
  if (rc) return rc;
  return check_cuda(c, cudaStreamSynchronize(nullptr), "dgfs_reserve");
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
  if (c->use_v1) return flops_per_pair_eval_v1(c, p * c->ns + q);
  const double N3 = c->N3, fft3 = 15.0 * N3 * log2((double)c->N);
  const double tail = 2.0 * fft3 + 11.0 * N3 + fft3 / c->ns;
  const double rs = (double)c->N_rho * c->M;
  const int pair = p * c->ns + q;
  if (c->full[pair]) return rs * (3.0 * fft3 + 26.0 * N3) + tail;                        // verbatim Algo 2
  // with R-1; R-10 / R-11: only `run` of the M sphere points are shifted and multiplied, a transposed pair none
  int run = 0;
  for (int s = 0; s < c->M; ++s) run += !c->v0_sskip[(size_t)pair * c->M + s];
  const double fwd = (c->v0_tsrc[pair] == pair) ? fft3 + 4.0 * N3 : fft3 * 2.0 / 3.0 + 4.0 * N3;
  return (double)c->N_rho * run * (2.0 * fft3 + 22.0 * N3) + c->N_rho * fwd + tail;
}
