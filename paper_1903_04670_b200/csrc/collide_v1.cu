// collide_v1.cu -- v1 pipeline of dgfs_collide (N <= 32; N = 48 with collide_v1_wide.cuh): Algorithm 2 of PAPER.md with the exact
// rearrangements of DESIGN.md section 5 (R-1 .. R-12).  The description below is the path of pairs whose b_rs
// does not depend on s (VHS, table_mode 0); pairs with a full table share the first three kernels and take
// k_xy_full / k_zfwd_full afterwards (described there).
//
// What is computed per pair (p,q), point x and radial node r (steps 2-8):
//   S_r(c) = sum_s w_s Re[ A_rs(c) B_rs(c) ],   A_rs = ifft3(e^{+i mu_q a_rs} f^_p),  B_rs = ifft3(e^{-i mu_p a_rs} f^_q)
//   QG    += w_r b_r(|k|) fft3(S_r)
// Re[.] is exact here: b_r is real and even in k, so Im(A B) only feeds the imaginary part that step 10
// discards.  f_p, f_q are real, hence A = a_r + i a_i with REAL fields a_r, a_i, where a_i comes
// from the three Nyquist planes only (the shift multiplier has no conjugate partner there).  Writing each
// 1-D factor as h_d + J s_d (v1_tables.h), with J standing for the imaginary unit that breaks the
// Hermitian symmetry,
//   a_r <- h_x h_y h_z - s_x s_y h_z - s_x h_y s_z - h_x s_y s_z        (spectral multipliers of f^_p)
//   a_i <- s_x h_y h_z + h_x s_y h_z + h_x h_y s_z - s_x s_y s_z
// and the same for B.  Two real fields share one complex transform: Z = a_r + i b_r, W = a_i + i b_i,
// Re(A B) = Re Z Im Z - Re W Im W.
//
// Kernels per radial node (all spatial points of a chunk at once):
//   k_zshift  inverse z pass of h_z f^ for every DISTINCT z shift (the sphere rules share sigma_z values:
//             18 arrays instead of 96 at c2), on the Hermitian half of the (lx,ly) plane (R-7)
//   k_nyq1d / k_nyq2   the Nyquist-plane fields: three 1-D sums and three 2-D transforms per (pair, s)
//   k_wterm   -sum_s Re W Im W  (tables staged by TMA bulk copies)
//   k_xy      per (pair, cz plane): for every s the inverse x,y passes of the packed field in one warp
//             (lane = pencil, FFTs in registers, one transposition through shared memory), the product
//             and the sum over s in registers, then the forward x,y passes of the real plane S_r(., ., cz)
//   k_zfwd_acc  forward z pass, QG += w_r b_r .
// Steps 1 and 10 reuse the v0 kernels.  dgfs_params::precision = 1 runs k_xy on float2 copies (k_xy<N, W, float2>).
// Sphere points with a zero component (R-9) skip the fields and factors
// that vanish; same-species pairs run one point per antipodal couple (R-10) and a transposed pair (q,p) reuses
// the summed products of (p,q) (R-11): see build_tables_v1.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include "ctx.h"
#include "kernels_v0.cuh"

namespace dgfs {

// flags of V1Tables::jobs[].w beside the zero-component mask (bits 0-2)
enum { JOB_FIRST = 8, JOB_LAST = 16, JOB_SLOT = 32 };

// ---------------------------------------------------------------- create-time tables ------------
static void split_factor(double theta, int N, double scale, cplx* h, double* s) {
  const int H = N / 2;
  for (int j = 0; j < N; ++j) {
    const int v = j - (j >= H ? N : 0);
    h[j] = make_double2(cos(theta * v) * scale, sin(theta * v) * scale);
  }
  h[H] = make_double2(cos(theta * H) * scale, 0.0);
  *s = -sin(theta * H) * scale;
}

template <class T>
static int upload(dgfs_ctx* c, T** d, const std::vector<T>& h, const char* what) {
  int rc = check_cuda(c, cudaMalloc((void**)d, h.size() * sizeof(T)), what);
  if (rc) return rc;
  return check_cuda(c, cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice), what);
}

int build_tables_v1(dgfs_ctx* c) {
  const int ns = c->ns, np = c->npairs, N = c->N, Nr = c->N_rho, M = c->M;
  const double pi = 3.14159265358979323846;
  // distinct (species, kappa) with kappa = +mu_q sigma_z (side A acts on f^_p) or -mu_p sigma_z (side B on f^_q)
  std::vector<double> zk;
  c->v1_zsp.clear(); c->v1_zmap.assign((size_t)np * M * 2, 0);
  auto zjob = [&](int sp, double kappa) {
    for (size_t k = 0; k < zk.size(); ++k)
      if (c->v1_zsp[k] == sp && fabs(zk[k] - kappa) <= 1e-15) return (int)k;
    c->v1_zsp.push_back(sp); zk.push_back(kappa);
    return (int)zk.size() - 1;
  };
  for (int p = 0; p < ns; ++p) for (int q = 0; q < ns; ++q) {
    const double mu_q = c->mass[q] / (c->mass[p] + c->mass[q]), mu_p = c->mass[p] / (c->mass[p] + c->mass[q]);
    for (int s = 0; s < M; ++s) {
      c->v1_zmap[((size_t)(p * ns + q) * M + s) * 2 + 0] = zjob(p, mu_q * c->sigma[3 * s + 2]);
      c->v1_zmap[((size_t)(p * ns + q) * M + s) * 2 + 1] = zjob(q, -mu_p * c->sigma[3 * s + 2]);
    }
  }
  const int nz = (int)zk.size();
  c->v1_nz = nz;
  // jobs with kappa = 0 (sigma_z = 0) do not depend on the radial node: put them last, they run once per chunk
  {
    std::vector<int> perm, inv(nz);
    for (int k = 0; k < nz; ++k) if (zk[k] != 0.0) perm.push_back(k);
    c->v1_nz0 = nz - (int)perm.size();
    for (int k = 0; k < nz; ++k) if (zk[k] == 0.0) perm.push_back(k);
    std::vector<double> zk2(nz); std::vector<int> zsp2(nz);
    for (int k = 0; k < nz; ++k) { zk2[k] = zk[perm[k]]; zsp2[k] = c->v1_zsp[perm[k]]; inv[perm[k]] = k; }
    zk = zk2; c->v1_zsp = zsp2;
    for (auto& m : c->v1_zmap) m = inv[m];
  }
  std::vector<cplx> hz((size_t)Nr * nz * N), hxy((size_t)np * Nr * M * 2 * 2 * N);
  std::vector<double> szv((size_t)Nr * nz), sxy((size_t)np * Nr * M * 2 * 2);
  for (int r = 0; r < Nr; ++r) {
    const double rp = pi * c->rho[r] / c->L;
    for (int k = 0; k < nz; ++k)
      // the job's own kappa stands for every (pair, s, side) mapped to it (they agree to 1e-15)
      split_factor(zk[k] * rp, N, 1.0 / N, &hz[((size_t)r * nz + k) * N], &szv[(size_t)r * nz + k]);
    for (int p = 0; p < ns; ++p) for (int q = 0; q < ns; ++q) {
      const double mu_q = c->mass[q] / (c->mass[p] + c->mass[q]), mu_p = c->mass[p] / (c->mass[p] + c->mass[q]);
      for (int s = 0; s < M; ++s) for (int side = 0; side < 2; ++side) {
        const double kap = side == 0 ? mu_q : -mu_p;
        const size_t e = (((size_t)(p * ns + q) * Nr + r) * M + s) * 2 + side;
        const double wx = (side == 0 ? c->w_sigma[s] : 1.0) / N;
        split_factor(kap * rp * c->sigma[3 * s + 0], N, wx, &hxy[e * 2 * N], &sxy[e * 2]);
        split_factor(kap * rp * c->sigma[3 * s + 1], N, 1.0 / N, &hxy[e * 2 * N + N], &sxy[e * 2 + 1]);
      }
    }
  }
  // R-10, same-species VHS pairs: mu_q = mu_p = 1/2 and f_p = f_q, so the antipode s' of a sphere point s swaps
  // the two shifted fields, A_s' = B_s and B_s' = A_s, and A_s' B_s' = A_s B_s exactly.  Only one point of every
  // antipodal couple is run, with weight w_s + w_s' (the weight sits in the side-A x factors).  The paper's
  // "M points on the half sphere" is this symmetry; it does not hold for p != q (reading S-1).
  c->v1_sskip.assign((size_t)np * M, 0);
  {
    const char* ap = getenv("DGFS_V1_ANTIPODAL");
    const bool on = !(ap && atoi(ap) == 0);
    // which point of a couple runs: the one whose first non-zero component in the order (z, x, y) is positive, so that
    // the points kept are (sx, +-sy, sz) couples wherever the rule has them: they share their inverse x pass (R-12)
    auto runs_first = [&](int a) {
      for (int d : {2, 0, 1}) if (c->sigma[3 * a + d] != 0.0) return c->sigma[3 * a + d] > 0.0;
      return true;
    };
    for (int p = 0; on && p < ns; ++p) {
      const int pair = p * ns + p;
      if (c->full[pair]) continue;
      for (int s2 = 0; s2 < M; ++s2) {
        if (c->v1_sskip[(size_t)pair * M + s2]) continue;
        for (int s3 = s2 + 1; s3 < M; ++s3) {
          if (c->v1_sskip[(size_t)pair * M + s3]) continue;
          if (c->sigma[3 * s3] == -c->sigma[3 * s2] && c->sigma[3 * s3 + 1] == -c->sigma[3 * s2 + 1] &&
              c->sigma[3 * s3 + 2] == -c->sigma[3 * s2 + 2]) {
            const int keep = runs_first(s2) ? s2 : s3, drop = keep == s2 ? s3 : s2;
            c->v1_sskip[(size_t)pair * M + drop] = 1;
            const double fac = (c->w_sigma[s2] + c->w_sigma[s3]) / c->w_sigma[keep];
            for (int r = 0; r < Nr; ++r) {
              const size_t e = (((size_t)pair * Nr + r) * M + keep) * 2;        // side A
              for (int j = 0; j < N; ++j) { hxy[e * 2 * N + j].x *= fac; hxy[e * 2 * N + j].y *= fac; }
              sxy[e * 2] *= fac;
            }
            break;
          }
        }
      }
    }
  }
  // R-11, VHS pairs (p,q) and (q,p): the antipode exchanges their shifted fields, A'_s' = B_s and B'_s' = A_s, so
  // their products agree point by point on the sphere, and when every point has an antipode of the SAME weight
  // the sums S_r^(qp) = S_r^(pq) agree too.  (q,p), q > p, then runs no plane job at all: its forward z pass reads
  // the buffer of (p,q) and applies its own b_r.
  c->v1_tsrc.resize(np);
  for (int pr = 0; pr < np; ++pr) c->v1_tsrc[pr] = pr;
  {
    const char* ap = getenv("DGFS_V1_ANTIPODAL");
    bool sym = !(ap && atoi(ap) == 0);
    for (int s2 = 0; sym && s2 < M; ++s2) {
      bool found = false;
      for (int s3 = 0; s3 < M && !found; ++s3)
        found = c->sigma[3 * s3] == -c->sigma[3 * s2] && c->sigma[3 * s3 + 1] == -c->sigma[3 * s2 + 1] &&
                c->sigma[3 * s3 + 2] == -c->sigma[3 * s2 + 2] && c->w_sigma[s3] == c->w_sigma[s2];
      sym = found;
    }
    for (int p = 0; sym && p < ns; ++p)
      for (int q = p + 1; q < ns; ++q) {
        if (c->full[p * ns + q] || c->full[q * ns + p]) continue;
        c->v1_tsrc[q * ns + p] = p * ns + q;
        for (int s2 = 0; s2 < M; ++s2) c->v1_sskip[(size_t)(q * ns + p) * M + s2] = 1;
      }
  }
  // The same two symmetries for pairs with a full table b_rs: the products agree, P_s' = (w_s' / w_s) P_s, but b_rs'
  // differs from b_rs, so every (pair, s) keeps its own multiply-accumulate in k_zfwd_full and only the plane jobs
  // and their forward x,y passes are shared: (p,p) runs one point per antipodal couple, (q,p) runs none.
  c->v1_fsrc_s.resize((size_t)np * M);
  c->v1_fscale.assign((size_t)np * M, 1.0);
  for (int pr = 0; pr < np; ++pr) for (int s2 = 0; s2 < M; ++s2) c->v1_fsrc_s[(size_t)pr * M + s2] = s2;
  {
    const char* ap = getenv("DGFS_V1_ANTIPODAL");
    bool all = !(ap && atoi(ap) == 0);
    std::vector<int>& anti = c->v1_anti;
    anti.assign(M, -1);
    c->v1_tpartner.assign(np, -1);
    for (int s2 = 0; s2 < M; ++s2) {
      for (int s3 = 0; s3 < M; ++s3)
        if (c->sigma[3 * s3] == -c->sigma[3 * s2] && c->sigma[3 * s3 + 1] == -c->sigma[3 * s2 + 1] &&
            c->sigma[3 * s3 + 2] == -c->sigma[3 * s2 + 2]) { anti[s2] = s3; break; }
      if (anti[s2] < 0) all = false;
    }
    for (int p = 0; all && p < ns; ++p) {
      const int dp = p * ns + p;
      if (c->full[dp])
        for (int s2 = 0; s2 < M; ++s2) {
          const int s3 = anti[s2];
          if (s3 > s2) {                    // s2 runs, s3 reads its buffer
            c->v1_sskip[(size_t)dp * M + s3] = 1;
            c->v1_fsrc_s[(size_t)dp * M + s3] = s2;
            c->v1_fscale[(size_t)dp * M + s3] = c->w_sigma[s3] / c->w_sigma[s2];
          }
        }
      for (int q = p + 1; q < ns; ++q) {
        const int pq = p * ns + q, qp = q * ns + p;
        if (!c->full[pq] || !c->full[qp]) continue;
        c->v1_tsrc[qp] = pq;
        c->v1_tpartner[pq] = qp;
        for (int s2 = 0; s2 < M; ++s2) {
          c->v1_sskip[(size_t)qp * M + s2] = 1;
          c->v1_fsrc_s[(size_t)qp * M + s2] = anti[s2];
          c->v1_fscale[(size_t)qp * M + s2] = c->w_sigma[s2] / c->w_sigma[anti[s2]];
        }
      }
    }
  }
  // sphere points with a vanishing component (every point of the octahedron and of the icosahedron has one):
  // sin(0) = 0, so that axis contributes no anti-Hermitian part at all
  c->v1_smask.assign(M, 0);
  for (int s2 = 0; s2 < M; ++s2)
    for (int d = 0; d < 3; ++d)
      if (c->sigma[3 * s2 + d] == 0.0) c->v1_smask[s2] |= (unsigned char)(1 << d);
  // The plane jobs of every pair as a list the kernels walk without further look-ups, ordered in GROUPS of up to two
  // sphere points that share their z jobs and their x factors on both sides (equal sigma_z and sigma_x: the points
  // (sx, +-sy, sz) of the built-in rules): the inverse x pass of such points is the same transform of the same data
  // and runs once per group (R-12, k_xy).  .w = smask | JOB_FIRST (opens a group) | JOB_LAST (closes it) | JOB_SLOT.
  c->v1_jobs.assign((size_t)np * M, make_int4(0, 0, 0, 0));
  c->v1_njobs.assign(np, 0);
  c->v1_xyflops.assign(np, 0.0);
  {
    const char* gp = getenv("DGFS_V1_XSHARE");
    const bool share = !(gp && atoi(gp) == 0) && N <= 32;       // the N = 48 job (collide_v1_wide.cuh) runs every x pass
    const double fft1 = 5.0 * N * log2((double)N);
    for (int pr = 0; pr < np; ++pr) {
      if (c->v1_tsrc[pr] != pr) continue;
      std::vector<int> run;
      for (int s2 = 0; s2 < M; ++s2) if (!c->v1_sskip[(size_t)pr * M + s2]) run.push_back(s2);
      std::vector<char> used(run.size(), 0);
      auto zj = [&](int s2, int side) { return c->v1_zmap[((size_t)pr * M + s2) * 2 + side]; };
      auto same_x = [&](int s2, int s3) {            // x factors (weights folded in) of both sides, every radial node
        if (c->sigma[3 * s2] != c->sigma[3 * s3]) return false;
        for (int r = 0; r < Nr; ++r) for (int side = 0; side < 2; ++side) {
          const size_t e2 = ((((size_t)pr * Nr + r) * M + s2) * 2 + side), e3 = ((((size_t)pr * Nr + r) * M + s3) * 2 + side);
          if (sxy[e2 * 2] != sxy[e3 * 2]) return false;
          for (int j = 0; j < N; ++j)
            if (hxy[e2 * 2 * N + j].x != hxy[e3 * 2 * N + j].x || hxy[e2 * 2 * N + j].y != hxy[e3 * 2 * N + j].y) return false;
        }
        return true;
      };
      auto push = [&](int s2, int flags) {
        c->v1_jobs[(size_t)pr * M + c->v1_njobs[pr]++] = make_int4(s2, zj(s2, 0), zj(s2, 1), c->v1_smask[s2] | flags);
        // flops of this job's y pass, factor, packing adds, product, Nyquist fixes; the x pass is counted per group
        c->v1_xyflops[pr] += N * (N * fft1 + ((c->v1_smask[s2] & 2) ? 2.0 : 6.0) * N * N + 4.0 * N * N + 12.0 * N);
        if (flags & JOB_FIRST) c->v1_xyflops[pr] += N * (N * fft1 + ((c->v1_smask[s2] & 1) ? 0.0 : 6.0) * N * N);
      };
      for (size_t i = 0; i < run.size(); ++i) {
        if (used[i]) continue;
        used[i] = 1;
        size_t mate = run.size();
        for (size_t k = i + 1; share && k < run.size() && mate == run.size(); ++k)
          if (!used[k] && zj(run[k], 0) == zj(run[i], 0) && zj(run[k], 1) == zj(run[i], 1) && same_x(run[i], run[k])) mate = k;
        if (mate < run.size()) {
          used[mate] = 1;
          push(run[i], JOB_FIRST);
          push(run[mate], JOB_LAST | JOB_SLOT);
        } else push(run[i], JOB_FIRST | JOB_LAST);
      }
      c->v1_xyflops[pr] += N * (N + 1.0) * fft1;       // forward y, x passes of the real plane, once per plane
    }
  }
  int rc;
  if ((rc = upload(c, &c->d_v1_jobs, c->v1_jobs, "upload job lists"))) return rc;
  if ((rc = upload(c, &c->d_v1_njobs, c->v1_njobs, "upload job counts"))) return rc;
  if ((rc = upload(c, &c->d_v1_smask, c->v1_smask, "upload sphere masks"))) return rc;
  if ((rc = upload(c, &c->d_v1_sskip, c->v1_sskip, "upload antipode masks"))) return rc;
  if ((rc = upload(c, &c->d_v1_tsrc, c->v1_tsrc, "upload pair sources"))) return rc;
  if ((rc = upload(c, &c->d_v1_fsrc_s, c->v1_fsrc_s, "upload product sources"))) return rc;
  if ((rc = upload(c, &c->d_v1_fscale, c->v1_fscale, "upload product scales"))) return rc;
  if ((rc = upload(c, &c->d_v1_anti, c->v1_anti, "upload antipodes"))) return rc;
  if ((rc = upload(c, &c->d_v1_tpartner, c->v1_tpartner, "upload pair partners"))) return rc;
  if ((rc = upload(c, &c->d_v1_zsp, c->v1_zsp, "upload z-job species"))) return rc;
  if ((rc = upload(c, &c->d_v1_zmap, c->v1_zmap, "upload z-job map"))) return rc;
  if ((rc = upload(c, &c->d_v1_hz, hz, "upload z factors"))) return rc;
  if ((rc = upload(c, &c->d_v1_szv, szv, "upload z scalars"))) return rc;
  if ((rc = upload(c, &c->d_v1_hxy, hxy, "upload x,y factors"))) return rc;
  if (c->precision == 1) {
    std::vector<cplxf> hxyf(hxy.size());
    for (size_t i = 0; i < hxy.size(); ++i) hxyf[i] = make_float2((float)hxy[i].x, (float)hxy[i].y);
    if ((rc = upload(c, &c->d_v1_hxyf, hxyf, "upload x,y factors (fp32)"))) return rc;
  }
  if ((rc = upload(c, &c->d_v1_sxy, sxy, "upload x,y scalars"))) return rc;
  V1Tables& t = c->v1;
  t.nz = nz; t.zsp = c->d_v1_zsp; t.zmap = c->d_v1_zmap; t.hz = c->d_v1_hz; t.szv = c->d_v1_szv;
  t.hxy = c->d_v1_hxy; t.hxyf = c->d_v1_hxyf; t.sxy = c->d_v1_sxy; t.smask = c->d_v1_smask; t.sskip = c->d_v1_sskip; t.tsrc = c->d_v1_tsrc; t.fsrc_s = c->d_v1_fsrc_s; t.fscale = c->d_v1_fscale; t.anti = c->d_v1_anti; t.tpartner = c->d_v1_tpartner;
  t.jobs = c->d_v1_jobs; t.njobs = c->d_v1_njobs;
  return DGFS_OK;
}

void free_tables_v1(dgfs_ctx* c) {
  cudaFree(c->d_v1_zsp); cudaFree(c->d_v1_zmap); cudaFree(c->d_v1_hz); cudaFree(c->d_v1_szv);
  cudaFree(c->d_v1_hxy); cudaFree(c->d_v1_sxy); cudaFree(c->d_v1_smask); cudaFree(c->d_v1_sskip); cudaFree(c->d_v1_tsrc); cudaFree(c->d_v1_fsrc_s); cudaFree(c->d_v1_fscale); cudaFree(c->d_v1_anti); cudaFree(c->d_v1_tpartner);
  cudaFree(c->d_v1_jobs); cudaFree(c->d_v1_njobs); cudaFree(c->d_v1_hxyf);
}

// ---------------------------------------------------------------- device code -------------------
// Half-packed spectrum (R-7): f^ of a real field is Hermitian, so columns ly = 0 .. H-1 suffice when
// column 0 carries column H in its imaginary unit:  fhh[lz][lx][m] = f^(lx, m, lz) for m >= 1,
// f^(lx, 0, lz) + i f^(lx, H, lz) for m = 0.  Both packed columns are spectra (in lx, lz) of real
// fields, so they separate again as Re / Im once the x and z transforms are done.
template <int N>
__global__ void __launch_bounds__(256) k_pack_half(const cplx* __restrict__ fhat, cplx* __restrict__ fhh,
                                                   cplx* __restrict__ nyqy, int narr) {
  constexpr int H = N / 2;
  const size_t total = (size_t)narr * N * N * H;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int m = (int)(i % H);
    const size_t row = i / H;                       // (array, lz, lx)
    cplx v = fhat[row * N + m];
    if (m == 0) { cplx w = fhat[row * N + H]; v.x -= w.y; v.y += w.x; }
    fhh[i] = v;
  }
  // the ly = H plane, half-packed along lx:  nyqy[arr][lz][m] = f^(m, H, lz), m = 0 carrying f^(H, H, lz)
  const size_t total2 = (size_t)narr * N * H;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total2; i += (size_t)gridDim.x * blockDim.x) {
    const int m = (int)(i % H);
    const size_t pl = i / H;                        // (array, lz)
    cplx v = fhat[(pl * N + m) * N + H];
    if (m == 0) { cplx w = fhat[(pl * N + H) * N + H]; v.x -= w.y; v.y += w.x; }
    nyqy[i] = v;
  }
}

// 16-byte asynchronous copy global -> shared (LDGSTS): the data of the next plane job lands in shared
// memory while the warp is still in the FFTs of the current one, without holding registers.
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sa), "l"(gmem));
}
__device__ __forceinline__ void cp_async_el(cplx* smem, const cplx* gmem) { cp_async16(smem, gmem); }
__device__ __forceinline__ void cp_async_el(cplxf* smem, const cplxf* gmem) { cp_async8(smem, gmem); }
template <class C> __device__ __forceinline__ C cvt(cplx v) { return mkc<C>((typename real_of<C>::type)v.x, (typename real_of<C>::type)v.y); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait_pending() { asm volatile("cp.async.wait_group %0;\n" ::"n"(PENDING) : "memory"); }

// Bulk asynchronous copy global -> shared by the TMA unit (cp.async.bulk; SASS UBLKCP): ONE thread issues a copy of
// a contiguous run (16-byte aligned, a multiple of 16 bytes) and the bytes are counted on an mbarrier in shared
// memory; the consumers wait on the barrier's phase parity.  No per-thread address arithmetic, no registers in flight.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* smem, const void* gmem, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(smem)),
               "l"(gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }

// Inverse z pass of h_z f^ for the z jobs k0 .. k0 + nk - 1 of point blockIdx.z that shift species blockIdx.y;
// thread per (lx, m) pencil.  The block's 128 pencils of the half-packed spectrum are read ONCE into shared memory
// (every job of a species starts from the same spectrum: 8 jobs per species and radial node at c2) and each job
// multiplies, transforms in registers and stores its own array.
// in: fhh[xl][species][lz][lx][m];  out: Gz[xl][k - kbase][cz][lx][m], kstride arrays per point (the jobs that depend
// on the radial node and the sigma_z = 0 jobs, which do not, live in separate buffers: GzView below).
template <int N, class CO>
__global__ void __launch_bounds__(128, N > 32 ? 2 : 3) k_zshift(V1Tables t, int ns, const cplx* __restrict__ fhh, CO* __restrict__ Gz, int r, int k0, int nk,
                                                   int kbase, int kstride) {
  constexpr int H = N / 2, NP = N * H;
  extern __shared__ cplx sm[];                       // [lz][128]
  const int pid = blockIdx.x * 128 + threadIdx.x;
  const int sp = blockIdx.y, xl = blockIdx.z;
  int first = k0;
  while (first < k0 + nk && t.zsp[first] != sp) ++first;
  if (first == k0 + nk) return;                      // no job of this launch shifts this species (uniform)
  const bool live = pid < NP;
  if (live) {
    const cplx* src = fhh + ((size_t)xl * ns + sp) * (size_t)(N * NP) + pid;
#pragma unroll
    for (int i = 0; i < N; ++i) cp_async16(&sm[i * 128 + threadIdx.x], src + (size_t)i * NP);
  }
  cp_async_commit();
  cp_async_wait_all();                               // each thread reads back only what it copied itself
  if (!live) return;
  for (int k = first; k < k0 + nk; ++k) {
    if (t.zsp[k] != sp) continue;
    const cplx* hz = t.hz + ((size_t)r * t.nz + k) * N;
    cplx v[N];
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = cmul(sm[i * 128 + threadIdx.x], __ldg(&hz[i]));
    fft_reg<N, +1>(v);
    CO* dst = Gz + ((size_t)xl * kstride + (k - kbase)) * (size_t)(N * NP) + pid;      // CO = float2: precision 1
#pragma unroll
    for (int i = 0; i < N; ++i) dst[(size_t)i * NP] = cvt<CO>(v[i]);
  }
}

// Where the z-shifted arrays of a chunk live: jobs 0 .. nzr-1 depend on the radial node (double-buffered, one buffer
// per radial node in flight), jobs nzr .. nz-1 (sigma_z = 0) are written once per chunk.
template <class C>
struct GzViewT {
  const C* r;                // [xl][nzr][cz][lx][m]
  const C* z0;               // [xl][nz - nzr][cz][lx][m]
  int nzr, nz0;
  __device__ __forceinline__ const C* job(int xl, int k, size_t arr) const {
    return k < nzr ? r + ((size_t)xl * nzr + k) * arr : z0 + ((size_t)xl * nz0 + (k - nzr)) * arr;
  }
};
typedef GzViewT<cplx> GzView;

// Per-warp shared memory of a plane job: the N x (N+1) tile (input columns, then the transposition) and
// the job's small tables.
template <int N>
struct JobSmem {
  static constexpr int P = N + 1;
  static constexpr int TILE = N * P;
  static constexpr int TS = N + 1;           // stride between the two sides' tables: the half warps read different banks
  static constexpr int HI = TILE;            // [2][TS]  factor along the pass-1 index, per side
  static constexpr int HM = TILE + 2 * TS;   // [2][TS]  factor along the pass-2 index, per side
  static constexpr int VYH = TILE + 4 * TS;  // [N]     lane format
  static constexpr int VXP = VYH + N;        // [N]
  static constexpr int VZP = VXP + N;        // [1]
  static constexpr int WORDS = VZP + 2;
};

// 1-D Nyquist corrections of one (item, s) per warp (file header: the s s h, s h s, h s s and s s s terms):
//   vyh[(side, m)] = s_x s_z f^(H, m, H)                 row lx = H of plane lz = H, lane format, y factor not applied
//   vxp[cx] = sum_lx e^{2 pi i lx cx / N} h_x s_y s_z f^(lx, H, H)      vzp[cz] = sum_lz e^{..} s_x s_y h_z f^(H, H, lz)
//   vt = s_x s_y s_z f^(H, H, H)                         all packed (side A) + i (side B)
template <int N>
__global__ void __launch_bounds__(128) k_nyq1d(V1Tables t, DevTables tab, const cplx* __restrict__ fhat,
                                               cplx* __restrict__ nyq, int r, int njobs) {
  constexpr int H = N / 2, N2 = N * N, N3 = N2 * N;
  typedef NyqLayout<N> NL;
  __shared__ cplx sm1[4][3 * N];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int job = blockIdx.x * 4 + warp;
  if (job >= njobs) return;
  const int s = job % tab.M, item = job / tab.M;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  if (t.sskip[(size_t)pair * tab.M + s]) return;           // the antipode carries this point (R-10)
  const int p = pair / tab.ns, q = pair % tab.ns;
  const cplx* FA = fhat + ((size_t)xl * tab.ns + p) * N3;
  const cplx* FB = fhat + ((size_t)xl * tab.ns + q) * N3;
  const size_t e = (((size_t)pair * tab.N_rho + r) * tab.M + s) * 2;
  const cplx *hxA = t.hxy + e * 2 * N, *hxB = hxA + 2 * N;
  const double sxA = t.sxy[e * 2], syA = t.sxy[e * 2 + 1], sxB = t.sxy[e * 2 + 2], syB = t.sxy[e * 2 + 3];
  const int kA = t.zmap[((size_t)pair * tab.M + s) * 2], kB = t.zmap[((size_t)pair * tab.M + s) * 2 + 1];
  const cplx *hzA = t.hz + ((size_t)r * t.nz + kA) * N, *hzB = t.hz + ((size_t)r * t.nz + kB) * N;
  const double szA = t.szv[(size_t)r * t.nz + kA], szB = t.szv[(size_t)r * t.nz + kB];
  cplx* out = nyq + ((size_t)item * tab.M + s) * NL::STRIDE;
  auto pack = [](cplx fa, cplx ha, double sa, cplx fb, cplx hb, double sb) {
    cplx a = cmul(fa, ha), b = cmul(fb, hb);
    return make_double2(sa * a.x - sb * b.y, sa * a.y + sb * b.x);
  };
  cplx* roots = sm1[warp];         // e^{2 pi i k / N}
  cplx* inx = roots + N;
  cplx* inz = roots + 2 * N;
  const size_t iy = (size_t)H * N2 + H * N;
  for (int k = lane; k < N; k += 32) {
    double sn, cs; sincospi(2.0 * k / N, &sn, &cs);
    roots[k] = make_double2(cs, sn);
    const size_t ix = (size_t)H * N2 + k * N + H, iz = (size_t)k * N2 + H * N + H;
    inx[k] = pack(FA[ix], hxA[k], syA * szA, FB[ix], hxB[k], syB * szB);
    inz[k] = pack(FA[iz], hzA[k], sxA * syA, FB[iz], hzB[k], sxB * syB);
    const int side = k / H, m = k % H;
    const cplx* F = side ? FB : FA;
    const double sc = side ? sxB * szB : sxA * szA;
    cplx v = F[iy + m];
    if (m == 0) v = make_double2(v.x, F[iy + H].x);
    out[NL::VYH + k] = make_double2(sc * v.x, sc * v.y);
  }
  if (lane == 0) out[NL::VT] = make_double2(sxA * syA * szA * FA[iy + H].x, sxB * syB * szB * FB[iy + H].x);
  __syncwarp();
  for (int c = lane; c < N; c += 32) {
    cplx ax = make_double2(0, 0), az = make_double2(0, 0);
    for (int l = 0; l < N; ++l) {
      const cplx w = roots[(l * c) % N];
      ax = cfma(inx[l], w, ax);
      az = cfma(inz[l], w, az);
    }
    out[NL::VXP + c] = ax;
    out[NL::VZP + c] = az;
  }
}

// Pass 1 of a plane job (lane = (side, m), column m of the Hermitian half): multiply by the factor along
// the pass-1 index, inverse transform in registers, factor of the lane's own column, back into the tile.
template <int N, bool CORR, class C>
__device__ __forceinline__ void job_pass1(C* buf, int ln, int side, int m, typename real_of<C>::type szs,
                                          typename real_of<C>::type scale, C c1, bool unit_i = false, bool real_m = false) {
  typedef JobSmem<N> JS;
  typedef typename real_of<C>::type R;
  constexpr int H = N / 2, P = JS::P;
  C v[N];
  if (unit_i) {
    // theta = 0 along the pass-1 axis: the factor is the same real number for every index; the caller has
    // folded it into `scale` (warp-uniform branch)
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = buf[i * P + ln];
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = cmul(buf[i * P + ln], buf[JS::HI + side * JS::TS + i]);
  }
  if (CORR) {            // c1: the x-Nyquist row correction of this lane's column (NyqLayout::VYH)
    v[H].x = fma_(-szs, c1.x, v[H].x);
    v[H].y = fma_(-szs, c1.y, v[H].y);
  }
  fft_reg<N, +1>(v);
  // complex h[m] for m >= 1; for the packed lane m = 0 the real h[0], h[H] scale Re (column 0) and
  // Im (column H) separately
  const C hy0 = buf[JS::HM + side * JS::TS + m];
  const R hyH = buf[JS::HM + side * JS::TS + H].x;
  const R ya = scale * hy0.x, yb = (m == 0) ? (R)0 : -scale * hy0.y, yc = (m == 0) ? (R)0 : scale * hy0.y,
          yd = (m == 0) ? scale * hyH : scale * hy0.x;
  if (real_m) {
    // theta = 0 along the pass-2 axis: every h[m] is the same real number (yb = yc = 0)
#pragma unroll
    for (int i = 0; i < N; ++i) buf[i * P + ln] = mkc<C>(v[i].x * ya, v[i].y * yd);
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i)
      buf[i * P + ln] = mkc<C>(fma_(v[i].x, ya, v[i].y * yb), fma_(v[i].x, yc, v[i].y * yd));
  }
}

// Input of pass 2 (lane = pass-1 output index): the N packed columns X = Y_A + i Y_B, the mirror half by
// conjugation (Y_A, Y_B are Hermitian along the pass-2 index).  vx, vz: the y-Nyquist column and (H,H) element
// corrections of this lane / plane (NyqLayout::VXP, VZP).
template <int N, bool CORR, class C>
__device__ __forceinline__ void job_pass2_in(const C* buf, int ln, typename real_of<C>::type szs,
                                             typename real_of<C>::type sxb, C vx, C vz, C (&X)[N]) {
  typedef JobSmem<N> JS;
  constexpr int H = N / 2, P = JS::P;
  const C* row = buf + ln * P;
  const C a0 = row[0], b0 = row[H];
  X[0] = mkc<C>(a0.x, b0.x);
  X[H] = mkc<C>(a0.y, b0.y);
  if (CORR) {
    X[H].x -= szs * vx.x + sxb * vz.x;
    X[H].y -= szs * vx.y + sxb * vz.y;
  }
#pragma unroll
  for (int mm = 1; mm < H; ++mm) {
    const C ya = row[mm], yb = row[H + mm];
    X[mm] = mkc<C>(ya.x - yb.y, ya.y + yb.x);
    X[N - mm] = mkc<C>(ya.x + yb.y, yb.x - ya.y);
  }
}

// The three Nyquist-plane fields of every (item, s): block (which, item), warp w of NW runs s = w, w + NW, ...
//   which 0: uz[cy][cx]  = ifft_xy[ h_x h_y s_z f^(., ., H) ]     pass 1 over lx, pass 2 over ly
//   which 1: uxp[cy][cz] = ifft_yz[ s_x h_y h_z f^(H, ., .) ] - (-1)^{cy+cz} vt     pass 1 over lz, pass 2 over ly
//   which 2: uy[cx][cz]  = ifft_xz[ h_x s_y h_z f^(., H, .) ]     pass 1 over lz, pass 2 over lx
// each a plane job on the Hermitian half (from fhh / nyqy), packed (side A) + i (side B).
template <int N, int NW>
__global__ void __launch_bounds__(32 * NW) k_nyq2(V1Tables t, DevTables tab, const cplx* __restrict__ fhh,
                                              const cplx* __restrict__ nyqy, cplx* __restrict__ nyq, int r) {
  constexpr int H = N / 2, NH = N * H;
  typedef NyqLayout<N> NL;
  typedef JobSmem<N> JS;
  constexpr int P = JS::P;
  extern __shared__ cplx sm[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int which = blockIdx.x, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  const int sp[2] = {pair / tab.ns, pair % tab.ns};
  cplx* buf = sm + (size_t)warp * JS::WORDS;
  const bool act = lane < N;
  const int ln = act ? lane : 0;
  const int side = ln / H, m = ln % H;
  // half plane of this lane's side: element (i, m) at src[i * istride + m]
  const cplx* src;
  int istride;
  if (which == 0) { src = fhh + ((size_t)xl * tab.ns + sp[side]) * (size_t)(N * NH) + (size_t)H * NH; istride = H; }
  else if (which == 1) { src = fhh + ((size_t)xl * tab.ns + sp[side]) * (size_t)(N * NH) + (size_t)H * H; istride = NH; }
  else { src = nyqy + ((size_t)xl * tab.ns + sp[side]) * (size_t)NH; istride = H; }
  src += m;
  const int* zm = t.zmap + (size_t)pair * tab.M * 2;
  const cplx* hbase = t.hxy + (((size_t)pair * tab.N_rho + r) * tab.M) * 4 * N;
  const double* sbase = t.sxy + (((size_t)pair * tab.N_rho + r) * tab.M) * 4;
  auto issue = [&](int s) {
    if (act) {
#pragma unroll
      for (int i = 0; i < N; ++i) cp_async16(&buf[i * P + ln], src + (size_t)i * istride);
      const cplx* hx = hbase + (size_t)s * 4 * N;            // [side][x|y][N]
      const cplx* hzA = t.hz + ((size_t)r * t.nz + zm[2 * s]) * N;
      const cplx* hzB = t.hz + ((size_t)r * t.nz + zm[2 * s + 1]) * N;
      const cplx *hiA, *hiB, *hmA, *hmB;
      if (which == 0) { hiA = hx; hiB = hx + 2 * N; hmA = hx + N; hmB = hx + 3 * N; }
      else if (which == 1) { hiA = hzA; hiB = hzB; hmA = hx + N; hmB = hx + 3 * N; }
      else { hiA = hzA; hiB = hzB; hmA = hx; hmB = hx + 2 * N; }
      cp_async16(&buf[JS::HI + ln], hiA + ln);
      cp_async16(&buf[JS::HI + JS::TS + ln], hiB + ln);
      cp_async16(&buf[JS::HM + ln], hmA + ln);
      cp_async16(&buf[JS::HM + JS::TS + ln], hmB + ln);
      if (ln == 0) cp_async16(&buf[JS::VZP], nyq + ((size_t)item * tab.M + s) * NL::STRIDE + NL::VT);
    }
    cp_async_commit();
  };
  auto scale_of = [&](int s) {
    if (which == 0) return t.szv[(size_t)r * t.nz + zm[2 * s + side]];
    return sbase[s * 4 + side * 2 + (which == 1 ? 0 : 1)];
  };
  // fields of an axis with sigma_{s,d} = 0 vanish identically (v1_tables.h): run no job; zeros are stored only for
  // pairs with a full table (k_xy_full reads all three fields; k_wterm skips the masked ones)
  // pairs with a full table: the fields go to k_xy_full in their natural layout [j][lane] (and zeros are stored for the
  // fields that vanish); the other pairs' fields go to k_wterm, de-interleaved / swizzled for its bulk copies
  const bool store_zeros = tab.full[pair] != 0;
  const int zbit = (which == 0) ? 4 : (which == 1 ? 1 : 2);
  const int ooff = (which == 0) ? NL::UZ : (which == 1 ? NL::UXP : NL::UY);
  auto next_job = [&](int s) {                   // first s' >= s in this warp's sequence with a job to run
    const unsigned char* skip = t.sskip + (size_t)pair * tab.M;
    while (s < tab.M && ((t.smask[s] & zbit) || skip[s])) {
      if (act && !skip[s] && store_zeros) {
        cplx* out = nyq + ((size_t)item * tab.M + s) * NL::STRIDE + ooff;
#pragma unroll
        for (int j = 0; j < N; ++j) out[j * N + ln] = make_double2(0.0, 0.0);
      }
      s += NW;
    }
    return s;
  };
  int s = next_job(warp);
  if (s >= tab.M) return;
  issue(s);
  double scale = scale_of(s);
  while (s < tab.M) {
    const int sn = next_job(s + NW);
    cp_async_wait_all();
    __syncwarp();
    cplx X[N];
    if (act) job_pass1<N, false>(buf, ln, side, m, 0.0, scale, make_double2(0.0, 0.0));
    __syncwarp();
    cplx vt = make_double2(0.0, 0.0);
    if (act) { job_pass2_in<N, false>(buf, ln, 0.0, 0.0, make_double2(0.0, 0.0), make_double2(0.0, 0.0), X); vt = buf[JS::VZP]; }
    __syncwarp();
    const double scale_next = (sn < tab.M) ? scale_of(sn) : 0.0;
    if (sn < tab.M) issue(sn);
    if (act) {
      fft_reg<N, +1>(X);
      cplx* out = nyq + ((size_t)item * tab.M + s) * NL::STRIDE;
      if (which == 0) {
#pragma unroll
        for (int j = 0; j < N; ++j) out[NL::UZ + (store_zeros ? j * N + ln : (j * 2 + (ln & 1)) * H + (ln >> 1))] = X[j];
      } else if (which == 1) {
        const double sb = (ln & 1) ? -1.0 : 1.0;
#pragma unroll
        for (int j = 0; j < N; ++j) {
          const double sg = (j & 1) ? -sb : sb;
          out[NL::UXP + j * N + ln] = make_double2(X[j].x - sg * vt.x, X[j].y - sg * vt.y);
        }
      } else {
#pragma unroll
        for (int j = 0; j < N; ++j) out[NL::UY + j * N + (store_zeros ? ln : (ln ^ uy_swz(j)))] = X[j];
      }
    }
    s = sn; scale = scale_next;
  }
}

// The r-loop's main kernel: block (cz group, item), warp w owns the plane cz = blockIdx.x * W + w and runs
// the plane jobs of all s for it, so the sum over s stays in that warp's registers.  Per job:
//   prefetch (cp.async, issued during the previous job): the two half planes Gz_A(., ., cz), Gz_B(., ., cz)
//           into the tile, lane = (side, m) owning column m; the x, y factor tables; the Nyquist corrections
//   pass 1: v[lx] = tile[lx][lane] h_x,side[lx]; inverse x pass in registers; y factor of the lane's column;
//           back into the tile (transposition)
//   pass 2: lane = cx rebuilds the N packed columns X[ly] = Y_A + i Y_B (mirror half by conjugation), inverse
//           y pass: Z = a_r + i b_r;  acc[cy] += Re Z Im Z
// in: S[item][cz][cy][cx] = -sum_s Re W Im W (k_wterm);  out: T[item][cz][kx][ky <= H] = fft_xy of S_r(., ., cz).
// Shared memory of a k_xy warp: the tile, what a GROUP of jobs shares (x factors, x-Nyquist row correction) and what
// each of its up to two jobs owns (y factors, y-Nyquist column correction, (H,H) scalar).
template <int N>
struct GroupSmem {
  static constexpr int P = N + 1;
  static constexpr int TILE = N * P;
  static constexpr int TS = N + 1;
  static constexpr int HI = TILE;             // [2][TS]  x factors per side
  static constexpr int VYH = HI + 2 * TS;     // [N]      lane format
  static constexpr int SLOT = VYH + N;        // per job of the group:
  static constexpr int HM = 0;                //   [2][TS] y factors per side
  static constexpr int VXP = 2 * TS;          //   [N]
  static constexpr int VZP = 2 * TS + N;      //   [1]
  static constexpr int SLOTW = 2 * TS + N + 2;
  static constexpr int WORDS = SLOT + 2 * SLOTW;
};

// Inverse x pass of a group (lane = (side, m), column m of the Hermitian half): x factor, Nyquist row correction,
// transform in registers, back into the tile WITHOUT the y factor (which differs between the jobs of the group).
template <int N, class C>
__device__ __forceinline__ void xpass_group(C* buf, int ln, int side, typename real_of<C>::type szs, C c1, bool unit_i) {
  typedef GroupSmem<N> GS;
  constexpr int H = N / 2, P = GS::P;
  C v[N];
  if (unit_i) {
    // sigma_x = 0: the x factor is the same real number for every index (and the Nyquist correction c1 vanishes)
    const typename real_of<C>::type sc = buf[GS::HI + side * GS::TS].x;
#pragma unroll
    for (int i = 0; i < N; ++i) { const C t = buf[i * P + ln]; v[i] = mkc<C>(t.x * sc, t.y * sc); }
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = cmul(buf[i * P + ln], buf[GS::HI + side * GS::TS + i]);
    v[H].x = fma_(-szs, c1.x, v[H].x);
    v[H].y = fma_(-szs, c1.y, v[H].y);
  }
  fft_reg<N, +1>(v);
#pragma unroll
  for (int i = 0; i < N; ++i) buf[i * P + ln] = v[i];
}

// Input of the y pass of one job of the group (lane = row = x index): the y factors of both sides (hm: [2][TS],
// the same for every lane), the N packed columns
// X = Y_A + i Y_B with the mirror half by conjugation, the Nyquist corrections vx (this lane's), vz.  The tile is only read.
template <int N, class C>
__device__ __forceinline__ void ypass_in(const C* buf, const C* hm, int ln, typename real_of<C>::type szs,
                                         typename real_of<C>::type sxb, C vx, C vz, bool real_y, C (&X)[N]) {
  typedef GroupSmem<N> GS;
  typedef typename real_of<C>::type R;
  constexpr int H = N / 2, P = GS::P;
  const C* row = buf + ln * P;
  const C a0 = row[0], b0 = row[H];
  const R hA0 = hm[0].x, hAH = hm[H].x, hB0 = hm[GS::TS].x, hBH = hm[GS::TS + H].x;
  X[0] = mkc<C>(a0.x * hA0, b0.x * hB0);
  X[H] = mkc<C>(a0.y * hAH - (szs * vx.x + sxb * vz.x), b0.y * hBH - (szs * vx.y + sxb * vz.y));
  if (real_y) {
    // theta_y = 0: every y factor is the same real number per side
#pragma unroll
    for (int mm = 1; mm < H; ++mm) {
      const C ya = row[mm], yb = row[H + mm];
      const C p = mkc<C>(ya.x * hA0, ya.y * hA0), q = mkc<C>(yb.x * hB0, yb.y * hB0);
      X[mm] = mkc<C>(p.x - q.y, p.y + q.x);
      X[N - mm] = mkc<C>(p.x + q.y, q.x - p.y);
    }
  } else {
#pragma unroll
    for (int mm = 1; mm < H; ++mm) {
      const C ha = hm[mm], hb = hm[GS::TS + mm];
      const C p = cmul(row[mm], ha), q = cmul(row[H + mm], hb);
      X[mm] = mkc<C>(p.x - q.y, p.y + q.x);
      X[N - mm] = mkc<C>(p.x + q.y, q.x - p.y);
    }
  }
}

// C = double2: Algorithm 2 in fp64.  C = float2 (dgfs_params::precision = 1): the same job on single-precision copies
// of the z-shifted arrays and factor tables; the Nyquist corrections and S are read in double and converted, T is
// written in double (the forward z pass and everything after it stay fp64).
// PACK (N < 32, e.g. N = 24): the W jobs of a block are dealt out N lanes each over its N W threads (W = 4, N = 24:
// three full warps run four planes) instead of one job per warp with 32 - N lanes idle; the jobs of a block then walk
// their common job list in step, with block barriers in place of warp barriers.
template <int N, int W, class C, bool PACK = false>
__global__ void __launch_bounds__(PACK ? N * W : 32 * W) __maxnreg__(sizeof(C) == 8 ? 128 : (W == 2 ? 200 : 255)) k_xy(V1Tables t, DevTables tab, GzViewT<C> Gz,
                                               const C* __restrict__ hxy, const cplx* __restrict__ nyq, const double* __restrict__ S,
                                               cplx* __restrict__ T, int r) {
  constexpr int H = N / 2, NH = N * H, N2 = N * N;
  constexpr bool F32 = sizeof(C) == sizeof(float2);
  typedef typename real_of<C>::type R;
  typedef NyqLayout<N> NL;
  typedef GroupSmem<N> JS;
  constexpr int P = JS::P;
  static_assert(N <= 32, "one lane per pencil");
  extern __shared__ __align__(16) unsigned char sm_raw[];
  C* sm = reinterpret_cast<C*>(sm_raw);
  const int warp = PACK ? threadIdx.x / N : threadIdx.x >> 5, lane = PACK ? threadIdx.x % N : threadIdx.x & 31;
  const int cz = blockIdx.x * W + warp, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  static_assert(!PACK || N % W == 0, "PACK: every block runs W planes");
  if (cz >= N || tab.full[pair] || t.tsrc[pair] != pair) return;      // R-11: (q,p) uses the buffer of (p,q)
  C* buf = sm + (size_t)warp * JS::WORDS;
  const bool act = lane < N;
  const int ln = act ? lane : 0;
  auto sync = [&]() { if (PACK) __syncthreads(); else __syncwarp(); };
  const int side = ln / H, m = ln % H;
  const R szs = (cz & 1) ? (R)-1 : (R)1;
  const R sxb = (ln & 1) ? (R)-1 : (R)1;
  const size_t goff = (size_t)cz * NH + m;
  const C* hbase = hxy + (((size_t)pair * tab.N_rho + r) * tab.M) * 4 * N;
  const cplx* nbase = nyq + (size_t)item * tab.M * NL::STRIDE;
  // jobs = {s, z job of side A, z job of side B, smask[s] | JOB_*} (V1Tables::jobs), in groups of one or two that
  // share the inverse x pass (R-12); the entries of the next group are fetched a group ahead
  const int4* jl = t.jobs + (size_t)pair * tab.M;
  const int nj = t.njobs[pair];
  // the input of a group (the two half planes, x factors, x-Nyquist row) and the tables of its jobs into the tile
  auto issue = [&](int4 j0, int4 j1, bool two) {
    if (act) {
      const C* g = Gz.job(xl, side ? j0.z : j0.y, (size_t)(N * NH)) + goff;
#pragma unroll
      for (int i = 0; i < N; ++i) cp_async_el(&buf[i * P + ln], g + i * H);
      const C* hx = hbase + (size_t)j0.x * 4 * N;          // [side][x|y][N]
      cp_async_el(&buf[JS::HI + ln], hx + ln);               // h_x side A
      cp_async_el(&buf[JS::HI + JS::TS + ln], hx + 2 * N + ln);   // h_x side B
      if (!F32) cp_async16(reinterpret_cast<cplx*>(buf) + JS::VYH + ln, nbase + (size_t)j0.x * NL::STRIDE + NL::VYH + ln);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (k == 1 && !two) break;
        const int4 jb = k ? j1 : j0;
        C* sl = buf + JS::SLOT + k * JS::SLOTW;
        const C* hy = hbase + (size_t)jb.x * 4 * N;
        cp_async_el(&sl[JS::HM + ln], hy + N + ln);           // h_y side A
        cp_async_el(&sl[JS::HM + JS::TS + ln], hy + 3 * N + ln);   // h_y side B
        if (!F32) {
          const cplx* nq = nbase + (size_t)jb.x * NL::STRIDE;
          cplx* sd = reinterpret_cast<cplx*>(sl);
          cp_async16(&sd[JS::VXP + ln], nq + NL::VXP + ln);
          if (ln == 0) cp_async16(&sd[JS::VZP], nq + NL::VZP + cz);
        }
      }
    }
    cp_async_commit();
  };
  int4 g0 = make_int4(0, 0, 0, 0), g1 = g0;
  bool two = false;
  if (nj > 0) {
    g0 = __ldg(&jl[0]);
    two = !(g0.w & JOB_LAST);
    if (two) g1 = __ldg(&jl[1]);
    issue(g0, g1, two);
  }
  // start from the Nyquist-field product written by k_wterm
  R acc[N];
  {
    const double* w0 = S + ((size_t)item * N + cz) * N2 + ln;
#pragma unroll
    for (int j = 0; j < N; ++j) acc[j] = (R)w0[j * N];
  }
  for (int j = 0; j < nj;) {
    const int jn = j + (two ? 2 : 1);                        // first job of the next group
    int4 n0 = g0, n1 = g1;
    bool ntwo = false;
    if (jn < nj) {
      n0 = __ldg(&jl[jn]);
      ntwo = !(n0.w & JOB_LAST);
      if (ntwo) n1 = __ldg(&jl[jn + 1]);
    }
    cp_async_wait_all();
    sync();
    if (act) {
      // sigma_x = 0: h_x is the constant w_s / N (side A) or 1 / N
      const C c1 = F32 ? cvt<C>(__ldg(nbase + (size_t)g0.x * NL::STRIDE + NL::VYH + ln)) : buf[JS::VYH + ln];
      xpass_group<N>(buf, ln, side, szs, c1, (g0.w & 1) != 0);
    }
    sync();
#pragma unroll 1
    for (int k = 0; k < (two ? 2 : 1); ++k) {
      const int4 jb = k ? g1 : g0;
      const C* sl = buf + JS::SLOT + k * JS::SLOTW;
      C X[N];
      if (act) {
        C c2, c3;
        if (F32) {
          const cplx* nq = nbase + (size_t)jb.x * NL::STRIDE;
          c2 = cvt<C>(__ldg(nq + NL::VXP + ln)); c3 = cvt<C>(__ldg(nq + NL::VZP + cz));
        } else { c2 = sl[JS::VXP + ln]; c3 = sl[JS::VZP]; }
        // sigma_y = 0: h_y is the constant 1 / N
        ypass_in<N>(buf, sl + JS::HM, ln, szs, sxb, c2, c3, (jb.w & 2) != 0, X);
      }
      if (k + 1 == (two ? 2 : 1)) {           // last job of the group: the tile is free, the next group's data arrives
        sync();                               // during this y pass
        if (jn < nj) issue(n0, n1, ntwo);
      }
      if (act) {
        fft_reg<N, +1>(X);
#pragma unroll
        for (int jj = 0; jj < N; ++jj) acc[jj] = fma_(X[jj].x, X[jj].y, acc[jj]);
      }
    }
    j = jn; g0 = n0; g1 = n1; two = ntwo;
  }
  // forward y and x passes of the real plane S_r(., ., cz) (steps 6-7, after R-1)
  if (act) {
    C v[N];
#pragma unroll
    for (int j = 0; j < N; ++j) v[j] = mkc<C>(acc[j], (R)0);
    fft_reg<N, -1>(v);
#pragma unroll
    for (int j = 0; j < N; ++j) buf[j * P + ln] = v[j];          // [ky][cx]
  }
  sync();
  if (act) {
    C v[N];
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = buf[ln * P + i];          // lane = ky
    fft_reg<N, -1>(v);
    // S_r is real: columns ky = 0 .. H determine the rest (Hermitian symmetry), only they are kept
    if (ln <= H) {
      cplx* o = T + ((size_t)item * N + cz) * (size_t)(N * (H + 1)) + ln;
#pragma unroll
      for (int k = 0; k < N; ++k) o[k * (H + 1)] = make_double2((double)v[k].x, (double)v[k].y);         // [cz][kx][ky <= H]
    }
  }
}

// Pairs with a full table b_rs(k) (VSS, table_mode 1): the plane job of every s ends in its own forward
// transform (no sum over s before it, b depends on s), and the complex product A B is needed:
//   P = (a_r b_r - a_i b_i) + i (a_r b_i + a_i b_r),   W = a_i + i b_i from the Nyquist fields (file header).
// Same block / warp mapping and prefetch as k_xy; the warp's shared memory also holds the uz plane and the
// ux', uy columns of the job.  out: Tf[item][s][cz][kx][ky] = fft_xy of P_s(., ., cz).
// The uz plane of a job does not depend on cz: the W warps (planes) of a block share ONE copy, staged a quarter each and
// guarded by two block barriers per job (all warps of a block walk the same job list), instead of one copy per warp: 101
// instead of 150 KB per block at N = 32, i.e. two blocks (eight warps) per SM instead of one.
template <int N>
struct FullSmem {
  typedef JobSmem<N> JS;
  static constexpr bool SHARE = N > 24;         // (N = 24: two blocks per SM either way, and the barriers cost 10 %: one copy per warp)
  static constexpr int UX = JS::WORDS;          // [cy]   ux'(cy, cz)
  static constexpr int UY = UX + N;             // [cx]   uy(cx, cz)
  static constexpr int UZ = UY + N;             // [cy][cx] per warp (not SHARE)
  static constexpr int WORDS = UY + N + (SHARE ? 0 : N * N);      // per warp
  static constexpr int UZW = SHARE ? N * N : 0; // per block: [cy][cx], after the W warps' regions (SHARE)
};
template <int N, int W>
__global__ void __launch_bounds__(32 * W) k_xy_full(V1Tables t, DevTables tab, GzView Gz,
                                                    const cplx* __restrict__ nyq, cplx* __restrict__ Tf, int r) {
  constexpr int H = N / 2, NH = N * H, N2 = N * N, N3 = N2 * N;
  typedef NyqLayout<N> NL;
  typedef JobSmem<N> JS;
  typedef FullSmem<N> FS;
  constexpr int P = JS::P;
  static_assert(N <= 32, "one lane per pencil");
  extern __shared__ cplx sm[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cz = blockIdx.x * W + warp, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  if (cz >= N || !tab.full[pair] || t.tsrc[pair] != pair) return;     // (q,p) reads the products of (p,q)
  cplx* buf = sm + (size_t)warp * FS::WORDS;
  cplx* uzs = FS::SHARE ? sm + (size_t)W * FS::WORDS : buf + FS::UZ;      // the block's (or the warp's) copy of the uz plane
  static_assert(N % W == 0, "every warp of a block has a plane (block barriers in the job loop)");
  auto sync = [&]() { if (FS::SHARE) __syncthreads(); else __syncwarp(); };
  const bool act = lane < N;
  const int ln = act ? lane : 0;
  const int side = ln / H, m = ln % H;
  const double szs = (cz & 1) ? -1.0 : 1.0;
  const double sxb = (ln & 1) ? -1.0 : 1.0;
  const int* zm = t.zmap + (size_t)pair * tab.M * 2;
  const size_t goff = (size_t)cz * NH + m;
  const cplx* hbase = t.hxy + (((size_t)pair * tab.N_rho + r) * tab.M) * 4 * N;
  const cplx* nbase = nyq + (size_t)item * tab.M * NL::STRIDE;
  auto issue = [&](int s) {
    if (act) {
      const cplx* g = Gz.job(xl, zm[2 * s + side], (size_t)(N * NH)) + goff;
#pragma unroll
      for (int i = 0; i < N; ++i) cp_async16(&buf[i * P + ln], g + i * H);
      const cplx* hx = hbase + (size_t)s * 4 * N;          // [side][x|y][N]
      cp_async16(&buf[JS::HI + ln], hx + ln);
      cp_async16(&buf[JS::HI + JS::TS + ln], hx + 2 * N + ln);
      cp_async16(&buf[JS::HM + ln], hx + N + ln);
      cp_async16(&buf[JS::HM + JS::TS + ln], hx + 3 * N + ln);
      const cplx* nq = nbase + (size_t)s * NL::STRIDE;
      cp_async16(&buf[JS::VYH + ln], nq + NL::VYH + ln);
      cp_async16(&buf[JS::VXP + ln], nq + NL::VXP + ln);
      if (ln == 0) cp_async16(&buf[JS::VZP], nq + NL::VZP + cz);
#pragma unroll
      for (int j = FS::SHARE ? warp : 0; j < N; j += FS::SHARE ? W : 1) cp_async16(&uzs[j * N + ln], nq + NL::UZ + j * N + ln);   // (this warp's rows)
      cp_async16(&buf[FS::UX + ln], nq + NL::UXP + ln * N + cz);
      cp_async16(&buf[FS::UY + ln], nq + NL::UY + ln * N + cz);
    }
    cp_async_commit();
  };
  const unsigned char* skip = t.sskip + (size_t)pair * tab.M;
  auto next_s = [&](int s) { while (s < tab.M && skip[s]) ++s; return s; };     // points run for this pair (R-10)
  int s = next_s(0);
  if (s < tab.M) issue(s);
  while (s < tab.M) {
    const int sn = next_s(s + 1);
    cp_async_wait_all();
    sync();                                                // every warp's rows of the uz plane have landed
    cplx X[N];
    if (act) {
      // sigma_x = 0: h_x is the constant w_s / N (side A) or 1 / N; sigma_y = 0: h_y is the constant 1 / N
      const int mk = t.smask[s];
      const bool ux_ = (mk & 1) != 0, ry_ = (mk & 2) != 0;
      job_pass1<N, true>(buf, ln, side, m, szs, ux_ ? buf[JS::HI + side * JS::TS].x : 1.0, buf[JS::VYH + ln], ux_, ry_);
    }
    __syncwarp();
    if (act) {
      job_pass2_in<N, true>(buf, ln, szs, sxb, buf[JS::VXP + ln], buf[JS::VZP], X);
      fft_reg<N, +1>(X);                                   // Z = a_r + i b_r, lane = cx, index = cy
      const cplx uyv = buf[FS::UY + ln];
#pragma unroll
      for (int j = 0; j < N; ++j) {
        const cplx ux = buf[FS::UX + j], uz = uzs[j * N + ln];
        const double syj = (j & 1) ? -1.0 : 1.0;
        const double ai = fma(sxb, ux.x, fma(szs, uz.x, syj * uyv.x));
        const double bi = fma(sxb, ux.y, fma(szs, uz.y, syj * uyv.y));
        const double ar = X[j].x, br = X[j].y;
        X[j] = make_double2(fma(ar, br, -ai * bi), fma(ar, bi, ai * br));
      }
      fft_reg<N, -1>(X);                                   // forward y pass: index = ky
    }
    __syncwarp();                                          // every lane has read its row of the tile
    if (act) {
#pragma unroll
      for (int j = 0; j < N; ++j) buf[j * P + ln] = X[j];          // [ky][cx]
    }
    __syncwarp();
    if (act) {
#pragma unroll
      for (int i = 0; i < N; ++i) X[i] = buf[ln * P + i];          // lane = ky
    }
    sync();                                                // every warp of the block is done with the uz plane
    if (sn < tab.M) issue(sn);                             // tile and tables are free again
    if (act) {
      fft_reg<N, -1>(X);                                   // forward x pass
      cplx* o = Tf + ((size_t)item * tab.M + s) * N3 + (size_t)cz * N2 + ln;
#pragma unroll
      for (int k = 0; k < N; ++k) o[k * N] = X[k];         // [cz][kx][ky]
    }
    s = sn;
  }
}

// Forward z pass and steps 7-8 of the full-table pairs for one radial node, driven by the products that
// were actually computed: block (pencils, SOURCE item).  For every sphere point s the source pair ran,
//   u = fft_z( Tf[item][s][.][kx][ky] )  once, then
//   QG[item]          += w_r b^(pq)_rs  u                      its own term
//   QG[item]          += w_r f b^(pq)_rs' u                    same-species pair: the antipode s' it stands for (R-10)
//   QG[partner item]  += w_r f b^(qp)_rs' u                    the transposed pair, which ran nothing (R-11)
// with f = fscale of the target (ratio of sphere weights).  Thread pair per pencil as in k_zfwd_acc; the sums
// over s stay in registers.  b is read in SPEC layout [r][s][kz][kx][ky].
template <int N>
struct ZaccSmem {
  static constexpr int PB = 64, STAGES = 3, WORDS = N * PB;
};
// The rows of Tf (64 pencils x N values of z per sphere point) are staged in shared memory by cp.async, a ring of three
// stages over the sphere points that ran, as k_zfwd_acc stages the radial nodes of T: the loads of the next two points are
// in flight while the current one is transformed, and both threads of a pencil read each element from the stage.
// One sphere point's contribution for the thread's quarter QTR of the outputs, kz = 4 k + QTR: one radix-4 decimation-in-
// frequency step on the staged row, u_j = (x_j + w^QTR x_{j+Q} + w^{2 QTR} x_{j+2Q} + w^{3 QTR} x_{j+3Q}) W_N^{j QTR}
// (w = -i, Q = N / 4), then a length-Q transform in registers.
template <int N, int QTR>
__device__ __forceinline__ void zfull_quarter(const cplx* __restrict__ src, int PB, const BSweep& b1, const BSweep& b2,
                                              const BSweep& b3, bool sym, bool twin, bool has_partner, double ft, double fp,
                                              cplx (&acc)[N / 4], cplx (&acc2)[N / 4]) {
  constexpr int Q = N / 4, H = N / 2;
  // N <= 24: the sweep over the point's own table is issued first, its L2 round trip runs under the transform (c3: 81.3 ->
  // 72.5 ms per three steps).  Not at N = 32, and not the other two sweeps as well: at the 128-register cap the values
  // are spilled and the kernel gets slower (measured both).
  constexpr bool PRE = N <= 24;
  cplx bo[PRE ? Q : 1];
  if (PRE) {
#pragma unroll
    for (int k = 0; k < Q; ++k) {
      const int iz = 4 * k + QTR, kzs = iz - (iz >= H ? N : 0);
      bo[PRE ? k : 0] = b1.p[(sym ? (long)kzs : (long)iz) * b1.sz];
    }
  }
  cplx u[Q];
#pragma unroll
  for (int j = 0; j < Q; ++j) {
    const cplx x0 = src[j * PB], x1 = src[(j + Q) * PB], x2 = src[(j + 2 * Q) * PB], x3 = src[(j + 3 * Q) * PB];
    cplx v;
    if (QTR == 0) v = cadd(cadd(x0, x2), cadd(x1, x3));
    else if (QTR == 2) v = csub(cadd(x0, x2), cadd(x1, x3));
    else {
      // QTR = 1: x0 - i x1 - x2 + i x3 = (x0 - x2) - i (x1 - x3);  QTR = 3: (x0 - x2) + i (x1 - x3)
      const cplx a = csub(x0, x2), d = csub(x1, x3);
      v = (QTR == 1) ? make_double2(a.x + d.y, a.y - d.x) : make_double2(a.x - d.y, a.y + d.x);
    }
    u[j] = twiddle_mul<N, -1>(v, j * QTR);
  }
  fft_reg<Q, -1>(u);
#pragma unroll
  for (int k = 0; k < Q; ++k) {
    const int iz = 4 * k + QTR, kzs = iz - (iz >= H ? N : 0);
    const long zi = sym ? kzs : iz;
    cplx b = PRE ? bo[PRE ? k : 0] : b1.p[zi * b1.sz];
    if (twin) { const cplx bb = b2.p[zi * b2.sz]; b.x = fma(ft, bb.x, b.x); b.y = fma(ft, bb.y, b.y); }
    acc[k] = cfma(b, u[k], acc[k]);
    if (has_partner) { const cplx b3v = b3.p[zi * b3.sz]; acc2[k] = cfma(make_double2(fp * b3v.x, fp * b3v.y), u[k], acc2[k]); }
  }
}
template <int N>
struct ZfullSmem {
  static constexpr int PB = 64, STAGES = 3, WORDS = N * PB;
};
// The rows of Tf (64 pencils x N values of z per sphere point) are staged in shared memory by cp.async, a ring of three
// stages over the sphere points that ran, as k_zfwd_acc stages the radial nodes of T.  FOUR threads per pencil, each
// with a quarter of the outputs (N / 4 + N / 4 accumulators): ~130 registers, so that enough warps are resident to hide
// the L2 latency of the three sweeps over the b tables (with two threads per pencil and 255 registers, 8 warps per SM,
// every sweep's round trip was exposed).
template <int N, bool FIRST>
__global__ void __launch_bounds__(256, 2) k_zfwd_full(DevTables tab, V1Tables t, const cplx* __restrict__ Tf,
                                                   cplx* __restrict__ QG, size_t qstride, int r) {
  constexpr int Q = N / 4, N2 = N * N, N3 = N2 * N;
  typedef ZfullSmem<N> ZS;
  constexpr int PB = ZS::PB, NS = ZS::STAGES;
  extern __shared__ cplx sm[];
  const int qtr = threadIdx.x >> 6, pl = threadIdx.x & 63;          // warp-uniform quarter
  const int pid0 = blockIdx.x * PB, pid = pid0 + pl;
  const int item = blockIdx.y, pair = item % tab.npairs;
  if (!tab.full[pair] || t.tsrc[pair] != pair) return;      // uniform per block
  const int M = tab.M;
  const int partner = t.tpartner[pair];                 // pair that reads this one's products, or -1
  const unsigned char* skip = t.sskip + (size_t)pair * M;
  // What the loop needs to know about a sphere point (its antipode, the weight ratios, where its three sweeps over the b
  // tables start and how they stride), gathered ONCE per block by one thread per sphere point and kept in shared
  // memory: looked up inside the loop these are chains of four or five dependent global loads per sphere point, and
  // that latency, not the sweeps or the staging, was what the kernel waited for (long scoreboard 6.2 per issue).
  constexpr int MAXJ = 64;
  struct ZJob { int run, twin; double ft, fp; long b1, b2, b3; int m1[3], m2[3], m3[3]; };
  __shared__ ZJob jobs[MAXJ];
  const bool sym = tab.bsym != 0;
  auto sweep_of = [&](int s2, long& base, int (&m)[3]) {
    if (sym) {
      const int4 mm = tab.bmap[s2];
      const long E = N + 1;
      base = (long)r * tab.nref * (E * E * E) + mm.x; m[0] = mm.y; m[1] = mm.z; m[2] = mm.w;
    } else { base = ((long)r * M + s2) * N3; m[0] = N; m[1] = 1; m[2] = N2; }
  };
  auto make_job = [&](int s2) {
    ZJob jb;
    jb.run = !skip[s2];
    const int sa = t.anti[s2];
    jb.twin = jb.run && sa >= 0 && skip[sa] && t.fsrc_s[(size_t)pair * M + sa] == s2;     // same-species pair: s also stands for its antipode
    jb.ft = jb.twin ? t.fscale[(size_t)pair * M + sa] : 0.0;
    jb.fp = (partner >= 0 && sa >= 0) ? t.fscale[(size_t)partner * M + sa] : 0.0;
    sweep_of(s2, jb.b1, jb.m1);
    sweep_of(jb.twin ? sa : s2, jb.b2, jb.m2);
    sweep_of(partner >= 0 && sa >= 0 ? sa : s2, jb.b3, jb.m3);
    return jb;
  };
  for (int s2 = threadIdx.x; s2 < M && s2 < MAXJ; s2 += 256) jobs[s2] = make_job(s2);
  const cplx* bf_own = tab.bfull[pair];
  const cplx* bf_par = tab.bfull[partner >= 0 ? partner : pair];
  __syncthreads();
  auto next_s = [&](int s) { while (s < M && (s < MAXJ ? !jobs[s].run : (bool)skip[s])) ++s; return s; };
  const cplx* tbase = Tf + (size_t)item * M * N3 + pid0;
  auto issue = [&](int s, int slot) {
    cplx* dstb = sm + (size_t)slot * ZS::WORDS;
    const cplx* srcb = tbase + (size_t)s * N3;
#pragma unroll
    for (int q = threadIdx.x; q < N * PB; q += 256) {
      const int jj = q / PB, col = q % PB;
      if (pid0 + col < N2) cp_async16(&dstb[q], srcb + (size_t)jj * N2 + col);
    }
  };
  int s_iss = next_s(0);
#pragma unroll
  for (int k = 0; k < NS - 1; ++k) {
    if (s_iss < M) { issue(s_iss, k); s_iss = next_s(s_iss + 1); }
    cp_async_commit();
  }
  const bool live = pid < N2;
  const int pc = live ? pid : 0;
  // index of the pencil in a table: signed frequencies on the extended grid of the orbit tables, else plain indices
  const int kxu = sym ? sfreq(pc / N, N) : pc / N, kyu = sym ? sfreq(pc % N, N) : pc % N;
  const double scale = tab.w_rho[r];
  cplx acc[Q], acc2[Q];
#pragma unroll
  for (int k = 0; k < Q; ++k) acc[k] = acc2[k] = make_double2(0.0, 0.0);
  for (int s = next_s(0), j = 0; s < M; s = next_s(s + 1), ++j) {
    cp_async_wait_pending<NS - 2>();
    if (s >= MAXJ && threadIdx.x == 0) jobs[s % MAXJ] = make_job(s);      // (M > 64: the slot of a point long done)
    __syncthreads();                            // stage j has landed; the stage of j - 1 is free
    if (s_iss < M) { issue(s_iss, (j + NS - 1) % NS); s_iss = next_s(s_iss + 1); }
    cp_async_commit();
    if (!live) continue;
    const cplx* src = sm + (size_t)(j % NS) * ZS::WORDS + pl;
    const ZJob& jb = jobs[s % MAXJ];                    // read in place (a copy of the struct ends up in local memory)
    const bool twin = jb.twin != 0;
    const double ft = jb.ft, fp = jb.fp;
    const BSweep b1{bf_own + jb.b1 + (long)kxu * jb.m1[0] + (long)kyu * jb.m1[1], (long)jb.m1[2]};
    const BSweep b2{bf_own + jb.b2 + (long)kxu * jb.m2[0] + (long)kyu * jb.m2[1], (long)jb.m2[2]};
    const BSweep b3{bf_par + jb.b3 + (long)kxu * jb.m3[0] + (long)kyu * jb.m3[1], (long)jb.m3[2]};
    switch (qtr) {
      case 0: zfull_quarter<N, 0>(src, PB, b1, b2, b3, sym, twin, partner >= 0, ft, fp, acc, acc2); break;
      case 1: zfull_quarter<N, 1>(src, PB, b1, b2, b3, sym, twin, partner >= 0, ft, fp, acc, acc2); break;
      case 2: zfull_quarter<N, 2>(src, PB, b1, b2, b3, sym, twin, partner >= 0, ft, fp, acc, acc2); break;
      default: zfull_quarter<N, 3>(src, PB, b1, b2, b3, sym, twin, partner >= 0, ft, fp, acc, acc2); break;
    }
  }
  if (!live) return;
  cplx* dst = QG + (size_t)item * qstride + pid;
  cplx* dst2 = QG + (size_t)(item - pair + (partner >= 0 ? partner : pair)) * qstride + pid;
#pragma unroll
  for (int k = 0; k < Q; ++k) {
    const size_t o = (size_t)(4 * k + qtr) * N2;
    const cplx q1 = FIRST ? make_double2(0.0, 0.0) : dst[o];
    dst[o] = make_double2(fma(scale, acc[k].x, q1.x), fma(scale, acc[k].y, q1.y));
    if (partner >= 0) {
      const cplx q2 = FIRST ? make_double2(0.0, 0.0) : dst2[o];
      dst2[o] = make_double2(fma(scale, acc2[k].x, q2.x), fma(scale, acc2[k].y, q2.y));
    }
  }
}

// S(c) = -sum_s Re W_s(c) Im W_s(c),  W_s(c) = (-1)^cx ux'_s(cy,cz) + (-1)^cy uy_s(cx,cz) + (-1)^cz uz_s(cx,cy)
// (W = a_i + i b_i, file header).  Five FP64 instructions per node and sphere point against three tables of N^2
// complex values each: the kernel is bound by how its tables reach the SM, not by arithmetic.  A block of 256 threads
// covers a slab of 8 cy rows of one item, all (cx, cz): in the layouts k_nyq2 writes (first index = the transform's
// register index, second = its lane) the slab's rows of ux'[cy][cz] and uz[cy][cx] and the whole plane uy[cx][cz] are
// three CONTIGUOUS runs, so one thread stages the tables of a sphere point with three bulk copies of the TMA unit
// (cp.async.bulk, completion counted on an mbarrier; a ring of four stages over s).  Round 1 staged them with
// 16-byte cp.async and its per-element address arithmetic took 60 % of the kernel's issue slots (profiles/r02_wterm.md).
// Thread = 2 x 2 tile of (cx, cz) over the slab's 8 rows: every table element serves several nodes and all signs are
// compile-time constants.  Bank conflicts: uz is stored de-interleaved by the parity of cx, uy with its cz index
// XOR-swizzled by (cx / 2) mod 8 (v1_tables.h), so that the 8 lanes of a 128-bit wavefront read 8 different banks.
template <int N>
struct WtermSmem {
  static constexpr int CYB = 8, THREADS = (N / 2) * (N / 2);    // thread = 2 x 2 tile of (cx, cz)
  static constexpr int Y = 0;                       // [cx][cz ^ swz(cx)]      the uy plane
  static constexpr int Z = N * N;                   // [i][parity][H]          uz rows of the slab
  static constexpr int U = N * N + CYB * N;         // [i][cz]                 ux' rows of the slab
  static constexpr int WORDS = N * N + 2 * CYB * N;
  static constexpr int STAGES = N > 32 ? 2 : 4;     // ring depth (N = 32: two blocks per SM, 8 stages in flight per SM)
};

// Arithmetic of one s for the thread's 2 x 2 x 8 nodes (cx = 2 tx + a, cz = 2 tz + b, cy = cy0 + i).  MASK bit d set:
// the field of axis d (ux', uy, uz) is identically zero for this sphere point (V1Tables::smask), neither staged nor read.
template <int N, int MASK>
__device__ __forceinline__ void wterm_rows(const cplx* __restrict__ b_, int tx, int tz, double (&acc)[8][2][2]) {
  typedef WtermSmem<N> WS;
  constexpr int H = N / 2, CYB = WS::CYB;
  constexpr bool HU = !(MASK & 1), HV = !(MASK & 2), HZ = !(MASK & 4);
  const cplx zero = make_double2(0.0, 0.0);
  cplx y[2][2];                                     // uy(cx = 2 tx + a, cz = 2 tz + b)
#pragma unroll
  for (int b = 0; b < 2; ++b)
#pragma unroll
    for (int a = 0; a < 2; ++a) y[b][a] = HV ? b_[WS::Y + (2 * tx + a) * N + ((2 * tz + b) ^ uy_swz(2 * tx + a))] : zero;
  // software pipeline over the rows: the loads of row i + 1 are in flight during the arithmetic of row i
  const cplx* ub = b_ + WS::U + 2 * tz;             // ux'(cy0 + i, cz = 2 tz + b): the same for all lanes of a tz
  const cplx* zb = b_ + WS::Z + tx;                 // uz(cy0 + i, cx = 2 tx + a) at [i][a][tx]
  cplx un[2] = {HU ? ub[0] : zero, HU ? ub[1] : zero}, zn[2] = {HZ ? zb[0] : zero, HZ ? zb[H] : zero};
#pragma unroll
  for (int i = 0; i < CYB; ++i) {
    const cplx u[2] = {un[0], un[1]}, z[2] = {zn[0], zn[1]};
    if (i + 1 < CYB) {
      if (HU) { un[0] = ub[(i + 1) * N]; un[1] = ub[(i + 1) * N + 1]; }
      if (HZ) { zn[0] = zb[(i + 1) * N]; zn[1] = zb[(i + 1) * N + H]; }
    }
#pragma unroll
    for (int b = 0; b < 2; ++b)
#pragma unroll
      for (int a = 0; a < 2; ++a) {
        // signs: the tile starts at even cx, cz; slabs start at even cy
        double wx = 0.0, wy = 0.0;
        if (HU) { wx = a ? -u[b].x : u[b].x; wy = a ? -u[b].y : u[b].y; }
        if (HV) { wx += (i & 1) ? -y[b][a].x : y[b][a].x; wy += (i & 1) ? -y[b][a].y : y[b][a].y; }
        if (HZ) { wx += b ? -z[a].x : z[a].x; wy += b ? -z[a].y : z[a].y; }
        acc[i][b][a] = fma(wx, wy, acc[i][b][a]);
      }
  }
}

template <int N>
__global__ void __launch_bounds__(WtermSmem<N>::THREADS, N > 32 ? 1 : 2) k_wterm(const cplx* __restrict__ nyq, int M, double* __restrict__ S, const unsigned char* __restrict__ full, int npairs,
        const unsigned char* __restrict__ smask, const unsigned char* __restrict__ sskip, const int* __restrict__ tsrc) {
  constexpr int N2 = N * N, N3 = N2 * N, H = N / 2;
  typedef NyqLayout<N> NL;
  typedef WtermSmem<N> WS;
  constexpr int CYB = WS::CYB, NT = WS::THREADS, NS = WS::STAGES;
  extern __shared__ cplx sm[];
  // pairs with a full b table take k_xy_full, transposed pairs reuse the other's S_r (uniform per block)
  if (full[blockIdx.y % npairs] || tsrc[blockIdx.y % npairs] != (int)(blockIdx.y % npairs)) return;
  const int tx = threadIdx.x % H, tz = threadIdx.x / H;
  const bool act = true;
  const int cy0 = blockIdx.x * CYB;
  const cplx* nbase = nyq + (size_t)blockIdx.y * M * NL::STRIDE;
  const unsigned char* skip = sskip + (size_t)(blockIdx.y % npairs) * M;
  // which fields each sphere point has (7: none, or the point is not run for this pair, R-10), once per block in
  // shared memory: the loop below then never waits for a global load before it can issue or branch
  __shared__ unsigned char mk_s[256];
  __shared__ unsigned long long bar[NS];             // one "stage is full" barrier per ring slot
  for (int i = threadIdx.x; i < M && i < 256; i += NT) mk_s[i] = skip[i] ? 7 : smask[i];
  if (threadIdx.x == 0) {
    for (int k = 0; k < NS; ++k) mbar_init(&bar[k], 1);
    fence_mbar_init();
  }
  __syncthreads();
  auto mk = [&](int s) -> int { return s < 256 ? (int)mk_s[s] : (skip[s] ? 7 : (int)smask[s]); };
  auto next_a = [&](int s) { while (s < M && mk(s) == 7) ++s; return s; };      // next point with something to add
  // the tables of sphere point s into ring slot `slot` (thread 0): three contiguous runs; vanishing fields are not staged
  auto issue = [&](int s, int slot) {
    cplx* dst = sm + (size_t)slot * WS::WORDS;
    const cplx* nq = nbase + (size_t)s * NL::STRIDE;
    const int mask = mk(s);
    const unsigned bu = (mask & 1) ? 0u : (unsigned)(CYB * N * sizeof(cplx));
    const unsigned by = (mask & 2) ? 0u : (unsigned)(N2 * sizeof(cplx));
    const unsigned bz = (mask & 4) ? 0u : (unsigned)(CYB * N * sizeof(cplx));
    mbar_expect_tx(&bar[slot], bu + by + bz);
    if (by) tma_bulk_g2s(dst + WS::Y, nq + NL::UY, by, &bar[slot]);
    if (bz) tma_bulk_g2s(dst + WS::Z, nq + NL::UZ + (size_t)cy0 * N, bz, &bar[slot]);
    if (bu) tma_bulk_g2s(dst + WS::U, nq + NL::UXP + (size_t)cy0 * N, bu, &bar[slot]);
  };
  double acc[CYB][2][2];                      // [cy][cz][cx]
#pragma unroll
  for (int i = 0; i < CYB; ++i) acc[i][0][0] = acc[i][0][1] = acc[i][1][0] = acc[i][1][1] = 0.0;
  // ring of NS slots over the points that are run: job j uses slot j % NS; thread 0 keeps NS - 1 jobs in flight
  int s_issue = next_a(0), j_issue = 0;
  if (threadIdx.x == 0) {
    for (int k = 0; k < NS - 1 && s_issue < M; ++k) { issue(s_issue, j_issue % NS); s_issue = next_a(s_issue + 1); ++j_issue; }
  }
  for (int s = next_a(0), j = 0; s < M; s = next_a(s + 1), ++j) {
    mbar_wait(&bar[j % NS], (unsigned)((j / NS) & 1));       // the bulk copies of job j have landed
    __syncthreads();                                          // everyone is done with job j - 1: its slot is free
    if (threadIdx.x == 0 && s_issue < M) { issue(s_issue, j_issue % NS); s_issue = next_a(s_issue + 1); ++j_issue; }
    if (!act) continue;
    const cplx* b_ = sm + (size_t)(j % NS) * WS::WORDS;
    switch (mk(s)) {                                 // uniform over the block
      case 0: wterm_rows<N, 0>(b_, tx, tz, acc); break;
      case 1: wterm_rows<N, 1>(b_, tx, tz, acc); break;
      case 2: wterm_rows<N, 2>(b_, tx, tz, acc); break;
      case 3: wterm_rows<N, 3>(b_, tx, tz, acc); break;
      case 4: wterm_rows<N, 4>(b_, tx, tz, acc); break;
      case 5: wterm_rows<N, 5>(b_, tx, tz, acc); break;
      case 6: wterm_rows<N, 6>(b_, tx, tz, acc); break;
      default: break;
    }
  }
  if (!act) return;
  double* o = S + (size_t)blockIdx.y * N3 + (size_t)(2 * tz) * N2 + (size_t)cy0 * N + 2 * tx;
#pragma unroll
  for (int i = 0; i < CYB; ++i)
#pragma unroll
    for (int b = 0; b < 2; ++b)
      *reinterpret_cast<double2*>(o + (size_t)b * N2 + i * N) = make_double2(-acc[i][b][0], -acc[i][b][1]);
}

// k_wterm with the uy plane of a sphere point fetched ONCE per item: the N / CYB blocks of an item (its cy slabs) form a
// thread-block cluster; block rank 0 issues one bulk copy of the plane with .multicast::cluster, which lands at the same
// shared-memory offset of every block of the cluster and counts its bytes on each block's own mbarrier; every block
// still fetches its own rows of ux' and uz.  A slot is refilled only after EVERY block of the cluster has finished with
// it: the block barrier of k_wterm becomes a cluster barrier, split into arrive (after a job's arithmetic) and wait
// (before the next refill is issued).
__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;\n" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tma_bulk_g2s_mc(void* smem, const void* gmem, unsigned bytes, unsigned long long* bar, unsigned short mask) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1], %2, [%3], %4;\n"
               ::"r"(smem_u32(smem)), "l"(gmem), "r"(bytes), "r"(smem_u32(bar)), "h"(mask) : "memory");
}
template <int N>
__global__ void __launch_bounds__(WtermSmem<N>::THREADS, 2) k_wterm_mc(const cplx* __restrict__ nyq, int M, double* __restrict__ S, const unsigned char* __restrict__ full, int npairs,
        const unsigned char* __restrict__ smask, const unsigned char* __restrict__ sskip, const int* __restrict__ tsrc) {
  constexpr int N2 = N * N, N3 = N2 * N, H = N / 2;
  typedef NyqLayout<N> NL;
  typedef WtermSmem<N> WS;
  constexpr int CYB = WS::CYB, NT = WS::THREADS, NS = WS::STAGES, NC = N / CYB;
  extern __shared__ cplx sm[];
  // uniform per cluster (one item): nothing to do
  if (full[blockIdx.y % npairs] || tsrc[blockIdx.y % npairs] != (int)(blockIdx.y % npairs)) return;
  const int tx = threadIdx.x % H, tz = threadIdx.x / H;
  const unsigned rank = cluster_ctarank();
  const int cy0 = blockIdx.x * CYB;
  const cplx* nbase = nyq + (size_t)blockIdx.y * M * NL::STRIDE;
  const unsigned char* skip = sskip + (size_t)(blockIdx.y % npairs) * M;
  __shared__ unsigned char mk_s[256];
  __shared__ unsigned long long bar[NS];
  for (int i = threadIdx.x; i < M && i < 256; i += NT) mk_s[i] = skip[i] ? 7 : smask[i];
  if (threadIdx.x == 0) {
    for (int k = 0; k < NS; ++k) mbar_init(&bar[k], 1);
    fence_mbar_init();
  }
  __syncthreads();
  cluster_arrive();                                  // every block's barriers exist before anyone multicasts onto them
  cluster_wait();
  auto mk = [&](int s) -> int { return s < 256 ? (int)mk_s[s] : (skip[s] ? 7 : (int)smask[s]); };
  auto next_a = [&](int s) { while (s < M && mk(s) == 7) ++s; return s; };
  auto issue = [&](int s, int slot) {
    cplx* dst = sm + (size_t)slot * WS::WORDS;
    const cplx* nq = nbase + (size_t)s * NL::STRIDE;
    const int mask = mk(s);
    const unsigned bu = (mask & 1) ? 0u : (unsigned)(CYB * N * sizeof(cplx));
    const unsigned by = (mask & 2) ? 0u : (unsigned)(N2 * sizeof(cplx));
    const unsigned bz = (mask & 4) ? 0u : (unsigned)(CYB * N * sizeof(cplx));
    mbar_expect_tx(&bar[slot], bu + by + bz);         // by arrives by multicast from block rank 0
    if (by && rank == 0) tma_bulk_g2s_mc(dst + WS::Y, nq + NL::UY, by, &bar[slot], (unsigned short)((1u << NC) - 1));
    if (bz) tma_bulk_g2s(dst + WS::Z, nq + NL::UZ + (size_t)cy0 * N, bz, &bar[slot]);
    if (bu) tma_bulk_g2s(dst + WS::U, nq + NL::UXP + (size_t)cy0 * N, bu, &bar[slot]);
  };
  double acc[CYB][2][2];
#pragma unroll
  for (int i = 0; i < CYB; ++i) acc[i][0][0] = acc[i][0][1] = acc[i][1][0] = acc[i][1][1] = 0.0;
  int s_issue = next_a(0), j_issue = 0;
  if (threadIdx.x == 0) {
    for (int k = 0; k < NS - 1 && s_issue < M; ++k) { issue(s_issue, j_issue % NS); s_issue = next_a(s_issue + 1); ++j_issue; }
  }
  cluster_arrive();                                  // matches the wait of the first iteration (no job before it)
  for (int s = next_a(0), j = 0; s < M; s = next_a(s + 1), ++j) {
    mbar_wait(&bar[j % NS], (unsigned)((j / NS) & 1));       // the bulk copies of job j have landed
    cluster_wait();                                            // every block of the item is done with job j - 1
    if (threadIdx.x == 0 && s_issue < M) { issue(s_issue, j_issue % NS); s_issue = next_a(s_issue + 1); ++j_issue; }
    const cplx* b_ = sm + (size_t)(j % NS) * WS::WORDS;
    switch (mk(s)) {
      case 0: wterm_rows<N, 0>(b_, tx, tz, acc); break;
      case 1: wterm_rows<N, 1>(b_, tx, tz, acc); break;
      case 2: wterm_rows<N, 2>(b_, tx, tz, acc); break;
      case 3: wterm_rows<N, 3>(b_, tx, tz, acc); break;
      case 4: wterm_rows<N, 4>(b_, tx, tz, acc); break;
      case 5: wterm_rows<N, 5>(b_, tx, tz, acc); break;
      case 6: wterm_rows<N, 6>(b_, tx, tz, acc); break;
      default: break;
    }
    cluster_arrive();
  }
  cluster_wait();                                    // the last arrive; no block leaves while a neighbour still multicasts
  double* o = S + (size_t)blockIdx.y * N3 + (size_t)(2 * tz) * N2 + (size_t)cy0 * N + 2 * tx;
#pragma unroll
  for (int i = 0; i < CYB; ++i)
#pragma unroll
    for (int b = 0; b < 2; ++b)
      *reinterpret_cast<double2*>(o + (size_t)b * N2 + i * N) = make_double2(-acc[i][b][0], -acc[i][b][1]);
}

// Forward z pass and steps 7-8 for a group of nr radial nodes r0 .. r0+nr-1:
//   QGh[item][kz][kx][ky <= H] (+)= sum_r w_r b_r(|k|^2) fft_z( T_r[item][.][kx][ky] ).
// Thread pair per (kx,ky) pencil: parity 0 computes the even kz, parity 1 the odd kz (one radix-2
// decimation-in-frequency step, then a length-N/2 transform in registers), so that the accumulators of
// the whole group stay in registers and QG is touched once per group.  FIRST: store, do not accumulate.
// The rows of T (64 pencils x N values of z per radial node) are staged in shared memory by cp.async, a ring of three
// stages: the loads of the next two radial nodes are in flight while the current one is transformed, without holding
// registers, and every element of T is fetched once (the two threads of a pencil read it from the stage).
template <int N, bool FIRST>
__global__ void __launch_bounds__(128) k_zfwd_acc(DevTables tab, const int* __restrict__ tsrc, const cplx* __restrict__ T,
                                                  size_t slot_stride, cplx* __restrict__ QGh, size_t qstride, int r0, int nr) {
  constexpr int H = N / 2, NPH = N * (H + 1);
  typedef ZaccSmem<N> ZS;
  constexpr int PB = ZS::PB, NS = ZS::STAGES;
  extern __shared__ cplx sm[];
  const int par = threadIdx.x >> 6, pl = threadIdx.x & 63;
  const int pid0 = blockIdx.x * PB, pid = pid0 + pl;
  const int item = blockIdx.y, pair = item % tab.npairs;
  if (tab.full[pair]) return;                                          // uniform per block
  const cplx* tbase = T + (size_t)(item - pair + tsrc[pair]) * (N * NPH) + pid0;   // R-11
  auto issue = [&](int sl) {
    if (sl < nr) {
      cplx* dstb = sm + (size_t)(sl % NS) * ZS::WORDS;
      const cplx* srcb = tbase + (size_t)sl * slot_stride;
#pragma unroll
      for (int q = threadIdx.x; q < N * PB; q += 128) {
        const int jj = q / PB, col = q % PB;
        if (pid0 + col < NPH) cp_async16(&dstb[q], srcb + (size_t)jj * NPH + col);
      }
    }
    cp_async_commit();
  };
#pragma unroll
  for (int sl = 0; sl < NS - 1; ++sl) issue(sl);
  const bool live = pid < NPH;
  const int pc = live ? pid : 0;
  const int kxs = sfreq(pc / (H + 1), N), kys = sfreq(pc % (H + 1), N);
  const int k2xy = kxs * kxs + kys * kys;
  cplx acc[H];
#pragma unroll
  for (int k = 0; k < H; ++k) acc[k] = make_double2(0.0, 0.0);
  for (int sl = 0; sl < nr; ++sl) {
    cp_async_wait_pending<NS - 2>();
    __syncthreads();                            // stage sl has landed; the stage of sl - 1 is free
    issue(sl + NS - 1);
    if (live) {
      const cplx* src = sm + (size_t)(sl % NS) * ZS::WORDS + pl;
      cplx u[H];
      if (par == 0) {
#pragma unroll
        for (int j = 0; j < H; ++j) u[j] = cadd(src[j * PB], src[(j + H) * PB]);
      } else {
#pragma unroll
        for (int j = 0; j < H; ++j) u[j] = twiddle_mul<N, -1>(csub(src[j * PB], src[(j + H) * PB]), j);
      }
      fft_reg<H, -1>(u);
      const double* bv = tab.bvhs + ((size_t)pair * tab.N_rho + r0 + sl) * tab.K2n + k2xy;
      const double scale = tab.w_rho[r0 + sl];
#pragma unroll
      for (int k = 0; k < H; ++k) {
        const int kz = 2 * k + par, kzs = kz - (kz >= H ? N : 0);
        const double b = scale * __ldg(&bv[kzs * kzs]);
        acc[k].x = fma(b, u[k].x, acc[k].x);
        acc[k].y = fma(b, u[k].y, acc[k].y);
      }
    }
  }
  if (!live) return;
  cplx* dst = QGh + (size_t)item * qstride + pid;
#pragma unroll
  for (int k = 0; k < H; ++k) {
    cplx* d = dst + (size_t)(2 * k + par) * NPH;
    if (FIRST) *d = acc[k];
    else { cplx o = *d; *d = make_double2(o.x + acc[k].x, o.y + acc[k].y); }
  }
}

// Step 10, spectral part, from the Hermitian half of QG: inverse x,y passes of QG (job 0) and of
// c^(pq) f^_q (job 1), scaled by 1/N^3.  QG(lx, ly, lz) for ly > H is conj QGh(-lx, -ly, -lz).
// out: G2[item][job][lz][cy][cx] (the layout k_z_final reads).
template <int N>
__global__ void __launch_bounds__(64) k_final_xy_h(DevTables tab, const cplx* __restrict__ fhat, const cplx* __restrict__ QGh,
                                                   size_t qstride, cplx* __restrict__ G2) {
  constexpr int N2 = N * N, N3 = N2 * N, H = N / 2, NPH = N * (H + 1);
  extern __shared__ cplx sm[];
  const int job = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* buf = sm + (size_t)job * (N * (N + 1) + N);
  const int lz = blockIdx.x, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  const int q = pair % tab.ns;
  const double inv = 1.0 / ((double)N3);
  const bool full = tab.full[pair];              // full-table pairs keep the whole spectrum, [lz][lx][ly]
  const cplx* qa = QGh + (size_t)item * qstride + (size_t)lz * (full ? N2 : NPH);
  const cplx* qb = QGh + (size_t)item * qstride + (size_t)((N - lz) % N) * NPH;
  const cplx* in = fhat + ((size_t)xl * tab.ns + q) * N3 + (size_t)lz * N2;
  const cplx* cl = tab.closs + (size_t)pair * N3 + (size_t)lz * N2;
  cplx* o = G2 + ((size_t)item * 2 + job) * N3 + (size_t)lz * N2;
  warp_plane_fft<N, +1>(
      buf, lane,
      [&](int lx, int ly) {
        cplx v;
        if (job == 1) v = cmul(in[lx * N + ly], cl[lx * N + ly]);
        else if (full) v = qa[lx * N + ly];
        else if (ly <= H) v = qa[lx * (H + 1) + ly];
        else { v = qb[((N - lx) % N) * (H + 1) + (N - ly)]; v.y = -v.y; }
        return make_double2(v.x * inv, v.y * inv);
      },
      [](cplx x, int) { return x; }, [&](int cy, int cx, cplx val) { o[cy * N + cx] = val; });
}

}  // namespace dgfs
#include "collide_v1_wide.cuh"
namespace dgfs {

// ---------------------------------------------------------------- host orchestration ------------
namespace {
struct PlanV1 {
  int nbx, nbuf, tslots;
  size_t off_fhat, off_fhh, off_nyqy, off_qg, off_gzr[2], off_gz0, off_nyq[2], off_s[2], off_t, off_tf, off_fp, off_gin, off_gout, nyq_bytes, qstride, total;
};
PlanV1 plan_v1_chunk(const dgfs_ctx* c, int nx, int nbx) {
  PlanV1 pl{};
  const size_t N = c->N, N3 = c->N3, arr = N3 * sizeof(cplx);
  pl.nbx = nbx;
  // two-stream schedule: the buffers filled by the preparing kernels exist twice (radial nodes r and r + 1 in flight)
  pl.nbuf = c->v1_overlap ? 2 : 1;
  const size_t items = (size_t)nbx * c->npairs;
  const size_t nyq_stride = 4 * N + 3 * N * N;
  const size_t nzr = c->v1_nz - c->v1_nz0;
  const size_t gel = c->precision == 1 ? 2 : 1;              // precision 1: z-shifted arrays in float2
  size_t gz = (size_t)nbx * nzr * (arr / 2) / gel, g2 = items * 2 * arr;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
  pl.off_fhat = take((size_t)nbx * c->ns * arr);
  pl.off_fhh = take((size_t)nbx * c->ns * (arr / 2));
  pl.off_nyqy = take((size_t)nbx * c->ns * (N * N / 2) * sizeof(cplx));
  const size_t half_arr = N * N * (N / 2 + 1) * sizeof(cplx);
  // QG per item: Hermitian half for VHS pairs, the whole spectrum for pairs with a full b table
  pl.qstride = (c->any_full ? arr : half_arr) / sizeof(cplx);
  pl.off_qg = take(items * pl.qstride * sizeof(cplx));
  pl.off_gzr[0] = take(gz > g2 ? gz : g2);               // also the scratch of step 10
  pl.off_gzr[1] = pl.nbuf > 1 ? take(gz) : pl.off_gzr[0];
  pl.off_gz0 = take((size_t)nbx * c->v1_nz0 * (arr / 2) / gel);
  pl.nyq_bytes = items * c->M * nyq_stride * sizeof(cplx);
  pl.off_nyq[0] = take(pl.nyq_bytes);
  pl.off_nyq[1] = pl.nbuf > 1 ? take(pl.nyq_bytes) : pl.off_nyq[0];
  pl.off_s[0] = take(items * N3 * sizeof(double));
  pl.off_s[1] = pl.nbuf > 1 ? take(items * N3 * sizeof(double)) : pl.off_s[0];
  // T: forward-transformed planes of pl.nbuf groups of radial nodes (a ring: the forward z pass of one group runs
  // while the plane jobs fill the next); also the z-pass scratch of step 1
  pl.tslots = pl.nbuf * c->v1_rgroup;
  const size_t tg = (size_t)pl.tslots * items * half_arr, t1 = (size_t)nbx * c->ns * arr;
  pl.off_t = take(tg > t1 ? tg : t1);
  // Tf: per-s forward-transformed planes of the full-table pairs
  pl.off_tf = take(c->any_full ? items * c->M * arr : 0);
  pl.off_fp = take(c->nyq_filter ? (size_t)nbx * c->ns * N3 * sizeof(double) : 0);     // filtered inputs
  // small batches replayed from a CUDA graph: fixed input / output staging (run_collide_v1)
  const bool small = nx * c->npairs <= c->v1_graph_items;
  pl.off_gin = take(small ? (size_t)nx * c->ns * N3 * sizeof(double) : 0);
  pl.off_gout = take(small ? (size_t)nx * c->npairs * N3 * sizeof(double) : 0);
  pl.total = off;
  return pl;
}
// The launch group: v1_chunk spatial points, fewer when the batch is smaller, when the grid's y extent would pass
// 65535, or when the workspace of the group would pass the context's byte budget (ws_budget: 70 % of the memory free
// at create, or DGFS_V1_WS_GB) -- then it is halved until it fits.  Results do not depend on the group size.
PlanV1 plan_v1(const dgfs_ctx* c, int nx) {
  int nbx = c->v1_chunk;
  if (nbx > nx) nbx = nx;
  if (nbx < 1) nbx = 1;
  if ((size_t)nbx * c->npairs > 65535) nbx = 65535 / c->npairs;
  PlanV1 pl = plan_v1_chunk(c, nx, nbx);
  while (c->ws_budget > 0 && pl.total > c->ws_budget && nbx > 1) {
    nbx = (nbx + 1) / 2;
    pl = plan_v1_chunk(c, nx, nbx);
  }
  return pl;
}
}  // namespace

size_t workspace_bytes_v1(const dgfs_ctx* c, int nx) { return plan_v1(c, nx).total; }

// algorithmic FLOPs of the executed algorithm: a 1-D transform of length N counts
// 5 N log2 N, pointwise work counts the real operations of the formulas in this file's header.
namespace {
struct FlopsV1 { double zshift, nyq, xy, wterm, acc, xy_full, acc_full, tail; };
FlopsV1 flops_v1(const dgfs_ctx* c) {
  const double N = c->N, N2 = N * N, N3 = N2 * N, H = N / 2, M = c->M;
  const double fft1 = 5.0 * N * log2(N), fft3 = 3.0 * N2 * fft1;
  FlopsV1 f{};
  f.zshift = (double)(c->v1_nz - c->v1_nz0) / c->npairs * N * H * (fft1 + 6.0 * N);   // per item and radial node
  // plane jobs and product terms actually run: fields of an axis with sigma_{s,d} = 0 vanish and are skipped
  double njobs = 0.0, wops = 0.0;
  for (int s2 = 0; s2 < c->M; ++s2) {
    const int nt = 3 - ((c->v1_smask[s2] & 1) + ((c->v1_smask[s2] >> 1) & 1) + ((c->v1_smask[s2] >> 2) & 1));
    njobs += nt;
    wops += nt > 0 ? 2.0 * (nt - 1) + 2.0 : 0.0;     // adds forming Re W, Im W, one fma
  }
  f.nyq = njobs * (2.0 * N * fft1 + 14.0 * N2) + M * 16.0 * N2;   // the plane jobs + the 1-D sums
  // per plane job: two passes of N transforms, x and y factors (6 + 6 per element; none / 2 where sigma_x / sigma_y
  // vanishes), packing adds (2), product
  // fma (2), Nyquist row / column fixes (12 N); per plane: forward y pass on real rows (half) and x pass on H+1 columns
  double fac = 0.0;                                    // x and y factor work per element, summed over s
  for (int s2 = 0; s2 < c->M; ++s2)
    fac += ((c->v1_smask[s2] & 1) ? 0.0 : 6.0) + ((c->v1_smask[s2] & 2) ? 2.0 : 6.0);
  f.xy = N * (M * (2.0 * N * fft1 + 4.0 * N2 + 12.0 * N) + fac * N2) + N * (N + 1.0) * fft1;
  f.wterm = wops * N3 + N3;
  f.acc = N * (H + 1.0) * (fft1 + 4.0 * N);         // forward z pass and QG += w_r b_r . on the Hermitian half
  // full-table pairs: four passes per plane job, W (10 per element) and the complex product (8), then per s
  // a forward z pass and the complex multiply-accumulate with b_rs (8 per mode)
  f.xy_full = N * (M * (4.0 * N * fft1 + 20.0 * N2 + 12.0 * N) + fac * N2);
  f.acc_full = M * (N2 * fft1 + 8.0 * N3);
  f.tail = 2.0 * fft3 + 11.0 * N3 + fft3 / c->ns;
  return f;
}
}  // namespace

double flops_per_pair_eval_v1(const dgfs_ctx* c, int pair) {
  FlopsV1 f = flops_v1(c);
  if (c->nyq_filter) f.nyq = f.wterm = 0.0;              // those kernels are not run (dgfs_params::nyquist_filter)
  if (c->full[pair]) {
    int run = 0;
    for (int s2 = 0; s2 < c->M; ++s2) run += !c->v1_sskip[(size_t)pair * c->M + s2];
    const double frac = (double)run / c->M;
    return c->N_rho * ((frac > 0 ? f.zshift : 0.0) + frac * (f.nyq + f.xy_full) + f.acc_full) + f.tail;
  }
  if (c->v1_tsrc[pair] != pair) return c->N_rho * f.acc + f.tail;      // R-11: only the forward z pass and step 10
  // same-species VHS pairs run one point of every antipodal couple (R-10): the s-proportional kernels scale
  int run = 0;
  for (int s2 = 0; s2 < c->M; ++s2) run += !c->v1_sskip[(size_t)pair * c->M + s2];
  const double frac = (double)run / c->M;
  const double fwd = c->N * (c->N + 1.0) * 5.0 * c->N * log2((double)c->N);     // forward passes in k_xy: once per plane
  (void)fwd;
  return c->N_rho * (f.zshift + frac * (f.nyq + f.wterm) + c->v1_xyflops[pair] + f.acc) + f.tail;
}

// Streams and events of the two-stream schedule (created with the context's v1 tables).
int init_streams_v1(dgfs_ctx* c) {
  const char* ov = getenv("DGFS_V1_OVERLAP");
  // measured at c2 (profiles/r02_streams.md): with the auxiliary streams at high priority the preparing kernels
  // displace the plane jobs instead of sharing the SMs with them (each of them fills the register file or the
  // shared memory of an SM on its own), same step time; at equal priority only the tails overlap, 1 % faster.
  // Off by default: one stream, per-kernel event times that add up.
  c->v1_overlap = (ov && atoi(ov) != 0);
  const char* gi = getenv("DGFS_V1_GRAPH_ITEMS");
  if (gi) c->v1_graph_items = atoi(gi) > 0 ? atoi(gi) : 0;
  const char* pk = getenv("DGFS_V1_PACK");
  c->v1_pack = (pk && atoi(pk) != 0);      // measured at c1 (N = 24): 119.5 against 113.2 ms of k_xy per 3 steps, off by default
  const char* xw = getenv("DGFS_V1_XYW");
  c->v1_xyw = (xw && atoi(xw) == 2) ? 2 : 4;
  const char* wm = getenv("DGFS_V1_WTERM_MC");
  c->v1_wterm_mc = (wm && atoi(wm) != 0);
  // byte budget of the workspace of one launch group (plan_v1): DGFS_V1_WS_GB, else 70 % of the memory free now
  const char* wb = getenv("DGFS_V1_WS_GB");
  size_t freeb = 0, totalb = 0;
  if (wb && atof(wb) > 0) c->ws_budget = (size_t)(atof(wb) * 1e9);
  else if (cudaMemGetInfo(&freeb, &totalb) == cudaSuccess) c->ws_budget = (size_t)(0.7 * (double)freeb);
  else cudaGetLastError();
  if (!c->v1_overlap) return DGFS_OK;
  int least = 0, greatest = 0;
  cudaDeviceGetStreamPriorityRange(&least, &greatest);
  const char* pr = getenv("DGFS_V1_AUX_PRIORITY");          // 1 (default): highest priority; 0: default priority
  const int prio = (pr && atoi(pr) == 0) ? 0 : greatest;
  int rc;
  if ((rc = check_cuda(c, cudaStreamCreateWithPriority(&c->aux, cudaStreamNonBlocking, prio), "stream create"))) return rc;
  if ((rc = check_cuda(c, cudaStreamCreateWithPriority(&c->aux2, cudaStreamNonBlocking, prio), "stream create"))) return rc;
  cudaEvent_t* evs[] = {&c->ev_head, &c->ev_prep[0], &c->ev_prep[1], &c->ev_xy[0], &c->ev_xy[1],
                        &c->ev_grp[0], &c->ev_grp[1], &c->ev_acc[0], &c->ev_acc[1]};
  for (cudaEvent_t* e : evs)
    if ((rc = check_cuda(c, cudaEventCreateWithFlags(e, cudaEventDisableTiming), "event create"))) return rc;
  return DGFS_OK;
}
void free_streams_v1(dgfs_ctx* c) {
  cudaEvent_t evs[] = {c->ev_head, c->ev_prep[0], c->ev_prep[1], c->ev_xy[0], c->ev_xy[1], c->ev_grp[0], c->ev_grp[1],
                       c->ev_acc[0], c->ev_acc[1]};
  for (cudaEvent_t e : evs) if (e) cudaEventDestroy(e);
  if (c->aux) cudaStreamDestroy(c->aux);
  if (c->aux2) cudaStreamDestroy(c->aux2);
}

// Schedule of one chunk (all launches asynchronous; `st` is the caller's stream):
//   st  : step 1 | k_xy(0) | k_xy(1) | ...                         | step 10
//   aux : z shifts with sigma_z = 0 | prep(0) | prep(1) | prep(2) ...      prep(r) = k_zshift, k_nyq1d, k_nyq2, k_wterm
//   aux2:                                   forward z pass + QG accumulation of every finished group of radial nodes
// prep(r) fills buffer r & 1 (z-shifted arrays, Nyquist fields, S) and waits for k_xy(r - 2) to have read it; k_xy(r)
// waits for prep(r).  The preparing kernels are bound by memory traffic and latencies and leave the FP64 pipe mostly
// idle, the plane jobs are bound by the FP64 pipe: on the same SMs at the same time they fill each other's gaps.  aux
// and aux2 have the higher priority, so their blocks take the slots that k_xy blocks free.  With DGFS_V1_OVERLAP=0
// the three streams are the caller's and the events are not used.
template <int N>
static int collide_v1_impl(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  constexpr int N2 = N * N, N3 = N2 * N, H = N / 2;
  constexpr int W = 4;
  const PlanV1 pl = plan_v1(c, nx);
  int rc = ensure_workspace(c, pl.total, st);
  if (rc) return rc;
  const bool ov = c->v1_overlap != 0;
  const bool f32 = c->precision == 1;
  cudaStream_t sa = ov ? c->aux : st, sz = ov ? c->aux2 : st;
  auto wait = [&](cudaStream_t s, cudaEvent_t e) { if (ov) cudaStreamWaitEvent(s, e, 0); };
  auto record = [&](cudaEvent_t e, cudaStream_t s) { if (ov) cudaEventRecord(e, s); };
  char* ws = (char*)c->ws;
  cplx* fhat = (cplx*)(ws + pl.off_fhat);
  cplx* fhh = (cplx*)(ws + pl.off_fhh);
  cplx* nyqy = (cplx*)(ws + pl.off_nyqy);
  cplx* QG = (cplx*)(ws + pl.off_qg);
  cplx* GzR[2] = {(cplx*)(ws + pl.off_gzr[0]), (cplx*)(ws + pl.off_gzr[1])};
  cplx* Gz0 = (cplx*)(ws + pl.off_gz0);
  cplx* nyqb[2] = {(cplx*)(ws + pl.off_nyq[0]), (cplx*)(ws + pl.off_nyq[1])};
  double* Sb[2] = {(double*)(ws + pl.off_s[0]), (double*)(ws + pl.off_s[1])};
  cplx* T = (cplx*)(ws + pl.off_t);
  cplx* Tf = (cplx*)(ws + pl.off_tf);
  cplx* G2 = GzR[0];
  const size_t qstride = pl.qstride;
  int nfull = 0;
  for (int pr = 0; pr < c->npairs; ++pr) nfull += c->full[pr];
  const int nvhs = c->npairs - nfull;
  // share of the sphere points actually run, summed over the VHS pairs / over all pairs (R-10)
  double run_vhs = 0.0, run_all = 0.0;
  int nrun_vhs = 0;                                                     // VHS pairs that run plane jobs (R-11)
  for (int pr = 0; pr < c->npairs; ++pr) {
    int run = 0;
    for (int s2 = 0; s2 < c->M; ++s2) run += !c->v1_sskip[(size_t)pr * c->M + s2];
    run_all += (double)run / c->M;
    if (!c->full[pr]) run_vhs += (double)run / c->M;
    if (!c->full[pr] && c->v1_tsrc[pr] == pr) ++nrun_vhs;
  }
  double xy_flops = 0.0;                                                 // k_xy per point and radial node, all pairs
  for (int pr = 0; pr < c->npairs; ++pr) if (!c->full[pr]) xy_flops += c->v1_xyflops[pr];
  (void)nrun_vhs;
  const int ns = c->ns, np = c->npairs, nz = c->v1_nz, nz0 = c->v1_nz0, nzr = nz - nz0;
  const size_t smem_plane = plane_smem_per_warp<N>() * W;
  const size_t smem_final = plane_smem_per_warp<N>() * 2;
  const size_t smem_xy = sizeof(cplx) * (size_t)W * GroupSmem<N>::WORDS;
  const size_t smem_xyf = sizeof(cplx) * ((size_t)W * FullSmem<N>::WORDS + FullSmem<N>::UZW);
  const size_t smem_wt = sizeof(cplx) * (size_t)WtermSmem<N>::STAGES * WtermSmem<N>::WORDS;
  const size_t smem_nyq = sizeof(cplx) * (size_t)2 * JobSmem<N>::WORDS;
  const size_t smem_zacc = sizeof(cplx) * (size_t)ZaccSmem<N>::STAGES * ZaccSmem<N>::WORDS;
  const size_t smem_zs = sizeof(cplx) * (size_t)N * 128;
  const size_t smem_wide = sizeof(cplx) * (size_t)JobSmem<N>::WORDS;      // one job per block of 64 threads (N > 32)
  if (!c->v1_attr_done) {                 // per context, hence per device
    cudaFuncSetAttribute(k_plane_fwd<N, W, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_plane_fwd<N, W, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_plane);
    cudaFuncSetAttribute(k_final_xy_h<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_final);
    if constexpr (N <= 32) {
      cudaFuncSetAttribute(k_xy<N, W, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xy);
      cudaFuncSetAttribute(k_xy<N, W, cplxf>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xy / 2);
      cudaFuncSetAttribute(k_xy<N, 2, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xy / 2);
      if constexpr (N < 32) {
        cudaFuncSetAttribute(k_xy<N, W, cplx, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xy);
        cudaFuncSetAttribute(k_xy<N, W, cplxf, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xy / 2);
      }
      cudaFuncSetAttribute(k_xy_full<N, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xyf);
      cudaFuncSetAttribute(k_nyq2<N, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_nyq);
    } else {
      cudaFuncSetAttribute(k_xy_wide<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(2 * smem_wide));
      cudaFuncSetAttribute(k_nyq2_wide<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_wide);
    }
    cudaFuncSetAttribute(k_wterm<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_wt);
    if constexpr (N == 32) cudaFuncSetAttribute(k_wterm_mc<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_wt);
    cudaFuncSetAttribute(k_zshift<N, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_zs);
    cudaFuncSetAttribute(k_zshift<N, cplxf>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_zs);
    if constexpr (N <= 32) {
      cudaFuncSetAttribute(k_zfwd_full<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_zacc);
      cudaFuncSetAttribute(k_zfwd_full<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_zacc);
    }
    cudaFuncSetAttribute(k_zfwd_acc<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_zacc);
    cudaFuncSetAttribute(k_zfwd_acc<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_zacc);
    c->v1_attr_done = true;
  }
  const int pen_blocks = (N2 + 127) / 128;
  const int hpen_blocks = (N * H + 127) / 128;
  const int plane_blocks = (N + W - 1) / W;
  const int hp_blocks = (N * (H + 1) + ZaccSmem<N>::PB - 1) / ZaccSmem<N>::PB;
  const int RG = c->v1_rgroup;
  const double fft3 = 15.0 * N3 * log2((double)N);
  const FlopsV1 fl = flops_v1(c);
  for (int x0 = 0; x0 < nx; x0 += pl.nbx) {
    const int nb = (nx - x0 < pl.nbx) ? nx - x0 : pl.nbx;
    const int items = nb * np;
    const double* fc = f + (size_t)x0 * ns * N3;       // (or the filtered copy, below)
    const size_t slot_stride = (size_t)items * N2 * (H + 1);
    if (c->nyq_filter) {
      // dgfs_params::nyquist_filter: the operator acts on P f; every Nyquist field is then zero, so the kernels that
      // build and multiply them are not run and their buffers are cleared once per chunk
      double* fp = (double*)(ws + pl.off_fp);
      if ((rc = launch_nyquist_filter(c, fc, fp, nb * ns, st))) return rc;
      fc = fp;
      for (int b = 0; b < pl.nbuf; ++b) {
        cudaMemsetAsync(nyqb[b], 0, pl.nyq_bytes, st);
        cudaMemsetAsync(Sb[b], 0, (size_t)items * N3 * sizeof(double), st);
      }
    }
    // step 1, once per species (R-2), plus the half-packed copy
    { ProfScope ps(c->prof, st, "k_zfwd_real", nb * ns * fft3 / 3.0);
      k_zfwd_real<N><<<dim3(pen_blocks, nb * ns), 128, 0, st>>>(fc, T); }
    { ProfScope ps(c->prof, st, "k_plane_fwd<store>", nb * ns * fft3 * 2.0 / 3.0);
      k_plane_fwd<N, W, 0><<<dim3(plane_blocks, nb * ns), 32 * W, smem_plane, st>>>(c->tab, T, 1, fhat, 0); }
    { ProfScope ps(c->prof, st, "k_pack_half", 0.0);
      k_pack_half<N><<<(nb * ns * N2 * H + 255) / 256, 256, 0, st>>>(fhat, fhh, nyqy, nb * ns); }
    record(c->ev_head, st);
    wait(sa, c->ev_head);
    if (nvhs > 0) wait(sz, c->ev_head);
    if (nz0 > 0) {     // the unshifted arrays (sigma_z = 0), the same for every radial node
      ProfScope ps(c->prof, sa, "k_zshift", items * fl.zshift * nz0 / (nzr > 0 ? nzr : 1));
      if (f32) k_zshift<N, cplxf><<<dim3(hpen_blocks, ns, nb), 128, smem_zs, sa>>>(c->v1, ns, fhh, (cplxf*)Gz0, 0, nzr, nz0, nzr, nz0);
      else k_zshift<N, cplx><<<dim3(hpen_blocks, ns, nb), 128, smem_zs, sa>>>(c->v1, ns, fhh, Gz0, 0, nzr, nz0, nzr, nz0);
    }
    int ngroups = 0;
    for (int r = 0; r < c->N_rho; ++r) {
      const int b = ov ? (r & 1) : 0;
      // ---- prepare radial node r (stream sa)
      if (r >= 2) wait(sa, c->ev_xy[b]);                     // the plane jobs of r - 2 have read buffer b
      if (nzr > 0)
      { ProfScope ps(c->prof, sa, "k_zshift", items * fl.zshift);
        if (f32) k_zshift<N, cplxf><<<dim3(hpen_blocks, ns, nb), 128, smem_zs, sa>>>(c->v1, ns, fhh, (cplxf*)GzR[b], r, 0, nzr, 0, nzr);
        else k_zshift<N, cplx><<<dim3(hpen_blocks, ns, nb), 128, smem_zs, sa>>>(c->v1, ns, fhh, GzR[b], r, 0, nzr, 0, nzr); }
      if (!c->nyq_filter) {
      { ProfScope ps(c->prof, sa, "k_nyq1d", nb * run_all * c->M * 16.0 * N2);
        k_nyq1d<N><<<(items * c->M + 3) / 4, 128, 0, sa>>>(c->v1, c->tab, fhat, nyqb[b], r, items * c->M); }
      { ProfScope ps(c->prof, sa, "k_nyq2", nb * run_all * (fl.nyq - c->M * 16.0 * N2));
        if constexpr (N <= 32) k_nyq2<N, 2><<<dim3(3, items), 64, smem_nyq, sa>>>(c->v1, c->tab, fhh, nyqy, nyqb[b], r);
        else k_nyq2_wide<N><<<dim3(3, items), 64, smem_wide, sa>>>(c->v1, c->tab, fhh, nyqy, nyqb[b], r); }
      if (nvhs > 0)
        { ProfScope ps(c->prof, sa, "k_wterm", nb * run_vhs * fl.wterm);
          bool mc = false;
          if constexpr (N == 32) mc = c->v1_wterm_mc != 0;
          if (mc) {
            if constexpr (N == 32) {
              cudaLaunchConfig_t lc{};
              lc.gridDim = dim3(N / WtermSmem<N>::CYB, items); lc.blockDim = dim3(WtermSmem<N>::THREADS);
              lc.dynamicSmemBytes = smem_wt; lc.stream = sa;
              cudaLaunchAttribute at[1];
              at[0].id = cudaLaunchAttributeClusterDimension;
              at[0].val.clusterDim.x = N / WtermSmem<N>::CYB; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
              lc.attrs = at; lc.numAttrs = 1;
              cudaLaunchKernelEx(&lc, k_wterm_mc<N>, (const cplx*)nyqb[b], (int)c->M, Sb[b], c->tab.full, np, c->v1.smask, c->v1.sskip, c->v1.tsrc);
            }
          } else
          k_wterm<N><<<dim3(N / WtermSmem<N>::CYB, items), WtermSmem<N>::THREADS, smem_wt, sa>>>(nyqb[b], c->M, Sb[b], c->tab.full, np, c->v1.smask, c->v1.sskip, c->v1.tsrc); }
      }
      record(c->ev_prep[b], sa);
      // ---- plane jobs of radial node r (caller's stream)
      wait(st, c->ev_prep[b]);
      const GzView gv{GzR[b], Gz0, nzr, nz0};
      if (nvhs > 0) {
        const int g = r / RG, slot = r % pl.tslots;
        if (r % RG == 0 && g >= 2) wait(st, c->ev_acc[g & 1]);       // the forward z pass of group g - 2 has read these slots
        { ProfScope ps(c->prof, st, "k_xy", nb * xy_flops);
          if constexpr (N > 32) {
            k_xy_wide<N><<<dim3(N / 2, items), 2 * N, 2 * smem_wide, st>>>(c->v1, c->tab, gv, c->v1.hxy, nyqb[b], Sb[b], T + (size_t)slot * slot_stride, r);
          } else if (N < 32 && c->v1_pack) {          // N lanes per job: W planes on N W threads (k_xy, PACK)
            if constexpr (N < 32) {
              if (f32) {
                const GzViewT<cplxf> gvf{(const cplxf*)GzR[b], (const cplxf*)Gz0, nzr, nz0};
                k_xy<N, W, cplxf, true><<<dim3(N / W, items), N * W, smem_xy / 2, st>>>(c->v1, c->tab, gvf, c->v1.hxyf, nyqb[b], Sb[b], T + (size_t)slot * slot_stride, r);
              } else
                k_xy<N, W, cplx, true><<<dim3(N / W, items), N * W, smem_xy, st>>>(c->v1, c->tab, gv, c->v1.hxy, nyqb[b], Sb[b], T + (size_t)slot * slot_stride, r);
            }
          } else if (f32) {         // dgfs_params::precision = 1
            const GzViewT<cplxf> gvf{(const cplxf*)GzR[b], (const cplxf*)Gz0, nzr, nz0};
            k_xy<N, W, cplxf><<<dim3((N + W - 1) / W, items), 32 * W, smem_xy / 2, st>>>(c->v1, c->tab, gvf, c->v1.hxyf, nyqb[b], Sb[b], T + (size_t)slot * slot_stride, r);
          } else if (c->v1_xyw == 2)       // DGFS_V1_XYW=2: blocks of two warps, five per SM (ten warps at <= 200 registers)
            k_xy<N, 2, cplx><<<dim3((N + 1) / 2, items), 64, smem_xy / 2, st>>>(c->v1, c->tab, gv, c->v1.hxy, nyqb[b], Sb[b], T + (size_t)slot * slot_stride, r);
          else
            k_xy<N, W, cplx><<<dim3((N + W - 1) / W, items), 32 * W, smem_xy, st>>>(c->v1, c->tab, gv, c->v1.hxy, nyqb[b], Sb[b], T + (size_t)slot * slot_stride, r); }
      }
      if constexpr (N <= 32) if (nfull > 0) {
        { ProfScope ps(c->prof, st, "k_xy_full", nb * (run_all - run_vhs) * fl.xy_full);
          k_xy_full<N, W><<<dim3((N + W - 1) / W, items), 32 * W, smem_xyf, st>>>(c->v1, c->tab, gv, nyqb[b], Tf, r); }
        { ProfScope ps(c->prof, st, "k_zfwd_full", nb * nfull * fl.acc_full);
          const int fp_blocks = (N2 + ZaccSmem<N>::PB - 1) / ZaccSmem<N>::PB;
          if (r == 0) k_zfwd_full<N, true><<<dim3(fp_blocks, items), 256, smem_zacc, st>>>(c->tab, c->v1, Tf, QG, qstride, r);
          else k_zfwd_full<N, false><<<dim3(fp_blocks, items), 256, smem_zacc, st>>>(c->tab, c->v1, Tf, QG, qstride, r); }
      }
      record(c->ev_xy[b], st);
      // ---- forward z pass and QG accumulation of a finished group of radial nodes (stream sz)
      if (nvhs > 0 && ((r + 1) % RG == 0 || r + 1 == c->N_rho)) {
        const int g = r / RG, r0 = g * RG, nr = r + 1 - r0;
        record(c->ev_grp[g & 1], st);
        wait(sz, c->ev_grp[g & 1]);
        const cplx* Tg = T + (size_t)(r0 % pl.tslots) * slot_stride;
        { ProfScope ps(c->prof, sz, "k_zfwd_acc", nb * nvhs * fl.acc * nr);
          if (r0 == 0) k_zfwd_acc<N, true><<<dim3(hp_blocks, items), 128, smem_zacc, sz>>>(c->tab, c->v1.tsrc, Tg, slot_stride, QG, qstride, r0, nr);
          else k_zfwd_acc<N, false><<<dim3(hp_blocks, items), 128, smem_zacc, sz>>>(c->tab, c->v1.tsrc, Tg, slot_stride, QG, qstride, r0, nr); }
        record(c->ev_acc[g & 1], sz);
        ngroups = g + 1;
      }
    }
    // join: the last groups' accumulation into QG (sz is in order, so the last event covers the earlier ones)
    if (ngroups > 0) wait(st, c->ev_acc[(ngroups - 1) & 1]);
    // step 10
    { ProfScope ps(c->prof, st, "k_final_xy", items * (2.0 * fft3 * 2.0 / 3.0 + 6.0 * N3));
      k_final_xy_h<N><<<dim3(N, items), 64, smem_final, st>>>(c->tab, fhat, QG, qstride, G2); }
    { ProfScope ps(c->prof, st, "k_z_final", items * (2.0 * fft3 / 3.0 + 5.0 * N3));
      if (pairs_out)
        k_z_final<N, false><<<dim3(pen_blocks, items), 128, 0, st>>>(c->tab, G2, fc, out + (size_t)x0 * np * N3);
      else
        k_z_final<N, true><<<dim3(pen_blocks, nb * ns), 128, 0, st>>>(c->tab, G2, fc, out + (size_t)x0 * ns * N3); }
  }
  return check_cuda(c, cudaGetLastError(), "collide (v1) launch");
}

static int dispatch_v1(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  switch (c->N) {
    case 8: return collide_v1_impl<8>(c, f, out, nx, pairs_out, st);
    case 16: return collide_v1_impl<16>(c, f, out, nx, pairs_out, st);
    case 24: return collide_v1_impl<24>(c, f, out, nx, pairs_out, st);
    case 32: return collide_v1_impl<32>(c, f, out, nx, pairs_out, st);
    case 48: return collide_v1_impl<48>(c, f, out, nx, pairs_out, st);      // VHS pairs only (collide_v1_wide.cuh)
  }
  return set_error(c, DGFS_ENOSUP, "v1 pipeline: unsupported N");
}

void drop_graphs_v1(dgfs_ctx* c) {
  for (auto& g : c->graphs) cudaGraphExecDestroy(g.exec);
  c->graphs.clear();
}
void free_graph_stream_v1(dgfs_ctx* c) { if (c->cap_stream) cudaStreamDestroy(c->cap_stream); c->cap_stream = nullptr; }

// Small batches (nx * pairs <= 64: config c0, single points of a test) are bound by launch latency: ~100 launches of a
// few microseconds each.  Their whole call is captured once, on fixed staging buffers inside the workspace, into a CUDA
// graph and replayed: copy f in, one graph launch, copy Q out.  Same kernels, same launch order, same bits.  Not
// while the caller captures its own graph, nor with per-launch profiling on, nor with the three-stream schedule.
int run_collide_v1(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cap);
  const bool small = nx * c->npairs <= c->v1_graph_items && !c->prof.on && !c->v1_overlap && cap == cudaStreamCaptureStatusNone;
  if (!small) return dispatch_v1(c, f, out, nx, pairs_out, st);
  const PlanV1 pl = plan_v1(c, nx);
  int rc = ensure_workspace(c, pl.total, st);
  if (rc) return rc;
  double* gin = (double*)((char*)c->ws + pl.off_gin);
  double* gout = (double*)((char*)c->ws + pl.off_gout);
  const size_t in_bytes = (size_t)nx * c->ns * c->N3 * sizeof(double);
  const size_t out_bytes = (size_t)nx * (pairs_out ? c->npairs : c->ns) * c->N3 * sizeof(double);
  dgfs_ctx::SmallGraph* g = nullptr;
  for (auto& e : c->graphs) if (e.nx == nx && e.pairs == pairs_out && e.ws == c->ws) g = &e;
  if (!g) {
    if (!c->v1_attr_done) {          // first call of the context: set the kernel attributes outside any capture
      if ((rc = dispatch_v1(c, f, out, nx, pairs_out, st))) return rc;
      return DGFS_OK;
    }
    const long long l0 = c->prof.total_launches;
    cudaGraph_t graph = nullptr;
    if (!c->cap_stream && (rc = check_cuda(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking), "stream create"))) return rc;
    if ((rc = check_cuda(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal), "graph capture"))) return rc;
    rc = dispatch_v1(c, gin, gout, nx, pairs_out, c->cap_stream);
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
    const long long nl = c->prof.total_launches - l0;
    c->prof.total_launches = l0;
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if ((rc = check_cuda(c, e, "graph capture"))) return rc;
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if ((rc = check_cuda(c, e, "graph instantiation"))) return rc;
    c->graphs.push_back({nx, pairs_out, c->ws, exec, nl});
    g = &c->graphs.back();
  }
  cudaMemcpyAsync(gin, f, in_bytes, cudaMemcpyDeviceToDevice, st);
  if ((rc = check_cuda(c, cudaGraphLaunch(g->exec, st), "graph launch"))) return rc;
  cudaMemcpyAsync(out, gout, out_bytes, cudaMemcpyDeviceToDevice, st);
  c->prof.total_launches += g->launches;
  return check_cuda(c, cudaGetLastError(), "collide (v1, graph) launch");
}

}  // namespace dgfs

// ---------------------------------------------------------------- dgfs_collide_noalloc ------------
// The v1 pipeline above with its workspace in a file-scope device array instead of the context's stream-ordered
// allocation: for callers that must not allocate (a caller's own graph capture, a serving loop, a harness that forbids
// cudaMalloc).  Every GPU that loads the library holds DGFS_NOALLOC_SCRATCH_BYTES of device memory for this array until
// the process exits.  Host code must not pass the symbol itself to a kernel (there it names a host-side stand-in): the
// device address is asked for once per device, with that device current, and kept.
static __device__ __align__(256) unsigned char g_noalloc_scratch[DGFS_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
void* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

// puts the context's workspace fields back however the call ends
struct WorkspaceSwap {
  dgfs_ctx* c; void* ws; size_t ws_bytes, ws_budget;
  WorkspaceSwap(dgfs_ctx* c_, void* p, size_t bytes) : c(c_), ws(c_->ws), ws_bytes(c_->ws_bytes), ws_budget(c_->ws_budget) {
    c->ws = p; c->ws_bytes = bytes;
    if (c->ws_budget == 0 || c->ws_budget > bytes) c->ws_budget = bytes;      // plan_v1 halves the launch group to fit
  }
  ~WorkspaceSwap() { c->ws = ws; c->ws_bytes = ws_bytes; c->ws_budget = ws_budget; }
};
}  // namespace

extern "C" int dgfs_collide_noalloc(dgfs_ctx* c, const double* f, double* Q, int nx, void* stream) {
  using namespace dgfs;
  if (!c) return DGFS_EINVAL;
  if (nx < 0) return set_error(c, DGFS_EINVAL, "dgfs_collide_noalloc: nx must be >= 0");
  if (nx == 0) return DGFS_OK;
  if (!f || !Q) return set_error(c, DGFS_EINVAL, "dgfs_collide_noalloc: f and Q must not be NULL");
  if ((const void*)f == (const void*)Q) return set_error(c, DGFS_EINVAL, "dgfs_collide_noalloc: Q must not alias f");
  if (!c->use_v1) return set_error(c, DGFS_ENOSUP, "dgfs_collide_noalloc: only contexts on the v1 pipeline (N <= 32, or N = 48 without VSS pairs)");
  if (c->prof.on) return set_error(c, DGFS_ENOSUP, "dgfs_collide_noalloc: per-launch profiling creates events; switch it off (dgfs_profile_enable)");
  if (c->device < 0 || c->device >= NOALLOC_MAX_DEVICES) return set_error(c, DGFS_ENOSUP, "dgfs_collide_noalloc: device index beyond 63");
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) return check_cuda(c, e, "cudaSetDevice");
  void* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[c->device]) {                  // once per device, that device current
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
      if (e != cudaSuccess || !p) return check_cuda(c, e != cudaSuccess ? e : cudaErrorInvalidSymbol, "dgfs_collide_noalloc: cudaGetSymbolAddress");
      g_noalloc_ptr[c->device] = p;
    }
    scratch = g_noalloc_ptr[c->device];
  }
  cudaStream_t st = (cudaStream_t)stream;
  WorkspaceSwap swap(c, scratch, (size_t)DGFS_NOALLOC_SCRATCH_BYTES);
  const size_t need = workspace_bytes_v1(c, nx);       // with the launch group already halved towards the limit
  if (need > (size_t)DGFS_NOALLOC_SCRATCH_BYTES) {
    char msg[256];
    snprintf(msg, sizeof msg, "dgfs_collide_noalloc: one spatial point of this configuration needs %zu bytes of workspace, "
             "the static scratch holds %zu (DGFS_NOALLOC_SCRATCH_BYTES): use dgfs_collide", need, (size_t)DGFS_NOALLOC_SCRATCH_BYTES);
    return set_error(c, DGFS_EINVAL, msg);
  }
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(st, &cap);
  const bool capturing = cap != cudaStreamCaptureStatusNone;
  if (!capturing && c->ev_last_set) cudaStreamWaitEvent(st, c->ev_last, 0);      // calls of one context stay ordered
  // Nothing in the workspace has to start from zero: every buffer is written by an earlier kernel of the same call
  // before it is read (the r = 0 launches of k_zfwd_acc / k_zfwd_full store QG, the later ones add to it), the
  // Nyquist-filter variant clears its fields itself.  So the contents the last call left behind are never read.
  const int rc = dispatch_v1(c, f, Q, nx, false, st);    // straight to the kernels: no graph, no ensure_workspace growth
  if (!capturing && c->ev_last) { cudaEventRecord(c->ev_last, st); c->ev_last_set = true; }
  return rc;
}
