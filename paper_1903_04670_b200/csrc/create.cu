// create.cu -- dgfs_create: Algorithm 1 of PAPER.md on the device.
//
// Host part: argument validation, Gauss-Legendre radial rule, built-in sphere rules standing in
// for the spherical designs of ref. [18] (reading S-2), truncation radius (Eq. 9, reading RAD-1),
// prefactors (Eq. 6).  Device part: the kernel-mode tables.  The paper stores a[N_rho][M][N^3] and
// b[N_rho][M][N^3] in full; here
//   * exp(+-i mu a_rs) is kept as three 1-D factors per (r, s, side)          (exact: a_rs is linear in l),
//   * b_r of a VHS pair depends on |k|^2 only and is stored as such           (Eq. 16 with eta = 0),
//   * b_rs of a VSS pair is stored in full, evaluated from the Legendre / spherical-Bessel expansion of
//     the angular integral of Eq. 16 (exact to round-off; see k_bfull_series),
//   * table_mode 1 reproduces Algo 1 steps 9-14 literally with the caller's pre-computation sphere.
#include <cmath>
#include <cstdio>
#include <cstring>
#include "ctx.h"

namespace dgfs {

static thread_local std::string g_create_error;   // per thread: dgfs_last_error(NULL) reports the calling thread's last failed dgfs_create

int set_error(dgfs_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}
int check_cuda(dgfs_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return DGFS_OK;
  return set_error(c, e == cudaErrorMemoryAllocation ? DGFS_ENOMEM : DGFS_ECUDA,
                   std::string(what) + ": " + cudaGetErrorString(e));
}

// ---------------------------------------------------------------- host quadrature -----------------
// N_rho-point Gauss-Legendre on [-1,1] by Newton iteration on P_n (ascending nodes).
static void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
  x.resize(n); w.resize(n);
  const long double pi = 3.14159265358979323846264338327950288L;
  for (int i = 0; i < n; ++i) {
    long double z = cosl(pi * (i + 0.75L) / (n + 0.5L)), pp = 0;
    for (int it = 0; it < 100; ++it) {
      long double p0 = 1, p1 = z;
      for (int k = 2; k <= n; ++k) { long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
      if (n == 1) { p0 = 1; p1 = z; }
      pp = n * (z * p1 - p0) / (z * z - 1);
      long double dz = p1 / pp;
      z -= dz;
      if (fabsl(dz) < 1e-19L) break;
    }
    {  // derivative at the converged node
      long double p0 = 1, p1 = z;
      for (int k = 2; k <= n; ++k) { long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
      pp = n * (z * p1 - p0) / (z * z - 1);
    }
    x[n - 1 - i] = (double)z;
    w[n - 1 - i] = (double)(2 / ((1 - z * z) * pp * pp));
  }
}

// Built-in sphere rules (reading S-2): octahedron (degree 3), icosahedron (5), icosahedron + its dual
// dodecahedron with weights 5/168 and 9/280 of 4 pi (degree 9).
static bool builtin_sphere(int M, std::vector<double>& sig, std::vector<double>& w) {
  const double pi = 3.14159265358979323846;
  const double phi = 0.5 * (1.0 + sqrt(5.0));
  sig.clear(); w.clear();
  auto push = [&](double x, double y, double z, double wt) {
    double n = sqrt(x * x + y * y + z * z);
    sig.push_back(x / n); sig.push_back(y / n); sig.push_back(z / n); w.push_back(wt);
  };
  if (M == 6) {
    for (int d = 0; d < 3; ++d) for (int sgn = 1; sgn >= -1; sgn -= 2) {
      double v[3] = {0, 0, 0}; v[d] = sgn; push(v[0], v[1], v[2], 4 * pi / 6);
    }
    return true;
  }
  if (M == 12 || M == 32) {
    const double wi = (M == 12) ? 4 * pi / 12 : 4 * pi * 5.0 / 168.0;
    for (int rot = 0; rot < 3; ++rot) for (int a = 1; a >= -1; a -= 2) for (int b = 1; b >= -1; b -= 2) {
      double v[3]; v[rot] = 0; v[(rot + 1) % 3] = a; v[(rot + 2) % 3] = b * phi;   // (0, +-1, +-phi) cyclic
      push(v[0], v[1], v[2], wi);
    }
    if (M == 32) {
      const double wd = 4 * pi * 9.0 / 280.0;
      for (int a = 1; a >= -1; a -= 2) for (int b = 1; b >= -1; b -= 2) for (int c = 1; c >= -1; c -= 2) push(a, b, c, wd);
      // face centres of the icosahedron above: cyclic permutations of (+-1/phi, 0, +-phi)
      for (int rot = 0; rot < 3; ++rot) for (int a = 1; a >= -1; a -= 2) for (int b = 1; b >= -1; b -= 2) {
        double v[3]; v[rot] = a / phi; v[(rot + 1) % 3] = 0; v[(rot + 2) % 3] = b * phi;
        push(v[0], v[1], v[2], wd);
      }
    }
    return true;
  }
  return false;
}

// ---------------------------------------------------------------- device table kernels -----------
__device__ __forceinline__ int signed_freq(int j, int N) { return j - (j >= N / 2 ? N : 0); }   // Algo 1 steps 1-3
__device__ __forceinline__ double sinc_u(double x) { return x == 0.0 ? 1.0 : sin(x) / x; }

// SPEC layout index -> signed frequency triple
__device__ __forceinline__ void spec_freq(int idx, int N, int& kx, int& ky, int& kz) {
  int iy = idx % N, ix = (idx / N) % N, iz = idx / (N * N);
  kx = signed_freq(ix, N); ky = signed_freq(iy, N); kz = signed_freq(iz, N);
}

// phase[pair][r][s][side][d][j]
__global__ void k_phase(cplx* out, int ns, int N, int N_rho, int M, double L, const double* mass,
                        const double* rho, const double* sigma, const double* w_sigma, const double* wfac) {
  const long total = (long)ns * ns * N_rho * M * 2 * 3 * N;
  const double pi = 3.14159265358979323846;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int j = i % N; long t = i / N;
    int d = t % 3; t /= 3;
    int side = t % 2; t /= 2;
    int s = t % M; t /= M;
    int r = t % N_rho; t /= N_rho;
    int q = t % ns, p = t / ns;
    double mu = (side == 0) ? mass[q] / (mass[p] + mass[q]) : -mass[p] / (mass[p] + mass[q]);
    double theta = mu * (pi * rho[r] / L) * sigma[s * 3 + d] * (double)signed_freq(j, N);
    double sn, cs; sincos(theta, &sn, &cs);
    double scale = 1.0;
    if (d == 0) { scale = 1.0 / ((double)N * N * N); if (side == 0) scale *= w_sigma[s] * wfac[(size_t)(p * ns + q) * M + s]; }
    out[i] = make_double2(cs * scale, sn * scale);
  }
}

// bvhs[pair][r][K2] = 4 pi rho^{gamma+2} sinc(mu_q rho' sqrt(K2))          (Eq. 16 with eta = 0, reading P-1)
__global__ void k_bvhs(double* out, int ns, int N_rho, int K2n, double L, const double* mass, const double* gam,
                       const double* rho) {
  const long total = (long)ns * ns * N_rho * K2n;
  const double pi = 3.14159265358979323846;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int k2 = i % K2n; long t = i / K2n;
    int r = t % N_rho; int pair = t / N_rho;
    int q = pair % ns, p = pair / ns;
    double mu_q = mass[q] / (mass[p] + mass[q]);
    double z = mu_q * (pi * rho[r] / L) * sqrt((double)k2);
    out[i] = 4.0 * pi * pow(rho[r], gam[pair] + 2.0) * sinc_u(z);
  }
}

// closs[pair][idx] (mode 0) = sum_r w_r rho^{gamma+2} C_eta 4 pi sinc(rho'_r |l|)   (Eq. 17, reading O-8)
__global__ void k_closs0(cplx* out, int ns, int N, int N_rho, double L, const double* gam, const double* eta,
                         const double* rho, const double* w_rho) {
  const int N3 = N * N * N;
  const long total = (long)ns * ns * N3;
  const double pi = 3.14159265358979323846;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int idx = i % N3, pair = i / N3;
    int kx, ky, kz; spec_freq(idx, N, kx, ky, kz);
    double ln = sqrt((double)(kx * kx + ky * ky + kz * kz));
    double e = eta[pair], g = gam[pair];
    double Ceta = 2.0 * pi * exp2(e + 1.0) / (e + 1.0);
    double acc = 0.0;
    for (int r = 0; r < N_rho; ++r)
      acc += w_rho[r] * pow(rho[r], g + 2.0) * Ceta * 4.0 * pi * sinc_u(pi * rho[r] / L * ln);
    out[i] = make_double2(acc, 0.0);
  }
}

// Full b for a VSS pair, table_mode 0.  Angular integral of Eq. 16,
//   F = int_{S^2} (1 + sigma_s.u)^eta exp(-i z lhat.u) du ,  z = mu_q rho'_r |l| ,
// expanded in Legendre polynomials: (1+t)^eta = sum_n a_n P_n(t), exp(-i z t) = sum_n (2n+1)(-i)^n j_n(z) P_n(t),
// addition theorem  =>  F = 4 pi sum_n a_n (-i)^n j_n(z) P_n(kappa), kappa = lhat.sigma_s,
// a_n = (2n+1)/2 I_n, I_0 = 2^{eta+1}/(eta+1), I_{n+1} = I_n (eta - n)/(eta + n + 2).
// j_n by Miller's backward recurrence normalised with sum (2n+1) j_n^2 = 1 and the sign of j_0 / j_1.
#define DGFS_NSER 224
// F of the comment above times rho^{gamma+2}: one mode (kx, ky, kz) (signed frequencies), one sphere point sigma.
__device__ cplx b_series(int kx, int ky, int kz, const double* sigma3, double mu_q, double rho_r, double L, double gam,
                         double eta) {
  const double pi = 3.14159265358979323846;
  double ln = sqrt((double)(kx * kx + ky * ky + kz * kz));
  double z = mu_q * (pi * rho_r / L) * ln;
  double pref = 4.0 * pi * pow(rho_r, gam + 2.0);
  double I0 = exp2(eta + 1.0) / (eta + 1.0);
  if (ln == 0.0) return make_double2(pref * 0.5 * I0, 0.0);
  double kappa = (kx * sigma3[0] + ky * sigma3[1] + kz * sigma3[2]) / ln;
  kappa = fmin(1.0, fmax(-1.0, kappa));
  // spherical Bessel j_0..j_nmax(z)
  int nmax = (int)(z + 12.0 * cbrt(z + 1.0) + 20.0);
  if (nmax > DGFS_NSER - 1) nmax = DGFS_NSER - 1;
  double jn[DGFS_NSER];
  if (z < 1e-3) {            // series j_n ~ z^n/(2n+1)!! (1 - z^2/(2(2n+3)))
    double tterm = 1.0;
    for (int n = 0; n <= nmax; ++n) { jn[n] = tterm * (1.0 - z * z / (2.0 * (2 * n + 3))); tterm *= z / (2 * n + 3); }
  } else {
    int nstart = nmax + 40;
    double fp1 = 0.0, f = 1e-120, norm = 0.0;
    for (int n = nstart; n >= 0; --n) {
      // j_{n-1} = (2n+1)/z j_n - j_{n+1}
      if (n <= nmax) jn[n] = f;
      norm += (2 * n + 1) * f * f;
      double fm1 = (2 * n + 1) / z * f - fp1;
      fp1 = f; f = fm1;
      if (fabs(f) > 1e120) {   // rescale so that f^2 in the norm cannot overflow
        f *= 1e-120; fp1 *= 1e-120; norm *= 1e-240;
        for (int m = n; m <= nmax; ++m) jn[m] *= 1e-120;
      }
    }
    double scale = rsqrt(norm);
    // fix the sign with whichever of j_0 = sin z / z, j_1 = sin z / z^2 - cos z / z is larger in magnitude
    double sn, cs; sincos(z, &sn, &cs);
    double j0 = sn / z, j1 = sn / (z * z) - cs / z;
    if (fabs(j0) >= fabs(j1)) { if ((jn[0] * scale > 0) != (j0 > 0)) scale = -scale; }
    else { if ((jn[1] * scale > 0) != (j1 > 0)) scale = -scale; }
    for (int n = 0; n <= nmax; ++n) jn[n] *= scale;
  }
  double re = 0.0, im = 0.0;
  double In = I0, Pm1 = 0.0, Pn = 1.0;     // P_{n-1}, P_n at kappa
  for (int n = 0; n <= nmax; ++n) {
    double term = 0.5 * (2 * n + 1) * In * jn[n] * Pn;
    switch (n & 3) {            // (-i)^n
      case 0: re += term; break;
      case 1: im -= term; break;
      case 2: re -= term; break;
      default: im += term; break;
    }
    double Pp1 = ((2 * n + 1) * kappa * Pn - n * Pm1) / (n + 1);
    Pm1 = Pn; Pn = Pp1;
    In *= (eta - n) / (eta + n + 2.0);
  }
  return make_double2(pref * re, pref * im);
}

// out[r][s][N^3] (SPEC layout): every sphere point of the rule in full
__global__ void k_bfull_series(cplx* out, int p, int q, int N, int N_rho, int M, double L, const double* mass,
                               double gam, double eta, const double* rho, const double* sigma) {
  const int N3 = N * N * N;
  const long total = (long)N_rho * M * N3;
  const double mu_q = mass[q] / (mass[p] + mass[q]);
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int idx = i % N3; long t = i / N3;
    int s = t % M, r = t / M;
    int kx, ky, kz; spec_freq(idx, N, kx, ky, kz);
    out[i] = b_series(kx, ky, kz, sigma + 3 * s, mu_q, rho[r], L, gam, eta);
  }
}

// Symmetry-compressed b (DevTables::bsym): out[r][u][(N+1)^3] for the nref reference sphere points refs[u] only, on the
// EXTENDED frequency grid [-N/2, N/2]^3 ([kz][kx][ky], ky fastest): b_rs(k) depends on k through |k| and k . sigma_s,
// so for sigma_s = G sigma_u (G a signed permutation of the axes) b_rs(k) = b_ru(G^T k), and G^T maps the grid
// [-N/2, N/2) into the extended one (the Nyquist index -N/2 may change sign).
__global__ void k_bsym_series(cplx* out, int p, int q, int N, int N_rho, int nref, const int* refs, double L,
                              const double* mass, double gam, double eta, const double* rho, const double* sigma) {
  const int E = N + 1, H = N / 2, E3 = E * E * E;
  const long total = (long)N_rho * nref * E3;
  const double mu_q = mass[q] / (mass[p] + mass[q]);
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int idx = i % E3; long t = i / E3;
    int u = t % nref, r = t / nref;
    int ky = idx % E - H, kx = (idx / E) % E - H, kz = idx / (E * E) - H;
    out[i] = b_series(kx, ky, kz, sigma + 3 * refs[u], mu_q, rho[r], L, gam, eta);
  }
}

// Full b, table_mode 1: Algo 1 steps 9-13 with the caller's pre-computation sphere.
__global__ void k_bfull_pre(cplx* out, int p, int q, int N, int N_rho, int M, double L, const double* mass,
                            double gam, double eta, const double* rho, const double* sigma,
                            int M_pre, const double* sig_pre, const double* w_pre) {
  const int N3 = N * N * N;
  const long total = (long)N_rho * M * N3;
  const double pi = 3.14159265358979323846;
  const double mu_q = mass[q] / (mass[p] + mass[q]);
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int idx = i % N3; long t = i / N3;
    int s = t % M, r = t / M;
    int kx, ky, kz; spec_freq(idx, N, kx, ky, kz);
    double rg = pow(rho[r], gam + 2.0), rp = pi * rho[r] / L;
    double re = 0.0, im = 0.0;
    for (int y = 0; y < M_pre; ++y) {
      double dot = sigma[s * 3] * sig_pre[y * 3] + sigma[s * 3 + 1] * sig_pre[y * 3 + 1] + sigma[s * 3 + 2] * sig_pre[y * 3 + 2];
      double B = pow(1.0 + dot, eta);
      double th = -mu_q * rp * (kx * sig_pre[y * 3] + ky * sig_pre[y * 3 + 1] + kz * sig_pre[y * 3 + 2]);
      double sn, cs; sincos(th, &sn, &cs);
      re += B * w_pre[y] * rg * cs; im += B * w_pre[y] * rg * sn;
    }
    out[i] = make_double2(re, im);
  }
}
// closs, table_mode 1: Algo 1 step 14, sums over r, s and the pre-sphere (reading Q-3).
__global__ void k_closs1(cplx* out, int pair, int N, int N_rho, int M, double L, double gam, double eta,
                         const double* rho, const double* w_rho, const double* sigma, const double* w_sigma,
                         int M_pre, const double* sig_pre, const double* w_pre) {
  const int N3 = N * N * N;
  const double pi = 3.14159265358979323846;
  for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < N3; idx += gridDim.x * blockDim.x) {
    int kx, ky, kz; spec_freq(idx, N, kx, ky, kz);
    double re = 0.0, im = 0.0;
    for (int r = 0; r < N_rho; ++r) {
      double rg = pow(rho[r], gam + 2.0), rp = pi * rho[r] / L;
      for (int s = 0; s < M; ++s)
        for (int y = 0; y < M_pre; ++y) {
          double dot = sigma[s * 3] * sig_pre[y * 3] + sigma[s * 3 + 1] * sig_pre[y * 3 + 1] + sigma[s * 3 + 2] * sig_pre[y * 3 + 2];
          double wgt = w_rho[r] * w_sigma[s] * pow(1.0 + dot, eta) * w_pre[y] * rg;
          double th = -rp * (kx * sig_pre[y * 3] + ky * sig_pre[y * 3 + 1] + kz * sig_pre[y * 3 + 2]);
          double sn, cs; sincos(th, &sn, &cs);
          re += wgt * cs; im += wgt * sn;
        }
    }
    out[(size_t)pair * N3 + idx] = make_double2(re, im);
  }
}

// ---- expansion kernels for dgfs_get_tables (Algorithm 1's layout: z = (ix*N+iy)*N+iz) ----
__global__ void k_expand_a(double* a, int N, int N_rho, int M, double L, const double* rho, const double* sigma) {
  const int N3 = N * N * N;
  const long total = (long)N_rho * M * N3;
  const double pi = 3.14159265358979323846;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int z = i % N3; long t = i / N3; int s = t % M, r = t / M;
    int iz = z % N, iy = (z / N) % N, ix = z / (N * N);
    double dot = signed_freq(ix, N) * sigma[s * 3] + signed_freq(iy, N) * sigma[s * 3 + 1] + signed_freq(iz, N) * sigma[s * 3 + 2];
    a[i] = pi / L * rho[r] * dot;                                          // Algo 1 step 7
  }
}
__global__ void k_expand_b(cplx* b, int pair, DevTables tab) {
  const int N = tab.N, N3 = tab.N3;
  const long total = (long)tab.N_rho * tab.M * N3;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    int z = i % N3; long t = i / N3; int s = t % tab.M, r = t / tab.M;
    int iz = z % N, iy = (z / N) % N, ix = z / (N * N);
    if (tab.full[pair]) {
      b[i] = bfull_at(tab, pair, r, s, signed_freq(ix, N), signed_freq(iy, N), signed_freq(iz, N));
    } else {
      int kx = signed_freq(ix, N), ky = signed_freq(iy, N), kz = signed_freq(iz, N);
      b[i] = make_double2(tab.bvhs[((size_t)pair * tab.N_rho + r) * tab.K2n + kx * kx + ky * ky + kz * kz], 0.0);
    }
  }
}
__global__ void k_expand_c(cplx* cc, int pair, DevTables tab) {
  const int N = tab.N, N3 = tab.N3;
  for (int z = blockIdx.x * blockDim.x + threadIdx.x; z < N3; z += gridDim.x * blockDim.x) {
    int iz = z % N, iy = (z / N) % N, ix = z / (N * N);
    cc[z] = tab.closs[(size_t)pair * N3 + ((size_t)iz * N + ix) * N + iy];
  }
}

template <class T>
static int dev_upload(dgfs_ctx* c, T** dptr, const T* h, size_t n, const char* what) {
  int rc = check_cuda(c, cudaMalloc((void**)dptr, n * sizeof(T)), what);
  if (rc) return rc;
  return check_cuda(c, cudaMemcpy(*dptr, h, n * sizeof(T), cudaMemcpyHostToDevice), what);
}

int build_tables(dgfs_ctx* c) {
  const int ns = c->ns, N = c->N, Nr = c->N_rho, M = c->M, np = c->npairs, N3 = c->N3;
  int rc;
  double *d_mass = nullptr, *d_gam = nullptr, *d_eta = nullptr, *d_wsig = nullptr, *d_sigpre = nullptr, *d_wpre = nullptr;
  if ((rc = dev_upload(c, &d_mass, c->mass.data(), ns, "upload mass"))) return rc;
  if ((rc = dev_upload(c, &d_gam, c->gam.data(), np, "upload gamma"))) return rc;
  if ((rc = dev_upload(c, &d_eta, c->eta.data(), np, "upload eta"))) return rc;
  if ((rc = dev_upload(c, &c->d_rho, c->rho.data(), Nr, "upload rho"))) return rc;
  if ((rc = dev_upload(c, &c->d_w_rho, c->w_rho.data(), Nr, "upload w_rho"))) return rc;
  if ((rc = dev_upload(c, &c->d_sigma, c->sigma.data(), 3 * M, "upload sigma"))) return rc;
  if ((rc = dev_upload(c, &d_wsig, c->w_sigma.data(), M, "upload w_sigma"))) return rc;
  if ((rc = dev_upload(c, &c->d_beta, c->beta.data(), np, "upload beta"))) return rc;
  if ((rc = dev_upload(c, &c->d_full, c->full.data(), np, "upload flags"))) return rc;
  if (c->table_mode == 1) {
    if ((rc = dev_upload(c, &d_sigpre, c->sigma_pre.data(), c->sigma_pre.size(), "upload sigma_pre"))) return rc;
    if ((rc = dev_upload(c, &d_wpre, c->w_pre.data(), c->w_pre.size(), "upload w_pre"))) return rc;
  }
  // v0 pipeline: antipodal symmetries of VHS pairs (R-10, R-11; same reasoning as in collide_v1.cu)
  c->v0_sskip.assign((size_t)np * M, 0);
  c->v0_wfac.assign((size_t)np * M, 1.0);
  c->v0_tsrc.resize(np);
  for (int pr = 0; pr < np; ++pr) c->v0_tsrc[pr] = pr;
  {
    const char* ap = getenv("DGFS_V1_ANTIPODAL");
    const bool on = !(ap && atoi(ap) == 0);
    std::vector<int> anti(M, -1);
    bool sym_w = on;
    for (int s2 = 0; s2 < M; ++s2) {
      for (int s3 = 0; s3 < M; ++s3)
        if (c->sigma[3 * s3] == -c->sigma[3 * s2] && c->sigma[3 * s3 + 1] == -c->sigma[3 * s2 + 1] &&
            c->sigma[3 * s3 + 2] == -c->sigma[3 * s2 + 2]) { anti[s2] = s3; break; }
      if (anti[s2] < 0 || c->w_sigma[anti[s2]] != c->w_sigma[s2]) sym_w = false;
    }
    for (int p = 0; on && p < ns; ++p) {
      const int dp = p * ns + p;
      if (!c->full[dp])
        for (int s2 = 0; s2 < M; ++s2)
          if (anti[s2] > s2) {
            c->v0_sskip[(size_t)dp * M + anti[s2]] = 1;
            c->v0_wfac[(size_t)dp * M + s2] = (c->w_sigma[s2] + c->w_sigma[anti[s2]]) / c->w_sigma[s2];
          }
      for (int q = p + 1; sym_w && q < ns; ++q) {
        if (c->full[p * ns + q] || c->full[q * ns + p]) continue;
        c->v0_tsrc[q * ns + p] = p * ns + q;
        for (int s2 = 0; s2 < M; ++s2) c->v0_sskip[(size_t)(q * ns + p) * M + s2] = 1;
      }
    }
  }
  if ((rc = dev_upload(c, &c->d_v0_sskip, c->v0_sskip.data(), c->v0_sskip.size(), "upload antipode masks"))) return rc;
  if ((rc = dev_upload(c, &c->d_v0_tsrc, c->v0_tsrc.data(), c->v0_tsrc.size(), "upload pair sources"))) return rc;
  if ((rc = dev_upload(c, &c->d_v0_wfac, c->v0_wfac.data(), c->v0_wfac.size(), "upload weight factors"))) return rc;
  const int TB = 256;
  auto blocks = [&](long total) { long b = (total + TB - 1) / TB; return (int)(b > 65535 * 8 ? 65535 * 8 : b); };

  size_t nphase = (size_t)np * Nr * M * 2 * 3 * N;
  if ((rc = check_cuda(c, cudaMalloc((void**)&c->d_phase, nphase * sizeof(cplx)), "alloc phase table"))) return rc;
  k_phase<<<blocks(nphase), TB>>>(c->d_phase, ns, N, Nr, M, c->L, d_mass, c->d_rho, c->d_sigma, d_wsig, c->d_v0_wfac);

  size_t nb = (size_t)np * Nr * c->K2n;
  if ((rc = check_cuda(c, cudaMalloc((void**)&c->d_bvhs, nb * sizeof(double)), "alloc b (VHS) table"))) return rc;
  k_bvhs<<<blocks(nb), TB>>>(c->d_bvhs, ns, Nr, c->K2n, c->L, d_mass, d_gam, c->d_rho);

  if ((rc = check_cuda(c, cudaMalloc((void**)&c->d_closs, (size_t)np * N3 * sizeof(cplx)), "alloc c table"))) return rc;
  if (c->table_mode == 0)
    k_closs0<<<blocks((long)np * N3), TB>>>(c->d_closs, ns, N, Nr, c->L, d_gam, d_eta, c->d_rho, c->d_w_rho);

  // Full tables (VSS pairs, table_mode 1).  table_mode 0: b_rs(k) depends on k through |k| and k . sigma_s only, so
  // sphere points that are signed axis permutations of one another share one table on the extended grid (bfull_at in
  // ctx.h).  DGFS_BTABLE=full keeps [r][s][N^3] (the paper's layout).
  c->bsym = 0; c->nref = 0; c->bref.clear(); c->bmap.assign(M, make_int4(0, 0, 0, 0));
  if (c->any_full && c->table_mode == 0) {
    const char* bt = getenv("DGFS_BTABLE");
    const int E = N + 1, H = N / 2;
    const int S3[3] = {E, 1, E * E};                                   // stride of the x, y, z index ([kz][kx][ky])
    // only the permutations that keep y in place: the consumers' lanes run along ky, and with ky mapped to another
    // axis of the reference table every lane of a load would touch its own 128-byte line (measured on config c3:
    // k_zfwd_full 3.2x slower with the full group of 48, whose one orbit would store the icosahedron 12x smaller)
    static const int perms[2][3] = {{0, 1, 2}, {2, 1, 0}};
    for (int s2 = 0; s2 < M; ++s2) {
      bool found = false;
      for (int u = 0; u < (int)c->bref.size() && !found; ++u) {
        const double* su = &c->sigma[3 * c->bref[u]];
        for (int pi_ = 0; pi_ < 2 && !found; ++pi_) {
          int eps[3]; bool ok = true;
          for (int d = 0; d < 3 && ok; ++d) {                          // sigma_s[d] = eps_d sigma_u[perm(d)]
            const double a = c->sigma[3 * s2 + d], b = su[perms[pi_][d]];
            if (fabs(a - b) <= 1e-15) eps[d] = 1;
            else if (fabs(a + b) <= 1e-15) eps[d] = -1;
            else ok = false;
          }
          if (!ok) continue;
          // k . sigma_s = k' . sigma_u with k'_{perm(d)} = eps_d k_d
          c->bmap[s2] = make_int4(u * E * E * E + H * (E * E + E + 1), eps[0] * S3[perms[pi_][0]],
                                  eps[1] * S3[perms[pi_][1]], eps[2] * S3[perms[pi_][2]]);
          found = true;
        }
      }
      if (!found) {
        c->bmap[s2] = make_int4((int)c->bref.size() * E * E * E + H * (E * E + E + 1), S3[0], S3[1], S3[2]);
        c->bref.push_back(s2);
      }
    }
    c->nref = (int)c->bref.size();
    c->bsym = !(bt && std::string(bt) == "full") && (size_t)c->nref * E * E * E < (size_t)M * N3;
    if (c->bsym) {
      if ((rc = dev_upload(c, &c->d_bref, c->bref.data(), c->bref.size(), "upload reference points"))) return rc;
      if ((rc = dev_upload(c, &c->d_bmap, c->bmap.data(), c->bmap.size(), "upload table maps"))) return rc;
    }
  }
  c->h_bfull.assign(np, nullptr);
  c->table_bytes = 0;
  for (int pair = 0; pair < np; ++pair) {
    int p = pair / ns, q = pair % ns;
    if (c->full[pair]) {
      const size_t E3 = (size_t)(N + 1) * (N + 1) * (N + 1);
      size_t n = c->bsym ? (size_t)Nr * c->nref * E3 : (size_t)Nr * M * N3;
      if ((rc = check_cuda(c, cudaMalloc((void**)&c->h_bfull[pair], n * sizeof(cplx)), "alloc full b table"))) return rc;
      c->table_bytes += n * sizeof(cplx);
      if (c->bsym)
        k_bsym_series<<<blocks(n), 128>>>(c->h_bfull[pair], p, q, N, Nr, c->nref, c->d_bref, c->L, d_mass, c->gam[pair],
                                          c->eta[pair], c->d_rho, c->d_sigma);
      else if (c->table_mode == 0)
        k_bfull_series<<<blocks(n), 128>>>(c->h_bfull[pair], p, q, N, Nr, M, c->L, d_mass, c->gam[pair], c->eta[pair],
                                           c->d_rho, c->d_sigma);
      else
        k_bfull_pre<<<blocks(n), TB>>>(c->h_bfull[pair], p, q, N, Nr, M, c->L, d_mass, c->gam[pair], c->eta[pair],
                                       c->d_rho, c->d_sigma, c->M_pre_count(), d_sigpre, d_wpre);
    }
    if (c->table_mode == 1)
      k_closs1<<<blocks(N3), TB>>>(c->d_closs, pair, N, Nr, M, c->L, c->gam[pair], c->eta[pair], c->d_rho, c->d_w_rho,
                                   c->d_sigma, d_wsig, c->M_pre_count(), d_sigpre, d_wpre);
  }
  if ((rc = dev_upload(c, &c->d_bfull, c->h_bfull.data(), np, "upload b pointers"))) return rc;
  if ((rc = check_cuda(c, cudaGetLastError(), "table kernels launch"))) return rc;
  if ((rc = check_cuda(c, cudaDeviceSynchronize(), "table kernels"))) return rc;
  cudaFree(d_mass); cudaFree(d_gam); cudaFree(d_eta); cudaFree(d_wsig); cudaFree(d_sigpre); cudaFree(d_wpre);

  DevTables& t = c->tab;
  t.ns = ns; t.npairs = np; t.N = N; t.N3 = N3; t.N_rho = Nr; t.M = M; t.K2n = c->K2n;
  t.phase = c->d_phase; t.bvhs = c->d_bvhs; t.bfull = c->d_bfull; t.closs = c->d_closs;
  t.w_rho = c->d_w_rho; t.beta = c->d_beta; t.full = c->d_full; t.sskip = c->d_v0_sskip; t.tsrc = c->d_v0_tsrc;
  t.bsym = c->bsym; t.nref = c->nref; t.bmap = c->d_bmap;
  return DGFS_OK;
}

}  // namespace dgfs

using namespace dgfs;

extern "C" const char* dgfs_last_error(const dgfs_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

extern "C" int dgfs_create(const dgfs_params* P, dgfs_ctx** out) {
  if (!out) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: out is NULL");
  *out = nullptr;
  if (!P) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: params is NULL");
  if (P->ns < 1 || P->ns > 16) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: ns must be in 1..16");
  if (!P->mass || !P->omega || !P->alpha) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: mass, omega, alpha must not be NULL");
  const int N = P->N;
  if (!(N == 8 || N == 16 || N == 24 || N == 32 || N == 48))
    return set_error(nullptr, (N > 0 && N % 2 == 0) ? DGFS_ENOSUP : DGFS_EINVAL,
                     "dgfs_create: N must be even; supported values are 8, 16, 24, 32, 48");
  if (P->N_rho < 1 || P->N_rho > 4096) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: N_rho must be in 1..4096");
  if (P->M < 1 || P->M > 4096) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: M must be in 1..4096");
  if (!(P->L > 0) || !std::isfinite(P->L)) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: L must be positive");
  if ((P->sigma == nullptr) != (P->w_sigma == nullptr))
    return set_error(nullptr, DGFS_EINVAL, "dgfs_create: sigma and w_sigma must both be given or both be NULL");
  if (P->table_mode != 0 && P->table_mode != 1) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: table_mode must be 0 or 1");
  if (P->precision != 0 && P->precision != 1) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: precision must be 0 (fp64) or 1 (fp32 inner loop)");
  if (P->table_mode == 1 && (P->M_pre < 1 || !P->sigma_pre || !P->w_pre))
    return set_error(nullptr, DGFS_EINVAL, "dgfs_create: table_mode 1 needs M_pre >= 1, sigma_pre and w_pre");
  const int ns = P->ns, np = ns * ns;
  for (int p = 0; p < ns; ++p)
    if (!(P->mass[p] > 0) || !std::isfinite(P->mass[p])) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: masses must be positive");
  for (int i = 0; i < np; ++i) {
    if (!(P->alpha[i] > 0) || !std::isfinite(P->alpha[i])) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: alpha_pq must be positive");
    if (!(P->omega[i] < 2.5) || !std::isfinite(P->omega[i]))
      return set_error(nullptr, DGFS_EINVAL, "dgfs_create: omega_pq must be < 2.5 (Gamma(2.5 - omega) pole in Eq. 6)");
    if (P->kn && !(P->kn[i] > 0)) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: Kn_pq must be positive");
  }
  const double pi = 3.14159265358979323846;
  std::vector<double> sig, wsig;
  if (P->sigma) {
    sig.assign(P->sigma, P->sigma + 3 * P->M); wsig.assign(P->w_sigma, P->w_sigma + P->M);
    double sw = 0;
    for (int s = 0; s < P->M; ++s) {
      double n2 = sig[3 * s] * sig[3 * s] + sig[3 * s + 1] * sig[3 * s + 1] + sig[3 * s + 2] * sig[3 * s + 2];
      if (fabs(n2 - 1.0) > 1e-12) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: sigma rows must be unit vectors");
      sw += wsig[s];
    }
    if (fabs(sw - 4 * pi) > 1e-12 * 4 * pi) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: w_sigma must sum to 4 pi");
  } else if (!builtin_sphere(P->M, sig, wsig)) {
    return set_error(nullptr, DGFS_EINVAL, "dgfs_create: built-in sphere rules exist for M in {6, 12, 32}; pass sigma/w_sigma");
  }
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev == 0)
    return set_error(nullptr, DGFS_ECUDA, std::string("dgfs_create: no CUDA device (") + cudaGetErrorString(ce) + "); there is no CPU fallback");
  if (P->device < 0 || P->device >= ndev) return set_error(nullptr, DGFS_EINVAL, "dgfs_create: device ordinal out of range");
  if ((ce = cudaSetDevice(P->device)) != cudaSuccess) return set_error(nullptr, DGFS_ECUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(ce));

  dgfs_ctx* c = new dgfs_ctx();
  c->device = P->device; c->ns = ns; c->npairs = np; c->N = N; c->N3 = N * N * N; c->N_rho = P->N_rho; c->M = P->M;
  c->L = P->L; c->table_mode = P->table_mode;
  c->nyq_filter = P->nyquist_filter != 0;
  c->precision = P->precision;
  c->K2n = 3 * (N / 2) * (N / 2) + 1;
  c->mass.assign(P->mass, P->mass + ns);
  c->omega.assign(P->omega, P->omega + np);
  c->alpha.assign(P->alpha, P->alpha + np);
  c->kn.assign(np, 1.0);
  if (P->kn) c->kn.assign(P->kn, P->kn + np);
  c->sigma = sig; c->w_sigma = wsig;
  if (P->table_mode == 1) {
    c->sigma_pre.assign(P->sigma_pre, P->sigma_pre + 3 * P->M_pre);
    c->w_pre.assign(P->w_pre, P->w_pre + P->M_pre);
  }
  // Eq. 9, reading RAD-1: one global R from (max mass, min mass)
  double ma = c->mass[0], mb = c->mass[0];
  for (double m : c->mass) { ma = fmax(ma, m); mb = fmin(mb, m); }
  c->R = (P->R > 0) ? P->R : 4.0 * P->L / (1.0 + fmax(4.0 * ma / (mb + ma), 2.0) + sqrt(1.0 + ma / mb));
  // radial rule on [0, R] (O-2)
  std::vector<double> gx, gw;
  gauss_legendre(P->N_rho, gx, gw);
  c->rho.resize(P->N_rho); c->w_rho.resize(P->N_rho);
  for (int r = 0; r < P->N_rho; ++r) { c->rho[r] = 0.5 * c->R * (gx[r] + 1.0); c->w_rho[r] = 0.5 * c->R * gw[r]; }
  // exponents (reading G-1) and prefactors (Eq. 6)
  c->gam.resize(np); c->eta.resize(np); c->beta.resize(np); c->full.resize(np);
  for (int p = 0; p < ns; ++p) for (int q = 0; q < ns; ++q) {
    int i = p * ns + q;
    c->gam[i] = 2.0 * (1.0 - c->omega[i]);
    c->eta[i] = c->alpha[i] - 1.0;
    double mp = c->mass[p], mq = c->mass[q];
    c->beta[i] = P->prefactor ? P->prefactor[i]
                              : (1.0 / c->kn[i]) / sqrt(1.0 + mp / mq) / pow(mp * mq / (mp + mq), c->omega[i] - 0.5) *
                                    c->alpha[i] / (exp2(1.0 + c->alpha[i]) * tgamma(2.5 - c->omega[i]) * pi);
    c->full[i] = (c->table_mode == 1 || c->eta[i] != 0.0) ? 1 : 0;
    c->any_full = c->any_full || c->full[i];
  }
  const char* env = getenv("DGFS_SCRATCH_MB");
  c->scratch_budget = (size_t)(env ? atol(env) : 3072) << 20;
  int rc = build_tables(c);
  if (rc != DGFS_OK) { g_create_error = c->err; dgfs_destroy(c); return rc; }
  // DGFS_PIPELINE=v0 forces the stage-per-kernel pipeline (the parity tests cover both)
  const char* pipe = getenv("DGFS_PIPELINE");
  // pipeline choice: v1 (collide_v1.cu): N <= 32, or N = 48 when no pair needs a full b table (collide_v1_wide.cuh)
  c->use_v1 = (N <= 32 || !c->any_full) && !(pipe && std::string(pipe) == "v0");
  if (c->precision == 1 && (!c->use_v1 || c->any_full || N > 32)) {
    g_create_error = "dgfs_create: precision 1 is implemented for VHS pairs (alpha = 1, table_mode 0) with N <= 32 on the default pipeline";
    dgfs_destroy(c);
    return DGFS_ENOSUP;
  }
  if (c->use_v1) {
    const char* ch = getenv("DGFS_V1_CHUNK");
    if (N > 32) c->v1_chunk = 256;                  // 1.7 MB arrays: half the points per launch group for the same workspace
    if (ch && atoi(ch) > 0) c->v1_chunk = atoi(ch);
    const char* rg = getenv("DGFS_V1_RGROUP");
    if (rg && atoi(rg) > 0) c->v1_rgroup = atoi(rg);
    if (c->v1_rgroup > c->N_rho) c->v1_rgroup = c->N_rho;
    rc = build_tables_v1(c);
    if (rc == DGFS_OK) rc = init_streams_v1(c);
    if (rc != DGFS_OK) { g_create_error = c->err; dgfs_destroy(c); return rc; }
  }
  if ((rc = check_cuda(c, cudaEventCreateWithFlags(&c->ev_last, cudaEventDisableTiming), "event create")) != DGFS_OK) {
    g_create_error = c->err; dgfs_destroy(c); return rc;
  }
  *out = c;
  return DGFS_OK;
}

extern "C" void dgfs_destroy(dgfs_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaFree(c->d_phase); cudaFree(c->d_bvhs); cudaFree(c->d_closs); cudaFree(c->d_w_rho); cudaFree(c->d_beta);
  cudaFree(c->d_rho); cudaFree(c->d_sigma); cudaFree(c->d_full); cudaFree(c->d_bfull);
  cudaFree(c->d_v0_sskip); cudaFree(c->d_v0_tsrc); cudaFree(c->d_v0_wfac); cudaFree(c->d_bref); cudaFree(c->d_bmap);
  for (auto p : c->h_bfull) cudaFree(p);
  cudaFree(c->ws); cudaFree(c->dg_ws);
  drop_graphs_v1(c);
  free_graph_stream_v1(c);
  free_tables_v1(c);
  free_streams_v1(c);
  if (c->ev_last) cudaEventDestroy(c->ev_last);
  for (int b = 0; b < 2; ++b) { cudaFree(c->hp_f[b]); cudaFree(c->hp_q[b]); }
  for (int i = 0; i < 3; ++i) {
    if (c->hp_stream[i]) cudaStreamDestroy(c->hp_stream[i]);
    for (int b = 0; b < 2; ++b) if (c->hp_ev[i][b]) cudaEventDestroy(c->hp_ev[i][b]);
  }
  c->prof.drain();
  for (auto e : c->prof.pool) cudaEventDestroy(e);
  delete c;
}

extern "C" size_t dgfs_table_bytes(const dgfs_ctx* c) { return c ? c->table_bytes : 0; }

extern "C" int dgfs_get_quadrature(const dgfs_ctx* c, double* R, double* rho, double* w_rho, double* sigma,
                                   double* w_sigma, double* beta) {
  if (!c) return DGFS_EINVAL;
  if (R) *R = c->R;
  if (rho) memcpy(rho, c->rho.data(), sizeof(double) * c->N_rho);
  if (w_rho) memcpy(w_rho, c->w_rho.data(), sizeof(double) * c->N_rho);
  if (sigma) memcpy(sigma, c->sigma.data(), sizeof(double) * 3 * c->M);
  if (w_sigma) memcpy(w_sigma, c->w_sigma.data(), sizeof(double) * c->M);
  if (beta) memcpy(beta, c->beta.data(), sizeof(double) * c->npairs);
  return DGFS_OK;
}

extern "C" int dgfs_get_tables(dgfs_ctx* c, int p, int q, double* a, double* b, double* cc) {
  if (!c) return DGFS_EINVAL;
  if (p < 0 || p >= c->ns || q < 0 || q >= c->ns) return set_error(c, DGFS_EINVAL, "dgfs_get_tables: pair out of range");
  cudaSetDevice(c->device);
  const size_t n = (size_t)c->N_rho * c->M * c->N3;
  const int pair = p * c->ns + q;
  int rc;
  if (a) {
    double* d; if ((rc = check_cuda(c, cudaMalloc((void**)&d, n * sizeof(double)), "dgfs_get_tables alloc"))) return rc;
    k_expand_a<<<4096, 256>>>(d, c->N, c->N_rho, c->M, c->L, c->d_rho, c->d_sigma);
    rc = check_cuda(c, cudaMemcpy(a, d, n * sizeof(double), cudaMemcpyDeviceToHost), "dgfs_get_tables copy a");
    cudaFree(d); if (rc) return rc;
  }
  if (b) {
    cplx* d; if ((rc = check_cuda(c, cudaMalloc((void**)&d, n * sizeof(cplx)), "dgfs_get_tables alloc"))) return rc;
    k_expand_b<<<4096, 256>>>(d, pair, c->tab);
    rc = check_cuda(c, cudaMemcpy(b, d, n * sizeof(cplx), cudaMemcpyDeviceToHost), "dgfs_get_tables copy b");
    cudaFree(d); if (rc) return rc;
  }
  if (cc) {
    cplx* d; if ((rc = check_cuda(c, cudaMalloc((void**)&d, c->N3 * sizeof(cplx)), "dgfs_get_tables alloc"))) return rc;
    k_expand_c<<<128, 256>>>(d, pair, c->tab);
    rc = check_cuda(c, cudaMemcpy(cc, d, c->N3 * sizeof(cplx), cudaMemcpyDeviceToHost), "dgfs_get_tables copy c");
    cudaFree(d); if (rc) return rc;
  }
  return DGFS_OK;
}
