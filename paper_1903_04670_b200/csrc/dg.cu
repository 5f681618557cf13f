// dg.cu -- dgfs_step / dgfs_advect_rhs: 1-D nodal DG transport and SSP-RK3 around dgfs_collide
// (secondary rows D1-D4 of SURVEY.md section 8(a); Table 2).
//
// The paper gives no formulas for its spatial scheme; readings DG-1..DG-3 of DESIGN.md section 2:
//   d/dt f_e = -(2/h) c_x D f_e + (2/h) M^-1 [ e_K (c_x f_{e,K} - F*_{e+1/2}) - e_1 (c_x f_{e,1} - F*_{e-1/2}) ] + Q
// on K = order+1 Gauss-Lobatto-Legendre nodes, exact mass matrix, upwind F*, purely diffuse walls (incoming
// half range = n_w Maxw(1, u_w, T_w; m_p), n_w from zero net mass flux per species with the discrete velocity
// sums), Shu-Osher SSP-RK3.  Transport is HBM-bound (one read of the stage state, of Q and of the step's
// start state, one write, per stage); one kernel per stage fuses volume term, interface flux, lift, wall
// inflow and the Runge-Kutta combination.
#include <cmath>
#include <cstring>
#include "ctx.h"

namespace dgfs {

constexpr int DG_MAXK = 8;

struct DgOps {
  int K;
  double D[DG_MAXK][DG_MAXK];     // D[i][j] = l_j'(xi_i)
  double lift_r[DG_MAXK];         // column K-1 of M^-1
  double lift_l[DG_MAXK];         // column 0 of M^-1
};

// ---- host: Gauss-Lobatto-Legendre nodes, differentiation matrix, M^-1 = V V^T -----------------------
static void legendre(int n, double x, double* P, double* dP) {   // P_n(x), P_n'(x)
  double p0 = 1.0, p1 = x, d0 = 0.0, d1 = 1.0;
  if (n == 0) { *P = 1.0; *dP = 0.0; return; }
  for (int k = 2; k <= n; ++k) {
    const double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
    const double d2 = d0 + (2 * k - 1) * p1;
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  *P = p1; *dP = d1;
}

static void build_ops(int order, DgOps* ops) {
  const int K = order + 1, n = K - 1;
  const double pi = 3.14159265358979323846;
  double xi[DG_MAXK];
  xi[0] = -1.0; xi[K - 1] = 1.0;
  for (int i = 1; i < K - 1; ++i) {
    // Newton on q(x) = P_n'(x), q' = (2x P_n' - n(n+1) P_n) / (1 - x^2), from the Chebyshev-Gauss-Lobatto guess
    double x = -cos(pi * i / n);
    for (int it = 0; it < 100; ++it) {
      double P, dP; legendre(n, x, &P, &dP);
      const double ddP = (2.0 * x * dP - n * (n + 1.0) * P) / (1.0 - x * x);
      const double dx = dP / ddP;
      x -= dx;
      if (fabs(dx) < 1e-16) break;
    }
    xi[i] = x;
  }
  for (int i = 0; i < K / 2; ++i) { const double a = 0.5 * (xi[K - 1 - i] - xi[i]); xi[i] = -a; xi[K - 1 - i] = a; }
  if (K % 2) xi[K / 2] = 0.0;
  // barycentric differentiation matrix
  double w[DG_MAXK];
  for (int j = 0; j < K; ++j) { w[j] = 1.0; for (int k = 0; k < K; ++k) if (k != j) w[j] /= (xi[j] - xi[k]); }
  ops->K = K;
  memset(ops->D, 0, sizeof(ops->D));
  for (int i = 0; i < K; ++i) {
    double s = 0.0;
    for (int j = 0; j < K; ++j) if (j != i) { ops->D[i][j] = (w[j] / w[i]) / (xi[i] - xi[j]); s += ops->D[i][j]; }
    ops->D[i][i] = -s;
  }
  // M^-1 = V V^T with the orthonormal Legendre Vandermonde V[i][j] = sqrt((2j+1)/2) P_j(xi_i)
  double V[DG_MAXK][DG_MAXK];
  for (int i = 0; i < K; ++i) for (int j = 0; j < K; ++j) {
    double P, dP; legendre(j, xi[i], &P, &dP);
    V[i][j] = sqrt(0.5 * (2 * j + 1)) * P;
  }
  for (int i = 0; i < K; ++i) {
    double a = 0.0, b = 0.0;
    for (int j = 0; j < K; ++j) { a += V[i][j] * V[K - 1][j]; b += V[i][j] * V[0][j]; }
    ops->lift_r[i] = a; ops->lift_l[i] = b;
  }
}

// ---- device ---------------------------------------------------------------------------------------
__device__ __forceinline__ double node_cx(int z, int N, double L) {
  return -L + ((z / (N * N)) + 0.5) * (2.0 * L / N);
}

// wall Maxwellians Maxw(1, u_w, T_w; m_p) on the grid (reading M-1): Wt[wall][p][z]
__global__ void k_dg_wallmaxw(double* __restrict__ Wt, int ns, int N, double L, const double* __restrict__ mass,
                              double T0, double T1, double u0x, double u0y, double u0z, double u1x, double u1y, double u1z) {
  const int N3 = N * N * N;
  const double pi = 3.14159265358979323846;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < 2 * ns * N3; i += gridDim.x * blockDim.x) {
    const int z = i % N3, p = (i / N3) % ns, wall = i / (N3 * ns);
    const double T = wall ? T1 : T0, ux = wall ? u1x : u0x, uy = wall ? u1y : u0y, uz = wall ? u1z : u0z;
    const double h = 2.0 * L / N;
    const double cx = -L + ((z / (N * N)) + 0.5) * h, cy = -L + (((z / N) % N) + 0.5) * h, cz = -L + ((z % N) + 0.5) * h;
    const double m = mass[p];
    const double e = exp(-m * (cx - ux) * (cx - ux) / T) * exp(-m * (cy - uy) * (cy - uy) / T) * exp(-m * (cz - uz) * (cz - uz) / T);
    Wt[i] = pow(m / (pi * T), 1.5) * e;
  }
}

// n_w[wall][p] = (outgoing mass flux of the adjacent trace) / (incoming flux of the unit wall Maxwellian); block per (wall, p)
__global__ void __launch_bounds__(256) k_dg_wall(const double* __restrict__ f, const double* __restrict__ Wt,
                                                 double* __restrict__ nw, int ne, int K, int ns, int N, double L) {
  const int N3 = N * N * N;
  const int p = blockIdx.x % ns, wall = blockIdx.x / ns;
  const double* tr = f + ((size_t)(wall ? (ne - 1) * K + (K - 1) : 0) * ns + p) * N3;
  const double* W = Wt + ((size_t)wall * ns + p) * N3;
  double out = 0.0, in = 0.0;
  for (int z = threadIdx.x; z < N3; z += 256) {
    const double cx = node_cx(z, N, L);
    const bool leaving = wall ? (cx > 0) : (cx < 0);
    if (leaving) out += fabs(cx) * tr[z]; else in += fabs(cx) * W[z];
  }
  __shared__ double so[256], si[256];
  so[threadIdx.x] = out; si[threadIdx.x] = in;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) { so[threadIdx.x] += so[threadIdx.x + s]; si[threadIdx.x] += si[threadIdx.x + s]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) nw[blockIdx.x] = so[0] / si[0];
}

// One Runge-Kutta stage (or the bare right-hand side): thread per (element, species, velocity node).
//   rhs = transport(u) [+ Q];   out = rhs                      if a == 0 && b == 0 (dgfs_advect_rhs)
//                               out = a u0 + b (u + dt rhs)    otherwise
template <int K>
__global__ void __launch_bounds__(256) k_dg_stage(DgOps ops, const double* __restrict__ u, const double* u0,
                                                  const double* __restrict__ Q, double* out,
                                                  const double* __restrict__ Wt, const double* __restrict__ nw,
                                                  int ne, int ns, int N, double L, double jac, double dt, double a, double b) {
  const int N3 = N * N * N;
  const size_t total = (size_t)ne * ns * N3;
  const size_t i = blockIdx.x * (size_t)256 + threadIdx.x;
  if (i >= total) return;
  const int z = (int)(i % N3), p = (int)((i / N3) % ns), e = (int)(i / ((size_t)N3 * ns));
  const size_t nstride = (size_t)ns * N3;                       // between nodes of an element
  const size_t base = ((size_t)e * K * ns + p) * N3 + z;
  const double cx = node_cx(z, N, L);
  double fe[K];
#pragma unroll
  for (int k = 0; k < K; ++k) fe[k] = u[base + k * nstride];
  // upwind interface values (reading DG-1) and diffuse walls (DG-2)
  double jump_l = 0.0, jump_r = 0.0;
  if (cx > 0) {
    const double up = (e > 0) ? u[base - nstride] : nw[p] * Wt[(size_t)p * N3 + z];
    jump_l = cx * (fe[0] - up);
  } else {
    const double up = (e < ne - 1) ? u[base + K * nstride] : nw[ns + p] * Wt[((size_t)ns + p) * N3 + z];
    jump_r = cx * (fe[K - 1] - up);
  }
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double d = 0.0;
#pragma unroll
    for (int j = 0; j < K; ++j) d = fma(ops.D[k][j], fe[j], d);
    double rhs = jac * (-cx * d + ops.lift_r[k] * jump_r - ops.lift_l[k] * jump_l);
    const size_t o = base + k * nstride;
    if (Q) rhs += Q[o];
    out[o] = (a == 0.0 && b == 0.0) ? rhs : a * u0[o] + b * (fe[k] + dt * rhs);
  }
}

template <int K>
static void launch_stage(const DgOps& ops, const double* u, const double* u0, const double* Q, double* out, const double* Wt,
                         const double* nw, int ne, int ns, int N, double L, double jac, double dt, double a, double b,
                         cudaStream_t st) {
  const size_t total = (size_t)ne * ns * N * N * N;
  k_dg_stage<K><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b);
}

static void stage(const DgOps& ops, const double* u, const double* u0, const double* Q, double* out, const double* Wt,
                  const double* nw, int ne, int ns, int N, double L, double jac, double dt, double a, double b, cudaStream_t st) {
  switch (ops.K) {
    case 2: launch_stage<2>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
    case 3: launch_stage<3>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
    case 4: launch_stage<4>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
    case 5: launch_stage<5>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
    case 6: launch_stage<6>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
    case 7: launch_stage<7>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
    case 8: launch_stage<8>(ops, u, u0, Q, out, Wt, nw, ne, ns, N, L, jac, dt, a, b, st); break;
  }
}

struct DgBuffers { double *w1, *w2, *Qb, *Wt, *nw, *mass; };

static int dg_setup(dgfs_ctx* c, const dgfs_mesh1d* mesh, const char* who, DgOps* ops, DgBuffers* B, cudaStream_t st) {
  if (!mesh) return set_error(c, DGFS_EINVAL, std::string(who) + ": mesh is NULL");
  if (mesh->ne < 1) return set_error(c, DGFS_EINVAL, std::string(who) + ": ne must be >= 1");
  if (mesh->order < 1 || mesh->order + 1 > DG_MAXK) return set_error(c, DGFS_EINVAL, std::string(who) + ": order must be in 1..7");
  if (!(mesh->x1 > mesh->x0)) return set_error(c, DGFS_EINVAL, std::string(who) + ": x1 must exceed x0");
  if (!(mesh->wall_T[0] > 0) || !(mesh->wall_T[1] > 0)) return set_error(c, DGFS_EINVAL, std::string(who) + ": wall temperatures must be positive");
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) return check_cuda(c, e, "cudaSetDevice");
  build_ops(mesh->order, ops);
  const size_t N3 = c->N3, state = (size_t)mesh->ne * ops->K * c->ns * N3;
  const size_t need = (3 * state + 2 * (size_t)c->ns * N3 + 2 * c->ns + c->ns + 64) * sizeof(double);
  if (need > c->dg_ws_bytes) {       // ordered on the caller's stream, like the collision workspace (collide.cu)
    if (c->ev_last_set) cudaStreamWaitEvent(st, c->ev_last, 0);
    if (c->dg_ws) cudaFreeAsync(c->dg_ws, st);
    c->dg_ws = nullptr; c->dg_ws_bytes = 0;
    int rc = check_cuda(c, cudaMallocAsync(&c->dg_ws, need, st), "DG workspace allocation");
    if (rc) { c->dg_ws = nullptr; return rc; }
    c->dg_ws_bytes = need;
  }
  double* w = (double*)c->dg_ws;
  B->w1 = w; B->w2 = w + state; B->Qb = w + 2 * state; B->Wt = w + 3 * state;
  B->nw = B->Wt + 2 * (size_t)c->ns * N3; B->mass = B->nw + 2 * c->ns;
  int rc = check_cuda(c, cudaMemcpyAsync(B->mass, c->mass.data(), c->ns * sizeof(double), cudaMemcpyHostToDevice, st), "upload masses");
  if (rc) return rc;
  k_dg_wallmaxw<<<256, 256, 0, st>>>(B->Wt, c->ns, c->N, c->L, B->mass, mesh->wall_T[0], mesh->wall_T[1], mesh->wall_u[0][0],
                                     mesh->wall_u[0][1], mesh->wall_u[0][2], mesh->wall_u[1][0], mesh->wall_u[1][1], mesh->wall_u[1][2]);
  return DGFS_OK;
}

}  // namespace dgfs

using namespace dgfs;

extern "C" int dgfs_advect_rhs(dgfs_ctx* c, const dgfs_mesh1d* mesh, const double* f, double* rhs, void* stream) {
  if (!c) return DGFS_EINVAL;
  if (!f || !rhs) return set_error(c, DGFS_EINVAL, "dgfs_advect_rhs: f and rhs must not be NULL");
  if (f == rhs) return set_error(c, DGFS_EINVAL, "dgfs_advect_rhs: rhs must not alias f");
  cudaStream_t st = (cudaStream_t)stream;
  DgOps ops; DgBuffers B;
  int rc = dg_setup(c, mesh, "dgfs_advect_rhs", &ops, &B, st);
  if (rc) return rc;
  const double jac = 2.0 * mesh->ne / (mesh->x1 - mesh->x0);
  k_dg_wall<<<2 * c->ns, 256, 0, st>>>(f, B.Wt, B.nw, mesh->ne, ops.K, c->ns, c->N, c->L);
  stage(ops, f, f, nullptr, rhs, B.Wt, B.nw, mesh->ne, c->ns, c->N, c->L, jac, 0.0, 0.0, 0.0, st);
  return check_cuda(c, cudaGetLastError(), "dgfs_advect_rhs launch");
}

// Forward Euler (the time stepping of the paper's Couette case, Table 2): f <- f + dt L(f).  One stage
// kernel per step (a = 0, b = 1); the stage reads the neighbour traces of its input, so it cannot run in place:
// f and the scratch state w1 alternate, with one device copy at the end when nsteps is odd.
extern "C" int dgfs_step_euler(dgfs_ctx* c, const dgfs_mesh1d* mesh, double* f, double dt, int nsteps, void* stream) {
  if (!c) return DGFS_EINVAL;
  if (!f) return set_error(c, DGFS_EINVAL, "dgfs_step_euler: f must not be NULL");
  if (nsteps < 0) return set_error(c, DGFS_EINVAL, "dgfs_step_euler: nsteps must be >= 0");
  if (!(dt > 0) || !std::isfinite(dt)) return set_error(c, DGFS_EINVAL, "dgfs_step_euler: dt must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  DgOps ops; DgBuffers B;
  int rc = dg_setup(c, mesh, "dgfs_step_euler", &ops, &B, st);
  if (rc) return rc;
  const int ne = mesh->ne, ns = c->ns, nx = ne * ops.K;
  const double jac = 2.0 * ne / (mesh->x1 - mesh->x0);
  const size_t bytes = (size_t)nx * ns * c->N * c->N * c->N * sizeof(double);
  double* u = f;
  double* v = B.w1;
  for (int n = 0; n < nsteps; ++n) {
    k_dg_wall<<<2 * ns, 256, 0, st>>>(u, B.Wt, B.nw, ne, ops.K, ns, c->N, c->L);
    if ((rc = run_collide(c, u, B.Qb, nx, false, st))) return rc;                    // sum_q beta_pq Q^(pq), Eq. 1
    stage(ops, u, u, B.Qb, v, B.Wt, B.nw, ne, ns, c->N, c->L, jac, dt, 0.0, 1.0, st);
    double* t = u; u = v; v = t;
  }
  if (u != f && (rc = check_cuda(c, cudaMemcpyAsync(f, u, bytes, cudaMemcpyDeviceToDevice, st), "dgfs_step_euler copy"))) return rc;
  return check_cuda(c, cudaGetLastError(), "dgfs_step_euler launch");
}

extern "C" int dgfs_step(dgfs_ctx* c, const dgfs_mesh1d* mesh, double* f, double dt, int nsteps, void* stream) {
  if (!c) return DGFS_EINVAL;
  if (!f) return set_error(c, DGFS_EINVAL, "dgfs_step: f must not be NULL");
  if (nsteps < 0) return set_error(c, DGFS_EINVAL, "dgfs_step: nsteps must be >= 0");
  if (!(dt > 0) || !std::isfinite(dt)) return set_error(c, DGFS_EINVAL, "dgfs_step: dt must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  DgOps ops; DgBuffers B;
  int rc = dg_setup(c, mesh, "dgfs_step", &ops, &B, st);
  if (rc) return rc;
  const int ne = mesh->ne, ns = c->ns, nx = ne * ops.K;
  const double jac = 2.0 * ne / (mesh->x1 - mesh->x0);
  // SSP-RK3 (reading DG-3): (state read, output, a, b) per stage; u0 = f throughout the step
  struct { const double* u; double* out; double a, b; } S[3] = {
      {f, B.w1, 0.0, 1.0}, {B.w1, B.w2, 0.75, 0.25}, {B.w2, f, 1.0 / 3.0, 2.0 / 3.0}};
  for (int n = 0; n < nsteps; ++n)
    for (int s = 0; s < 3; ++s) {
      k_dg_wall<<<2 * ns, 256, 0, st>>>(S[s].u, B.Wt, B.nw, ne, ops.K, ns, c->N, c->L);
      if ((rc = run_collide(c, S[s].u, B.Qb, nx, false, st))) return rc;          // sum_q beta_pq Q^(pq), Eq. 1
      stage(ops, S[s].u, f, B.Qb, S[s].out, B.Wt, B.nw, ne, ns, c->N, c->L, jac, dt, S[s].a, S[s].b, st);
    }
  return check_cuda(c, cudaGetLastError(), "dgfs_step launch");
}
