/*
 * dgfs.h -- C ABI of the B200-native multi-species DGFS Boltzmann collision operator.
 *
 * What the library computes is the fast Fourier-spectral collision operator Q^(pq)(f^(p), f^(q))
 * of arXiv 1903.04670 ("PAPER.md", cited as P:line):
 *   - Eq. 1       right-hand side  sum_q Kn_pq^-1 Q^(pq)            -> dgfs_collide
 *   - Eq. 2    definition of Q^(pq)
 *   - Eq. 13-17 low-rank separated kernel modes
 *   - Algorithm 1  precomputed tables a, b^(pq), c^(pq)          -> dgfs_create
 *   - Algorithm 2  FFT -> phase -> 2 iFFT -> product -> FFT -> weighted sum,
 *                              loss term as one convolution, prefactor beta   -> dgfs_collide[_pairs]
 *   - 1-D RKDG transport around it (readings DG-1..4)      -> dgfs_step
 *
 * Conventions (identical to DESIGN.md "Boundary"):
 *   - all floating point data is IEEE fp64;
 *   - velocity node z = (ix*N + iy)*N + iz (iz fastest), c = (c[ix], c[iy], c[iz]),
 *     c[j] = -L + (j + 1/2) * 2L/N (cell centred);
 *   - distribution functions  f[nx][ns][N^3]  (point slowest, species, velocity node fastest);
 *   - pointers documented "device" are CUDA device pointers on the context's device, pointers
 *     documented "host" are ordinary host pointers; the library never takes ownership of either;
 *   - `stream` is the caller's cudaStream_t passed as void* (NULL = legacy default stream);
 *     dgfs_collide* / dgfs_step enqueue work on it and return without synchronising;
 *   - the workspace of a context belongs to one call at a time: every call first waits, on its own stream, for the
 *     last launch of the previous call on that context, whichever stream that was issued on, so calls on different
 *     streams are safe and serialised; when a batch needs a larger workspace it is re-allocated in stream order
 *     (cudaFreeAsync / cudaMallocAsync on `stream`, no device-wide synchronisation) -- not possible while `stream`
 *     is being captured into a CUDA graph: call dgfs_reserve first;
 *   - every int-returning call returns DGFS_OK (0) or a negative DGFS_E* code, validates its
 *     arguments before any launch, and records a message readable with dgfs_last_error();
 *   - there is no CPU fallback: without a CUDA device dgfs_create fails with DGFS_ECUDA.
 */
#ifndef DGFS_H
#define DGFS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DGFS_OK        0
#define DGFS_EINVAL   -1   /* invalid argument (message says which)            */
#define DGFS_ECUDA    -2   /* CUDA runtime error (message carries the string)  */
#define DGFS_ENOMEM   -3   /* device allocation failed                         */
#define DGFS_ENOSUP   -4   /* valid request the library does not implement     */

typedef struct dgfs_ctx dgfs_ctx;   /* opaque: owns device tables + workspace */

/* Inputs of Algorithm 1 plus the physical parameters of Eq. 4-6. All host. */
typedef struct dgfs_params {
  int ns;                  /* number of species n (Eq. 1)                                        */
  const double *mass;      /* [ns]     non-dimensional masses m_p > 0                             */
  const double *omega;     /* [ns*ns]  viscosity index omega_pq (Eq. 4); gamma_pq = 2(1-omega_pq) */
  const double *alpha;     /* [ns*ns]  VSS scattering parameter alpha_pq > 0; 1.0 = VHS           */
  const double *kn;        /* [ns*ns]  Knudsen numbers Kn_pq (Eq. 5), or NULL => 1.0              */
  const double *prefactor; /* [ns*ns]  beta_pq override (Eq. 6), or NULL => Eq. 6 from kn         */
  int N;                   /* velocity points per dimension; supported: 8, 16, 24, 32, 48         */
  int N_rho;               /* Gauss-Legendre radial nodes on [0, R]                       */
  int M;                   /* points on the full sphere (reading S-1)                      */
  double L;                /* velocity box [-L, L]^3                                              */
  double R;                /* relative-velocity truncation radius; <= 0 => Eq. 9 with
                              (max mass, min mass) (reading RAD-1)                                */
  const double *sigma;     /* [M*3] unit vectors, or NULL => built-in rule for M in {6, 12, 32}   */
  const double *w_sigma;   /* [M] weights summing to 4 pi; must be NULL iff sigma is NULL         */
  int table_mode;          /* 0 = angular integrals of Eq. 16/17 evaluated exactly (default)
                              1 = Algo 1's pre-computation sphere quadrature (needs *_pre)        */
  int M_pre;               /* table_mode 1: number of pre-computation sphere points               */
  const double *sigma_pre; /* [M_pre*3]                                                           */
  const double *w_pre;     /* [M_pre]                                                             */
  int device;              /* CUDA device ordinal                                                 */
  int nyquist_filter;      /* 0 (default): Algorithm 2 as printed.  1: the operator is applied to the
                              inputs with their three Nyquist planes (l_d = -N/2) removed,
                              Q(P f_p, P f_q) with P = prod_d (1 - E_d), (E_d f)(c) = (-1)^{c_d} mean over
                              c_d' of (-1)^{c_d'} f.  A different discrete operator:
                              every shifted field is then exactly real, so the Nyquist-field kernels of
                              the N <= 32 pipeline are not run.                                    */
  int precision;           /* 0 (default): every step in fp64 (tolerance 1e-10 of max|Q| against the oracle).
                              1: the shifted fields, their transforms in x and y, the product and the sum over
                              sphere points (steps 4-6 of Algorithm 2: 3/4 of the work) run in fp32 on
                              single-precision copies of the z-shifted spectra and phase factors; step 1, the z
                              shifts, the forward z pass, steps 7-10 and the Nyquist-plane terms stay fp64.  Errors of
                              ~1e-6 of the GAIN term: within 1e-4 of max|Q| away from equilibrium, not near it
                              (DESIGN.md section 8e).  VHS pairs, table_mode 0, N <= 32 only: DGFS_ENOSUP otherwise. */
} dgfs_params;

/* Algorithm 1: quadratures, truncation radius (Eq. 9), prefactors (Eq. 6) and the
 * kernel-mode tables for every (radial node r, sphere point s, pair p,q), built on the device
 * and kept there. Synchronous. On success *out owns the tables until dgfs_destroy. */
int dgfs_create(const dgfs_params *p, dgfs_ctx **out);

/* Frees tables and workspace. NULL is allowed. */
void dgfs_destroy(dgfs_ctx *c);

/* Message of the last failed call on this context (or of the last failed dgfs_create when
 * c == NULL). The string is owned by the library and valid until the next call. */
const char *dgfs_last_error(const dgfs_ctx *c);

/* Right-hand side of Eq. 1 at nx spatial points, Algorithm 2 for all pairs:
 *   Q[x][p][:] = sum_q beta_pq * Q^(pq)(f[x][p], f[x][q]).
 * f: device, [nx][ns][N^3], read only.  Q: device, [nx][ns][N^3], overwritten; must not
 * alias f.  nx >= 0 (0 is a no-op).  Workspace is grown on demand (see dgfs_reserve). */
int dgfs_collide(dgfs_ctx *c, const double *f, double *Q, int nx, void *stream);

/* Same, every pair separately: Qpq[x][p][q][:] = beta_pq * Q^(pq)(f[x][p], f[x][q]).
 * Qpq: device, [nx][ns][ns][N^3]. */
int dgfs_collide_pairs(dgfs_ctx *c, const double *f, double *Qpq, int nx, void *stream);

/* End-to-end form of dgfs_collide with HOST buffers (pageable or pinned): f_host [nx][ns][N^3] is
 * copied to the device in slabs, collided (same kernels as dgfs_collide) and Q_host [nx][ns][N^3]
 * is copied back; uploads, kernels and downloads of consecutive slabs overlap on the library's own
 * streams.  Synchronous: on return Q_host is complete.  This is the call bench.py's "e2e" line
 * times.  The device staging buffers are owned by the context and grown on demand. */
int dgfs_collide_host(dgfs_ctx *c, const double *f_host, double *Q_host, int nx);

/* dgfs_collide for callers that must not allocate device memory (their own CUDA graph capture, a serving loop, a
 * harness that forbids cudaMalloc): same kernels, same launch order and same result as dgfs_collide, bit for bit, but
 * the workspace is a static device array of DGFS_NOALLOC_SCRATCH_BYTES inside the library instead of the context's
 * allocation; the call makes no cudaMalloc / cudaFree / cudaMallocAsync and no call that allocates on its behalf
 * (no CUDA graph is built, the context's workspace is not grown).  Every GPU that loads the library holds the array
 * until the process exits.  f, Q, nx, stream: as dgfs_collide.  The batch runs in launch groups small enough for
 * the array; the call fails with DGFS_EINVAL, before any launch, when one spatial point alone needs more (compare
 * dgfs_workspace_bytes(c, 1): about 13 MB at N = 32, 2 species; N = 48 does not fit), with DGFS_ENOSUP for a context
 * on the v0 pipeline (N = 48 with VSS pairs, DGFS_PIPELINE=v0) or with per-launch profiling switched on.
 * The array is shared by every context and every call of the process on that GPU and keeps what the last call left;
 * no kernel reads it before writing it, so nothing has to be cleared.  Calls that overlap on the GPU (two streams,
 * two contexts, two host threads) race on it: the caller orders them.  Calls of ONE context are ordered by the
 * library as for dgfs_collide.  The first call of a context sets kernel attributes (not an allocation). */
#define DGFS_NOALLOC_SCRATCH_BYTES (64u << 20)
int dgfs_collide_noalloc(dgfs_ctx *c, const double *f, double *Q, int nx, void *stream);

/* Bytes of device workspace dgfs_collide* needs for a batch of nx points (tables excluded).  A batch runs in launch
 * groups of a fixed number of points; the group is halved until its workspace fits a byte budget fixed at
 * dgfs_create: 70 % of the device memory free at that moment, or the environment variable DGFS_V1_WS_GB (in GB).
 * Results do not depend on the group size. */
size_t dgfs_workspace_bytes(const dgfs_ctx *c, int nx);

/* Allocate the workspace for batches of up to nx points now, so that later dgfs_collide* calls
 * with <= nx points never allocate (required before capturing them into a CUDA graph). */
int dgfs_reserve(dgfs_ctx *c, int nx);

/* Read back what dgfs_create derived (host outputs; any pointer may be NULL):
 * R (scalar), rho[N_rho], w_rho[N_rho], sigma[M*3], w_sigma[M], beta[ns*ns]. */
int dgfs_get_quadrature(const dgfs_ctx *c, double *R, double *rho, double *w_rho,
                        double *sigma, double *w_sigma, double *beta);

/* Copy the kernel-mode tables of pair (p,q) to HOST buffers, in Algorithm 1's layout and meaning
 * (for verification): a[N_rho][M][N^3] real, b[N_rho][M][N^3] complex interleaved
 * (re,im) (Eq. 16), c[N^3] complex interleaved (Eq. 17). Any pointer may be
 * NULL. The internal device tables are factored/compressed; this call expands them with the
 * library's own kernels. */
int dgfs_get_tables(dgfs_ctx *c, int p, int q, double *a, double *b, double *cc);

/* Device bytes held by the full kernel-mode tables b^(pq)_rs(k) of the pairs that need one (VSS, table_mode 1).  With
 * table_mode 0 these are stored once per orbit of the sphere rule under sign flips and the x <-> z swap, on the extended grid
 * [-N/2, N/2]^3 (b_rs(k) depends on k through |k| and k . sigma_s only, Eq. 16): [N_rho][orbits][(N+1)^3] complex
 * instead of the paper's [N_rho][M][N^3].  Environment DGFS_BTABLE=full keeps the paper's layout. */
size_t dgfs_table_bytes(const dgfs_ctx *c);

/* FLOP count of one pair evaluation as executed (SURVEY 8(d) / DESIGN.md "Roofline"), for the
 * benchmark's roofline line. */
double dgfs_flops_per_pair_eval(const dgfs_ctx *c, int p, int q);

/* Instrumentation for the benchmark.  dgfs_launch_count: number of
 * kernels this context has enqueued since dgfs_create.  dgfs_profile_enable(on != 0): from now on
 * every kernel launch is bracketed by a pair of CUDA events recorded on the caller's stream, and
 * launches, elapsed time and algorithmic FLOPs are accumulated per kernel class (a few
 * microseconds of overhead per launch; off by default).  dgfs_profile_get: entry i of
 * dgfs_profile_count; synchronises with the recorded events; *name is owned by the library.
 * dgfs_profile_reset: zero the accumulators. */
long long dgfs_launch_count(const dgfs_ctx *c);
int dgfs_profile_enable(dgfs_ctx *c, int on);
int dgfs_profile_count(const dgfs_ctx *c);
int dgfs_profile_get(dgfs_ctx *c, int i, const char **name, long long *launches, double *ms, double *flops);
int dgfs_profile_reset(dgfs_ctx *c);

/* Roofline denominator: throughput of the plain FP64 pipe of `device`
 * measured with dependency-free DFMA chains for about `seconds` (0 < seconds <= 30): best single
 * launch (*tflops_burst) and the average over the whole interval (*tflops_sustained). Host outputs,
 * either may be NULL.  Synchronous; needs no context. */
int dgfs_measure_fp64_peak(int device, double seconds, double *tflops_burst, double *tflops_sustained);

/* Do the plain FP64 pipe (DFMA) and the FP64 tensor path (mma.sync.m8n8k4.f64) of `device` run side by side?  A kernel
 * in which every thread carries n_dfma independent DFMA chains and every warp n_dmma independent MMA chains, no memory
 * traffic, timed for about `seconds` (0 < seconds <= 30); (n_dfma, n_dmma) one of (8,0), (0,8), (8,8), (8,2), (4,4),
 * else DGFS_EINVAL.  Host outputs (either may be NULL): the TFLOP/s each kind of instruction reached in the best launch
 * (m8n8k4 = 512 flop).  Separate pipes would give a mixed run both pure rates at once; B200 gives their times added
 * (profiles/r02_dft_probe.md).  Synchronous; needs no context. */
int dgfs_measure_fp64_mix(int device, int n_dfma, int n_dmma, double seconds, double *tflops_dfma, double *tflops_dmma);

/* Evidence for the transform kernels' design (BASELINE.json north_star: "shared-memory radix stages ... or per-axis DFT as
 * a dense contraction on FP64 tensor cores where N makes that the faster choice"): complex 1-D DFTs of length N
 * (8, 16, 24, 32 or 48) per second on `device`, on chip (registers / shared memory only inside the timed loop), by
 * method 0 = the register FFT every pass of the pipeline uses, method 1 = the same DFT as a real (2N x 2N) matrix
 * product on the FP64 tensor path (mma.sync.m8n8k4.f64).  *rel_err: one transform of each method against the direct
 * sum evaluated on the host, relative to the largest output.  Host outputs; synchronous; needs no context. */
int dgfs_measure_dft(int device, int N, int method, double seconds, double *dfts_per_second, double *rel_err);

/* 1-D mesh for dgfs_step: ne uniform elements on [x0, x1], nodal DG of polynomial degree
 * `order` on K = order+1 Gauss-Lobatto-Legendre nodes, purely diffuse walls at both ends
 * (Table 2; readings DG-1, DG-2). */
typedef struct dgfs_mesh1d {
  int ne;
  int order;
  double x0, x1;
  double wall_T[2];        /* wall temperatures at x0 and x1                                  */
  double wall_u[2][3];     /* wall velocities at x0 and x1                                    */
} dgfs_mesh1d;

/* nsteps explicit SSP-RK3 steps (reading DG-3) of Eq. 1 in one space dimension:
 *   d/dt f = -c_x d/dx f + sum_q beta_pq Q^(pq),  upwind interface flux, diffuse walls.
 * f: device, [ne][K][ns][N^3], updated in place. */
int dgfs_step(dgfs_ctx *c, const dgfs_mesh1d *mesh, double *f, double dt, int nsteps, void *stream);

/* nsteps forward-Euler steps f <- f + dt L(f) of the same equation (the time stepping of the paper's
 * Couette case, Table 2).  Same arguments, layout and error behaviour as dgfs_step. */
int dgfs_step_euler(dgfs_ctx *c, const dgfs_mesh1d *mesh, double *f, double dt, int nsteps, void *stream);

/* The spatial right-hand side alone (verification of D1-D3): rhs = -c_x d/dx f with upwind
 * fluxes and diffuse walls, no collisions.  f, rhs: device, [ne][K][ns][N^3]. */
int dgfs_advect_rhs(dgfs_ctx *c, const dgfs_mesh1d *mesh, const double *f, double *rhs, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* DGFS_H */
