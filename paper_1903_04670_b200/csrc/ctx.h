// ctx.h -- internal context of libdgfs (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <vector>
#include "../../include/dgfs.h"
#include "fft_reg.cuh"
#include "v1_tables.h"

namespace dgfs {

// Device-side view of the tables built by dgfs_create (Algorithm 1).
// "SPEC layout" = spectral index order [lz][lx][ly] (ly fastest): the order in which the
// warp-per-plane transforms produce and consume spectra.
struct DevTables {
  int ns, npairs, N, N3, N_rho, M, K2n;
  // separable phase factors  e^{ +i mu_q rho'_r sigma_s,d v } (side 0, acts on f^_p) and
  // e^{ -i mu_p rho'_r sigma_s,d v } (side 1, acts on f^_q)  == exp(+-i mu a_rs), Algo 2 steps 4-5
  // with a_rs of Algo 1 step 7 split per axis.  d = 0 carries the folded
  // normalisation: side 0: w_sigma_s / N^3, side 1: 1 / N^3.
  const cplx* phase;            // [pair][r][s][side][3][N]
  // b^(pq)_r(|k|^2) for pairs whose b does not depend on s (VHS, table_mode 0; Eq. 16)
  const double* bvhs;           // [pair][r][K2n]
  // full b^(pq)_rs(k) in SPEC layout for the other pairs (VSS or table_mode 1), else nullptr
  const cplx* const* bfull;     // [pair] -> [r][s][N3], or (bsym) [r][nref][(N+1)^3]: see bfull_at below
  int bsym, nref;               // symmetry-compressed full tables: reference sphere points only, extended grid
  const int4* bmap;             // [s] {offset, stride of kx, of ky, of kz} into the reference tables (signed frequencies)
  const cplx* closs;            // [pair][N3]  c^(pq)(k), SPEC layout (Eq. 17)
  const double* w_rho;          // [N_rho]
  const double* beta;           // [pair]      beta_pq (Eq. 6)
  const unsigned char* full;    // [pair]      1 = uses bfull and per-s forward transforms
  // v0 pipeline, VHS pairs (R-10, R-11): sphere points not run, pair whose summed products are used
  const unsigned char* sskip;   // [pair][s]
  const int* tsrc;              // [pair]
};

// b^(pq)_rs(k) of a pair with a full table, at SIGNED frequencies (kx, ky, kz) in [-N/2, N/2).
// bsym: b_rs(k) = F_r(|k|, k . sigma_s) (Eq. 16), so for sigma_s = G sigma_u with G a signed permutation of the
// axes, b_rs(k) = b_ru(G^T k): only the reference points u are stored, on the extended grid [-N/2, N/2]^3 (G^T may flip
// the sign of the Nyquist index), and the index of G^T k is linear in (kx, ky, kz): bmap[s].  G ranges over the sign
// flips and the x <-> z swap (ky stays the fastest index, loads stay coalesced): 3 tables for the 12 points of the
// icosahedron, 7 for the 32-point rule: 2.7 GB -> 0.63 GB per pair at (48, 48, 32).
// Written without branches (both index forms are a few integer operations; the load is unconditional).
__device__ __forceinline__ size_t bfull_index(const DevTables& tab, int r, int s, int kx, int ky, int kz) {
  const int N = tab.N;
  const int4 m = tab.bsym ? tab.bmap[s] : make_int4(0, 0, 0, 0);
  const size_t E = N + 1;
  const int ix = kx < 0 ? kx + N : kx, iy = ky < 0 ? ky + N : ky, iz = kz < 0 ? kz + N : kz;
  const size_t isym = (size_t)r * tab.nref * (E * E * E) + (size_t)(m.x + kx * m.y + ky * m.z + kz * m.w);
  const size_t ifull = ((size_t)r * tab.M + s) * tab.N3 + ((size_t)iz * N + ix) * N + iy;
  return tab.bsym ? isym : ifull;
}
__device__ __forceinline__ cplx bfull_at(const DevTables& tab, int pair, int r, int s, int kx, int ky, int kz) {
  return tab.bfull[pair][bfull_index(tab, r, s, kx, ky, kz)];
}
// The same for a sweep over kz at fixed (kx, ky): pointer to the element of kz = 0 and the stride (in elements) per
// unit of the index zi = kz (signed, bsym) or iz = kz mod N (full layout).
struct BSweep { const cplx* p; long sz; };
__device__ __forceinline__ BSweep bfull_sweep(const DevTables& tab, int pair, int r, int s, int kx, int ky) {
  const int4 m = tab.bsym ? tab.bmap[s] : make_int4(0, 0, 0, 0);
  BSweep b;
  b.p = tab.bfull[pair] + bfull_index(tab, r, s, kx, ky, 0);
  b.sz = tab.bsym ? (long)m.w : (long)tab.N * tab.N;
  return b;
}

}  // namespace dgfs

namespace dgfs {
// per-kernel-class accumulators behind dgfs_profile_* (include/dgfs.h)
struct ProfEntry {
  std::string name;
  long long launches = 0;
  double ms = 0.0, flops = 0.0;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> pending;
};
struct Profiler {
  bool on = false;
  long long total_launches = 0;
  std::vector<ProfEntry> entries;
  std::vector<cudaEvent_t> pool;
  int find(const char* name) {
    for (size_t i = 0; i < entries.size(); ++i) if (entries[i].name == name) return (int)i;
    entries.emplace_back(); entries.back().name = name; return (int)entries.size() - 1;
  }
  cudaEvent_t get_event() {
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e; cudaEventCreate(&e); return e;
  }
  void drain() {
    for (auto& en : entries) {
      for (auto& pr : en.pending) {
        cudaEventSynchronize(pr.second);
        float t = 0; cudaEventElapsedTime(&t, pr.first, pr.second);
        en.ms += t; pool.push_back(pr.first); pool.push_back(pr.second);
      }
      en.pending.clear();
    }
  }
};
// RAII bracket around one launch
struct ProfScope {
  Profiler& P; cudaStream_t st; int id = -1; cudaEvent_t e0{}, e1{};
  ProfScope(Profiler& p, cudaStream_t s, const char* name, double flops) : P(p), st(s) {
    ++P.total_launches;
    if (!P.on) return;
    id = P.find(name); P.entries[id].launches++; P.entries[id].flops += flops;
    e0 = P.get_event(); e1 = P.get_event(); cudaEventRecord(e0, st);
  }
  ~ProfScope() { if (id >= 0) { cudaEventRecord(e1, st); P.entries[id].pending.emplace_back(e0, e1); } }
};
}  // namespace dgfs

struct dgfs_ctx {
  int device = 0;
  dgfs::Profiler prof;
  int ns = 0, N = 0, N_rho = 0, M = 0, npairs = 0, N3 = 0, K2n = 0;
  double L = 0, R = 0;
  int table_mode = 0;
  bool nyq_filter = false;               // dgfs_params::nyquist_filter
  int precision = 0;                     // dgfs_params::precision
  bool any_full = false;
  std::vector<double> mass, omega, alpha, kn, beta, gam, eta, rho, w_rho, sigma, w_sigma;
  std::vector<double> sigma_pre, w_pre;
  int M_pre_count() const { return (int)w_pre.size(); }
  std::vector<unsigned char> full;
  // device tables
  dgfs::cplx* d_phase = nullptr;
  double* d_bvhs = nullptr;
  std::vector<dgfs::cplx*> h_bfull;      // device pointers, one per pair (or nullptr)
  int bsym = 0, nref = 0;                // symmetry-compressed full tables (DevTables::bsym)
  std::vector<int> bref;                 // [nref] sphere point each reference table belongs to
  std::vector<int4> bmap;                // [M]
  int* d_bref = nullptr;
  int4* d_bmap = nullptr;
  size_t table_bytes = 0;                // device bytes of the b tables (reported by dgfs_table_bytes)
  dgfs::cplx** d_bfull = nullptr;
  dgfs::cplx* d_closs = nullptr;
  double* d_w_rho = nullptr;
  double* d_beta = nullptr;
  double* d_rho = nullptr;
  double* d_sigma = nullptr;
  unsigned char* d_full = nullptr;
  std::vector<unsigned char> v0_sskip;      // antipodal symmetries of VHS pairs for the v0 pipeline
  std::vector<int> v0_tsrc;
  std::vector<double> v0_wfac;              // [pair][s] weight factor of the points that run
  unsigned char* d_v0_sskip = nullptr;
  int* d_v0_tsrc = nullptr;
  double* d_v0_wfac = nullptr;
  dgfs::DevTables tab{};
  // v1 pipeline (collide_v1.cu): tables built by build_tables_v1, used for N <= 32
  bool use_v1 = false;
  int v1_chunk = 512;                    // spatial points per launch group (large launches amortise the tails)
  size_t ws_budget = 0;                  // bytes the workspace of one launch group may take (0: no limit); plan_v1
  int v1_rgroup = 16;                    // radial nodes per forward-z / QG accumulation launch
  int v1_nz = 0, v1_nz0 = 0;             // z jobs; the last v1_nz0 of them have sigma_z = 0
  std::vector<int> v1_zsp, v1_zmap, v1_tsrc, v1_fsrc_s, v1_anti, v1_tpartner;
  std::vector<double> v1_fscale;
  std::vector<int4> v1_jobs;
  std::vector<int> v1_njobs;
  std::vector<double> v1_xyflops;        // [pair] executed flops of k_xy per item and radial node (x passes per group)
  int4* d_v1_jobs = nullptr;
  int* d_v1_njobs = nullptr;
  int *d_v1_zsp = nullptr, *d_v1_zmap = nullptr, *d_v1_tsrc = nullptr, *d_v1_fsrc_s = nullptr, *d_v1_anti = nullptr, *d_v1_tpartner = nullptr;
  double* d_v1_fscale = nullptr;
  dgfs::cplx *d_v1_hz = nullptr, *d_v1_hxy = nullptr;
  dgfs::cplxf* d_v1_hxyf = nullptr;      // precision 1: single-precision copy of the x, y factors
  double *d_v1_szv = nullptr, *d_v1_sxy = nullptr;
  std::vector<unsigned char> v1_smask, v1_sskip;
  unsigned char *d_v1_smask = nullptr, *d_v1_sskip = nullptr;
  dgfs::V1Tables v1{};
  // v1 pipeline, two-stream schedule (collide_v1.cu "host orchestration"): the kernels that prepare radial node
  // r + 1 (z shifts, Nyquist fields, their product term; bound by memory and latency) run on `aux`, a
  // high-priority stream of the library, while the plane jobs of radial node r (bound by the FP64 pipe) run on
  // the caller's stream; double-buffered intermediates, ordered by these events
  int v1_pack = 0;                       // DGFS_V1_PACK=1, N < 32: plane jobs dealt out N lanes each instead of one per warp
  int v1_xyw = 4;                        // warps per k_xy block (DGFS_V1_XYW)
  int v1_wterm_mc = 0;                   // DGFS_V1_WTERM_MC=1 (N = 32): k_wterm as clusters of 4 blocks, uy plane by TMA multicast
  int v1_overlap = 0;                    // DGFS_V1_OVERLAP=1: three streams (default: everything on the caller's stream)
  cudaStream_t aux = nullptr, aux2 = nullptr;
  bool v1_attr_done = false, v0_attr_done = false;   // dynamic shared-memory opt-in, once per context (= per device)
  cudaEvent_t ev_head = nullptr, ev_prep[2] = {nullptr, nullptr}, ev_xy[2] = {nullptr, nullptr};
  cudaEvent_t ev_grp[2] = {nullptr, nullptr}, ev_acc[2] = {nullptr, nullptr};
  // the workspace belongs to one call at a time: every call waits for the previous one's last launch
  cudaEvent_t ev_last = nullptr;
  bool ev_last_set = false;
  bool pool_set = false;                 // release threshold of the stream-ordered allocator raised
  // small batches (collide_v1.cu, run_collide_v1): the whole call captured once into a CUDA graph and replayed
  struct SmallGraph { int nx; bool pairs; void* ws; cudaGraphExec_t exec; long long launches; };
  std::vector<SmallGraph> graphs;
  cudaStream_t cap_stream = nullptr;     // captures happen on a stream of the library (the legacy default stream cannot capture)
  int v1_graph_items = 64;               // largest nx * pairs served that way (DGFS_V1_GRAPH_ITEMS; 0 = never)
  // workspace (grown on demand)
  void* ws = nullptr;
  size_t ws_bytes = 0;
  size_t scratch_budget = 0;             // bytes allowed for the transposition scratch G
  // dgfs_collide_host: two device slabs each for f and Q, three streams, per-slab events
  double* hp_f[2] = {nullptr, nullptr};
  double* hp_q[2] = {nullptr, nullptr};
  int hp_pts = 0;
  cudaStream_t hp_stream[3] = {nullptr, nullptr, nullptr};
  cudaEvent_t hp_ev[3][2] = {};
  // DG operator storage (dgfs_step)
  void* dg_ws = nullptr;
  size_t dg_ws_bytes = 0;
  std::string err;
};

namespace dgfs {

int set_error(dgfs_ctx* c, int code, const std::string& msg);
int check_cuda(dgfs_ctx* c, cudaError_t e, const char* what);

// create.cu
int build_tables(dgfs_ctx* c);
// collide.cu
struct ChunkPlan {
  int nbx;                 // spatial points per chunk
  size_t off_fhat, off_qg, off_g, off_t, off_fp, total;
};
ChunkPlan plan_chunks(const dgfs_ctx* c, int nx);
int run_collide(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st);
int ensure_workspace(dgfs_ctx* c, size_t bytes, cudaStream_t st);
// P f = prod_d (1 - E_d) f on `narr` arrays of N^3 values (dgfs_params::nyquist_filter): src -> dst
int launch_nyquist_filter(dgfs_ctx* c, const double* src, double* dst, int narr, cudaStream_t st);
// collide_v1.cu
int build_tables_v1(dgfs_ctx* c);
void free_tables_v1(dgfs_ctx* c);
int init_streams_v1(dgfs_ctx* c);
void free_streams_v1(dgfs_ctx* c);
void drop_graphs_v1(dgfs_ctx* c);
void free_graph_stream_v1(dgfs_ctx* c);
size_t workspace_bytes_v1(const dgfs_ctx* c, int nx);
int run_collide_v1(dgfs_ctx* c, const double* f, double* out, int nx, bool pairs_out, cudaStream_t st);
double flops_per_pair_eval_v1(const dgfs_ctx* c, int pair);

}  // namespace dgfs
