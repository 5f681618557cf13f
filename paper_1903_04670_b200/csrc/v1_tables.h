// v1_tables.h -- create-time tables of the v1 collision pipeline (internal, not part of the ABI).
//
// The shift e^{i theta.l} of Algorithm 2 steps 4-5 (a_rs of Algo 1 step 7,
// P:185, is linear in l) is a product of three 1-D factors.  Each factor is split into the part that
// keeps the spectrum of a real field Hermitian ("h": e^{i theta_d v} for |v| < N/2, cos(theta_d N/2)
// on the Nyquist index) and the part that does not ("s" = -sin(theta_d N/2), Nyquist index only);
// DESIGN.md section 5, R-6.  1/N per axis (unnormalised inverse transforms, reading C-3) and the
// sphere weight w_s (side A, x axis) are folded into both parts.
#pragma once
#include "fft_reg.cuh"

namespace dgfs {

struct V1Tables {
  int nz;                    // number of distinct z shifts ("z jobs") per radial node
  const int* zsp;            // [nz]                 species whose spectrum the job shifts
  const int* zmap;           // [pair][s][side]      -> z job
  const cplx* hz;            // [r][nz][N]           Hermitian-preserving z factor (1/N folded)
  const double* szv;         // [r][nz]              anti-Hermitian z scalar (1/N folded)
  const cplx* hxy;           // [pair][r][s][side][2][N]   x factors then y factors
  const cplxf* hxyf;         // the same in single precision (dgfs_params::precision = 1), else nullptr
  const double* sxy;         // [pair][r][s][side][2]      anti-Hermitian x, y scalars
  const int* tsrc;           // [pair]  pair whose S_r (buffer T) this pair uses: itself, or its transpose (q,p) -> (p,q) (R-11)
  const int* anti;           // [s]     antipode of sphere point s, or -1
  const int* tpartner;       // [pair]  full-table pair whose products this pair also serves (its transpose), or -1
  const int* fsrc_s;         // [pair][s]  full-table pairs: sphere point whose transformed product P_s (buffer Tf of pair
                             //            tsrc[pair]) equals this one's up to the factor fscale (R-10 / R-11)
  const double* fscale;      // [pair][s]
  const unsigned char* sskip; // [pair][s]  1: sphere point not run for this pair, its antipode carries both weights (R-10)
  const int4* jobs;          // [pair][M]  plane jobs the pair runs, in order: {s, z job of side A, z job of side B, smask[s]}
  const int* njobs;          // [pair]     how many (0 for a pair that reuses another pair's products)
  const unsigned char* smask; // [s]  bit d set: sigma_{s,d} = 0, so s_d = 0 for every pair and radial node and
                             //      the Nyquist field of that axis (ux', uy, uz for d = x, y, z) vanishes identically
};

// swizzle of the cz index of uy within its row (NyqLayout::UY)
__host__ __device__ __forceinline__ int uy_swz(int cx) { return (cx >> 1) & 7; }

// per (item, s) block of Nyquist-plane fields written by k_nyq.  UY and UZ as commented for the pairs whose fields go to
// k_wterm; for pairs with a full table (k_xy_full) they are plain [cx][cz] and [cy][cx], in units of cplx
template <int N>
struct NyqLayout {
  static constexpr int VYH = 0;            // [N]     lane format, x-Nyquist row correction (no y factor)
  static constexpr int VXP = N;            // [N]     packed (A + iB), y-Nyquist column correction
  static constexpr int VZP = 2 * N;        // [N]     packed, (H,H) element correction per cz
  static constexpr int VT = 3 * N;         // [1]     packed, s_x s_y s_z f^(H,H,H)
  static constexpr int UXP = 4 * N;        // [cy][cz]
  static constexpr int UY = 4 * N + N * N; // [cx][cz ^ ((cx / 2) mod 8)]: cz XOR-swizzled within its row (uy_swz), conflict-free plane reads in k_wterm
  static constexpr int UZ = 4 * N + 2 * N * N;   // [cy][cx & 1][cx / 2]: de-interleaved by the parity of cx, the shared-memory image k_wterm reads
  static constexpr int STRIDE = 4 * N + 3 * N * N;
};

}  // namespace dgfs
