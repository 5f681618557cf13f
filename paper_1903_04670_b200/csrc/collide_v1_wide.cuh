// collide_v1_wide.cuh -- the plane job of collide_v1.cu for 32 < N <= 64 (N = 48: config c4 of BASELINE.json).
//
// Same arithmetic as k_xy / k_nyq2 (file header of collide_v1.cu): lane = pencil, 1-D transforms in registers, one
// transposition through a shared-memory tile.  What changes with N = 48:
//   * a job needs N = 48 lanes: it runs on a block of 64 threads (two warps, 16 lanes idle), barriers are block barriers;
//   * 48 complex values plus 48 accumulators do not fit a thread's registers, so every length-N transform is split by
//     one radix-2 decimation-in-frequency step,  u_j = x_j + x_{j+N/2},  v_j = (x_j - x_{j+N/2}) w^j :  u (N/2 values)
//     stays in registers, v is parked in the lane's own column (pass 1) or row (pass 2) of the tile, where the inputs
//     it replaces have just been consumed; FFT_{N/2}(u) gives the even outputs, FFT_{N/2}(v) the odd ones;
//   * pass 1 therefore leaves its outputs in the tile in the order row p <-> cx = perm(p) = 2p (p < N/2), 2(p-N/2)+1
//     (p >= N/2): the lane that runs pass 2 on row p owns the column cx = perm(p) of the plane for the whole job list.
// Included by collide_v1.cu (needs JobSmem, NyqLayout, GzView, cp_async16, ...).
#pragma once

namespace dgfs {

template <int N>
__device__ __forceinline__ int wide_perm(int p) { return p < N / 2 ? 2 * p : 2 * (p - N / 2) + 1; }
template <int N>
__host__ __device__ constexpr int wide_invperm(int cx) { return (cx & 1) ? N / 2 + cx / 2 : cx / 2; }

// Pass 1 (lane g = (side, m), column m of the Hermitian half of that side): factor along the pass-1 index, inverse
// transform, factor of the lane's own column, back into the tile (rows in perm order).
template <int N, bool CORR>
__device__ __forceinline__ void wide_pass1(cplx* buf, int g, int side, int m, double szs, double scale, cplx c1,
                                           bool unit_i, bool real_m) {
  typedef JobSmem<N> JS;
  constexpr int H = N / 2, P = JS::P;
  const cplx hy0 = buf[JS::HM + side * JS::TS + m];
  const double hyH = buf[JS::HM + side * JS::TS + H].x;
  const double ya = scale * hy0.x, yb = (m == 0) ? 0.0 : -scale * hy0.y, yc = (m == 0) ? 0.0 : scale * hy0.y,
               yd = (m == 0) ? scale * hyH : scale * hy0.x;
  cplx u[H];
#pragma unroll
  for (int j = 0; j < H; ++j) {
    cplx x0 = buf[j * P + g], x1 = buf[(j + H) * P + g];
    if (!unit_i) {
      x0 = cmul(x0, buf[JS::HI + side * JS::TS + j]);
      x1 = cmul(x1, buf[JS::HI + side * JS::TS + j + H]);
    }
    if (CORR && j == 0) {                       // element H: the x-Nyquist row correction (NyqLayout::VYH)
      x1.x = fma(-szs, c1.x, x1.x);
      x1.y = fma(-szs, c1.y, x1.y);
    }
    u[j] = cadd(x0, x1);
    buf[(j + H) * P + g] = twiddle_mul<N, +1>(csub(x0, x1), j);
  }
  fft_reg<H, +1>(u);
#pragma unroll
  for (int k = 0; k < H; ++k) {                 // even outputs 2k -> row k
    const cplx v = u[k];
    buf[k * P + g] = real_m ? make_double2(v.x * ya, v.y * yd) : make_double2(fma(v.x, ya, v.y * yb), fma(v.x, yc, v.y * yd));
  }
#pragma unroll
  for (int j = 0; j < H; ++j) u[j] = buf[(j + H) * P + g];
  fft_reg<H, +1>(u);
#pragma unroll
  for (int k = 0; k < H; ++k) {                 // odd outputs 2k + 1 -> row H + k
    const cplx v = u[k];
    buf[(k + H) * P + g] = real_m ? make_double2(v.x * ya, v.y * yd) : make_double2(fma(v.x, ya, v.y * yb), fma(v.x, yc, v.y * yd));
  }
}

// Pass 2 (lane g runs row g of the tile): the N packed columns X = Y_A + i Y_B with the mirror half by conjugation,
// inverse transform.  Two halves, so that the caller can put a block barrier and the next job's prefetch between them:
// wide_pass2_even delivers the even outputs through out(index, value) (index known at compile time) and returns with
// v (the input of the odd half) in registers, after which the lane does not touch the tile again.
template <int N, bool CORR, class Out>
__device__ __forceinline__ void wide_pass2_even(cplx* buf, int g, double szs, double sxb, cplx vx, cplx vz, cplx (&u)[N / 2], Out out) {
  typedef JobSmem<N> JS;
  constexpr int H = N / 2, Q = H / 2, P = JS::P;
  static_assert(H % 2 == 0, "N must be a multiple of 4");
  cplx* row = buf + g * P;
  {
    const cplx a0 = row[0], b0 = row[H];
    cplx X0 = make_double2(a0.x, b0.x), XH = make_double2(a0.y, b0.y);
    if (CORR) {
      XH.x -= szs * vx.x + sxb * vz.x;
      XH.y -= szs * vx.y + sxb * vz.y;
    }
    u[0] = cadd(X0, XH);
    row[0] = csub(X0, XH);
  }
#pragma unroll
  for (int jj = 1; jj < Q; ++jj) {              // column pairs jj and H - jj give X[jj], X[N-jj], X[H-jj], X[H+jj]
    const cplx ya = row[jj], yb = row[H + jj], yc = row[H - jj], yd = row[N - jj];
    const cplx Xa = make_double2(ya.x - yb.y, ya.y + yb.x), Xb = make_double2(ya.x + yb.y, yb.x - ya.y);
    const cplx Xc = make_double2(yc.x - yd.y, yc.y + yd.x), Xd = make_double2(yc.x + yd.y, yd.x - yc.y);
    u[jj] = cadd(Xa, Xd);
    row[jj] = twiddle_mul<N, +1>(csub(Xa, Xd), jj);
    u[H - jj] = cadd(Xc, Xb);
    row[H - jj] = twiddle_mul<N, +1>(csub(Xc, Xb), H - jj);
  }
  {
    const cplx ya = row[Q], yb = row[H + Q];
    const cplx Xa = make_double2(ya.x - yb.y, ya.y + yb.x), Xb = make_double2(ya.x + yb.y, yb.x - ya.y);
    u[Q] = cadd(Xa, Xb);
    row[Q] = twiddle_mul<N, +1>(csub(Xa, Xb), Q);
  }
  fft_reg<H, +1>(u);
#pragma unroll
  for (int k = 0; k < H; ++k) out(2 * k, u[k]);
#pragma unroll
  for (int j = 0; j < H; ++j) u[j] = row[j];
}
template <int N, class Out>
__device__ __forceinline__ void wide_pass2_odd(cplx (&u)[N / 2], Out out) {
  constexpr int H = N / 2;
  fft_reg<H, +1>(u);
#pragma unroll
  for (int k = 0; k < H; ++k) out(2 * k + 1, u[k]);
}

// The r-loop's main kernel for 32 < N <= 64: a block of 2 N threads (N = 48: three full warps) runs the planes
// cz = 2 blockIdx.x and 2 blockIdx.x + 1 of one item side by side, thread t = (plane t / N, lane t % N); both walk the
// pair's job list in step (block barriers), each with its own tile and the sum over s in its lanes' registers (48
// accumulators per lane), then the forward x,y passes of the real plane.  Same inputs and outputs as k_xy<N, W, double2>.
template <int N>
__global__ void __launch_bounds__(2 * N) k_xy_wide(V1Tables t, DevTables tab, GzView Gz, const cplx* __restrict__ hxy,
                                                const cplx* __restrict__ nyq, const double* __restrict__ S,
                                                cplx* __restrict__ T, int r) {
  constexpr int H = N / 2, NH = N * H, N2 = N * N;
  typedef NyqLayout<N> NL;
  typedef JobSmem<N> JS;
  constexpr int P = JS::P;
  static_assert(N > 32 && N <= 64 && N % 2 == 0, "two jobs of N lanes per block");
  extern __shared__ cplx sm[];
  const int jp = threadIdx.x / N, g = threadIdx.x % N;      // plane of the block, lane of the job
  cplx* buf = sm + (size_t)jp * JS::WORDS;
  const int cz = blockIdx.x * 2 + jp, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  if (tab.full[pair] || t.tsrc[pair] != pair) return;      // R-11: (q,p) uses the buffer of (p,q)
  constexpr bool act = true;
  const int side = g / H, m = g % H;
  const int cx = wide_perm<N>(g);                           // column of the plane this lane owns in pass 2
  const double szs = (cz & 1) ? -1.0 : 1.0;
  const double sxb = (cx & 1) ? -1.0 : 1.0;
  const size_t goff = (size_t)cz * NH + m;
  const cplx* hbase = hxy + (((size_t)pair * tab.N_rho + r) * tab.M) * 4 * N;
  const cplx* nbase = nyq + (size_t)item * tab.M * NL::STRIDE;
  const int4* jl = t.jobs + (size_t)pair * tab.M;
  const int nj = t.njobs[pair];
  auto issue = [&](int4 jb) {
    if (act) {
      const cplx* gsrc = Gz.job(xl, side ? jb.z : jb.y, (size_t)(N * NH)) + goff;
#pragma unroll
      for (int i = 0; i < N; ++i) cp_async16(&buf[i * P + g], gsrc + i * H);
      const cplx* hx = hbase + (size_t)jb.x * 4 * N;          // [side][x|y][N]
      cp_async16(&buf[JS::HI + g], hx + g);
      cp_async16(&buf[JS::HI + JS::TS + g], hx + 2 * N + g);
      cp_async16(&buf[JS::HM + g], hx + N + g);
      cp_async16(&buf[JS::HM + JS::TS + g], hx + 3 * N + g);
      const cplx* nq = nbase + (size_t)jb.x * NL::STRIDE;
      cp_async16(&buf[JS::VYH + g], nq + NL::VYH + g);         // lane format (side, m)
      cp_async16(&buf[JS::VXP + g], nq + NL::VXP + cx);        // the lane's own cx
      if (g == 0) cp_async16(&buf[JS::VZP], nq + NL::VZP + cz);
    }
    cp_async_commit();
  };
  int mask = 0;
  if (nj > 0) { const int4 j0 = __ldg(&jl[0]); issue(j0); mask = j0.w; }
  double acc[N];
  {
    const double* w0 = S + ((size_t)item * N + cz) * N2 + cx;
#pragma unroll
    for (int j = 0; j < N; ++j) acc[j] = w0[j * N];
  }
  auto accumulate = [&](int idx, cplx v) { acc[idx] = fma(v.x, v.y, acc[idx]); };
  for (int j = 0; j < nj; ++j) {
    const int4 jn = __ldg(&jl[j + 1 < nj ? j + 1 : j]);
    cp_async_wait_all();
    __syncthreads();
    if (act) {
      const bool ux_ = (mask & 1) != 0, ry_ = (mask & 2) != 0;
      wide_pass1<N, true>(buf, g, side, m, szs, ux_ ? buf[JS::HI + side * JS::TS].x : 1.0, buf[JS::VYH + g], ux_, ry_);
    }
    __syncthreads();
    cplx u[H];
    if (act) wide_pass2_even<N, true>(buf, g, szs, sxb, buf[JS::VXP + g], buf[JS::VZP], u, accumulate);
    __syncthreads();                         // every lane has read its row for the last time: the tile is free
    if (j + 1 < nj) issue(jn);
    if (act) wide_pass2_odd<N>(u, accumulate);
    mask = jn.w;
  }
  // forward y and x passes of the real plane S_r(., ., cz)
  __syncthreads();
  if (act) {
    cplx v[N];
#pragma unroll
    for (int j = 0; j < N; ++j) v[j] = make_double2(acc[j], 0.0);
    fft_reg<N, -1>(v);
#pragma unroll
    for (int j = 0; j < N; ++j) buf[j * P + g] = v[j];          // [ky][lane of cx = perm(g)]
  }
  __syncthreads();
  if (act && g <= H) {                                          // lane = ky; S_r is real: ky = 0 .. H suffice
    cplx v[N];
#pragma unroll
    for (int i = 0; i < N; ++i) v[i] = buf[g * P + wide_invperm<N>(i)];
    fft_reg<N, -1>(v);
    cplx* o = T + ((size_t)item * N + cz) * (size_t)(N * (H + 1)) + g;
#pragma unroll
    for (int k = 0; k < N; ++k) o[k * (H + 1)] = v[k];           // [cz][kx][ky <= H]
  }
}

// The three Nyquist-plane fields of every (item, s) for 32 < N <= 64: block of 64 threads = (which, item), all sphere
// points in turn.  Same inputs, outputs and layouts as k_nyq2.
template <int N>
__global__ void __launch_bounds__(64) k_nyq2_wide(V1Tables t, DevTables tab, const cplx* __restrict__ fhh,
                                                  const cplx* __restrict__ nyqy, cplx* __restrict__ nyq, int r) {
  constexpr int H = N / 2, NH = N * H;
  typedef NyqLayout<N> NL;
  typedef JobSmem<N> JS;
  constexpr int P = JS::P;
  extern __shared__ cplx sm[];
  cplx* buf = sm;
  const int which = blockIdx.x, item = blockIdx.y;
  const int pair = item % tab.npairs, xl = item / tab.npairs;
  const int sp[2] = {pair / tab.ns, pair % tab.ns};
  const bool act = threadIdx.x < N;
  const int g = act ? threadIdx.x : 0;
  const int side = g / H, m = g % H;
  const int co = wide_perm<N>(g);                  // pass-1 output index this lane owns in pass 2
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
      for (int i = 0; i < N; ++i) cp_async16(&buf[i * P + g], src + (size_t)i * istride);
      const cplx* hx = hbase + (size_t)s * 4 * N;            // [side][x|y][N]
      const cplx* hzA = t.hz + ((size_t)r * t.nz + zm[2 * s]) * N;
      const cplx* hzB = t.hz + ((size_t)r * t.nz + zm[2 * s + 1]) * N;
      const cplx *hiA, *hiB, *hmA, *hmB;
      if (which == 0) { hiA = hx; hiB = hx + 2 * N; hmA = hx + N; hmB = hx + 3 * N; }
      else if (which == 1) { hiA = hzA; hiB = hzB; hmA = hx + N; hmB = hx + 3 * N; }
      else { hiA = hzA; hiB = hzB; hmA = hx; hmB = hx + 2 * N; }
      cp_async16(&buf[JS::HI + g], hiA + g);
      cp_async16(&buf[JS::HI + JS::TS + g], hiB + g);
      cp_async16(&buf[JS::HM + g], hmA + g);
      cp_async16(&buf[JS::HM + JS::TS + g], hmB + g);
      if (g == 0) cp_async16(&buf[JS::VZP], nyq + ((size_t)item * tab.M + s) * NL::STRIDE + NL::VT);
    }
    cp_async_commit();
  };
  auto scale_of = [&](int s) {
    if (which == 0) return t.szv[(size_t)r * t.nz + zm[2 * s + side]];
    return sbase[s * 4 + side * 2 + (which == 1 ? 0 : 1)];
  };
  const bool store_zeros = tab.full[pair] != 0;
  const int zbit = (which == 0) ? 4 : (which == 1 ? 1 : 2);
  const int ooff = (which == 0) ? NL::UZ : (which == 1 ? NL::UXP : NL::UY);
  const unsigned char* skip = t.sskip + (size_t)pair * tab.M;
  auto next_job = [&](int s) {                   // first s' >= s with a job to run
    while (s < tab.M && ((t.smask[s] & zbit) || skip[s])) {
      if (act && !skip[s] && store_zeros) {
        cplx* out = nyq + ((size_t)item * tab.M + s) * NL::STRIDE + ooff;
#pragma unroll
        for (int j = 0; j < N; ++j) out[j * N + g] = make_double2(0.0, 0.0);
      }
      ++s;
    }
    return s;
  };
  int s = next_job(0);
  if (s >= tab.M) return;
  issue(s);
  double scale = scale_of(s);
  while (s < tab.M) {
    const int sn = next_job(s + 1);
    cp_async_wait_all();
    __syncthreads();
    if (act) wide_pass1<N, false>(buf, g, side, m, 0.0, scale, make_double2(0.0, 0.0), false, false);
    __syncthreads();
    cplx* out = nyq + ((size_t)item * tab.M + s) * NL::STRIDE;
    const cplx vt = buf[JS::VZP];
    const double sb = (co & 1) ? -1.0 : 1.0;
    auto store = [&](int j, cplx v) {            // j: pass-2 output index (compile time), co: this lane's pass-1 output index
      if (which == 0) out[NL::UZ + (j * 2 + (co & 1)) * H + (co >> 1)] = v;
      else if (which == 1) {
        const double sg = (j & 1) ? -sb : sb;
        out[NL::UXP + j * N + co] = make_double2(v.x - sg * vt.x, v.y - sg * vt.y);
      } else out[NL::UY + j * N + (co ^ uy_swz(j))] = v;
    };
    cplx u[H];
    if (act) wide_pass2_even<N, false>(buf, g, 0.0, 0.0, make_double2(0.0, 0.0), make_double2(0.0, 0.0), u, store);
    __syncthreads();
    const double scale_next = (sn < tab.M) ? scale_of(sn) : 0.0;
    if (sn < tab.M) issue(sn);
    if (act) wide_pass2_odd<N>(u, store);
    s = sn; scale = scale_next;
  }
}

}  // namespace dgfs
