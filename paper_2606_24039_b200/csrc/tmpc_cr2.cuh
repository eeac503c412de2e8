// tmpc_cr2.cuh — a11, chunked form of the fused ADMM loop on the cyclic-reduction factor of tmpc_cr.cuh (config 5).
//
// cr_admm_kernel runs every elimination level grid-wide: ~30 phases per iteration, each paying an L2 round trip
// (~1.5-2 us) whatever the barrier costs.  Here the stages are cut into chunks of CS = 64 = 2^6 consecutive stages with
// the multiples of 64 as SEPARATORS.  Levels 0..5 of the odd-even elimination only ever couple a stage with stages of
// its own closed chunk [64c, 64c+64], so each CTA runs them on shared-memory copies of its factor blocks with
// __syncthreads; the separators only ACCUMULATE during these levels (partial sums from their two chunks are added
// later).  One extra CTA owns the separator system (levels >= 6, the root and the way back up) in its shared memory.
// Per iteration: [eta, local down-sweep] -> barrier -> [separator solve, one CTA] -> barrier -> [local up-sweep,
// eq. 9-16 for the chunk] -> barrier (r of the last dynamics block crosses the chunk boundary): 3 grid barriers and no
// global-memory latency inside the levels.  All ADMM state of a chunk lives in its shared memory for the whole launch.
// Same recurrences as tmpc_cr.cuh (gather form, deterministic), same factor arrays (Th, Lo, U, FA, FB from cr_factor).
#pragma once
#include "tmpc_cr.cuh"

namespace tmpc {

constexpr int CR2_CS = 64, CR2_LV = 6;

// local levels on a chunk: arrays indexed by local stage 0..nl (0 = left separator, CS = right separator if it exists)
template <typename T, int NC>
__device__ __forceinline__ void cr2_down(const T* FA, const T* FB, T* eta, int nl, int h, int tid, int nt) {
  constexpr int n = NC, nn = NC * NC;
  for (int w = tid;; w += nt) {
    const int k = w / n, i = w - k * n, s = 2 * h * k;
    if (s > nl) break;
    T acc = T(0);
    if (s + h <= nl) { const T* F = FA + (s + h) * nn + i * n; const T* e = eta + (s + h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc += F[m] * e[m]; }
    if (s - h >= 0) { const T* F = FB + (s - h) * nn + i * n; const T* e = eta + (s - h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc += F[m] * e[m]; }
    eta[s * n + i] -= acc;
  }
}
template <typename T, int NC>
__device__ __forceinline__ void cr2_up(const T* FA, const T* FB, const T* U, const T* eta, T* xt, int nl, int h, int tid, int nt) {
  constexpr int n = NC, nn = NC * NC;
  for (int w = tid;; w += nt) {
    const int k = w / n, i = w - k * n, j = h * (2 * k + 1);
    if (j > nl) break;
    const T* Uj = U + j * nn + i * n; const T* e = eta + j * n;
    T acc = T(0);
#pragma unroll
    for (int m = 0; m < n; ++m) acc += Uj[m] * e[m];
    { const T* F = FA + j * nn + i; const T* xa = xt + (j - h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc -= F[m * n] * xa[m]; }
    if (j + h <= nl) { const T* F = FB + j * nn + i; const T* xb = xt + (j + h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc -= F[m * n] * xb[m]; }
    xt[j * n + i] = acc;
  }
}

template <typename T, int NC, int NX>
__host__ __device__ inline size_t cr2_smem_elems(int ng, int S) {
  const size_t chunk = (size_t)3 * (CR2_CS + 1) * NC * NC + 2 * CR2_CS * NX * NC + (size_t)CR2_CS * ng * NC + 4 * (CR2_CS + 1) * NC + 5 * CR2_CS * ng + 3 * (CR2_CS + 1) * NX + NX * NC + 64;
  const size_t top = (size_t)3 * S * NC * NC + 2 * (size_t)S * NC + 64;
  return chunk > top ? chunk : top;
}

template <typename T, int NC, int NX>
__global__ void __launch_bounds__(256) cr2_admm_kernel(CrAdmmArgs<T> a, int nchunks) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  const Dims& d = a.d;
  constexpr int n = NC, nn = NC * NC, nx = NX, CS = CR2_CS;
  const int ng = d.ng, N = d.N, T_ = d.T, nz = d.nz, mf = d.mf, mg = d.mg, p = blockIdx.y, tid = threadIdx.x, nt = blockDim.x;
  CrBuf<T> b = cr_carve<T>(d, a.ws, p);
  GridBar grid = cr_gridbar<T>(b);
  const int S = N / CS + 1;                             // separators 0, 64, .., 64 (S-1)
  T* gEta = b.part; T* gPart = gEta + S * n; T* gX = gPart + S * n; T* gR = gX + S * n;   // exchange through global memory
  const int L = cr_levels(T_);
  const int iters = a.kkt_only ? 1 : a.iters;

  // ================================================================ separator CTA
  if ((int)blockIdx.x == nchunks) {
    T* FA = sm; T* FB = FA + (size_t)S * nn; T* U = FB + (size_t)S * nn; T* eta = U + (size_t)S * nn; T* xt = eta + S * n;
    for (int e = tid; e < S * nn; e += nt) { const int k = e / nn, r = e - k * nn; const size_t g = (size_t)k * CS * nn + r; FA[e] = b.FA[g]; FB[e] = b.FB[g]; U[e] = b.U[g]; }
    __syncthreads();
    if (!a.kkt_only) grid.sync();                       // pairs with the chunks' set-up barrier
    for (int it = 0; it < iters; ++it) {
      grid.sync();
      for (int e = tid; e < S * n; e += nt) { const int k = e / n; eta[e] = __ldcg(gEta + e) + (k > 0 ? __ldcg(gPart + e - n) : T(0)); }
      __syncthreads();
      for (int l = CR2_LV; l < L; ++l) { cr2_down<T, NC>(FA, FB, eta, S - 1, 1 << (l - CR2_LV), tid, nt); __syncthreads(); }
      if (tid < n) { T acc = T(0);
#pragma unroll
        for (int m = 0; m < n; ++m) acc += U[tid * n + m] * eta[m];
        xt[tid] = acc; }
      __syncthreads();
      for (int l = L - 1; l >= CR2_LV; --l) { cr2_up<T, NC>(FA, FB, U, eta, xt, S - 1, 1 << (l - CR2_LV), tid, nt); __syncthreads(); }
      for (int e = tid; e < S * n; e += nt) gX[e] = xt[e];
      grid.sync();
      if (!a.kkt_only) grid.sync();
    }
    if (!a.kkt_only && tid == 0 && a.status && *b.flag) atomicOr(&a.status[p], TMPC_ST_PIVOT);
    return;
  }

  // ================================================================ chunk CTAs
  const int c = blockIdx.x, a0 = c * CS;
  const int nl = (N - a0) < CS ? (N - a0) : CS;         // last local stage index (CS = the right separator)
  const int nown = nl < CS ? nl + 1 : CS;               // stages owned: a0 .. a0+nown-1
  const int nblk = (N - a0) < CS ? (N - a0) : CS;       // dynamics blocks owned: t = a0 .. a0+nblk-1
  T* FA = sm; T* FB = FA + (size_t)(CS + 1) * nn; T* U = FB + (size_t)(CS + 1) * nn;
  T* sAm = U + (size_t)(CS + 1) * nn; T* sAp = sAm + (size_t)CS * nx * n; T* sG = sAp + (size_t)CS * nx * n;
  T* eta = sG + (size_t)CS * ng * n; T* xt = eta + (CS + 1) * n; T* xs = xt + (CS + 1) * n; T* qs = xs + (CS + 1) * n;
  T* zg = qs + (CS + 1) * n; T* yg = zg + CS * ng; T* lo = yg + CS * ng; T* hi = lo + CS * ng; T* sv = hi + CS * ng;
  T* yf = sv + CS * ng; T* cv = yf + (CS + 1) * nx; T* rv = cv + (CS + 1) * nx;     // slot 0 = the block before the chunk (or init rows)
  T* sApP = rv + (CS + 1) * nx;                         // A^+ of the block before the chunk
  // interior stages keep their factor blocks here for the whole launch (separators' blocks belong to the separator CTA)
  for (int e = tid; e < (nl + 1) * nn; e += nt) { const size_t g = (size_t)a0 * nn + e; const int ls = e / nn; const bool sep = ls == 0 || ls == CS; FA[e] = sep ? T(0) : b.FA[g]; FB[e] = sep ? T(0) : b.FB[g]; U[e] = sep ? T(0) : b.U[g]; }
  const T sigma = a.prm.sigma, rho_f = a.prm.rho_f, rho_g = a.prm.rho_g, alpha = a.prm.alpha;
  const T inv_rho_g = T(1) / rho_g, inv_rg = T(1) / (rho_g + a.prm.gamma), lam = a.prm.lam;
  const size_t gxo = (size_t)p * nz + (size_t)a0 * n, ggo = (size_t)p * mg + (size_t)a0 * ng;
  auto local_solve_down = [&]() { for (int l = 0; l < CR2_LV && l < L; ++l) { cr2_down<T, NC>(FA, FB, eta, nl, 1 << l, tid, nt); __syncthreads(); } };
  auto local_solve_up = [&]() { for (int l = (L < CR2_LV ? L : CR2_LV) - 1; l >= 0; --l) { cr2_up<T, NC>(FA, FB, U, eta, xt, nl, 1 << l, tid, nt); __syncthreads(); } };
  auto publish_down = [&]() {
    if (tid < n) { gEta[c * n + tid] = eta[tid]; if (nl == CS) gPart[c * n + tid] = eta[CS * n + tid]; }
  };
  auto fetch_x = [&]() {
    if (tid < n) { xt[tid] = __ldcg(gX + c * n + tid); if (nl == CS) xt[CS * n + tid] = __ldcg(gX + (c + 1) * n + tid); }
    __syncthreads();
  };

  if (a.kkt_only) {
    for (int e = tid; e < (nl + 1) * n; e += nt) eta[e] = (e < nown * n) ? a.eta_in[gxo + e] : T(0);
    __syncthreads();
    local_solve_down(); publish_down();
    grid.sync(); grid.sync();
    fetch_x(); local_solve_up();
    for (int e = tid; e < nown * n; e += nt) a.xt_out[gxo + e] = xt[e];
    return;
  }

  // ---- chunk data and state into shared memory
  {
    const T* Am = a.qp.Am + ((size_t)p * N + a0) * nx * n; const T* Ap = a.qp.Ap + ((size_t)p * N + a0) * nx * n;
    for (int e = tid; e < nblk * nx * n; e += nt) { sAm[e] = Am[e]; sAp[e] = Ap[e]; }
    if (c > 0) for (int e = tid; e < nx * n; e += nt) sApP[e] = a.qp.Ap[((size_t)p * N + a0 - 1) * nx * n + e];
    if (!d.g_sel && ng > 0) { const T* G = a.qp.G + a.qp.sG * p + (size_t)a0 * ng * n; for (int e = tid; e < nown * ng * n; e += nt) sG[e] = G[e]; }
    for (int e = tid; e < nown * n; e += nt) { xs[e] = a.x[gxo + e]; qs[e] = a.qp.q[gxo + e]; }
    for (int e = tid; e < nown * ng; e += nt) { lo[e] = a.qp.lo[ggo + e]; hi[e] = a.qp.hi[ggo + e]; yg[e] = a.yg[ggo + e]; zg[e] = a.zg_given ? a.zg[ggo + e] : T(0); }
    // equality rows: slot 0 = init rows (chunk 0 only), slot 1 + k = dynamics block a0 + k
    for (int e = tid; e < (nblk + 1) * nx; e += nt) {
      const int k = e / nx - 1, i = e - (k + 1) * nx;
      if (k < 0) { const bool has = c == 0; yf[e] = has ? a.yf[(size_t)p * mf + i] : T(0); cv[e] = has ? a.qp.x_init[(size_t)p * nx + i] : T(0); }
      else { yf[e] = a.yf[(size_t)p * mf + nx + (size_t)(a0 + k) * nx + i]; cv[e] = a.qp.b[((size_t)p * N + a0 + k) * nx + i]; }
    }
  }
  __syncthreads();
  auto g_dot = [&](int ls, int r, const T* vec) -> T {
    if (d.g_sel) return vec[ls * n + d.g_col[r]];
    const T* g = sG + (ls * ng + r) * n; T s = T(0);
#pragma unroll
    for (int j = 0; j < n; ++j) s += g[j] * vec[ls * n + j];
    return s;
  };
  for (int e = tid; e < nown * ng; e += nt) {
    const int ls = e / ng, r = e - ls * ng;
    if (!a.zg_given) { zg[e] = tmin(tmax(g_dot(ls, r, xs), lo[e]), hi[e]); if (a.iters == 0) a.xi[ggo + e] = T(0); }
    sv[e] = rho_g * zg[e] - yg[e];
  }
  for (int e = tid; e < (nblk + 1) * nx; e += nt) rv[e] = (e >= nx || c == 0) ? rho_f * cv[e] - yf[e] : T(0);
  __syncthreads();
  if (nblk == CS && tid < nx) gR[c * nx + tid] = rv[CS * nx + tid];      // r of my last block, for the next chunk's first stage
  grid.sync();

  for (int it = 0; it < a.iters; ++it) {
    // ---- a4 (eq. 51) for my stages; rows of the block before the chunk come through gR
    if (c > 0 && tid < nx) rv[tid] = __ldcg(gR + (c - 1) * nx + tid);
    __syncthreads();
    for (int e = tid; e < (nl + 1) * n; e += nt) {
      const int ls = e / n, i = e - ls * n;
      T s = T(0);
      if (ls < nown) {
        s = sigma * xs[e] - qs[e];
        if (c == 0 && ls == 0) { if (i < nx) s += rv[i]; }
        else if (ls == 0) { const T* A_ = sApP + i; for (int k = 0; k < nx; ++k) s += A_[k * n] * rv[k]; }
        if (ls < nblk) { const T* A_ = sAm + ls * nx * n + i; const T* r = rv + (ls + 1) * nx; for (int k = 0; k < nx; ++k) s += A_[k * n] * r[k]; }
        if (ls > 0) { const T* A_ = sAp + (ls - 1) * nx * n + i; const T* r = rv + ls * nx; for (int k = 0; k < nx; ++k) s += A_[k * n] * r[k]; }
        if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) s += sv[ls * ng + r]; }
        else { const T* g = sG + ls * ng * n + i; for (int r = 0; r < ng; ++r) s += g[r * n] * sv[ls * ng + r]; }
      }
      eta[e] = s;                                       // the right separator slot starts at zero: it only accumulates
    }
    __syncthreads();
    local_solve_down(); publish_down();
    grid.sync();                                        // separator CTA solves
    grid.sync();
    fetch_x(); local_solve_up();
    // ---- a7 + a8 for my blocks and stages (x~ of the right separator is in xt[CS])
    for (int e = tid; e < (nblk + 1) * nx; e += nt) {
      const int k = e / nx - 1, i = e - (k + 1) * nx;
      T ztf;
      if (k < 0) { if (c != 0) continue; ztf = xt[i]; }
      else {
        const T* am = sAm + (k * nx + i) * n; const T* ap = sAp + (k * nx + i) * n; T s = T(0);
#pragma unroll
        for (int j = 0; j < n; ++j) s += am[j] * xt[k * n + j] + ap[j] * xt[(k + 1) * n + j];
        ztf = s;
      }
      const T y = yf[e] + rho_f * alpha * (ztf - cv[e]);
      yf[e] = y; rv[e] = rho_f * cv[e] - y;
    }
    for (int e = tid; e < nown * ng; e += nt) {
      const int ls = e / ng, r = e - ls * ng;
      const T zh = alpha * g_dot(ls, r, xt) + (T(1) - alpha) * zg[e];
      const T v = zh + yg[e] * inv_rho_g;
      T z, s;
      project_row<T>(((d.soft_mask >> r) & 1u) != 0, v, lo[e], hi[e], rho_g, inv_rg, lam, z, s);
      const T y = yg[e] + rho_g * (zh - z);
      zg[e] = z; yg[e] = y; sv[e] = rho_g * z - y;
      if (it == a.iters - 1) a.xi[ggo + e] = s;
    }
    for (int e = tid; e < nown * n; e += nt) xs[e] = alpha * xt[e] + (T(1) - alpha) * xs[e];
    __syncthreads();
    if (nblk == CS && tid < nx) gR[c * nx + tid] = rv[CS * nx + tid];
    grid.sync();
  }
  // ---- write back the state
  for (int e = tid; e < nown * n; e += nt) a.x[gxo + e] = xs[e];
  for (int e = tid; e < nown * ng; e += nt) { a.zg[ggo + e] = zg[e]; a.yg[ggo + e] = yg[e]; }
  for (int e = tid; e < (nblk + 1) * nx; e += nt) {
    const int k = e / nx - 1, i = e - (k + 1) * nx;
    if (k < 0) { if (c == 0) a.yf[(size_t)p * mf + i] = yf[e]; }
    else a.yf[(size_t)p * mf + nx + (size_t)(a0 + k) * nx + i] = yf[e];
  }
}

}  // namespace tmpc
