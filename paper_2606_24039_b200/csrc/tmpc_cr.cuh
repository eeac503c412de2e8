// tmpc_cr.cuh — a11: parallel-in-time factor and solve of the block-tridiagonal S by block cyclic reduction
// (odd-even elimination; textbook, cited as prior art at PAPER.md:86) for a single long horizon (config 5).
//
// Level l (h = 2^l) eliminates the stages j = h(2k+1) < T; survivors are the multiples of 2h.  With Lo_j the
// current block (j, j-h) and a = j-h, b = j+h the neighbours of an eliminated stage j:
//     U_j = Theta_j^{-1},   FA_j = Lo_j' U_j,   FB_j = Lo_b U_j                      (stored for the solves)
//     Theta_a -= FA_j Lo_j,   Theta_b -= FB_j Lo_b',   Lo_b(new, couples b and a) = -FB_j Lo_j
//     down-sweep  eta_a -= FA_j eta_j,  eta_b -= FB_j eta_j ;  root x_0 = U_0 eta_0
//     up-sweep    x_j = U_j eta_j - FA_j' x_a - FB_j' x_b.
// Every Theta met is a Schur complement of the SPD matrix S, hence SPD: each pivot block is inverted through its
// Cholesky factor.  ceil(log2 T) levels; T need not be a power of two (out-of-range neighbours simply vanish).
// All updates are written in GATHER form (each survivor pulls from its two eliminated neighbours) so that there are
// no write conflicts and the result is deterministic.
//
// v1 layout: everything in global memory (L2-resident: 5 T n^2 elements), one cooperative grid, grid-wide barrier
// between levels.  The fused ADMM loop (Alg. 3) runs entirely inside cr_admm_kernel.
#pragma once
#include <cooperative_groups.h>
#include "tmpc_common.cuh"

namespace tmpc {
namespace cg = cooperative_groups;

template <typename T>
struct CrBuf {         // per problem, carved from the workspace
  T* Th; T* Lo; T* U; T* FA; T* FB;    // [T][n][n]
  T* eta; T* xt;                       // [T][n]
  T* rv; T* sv;                        // [mf], [mg]
  T* part;                             // [3 * max CTAs] reduction partials
  int32_t* flag;
};

inline size_t cr_workspace_bytes(const Dims& d, size_t es) {
  const size_t nn = (size_t)d.n * d.n;
  size_t per = 5 * (size_t)d.T * nn + 2 * (size_t)d.nz + d.mf + d.mg + 3 * 4096;
  return (size_t)d.B * per * es + 256 * (size_t)d.B + 1024;
}
template <typename T>
__host__ __device__ inline CrBuf<T> cr_carve(const Dims& d, unsigned char* ws, int p) {
  const size_t nn = (size_t)d.n * d.n;
  const size_t per = 5 * (size_t)d.T * nn + 2 * (size_t)d.nz + d.mf + d.mg + 3 * 4096;
  T* base = reinterpret_cast<T*>(ws) + (size_t)p * per;
  CrBuf<T> b;
  b.Th = base; b.Lo = b.Th + d.T * nn; b.U = b.Lo + d.T * nn; b.FA = b.U + d.T * nn; b.FB = b.FA + d.T * nn;
  b.eta = b.FB + d.T * nn; b.xt = b.eta + d.nz; b.rv = b.xt + d.nz; b.sv = b.rv + d.mf; b.part = b.sv + d.mg;
  b.flag = reinterpret_cast<int32_t*>(ws + (size_t)d.B * per * sizeof(T)) + 64 * p;
  return b;
}
__host__ __device__ inline int cr_levels(int T_) { int L = 0; while ((1 << L) < T_) ++L; return L; }

// Light-weight barrier over the gridDim.x CTAs of ONE problem (cooperative launch guarantees co-residency): one
// acq_rel atomic per CTA on a counter; the last arriver resets the counter and bumps a generation word with release
// semantics; the others poll the generation word with acquire loads.  Each CTA counts its own barriers (the expected
// generation lives in a register), so a barrier costs one atomic round trip plus the release/acquire hand-over.
struct GridBar {
  unsigned* cnt; unsigned* gen; unsigned nblocks; unsigned expect;      // expect: generation value that ends my next barrier
  __device__ __forceinline__ void sync() {
    __syncthreads();
    if (threadIdx.x == 0) {
      unsigned old;
      asm volatile("atom.add.acq_rel.gpu.u32 %0, [%1], 1;" : "=r"(old) : "l"(cnt) : "memory");
      if (old == nblocks - 1) {
        asm volatile("st.relaxed.gpu.u32 [%0], %1;" ::"l"(cnt), "r"(0u) : "memory");
        asm volatile("red.release.gpu.add.u32 [%0], 1;" ::"l"(gen) : "memory");
      } else {
        unsigned g;
        do { asm volatile("ld.acquire.gpu.u32 %0, [%1];" : "=r"(g) : "l"(gen) : "memory"); } while ((int)(g - expect) < 0);
      }
    }
    ++expect;
    __syncthreads();
  }
};
template <typename T>
__device__ __forceinline__ GridBar cr_gridbar(const CrBuf<T>& b) {
  unsigned* gen = reinterpret_cast<unsigned*>(b.flag) + 32;
  unsigned g0;                                          // every CTA reads the generation before anyone can have passed a barrier of this launch
  asm volatile("ld.acquire.gpu.u32 %0, [%1];" : "=r"(g0) : "l"(gen) : "memory");
  return GridBar{reinterpret_cast<unsigned*>(b.flag) + 16, gen, gridDim.x, g0 + 1};
}

template <typename T>
struct CrFactorArgs { Dims d; QpView<T> qp; T sigma, rho_f, rho_g; unsigned char* ws; };

// ---- factor: assemble Theta_t, Lo_t = Phi_{t-1}, then ceil(log2 T) elimination levels
template <typename T, int NC>
__global__ void __launch_bounds__(256) cr_factor_kernel(CrFactorArgs<T> a) {
  const Dims& d = a.d;
  constexpr int n = NC, nn = NC * NC;
  const int nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, p = blockIdx.y;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x, gsz = (long long)gridDim.x * blockDim.x;
  CrBuf<T> b = cr_carve<T>(d, a.ws, p);
  GridBar grid = cr_gridbar<T>(b);
  const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Amp = a.qp.Am + (size_t)p * N * nx * n; const T* App = a.qp.Ap + (size_t)p * N * nx * n;
  const T* Gp = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  for (long long e = gid; e < (long long)T_ * nn; e += gsz) {
    const int t = (int)(e / nn), r_ = (int)(e - (long long)t * nn), i = r_ / n, j = r_ - i * n;
    const T* Amt = Amp + (size_t)t * nx * n; const T* Apm = App + (size_t)(t - 1) * nx * n;
    T s = Dp[(size_t)t * nn + r_];
    if (i == j) s += a.sigma;
    T acc = T(0);
    if (t < N) for (int r = 0; r < nx; ++r) acc += Amt[r * n + i] * Amt[r * n + j];
    if (t > 0) for (int r = 0; r < nx; ++r) acc += Apm[r * n + i] * Apm[r * n + j];
    if (t == 0 && i == j && i < nx) acc += T(1);
    s += a.rho_f * acc;
    if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i && i == j) s += a.rho_g; }
    else { const T* Gt = Gp + (size_t)t * ng * n; for (int r = 0; r < ng; ++r) s += a.rho_g * Gt[r * n + i] * Gt[r * n + j]; }
    b.Th[e] = s;
    T lo = T(0);
    if (t > 0) {   // Lo_t = Phi_{t-1} = E_{t-1} + rho_f A^+_{t-1}' A^-_{t-1}
      const T* Amm = Amp + (size_t)(t - 1) * nx * n;
      T c = T(0);
      for (int r = 0; r < nx; ++r) c += Apm[r * n + i] * Amm[r * n + j];
      lo = Ep[(size_t)(t - 1) * nn + r_] + a.rho_f * c;
    }
    b.Lo[e] = lo;
  }
  if (gid == 0) *b.flag = 0;
  grid.sync();
  const int L = cr_levels(T_);
  // One WARP per stage from here on: lane e owns matrix element e (and e + 32 when nn > 32); the small products go
  // through a per-warp shared scratch, the pivot block is inverted in place by Gauss-Jordan (no pivoting: SPD).
  __shared__ T scr[8][6 * NC * NC];
  constexpr int EPL = (nn + 31) / 32;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const long long gw = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
  T* M0 = scr[wib]; T* M1 = M0 + nn; T* M2 = M1 + nn; T* M3 = M2 + nn; T* M4 = M3 + nn;
  auto ld_mat = [&](T* dst, const T* src) {
#pragma unroll
    for (int u = 0; u < EPL; ++u) { const int e = lane + 32 * u; if (e < nn) dst[e] = src ? src[e] : T(0); }
  };
  auto gj_inverse = [&](T* A) -> int {                 // in-place inverse of an SPD block; returns 1 on a bad pivot
    int bad = 0;
#pragma unroll 1
    for (int k = 0; k < n; ++k) {
      T dk = A[k * n + k];
      if (!(dk > T(0)) || !isfinite(dk)) { bad = 1; dk = T(1); }
      const T pinv = T(1) / dk;
      __syncwarp();
#pragma unroll
      for (int u = 0; u < EPL; ++u) { const int e = lane + 32 * u, i = e / n, j = e % n; if (e < nn && i == k && j != k) A[e] *= pinv; }
      __syncwarp();
#pragma unroll
      for (int u = 0; u < EPL; ++u) { const int e = lane + 32 * u, i = e / n, j = e % n; if (e < nn && i != k && j != k) A[e] -= A[i * n + k] * A[k * n + j]; }
      __syncwarp();
#pragma unroll
      for (int u = 0; u < EPL; ++u) { const int e = lane + 32 * u, i = e / n, j = e % n; if (e < nn && j == k) A[e] = (i == k) ? pinv : -A[e] * pinv; }
      __syncwarp();
    }
    return bad;
  };
  for (int l = 0; l < L; ++l) {
    const int h = 1 << l;
    // (1) eliminated stages j = h(2k+1): U_j = Theta_j^{-1}, FA_j = Lo_j' U_j, FB_j = Lo_b U_j
    for (long long k = gw;; k += nw) {
      const long long j = (long long)h * (2 * k + 1);
      if (j >= T_) break;
      const bool hb = j + h < T_;
      ld_mat(M0, b.Th + j * nn); ld_mat(M1, b.Lo + j * nn); ld_mat(M2, hb ? b.Lo + (j + h) * nn : nullptr);
      __syncwarp();
      if (gj_inverse(M0) && lane == 0) atomicOr(b.flag, 1);
#pragma unroll
      for (int u = 0; u < EPL; ++u) {
        const int e = lane + 32 * u, i = e / n, c = e % n;
        if (e >= nn) continue;
        T fa = T(0), fb = T(0);
#pragma unroll
        for (int m = 0; m < n; ++m) { fa += M1[m * n + i] * M0[m * n + c]; fb += M2[i * n + m] * M0[m * n + c]; }
        b.U[j * nn + e] = M0[e]; b.FA[j * nn + e] = fa; if (hb) b.FB[j * nn + e] = fb;
      }
      __syncwarp();
    }
    grid.sync();
    // (2) survivors s = 2hk: Theta_s -= FA_{s+h} Lo_{s+h} + FB_{s-h} Lo_s' ;  Lo_s <- -FB_{s-h} Lo_{s-h}
    for (long long k = gw;; k += nw) {
      const long long s_ = 2LL * h * k;
      if (s_ >= T_) break;
      const bool hp = s_ + h < T_, hm = s_ - h >= 0;
      ld_mat(M0, hp ? b.FA + (s_ + h) * nn : nullptr); ld_mat(M1, hp ? b.Lo + (s_ + h) * nn : nullptr);
      ld_mat(M2, hm ? b.FB + (s_ - h) * nn : nullptr); ld_mat(M3, b.Lo + s_ * nn); ld_mat(M4, hm ? b.Lo + (s_ - h) * nn : nullptr);
      __syncwarp();
#pragma unroll
      for (int u = 0; u < EPL; ++u) {
        const int e = lane + 32 * u, i = e / n, c = e % n;
        if (e >= nn) continue;
        T acc = T(0), nlo = T(0);
#pragma unroll
        for (int m = 0; m < n; ++m) { acc += M0[i * n + m] * M1[m * n + c] + M2[i * n + m] * M3[c * n + m]; nlo -= M2[i * n + m] * M4[m * n + c]; }
        b.Th[s_ * nn + e] -= acc; b.Lo[s_ * nn + e] = nlo;
      }
      __syncwarp();
    }
    grid.sync();
  }
  if (gw == 0) {
    ld_mat(M0, b.Th); __syncwarp();
    if (gj_inverse(M0) && lane == 0) atomicOr(b.flag, 1);
#pragma unroll
    for (int u = 0; u < EPL; ++u) { const int e = lane + 32 * u; if (e < nn) b.U[e] = M0[e]; }
  }
}

}  // namespace tmpc

namespace tmpc {

// ---- the solve with the CR factor, gather form; eta is consumed, x written to xt.
// Levels with many stages run grid-wide (one barrier per level); once at most CR_SMALL stages survive, CTA 0 finishes
// the down-sweep, the root and the first up-sweep levels alone with __syncthreads, the other CTAs wait at one barrier.
constexpr int CR_SMALL = 512;
template <typename T, int NC>
__device__ __forceinline__ void cr_down_level(const CrBuf<T>& b, int T_, long long h, long long w0, long long wstep) {
  constexpr int n = NC, nn = NC * NC;
  for (long long w = w0;; w += wstep) {               // survivors s = 2hk pull from s+h and s-h
    const long long k = w / n; const int i = (int)(w - k * n);
    const long long s_ = 2 * h * k;
    if (s_ >= T_) break;
    T acc = T(0);
    if (s_ + h < T_) { const T* F = b.FA + (s_ + h) * nn + i * n; const T* e = b.eta + (s_ + h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc += F[m] * e[m]; }
    if (s_ - h >= 0) { const T* F = b.FB + (s_ - h) * nn + i * n; const T* e = b.eta + (s_ - h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc += F[m] * e[m]; }
    b.eta[s_ * n + i] -= acc;
  }
}
template <typename T, int NC>
__device__ __forceinline__ void cr_up_level(const CrBuf<T>& b, int T_, long long h, long long w0, long long wstep) {
  constexpr int n = NC, nn = NC * NC;
  for (long long w = w0;; w += wstep) {               // eliminated j = h(2k+1)
    const long long k = w / n; const int i = (int)(w - k * n);
    const long long j = h * (2 * k + 1);
    if (j >= T_) break;
    const T* U = b.U + j * nn + i * n; const T* e = b.eta + j * n;
    T acc = T(0);
#pragma unroll
    for (int m = 0; m < n; ++m) acc += U[m] * e[m];
    { const T* F = b.FA + j * nn + i; const T* xa = b.xt + (j - h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc -= F[m * n] * xa[m]; }
    if (j + h < T_) { const T* F = b.FB + j * nn + i; const T* xb = b.xt + (j + h) * n;
#pragma unroll
      for (int m = 0; m < n; ++m) acc -= F[m * n] * xb[m]; }
    b.xt[j * n + i] = acc;
  }
}
template <typename T, int NC>
__device__ void cr_solve(GridBar& gb, const CrBuf<T>& b, int T_, long long gid, long long gsz) {
  constexpr int n = NC;
  const int L = cr_levels(T_);
  int LS = 0;                                          // levels run grid-wide
  while (LS < L && ((T_ + (1 << LS) - 1) >> LS) > CR_SMALL) ++LS;
  for (int l = 0; l < LS; ++l) { cr_down_level<T, NC>(b, T_, 1LL << l, gid, gsz); gb.sync(); }
  if (blockIdx.x == 0) {
    for (int l = LS; l < L; ++l) { cr_down_level<T, NC>(b, T_, 1LL << l, threadIdx.x, blockDim.x); __syncthreads(); }
    if (threadIdx.x < n) { T acc = T(0);
#pragma unroll
      for (int m = 0; m < n; ++m) acc += b.U[threadIdx.x * n + m] * b.eta[m];
      b.xt[threadIdx.x] = acc; }
    __syncthreads();
    for (int l = L - 1; l >= LS; --l) { cr_up_level<T, NC>(b, T_, 1LL << l, threadIdx.x, blockDim.x); __syncthreads(); }
  }
  gb.sync();
  for (int l = LS - 1; l >= 0; --l) { cr_up_level<T, NC>(b, T_, 1LL << l, gid, gsz); gb.sync(); }
}

template <typename T>
struct CrAdmmArgs {
  Dims d; Params<T> prm; QpView<T> qp; unsigned char* ws;
  T* x; T* zg; T* yf; T* yg; T* xi; T* r_prim; T* r_dual; T* objective; int32_t* status;
  int iters, zg_given, kkt_only;
  const T* eta_in; T* xt_out;
};

// ---- fused ADMM loop (Alg. 3) on the CR factor: one cooperative grid, blockIdx.y = problem
template <typename T, int NC>
__global__ void __launch_bounds__(256) cr_admm_kernel(CrAdmmArgs<T> a) {
  __shared__ T red[64];
  const Dims& d = a.d;
  constexpr int n = NC, nn = NC * NC;
  const int nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nz = d.nz, mf = d.mf, mg = d.mg, p = blockIdx.y;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x, gsz = (long long)gridDim.x * blockDim.x;
  CrBuf<T> b = cr_carve<T>(d, a.ws, p);
  GridBar grid = cr_gridbar<T>(b);
  if (a.kkt_only) {
    for (long long e = gid; e < nz; e += gsz) b.eta[e] = a.eta_in[(size_t)p * nz + e];
    grid.sync();
    cr_solve<T, NC>(grid, b, T_, gid, gsz);
    for (long long e = gid; e < nz; e += gsz) a.xt_out[(size_t)p * nz + e] = b.xt[e];
    return;
  }
  const T sigma = a.prm.sigma, rho_f = a.prm.rho_f, rho_g = a.prm.rho_g, alpha = a.prm.alpha;
  const T inv_rho_g = T(1) / rho_g, inv_rg = T(1) / (rho_g + a.prm.gamma), lam = a.prm.lam, gam = a.prm.gamma;
  T* x = a.x + (size_t)p * nz; T* zg = a.zg + (size_t)p * mg; T* yf = a.yf + (size_t)p * mf; T* yg = a.yg + (size_t)p * mg; T* xi = a.xi + (size_t)p * mg;
  const T* q = a.qp.q + (size_t)p * nz; const T* lo = a.qp.lo + (size_t)p * mg; const T* hi = a.qp.hi + (size_t)p * mg;
  const T* Am = a.qp.Am + (size_t)p * N * nx * n; const T* Ap = a.qp.Ap + (size_t)p * N * nx * n;
  const T* G = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  const T* xin = a.qp.x_init + (size_t)p * nx; const T* bb = a.qp.b + (size_t)p * N * nx;
  auto cval = [&](long long e) -> T { return e < nx ? xin[e] : bb[e - nx]; };
  auto g_dot = [&](int t, int r, const T* vec) -> T {
    if (d.g_sel) return vec[(size_t)t * n + d.g_col[r]];
    const T* g = G + ((size_t)t * ng + r) * n; const T* vt = vec + (size_t)t * n; T s = T(0);
#pragma unroll
    for (int j = 0; j < n; ++j) s += g[j] * vt[j];
    return s;
  };
  auto c_row = [&](long long e, const T* v) -> T {
    if (e < nx) return v[e];
    const long long t = (e - nx) / nx; const int i = (int)((e - nx) - t * nx);
    const T* am = Am + ((size_t)t * nx + i) * n; const T* ap = Ap + ((size_t)t * nx + i) * n; T s = T(0);
#pragma unroll
    for (int j = 0; j < n; ++j) s += am[j] * v[t * n + j] + ap[j] * v[(t + 1) * n + j];
    return s;
  };
  for (long long e = gid; e < mg; e += gsz) {
    const int t = (int)(e / ng), r = (int)(e - (long long)t * ng);
    if (!a.zg_given) { zg[e] = tmin(tmax(g_dot(t, r, x), lo[e]), hi[e]); xi[e] = T(0); }
    b.sv[e] = rho_g * zg[e] - yg[e];
  }
  for (long long e = gid; e < mf; e += gsz) b.rv[e] = rho_f * cval(e) - yf[e];
  grid.sync();
  for (int it = 0; it < a.iters; ++it) {
    for (long long e = gid; e < nz; e += gsz) {       // a4 (eq. 51)
      const long long t = e / n; const int i = (int)(e - t * n);
      T s = sigma * x[e] - q[e];
      if (t == 0 && i < nx) s += b.rv[i];
      if (t < N) { const T* A_ = Am + (size_t)t * nx * n + i; const T* r = b.rv + nx + t * nx; for (int k = 0; k < nx; ++k) s += A_[k * n] * r[k]; }
      if (t > 0) { const T* A_ = Ap + (size_t)(t - 1) * nx * n + i; const T* r = b.rv + nx + (t - 1) * nx; for (int k = 0; k < nx; ++k) s += A_[k * n] * r[k]; }
      if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) s += b.sv[t * ng + r]; }
      else { const T* g = G + (size_t)t * ng * n + i; for (int r = 0; r < ng; ++r) s += g[r * n] * b.sv[t * ng + r]; }
      b.eta[e] = s;
    }
    grid.sync();
    cr_solve<T, NC>(grid, b, T_, gid, gsz);          // a11 (eq. 8)
    for (long long e = gid; e < mf; e += gsz) {       // a7 + a8
      const T c = cval(e);
      const T y = yf[e] + rho_f * alpha * (c_row(e, b.xt) - c);
      yf[e] = y; b.rv[e] = rho_f * c - y;
    }
    for (long long e = gid; e < mg; e += gsz) {
      const int t = (int)(e / ng), r = (int)(e - (long long)t * ng);
      const T zh = alpha * g_dot(t, r, b.xt) + (T(1) - alpha) * zg[e];
      const T v = zh + yg[e] * inv_rho_g;
      T z, s;
      project_row<T>(((d.soft_mask >> r) & 1u) != 0, v, lo[e], hi[e], rho_g, inv_rg, lam, z, s);
      const T y = yg[e] + rho_g * (zh - z);
      zg[e] = z; xi[e] = s; yg[e] = y; b.sv[e] = rho_g * z - y;
    }
    for (long long e = gid; e < nz; e += gsz) x[e] = alpha * b.xt[e] + (T(1) - alpha) * x[e];
    grid.sync();
  }
  // ---- a9 residuals / objective: per-CTA partials, then CTA 0 reduces in a fixed order
  if (a.r_prim || a.r_dual || a.objective || a.status) {
    const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p;
    T rp = T(0), rd = T(0), ob = T(0);
    for (long long e = gid; e < mf; e += gsz) rp = tmax(rp, tabs(c_row(e, x) - cval(e)));
    for (long long e = gid; e < mg; e += gsz) {
      const int t = (int)(e / ng), r = (int)(e - (long long)t * ng);
      rp = tmax(rp, tabs(g_dot(t, r, x) - zg[e]));
      if (((d.soft_mask >> r) & 1u) && xi[e] != T(0)) {
        const T sg = xi[e] > T(0) ? T(1) : T(-1);
        rd = tmax(rd, tabs(gam * xi[e] + lam * sg + yg[e]));
        ob += lam * tabs(xi[e]) + T(0.5) * gam * xi[e] * xi[e];
      }
    }
    for (long long e = gid; e < nz; e += gsz) {
      const long long t = e / n; const int i = (int)(e - t * n);
      T px = T(0);
      const T* Dt = Dp + (size_t)t * nn + i * n;
      for (int j = 0; j < n; ++j) px += Dt[j] * x[t * n + j];
      if (t > 0) { const T* Et = Ep + (size_t)(t - 1) * nn + i * n; for (int j = 0; j < n; ++j) px += Et[j] * x[(t - 1) * n + j]; }
      if (t < N) { const T* Et = Ep + (size_t)t * nn + i; for (int j = 0; j < n; ++j) px += Et[j * n] * x[(t + 1) * n + j]; }
      T g = px + q[e];
      if (t == 0 && i < nx) g += yf[i];
      if (t < N) { const T* A_ = Am + (size_t)t * nx * n + i; for (int k = 0; k < nx; ++k) g += A_[k * n] * yf[nx + t * nx + k]; }
      if (t > 0) { const T* A_ = Ap + (size_t)(t - 1) * nx * n + i; for (int k = 0; k < nx; ++k) g += A_[k * n] * yf[nx + (t - 1) * nx + k]; }
      if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) g += yg[t * ng + r]; }
      else { const T* gg = G + (size_t)t * ng * n + i; for (int r = 0; r < ng; ++r) g += gg[r * n] * yg[t * ng + r]; }
      rd = tmax(rd, tabs(g));
      ob += T(0.5) * x[e] * px + q[e] * x[e];
    }
    rp = block_max(rp, red); rd = block_max(rd, red); ob = block_sum(ob, red);
    if (threadIdx.x == 0) { b.part[3 * blockIdx.x] = rp; b.part[3 * blockIdx.x + 1] = rd; b.part[3 * blockIdx.x + 2] = ob; }
    grid.sync();
    if (gid == 0) {
      T RP = T(0), RD = T(0), OB = T(0);
      for (unsigned c = 0; c < gridDim.x; ++c) { RP = tmax(RP, b.part[3 * c]); RD = tmax(RD, b.part[3 * c + 1]); OB += b.part[3 * c + 2]; }
      if (a.r_prim) a.r_prim[p] = RP;
      if (a.r_dual) a.r_dual[p] = RD;
      if (a.objective) a.objective[p] = OB;
      if (a.status) { int st = (*b.flag ? TMPC_ST_PIVOT : 0) | (isfinite(OB) ? 0 : TMPC_ST_NAN); if (st) atomicOr(&a.status[p], st); }
    }
  }
}

// ---- host launchers
template <typename K, typename A>
inline tmpc_status cr_launch(K kern, A& args, const Dims& d, cudaStream_t s, int64_t* launches) {
  int dev = 0, sms = 0, per_sm = 0, coop = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  if (!coop) return TMPC_E_UNSUPPORTED;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, 0) != cudaSuccess || per_sm < 1) return TMPC_E_CUDA;
  long long want = ((long long)d.nz + 255) / 256;
  long long cap = (long long)sms * per_sm / d.B;
  if (cap < 1) return TMPC_E_UNSUPPORTED;
  if (want > cap) want = cap;
  if (want > 4096) want = 4096;
  dim3 grid((unsigned)want, (unsigned)d.B), block(256);
  void* params[] = { (void*)&args };
  if (cudaLaunchCooperativeKernel((void*)kern, grid, block, params, 0, s) != cudaSuccess) { cudaGetLastError(); return TMPC_E_CUDA; }
  if (launches) ++*launches;
  return TMPC_OK;
}

template <typename T>
tmpc_status cr_factor(const Dims& d, const QpView<T>& qp, double sigma, double rho_f, double rho_g, unsigned char* ws, cudaStream_t s, int64_t* launches) {
  CrFactorArgs<T> a; a.d = d; a.qp = qp; a.sigma = (T)sigma; a.rho_f = (T)rho_f; a.rho_g = (T)rho_g; a.ws = ws;
  if (d.n == 6) return cr_launch(cr_factor_kernel<T, 6>, a, d, s, launches);
  if (d.n == 8) return cr_launch(cr_factor_kernel<T, 8>, a, d, s, launches);
  return TMPC_E_UNSUPPORTED;
}
template <typename T>
tmpc_status cr_admm(const Dims& d, const Params<T>& prm, const QpView<T>& qp, unsigned char* ws, T* x, T* zg, T* yf, T* yg, T* xi, T* r_prim, T* r_dual,
                    T* objective, int32_t* status, int iters, bool zg_given, cudaStream_t s, int64_t* launches) {
  CrAdmmArgs<T> a; memset(&a, 0, sizeof(a));
  a.d = d; a.prm = prm; a.qp = qp; a.ws = ws; a.x = x; a.zg = zg; a.yf = yf; a.yg = yg; a.xi = xi;
  a.r_prim = r_prim; a.r_dual = r_dual; a.objective = objective; a.status = status; a.iters = iters; a.zg_given = zg_given;
  if (d.n == 6) return cr_launch(cr_admm_kernel<T, 6>, a, d, s, launches);
  if (d.n == 8) return cr_launch(cr_admm_kernel<T, 8>, a, d, s, launches);
  return TMPC_E_UNSUPPORTED;
}
template <typename T>
tmpc_status cr_kkt_solve(const Dims& d, unsigned char* ws, const T* eta, T* xt, cudaStream_t s, int64_t* launches) {
  CrAdmmArgs<T> a; memset(&a, 0, sizeof(a));
  a.d = d; a.ws = ws; a.kkt_only = 1; a.eta_in = eta; a.xt_out = xt;
  if (d.n == 6) return cr_launch(cr_admm_kernel<T, 6>, a, d, s, launches);
  if (d.n == 8) return cr_launch(cr_admm_kernel<T, 8>, a, d, s, launches);
  return TMPC_E_UNSUPPORTED;
}

}  // namespace tmpc
