// tmpc_factor2.cuh — a2 + a3 for the resident fast path: twisted block Cholesky, one WARP per half chain with
// compile-time block sizes.
//
// Twisted ("burn at both ends") block LDL' factor for the resident fast path (tmpc_admm3.cuh).
//
// The block-tridiagonal S is eliminated from BOTH ends towards the middle stage m = T/2: the up chain runs over
// stages 0,1,..,m-1 and the down chain over N,N-1,..,m+1, independently; the middle pivot collects both Schur
// contributions.  With  Psi_t = block(next stage of the chain, t) of S  (up: Phi_t; down: Phi_{t-1}'),
//     Sigma_first = Theta_first,  L_t L_t' = Sigma_t,  W_t = Psi_t L_t^{-T},  Sigma_next = Theta_next - W_t W_t',
//     Sigma_m = Theta_m - W_{m-1} W_{m-1}' - W_{m+1} W_{m+1}'   (block Cholesky with the middle stage eliminated last).
// Stored with explicit inverses of the diagonal Cholesky blocks, X_t = L_t^{-1}, and the off-diagonal blocks pre- and
// post-multiplied by them, B_t = X_next W_t, so that the two sequential sweeps are pure mat-vecs on scaled variables:
//     eta~_t = X_t eta_t (stage-parallel),  w_next = eta~_next - B_t w_t,  w_m = eta~_m - B_{m-1} w_{m-1} - B_{m+1} w_{m+1},
//     y_m = w_m,  y_t = w_t - B_t' y_next (outwards from m),  x_t = X_t' y_t (stage-parallel).
// It is an exact factorisation of the same S (P A P' = L D L' for the permutation that orders stages
// 0, N, 1, N-1, ...), same flops and same storage as the one-directional form, but both substitution sweeps of a
// solve are two independent chains of half the length.
// Layout: Lam [B][T][n][n] holds B_t, indexed by the stage t the block belongs to (slot m unused); Sinv [B][T][n][n]
// holds X_t (lower triangular, zeros stored).
//
// The generic CTA-level factor_kernel (tmpc_factor.cuh) spends its time in CTA barriers, run-time integer divisions and
// dependent global loads; here a CTA is two warps (the up chain and the down chain of one problem), every phase of a stage is separated
// by __syncwarp only, the raw stage data (D_t, E_t, A^-_t, A^+_{t-1}, G_t) of the NEXT stage is prefetched into
// registers while the current stage is factored, and all index arithmetic is compile-time.  Arithmetic in double.
#pragma once
#include "tmpc_factor.cuh"

namespace tmpc {

// TW = true: twisted factor (X_t, B_t) for admm3_kernel.  TW = false: the one-directional block LDL' of factor_kernel
// (Lam_t = Phi_t Sigma_t^{-1}, Sinv_t = Sigma_t^{-1}; per-row weights w_rows supported) for the backward pass; one warp.
// WPC warps per chain: 1 for batches that fill the GPU (12 CTAs of two warps per SM, throughput bound); 4 (8 for n = 12) for small batches, where
// the launch is as long as ONE problem's chain (2000+ dependent warp instructions per stage for n = 12 on one warp) — the element loops are then
// spread over 128 (256) threads per chain and the phases are separated by a named barrier per chain instead of __syncwarp.  Same sums in the
// same order.  Measured at (64,40,8,4) fp64: 341 -> 128 -> 108 us per launch; two warps per chain for mid-size batches (B = 1024) lost to the
// register cap its eight CTAs per SM need (554 against 477 us).
template <typename T, int NC, int NX, bool TW, int WPC = 1, int MB = 0>
__global__ void __launch_bounds__(64 * WPC, MB ? MB : (WPC == 1 ? 12 : (WPC <= 4 ? 2 : 1))) factor_tw2_kernel(FactorArgs<T> a) {
  constexpr int n = NC, nx = NX, nn = NC * NC, an = NX * NC;
  constexpr int GT = 32 * WPC;                          // threads per chain
  constexpr int EPL = (nn + GT - 1) / GT;               // matrix elements per lane
  constexpr int GMAX = NC * NC;                         // room for ng <= n rows of G
  constexpr int RAW = 2 * nn + 2 * an + GMAX;           // D, E, Am, Ap, G
  constexpr int RPL = (RAW + GT - 1) / GT;
  __shared__ double sm[2][3 * nn + RAW + NC];
  const Dims& d = a.d;
  const int ng = d.ng, N = d.N, T_ = d.T;
  const int half = threadIdx.x / GT, lane = threadIdx.x % GT, p = blockIdx.x;
  auto gsync = [&]() { if constexpr (WPC == 1) __syncwarp(); else asm volatile("bar.sync %0, %1;" ::"r"(1 + half), "r"(GT) : "memory"); };
  double* A = sm[half]; double* Bm = A + nn; double* C = Bm + nn;
  double* rD = C + nn; double* rE = rD + nn; double* rAm = rE + nn; double* rAp = rAm + an; double* rG = rAp + an;
  const T* Dp = a.qp.D + a.qp.sD * p;
  const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Amp = a.qp.Am + (size_t)p * N * an;
  const T* App = a.qp.Ap + (size_t)p * N * an;
  const T* Gp = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  T* Lamp = a.Lam + (size_t)p * (TW ? T_ : N) * nn;
  T* Xp = a.Sinv + (size_t)p * T_ * nn;
  const int m = TW ? T_ / 2 : T_, cnt = half ? T_ - 1 - m : m;      // !TW: the up chain covers every stage, no middle
  const T* wr = a.w_rows ? a.w_rows + (size_t)p * T_ * ng : nullptr;
  if (a.mask && !a.mask[p]) return;
  const double w_in = a.rho_bar ? (double)a.rho_bar[p] : a.w_in, w_eq = a.rho_bar ? a.rho_scale * w_in : a.w_eq, sigma = a.sigma;
  int bad = 0;

  // raw data of stage t for this chain: D_t, the coupling block E_tc (tc = t for up, t-1 for down), A^-_t, A^+_{t-1}, G_t
  auto raw_src = [&](int t, int e) -> T {
    if (e < nn) return Dp[(size_t)t * nn + e];
    e -= nn;
    if (e < nn) { const int tc = half ? t - 1 : t; return (tc >= 0 && tc < N) ? Ep[(size_t)tc * nn + e] : T(0); }
    e -= nn;
    if (e < an) return t < N ? Amp[(size_t)t * an + e] : T(0);
    e -= an;
    if (e < an) return t > 0 ? App[(size_t)(t - 1) * an + e] : T(0);
    e -= an;
    return (Gp && e < ng * n) ? Gp[(size_t)t * ng * n + e] : T(0);
  };
  T pre[RPL];
  auto prefetch = [&](int t) {
#pragma unroll
    for (int u = 0; u < RPL; ++u) { const int e = lane + GT * u; pre[u] = e < RAW ? raw_src(t, e) : T(0); }
  };
  auto commit = [&]() {
#pragma unroll
    for (int u = 0; u < RPL; ++u) { const int e = lane + GT * u; if (e < RAW) rD[e] = (double)pre[u]; }
  };
  // The phases that touch the LOWER TRIANGLE only (Theta, the Cholesky updates, the triangular inverse) walk its n (n + 1) / 2 elements, TPL per
  // lane, instead of all n^2 with half of them masked: for n = 6 that is one pass of 21 lanes instead of two passes (36 > 32).  The (row, column)
  // of a lane's elements never changes, so it is worked out once.
  // Used where it saves a pass (n = 6, n = 12; measured: config 4 22.0 -> 21.7 ms, (1024,40,8,4) factor 459 -> 377 us); for n = 8 both walks take
  // two passes and the plain one is faster (config 2 1.053 vs 1.068 ms), so it keeps e = lane + GT u with the upper triangle masked.
  constexpr int NTRI = n * (n + 1) / 2, TPT = (NTRI + GT - 1) / GT;
  constexpr bool TRI = TPT < EPL;
  constexpr int TPL = TRI ? TPT : EPL;
  int tri_e[TRI ? TPL : 1];                             // triangular walk: i * n + j of my u-th element, -1 for none
  if constexpr (TRI) {
#pragma unroll
    for (int u = 0; u < TPL; ++u) {
      const int q = lane + GT * u;
      int i = 0;
#pragma unroll
      for (int r = 1; r < n; ++r) if (q >= r * (r + 1) / 2) i = r;
      tri_e[u] = q < NTRI ? i * n + (q - i * (i + 1) / 2) : -1;
    }
  }
  // Theta_t (lower triangle) minus W W' of up to two finished neighbours, from the raw data in shared memory
  auto theta = [&](int t, double* dst, const double* W1, const double* W2) {
#pragma unroll
    for (int u = 0; u < TPL; ++u) {
      int e;
      if constexpr (TRI) { e = tri_e[u]; if (e < 0) continue; }
      else { e = lane + GT * u; if (e >= nn) continue; }
      const int i = e / n, j = e % n;
      if constexpr (!TRI) { if (j > i) continue; }
      double s = rD[e];
      if (i == j) s += sigma;
      double acc = 0;
#pragma unroll
      for (int r = 0; r < nx; ++r) acc += rAm[r * n + i] * rAm[r * n + j] + rAp[r * n + i] * rAp[r * n + j];
      if (t == 0 && i == j && i < nx) acc += 1;        // A_init' A_init = blkdiag(I_nx, 0)
      s += w_eq * acc;
      if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i && i == j) s += wr ? (double)wr[t * ng + r] : w_in; }
      else { for (int r = 0; r < ng; ++r) s += (wr ? (double)wr[t * ng + r] : w_in) * rG[r * n + i] * rG[r * n + j]; }
      if (W1) { double c = 0;
#pragma unroll
        for (int k = 0; k < n; ++k) c += W1[i * n + k] * W1[j * n + k];
        s -= c; }
      if (W2) { double c = 0;
#pragma unroll
        for (int k = 0; k < n; ++k) c += W2[i * n + k] * W2[j * n + k];
        s -= c; }
      dst[e] = s;
    }
  };
  // in-place Cholesky of the lower triangle of Am_ (right-looking), then Xo <- L^{-1}.  One rsqrt per pivot and no
  // division: 1 / L_kk is kept in registers (compile-time k) and in `rsd` for the final row scaling.
  double* rsd = sm[half] + 3 * nn + RAW;
  auto chol_inv = [&](double* Am_, double* Xo) {
    double rsk[n];
#pragma unroll
    for (int k = 0; k < n; ++k) {
      double dk = Am_[k * n + k];
      if (!(dk > 0) || !isfinite(dk)) { bad = 1; dk = 1; }
      const double rs = rsqrt(dk), sq = dk * rs, inv = rs * rs;
      rsk[k] = rs;
#pragma unroll
      for (int u = 0; u < TPL; ++u) {
        if constexpr (TRI) { const int e = tri_e[u], i = e / n, j = e % n; if (e >= 0 && j > k) Am_[e] -= Am_[i * n + k] * Am_[j * n + k] * inv; }
        else { const int e = lane + GT * u, i = e / n, j = e % n; if (e < nn && j > k && j <= i) Am_[e] -= Am_[i * n + k] * Am_[j * n + k] * inv; }
      }
      gsync();
      if (lane < n && lane >= k) Am_[lane * n + k] = lane == k ? sq : Am_[lane * n + k] * rs;
      if (lane == 0) rsd[k] = rs;
      gsync();
    }
#pragma unroll
    for (int u = 0; u < EPL; ++u) { const int e = lane + GT * u; if (e < nn) Xo[e] = (e / n == e % n) ? 1.0 : 0.0; }
    gsync();
#pragma unroll
    for (int k = 0; k < n - 1; ++k) {
      const double inv = rsk[k];
#pragma unroll
      for (int u = 0; u < TPL; ++u) {
        if constexpr (TRI) { const int e = tri_e[u], i = e / n, j = e % n; if (e >= 0 && i > k && j <= k) Xo[e] -= Am_[i * n + k] * Xo[k * n + j] * inv; }
        else { const int e = lane + GT * u, i = e / n, j = e % n; if (e < nn && i > k && j <= k) Xo[e] -= Am_[i * n + k] * Xo[k * n + j] * inv; }
      }
      gsync();
    }
#pragma unroll
    for (int u = 0; u < EPL; ++u) { const int e = lane + GT * u; if (e < nn) Xo[e] = Xo[e] * rsd[e / n]; }
    gsync();
  };
  auto x_out = [&](int t, const double* X) {
#pragma unroll
    for (int u = 0; u < EPL; ++u) { const int e = lane + GT * u; if (e < nn) Xp[(size_t)t * nn + e] = (T)X[e]; }
  };
  auto b_out = [&](int tprev, const double* X, const double* W) {      // B = X_next W_prev
#pragma unroll
    for (int u = 0; u < EPL; ++u) {
      const int e = lane + GT * u;
      if (e >= nn) continue;
      const int i = e / n, j = e % n;
      double s = 0;
#pragma unroll
      for (int k = 0; k < n; ++k) if (k <= i) s += X[i * n + k] * W[k * n + j];
      Lamp[(size_t)tprev * nn + e] = (T)s;
    }
  };

  if (cnt > 0) prefetch(half ? N : 0);
  for (int k = 0; k < cnt; ++k) {
    const int t = half ? N - k : k;
    commit();
    gsync();
    if (k + 1 < cnt) prefetch(half ? t - 1 : t + 1);
    theta(t, A, k > 0 ? C : nullptr, nullptr);
    gsync();
    chol_inv(A, Bm);
    if constexpr (TW) { if (k > 0) b_out(half ? t + 1 : t - 1, Bm, C); x_out(t, Bm); }
    else {                                             // Sinv_t = X'X
#pragma unroll
      for (int u = 0; u < EPL; ++u) {
        const int e = lane + GT * u;
        if (e >= nn) continue;
        const int i = e / n, j = e % n;
        double s = 0;
#pragma unroll
        for (int kk = 0; kk < n; ++kk) if (kk >= i && kk >= j) s += Bm[kk * n + i] * Bm[kk * n + j];
        Xp[(size_t)t * nn + e] = (T)s;
      }
      if (t == N) break;
    }
    gsync();
    // A <- Psi_t: up Phi_t = E_t + w A^+_t' A^-_t ; down Phi_{t-1}' = E_{t-1}' + w A^-_{t-1}' A^+_{t-1}.
    // up needs A^+_t (not in this stage's raw data): read it from global; down has A^+_{t-1} (rAp) and needs A^-_{t-1}.
    {
      const int tc = half ? t - 1 : t;
      const T* other = half ? Amp + (size_t)tc * an : App + (size_t)tc * an;
#pragma unroll
      for (int u = 0; u < EPL; ++u) {
        const int e = lane + GT * u;
        if (e >= nn) continue;
        const int i = e / n, j = e % n;
        const int ii = half ? j : i, jj = half ? i : j; // Phi[ii][jj] = E[ii][jj] + w sum_r A^+[r][ii] A^-[r][jj]
        double acc = 0;
#pragma unroll
        for (int r = 0; r < nx; ++r) acc += half ? rAp[r * n + ii] * (double)other[r * n + jj] : (double)other[r * n + ii] * rAm[r * n + jj];
        A[e] = rE[ii * n + jj] + w_eq * acc;
      }
    }
    gsync();
#pragma unroll
    for (int u = 0; u < EPL; ++u) {                     // C <- W = Psi X'
      const int e = lane + GT * u;
      if (e >= nn) continue;
      const int i = e / n, j = e % n;
      double s = 0;
#pragma unroll
      for (int kk = 0; kk < n; ++kk) if (kk <= j) s += A[i * n + kk] * Bm[j * n + kk];
      C[e] = s;
    }
    gsync();
    if constexpr (!TW) {                                // Lambda_t = W X
#pragma unroll
      for (int u = 0; u < EPL; ++u) {
        const int e = lane + GT * u;
        if (e >= nn) continue;
        const int i = e / n, j = e % n;
        double s = 0;
#pragma unroll
        for (int kk = 0; kk < n; ++kk) if (kk >= j) s += C[i * n + kk] * Bm[kk * n + j];
        Lamp[(size_t)t * nn + e] = (T)s;
      }
    }
  }
  __syncthreads();
  // ---- middle stage m (warp 0): both chains' last W feed Sigma_m
  if (TW && half == 0) {
    const double* Wup = sm[0] + 2 * nn; const double* Wdn = sm[1] + 2 * nn;
    prefetch(m); commit();
    gsync();
    theta(m, A, m > 0 ? Wup : nullptr, (T_ - 1 - m) > 0 ? Wdn : nullptr);
    gsync();
    chol_inv(A, Bm);
    if (m > 0) b_out(m - 1, Bm, Wup);
    if (T_ - 1 - m > 0) b_out(m + 1, Bm, Wdn);
    x_out(m, Bm);
  }
  bad = __syncthreads_or(bad);
  if (a.status && threadIdx.x == 0) a.status[p] = bad ? TMPC_ST_PIVOT : 0;
}

}  // namespace tmpc
