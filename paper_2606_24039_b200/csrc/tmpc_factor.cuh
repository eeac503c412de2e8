// tmpc_factor.cuh — a2 + a3: assemble Theta_t, Phi_t and factor the block-tridiagonal S.
//
// Factor form: block LDL' with explicit inverses of the pivot blocks,
//     Sigma_0 = Theta_0,   Lambda_t = Phi_t Sigma_t^{-1},   Sigma_{t+1} = Theta_{t+1} - Lambda_t Phi_t',
// which is the block Cholesky of S with L_tt L_tt' = Sigma_t and L_{t+1,t} = Phi_t L_tt^{-T} written so that every
// step of the two substitution chains of the solve is ONE dense n x n mat-vec (no dependent triangular solve):
//     forward  w_t = eta_t - Lambda_{t-1} w_{t-1},   middle v_t = Sigma_t^{-1} w_t,   backward x_t = v_t - Lambda_t' x_{t+1}.
// Stored per problem in the workspace: Lam [N][n][n], Sinv [T][n][n] (working dtype).  Arithmetic of the factor
// is done in TA (double) whatever the working dtype, so that fp32 solves inherit a factor accurate to rounding.
//
// One CTA per problem, sequential in t, parallel inside the n x n blocks.  Three n x n shared buffers:
//   A: Sigma_t -> chol L (in place) ; later Phi_t ; later Lambda_t       Bm: X = L^{-1}      C: W_t = Phi_t X'
// with Sigma_{t+1} = Theta_{t+1} - W_t W_t'  (because Lambda_t Phi_t' = Phi_t X'X Phi_t').
#pragma once
#include "tmpc_common.cuh"

namespace tmpc {

template <typename T>
struct FactorArgs {
  Dims d;
  QpView<T> qp;
  double sigma, w_eq, w_in;     // weights: equality rows, inequality rows (scalar)
  const T* w_rows;              // optional per-inequality-row weights [B][T][ng] (overrides w_in), else null
  T* Lam; T* Sinv;              // outputs [B][N][n][n], [B][T][n][n]
  int32_t* status;              // [B], bits OR-ed in (may be null)
};

template <typename T, typename TA>
__global__ void __launch_bounds__(1024) factor_kernel(FactorArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TA* A = reinterpret_cast<TA*>(smem_raw);
  const Dims& d = a.d;
  const int n = d.n, nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nn = n * n;
  TA* Bm = A + nn;
  TA* C = Bm + nn;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const T* Dp = a.qp.D + a.qp.sD * p;
  const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Amp = a.qp.Am + (size_t)p * N * nx * n;
  const T* App = a.qp.Ap + (size_t)p * N * nx * n;
  const T* Gp = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  const T* wr = a.w_rows ? a.w_rows + (size_t)p * T_ * ng : nullptr;
  T* Lamp = a.Lam + (size_t)p * N * nn;
  T* Sinvp = a.Sinv + (size_t)p * T_ * nn;
  int bad = 0;

  for (int t = 0; t < T_; ++t) {
    const T* Dt = Dp + (size_t)t * nn;
    const T* Amt = Amp + (size_t)t * nx * n;            // valid for t < N
    const T* Apm = App + (size_t)(t - 1) * nx * n;      // A^+_{t-1}, valid for t > 0
    const T* Gt = Gp ? Gp + (size_t)t * ng * n : nullptr;
    // ---- A <- Theta_t - W_{t-1} W_{t-1}'   (lower triangle is enough; computed full for simplicity of indexing)
    for (int e = tid; e < nn; e += nt) {
      const int i = e / n, j = e - i * n;
      if (j > i) continue;
      TA s = (TA)Dt[e];
      if (i == j) s += a.sigma;
      TA acc = 0;
      if (t < N) for (int r = 0; r < nx; ++r) acc += (TA)Amt[r * n + i] * (TA)Amt[r * n + j];
      if (t > 0) for (int r = 0; r < nx; ++r) acc += (TA)Apm[r * n + i] * (TA)Apm[r * n + j];
      if (t == 0 && i == j && i < nx) acc += 1;        // A_init' A_init = blkdiag(I_nx, 0)
      s += a.w_eq * acc;
      if (d.g_sel) {
        for (int r = 0; r < ng; ++r) if (d.g_col[r] == i && i == j) s += wr ? (TA)wr[t * ng + r] : (TA)a.w_in;
      } else {
        for (int r = 0; r < ng; ++r) s += (wr ? (TA)wr[t * ng + r] : (TA)a.w_in) * (TA)Gt[r * n + i] * (TA)Gt[r * n + j];
      }
      if (t > 0) { TA c = 0; for (int k = 0; k < n; ++k) c += C[i * n + k] * C[j * n + k]; s -= c; }
      A[e] = s;
    }
    __syncthreads();
    // ---- in-place right-looking Cholesky of A (lower), one barrier per column
    for (int k = 0; k < n; ++k) {
      TA dk = A[k * n + k];
      if (!(dk > 0) || !isfinite(dk)) { bad = 1; dk = 1; }
      const TA inv = 1.0 / dk;
      const int m = n - 1 - k;                         // trailing size
      for (int e = tid; e < m * m; e += nt) {
        const int i = k + 1 + e / m, j = k + 1 + e % m;
        if (j <= i) A[i * n + j] -= A[i * n + k] * A[j * n + k] * inv;
      }
      __syncthreads();
      const TA rs = 1.0 / sqrt(dk);
      for (int i = k + tid; i < n; i += nt) A[i * n + k] = (i == k) ? sqrt(dk) : A[i * n + k] * rs;
    }
    __syncthreads();
    // ---- Bm <- X = L^{-1} (lower): Y = I; for k: rows i > k:  Y[i][:] -= L[i][k] * Y[k][:] / L[k][k];  final row scaling
    for (int e = tid; e < nn; e += nt) Bm[e] = (e / n == e % n) ? TA(1) : TA(0);
    __syncthreads();
    for (int k = 0; k < n - 1; ++k) {
      const TA inv = 1.0 / A[k * n + k];
      const int m = n - 1 - k, kk = k + 1;             // rows k+1..n-1, columns 0..k
      for (int e = tid; e < m * kk; e += nt) {
        const int i = k + 1 + e / kk, j = e % kk;
        Bm[i * n + j] -= A[i * n + k] * Bm[k * n + j] * inv;
      }
      __syncthreads();
    }
    for (int e = tid; e < nn; e += nt) { const int i = e / n; Bm[e] = Bm[e] / A[i * n + i]; }
    __syncthreads();
    // ---- Sinv_t = X'X -> global ;  A <- Phi_t = E_t + w_eq A^+_t' A^-_t  (t < N)
    for (int e = tid; e < nn; e += nt) {
      const int i = e / n, j = e - i * n;
      TA s = 0;
      for (int k = (i > j ? i : j); k < n; ++k) s += Bm[k * n + i] * Bm[k * n + j];
      Sinvp[(size_t)t * nn + e] = (T)s;
    }
    if (t < N) {
      const T* Apt = App + (size_t)t * nx * n;
      const T* Et = Ep + (size_t)t * nn;
      for (int e = tid; e < nn; e += nt) {
        const int i = e / n, j = e - i * n;
        TA acc = 0;
        for (int r = 0; r < nx; ++r) acc += (TA)Apt[r * n + i] * (TA)Amt[r * n + j];
        A[e] = (TA)Et[e] + a.w_eq * acc;
      }
      __syncthreads();
      // ---- C <- W_t = Phi_t X'   (X lower: sum over k <= j)
      for (int e = tid; e < nn; e += nt) {
        const int i = e / n, j = e - i * n;
        TA s = 0;
        for (int k = 0; k <= j; ++k) s += A[i * n + k] * Bm[j * n + k];
        C[e] = s;
      }
      __syncthreads();
      // ---- Lambda_t = W_t X -> global   (sum over k >= j)
      for (int e = tid; e < nn; e += nt) {
        const int i = e / n, j = e - i * n;
        TA s = 0;
        for (int k = j; k < n; ++k) s += C[i * n + k] * Bm[k * n + j];
        Lamp[(size_t)t * nn + e] = (T)s;
      }
    }
    __syncthreads();
  }
  if (a.status && tid == 0 && bad) atomicOr(&a.status[p], TMPC_ST_PIVOT);
}

// ===================================================================================================================
// Twisted ("burn at both ends") block LDL' factor for the resident fast path (tmpc_admm2.cuh).
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
// One CTA per problem, two halves of blockDim/2 threads, each with its own named barrier and shared buffers.
struct HalfBar {
  int id, cnt;
  __device__ __forceinline__ void sync() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(cnt) : "memory"); }
};

// in-place Cholesky of the lower triangle of A (n x n), then Bm <- X = L^{-1} (lower).  Returns 1 on a bad pivot.
template <typename TA>
__device__ int chol_and_inverse(TA* A, TA* Bm, int n, int ht, int hn, const HalfBar& bar) {
  const int nn = n * n; int bad = 0;
  for (int k = 0; k < n; ++k) {
    TA dk = A[k * n + k];
    if (!(dk > 0) || !isfinite(dk)) { bad = 1; dk = 1; }
    const TA inv = 1.0 / dk;
    const int m = n - 1 - k;
    for (int e = ht; e < m * m; e += hn) {
      const int i = k + 1 + e / m, j = k + 1 + e % m;
      if (j <= i) A[i * n + j] -= A[i * n + k] * A[j * n + k] * inv;
    }
    bar.sync();
    const TA rs = 1.0 / sqrt(dk);
    for (int i = k + ht; i < n; i += hn) A[i * n + k] = (i == k) ? sqrt(dk) : A[i * n + k] * rs;
  }
  for (int e = ht; e < nn; e += hn) Bm[e] = (e / n == e % n) ? TA(1) : TA(0);
  bar.sync();
  for (int k = 0; k < n - 1; ++k) {
    const TA inv = 1.0 / A[k * n + k];
    const int m = n - 1 - k, kk = k + 1;
    for (int e = ht; e < m * kk; e += hn) {
      const int i = k + 1 + e / kk, j = e % kk;
      Bm[i * n + j] -= A[i * n + k] * Bm[k * n + j] * inv;
    }
    bar.sync();
  }
  for (int e = ht; e < nn; e += hn) { const int i = e / n; Bm[e] = Bm[e] / A[i * n + i]; }
  bar.sync();
  return bad;
}

template <typename T, typename TA>
__global__ void __launch_bounds__(1024) factor_tw_kernel(FactorArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Dims& d = a.d;
  const int n = d.n, nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nn = n * n;
  const int hn = blockDim.x >> 1, half = threadIdx.x / hn, ht = threadIdx.x - half * hn;
  TA* A = reinterpret_cast<TA*>(smem_raw) + (size_t)half * 3 * nn;
  TA* Bm = A + nn;
  TA* C = Bm + nn;
  const HalfBar bar{1 + half, hn};
  const int p = blockIdx.x;
  const T* Dp = a.qp.D + a.qp.sD * p;
  const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Amp = a.qp.Am + (size_t)p * N * nx * n;
  const T* App = a.qp.Ap + (size_t)p * N * nx * n;
  const T* Gp = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  const T* wr = a.w_rows ? a.w_rows + (size_t)p * T_ * ng : nullptr;
  T* Lamp = a.Lam + (size_t)p * T_ * nn;
  T* Sinvp = a.Sinv + (size_t)p * T_ * nn;
  const int m = T_ / 2, cnt = half ? T_ - 1 - m : m;
  int bad = 0;

  // Theta_t (lower triangle) minus the Schur contributions W W' of up to two neighbours, into dst
  auto theta = [&](int t, TA* dst, const TA* W1, const TA* W2, int tt, int tn) {
    const T* Dt = Dp + (size_t)t * nn;
    const T* Amt = Amp + (size_t)t * nx * n;            // valid for t < N
    const T* Apm = App + (size_t)(t - 1) * nx * n;      // A^+_{t-1}, valid for t > 0
    const T* Gt = Gp ? Gp + (size_t)t * ng * n : nullptr;
    for (int e = tt; e < nn; e += tn) {
      const int i = e / n, j = e - i * n;
      if (j > i) continue;
      TA s = (TA)Dt[e];
      if (i == j) s += a.sigma;
      TA acc = 0;
      if (t < N) for (int r = 0; r < nx; ++r) acc += (TA)Amt[r * n + i] * (TA)Amt[r * n + j];
      if (t > 0) for (int r = 0; r < nx; ++r) acc += (TA)Apm[r * n + i] * (TA)Apm[r * n + j];
      if (t == 0 && i == j && i < nx) acc += 1;        // A_init' A_init = blkdiag(I_nx, 0)
      s += a.w_eq * acc;
      if (d.g_sel) {
        for (int r = 0; r < ng; ++r) if (d.g_col[r] == i && i == j) s += wr ? (TA)wr[t * ng + r] : (TA)a.w_in;
      } else {
        for (int r = 0; r < ng; ++r) s += (wr ? (TA)wr[t * ng + r] : (TA)a.w_in) * (TA)Gt[r * n + i] * (TA)Gt[r * n + j];
      }
      if (W1) { TA c = 0; for (int k = 0; k < n; ++k) c += W1[i * n + k] * W1[j * n + k]; s -= c; }
      if (W2) { TA c = 0; for (int k = 0; k < n; ++k) c += W2[i * n + k] * W2[j * n + k]; s -= c; }
      dst[e] = s;
    }
  };
  // X (lower triangular, zeros above) -> Sinv slot of stage t
  auto x_out = [&](int t, const TA* X, int tt, int tn) {
    for (int e = tt; e < nn; e += tn) Sinvp[(size_t)t * nn + e] = (T)X[e];
  };
  // B = X_next W_prev -> Lam slot of the stage W belongs to (coupling prev -> next)
  auto b_out = [&](int tprev, const TA* X, const TA* W, int tt, int tn) {
    for (int e = tt; e < nn; e += tn) {
      const int i = e / n, j = e - i * n;
      TA s = 0;
      for (int kk = 0; kk <= i; ++kk) s += X[i * n + kk] * W[kk * n + j];
      Lamp[(size_t)tprev * nn + e] = (T)s;
    }
  };
  for (int k = 0; k < cnt; ++k) {
    const int t = half ? N - k : k;
    theta(t, A, k > 0 ? C : nullptr, nullptr, ht, hn);
    bar.sync();
    bad |= chol_and_inverse<TA>(A, Bm, n, ht, hn, bar);
    if (k > 0) b_out(half ? t + 1 : t - 1, Bm, C, ht, hn);
    x_out(t, Bm, ht, hn);
    bar.sync();
    // A <- Psi_t: up Phi_t = E_t + w A^+_t' A^-_t ; down Phi_{t-1}' = E_{t-1}' + w A^-_{t-1}' A^+_{t-1}
    {
      const int tc = half ? t - 1 : t;                  // index of the coupling block Phi_tc
      const T* Apt = App + (size_t)tc * nx * n; const T* Amt = Amp + (size_t)tc * nx * n; const T* Et = Ep + (size_t)tc * nn;
      for (int e = ht; e < nn; e += hn) {
        const int i = e / n, j = e - i * n;
        const int ii = half ? j : i, jj = half ? i : j; // Phi[ii][jj]
        TA acc = 0;
        for (int r = 0; r < nx; ++r) acc += (TA)Apt[r * n + ii] * (TA)Amt[r * n + jj];
        A[e] = (TA)Et[ii * n + jj] + a.w_eq * acc;
      }
    }
    bar.sync();
    for (int e = ht; e < nn; e += hn) {                 // C <- W = Psi X'  (the Cholesky block L_{next,t})
      const int i = e / n, j = e - i * n;
      TA s = 0;
      for (int kk = 0; kk <= j; ++kk) s += A[i * n + kk] * Bm[j * n + kk];
      C[e] = s;
    }
    bar.sync();
  }
  __syncthreads();
  // ---- middle stage m: both halves' last W (if any) feed Sigma_m
  {
    TA* base = reinterpret_cast<TA*>(smem_raw);
    TA* A0 = base; TA* B0 = base + nn; const TA* Wup = base + 2 * nn; const TA* Wdn = base + 5 * nn;
    const HalfBar all{0, (int)blockDim.x};
    theta(m, A0, m > 0 ? Wup : nullptr, (T_ - 1 - m) > 0 ? Wdn : nullptr, threadIdx.x, blockDim.x);
    __syncthreads();
    bad |= chol_and_inverse<TA>(A0, B0, n, threadIdx.x, blockDim.x, all);
    if (m > 0) b_out(m - 1, B0, Wup, threadIdx.x, blockDim.x);
    if (T_ - 1 - m > 0) b_out(m + 1, B0, Wdn, threadIdx.x, blockDim.x);
    x_out(m, B0, threadIdx.x, blockDim.x);
  }
  bad = __syncthreads_or(bad);
  if (a.status && threadIdx.x == 0 && bad) atomicOr(&a.status[p], TMPC_ST_PIVOT);
}

}  // namespace tmpc
