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
  int32_t* status;              // [B], written: TMPC_ST_PIVOT or 0 (may be null)
  // f1 (adaptive step size): optional per-problem rho_bar [B] (w_in = rho_bar, w_eq = rho_scale rho_bar) and an optional refactor
  // mask [B]: problems with mask[p] == 0 keep their factor
  const T* rho_bar; double rho_scale;
  const int32_t* mask;
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
  if (a.mask && !a.mask[p]) return;
  const double w_in = a.rho_bar ? (double)a.rho_bar[p] : a.w_in, w_eq = a.rho_bar ? a.rho_scale * w_in : a.w_eq;
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
      s += (TA)w_eq * acc;
      if (d.g_sel) {
        for (int r = 0; r < ng; ++r) if (d.g_col[r] == i && i == j) s += wr ? (TA)wr[t * ng + r] : (TA)w_in;
      } else {
        for (int r = 0; r < ng; ++r) s += (wr ? (TA)wr[t * ng + r] : (TA)w_in) * (TA)Gt[r * n + i] * (TA)Gt[r * n + j];
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
        A[e] = (TA)Et[e] + (TA)w_eq * acc;
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
  if (a.status && tid == 0) a.status[p] = bad ? TMPC_ST_PIVOT : 0;
}

}  // namespace tmpc
