// tmpc_backward.cuh — a10: active-set VJP (Alg. 2; App. E).
//
//  bwd_prepare_kernel : classify each inequality row (reading A-16) into
//                       0 inactive / 1 hard-active / 2 soft-active, and build
//                         rhs_x = dL/dx - G_s' dL/dxi_s      (eq. 65 right-hand side in the signed slack xi = S xi_A of eq. 54)
//                       plus, per mode: adjoint row weights (REFINE) or the adjoint QP's data (REUSE, eq. 67).
//  bwd_refine_kernel  : iterative refinement of the active-set KKT system (eq. 62 / 65)
//                         [H A_a'; A_a 0][e_x; e_y] = [rhs_x; 0],  H = P + gamma G_s'G_s,  A_a = [C; G_h],
//                       with the regularised operator applied through the block-tridiagonal factor of
//                         S_adj = H + sigma I + rho_adj A_a'A_a :   dx = S_adj^{-1}(r1 + rho_adj A_a' r2),  dy = rho_adj (A_a dx - r2).
//                       dL/dq = -e_x, dL/dx_init = +e_f[0:nx]   (eq. 59 with dF/dq = [I;0;0], dF/dx_init = -I on the init rows).
#pragma once
#include "tmpc_common.cuh"
#include "tmpc_admm.cuh"

namespace tmpc {

template <typename T>
struct BwdArgs {
  Dims d;
  QpView<T> qp;
  const T* x; const T* yg; const T* xi;     // forward solution
  const T* dLdx; const T* dLdxi;            // upstream gradients (dLdxi may be null)
  T eps_abs, eps_rel, gamma, rho_adj, sigma;
  int8_t* cls;                              // [B][mg] out
  T* rhs;                                   // [B][nz] out: rhs_x
  T* w_rows;                                // [B][mg] out (REFINE): row weights for the adjoint factor
  T* lo_adj; T* hi_adj; int8_t* soft_adj;   // [B][mg] out (REUSE): bounds and soft flags of the adjoint QP
  T* q_adj;                                 // [B][nz] out (REUSE): -rhs_x
  int refine_codes;                         // 1: soft_adj holds the row codes of the resident-class refinement (see bwd_prepare_kernel)
  // refine
  const T* Lam; const T* Sinv;
  int sweeps;
  T* dq; T* dxinit;
};

template <typename T>
__device__ __forceinline__ T g_dot(const Dims& d, const T* G, int t, int r, const T* vec) {
  if (d.g_sel) return vec[t * d.n + d.g_col[r]];
  const T* g = G + ((size_t)t * d.ng + r) * d.n; const T* vt = vec + t * d.n;
  T s = T(0);
  for (int j = 0; j < d.n; ++j) s += g[j] * vt[j];
  return s;
}

template <typename T>
__global__ void bwd_prepare_kernel(BwdArgs<T> a) {
  __shared__ T red[64];
  const Dims& d = a.d;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x, n = d.n, ng = d.ng, mg = d.mg, nz = d.nz;
  const T* x = a.x + (size_t)p * nz; const T* yg = a.yg + (size_t)p * mg; const T* xi = a.xi + (size_t)p * mg;
  const T* lo = a.qp.lo + (size_t)p * mg; const T* hi = a.qp.hi + (size_t)p * mg;
  const T* G = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  T ym = T(0);
  for (int e = tid; e < mg; e += nt) ym = tmax(ym, tabs(yg[e]));
  ym = block_max(ym, red);
  const T eps_y = a.eps_abs + a.eps_rel * ym;
  int8_t* cls = a.cls + (size_t)p * mg;
  for (int e = tid; e < mg; e += nt) {
    const int t = e / ng, r = e - t * ng;
    const bool soft = (d.soft_mask >> r) & 1u;
    int c = 0;
    if (soft && tabs(xi[e]) > a.eps_abs) c = 2;
    else if (tabs(yg[e]) > eps_y) c = 1;
    else {
      const T gx = g_dot(d, G, t, r, x);
      const bool nl = isfinite(lo[e]) && (gx - lo[e] <= a.eps_abs + a.eps_rel * tabs(lo[e]));
      const bool nh = isfinite(hi[e]) && (hi[e] - gx <= a.eps_abs + a.eps_rel * tabs(hi[e]));
      if (nl || nh) c = 1;
    }
    cls[e] = (int8_t)c;
    if (a.w_rows) a.w_rows[(size_t)p * mg + e] = c == 1 ? a.rho_adj : (c == 2 ? a.gamma : T(0));
    if (a.lo_adj) {
      a.lo_adj[(size_t)p * mg + e] = c ? T(0) : -INFINITY; a.hi_adj[(size_t)p * mg + e] = c ? T(0) : INFINITY;
      // eq. 67 mode: soft-active rows are soft rows of the adjoint QP.  Refinement on the resident class (refine_codes): only the hard-active
      // rows are constraint rows; soft-active rows enter through the factor (weight gamma), inactive rows not at all -> both switched off (2)
      a.soft_adj[(size_t)p * mg + e] = a.refine_codes ? (int8_t)(c == 1 ? 0 : 2) : (int8_t)(c == 2);
    }
  }
  __syncthreads();
  for (int e = tid; e < nz; e += nt) {
    const int t = e / n, i = e - t * n;
    T s = a.dLdx[(size_t)p * nz + e];
    if (a.dLdxi) {
      for (int r = 0; r < ng; ++r) {
        const int row = t * ng + r;
        if (cls[row] != 2) continue;
        const T gi = d.g_sel ? (d.g_col[r] == i ? T(1) : T(0)) : G[((size_t)t * ng + r) * n + i];
        s -= gi * a.dLdxi[(size_t)p * mg + row];     // dL/dxi is w.r.t. the signed slack this library returns: no sign factor (tmpc.h)
      }
    }
    a.rhs[(size_t)p * nz + e] = s;
    if (a.q_adj) a.q_adj[(size_t)p * nz + e] = -s;
  }
}

// dynamic shared memory: e_x, dx(t0), t1, r1 [nz] ; e_f, r2f [mf] ; e_h, r2h [mg]
template <typename T, int NC>
__global__ void __launch_bounds__(1024) bwd_refine_kernel(BwdArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  const Dims& d = a.d;
  const int n = NC ? NC : d.n, nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nn = n * n, nz = d.nz, mf = d.mf, mg = d.mg;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  T* ex = sm; T* t0 = ex + nz; T* t1 = t0 + nz; T* ef = t1 + nz; T* r2f = ef + mf; T* eh = r2f + mf; T* r2h = eh + mg;
  const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Am = a.qp.Am + (size_t)p * N * nx * n; const T* Ap = a.qp.Ap + (size_t)p * N * nx * n;
  const T* G = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  const T* Lam = a.Lam + (size_t)p * N * nn; const T* Sinv = a.Sinv + (size_t)p * T_ * nn;
  const int8_t* cls = a.cls + (size_t)p * mg;
  const T* rhs = a.rhs + (size_t)p * nz;
  const T rho = a.rho_adj, gam = a.gamma;
  for (int e = tid; e < nz; e += nt) ex[e] = T(0);
  for (int e = tid; e < mf; e += nt) ef[e] = T(0);
  for (int e = tid; e < mg; e += nt) eh[e] = T(0);
  __syncthreads();
  auto c_row = [&](int e, const T* v) -> T {       // (C v)[e]
    if (e < nx) return v[e];
    const int t = (e - nx) / nx, i = (e - nx) - t * nx;
    const T* am = Am + ((size_t)t * nx + i) * n; const T* ap = Ap + ((size_t)t * nx + i) * n;
    T s = T(0);
    for (int j = 0; j < n; ++j) s += am[j] * v[t * n + j] + ap[j] * v[(t + 1) * n + j];
    return s;
  };
  for (int sw = 0; sw < a.sweeps; ++sw) {
    // r2 = -A_a e_x ; also the soft-active products gamma (G_s e_x) kept in r2h for the H term
    for (int e = tid; e < mf; e += nt) r2f[e] = -c_row(e, ex);
    for (int e = tid; e < mg; e += nt) { const int t = e / ng, r = e - t * ng; r2h[e] = cls[e] ? -g_dot(d, G, t, r, ex) : T(0); }
    __syncthreads();
    // t0 = r1 + rho A_a' r2,  r1 = rhs - (P e_x + gamma G_s'G_s e_x + C' e_f + G_h' e_h)
    for (int e = tid; e < nz; e += nt) {
      const int t = e / n, i = e - t * n;
      T px = T(0);
      const T* Dt = Dp + (size_t)t * nn + i * n;
      for (int j = 0; j < n; ++j) px += Dt[j] * ex[t * n + j];
      if (t > 0) { const T* Et = Ep + (size_t)(t - 1) * nn + i * n; for (int j = 0; j < n; ++j) px += Et[j] * ex[(t - 1) * n + j]; }
      if (t < N) { const T* Et = Ep + (size_t)t * nn + i; for (int j = 0; j < n; ++j) px += Et[j * n] * ex[(t + 1) * n + j]; }
      T s = rhs[e] - px;
      // C' (rho r2f - e_f)
      if (t == 0 && i < nx) s += rho * r2f[i] - ef[i];
      if (t < N) { const T* A_ = Am + (size_t)t * nx * n + i; for (int k = 0; k < nx; ++k) { const int row = nx + t * nx + k; s += A_[k * n] * (rho * r2f[row] - ef[row]); } }
      if (t > 0) { const T* A_ = Ap + (size_t)(t - 1) * nx * n + i; for (int k = 0; k < nx; ++k) { const int row = nx + (t - 1) * nx + k; s += A_[k * n] * (rho * r2f[row] - ef[row]); } }
      for (int r = 0; r < ng; ++r) {
        const int row = t * ng + r; const int c = cls[row];
        if (!c) continue;
        const T gi = d.g_sel ? (d.g_col[r] == i ? T(1) : T(0)) : G[((size_t)t * ng + r) * n + i];
        if (gi == T(0)) continue;
        // hard-active: G_h'(rho r2h - e_h);  soft-active: -gamma G_s'(G_s e_x) = +gamma G_s' r2h
        s += gi * (c == 1 ? (rho * r2h[row] - eh[row]) : gam * r2h[row]);
      }
      t0[e] = s;
    }
    __syncthreads();
    chain_forward<T, NC>(Lam, t0, n, T_, tid); __syncthreads();
    middle_apply<T, NC>(Sinv, t0, t1, n, nz, tid, nt); __syncthreads();
    chain_backward<T, NC>(Lam, t1, n, T_, tid); __syncthreads();
    // e_y += rho (A_a dx - r2) ; e_x += dx
    for (int e = tid; e < mf; e += nt) ef[e] += rho * (c_row(e, t1) - r2f[e]);
    for (int e = tid; e < mg; e += nt) if (cls[e] == 1) { const int t = e / ng, r = e - t * ng; eh[e] += rho * (g_dot(d, G, t, r, t1) - r2h[e]); }
    __syncthreads();
    for (int e = tid; e < nz; e += nt) ex[e] += t1[e];
    __syncthreads();
  }
  for (int e = tid; e < nz; e += nt) a.dq[(size_t)p * nz + e] = -ex[e];
  for (int e = tid; e < nx; e += nt) a.dxinit[(size_t)p * nx + e] = ef[e];
}

// eq. 66 in the signed slack: dL/dgamma_xi = sum over the soft-active rows of xi_i (G eta_x)_i with eta_x = -dL/dq;
// one CTA per problem, fixed summation order.
template <typename T>
__global__ void __launch_bounds__(256) bwd_dgamma_kernel(Dims d, QpView<T> qp, const int8_t* __restrict__ cls, const T* __restrict__ xi, const T* __restrict__ dq, T* __restrict__ out) {
  __shared__ T red[64];
  const int p = blockIdx.x, ng = d.ng, mg = d.mg, nz = d.nz;
  const T* G = qp.G ? qp.G + qp.sG * p : nullptr;
  T s = T(0);
  for (int e = threadIdx.x; e < mg; e += blockDim.x) {
    if (cls[(size_t)p * mg + e] != 2) continue;
    s -= xi[(size_t)p * mg + e] * g_dot(d, G, e / ng, e % ng, dq + (size_t)p * nz);
  }
  s = block_sum(s, red);
  if (threadIdx.x == 0) out[p] = s;
}

// REUSE mode epilogue: dq = -x_adj, dxinit = +yf_adj[0:nx]
template <typename T>
__global__ void bwd_reuse_finish_kernel(int B, int nz, int nx, int mf, const T* xa, const T* yfa, T* dq, T* dxinit) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid < (long long)B * nz) dq[gid] = -xa[gid];
  if (gid < (long long)B * nx) { const int p = (int)(gid / nx), i = (int)(gid - (long long)p * nx); dxinit[gid] = yfa[(size_t)p * mf + i]; }
}

}  // namespace tmpc
