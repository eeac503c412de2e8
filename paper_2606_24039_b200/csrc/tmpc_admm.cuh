// tmpc_admm.cuh — a4..a9: the fused ADMM iteration loop (Alg. 3), one CTA per problem,
// all `iters` iterations inside one launch, no host involvement.
//
// Work split inside a CTA:
//   * everything that is local to a stage (right-hand side eta eq. 51, v_t = Sigma_t^{-1} w_t, z~ = A x~ eq. 9,
//     relaxation eq. 10, projection eq. 12-15, dual update eq. 16) is done by ALL threads, one (stage,row) each;
//   * the two substitution chains  w_t = eta_t - Lambda_{t-1} w_{t-1}  and  x~_t = v_t - Lambda_t' x~_{t+1}
//     are sequential in t: warp 0 runs them with lane = row and warp shuffles (n <= 32), or the first ceil32(n)
//     threads with a shared-memory broadcast (n > 32).
// RESIDENT = true copies the factor (Lam, Sinv) and the constraint blocks (Am, Ap, G) into shared memory once and
// keeps them there for all iterations (configs 1, 2, 4); RESIDENT = false streams them from L2/HBM (config 3).
#pragma once
#include "tmpc_common.cuh"

namespace tmpc {

template <typename T>
struct AdmmArgs {
  Dims d;
  Params<T> prm;
  QpView<T> qp;
  const T* Lam; const T* Sinv;            // factor [B][N][n][n], [B][T][n][n]
  T* x; T* zg; T* yf; T* yg; T* xi;       // state in/out
  T* r_prim; T* r_dual; T* objective;     // info (may be null)
  int32_t* status;
  int iters, zg_given;
  int kkt_only;                           // 1: x <- S^{-1} x and return (tmpc_kkt_solve)
  const int8_t* soft_rows;                // optional [B][mg] per-row flag overriding d.soft_mask: 0 hard, 1 soft (adjoint QP, eq. 67), 2 = row switched off (resident class only)
  // f1 (adaptive step size): optional per-problem rho_bar [B] (rho_g = rho_bar, rho_f = rho_scale rho_bar) replacing
  // prm.rho_g / prm.rho_f, and an optional per-problem activity flag [B]: problems with active[p] == 0 (terminated by eq. 4) are left untouched
  const T* rho_bar; T rho_scale;
  const int32_t* active;
};

// shared-memory footprint in elements of T (host and device agree through this one function)
__host__ __device__ inline size_t admm_smem_elems(const Dims& d, bool resident) {
  const size_t nn = (size_t)d.n * d.n;
  size_t m = resident ? (size_t)d.N * nn + (size_t)d.T * nn + 2 * (size_t)d.N * d.nx * d.n + (d.g_sel ? 0 : (size_t)d.T * d.ng * d.n) : 0;
  m += 4 * (size_t)d.nz;                  // x, q, e0, e1
  m += 6 * (size_t)d.mg;                  // zg, yg, lo, hi, s, xi
  m += 3 * (size_t)d.mf;                  // yf, c, r
  m += 64;                                // reduction scratch
  return m;
}

// ---- the solve x~ = S^{-1} eta from the block LDL' factor: two sequential chains + one stage-parallel product
template <typename T, int NC>
__device__ __forceinline__ void chain_forward(const T* __restrict__ Lam, T* w, int n, int T_, int tid) {
  const int nn = n * n;
  {          // in place on w = eta:  w_t = eta_t - Lambda_{t-1} w_{t-1}
    if (n <= 32) {
      if (tid < 32) {
        const int i = tid < n ? tid : 0;
        T prev = w[i];
        for (int t = 1; t < T_; ++t) {
          const T* L = Lam + (size_t)(t - 1) * nn + i * n;
          T acc0 = w[t * n + i], acc1 = T(0);
#pragma unroll
          for (int j = 0; j < (NC ? NC : 32); j += 2) {
            if (j < n) acc0 -= L[j] * __shfl_sync(0xffffffffu, prev, j);
            if (j + 1 < n) acc1 -= L[j + 1] * __shfl_sync(0xffffffffu, prev, j + 1);
          }
          prev = acc0 + acc1;
          if (tid < n) w[t * n + i] = prev;
        }
      }
    } else {
      const int nth = ((n + 31) / 32) * 32;
      if (tid < nth) {
        for (int t = 1; t < T_; ++t) {
          if (tid < n) {
            const T* L = Lam + (size_t)(t - 1) * nn + tid * n;
            const T* wp = w + (t - 1) * n;
            T acc0 = T(0), acc1 = T(0), acc2 = T(0), acc3 = T(0);
            int j = 0;
            for (; j + 3 < n; j += 4) { acc0 += L[j] * wp[j]; acc1 += L[j + 1] * wp[j + 1]; acc2 += L[j + 2] * wp[j + 2]; acc3 += L[j + 3] * wp[j + 3]; }
            for (; j < n; ++j) acc0 += L[j] * wp[j];
            w[t * n + tid] -= (acc0 + acc1) + (acc2 + acc3);
          }
          asm volatile("bar.sync 1, %0;" ::"r"(nth) : "memory");
        }
      }
    }
  }
}
template <typename T, int NC>
__device__ __forceinline__ void chain_backward(const T* __restrict__ Lam, T* v, int n, int T_, int tid) {
  const int nn = n * n;
  {         // in place on v:  x_t = v_t - Lambda_t' x_{t+1}
    if (n <= 32) {
      if (tid < 32) {
        const int i = tid < n ? tid : 0;
        T prev = v[(T_ - 1) * n + i];
        for (int t = T_ - 2; t >= 0; --t) {
          const T* L = Lam + (size_t)t * nn + i;            // column i of Lambda_t
          T acc0 = v[t * n + i], acc1 = T(0);
#pragma unroll
          for (int j = 0; j < (NC ? NC : 32); j += 2) {
            if (j < n) acc0 -= L[j * n] * __shfl_sync(0xffffffffu, prev, j);
            if (j + 1 < n) acc1 -= L[(j + 1) * n] * __shfl_sync(0xffffffffu, prev, j + 1);
          }
          prev = acc0 + acc1;
          if (tid < n) v[t * n + i] = prev;
        }
      }
    } else {
      const int nth = ((n + 31) / 32) * 32;
      if (tid < nth) {
        for (int t = T_ - 2; t >= 0; --t) {
          if (tid < n) {
            const T* L = Lam + (size_t)t * nn + tid;
            const T* xp = v + (t + 1) * n;
            T acc0 = T(0), acc1 = T(0), acc2 = T(0), acc3 = T(0);
            int j = 0;
            for (; j + 3 < n; j += 4) { acc0 += L[j * n] * xp[j]; acc1 += L[(j + 1) * n] * xp[j + 1]; acc2 += L[(j + 2) * n] * xp[j + 2]; acc3 += L[(j + 3) * n] * xp[j + 3]; }
            for (; j < n; ++j) acc0 += L[j * n] * xp[j];
            v[t * n + tid] -= (acc0 + acc1) + (acc2 + acc3);
          }
          asm volatile("bar.sync 1, %0;" ::"r"(nth) : "memory");
        }
      }
    }
  }
}
template <typename T, int NC>
__device__ __forceinline__ void middle_apply(const T* __restrict__ Sinv, const T* w, T* v, int n, int nz, int tid, int nt) {
  const int nn = n * n;
  {      // v_t = Sigma_t^{-1} w_t
    for (int e = tid; e < nz; e += nt) {
      const int t = e / n, i = e - t * n;
      const T* S = Sinv + (size_t)t * nn + i * n;
      const T* wt = w + t * n;
      T acc0 = T(0), acc1 = T(0);
#pragma unroll
      for (int j = 0; j < (NC ? NC : 1024); j += 2) {
        if (j >= n) break;
        acc0 += S[j] * wt[j];
        if (j + 1 < n) acc1 += S[j + 1] * wt[j + 1];
      }
      v[e] = acc0 + acc1;
    }
  }
}


template <typename T, int NC, bool RESIDENT>
__global__ void __launch_bounds__(1024) admm_kernel(AdmmArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  const Dims& d = a.d;
  const int n = NC ? NC : d.n;
  const int nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nn = n * n, nz = T_ * n, mf = d.mf, mg = d.mg;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  if (a.active && !a.active[blockIdx.x]) return;        // terminated problem (f1): state stays as it is
  const T sigma = a.prm.sigma, rho_g = a.rho_bar ? a.rho_bar[blockIdx.x] : a.prm.rho_g, rho_f = a.rho_bar ? a.rho_scale * rho_g : a.prm.rho_f, alpha = a.prm.alpha;
  const T inv_rho_g = T(1) / rho_g, inv_rg = T(1) / (rho_g + a.prm.gamma), lam = a.prm.lam, gam = a.prm.gamma;

  // ---- carve shared memory
  T* ptr = sm;
  const T *Lam, *Sinv, *Am, *Ap, *G;
  {
    const T* gLam = a.Lam + (size_t)p * N * nn;
    const T* gSinv = a.Sinv + (size_t)p * T_ * nn;
    const T* gAm = a.kkt_only ? nullptr : a.qp.Am + (size_t)p * N * nx * n;
    const T* gAp = a.kkt_only ? nullptr : a.qp.Ap + (size_t)p * N * nx * n;
    const T* gG = (a.kkt_only || d.g_sel) ? nullptr : a.qp.G + a.qp.sG * p;
    if (RESIDENT) {
      T* sLam = ptr; ptr += (size_t)N * nn;
      T* sSinv = ptr; ptr += (size_t)T_ * nn;
      T* sAm = ptr; ptr += (size_t)N * nx * n;
      T* sAp = ptr; ptr += (size_t)N * nx * n;
      T* sG = ptr; if (!d.g_sel) ptr += (size_t)T_ * ng * n;
      for (int e = tid; e < N * nn; e += nt) sLam[e] = gLam[e];
      for (int e = tid; e < T_ * nn; e += nt) sSinv[e] = gSinv[e];
      if (gAm) for (int e = tid; e < N * nx * n; e += nt) { sAm[e] = gAm[e]; sAp[e] = gAp[e]; }
      if (gG) for (int e = tid; e < T_ * ng * n; e += nt) sG[e] = gG[e];
      Lam = sLam; Sinv = sSinv; Am = sAm; Ap = sAp; G = sG;
    } else { Lam = gLam; Sinv = gSinv; Am = gAm; Ap = gAp; G = gG; }
  }
  T* x = ptr; ptr += nz;
  T* q = ptr; ptr += nz;
  T* e0 = ptr; ptr += nz;
  T* e1 = ptr; ptr += nz;
  T* zg = ptr; ptr += mg;
  T* yg = ptr; ptr += mg;
  T* lo = ptr; ptr += mg;
  T* hi = ptr; ptr += mg;
  T* sv = ptr; ptr += mg;
  T* xi = ptr; ptr += mg;
  T* yf = ptr; ptr += mf;
  T* cv = ptr; ptr += mf;
  T* rv = ptr; ptr += mf;
  T* red = ptr;

  // ---- tmpc_kkt_solve: x <- S^{-1} x
  if (a.kkt_only) {
    for (int e = tid; e < nz; e += nt) e0[e] = a.x[(size_t)p * nz + e];
    __syncthreads();
    chain_forward<T, NC>(Lam, e0, n, T_, tid); __syncthreads();
    middle_apply<T, NC>(Sinv, e0, e1, n, nz, tid, nt); __syncthreads();
    chain_backward<T, NC>(Lam, e1, n, T_, tid); __syncthreads();
    for (int e = tid; e < nz; e += nt) a.xi[(size_t)p * nz + e] = e1[e];
    return;
  }

  // ---- load vectors
  for (int e = tid; e < nz; e += nt) { x[e] = a.x[(size_t)p * nz + e]; q[e] = a.qp.q[(size_t)p * nz + e]; }
  for (int e = tid; e < mg; e += nt) {
    lo[e] = a.qp.lo[(size_t)p * mg + e]; hi[e] = a.qp.hi[(size_t)p * mg + e]; yg[e] = a.yg[(size_t)p * mg + e];
    if (a.zg_given) { zg[e] = a.zg[(size_t)p * mg + e]; xi[e] = a.xi[(size_t)p * mg + e]; } else xi[e] = T(0);
  }
  for (int e = tid; e < mf; e += nt) {
    yf[e] = a.yf[(size_t)p * mf + e];
    cv[e] = e < nx ? a.qp.x_init[(size_t)p * nx + e] : a.qp.b[(size_t)p * N * nx + (e - nx)];
  }
  __syncthreads();

  auto g_row_dot = [&](int t, int r, const T* vec) -> T {      // (G_t vec_t)[r]
    if (d.g_sel) return vec[t * n + d.g_col[r]];
    const T* g = G + ((size_t)t * ng + r) * n; const T* vt = vec + t * n;
    T s = T(0);
    for (int j = 0; j < n; ++j) s += g[j] * vt[j];
    return s;
  };
  if (!a.zg_given) {                          // z_g^0 = clip(G x^0, lo, hi)
    for (int e = tid; e < mg; e += nt) { const int t = e / ng, r = e - t * ng; zg[e] = tmin(tmax(g_row_dot(t, r, x), lo[e]), hi[e]); }
  }
  for (int e = tid; e < mf; e += nt) rv[e] = rho_f * cv[e] - yf[e];
  __syncthreads();
  for (int e = tid; e < mg; e += nt) sv[e] = rho_g * zg[e] - yg[e];
  __syncthreads();

  const int8_t* srow = a.soft_rows ? a.soft_rows + (size_t)p * mg : nullptr;
  for (int it = 0; it < a.iters; ++it) {
    // a4: eta = sigma x - q + C'(rho_f c - y_f) + G'(rho_g z_g - y_g)                                   (eq. 51)
    for (int e = tid; e < nz; e += nt) {
      const int t = e / n, i = e - t * n;
      T s = sigma * x[e] - q[e];
      if (t == 0 && i < nx) s += rv[i];
      if (t < N) { const T* A_ = Am + (size_t)t * nx * n + i; const T* r = rv + nx + t * nx; for (int k = 0; k < nx; ++k) s += A_[k * n] * r[k]; }
      if (t > 0) { const T* A_ = Ap + (size_t)(t - 1) * nx * n + i; const T* r = rv + nx + (t - 1) * nx; for (int k = 0; k < nx; ++k) s += A_[k * n] * r[k]; }
      if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) s += sv[t * ng + r]; }
      else { const T* g = G + (size_t)t * ng * n + i; for (int r = 0; r < ng; ++r) s += g[r * n] * sv[t * ng + r]; }
      e0[e] = s;
    }
    __syncthreads();
    // a5, middle, a6: x~ = S^{-1} eta                                                                    (eq. 8)
    chain_forward<T, NC>(Lam, e0, n, T_, tid); __syncthreads();
    middle_apply<T, NC>(Sinv, e0, e1, n, nz, tid, nt); __syncthreads();
    chain_backward<T, NC>(Lam, e1, n, T_, tid); __syncthreads();
    // a7 + a8: z~ = A x~ (eq. 9), relaxation (eq. 10), projection (eq. 12-15), duals (eq. 16 / 44-45)
    for (int e = tid; e < mf; e += nt) {
      T ztf;
      if (e < nx) ztf = e1[e];
      else {
        const int t = (e - nx) / nx, i = (e - nx) - t * nx;
        const T* am = Am + ((size_t)t * nx + i) * n; const T* ap = Ap + ((size_t)t * nx + i) * n;
        const T* xa = e1 + t * n; const T* xb = xa + n;
        T s0 = T(0), s1 = T(0);
        for (int j = 0; j < n; ++j) { s0 += am[j] * xa[j]; s1 += ap[j] * xb[j]; }
        ztf = s0 + s1;
      }
      const T y = yf[e] + rho_f * alpha * (ztf - cv[e]);
      yf[e] = y; rv[e] = rho_f * cv[e] - y;
    }
    for (int e = tid; e < mg; e += nt) {
      const int t = e / ng, r = e - t * ng;
      const T ztg = g_row_dot(t, r, e1);
      const T zh = alpha * ztg + (T(1) - alpha) * zg[e];
      const T v = zh + yg[e] * inv_rho_g;
      T z, s;
      project_row<T>(srow ? (srow[e] != 0) : (((d.soft_mask >> r) & 1u) != 0), v, lo[e], hi[e], rho_g, inv_rg, lam, z, s);
      const T y = yg[e] + rho_g * (zh - z);
      zg[e] = z; xi[e] = s; yg[e] = y; sv[e] = rho_g * z - y;
    }
    for (int e = tid; e < nz; e += nt) x[e] = alpha * e1[e] + (T(1) - alpha) * x[e];
    __syncthreads();
  }

  // ---- write back the state
  for (int e = tid; e < nz; e += nt) a.x[(size_t)p * nz + e] = x[e];
  for (int e = tid; e < mg; e += nt) { a.zg[(size_t)p * mg + e] = zg[e]; a.yg[(size_t)p * mg + e] = yg[e]; a.xi[(size_t)p * mg + e] = xi[e]; }
  for (int e = tid; e < mf; e += nt) a.yf[(size_t)p * mf + e] = yf[e];

  // ---- a9: residuals (eq. 3) and objective at the last iterate
  if (a.r_prim || a.r_dual || a.objective || a.status) {
    const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p;
    T rp = T(0), rd = T(0), ob = T(0); int bad = 0;
    for (int e = tid; e < mf; e += nt) {
      T cx;
      if (e < nx) cx = x[e];
      else {
        const int t = (e - nx) / nx, i = (e - nx) - t * nx;
        const T* am = Am + ((size_t)t * nx + i) * n; const T* ap = Ap + ((size_t)t * nx + i) * n;
        T s = T(0);
        for (int j = 0; j < n; ++j) s += am[j] * x[t * n + j] + ap[j] * x[(t + 1) * n + j];
        cx = s;
      }
      rp = tmax(rp, tabs(cx - cv[e]));
    }
    for (int e = tid; e < mg; e += nt) {
      const int t = e / ng, r = e - t * ng;
      rp = tmax(rp, tabs(g_row_dot(t, r, x) - zg[e]));
      if (((d.soft_mask >> r) & 1u) && xi[e] != T(0)) {
        const T sg = xi[e] > T(0) ? T(1) : T(-1);
        rd = tmax(rd, tabs(gam * xi[e] + lam * sg + yg[e]));
        ob += lam * tabs(xi[e]) + T(0.5) * gam * xi[e] * xi[e];
      }
    }
    for (int e = tid; e < nz; e += nt) {
      const int t = e / n, i = e - t * n;
      T px = T(0);
      const T* Dt = Dp + (size_t)t * nn + i * n;
      for (int j = 0; j < n; ++j) px += Dt[j] * x[t * n + j];
      if (t > 0) { const T* Et = Ep + (size_t)(t - 1) * nn + i * n; for (int j = 0; j < n; ++j) px += Et[j] * x[(t - 1) * n + j]; }
      if (t < N) { const T* Et = Ep + (size_t)t * nn + i; for (int j = 0; j < n; ++j) px += Et[j * n] * x[(t + 1) * n + j]; }
      T g = px + q[e];                                   // + C'y_f + G'y_g
      if (t == 0 && i < nx) g += yf[i];
      if (t < N) { const T* A_ = Am + (size_t)t * nx * n + i; for (int k = 0; k < nx; ++k) g += A_[k * n] * yf[nx + t * nx + k]; }
      if (t > 0) { const T* A_ = Ap + (size_t)(t - 1) * nx * n + i; for (int k = 0; k < nx; ++k) g += A_[k * n] * yf[nx + (t - 1) * nx + k]; }
      if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) g += yg[t * ng + r]; }
      else { const T* gg = G + (size_t)t * ng * n + i; for (int r = 0; r < ng; ++r) g += gg[r * n] * yg[t * ng + r]; }
      rd = tmax(rd, tabs(g));
      ob += T(0.5) * x[e] * px + q[e] * x[e];
      if (!isfinite(x[e])) bad = 1;
    }
    rp = block_max(rp, red); rd = block_max(rd, red); ob = block_sum(ob, red);
    bad = __syncthreads_or(bad);
    if (tid == 0) {
      if (a.r_prim) a.r_prim[p] = rp;
      if (a.r_dual) a.r_dual[p] = rd;
      if (a.objective) a.objective[p] = ob;
      if (a.status && bad) atomicOr(&a.status[p], TMPC_ST_NAN);
    }
  }
}

}  // namespace tmpc
