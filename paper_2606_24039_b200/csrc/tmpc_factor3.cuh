// tmpc_factor3.cuh — a2 + a3 for the STREAMED class (n ~ 88): the one-directional block LDL' of factor_kernel
// (same outputs: Lam_t = Phi_t Sigma_t^{-1}, Sinv_t = Sigma_t^{-1}), restructured as register-tiled shared-memory
// matrix products.  factor_kernel spends its time on dependent global loads and two shared loads per FMA; here every
// product has the form  out(i,j) = sum_k A[k][i] B[k][j]  and runs on the FP64 tensor cores (DMMA m8n8k4: the A fragment
// of a lane is A[k + lane%4][i0 + lane/4], 8 contiguous doubles per k-row, two wavefronts per fragment load for ld = 88):
// 16 warps in a 4 x 4 grid, each owning up to 3 x 3 tiles of 8 x 8 (6 fragment loads per 9 DMMA; the 4 x 4 DFMA register
// tile it replaces needed 4 vector loads per 16 DFMA and was shared-memory bound).  Operands are staged in shared
// memory, and three n x n buffers suffice:
//   P: Sigma_t -> L (in-place Cholesky) -> Sigma_t^{-1} -> (next stage) Sigma_{t+1}
//   Q: X = L^{-1} -> Phi_t' (transposed)
//   R: Lambda_t' (transposed)
// with  Sigma^{-1} = X'X,  Lambda = Phi Sigma^{-1}  (out(j... ) from Q = Phi', P),  Sigma_{t+1} = Theta_{t+1} - Lambda Phi'
// (from R = Lambda', Q = Phi').  Arithmetic in double for both working dtypes.  One CTA per problem.
#pragma once
#include "tmpc_factor.cuh"

#include <type_traits>

namespace tmpc {

// fused Cholesky / inverse of factor3_kernel: 16 warps x F3_RMAX rows, 32 lanes x F3_CMAX chunks cover n <= 96; scratch buffer
// = colk[96], rowk[96], d_k (+ pad) doubles
constexpr int F3_RMAX = 6, F3_CMAX = 3, F3_SB = 2 * 96 + 2;
template <int V> using f3_ic = std::integral_constant<int, V>;
__device__ __forceinline__ double f3_lds(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ void f3_sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }

__device__ __forceinline__ void f3_cp16(unsigned dst, const void* src) { asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory"); }
__device__ __forceinline__ void f3_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void f3_cp_wait() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
template <typename T> __host__ __device__ constexpr int f3_ch() { return sizeof(T) == 4 ? 32 : 16; }   // rows of A^-/A^+/G staged per chunk (in the working dtype)

__host__ __device__ inline int f3_ld(int n) { return (n + 7) / 8 * 8; }
// D (8 x 8) += A (8 x 4, row) B (4 x 8, col): lane holds A[lane/4][lane%4], B[lane%4][lane/4], D[lane/4][2 (lane%4) + {0,1}]
__device__ __forceinline__ void f3_dmma(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
template <typename T> __host__ inline size_t factor3_smem(int n) { const int ld = f3_ld(n); return (size_t)3 * ld * ld * sizeof(double) + (size_t)2 * f3_ch<T>() * ld * sizeof(T) + 64; }

template <typename T>
__global__ void __launch_bounds__(512) factor3_kernel(FactorArgs<T> a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Dims& d = a.d;
  const int n = d.n, nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nn = n * n, ld = f3_ld(n), nt8 = ld / 8, n4 = (n + 3) & ~3;
  double* P = reinterpret_cast<double*>(smem_raw);
  double* Q = P + (size_t)ld * ld;
  double* R = Q + (size_t)ld * ld;
  constexpr int F3_CH = f3_ch<T>();
  T* S1 = reinterpret_cast<T*>(R + (size_t)ld * ld);              // staged chunk, [F3_CH][ld], working dtype (exact copy)
  T* S2 = S1 + (size_t)F3_CH * ld;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  if (a.mask && !a.mask[p]) return;
  const double w_in = a.rho_bar ? (double)a.rho_bar[p] : a.w_in, w_eq = a.rho_bar ? a.rho_scale * w_in : a.w_eq;
  const T* Dp = a.qp.D + a.qp.sD * p;
  const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Amp = a.qp.Am + (size_t)p * N * nx * n;
  const T* App = a.qp.Ap + (size_t)p * N * nx * n;
  const T* Gp = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  const T* wrow = a.w_rows ? a.w_rows + (size_t)p * T_ * ng : nullptr;
  T* Lamp = a.Lam + (size_t)p * N * nn;
  T* Sinvp = a.Sinv + (size_t)p * T_ * nn;
  int bad = 0;
  for (int e = tid; e < 3 * ld * ld; e += nt) P[e] = 0.0;          // pads stay zero
  __syncthreads();

  // stage rows [r0, r0+rows) of a row-major [*][n] global matrix into S (float), zero padded; optional per-row scale
  auto stage = [&](T* S, const T* src, int r0, int rows, const T* scale, double scale_all) {
    for (int e = tid; e < F3_CH * ld; e += nt) {
      const int r = e / ld, c = e - r * ld;
      T v = T(0);
      if (r < rows && c < n && src) { double x = (double)src[(size_t)(r0 + r) * n + c]; if (scale) x *= (double)scale[r0 + r]; v = (T)(x * scale_all); }
      S[e] = v;
    }
  };
  // asynchronous staging (LDGSTS, 16 bytes per copy, L2 only) of rows [r0, r0+rows) when a chunk is contiguous and aligned in
  // global AND shared memory (ld == n, 16-byte rows): the copies of the next chunk are in flight while the tensor cores work
  // on the current product; without it every chunk exposes a chain of dependent global-load latencies (measured: the staged
  // phases took 3-5x their DMMA time).  The tail rows of the chunk are zeroed.  Other shapes keep the synchronous path.
  constexpr int VE = 16 / (int)sizeof(T);
  const bool fast = ld == n && ((uintptr_t)Amp % 16 == 0) && ((uintptr_t)App % 16 == 0) && (((size_t)nx * n * sizeof(T)) % 16 == 0);
  auto stage_async = [&](T* S, const T* src, int r0, int rows) {
    const int nvec = rows * ld / VE, tot = F3_CH * ld / VE;
    const unsigned s0 = (unsigned)__cvta_generic_to_shared(S);
    const T* g0 = src + (size_t)r0 * n;
    for (int v = tid; v < tot; v += nt) {
      if (v < nvec) f3_cp16(s0 + 16u * v, g0 + (size_t)v * VE);
      else *reinterpret_cast<float4*>(reinterpret_cast<unsigned char*>(S) + 16 * (size_t)v) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  };
  auto clampr = [&](int r) { return r < 0 ? 0 : (r > F3_CH ? F3_CH : r); };

  // acc(i,j) += sum_k A[k][i] B[k][j], k in [k0, k1) (multiples of 4; pad rows are zero): warp (wr, wc) owns the 8 x 8 tiles
  // (3 wr + x, 3 wc + y); TRI skips the k-steps above the diagonal block of a tile (X lower triangular in X'X)
  const int lane = tid & 31, wid = tid >> 5, wr = wid >> 2, wc = wid & 3, lq = lane >> 2, lr = lane & 3;
  bool va[3], vb[3];
#pragma unroll
  for (int x = 0; x < 3; ++x) { va[x] = 3 * wr + x < nt8; vb[x] = 3 * wc + x < nt8; }
  auto mm = [&](double (&acc)[3][3][2], const auto* A, const auto* B, int k0, int k1, auto TRIc) {
    constexpr bool TRI = decltype(TRIc)::value != 0;
    for (int k = k0; k < k1; k += 4) {
      const auto* Ar = A + (size_t)(k + lr) * ld + 24 * wr + lq;
      const auto* Br = B + (size_t)(k + lr) * ld + 24 * wc + lq;
      double af[3], bf[3];
#pragma unroll
      for (int x = 0; x < 3; ++x) { af[x] = va[x] ? (double)Ar[8 * x] : 0.0; bf[x] = vb[x] ? (double)Br[8 * x] : 0.0; }
#pragma unroll
      for (int x = 0; x < 3; ++x)
#pragma unroll
        for (int y = 0; y < 3; ++y) {
          const int tmax = 3 * wr + x > 3 * wc + y ? 3 * wr + x : 3 * wc + y;
          if (va[x] && vb[y] && (!TRI || k >= 8 * tmax)) f3_dmma(acc[x][y], af[x], bf[y]);
        }
    }
  };
  // visit this lane's accumulator elements: fn(v, gi, gj), v = acc[x][y][e], (gi, gj) = (row, column) in the padded block
  auto for_acc = [&](double (&acc)[3][3][2], auto fn) {
#pragma unroll
    for (int x = 0; x < 3; ++x)
#pragma unroll
      for (int y = 0; y < 3; ++y)
        if (va[x] && vb[y]) {
#pragma unroll
          for (int e = 0; e < 2; ++e) fn(acc[x][y][e], 8 * (3 * wr + x) + lq, 8 * (3 * wc + y) + 2 * lr + e);
        }
  };

#ifdef TMPC_F3_PROF
  long long tk[8] = {}, tc = clock64();
#define F3_TICK(i) { long long c_ = clock64(); tk[i] += c_ - tc; tc = c_; }
#else
#define F3_TICK(i)
#endif
  for (int t = 0; t < T_; ++t) {
    // ---- P <- Theta_t - Lambda_{t-1} Phi_{t-1}'   (R = Lambda', Q = Phi' of the previous stage)
    {
      double acc[3][3][2] = {}, accA[3][3][2] = {};   // acc = G' w G - Lambda Phi' ; accA = A^-' A^- + A^+' A^+
      const int nps = (nx + 2 * F3_CH - 1) / (2 * F3_CH);
      auto pair_src = [&](int q_, int& r0) -> const T* {
        const int which = q_ / nps; r0 = (q_ - which * nps) * 2 * F3_CH;
        return which == 0 ? (t < N ? Amp + (size_t)t * nx * n : nullptr) : (t > 0 ? App + (size_t)(t - 1) * nx * n : nullptr);
      };
      auto next_valid = [&](int q_) { int r0; while (q_ < 2 * nps && !pair_src(q_, r0)) ++q_; return q_; };
      auto issue_pair = [&](int q_) {
        int r0; const T* src = pair_src(q_, r0);
        stage_async(S1, src, r0, clampr(nx - r0));
        if (nx - r0 - F3_CH > 0) stage_async(S2, src, r0 + F3_CH, clampr(nx - r0 - F3_CH));
        f3_cp_commit();
      };
      int q = next_valid(0);
      if (fast && q < 2 * nps) issue_pair(q);          // S1, S2 are idle since the barrier that ended the previous phase
      if (t > 0) {
        mm(acc, R, Q, 0, n4, f3_ic<0>{});
        for_acc(acc, [&](double& v, int, int) { v = -v; });
      }
      // A^-_t' A^-_t  and  A^+_{t-1}' A^+_{t-1}, two chunks (S1, S2) per step; step q = (which, r0)
      while (q < 2 * nps) {
        int r0; const T* src = pair_src(q, r0);
        const int rows1 = clampr(nx - r0), rows2 = clampr(nx - r0 - F3_CH);
        if (fast) { f3_cp_wait(); __syncthreads(); }
        else {
          __syncthreads();
          stage(S1, src, r0, rows1, nullptr, 1.0);
          if (rows2 > 0) stage(S2, src, r0 + F3_CH, rows2, nullptr, 1.0);
          __syncthreads();
        }
        mm(accA, S1, S1, 0, (rows1 + 3) & ~3, f3_ic<0>{});
        if (rows2 > 0) mm(accA, S2, S2, 0, (rows2 + 3) & ~3, f3_ic<0>{});
        q = next_valid(q + 1);
        if (fast && q < 2 * nps) { __syncthreads(); issue_pair(q); }
      }
      if (!d.g_sel && Gp) for (int r0 = 0; r0 < ng; r0 += F3_CH) {   // G' diag(w) G
        const int rows = ng - r0 < F3_CH ? ng - r0 : F3_CH;
        __syncthreads();
        stage(S1, Gp + (size_t)t * ng * n, r0, rows, nullptr, 1.0);
        stage(S2, Gp + (size_t)t * ng * n, r0, rows, wrow ? wrow + (size_t)t * ng : nullptr, wrow ? 1.0 : w_in);
        __syncthreads();
        mm(acc, S1, S2, 0, (rows + 3) & ~3, f3_ic<0>{});
      }
      __syncthreads();                                 // everyone is done reading R, Q, S before P is rewritten
#pragma unroll
      for (int x = 0; x < 3; ++x)
#pragma unroll
        for (int y = 0; y < 3; ++y)
          if (va[x] && vb[y]) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const int gi = 8 * (3 * wr + x) + lq, gj = 8 * (3 * wc + y) + 2 * lr + e;
              double s = 0.0;
              if (gi < n && gj < n) {
                s = (double)Dp[(size_t)t * nn + gi * n + gj] + w_eq * accA[x][y][e] + acc[x][y][e];
                if (gi == gj) {
                  s += a.sigma;
                  if (t == 0 && gi < nx) s += w_eq;      // A_init' A_init = blkdiag(I_nx, 0)
                  if (d.g_sel) for (int r = 0; r < ng; ++r) if (d.g_col[r] == gi) s += wrow ? (double)wrow[(size_t)t * ng + r] : w_in;
                }
              } else if (gi == gj) s = 1.0;              // identity on the padding keeps the factor well defined
              P[(size_t)gi * ld + gj] = s;
            }
          }
      __syncthreads();
    }
    F3_TICK(0)
    // ---- Cholesky of P and X = L^{-1} TOGETHER, both held in registers: warp w owns rows i = w + 16 r, lane l owns columns
    // j = l + 32 c of P (symmetric, being reduced) and of Y (starts as I, becomes diag(L) X).  Step k: the owners publish
    // column k of the reduced P (u_i, zero for i <= k), row k of Y and the pivot d_k in a double-buffered scratch (ONE CTA
    // barrier per column); then every thread applies  P[i][j] -= (u_i / d_k) u_j  and  Y[i][j] -= (u_i / d_k) Y[k][j]  to its
    // own registers (l_ik l_jk = u_i u_j / d_k and l_ik / l_kk = u_i / d_k: L itself is never formed).  The columns are
    // walked in six compile-time groups of 16 (row slot r of the pivot row and the live 32-column chunks are constants
    // inside a group; the only run-time conditions are warp uniform).  At the end X[i][j] = Y[i][j] / sqrt(d_i) goes to Q.
    {
      const unsigned scr = (unsigned)__cvta_generic_to_shared(S1);   // the staging chunks are idle here (>= 8 KB)
      const unsigned a_row = scr + 8u * wid, a_col = scr + 8u * lane;  // colk[i] broadcast per warp / colk[j], rowk[j] per lane
      double pv[F3_RMAX][F3_CMAX], yv[F3_RMAX][F3_CMAX];
      for (int e = tid; e < 2 * F3_SB + 96; e += nt) f3_sts(scr + 8u * e, 0.0);       // tails (i, j >= n) stay zero
#pragma unroll
      for (int r = 0; r < F3_RMAX; ++r)
#pragma unroll
        for (int c = 0; c < F3_CMAX; ++c) {
          const int i = wid + 16 * r, j = lane + 32 * c;
          pv[r][c] = (i < n && j < n) ? P[(size_t)i * ld + j] : 0.0;
          yv[r][c] = (i == j) ? 1.0 : 0.0;
        }
      __syncthreads();
      auto step = [&](auto RKc, auto BUFc, int kk) {
        constexpr int RK = decltype(RKc)::value, BUF = decltype(BUFc)::value, KC = RK / 2;
        constexpr unsigned OC = 8u * BUF * F3_SB, OR = OC + 8u * 96, OD = OR + 8u * 96;    // colk, rowk, d_k of this buffer
        const int k = 16 * RK + kk;
        if (k >= n) return;                                                              // uniform
        if (lane == 16 * (RK & 1) + kk) {                                                 // owners of column k
#pragma unroll
          for (int r = RK; r < F3_RMAX; ++r) {
            const int i = wid + 16 * r;
            if (i < n) f3_sts(a_row + OC + 128u * r, (r > RK || wid > kk) ? pv[r][KC] : 0.0);
          }
          if (wid == kk) { f3_sts(scr + OD, pv[RK][KC]); f3_sts(scr + 8u * (2 * F3_SB + k), pv[RK][KC]); }
        }
        if (wid == kk) {                                                                  // owners of row k
#pragma unroll
          for (int c = 0; c <= KC; ++c) f3_sts(a_col + OR + 256u * c, yv[RK][c]);
        }
        __syncthreads();
        double dk = f3_lds(scr + OD);
        if (!(dk > 0) || !isfinite(dk)) { bad = 1; dk = 1; }
        const double inv = 1.0 / dk;
        double uj[F3_CMAX], yk[F3_CMAX];
#pragma unroll
        for (int c = KC; c < F3_CMAX; ++c) uj[c] = f3_lds(a_col + OC + 256u * c);
#pragma unroll
        for (int c = 0; c <= KC; ++c) yk[c] = f3_lds(a_col + OR + 256u * c);
#pragma unroll
        for (int r = RK; r < F3_RMAX; ++r) {
          if (r > RK || wid > kk) {                    // rows i > k (rows beyond n read u_i = 0)
            const double f = f3_lds(a_row + OC + 128u * r) * inv;
#pragma unroll
            for (int c = KC; c < F3_CMAX; ++c) pv[r][c] -= f * uj[c];
#pragma unroll
            for (int c = 0; c <= KC; ++c) yv[r][c] -= f * yk[c];
          }
        }
      };
      auto group = [&](auto RKc) {
        for (int kk = 0; kk < 16; kk += 2) { step(RKc, f3_ic<0>{}, kk); step(RKc, f3_ic<1>{}, kk + 1); }
      };
      group(f3_ic<0>{}); group(f3_ic<1>{}); group(f3_ic<2>{}); group(f3_ic<3>{}); group(f3_ic<4>{}); group(f3_ic<5>{});
      __syncthreads();
      if (tid < 96) { const double di = f3_lds(scr + 8u * (2 * F3_SB + tid)); f3_sts(scr + 8u * (2 * F3_SB + tid), tid < n ? 1.0 / sqrt(di > 0 ? di : 1.0) : 0.0); }
      __syncthreads();
#pragma unroll
      for (int r = 0; r < F3_RMAX; ++r) {
        const int i = wid + 16 * r;
        const double si = f3_lds(a_row + 8u * 2 * F3_SB + 128u * r);
#pragma unroll
        for (int c = 0; c < F3_CMAX; ++c) {
          const int j = lane + 32 * c;
          if (i < ld && j < ld) Q[(size_t)i * ld + j] = (i < n && j < n) ? yv[r][c] * si : 0.0;
        }
      }
      __syncthreads();
    }
    F3_TICK(2)
    // ---- P <- Sigma^{-1} = X'X  (sum over k >= max(i,j): X lower triangular), also to global
    auto issue_phi = [&](int r0) {
      stage_async(S1, Amp + (size_t)t * nx * n, r0, clampr(nx - r0));
      stage_async(S2, App + (size_t)t * nx * n, r0, clampr(nx - r0));
      f3_cp_commit();
    };
    if (fast && t < N) issue_phi(0);                     // the Cholesky scratch in S1 is dead since the barrier above
    {
      double acc[3][3][2] = {};
      mm(acc, Q, Q, 0, n4, f3_ic<1>{});
      for_acc(acc, [&](double& v, int gi, int gj) {
        P[(size_t)gi * ld + gj] = (gi < n && gj < n) ? v : 0.0;
        if (gi < n && gj < n) Sinvp[(size_t)t * nn + gi * n + gj] = (T)v;
      });
    }
    __syncthreads();
    F3_TICK(3)
    if (t == N) break;
    // ---- Q <- Phi_t' : Q[k][i] = Phi[i][k] = E_t[i][k] + w sum_r A^+_t[r][i] A^-_t[r][k]   (tile (k-block, i-block))
    {
      double acc[3][3][2] = {};
      for (int r0 = 0; r0 < nx; r0 += F3_CH) {
        const int rows = nx - r0 < F3_CH ? nx - r0 : F3_CH;
        if (fast) { f3_cp_wait(); __syncthreads(); }
        else {
          __syncthreads();
          stage(S1, Amp + (size_t)t * nx * n, r0, rows, nullptr, 1.0);
          stage(S2, App + (size_t)t * nx * n, r0, rows, nullptr, 1.0);
          __syncthreads();
        }
        mm(acc, S1, S2, 0, (rows + 3) & ~3, f3_ic<0>{});   // acc(k, i) = sum_r A^-[r][k] A^+[r][i]
        if (fast && r0 + F3_CH < nx) { __syncthreads(); issue_phi(r0 + F3_CH); }
      }
      for_acc(acc, [&](double& v, int gk, int gi) {
        Q[(size_t)gk * ld + gi] = (gk < n && gi < n) ? (double)Ep[(size_t)t * nn + gi * n + gk] + w_eq * v : 0.0;
      });
      __syncthreads();
    }
    F3_TICK(4)
    // ---- Lambda = Phi Sigma^{-1}: Lambda(i,j) = sum_k Q[k][i] P[k][j] ; R <- Lambda' , Lambda to global
    {
      double acc[3][3][2] = {};
      mm(acc, Q, P, 0, n4, f3_ic<0>{});
      for_acc(acc, [&](double& v, int gi, int gj) {
        R[(size_t)gj * ld + gi] = (gi < n && gj < n) ? v : 0.0;
        if (gi < n && gj < n) Lamp[(size_t)t * nn + gi * n + gj] = (T)v;
      });
    }
    __syncthreads();
    F3_TICK(5)
  }
#ifdef TMPC_F3_PROF
  if (tid == 0 && p == 0) printf("f3 cycles: theta %lld chol+inv %lld - %lld xtx %lld phi %lld lam %lld\n", tk[0], tk[1], tk[2], tk[3], tk[4], tk[5]);
#endif
  bad = __syncthreads_or(bad);
  if (a.status && tid == 0) a.status[p] = bad ? TMPC_ST_PIVOT : 0;
}

}  // namespace tmpc
