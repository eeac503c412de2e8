// tmpc_admm2.cuh — a4..a8 for the RESIDENT class (configs 1, 2, 4): the fused ADMM loop of Alg. 3
// on the twisted block factor of tmpc_factor.cuh, all iterations in one launch.
//
// Design:
//  * a CTA owns PG problems (1 or 2).  Factor (Lam, Sinv) and constraint blocks (Am, Ap, G) are copied into shared
//    memory once and stay there for all iterations; the per-row ADMM state (x, q, y_f, c, z_g, y_g, lo, hi, xi) lives
//    in REGISTERS of the thread that owns the row: two (problem, stage, row) items per thread, fixed for the launch.
//  * x~ = S^{-1} eta (eq. 8) runs on warp 0: lanes = (problem, direction, row), 8 lanes per slot, so the up chain and
//    the down chain of the twisted factor of up to two problems advance together; a step is one n x n mat-vec whose
//    operand vector is exchanged with width-8 shuffles, and v_t = Sigma_t^{-1} w_t is folded into the forward step
//    (same shuffled values), so a solve is 2 * (T/2) dependent steps instead of 2T + a barrier-separated pass.
//  * everything local to a stage (eta eq. 51, z~ = A x~ eq. 9, relaxation eq. 10, projection eq. 12-15, duals eq. 16)
//    is done by all threads between three CTA barriers per iteration; several CTAs per SM overlap one CTA's chain
//    phase with another's stage-parallel phase.
//  * shared-memory layout is bank-conflict free for n = 8: rows of the factor blocks are XOR-swizzled by 16-byte
//    chunks (row-wise vector loads in the forward sweep, column-wise scalar loads in the backward sweep), and the
//    down-chain blocks / second problem are skewed by 8 / 16 elements so the four slots hit distinct banks.
// Residuals (a9) are computed by residual_kernel below from the state written back to global memory.
#pragma once
#include "tmpc_common.cuh"
#include "tmpc_admm.cuh"

namespace tmpc {

// ---- vector loads of L contiguous elements (base aligned to the widest chunk that divides the row)
template <int L> __device__ __forceinline__ void ld_vec(const float* __restrict__ p, float (&r)[L]) {
  if constexpr ((L * 4) % 16 == 0) {
#pragma unroll
    for (int c = 0; c < L / 4; ++c) { const float4 v = reinterpret_cast<const float4*>(p)[c]; r[4 * c] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w; }
  } else if constexpr ((L * 4) % 8 == 0) {
#pragma unroll
    for (int c = 0; c < L / 2; ++c) { const float2 v = reinterpret_cast<const float2*>(p)[c]; r[2 * c] = v.x; r[2 * c + 1] = v.y; }
  } else {
#pragma unroll
    for (int c = 0; c < L; ++c) r[c] = p[c];
  }
}
template <int L> __device__ __forceinline__ void ld_vec(const double* __restrict__ p, double (&r)[L]) {
  if constexpr (L % 2 == 0) {
#pragma unroll
    for (int c = 0; c < L / 2; ++c) { const double2 v = reinterpret_cast<const double2*>(p)[c]; r[2 * c] = v.x; r[2 * c + 1] = v.y; }
  } else {
#pragma unroll
    for (int c = 0; c < L; ++c) r[c] = p[c];
  }
}

// ---- dot products: packed FFMA2 (two fp32 FMAs per instruction on sm_100) for float, plain FMA chains for double
template <int L> __device__ __forceinline__ float dotv(const float (&a)[L], const float (&b)[L]) {
  float2 acc = make_float2(0.f, 0.f);
#pragma unroll
  for (int j = 0; j + 1 < L; j += 2) acc = __ffma2_rn(make_float2(a[j], a[j + 1]), make_float2(b[j], b[j + 1]), acc);
  float r = acc.x + acc.y;
  if constexpr (L % 2) r += a[L - 1] * b[L - 1];
  return r;
}
template <int L> __device__ __forceinline__ double dotv(const double (&a)[L], const double (&b)[L]) {
  double acc[2] = {0.0, 0.0};
#pragma unroll
  for (int j = 0; j < L; ++j) acc[j & 1] += a[j] * b[j];
  return acc[0] + acc[1];
}

// ---- shared-memory layout.  One RECORD per stage holds everything that multiplies or belongs to the stage variable
// v_t, at compile-time offsets from the record base (so a thread needs one address register per stage it touches):
//   AM  A^-_t             [nx][n]   (zero for t = N)
//   AP  A^+_{t-1}         [nx][n]   (A_init = [I 0] for t = 0: the rows x_0 = x_init are "dynamics block -1")
//   RM  r of block t      [nx]      r = rho_f c - y_f of the rows that AM belongs to
//   RP  r of block t-1    [nx]      (r_init for t = 0); written by the owner of that row together with RM of its own stage
//   S   s_t = rho_g z_g - y_g [n slots, ng used]
//   E0  eta_t -> w_t      [n]
//   E1  v_t -> x~_t       [n]
//   LAM Lambda_t          [n][n]    twisted factor, tmpc_factor.cuh
//   SINV Sigma_t^{-1}     [n][n]
//   G   G_t               [ng][n]   only when G is not a selection
// Rows of AM, AP, LAM, SINV are XOR-swizzled by 16-byte chunks for n = 8 (conflict-free row-wise vector loads AND
// column-wise scalar loads); the record stride is padded to 8 (mod 32) words so that the four stages a warp touches
// fall into distinct banks, records of the down chain are skewed by 8 words and the second problem by 16.
template <typename T, int NC, int NX>
struct Rec {
  static constexpr int V = 16 / (int)sizeof(T);
  static constexpr int up(int v) { return (v + V - 1) / V * V; }
  static constexpr int AM = 0, AP = AM + up(NX * NC), RM = AP + up(NX * NC), RP = RM + up(NX), S = RP + up(NX), E0 = S + up(NC),
                       E1 = E0 + up(NC), LAM = E1 + up(NC), SINV = LAM + up(NC * NC), G = SINV + up(NC * NC);
  static constexpr int SKEW = NC == 8 ? 8 : 0;
};
struct Admm2Plan { int R, per_problem; };

template <typename T, int NC, int NX>
__host__ __device__ inline Admm2Plan admm2_plan(const Dims& d, int pg) {
  using RC = Rec<T, NC, NX>;
  Admm2Plan P;
  int R = RC::G + (d.g_sel ? 0 : RC::up(d.ng * NC));
  if (NC == 8) { const int mod = 128 / (int)sizeof(T), want = sizeof(T) == 4 ? 8 : 8; while (R % (sizeof(T) == 4 ? 32 : 16) != want) R += RC::V; (void)mod; }
  P.R = R;
  int pp = d.T * R + RC::SKEW;
  if (pg == 2 && NC == 8) { const int half = 64 / (int)sizeof(T); while (pp % (2 * half) != half) pp += RC::V; }
  P.per_problem = pp;
  return P;
}
template <typename T, int NC, int NX>
__host__ __device__ inline size_t admm2_smem_bytes(const Dims& d, int pg) { return (size_t)admm2_plan<T, NC, NX>(d, pg).per_problem * pg * sizeof(T); }

// XOR swizzle (in elements) of 16-byte chunks inside an 8-element row (identity for other n)
template <typename T, int NC> __device__ __forceinline__ constexpr int swz_x(int row) {
  if (NC != 8) return 0;
  return sizeof(T) == 4 ? ((row >> 2) & 1) * 4 : ((row >> 1) & 3) * 2;
}

template <typename T>
struct Admm2Args {
  AdmmArgs<T> a;
  Admm2Plan pl;                       // host-computed: read straight from the constant bank, costs no registers
  T rfa, oma, inv_rho_g, inv_rg;      // rho_f alpha, 1 - alpha, 1 / rho_g, 1 / (rho_g + gamma)
};

// item flag bits
enum : unsigned { F_VALID = 1u, F_DYN = 2u, F_INEQ = 4u, F_SOFT = 8u, F_GMASK_SH = 8, F_GCOL_SH = 16 };

template <typename T, int NC, int NX, int PG, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) admm2_kernel(const __grid_constant__ Admm2Args<T> A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  using RC = Rec<T, NC, NX>;
  const AdmmArgs<T>& a = A.a;
  const Dims& d = a.d;
  constexpr int n = NC, nx = NX, nn = NC * NC, V = RC::V;
  const int R = A.pl.R, PP = A.pl.per_problem;
  const int ng = d.ng, N = d.N, T_ = d.T, nz = T_ * n, mf = d.mf, mg = d.mg;
  const int tid = threadIdx.x, nt = blockDim.x;
  const int m = T_ / 2;
  auto rec = [&](int t) { return t * R + (t > m ? RC::SKEW : 0); };

  // ---- stage the factor and the constraint blocks of every problem of this CTA into the records
#pragma unroll 1
  for (int g = 0; g < PG; ++g) {
    const int p = blockIdx.x * PG + g;
    T* P = sm + g * PP;
    for (int e = tid; e < PP; e += nt) P[e] = T(0);
    __syncthreads();
    if (p >= d.B) continue;
    const T* gLam = a.Lam + (size_t)p * T_ * nn;
    const T* gSinv = a.Sinv + (size_t)p * T_ * nn;
    for (int e = tid; e < T_ * nn; e += nt) {
      const int t = e / nn, rc = e - t * nn, row = rc / n, col = rc - row * n;
      const int o = rec(t) + row * n + (col ^ swz_x<T, NC>(row));
      if (t != m) P[o + RC::LAM] = gLam[e];
      P[o + RC::SINV] = gSinv[e];
    }
    if (!a.kkt_only) {
      const T* gAm = a.qp.Am + (size_t)p * N * nx * n; const T* gAp = a.qp.Ap + (size_t)p * N * nx * n;
      for (int e = tid; e < N * nx * n; e += nt) {
        const int t = e / (nx * n), rc = e - t * nx * n, row = rc / n, col = rc - row * n;
        const int o = row * n + (col ^ swz_x<T, NC>(row));
        P[rec(t) + RC::AM + o] = gAm[e];
        P[rec(t + 1) + RC::AP + o] = gAp[e];
      }
      for (int e = tid; e < nx; e += nt) P[rec(0) + RC::AP + e * n + (e ^ swz_x<T, NC>(e))] = T(1);   // A_init = [I 0]
      if (!d.g_sel) { const T* gG = a.qp.G + a.qp.sG * p; for (int e = tid; e < T_ * ng * n; e += nt) { const int t = e / (ng * n); P[rec(t) + RC::G + (e - t * ng * n)] = gG[e]; } }
    }
  }

  // ---- x~ = S^{-1} eta on warp 0: E0 (eta) -> E1 (x~)                                                    (eq. 8)
  // lanes = (problem, direction, row); the operand vector of every step is written to the record by its 8 owners and
  // read back as a broadcast vector load (3 instructions instead of 8 shuffles; in-order issue makes count = time).
  auto chain_solve = [&]() {
    const int lane = tid & 31, slot = lane >> 3, i8 = lane & 7;
    const int g = PG == 2 ? (slot >> 1) : 0, dir = slot & 1;
    const bool act = (PG == 2 || slot < 2) && i8 < n;
    const int ii = i8 < n ? i8 : 0, swx = swz_x<T, NC>(ii);
    const int cnt = act ? (dir ? T_ - 1 - m : m) : 0, t0 = dir ? N : 0, dR = dir ? -R : R;
    const int pb = g * PP, bm = pb + rec(m);
    int bt = cnt > 0 ? pb + rec(t0) : bm;
    T wv = cnt > 0 ? sm[bt + RC::E0 + ii] : T(0);
    // physical chunk c of a swizzled row holds logical columns (c*V) ^ swx ...: load the operand vector in the same order
    auto ld_operand = [&](int base, T (&w)[n]) {
      if constexpr (NC == 8) {
#pragma unroll
        for (int c = 0; c < n / V; ++c) { T part[V]; ld_vec<V>(sm + base + ((c * V) ^ swx), part);
#pragma unroll
          for (int e = 0; e < V; ++e) w[c * V + e] = part[e]; }
      } else ld_vec<n>(sm + base, w);
    };
#pragma unroll 1
    for (int k = 0; k < m; ++k) {                      // consumes the blocks of the current stage, produces w of the next
      const bool on = k < cnt, last = k == cnt - 1;
      if (on) sm[bt + RC::E0 + ii] = wv;
      __syncwarp();
      T W[n], Lr[n], Sr[n];
      ld_operand(bt + RC::E0, W);
      ld_vec<n>(sm + bt + RC::LAM + ii * n, Lr); ld_vec<n>(sm + bt + RC::SINV + ii * n, Sr);
      const int bnext = last ? bm : bt + dR;
      const T eta = (on && !(last && dir)) ? sm[bnext + RC::E0 + ii] : T(0);
      const T aL = dotv<n>(Lr, W), aS = dotv<n>(Sr, W);
      if (on) { sm[bt + RC::E1 + ii] = aS; wv = eta - aL; bt = bnext; }   // v = Sigma^{-1} w ; w_next = eta_next - Lambda w
    }
    // middle stage: w_m = eta_m - Lam_{m-1} w_{m-1} - Lam_{m+1} w_{m+1} ; x_m = Sigma_m^{-1} w_m (both slots redundantly)
    const T wm = wv + __shfl_xor_sync(0xffffffffu, wv, 8);
    if (act) sm[bm + RC::E0 + ii] = wm;
    __syncwarp();
    {
      T W[n], Sr[n];
      ld_operand(bm + RC::E0, W); ld_vec<n>(sm + bm + RC::SINV + ii * n, Sr);
      const T xm = dotv<n>(Sr, W);
      if (act) sm[bm + RC::E1 + ii] = xm;
    }
    __syncwarp();
    // outward sweep: x_t = v_t - Lam_t' x_prev, prev = the neighbour towards the middle
    int bc = cnt > 0 ? pb + rec(t0 + (cnt - 1) * (dir ? -1 : 1)) : bm, bp = bm;
#pragma unroll 1
    for (int k = m - 1; k >= 0; --k) {
      const bool on = k < cnt;
      T X[n], col[n];
      ld_vec<n>(sm + bp + RC::E1, X);
#pragma unroll
      for (int j = 0; j < n; ++j) col[j] = sm[bc + RC::LAM + j * n + (ii ^ swz_x<T, NC>(j))];
      const T v = sm[bc + RC::E1 + ii];
      const T xn = v - dotv<n>(col, X);
      if (on) { sm[bc + RC::E1 + ii] = xn; bp = bc; bc -= dR; }
      __syncwarp();
    }
  };

  // ---- tmpc_kkt_solve: xt <- S^{-1} eta
  if (a.kkt_only) {
    for (int e = tid; e < PG * nz; e += nt) {
      const int g = e / nz, el = e - g * nz, t = el / n, i = el - t * n, p = blockIdx.x * PG + g;
      sm[g * PP + rec(t) + RC::E0 + i] = p < d.B ? a.x[(size_t)p * nz + el] : T(0);
    }
    __syncthreads();
    if (tid < 32) chain_solve();
    __syncthreads();
    for (int e = tid; e < PG * nz; e += nt) {
      const int g = e / nz, el = e - g * nz, t = el / n, i = el - t * n, p = blockIdx.x * PG + g;
      if (p < d.B) a.xi[(size_t)p * nz + el] = sm[g * PP + rec(t) + RC::E1 + i];
    }
    return;
  }

  // ---- per-thread items: (problem g, stage t, row i), two per thread, state in registers.
  // Item (t, i < nx) owns the equality row i of dynamics block t (t < N) or of the init block (t = N: A^- = 0 in record N,
  // A^+ = A_init in record 0); item (t, i < ng) owns inequality row i of stage t.
  constexpr int IPT = 2;
  unsigned fl[IPT]; int bt[IPT], bn[IPT], it_i[IPT];
  T x[IPT], q[IPT], yf[IPT], cv[IPT], zg[IPT], yg[IPT], lo[IPT], hi[IPT];
#pragma unroll
  for (int u = 0; u < IPT; ++u) {
    const int e = tid + u * nt;
    const int g = e / nz, el = e - g * nz, t = el / n, i = el - t * n, p = blockIdx.x * PG + g;
    const bool valid = g < PG && p < d.B;
    fl[u] = 0u; it_i[u] = i; bt[u] = bn[u] = 0;
    x[u] = q[u] = yf[u] = cv[u] = zg[u] = yg[u] = lo[u] = hi[u] = T(0);
    if (valid) {
      fl[u] = F_VALID;
      bt[u] = g * PP + rec(t); bn[u] = g * PP + (t < N ? rec(t + 1) : rec(0));
      x[u] = a.x[(size_t)p * nz + el]; q[u] = a.qp.q[(size_t)p * nz + el];
      if (i < nx) {
        fl[u] |= F_DYN;
        if (t < N) { yf[u] = a.yf[(size_t)p * mf + nx + t * nx + i]; cv[u] = a.qp.b[((size_t)p * N + t) * nx + i]; }
        else { yf[u] = a.yf[(size_t)p * mf + i]; cv[u] = a.qp.x_init[(size_t)p * nx + i]; }
      }
      if (i < ng) {
        const size_t row = (size_t)p * mg + t * ng + i;
        fl[u] |= F_INEQ;
        lo[u] = a.qp.lo[row]; hi[u] = a.qp.hi[row]; yg[u] = a.yg[row];
        if (a.zg_given) zg[u] = a.zg[row];
        else if (a.iters == 0) a.xi[row] = T(0);
        if (a.soft_rows ? (a.soft_rows[row] != 0) : (((d.soft_mask >> i) & 1u) != 0)) fl[u] |= F_SOFT;
      }
      if (d.g_sel) {
#pragma unroll
        for (int r = 0; r < NC; ++r) if (r < ng) {       // static indices: no local copy of the parameter array
          if (r == i) fl[u] |= (unsigned)d.g_col[r] << F_GCOL_SH;
          if (d.g_col[r] == i) fl[u] |= 1u << (F_GMASK_SH + r);
        }
      }
    }
  }
  // (G_t vec_t)[row i] for the owner of inequality row (t, i); field = RC::E1 (or wherever vec_t sits in the record)
  auto g_dot_item = [&](int u, int field) -> T {
    if (d.g_sel) return sm[bt[u] + field + (int)((fl[u] >> F_GCOL_SH) & 15u)];
    T gr[n], vt[n];
    ld_vec<n>(sm + bt[u] + RC::G + it_i[u] * n, gr); ld_vec<n>(sm + bt[u] + field, vt);
    return dotv<n>(gr, vt);
  };
  auto g_row = [&](int u) -> size_t {                    // global index of the inequality row of item u (recomputed: not kept live)
    const int e = tid + u * nt, g = e / nz, el = e - g * nz, t = el / n;
    return (size_t)(blockIdx.x * PG + g) * mg + t * ng + it_i[u];
  };
  auto put_r = [&](int u) {                              // r = rho_f c - y_f, for both records that read it
    const T r = a.prm.rho_f * cv[u] - yf[u];
    sm[bt[u] + RC::RM + it_i[u]] = r; sm[bn[u] + RC::RP + it_i[u]] = r;
  };
  // z_g^0 = clip(G x^0, lo, hi) unless given; r = rho_f c - y_f ; s = rho_g z_g - y_g
#pragma unroll
  for (int u = 0; u < IPT; ++u) if (fl[u] & F_VALID) sm[bt[u] + RC::E1 + it_i[u]] = x[u];
  __syncthreads();
#pragma unroll
  for (int u = 0; u < IPT; ++u) {
    if (fl[u] & F_INEQ) {
      if (!a.zg_given) zg[u] = tmin(tmax(g_dot_item(u, RC::E1), lo[u]), hi[u]);
      sm[bt[u] + RC::S + it_i[u]] = a.prm.rho_g * zg[u] - yg[u];
    }
    if (fl[u] & F_DYN) put_r(u);
  }
  __syncthreads();

#pragma unroll 1
  for (int it = 0; it < a.iters; ++it) {
    // a4: eta = sigma x - q + C'(rho_f c - y_f) + G'(rho_g z_g - y_g)                                       (eq. 51)
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
      if (!(fl[u] & F_VALID)) continue;
      const int b = bt[u], i = it_i[u];
      T am[nx], ap[nx], rm[nx], rp[nx];
#pragma unroll
      for (int k = 0; k < nx; ++k) { am[k] = sm[b + RC::AM + k * n + (i ^ swz_x<T, NC>(k))]; ap[k] = sm[b + RC::AP + k * n + (i ^ swz_x<T, NC>(k))]; }
      ld_vec<nx>(sm + b + RC::RM, rm); ld_vec<nx>(sm + b + RC::RP, rp);
      T s = a.prm.sigma * x[u] - q[u];
      s += dotv<nx>(am, rm) + dotv<nx>(ap, rp);
      if (d.g_sel) { unsigned mk = (fl[u] >> F_GMASK_SH) & 255u; while (mk) { const int r = __ffs(mk) - 1; mk &= mk - 1; s += sm[b + RC::S + r]; } }
      else { for (int r = 0; r < ng; ++r) s += sm[b + RC::G + r * n + i] * sm[b + RC::S + r]; }
      sm[b + RC::E0 + i] = s;
    }
    __syncthreads();
    if (tid < 32) chain_solve();
    __syncthreads();
    // a7 + a8: z~ = A x~ (eq. 9), relaxation (eq. 10), projection (eq. 12-15), duals (eq. 16 / 44-45)
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
      if (!(fl[u] & F_VALID)) continue;
      const int b = bt[u], i = it_i[u];
      if (fl[u] & F_DYN) {
        T am[n], ap[n], xa[n], xb[n];
        ld_vec<n>(sm + b + RC::AM + i * n, am); ld_vec<n>(sm + bn[u] + RC::AP + i * n, ap);
        const int swx = swz_x<T, NC>(i);
        if constexpr (NC == 8) {
#pragma unroll
          for (int c = 0; c < n / V; ++c) { T pa[V], pb2[V]; ld_vec<V>(sm + b + RC::E1 + ((c * V) ^ swx), pa); ld_vec<V>(sm + bn[u] + RC::E1 + ((c * V) ^ swx), pb2);
#pragma unroll
            for (int e = 0; e < V; ++e) { xa[c * V + e] = pa[e]; xb[c * V + e] = pb2[e]; } }
        } else { ld_vec<n>(sm + b + RC::E1, xa); ld_vec<n>(sm + bn[u] + RC::E1, xb); }
        const T zt = dotv<n>(am, xa) + dotv<n>(ap, xb);
        yf[u] += A.rfa * (zt - cv[u]);
        put_r(u);
      }
      if (fl[u] & F_INEQ) {
        const T ztg = g_dot_item(u, RC::E1);
        const T zh = a.prm.alpha * ztg + A.oma * zg[u];
        const T v = zh + yg[u] * A.inv_rho_g;
        T z, s;
        project_row<T>((fl[u] & F_SOFT) != 0, v, lo[u], hi[u], a.prm.rho_g, A.inv_rg, a.prm.lam, z, s);
        yg[u] += a.prm.rho_g * (zh - z);
        zg[u] = z;
        sm[b + RC::S + i] = a.prm.rho_g * z - yg[u];
        if (it == a.iters - 1) a.xi[g_row(u)] = s;
      }
      x[u] = a.prm.alpha * sm[b + RC::E1 + i] + A.oma * x[u];
    }
    __syncthreads();
  }

  // ---- write back the state
#pragma unroll
  for (int u = 0; u < IPT; ++u) {
    if (!(fl[u] & F_VALID)) continue;
    const int e = tid + u * nt, g = e / nz, el = e - g * nz, t = el / n, i = it_i[u], p = blockIdx.x * PG + g;
    a.x[(size_t)p * nz + el] = x[u];
    if (fl[u] & F_DYN) a.yf[(size_t)p * mf + (t < N ? nx + t * nx + i : i)] = yf[u];
    if (fl[u] & F_INEQ) { const size_t row = g_row(u); a.zg[row] = zg[u]; a.yg[row] = yg[u]; }
  }
}

// ---- a9: residuals (eq. 3) and objective at the iterate in global memory; one CTA per problem
template <typename T>
struct ResidualArgs {
  Dims d; Params<T> prm; QpView<T> qp;
  const T* x; const T* zg; const T* yf; const T* yg; const T* xi;
  T* r_prim; T* r_dual; T* objective; int32_t* status;
};

template <typename T>
__global__ void __launch_bounds__(256) residual_kernel(ResidualArgs<T> a) {
  __shared__ T red[64];
  const Dims& d = a.d;
  const int n = d.n, nx = d.nx, ng = d.ng, N = d.N, nn = n * n, nz = d.nz, mf = d.mf, mg = d.mg;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const T gam = a.prm.gamma, lam = a.prm.lam;
  const T* x = a.x + (size_t)p * nz; const T* zg = a.zg + (size_t)p * mg; const T* yf = a.yf + (size_t)p * mf;
  const T* yg = a.yg + (size_t)p * mg; const T* xi = a.xi + (size_t)p * mg; const T* q = a.qp.q + (size_t)p * nz;
  const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p;
  const T* Am = a.qp.Am + (size_t)p * N * nx * n; const T* Ap = a.qp.Ap + (size_t)p * N * nx * n;
  const T* G = a.qp.G ? a.qp.G + a.qp.sG * p : nullptr;
  T rp = T(0), rd = T(0), ob = T(0); int bad = 0;
  for (int e = tid; e < mf; e += nt) {
    T cx, c;
    if (e < nx) { cx = x[e]; c = a.qp.x_init[(size_t)p * nx + e]; }
    else {
      const int t = (e - nx) / nx, i = (e - nx) - t * nx;
      const T* am = Am + ((size_t)t * nx + i) * n; const T* ap = Ap + ((size_t)t * nx + i) * n;
      T s = T(0);
      for (int j = 0; j < n; ++j) s += am[j] * x[t * n + j] + ap[j] * x[(t + 1) * n + j];
      cx = s; c = a.qp.b[(size_t)p * N * nx + (e - nx)];
    }
    rp = tmax(rp, tabs(cx - c));
  }
  for (int e = tid; e < mg; e += nt) {
    const int t = e / ng, r = e - t * ng;
    T gx;
    if (d.g_sel) gx = x[t * n + d.g_col[r]];
    else { const T* g = G + ((size_t)t * ng + r) * n; gx = T(0); for (int j = 0; j < n; ++j) gx += g[j] * x[t * n + j]; }
    rp = tmax(rp, tabs(gx - zg[e]));
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

}  // namespace tmpc
