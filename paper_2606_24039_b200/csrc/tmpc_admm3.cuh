// tmpc_admm3.cuh — a4..a8 for the RESIDENT class, second generation (round 2): the fused ADMM loop of Alg. 3
// on the twisted block factor of tmpc_factor2.cuh, all iterations in one launch.
//
// What changed against tmpc_admm2.cuh, and why (ncu of admm2 at config 2: 62 % of the warp samples wait at a barrier, the
// LSU pipe carries 1435 shared-memory wavefronts per problem-iteration = 52 % of its peak, 23 % of them excess):
//  * TWO lanes per stage instead of four.  Lane h of a stage owns the columns [h n/2, (h+1) n/2) of every block of
//    the stage record, the same rows of the stage variable, and half of the dynamics / inequality rows.  Every matrix
//    access is then a 16-byte load of "my column chunk of row k" (products with a transposed block: A~' r, X' y, G~' s)
//    or of a full row taken "my chunk first, the partner's second" (X d, A~ y, G~ y) — no scalar column loads, every
//    block element is read exactly once per use and no operand vector is loaded by four threads.
//  * the stage vector d = sigma x - q + G's is exchanged between the two lanes of a stage with one shuffle per
//    component instead of a shared-memory round trip plus a warp barrier.
//  * the records are NOT swizzled: with a record stride of 8 (mod 32) words the eight lanes of a quarter warp (four
//    stages x two halves) hit the eight distinct 16-byte bank groups in every access pattern above, and so do the eight
//    lanes of a chain slot once rows >= n/2 take their two chunks in the opposite order (admm2's 2-way conflict).
//  * half the item warps: a CTA of two problems is 7 item warps + the chain warp (256 threads), which leaves 128
//    registers per thread for the operand vectors.
// The chain warp (x~ = S^{-1} eta, eq. 8) and the named-barrier handshake are those of admm2.
#pragma once
#include "tmpc_common.cuh"
#include "tmpc_admm.cuh"
#include "tmpc_admm2.cuh"

namespace tmpc {

// ---- shared-memory record of one stage (elements of T); fields as in tmpc_admm2.cuh Rec, rows stored unswizzled
template <typename T, int NC, int NX>
struct Rec3 {
  static constexpr int V = 16 / (int)sizeof(T);
  static constexpr int up(int v) { return (v + V - 1) / V * V; }
  static constexpr int AM = 0, AP = AM + up(NX * NC), RM = AP + up(NX * NC), RP = RM + up(NX), E0 = RP + up(NX),
                       E1 = E0 + up(NC), LAM = E1 + up(NC), SINV = LAM + up(NC * NC), S = SINV + up(NC * NC), G = S + up(NC);   // S, G: dense G only
  static constexpr int SKEW = 32 / (int)sizeof(T);      // 32 bytes: the down-chain records sit one 8-bank group off
  static constexpr int pad_stride(int r) {               // record stride = 32 bytes (mod 128 bytes)
    constexpr int W128 = 128 / (int)sizeof(T), W32 = 32 / (int)sizeof(T);
    while (r % W128 != W32) r += V;
    return r;
  }
};
struct Admm3Plan { int R, per_problem; };

template <typename T, int NC, int NX>
inline Admm3Plan admm3_plan(const Dims& d, int pg) {
  using RC = Rec3<T, NC, NX>;
  Admm3Plan P;
  int R = d.g_sel ? RC::S : RC::G + ((d.ng * NC + RC::V - 1) / RC::V) * RC::V;
  P.R = RC::pad_stride(R);
  int pp = d.T * P.R + RC::SKEW;
  if (pg == 2) { const int w128 = 128 / (int)sizeof(T), w64 = 64 / (int)sizeof(T); while (pp % w128 != w64) pp += RC::V; }   // second problem: two bank groups off
  P.per_problem = pp;
  return P;
}
template <typename T, int NC, int NX>
inline size_t admm3_smem_bytes(const Dims& d, int pg) { return (size_t)admm3_plan<T, NC, NX>(d, pg).per_problem * pg * sizeof(T); }

template <typename T>
struct Admm3Args {
  AdmmArgs<T> a;
  Admm3Plan pl;
  T rfa, oma, inv_rho_g, inv_rg;      // rho_f alpha, 1 - alpha, 1 / rho_g, 1 / (rho_g + gamma)
};

// ---- H contiguous elements at a 16-byte aligned address (H * sizeof(T) a multiple of 16) or, for H = 3, the three
// elements of a lane's half of a 6-wide row: an 8-byte aligned pair plus one element (see chunk3 below)
template <int H> __device__ __forceinline__ void ld_chunk(const float* __restrict__ p, float (&r)[H]) {
  static_assert(H % 4 == 0, "float chunks are multiples of 16 bytes");
#pragma unroll
  for (int c = 0; c < H / 4; ++c) { const float4 v = reinterpret_cast<const float4*>(p)[c]; r[4 * c] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w; }
}
template <int H> __device__ __forceinline__ void ld_chunk(const double* __restrict__ p, double (&r)[H]) {
  static_assert(H % 2 == 0, "double chunks are multiples of 16 bytes");
#pragma unroll
  for (int c = 0; c < H / 2; ++c) { const double2 v = reinterpret_cast<const double2*>(p)[c]; r[2 * c] = v.x; r[2 * c + 1] = v.y; }
}
template <int H> __device__ __forceinline__ void st_chunk(float* __restrict__ p, const float (&r)[H]) {
#pragma unroll
  for (int c = 0; c < H / 4; ++c) reinterpret_cast<float4*>(p)[c] = make_float4(r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
}
template <int H> __device__ __forceinline__ void st_chunk(double* __restrict__ p, const double (&r)[H]) {
#pragma unroll
  for (int c = 0; c < H / 2; ++c) reinterpret_cast<double2*>(p)[c] = make_double2(r[2 * c], r[2 * c + 1]);
}
// acc[s] += m[s] * w for a chunk (packed FFMA2 for float)
template <int H> __device__ __forceinline__ void axpy_chunk(float (&acc)[H], const float (&m)[H], float w) {
#pragma unroll
  for (int s = 0; s + 1 < H; s += 2) { const float2 r = __ffma2_rn(make_float2(m[s], m[s + 1]), make_float2(w, w), make_float2(acc[s], acc[s + 1])); acc[s] = r.x; acc[s + 1] = r.y; }
  if constexpr (H % 2) acc[H - 1] = fmaf(m[H - 1], w, acc[H - 1]);
}
template <int H> __device__ __forceinline__ void axpy_chunk(double (&acc)[H], const double (&m)[H], double w) {
#pragma unroll
  for (int s = 0; s < H; ++s) acc[s] = fma(m[s], w, acc[s]);
}
__device__ __forceinline__ float shfl_x1(float v) { return __shfl_xor_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_x1(double v) { return __shfl_xor_sync(0xffffffffu, v, 1); }

// ---- x~ = S^{-1} eta on the scaled variables (tmpc_factor2.cuh): E1 holds eta~ on entry and w on exit, E0 receives y.
// One warp; lanes = (problem, direction, row), 8 lanes per slot (tmpc_admm2.cuh chain_warp_solve on the unswizzled record:
// row i >= n/2 takes its 16-byte chunks in the opposite order — `swb` — so that the eight rows of a slot cover the eight
// bank groups; the broadcast operand vector is read in the same order).
template <typename T, int NC, int NX, int PG>
__device__ __forceinline__ void chain3_solve(T* sm, int R, int PP, int T_, int lane, long long* tm = nullptr) {
  static_assert(NC == 8 || NC == 6, "chain lanes are written for n = 6 and n = 8");
  using RC = Rec3<T, NC, NX>;
  constexpr int n = NC;
  constexpr unsigned ES = sizeof(T);
  const unsigned sb = (unsigned)__cvta_generic_to_shared(sm);
  const int N = T_ - 1, m = T_ / 2;
  const int slot = lane >> 3, i8 = lane & 7;
  const int g = PG == 2 ? (slot >> 1) : 0, dir = slot & 1;
  const bool act = (PG == 2 || slot < 2) && i8 < n;
  const int ii = i8 < n ? i8 : 0;
  const unsigned swb = (unsigned)swz_x<T, NC>(ii) * ES;                 // chunk ORDER of my row (bytes); the data is not swizzled
  const int cnt = act ? (dir ? T_ - 1 - m : m) : 0, t0 = dir ? N : 0;
  const int dRb = (dir ? -R : R) * (int)ES;
  auto rec = [&](int t) { return t * R + (t > m ? RC::SKEW : 0); };
  const unsigned pb = sb + (unsigned)(g * PP) * ES, bm = pb + (unsigned)rec(m) * ES;
  constexpr unsigned oE0 = RC::E0 * ES, oE1 = RC::E1 * ES, oLAM = RC::LAM * ES;
  const unsigned me = (unsigned)ii * ES, myrow = oLAM + (unsigned)(ii * n) * ES;
  unsigned bt = cnt > 0 ? pb + (unsigned)rec(t0) * ES : bm;
  T wv = cnt > 0 ? lds_1(bt + oE1 + me, T(0)) : T(0);
  T Br[n];
  lds_row<T, NC>(bt + myrow, swb, Br);
  const int cmin = T_ - 1 - m;                          // = the down chain's length <= the up chain's (m)
  const int kmain = cmin > 1 ? ((cmin - 1) & ~1) : 0;   // even: the main loop is unrolled by two
  const int dRa = act ? dRb : 0;                        // idle lanes stay on record m
#ifdef TMPC_TIMING
  const long long q0 = clock64();
#endif
  // Main loop: every active slot is on and none is at its last stage, so no predicates.  Two steps per trip with the row
  // buffers Br / Bn swapping roles (no register copies: in admm2 the copies Br <- Bn sat in front of the final adds in program
  // order and made the in-order issue wait for the NEXT step's row load inside the dependent chain of THIS step).
#pragma unroll 1
  for (int k = 0; k < kmain; k += 2) {
    T W[n], Bn[n], eta;
    if (act) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    lds_row<T, NC>(bt + oE1, swb, W);
    bt += dRa;
    eta = lds_1(bt + oE1 + me, T(0));
    lds_row<T, NC>(bt + myrow, swb, Bn);
    wv = dotv_from<n>(Br, W, eta);
    if (act) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    lds_row<T, NC>(bt + oE1, swb, W);
    bt += dRa;
    eta = lds_1(bt + oE1 + me, T(0));
    lds_row<T, NC>(bt + myrow, swb, Br);
    wv = dotv_from<n>(Bn, W, eta);
  }
#ifdef TMPC_TIMING
  const long long q1 = clock64();
#endif
#pragma unroll 1
  for (int k = kmain; k < m; ++k) {                    // w_next = eta~_next + (-B_t) w_t
    const bool on = k < cnt, last = k == cnt - 1;
    if (on) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    T W[n];
    lds_row<T, NC>(bt + oE1, swb, W);
    pin_vec<n>(W);
    const unsigned bnext = last ? bm : bt + dRb;
    const T eta = (on && !(last && dir)) ? lds_1(bnext + oE1 + me, T(0)) : T(0);
    if (on) bt = bnext;
    T Bn[n];
    lds_row<T, NC>(bt + myrow, swb, Bn);               // next step's row (record m holds zeros: harmless)
    const T nw = dotv_from<n>(Br, W, eta);
    if (on) wv = nw;
#pragma unroll
    for (int j = 0; j < n; ++j) Br[j] = Bn[j];
  }
  // middle stage: w_m = eta~_m + both contributions; y_m = w_m
  const T wm = wv + __shfl_xor_sync(0xffffffffu, wv, 8);
  if (act) { sts_1(bm + oE1 + me, wm); sts_1(bm + oE0 + me, wm); }
  __syncwarp();
#ifdef TMPC_TIMING
  const long long q2 = clock64();
#endif
  // outward sweep: y_t = w_t + (-B_t)' y_next
  unsigned bc = cnt > 0 ? pb + (unsigned)rec(t0 + (cnt - 1) * (dir ? -1 : 1)) * ES : bm, bp = bm;
#pragma unroll 1
  for (int k = m - 1; k >= 0; --k) {
    const bool on = k < cnt;
    T Y[n], col[n];
    lds_row<T, NC>(bp + oE0, 0u, Y);
#pragma unroll
    for (int j = 0; j < n; ++j) col[j] = lds_1(bc + oLAM + (unsigned)(j * n) * ES + me, T(0));
    const T w = lds_1(bc + oE1 + me, T(0));
    const T y = dotv_from<n>(col, Y, w);
    if (on) { sts_1(bc + oE0 + me, y); bp = bc; bc -= dRb; }
    __syncwarp();
  }
#ifdef TMPC_TIMING
  if (tm) { const long long q3 = clock64(); tm[0] += q1 - q0; tm[1] += q2 - q1; tm[2] += q3 - q2; }
#endif
}

template <typename T, int H> __device__ __forceinline__ T dot2(const T (&a)[H], const T (&x)[H], const T (&b)[H], const T (&y)[H]) {
  return dotv<H>(a, x) + dotv<H>(b, y);      // first chunk with my half of the operand, second with the partner's
}

// Lane map of an item thread: (problem g of the CTA, stage t, half h).  Half h owns the columns / x-rows [h H, (h+1) H),
// the dynamics rows [h KA, ...) of ITS stage's block (block t for t < N; the rows x_0 = x_init for t = N, whose A^+ = [I 0]
// sits in record 0), and the inequality rows: for a selection G the rows whose column it owns, for a dense G the rows 2 s + h.
template <typename T, int NC, int NX, int PG, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) admm3_kernel(const __grid_constant__ Admm3Args<T> A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  using RC = Rec3<T, NC, NX>;
  static_assert(NC % 2 == 0 && ((NC / 2) * sizeof(T)) % 16 == 0, "a lane's column chunk must be a multiple of 16 bytes");
  const AdmmArgs<T>& a = A.a;
  const Dims& d = a.d;
  constexpr int n = NC, nx = NX, nn = NC * NC, H = NC / 2, KA = (NX + 1) / 2;
  const int R = A.pl.R, PP = A.pl.per_problem;
  const int ng = d.ng, N = d.N, T_ = d.T, nz = T_ * n, mf = d.mf, mg = d.mg;
  const int tid = threadIdx.x, nt = blockDim.x, nti = nt - 32, it_tid = tid - 32;
  const int m = T_ / 2;
  auto rec = [&](int t) { return t * R + (t > m ? RC::SKEW : 0); };

  // ---- stage 1: X_t and -B_t of every problem of this CTA into the records (all threads)
#pragma unroll 1
  for (int g = 0; g < PG; ++g) {
    const int p = blockIdx.x * PG + g;
    T* P = sm + g * PP;
    for (int e = tid; e < PP; e += nt) P[e] = T(0);
    __syncthreads();
    if (p >= d.B) continue;
    const T* gLam = a.Lam + (size_t)p * T_ * nn;
    const T* gX = a.Sinv + (size_t)p * T_ * nn;
    for (int e = tid; e < T_ * nn; e += nt) {
      const int t = e / nn, rc = e - t * nn;
      const int o = rec(t) + rc;
      if (t != m) P[o + RC::LAM] = -gLam[e];
      P[o + RC::SINV] = gX[e];
    }
  }
  __syncthreads();
  // ---- stage 2: constraint blocks in the scaled variables: A~^-_t = A^-_t X_t', A~^+_{t-1} = A^+_{t-1} X_t', G~_t = G_t X_t'
  if (!a.kkt_only) {
#pragma unroll 1
    for (int g = 0; g < PG; ++g) {
      const int p = blockIdx.x * PG + g;
      if (p >= d.B) continue;
      T* P = sm + g * PP;
      const T* gAm = a.qp.Am + (size_t)p * N * nx * n; const T* gAp = a.qp.Ap + (size_t)p * N * nx * n;
      for (int e = tid; e < T_ * nx * n; e += nt) {    // (t, row k, col j): sum_l M[k][l] X_t[j][l], l <= j
        const int t = e / (nx * n), rc = e - t * nx * n, k = rc / n, j = rc - k * n;
        const T* Xj = P + rec(t) + RC::SINV + j * n;
        T sa = T(0), sp = T(0);
        if (t < N) { const T* Mr = gAm + ((size_t)t * nx + k) * n; for (int l = 0; l <= j; ++l) sa += Mr[l] * Xj[l]; }
        if (t > 0) { const T* Mr = gAp + ((size_t)(t - 1) * nx + k) * n; for (int l = 0; l <= j; ++l) sp += Mr[l] * Xj[l]; }
        else if (k <= j) sp = Xj[k];                    // A_init = [I 0]
        P[rec(t) + RC::AM + rc] = sa;
        P[rec(t) + RC::AP + rc] = sp;
      }
      if (!d.g_sel) {
        const T* gG = a.qp.G + a.qp.sG * p;
        for (int e = tid; e < T_ * ng * n; e += nt) {
          const int t = e / (ng * n), rc = e - t * ng * n, k = rc / n, j = rc - k * n;
          const T* Xj = P + rec(t) + RC::SINV + j * n; const T* Mr = gG + ((size_t)t * ng + k) * n;
          T sg = T(0);
          for (int l = 0; l <= j; ++l) sg += Mr[l] * Xj[l];
          P[rec(t) + RC::G + rc] = sg;
        }
      }
    }
    __syncthreads();
  }

  // ================================================================ chain warp
  if (tid < 32) {
    const int iters = a.kkt_only ? 1 : a.iters;
#pragma unroll 1
#ifdef TMPC_TIMING
    long long tw = 0, ts = 0, tm[3] = {0, 0, 0};
#endif
    for (int it = 0; it < iters; ++it) {
#ifdef TMPC_TIMING
      const long long c0 = clock64();
#endif
      bar_sync(1, nt);
#ifdef TMPC_TIMING
      const long long c1 = clock64();
#endif
#ifdef TMPC_TIMING
      chain3_solve<T, NC, NX, PG>(sm, R, PP, T_, tid, tm);
#else
      chain3_solve<T, NC, NX, PG>(sm, R, PP, T_, tid);
#endif
      __syncwarp();
#ifdef TMPC_TIMING
      tw += c1 - c0; ts += clock64() - c1;
#endif
      bar_arrive(2, nt);
    }
#ifdef TMPC_TIMING
    if ((blockIdx.x == 0 || blockIdx.x == gridDim.x - 1) && tid == 0) printf("cta %d chain warp: wait %lld solve %lld cycles per iteration; fwd main %lld tail+mid %lld bwd %lld\n", blockIdx.x, tw / iters, ts / iters, tm[0] / iters, tm[1] / iters, tm[2] / iters);
#endif
    return;
  }

  // ================================================================ item warps
  const int per_p = 2 * T_;                              // lanes per problem
  const int g = it_tid / per_p, rem = it_tid - g * per_p, t = rem >> 1, h = rem & 1, p = blockIdx.x * PG + g;
  const bool valid = g < PG && p < d.B;
  const int c0 = h * H, oc = H - c0;                     // my column chunk, the partner's
  const int b = valid ? g * PP + rec(t) : 0, bn = valid ? g * PP + (t < N ? rec(t + 1) : rec(0)) : 0;
  const T* Xb = sm + b + RC::SINV;

  if (a.kkt_only) {                                      // xt <- S^{-1} eta : eta~ = X eta, solve, x = X' y
    T eo[H], er[H];
#pragma unroll
    for (int s = 0; s < H; ++s) eo[s] = valid ? a.x[(size_t)p * nz + t * n + c0 + s] : T(0);
#pragma unroll
    for (int s = 0; s < H; ++s) er[s] = shfl_x1(eo[s]);
    if (valid) {
      T acc[H];
#pragma unroll
      for (int s = 0; s < H; ++s) { T f[H], f2[H]; ld_chunk<H>(Xb + (c0 + s) * n + c0, f); ld_chunk<H>(Xb + (c0 + s) * n + oc, f2); acc[s] = dot2<T, H>(f, eo, f2, er); }
      st_chunk<H>(sm + b + RC::E1 + c0, acc);
    }
    bar_arrive(1, nt);
    bar_sync(2, nt);
    if (valid) {
      T yo[H], yr[H], xt[H];
      ld_chunk<H>(sm + b + RC::E0 + c0, yo); ld_chunk<H>(sm + b + RC::E0 + oc, yr);
#pragma unroll
      for (int s = 0; s < H; ++s) xt[s] = T(0);
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ld_chunk<H>(Xb + (c0 + jj) * n + c0, mk); axpy_chunk<H>(xt, mk, yo[jj]); }
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ld_chunk<H>(Xb + (oc + jj) * n + c0, mk); axpy_chunk<H>(xt, mk, yr[jj]); }
#pragma unroll
      for (int s = 0; s < H; ++s) a.xi[(size_t)p * nz + t * n + c0 + s] = xt[s];
    }
    return;
  }

  // ---- per-lane state in registers
  constexpr unsigned Q_VALID = 1u, Q_SOFT = 2u, Q_ROW_SH = 4;         // inequality slot flags: valid, soft, row index << 4
  T x[H], q[H], zg[H], yg[H], lo[H], hi[H], xi_last[H];
  T yf[KA], cv[KA];
  unsigned qf[H];                                                     // inequality slot s <-> (selection: my column c0 + s; dense: row 2 s + h)
  const int k0 = h * KA, nk = valid ? (h ? nx - KA : KA) : 0;         // my dynamics rows k0 .. k0 + nk - 1
#pragma unroll
  for (int s = 0; s < H; ++s) { x[s] = q[s] = zg[s] = yg[s] = lo[s] = hi[s] = xi_last[s] = T(0); qf[s] = 0u; }
#pragma unroll
  for (int s = 0; s < KA; ++s) yf[s] = cv[s] = T(0);
  if (valid) {
#pragma unroll
    for (int s = 0; s < H; ++s) { const size_t el = (size_t)p * nz + t * n + c0 + s; x[s] = a.x[el]; q[s] = a.qp.q[el]; }
#pragma unroll
    for (int s = 0; s < KA; ++s) if (s < nk) {
      const int k = k0 + s;
      if (t < N) { yf[s] = a.yf[(size_t)p * mf + nx + t * nx + k]; cv[s] = a.qp.b[((size_t)p * N + t) * nx + k]; }
      else { yf[s] = a.yf[(size_t)p * mf + k]; cv[s] = a.qp.x_init[(size_t)p * nx + k]; }
    }
#pragma unroll
    for (int s = 0; s < H; ++s) {
      int r = -1;
      if (d.g_sel) {
#pragma unroll
        for (int rr = 0; rr < NC; ++rr) if (rr < ng && d.g_col[rr] == c0 + s) r = rr;
      } else if (2 * s + h < ng) r = 2 * s + h;
      if (r < 0) continue;
      const size_t row = (size_t)p * mg + t * ng + r;
      qf[s] = Q_VALID | ((unsigned)r << Q_ROW_SH);
      lo[s] = a.qp.lo[row]; hi[s] = a.qp.hi[row]; yg[s] = a.yg[row];
      if (a.soft_rows ? (a.soft_rows[row] != 0) : (((d.soft_mask >> r) & 1u) != 0)) qf[s] |= Q_SOFT;
      if (a.zg_given) zg[s] = a.zg[row];
      else {                                             // z_g^0 = clip(G x^0, lo, hi) (x-space, straight from the problem data)
        T gx;
        if (d.g_sel) gx = x[s];
        else {
          const T* gr = a.qp.G + a.qp.sG * p + ((size_t)t * ng + r) * n; const T* xs = a.x + (size_t)p * nz + t * n;
          gx = T(0);
          for (int j = 0; j < n; ++j) gx += gr[j] * xs[j];
        }
        zg[s] = tmin(tmax(gx, lo[s]), hi[s]);
        if (a.iters == 0) a.xi[row] = T(0);
      }
      if (!d.g_sel) sm[b + RC::S + r] = a.prm.rho_g * zg[s] - yg[s];
    }
#pragma unroll
    for (int s = 0; s < KA; ++s) if (s < nk) { const T r = a.prm.rho_f * cv[s] - yf[s]; sm[b + RC::RM + k0 + s] = r; sm[bn + RC::RP + k0 + s] = r; }
  }
  bar_sync(3, nti);

#pragma unroll 1
  for (int it = 0; it < a.iters; ++it) {
    // ---- a4 in scaled variables (eq. 51): eta~_t = X_t (sigma x - q + G's) + A~^-_t' r_t + A~^+_{t-1}' r_{t-1}  [+ G~_t' s for a dense G]
    T dn[H], dr[H];
#pragma unroll
    for (int s = 0; s < H; ++s) {
      T dd = a.prm.sigma * x[s] - q[s];
      if (d.g_sel && (qf[s] & Q_VALID)) dd += a.prm.rho_g * zg[s] - yg[s];
      dn[s] = dd;
    }
#pragma unroll
    for (int s = 0; s < H; ++s) dr[s] = shfl_x1(dn[s]);            // the partner's half of the stage vector
    if (valid) {
      T acc[H], rm[nx], rp[nx];
      ld_vec<nx>(sm + b + RC::RM, rm); ld_vec<nx>(sm + b + RC::RP, rp);
#pragma unroll
      for (int s = 0; s < H; ++s) {                    // my rows of X_t: my chunk first, then the partner's (zero for h = 0: X is lower triangular)
        T f[H], f2[H];
        ld_chunk<H>(Xb + (c0 + s) * n + c0, f); ld_chunk<H>(Xb + (c0 + s) * n + oc, f2);
        acc[s] = dot2<T, H>(f, dn, f2, dr);
      }
#pragma unroll
      for (int k = 0; k < nx; ++k) {                   // my columns of A~^-_t and A~^+_{t-1}
        T mk[H];
        ld_chunk<H>(sm + b + RC::AM + k * n + c0, mk); axpy_chunk<H>(acc, mk, rm[k]);
        ld_chunk<H>(sm + b + RC::AP + k * n + c0, mk); axpy_chunk<H>(acc, mk, rp[k]);
      }
      if (!d.g_sel) for (int r = 0; r < ng; ++r) { T mk[H]; ld_chunk<H>(sm + b + RC::G + r * n + c0, mk); axpy_chunk<H>(acc, mk, sm[b + RC::S + r]); }
      st_chunk<H>(sm + b + RC::E1 + c0, acc);
    }
    bar_arrive(1, nt);
    bar_sync(2, nt);
    // ---- a7 + a8 on y: x~ = X_t' y_t, z~_f = A~^-_t y_t + A~^+_t y_{t+1}, z~_g = x~_col or G~_t y_t; relaxation (eq. 10),
    // projection (eq. 12-15), duals (eq. 16 / 44-45)
    if (valid) {
      T yo[H], yr[H], xt[H];
      ld_chunk<H>(sm + b + RC::E0 + c0, yo); ld_chunk<H>(sm + b + RC::E0 + oc, yr);
#pragma unroll
      for (int s = 0; s < H; ++s) xt[s] = T(0);
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ld_chunk<H>(Xb + (c0 + jj) * n + c0, mk); axpy_chunk<H>(xt, mk, yo[jj]); }   // rows of my half
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ld_chunk<H>(Xb + (oc + jj) * n + c0, mk); axpy_chunk<H>(xt, mk, yr[jj]); }   // rows of the partner's half
      if (nk > 0) {
        T y2o[H], y2r[H];
        ld_chunk<H>(sm + bn + RC::E0 + c0, y2o); ld_chunk<H>(sm + bn + RC::E0 + oc, y2r);
#pragma unroll
        for (int s = 0; s < KA; ++s) if (s < nk) {
          const int k = k0 + s;
          T f[H], f2[H];
          ld_chunk<H>(sm + b + RC::AM + k * n + c0, f); ld_chunk<H>(sm + b + RC::AM + k * n + oc, f2);
          T zt = dot2<T, H>(f, yo, f2, yr);
          ld_chunk<H>(sm + bn + RC::AP + k * n + c0, f); ld_chunk<H>(sm + bn + RC::AP + k * n + oc, f2);
          zt += dot2<T, H>(f, y2o, f2, y2r);
          yf[s] += A.rfa * (zt - cv[s]);
          const T r = a.prm.rho_f * cv[s] - yf[s];
          sm[b + RC::RM + k] = r; sm[bn + RC::RP + k] = r;
        }
      }
#pragma unroll
      for (int s = 0; s < H; ++s) {
        if (qf[s] & Q_VALID) {
          T ztg = xt[s];
          if (!d.g_sel) { const int r = (int)(qf[s] >> Q_ROW_SH); T f[H], f2[H]; ld_chunk<H>(sm + b + RC::G + r * n + c0, f); ld_chunk<H>(sm + b + RC::G + r * n + oc, f2); ztg = dot2<T, H>(f, yo, f2, yr); }
          const T zh = a.prm.alpha * ztg + A.oma * zg[s];
          const T v = zh + yg[s] * A.inv_rho_g;
          T z, sl;
          project_row<T>((qf[s] & Q_SOFT) != 0, v, lo[s], hi[s], a.prm.rho_g, A.inv_rg, a.prm.lam, z, sl);
          yg[s] += a.prm.rho_g * (zh - z);
          zg[s] = z;
          if (!d.g_sel) sm[b + RC::S + (int)(qf[s] >> Q_ROW_SH)] = a.prm.rho_g * z - yg[s];
          xi_last[s] = sl;
        }
        x[s] = a.prm.alpha * xt[s] + A.oma * x[s];
      }
    }
    bar_sync(3, nti);
  }

  // ---- write back the state
  if (valid) {
#pragma unroll
    for (int s = 0; s < H; ++s) a.x[(size_t)p * nz + t * n + c0 + s] = x[s];
#pragma unroll
    for (int s = 0; s < KA; ++s) if (s < nk) a.yf[(size_t)p * mf + (t < N ? nx + t * nx + k0 + s : k0 + s)] = yf[s];
#pragma unroll
    for (int s = 0; s < H; ++s) if (qf[s] & Q_VALID) {
      const size_t row = (size_t)p * mg + t * ng + (qf[s] >> Q_ROW_SH);
      a.zg[row] = zg[s]; a.yg[row] = yg[s]; if (a.iters > 0) a.xi[row] = xi_last[s];
    }
  }
}

}  // namespace tmpc
