// tmpc_admm2.cuh — a4..a8 for the RESIDENT class (configs 1, 2, 4): the fused ADMM loop of Alg. 3
// on the twisted block factor of tmpc_factor2.cuh, all iterations in one launch.
//
// Design:
//  * a CTA owns PG problems (1 or 2).  The factor (X_t, -B_t) and the constraint blocks carried into the scaled
//    variables (A~^- = A^- X', A~^+ = A^+ X_next', G~ = G X') sit in shared memory for all iterations; the per-row ADMM
//    state (x, q, y_f, c, z_g, y_g, lo, hi) lives in REGISTERS of the thread that owns the row: two or three rows of
//    ONE stage per thread, fixed for the launch, so the stage's operand vectors are loaded once per thread (the
//    stage-parallel phases are bound by shared-memory wavefronts).
//  * x~ = S^{-1} eta (eq. 8) runs on a dedicated chain warp (warp 0): lanes = (problem, direction, row), 8 lanes per
//    slot, so the up chain and the down chain of the twisted factor of up to two problems advance together; a step is
//    one n x n mat-vec whose operand vector is published with one STS and read back as a broadcast vector load.
//  * everything local to a stage (eta eq. 51, z~ = A x~ eq. 9, relaxation eq. 10, projection eq. 12-15, duals eq. 16)
//    is done by the item warps; chain warp and item warps hand over through named barriers (arrive / sync), and
//    several CTAs per SM overlap one CTA's chain phase with another's stage-parallel phase.
//  * shared-memory layout is bank-conflict free for n = 8: rows of the blocks are XOR-swizzled by 16-byte chunks
//    (row-wise vector loads AND column-wise scalar loads), the record stride is 8 (mod 32) words, the down-chain
//    records are skewed by 8 words and the second problem by 16 so the four slots hit distinct banks.
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
//   AM  A~^-_t = A^-_t X_t'     [nx][n]   (zero for t = N)
//   AP  A~^+_{t-1} = A^+_{t-1} X_t' [nx][n] (A_init = [I 0] for t = 0: the rows x_0 = x_init are "dynamics block -1")
//   RM  r of block t      [nx]      r = rho_f c - y_f of the rows that AM belongs to
//   RP  r of block t-1    [nx]      (r_init for t = 0); written by the owner of that row together with RM of its own stage
//   E0  y_t               [n]       solution of the scaled system (x~_t = X_t' y_t)
//   E1  eta~_t -> w_t     [n]
//   D   sigma x - q + G's [n]       exchanged inside the stage for the X_t product
//   LAM -B_t              [n][n]    twisted factor, tmpc_factor2.cuh
//   SINV X_t = L_t^{-1}   [n][n]
//   S   s_t = rho_g z_g - y_g [n slots, ng used]   only when G is not a selection
//   G   G~_t = G_t X_t'   [ng][n]                  only when G is not a selection
// Rows of AM, AP, LAM, SINV are XOR-swizzled by 16-byte chunks for n = 8 (conflict-free row-wise vector loads AND
// column-wise scalar loads); the record stride is padded to 8 (mod 32) words so that the four stages a warp touches
// fall into distinct banks, records of the down chain are skewed by 8 words and the second problem by 16.
template <typename T, int NC, int NX>
struct Rec {
  static constexpr int V = 16 / (int)sizeof(T);
  static constexpr int up(int v) { return (v + V - 1) / V * V; }
  static constexpr int AM = 0, AP = AM + up(NX * NC), RM = AP + up(NX * NC), RP = RM + up(NX), E0 = RP + up(NX),
                       E1 = E0 + up(NC), D = E1 + up(NC), LAM = D + up(NC), SINV = LAM + up(NC * NC), S = SINV + up(NC * NC), G = S + up(NC);   // S, G: dense G only
  static constexpr int SKEW = NC == 8 ? 8 : 0;
};
struct Admm2Plan { int R, per_problem; };

template <typename T, int NC, int NX>
__host__ __device__ inline Admm2Plan admm2_plan(const Dims& d, int pg) {
  using RC = Rec<T, NC, NX>;
  Admm2Plan P;
  int R = d.g_sel ? RC::S : RC::G + RC::up(d.ng * NC);
  // four lanes per stage, eight stages per warp: a stride of 4 (mod 32) words (fp32) puts the eight stages' rows in distinct banks
  // (any stride = 4 mod 8 words: k R mod 32 runs through all multiples of 4 for k = 0..7)
  if (NC == 8) { while (R % 8 != 4) R += RC::V; }
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


// ---- explicit shared-state-space accesses on 32-bit addresses (byte units).  Going through generic pointers makes the
// compiler rebuild the shared window base (S2UR SR_CgaCtaId + ULEA, ~25 cycles) inside every chain step.
__device__ __forceinline__ void lds_vec8(unsigned a0, unsigned a1, float (&r)[8]) {   // two 16-byte chunks, issued together
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%8];\n\tld.shared.v4.f32 {%4,%5,%6,%7}, [%9];"
               : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]) : "r"(a0), "r"(a1));
}
__device__ __forceinline__ void lds_vec8(unsigned a0, unsigned a1, unsigned a2, unsigned a3, double (&r)[8]) {
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%8];\n\tld.shared.v2.f64 {%2,%3}, [%9];\n\tld.shared.v2.f64 {%4,%5}, [%10];\n\tld.shared.v2.f64 {%6,%7}, [%11];"
               : "=d"(r[0]), "=d"(r[1]), "=d"(r[2]), "=d"(r[3]), "=d"(r[4]), "=d"(r[5]), "=d"(r[6]), "=d"(r[7]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3));
}
__device__ __forceinline__ void lds_vec6(unsigned a, float (&r)[6]) {
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%6];\n\tld.shared.v2.f32 {%2,%3}, [%6+8];\n\tld.shared.v2.f32 {%4,%5}, [%6+16];"
               : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]) : "r"(a));
}
__device__ __forceinline__ void lds_vec6(unsigned a, double (&r)[6]) {
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%6];\n\tld.shared.v2.f64 {%2,%3}, [%6+16];\n\tld.shared.v2.f64 {%4,%5}, [%6+32];"
               : "=d"(r[0]), "=d"(r[1]), "=d"(r[2]), "=d"(r[3]), "=d"(r[4]), "=d"(r[5]) : "r"(a));
}
__device__ __forceinline__ float lds_1(unsigned a, float) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ double lds_1(unsigned a, double) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts_1(unsigned a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_1(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
// contiguous NC-vector at byte address a; for NC = 8 the 16-byte chunks are taken in the order of a row swizzled by swb bytes
template <typename T, int NC> __device__ __forceinline__ void lds_row(unsigned a, unsigned swb, T (&r)[NC]) {
  if constexpr (NC == 8 && sizeof(T) == 4) lds_vec8(a + swb, a + 16u - swb, r);     // swb in {0,16}: chunks (0,16) or (16,0), one add each
  else if constexpr (NC == 8) lds_vec8(a + (0u ^ swb), a + (16u ^ swb), a + (32u ^ swb), a + (48u ^ swb), r);
  else lds_vec6(a, r);
}

// empty asm that "uses" a whole register vector: keeps ptxas from splitting a multi-chunk load into load - use - load - use
template <int L> __device__ __forceinline__ void pin_vec(float (&r)[L]) {
  if constexpr (L == 8) asm volatile("" : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]), "+f"(r[4]), "+f"(r[5]), "+f"(r[6]), "+f"(r[7]));
  else if constexpr (L == 6) asm volatile("" : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]), "+f"(r[4]), "+f"(r[5]));
}
template <int L> __device__ __forceinline__ void pin_vec(double (&r)[L]) {
  if constexpr (L == 8) asm volatile("" : "+d"(r[0]), "+d"(r[1]), "+d"(r[2]), "+d"(r[3]), "+d"(r[4]), "+d"(r[5]), "+d"(r[6]), "+d"(r[7]));
  else if constexpr (L == 6) asm volatile("" : "+d"(r[0]), "+d"(r[1]), "+d"(r[2]), "+d"(r[3]), "+d"(r[4]), "+d"(r[5]));
}

// rows of one stage handled by a thread: 3 for fp32 n = 6 (three CTAs per SM leave 80 registers per thread only with
// 256-thread CTAs), else 2
template <typename T, int NC> __host__ __device__ constexpr int admm2_ipt() { return (NC == 6 && sizeof(T) == 4) ? 3 : 2; }

template <typename T>
struct Admm2Args {
  AdmmArgs<T> a;
  Admm2Plan pl;                       // host-computed: read straight from the constant bank, costs no registers
  T rfa, oma, inv_rho_g, inv_rg;      // rho_f alpha, 1 - alpha, 1 / rho_g, 1 / (rho_g + gamma)
};

// item flag bits
enum : unsigned { F_VALID = 1u, F_DYN = 2u, F_INEQ = 4u, F_SOFT = 8u, F_ROW_SH = 8 };

// named barriers: 1 = right-hand side ready (item warps arrive, chain warp waits), 2 = solution ready (chain warp
// arrives, item warps wait), 3 = item warps only
__device__ __forceinline__ void bar_sync(int id, int cnt) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(cnt) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int cnt) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(cnt) : "memory"); }

template <int L> __device__ __forceinline__ float dotv_from(const float (&a)[L], const float (&b)[L], float init) {
  // two independent FFMA2 chains, one per half of the vectors: the second instruction already needs the second half, so
  // ptxas issues all operand loads back to back instead of serialising load - use - load - use on recycled registers
  static_assert(L % 2 == 0, "even length");
  constexpr int H = (L / 4) * 2;                       // first half length (even)
  float2 p = make_float2(init, 0.f), q = make_float2(0.f, 0.f);
#pragma unroll
  for (int j = 0; j < H; j += 2) {
    p = __ffma2_rn(make_float2(a[j], a[j + 1]), make_float2(b[j], b[j + 1]), p);
    if (H + j + 1 < L) q = __ffma2_rn(make_float2(a[H + j], a[H + j + 1]), make_float2(b[H + j], b[H + j + 1]), q);
  }
  if constexpr (L - 2 * H > 0) q = __ffma2_rn(make_float2(a[L - 2], a[L - 1]), make_float2(b[L - 2], b[L - 1]), q);
  return (p.x + q.x) + (p.y + q.y);
}
template <int L> __device__ __forceinline__ double dotv_from(const double (&a)[L], const double (&b)[L], double init) {
  double acc[2] = {init, 0.0};
#pragma unroll
  for (int j = 0; j < L; ++j) acc[j & 1] += a[j] * b[j];
  return acc[0] + acc[1];
}

// ---- x~ = S^{-1} eta on the scaled variables (tmpc_factor2.cuh): E1 holds eta~ on entry and w on exit, E0 receives y.
// One warp; lanes = (problem, direction, row), 8 lanes per slot.  Every step is: publish my component (STS), read the
// 8-vector back as a broadcast vector load, one row (forward) or column (outward) of -B_t, one FFMA2 dot.
template <typename T, int NC, int NX, int PG>
__device__ __forceinline__ void chain_warp_solve(T* sm, int R, int PP, int T_, int lane) {
  static_assert(NC == 8 || NC == 6, "chain lanes are written for n = 6 and n = 8");
  using RC = Rec<T, NC, NX>;
  constexpr int n = NC;
  constexpr unsigned ES = sizeof(T);
  const unsigned sb = (unsigned)__cvta_generic_to_shared(sm);
  const int N = T_ - 1, m = T_ / 2;
  const int slot = lane >> 3, i8 = lane & 7;
  const int g = PG == 2 ? (slot >> 1) : 0, dir = slot & 1;
  const bool act = (PG == 2 || slot < 2) && i8 < n;
  const int ii = i8 < n ? i8 : 0;
  const unsigned swb = (unsigned)swz_x<T, NC>(ii) * ES;                 // my row's chunk swizzle, bytes
  const int cnt = act ? (dir ? T_ - 1 - m : m) : 0, t0 = dir ? N : 0;
  const int dRb = (dir ? -R : R) * (int)ES;
  auto rec = [&](int t) { return t * R + (t > m ? RC::SKEW : 0); };
  const unsigned pb = sb + (unsigned)(g * PP) * ES, bm = pb + (unsigned)rec(m) * ES;
  constexpr unsigned oE0 = RC::E0 * ES, oE1 = RC::E1 * ES, oLAM = RC::LAM * ES;
  const unsigned me = (unsigned)ii * ES, myrow = oLAM + (unsigned)(ii * n) * ES;
  unsigned bt = cnt > 0 ? pb + (unsigned)rec(t0) * ES : bm;
  T wv = cnt > 0 ? lds_1(bt + oE1 + me, T(0)) : T(0);
  T Br[n];
  lds_row<T, NC>(bt + myrow, 0u, Br);
  // steps in which every active slot is on and none is at its last stage run without per-lane predicates
  const int cmin = T_ - 1 - m;                          // = the down chain's length <= the up chain's (m)
  const int kmain = cmin > 1 ? cmin - 1 : 0;
  const int dRa = act ? dRb : 0;                        // idle lanes stay on record m
#pragma unroll 1
  for (int k = 0; k < kmain; ++k) {
    if (act) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    T W[n];
    lds_row<T, NC>(bt + oE1, swb, W);
    bt += dRa;
    const T eta = lds_1(bt + oE1 + me, T(0));
    T Bn[n];
    lds_row<T, NC>(bt + myrow, 0u, Bn);
    wv = dotv_from<n>(Br, W, eta);
#pragma unroll
    for (int j = 0; j < n; ++j) Br[j] = Bn[j];
  }
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
    lds_row<T, NC>(bt + myrow, 0u, Bn);                // next step's row (record m holds zeros: harmless)
    const T nw = dotv_from<n>(Br, W, eta);
    if (on) wv = nw;
#pragma unroll
    for (int j = 0; j < n; ++j) Br[j] = Bn[j];
  }
  // middle stage: w_m = eta~_m + both contributions; y_m = w_m
  const T wm = wv + __shfl_xor_sync(0xffffffffu, wv, 8);
  if (act) { sts_1(bm + oE1 + me, wm); sts_1(bm + oE0 + me, wm); }
  __syncwarp();
  // outward sweep: y_t = w_t + (-B_t)' y_next
  unsigned bc = cnt > 0 ? pb + (unsigned)rec(t0 + (cnt - 1) * (dir ? -1 : 1)) * ES : bm, bp = bm;
  unsigned colo[n];
#pragma unroll
  for (int j = 0; j < n; ++j) colo[j] = oLAM + (unsigned)(j * n + (ii ^ swz_x<T, NC>(j))) * ES;
#pragma unroll 1
  for (int k = m - 1; k >= 0; --k) {
    const bool on = k < cnt;
    T Y[n], col[n];
    lds_row<T, NC>(bp + oE0, 0u, Y);
#pragma unroll
    for (int j = 0; j < n; ++j) col[j] = lds_1(bc + colo[j], T(0));
    const T w = lds_1(bc + oE1 + me, T(0));
    const T y = dotv_from<n>(col, Y, w);
    if (on) { sts_1(bc + oE0 + me, y); bp = bc; bc -= dRb; }
    __syncwarp();
  }
}

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
  const int tid = threadIdx.x, nt = blockDim.x, nti = nt - 32, it_tid = tid - 32;
  const int m = T_ / 2;
  auto rec = [&](int t) { return t * R + (t > m ? RC::SKEW : 0); };
  auto sw = [&](int row, int col) { return row * n + (col ^ swz_x<T, NC>(row)); };

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
      const int t = e / nn, rc = e - t * nn, row = rc / n, col = rc - row * n;
      const int o = rec(t) + sw(row, col);
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
        const T* Xj = P + rec(t) + RC::SINV;
        T sa = T(0), sp = T(0);
        if (t < N) { const T* Mr = gAm + ((size_t)t * nx + k) * n; for (int l = 0; l <= j; ++l) sa += Mr[l] * Xj[sw(j, l)]; }
        if (t > 0) { const T* Mr = gAp + ((size_t)(t - 1) * nx + k) * n; for (int l = 0; l <= j; ++l) sp += Mr[l] * Xj[sw(j, l)]; }
        else if (k <= j) sp = Xj[sw(j, k)];             // A_init = [I 0]
        P[rec(t) + RC::AM + sw(k, j)] = sa;
        P[rec(t) + RC::AP + sw(k, j)] = sp;
      }
      if (!d.g_sel) {
        const T* gG = a.qp.G + a.qp.sG * p;
        for (int e = tid; e < T_ * ng * n; e += nt) {
          const int t = e / (ng * n), rc = e - t * ng * n, k = rc / n, j = rc - k * n;
          const T* Xj = P + rec(t) + RC::SINV; const T* Mr = gG + ((size_t)t * ng + k) * n;
          T sg = T(0);
          for (int l = 0; l <= j; ++l) sg += Mr[l] * Xj[sw(j, l)];
          P[rec(t) + RC::G + k * n + j] = sg;
        }
      }
    }
    __syncthreads();
  }

  // ================================================================ chain warp
  if (tid < 32) {
    const int iters = a.kkt_only ? 1 : a.iters;
#ifdef TMPC_TIMING
    long long tw = 0, ts = 0;
#endif
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#ifdef TMPC_TIMING
      const long long c0 = clock64();
#endif
      bar_sync(1, nt);
#ifdef TMPC_TIMING
      const long long c1 = clock64();
#endif
#ifndef TMPC_NO_CHAIN                                    // debug builds: measure the stage-parallel phases alone
      chain_warp_solve<T, NC, NX, PG>(sm, R, PP, T_, tid);
#endif
      __syncwarp();
#ifdef TMPC_TIMING
      tw += c1 - c0; ts += clock64() - c1;
#endif
      bar_arrive(2, nt);
    }
#ifdef TMPC_TIMING
    if (blockIdx.x == 0 && tid == 0) printf("chain warp: wait %lld solve %lld cycles per iteration\n", tw / iters, ts / iters);
#endif
    return;
  }

  // ================================================================ item warps
  // group exchange of a per-stage vector: the NC owners of a stage sit in one warp when NC = 8, else use the item barrier
  auto group_sync = [&]() { if constexpr (NC == 8) __syncwarp(); else bar_sync(3, nti); };
  // operand vector of stage record `base`, field `f`, in the chunk order of swizzled row `row`
  auto ld_operand = [&](int base, int f, int row, T (&w)[n]) {
    if constexpr (NC == 8) {
      const int swx = swz_x<T, NC>(row);
#pragma unroll
      for (int c = 0; c < n / V; ++c) { T part[V]; ld_vec<V>(sm + base + f + ((c * V) ^ swx), part);
#pragma unroll
        for (int e = 0; e < V; ++e) w[c * V + e] = part[e]; }
    } else ld_vec<n>(sm + base + f, w);
  };

  if (a.kkt_only) {                                    // xt <- S^{-1} eta : eta~ = X eta, solve, x = X' y
    for (int e = it_tid; e < PG * nz; e += nti) {
      const int g = e / nz, el = e - g * nz, t = el / n, i = el - t * n, p = blockIdx.x * PG + g;
      sm[g * PP + rec(t) + RC::D + i] = p < d.B ? a.x[(size_t)p * nz + el] : T(0);
    }
    bar_sync(3, nti);
    for (int e = it_tid; e < PG * nz; e += nti) {
      const int g = e / nz, el = e - g * nz, t = el / n, i = el - t * n, b = g * PP + rec(t);
      T xr[n], dv[n];
      ld_vec<n>(sm + b + RC::SINV + i * n, xr); ld_operand(b, RC::D, i, dv);
      sm[b + RC::E1 + i] = dotv<n>(xr, dv);
    }
    bar_arrive(1, nt);
    bar_sync(2, nt);
    for (int e = it_tid; e < PG * nz; e += nti) {
      const int g = e / nz, el = e - g * nz, t = el / n, i = el - t * n, b = g * PP + rec(t), p = blockIdx.x * PG + g;
      T xc[n], yv[n];
#pragma unroll
      for (int j = 0; j < n; ++j) xc[j] = sm[b + RC::SINV + sw(j, i)];
      ld_vec<n>(sm + b + RC::E0, yv);
      if (p < d.B) a.xi[(size_t)p * nz + el] = dotv<n>(xc, yv);
    }
    return;
  }
  // ---- per-thread items: (problem g, stage t, row i), two per thread, state in registers.
  // Item (t, i < nx) owns the equality row i of dynamics block t (t < N) or of the init block (t = N: A^- = 0 in record N,
  // A^+ = A_init in record 0).  Inequality row r of stage t is owned by item (t, g_col[r]) for a selection G (so that
  // G'(.) and G x~ touch only the owner's own component) and by item (t, r) for a dense G.
  // The two items of a thread are rows i0 and i0 + n/2 of the SAME stage, so the stage's operand vectors (y_t, y_{t+1},
  // r_t, r_{t-1}, the exchange vector) are loaded once per thread and serve both rows: the stage-parallel phases are bound
  // by shared-memory wavefronts (measured: 0.69 of 1.22 ms at config 2 with the chain switched off), not by issue.
  // A row's chunk swizzle is undone on the registers (compile-time half swap for rows >= n/2, plus one select level for
  // fp64 n = 8).  PAIR needs registers for the shared vectors: not so for fp32 n = 6 under the 56-register cap of three
  // CTAs per SM (measured 4.72 vs 4.44 ms at config 4), which keeps two rows of different stages per thread.
  constexpr int IPT = admm2_ipt<T, NC>(), HALF = NC / IPT;     // rows i0, i0 + HALF, .. of one stage per thread
  constexpr bool PAIR = true;
  static_assert(NC % IPT == 0 && (NC != 8 || IPT == 2), "rows per thread");
  const int per_p = T_ * HALF;                           // PAIR: threads per problem
  const int pr_g = it_tid / per_p, pr_rem = it_tid - pr_g * per_p, pr_t = pr_rem / HALF, pr_i0 = pr_rem - pr_t * HALF;
  auto item_g = [&](int u) { return PAIR ? pr_g : (it_tid + u * nti) / nz; };
  auto item_el = [&](int u) { return PAIR ? pr_t * n + pr_i0 + u * HALF : (it_tid + u * nti) - item_g(u) * nz; };
  unsigned fl[IPT]; int bt[IPT], bn[IPT], it_i[IPT];
  T x[IPT], q[IPT], yf[IPT], cv[IPT], zg[IPT], yg[IPT], lo[IPT], hi[IPT];
  T xi_last[IPT];                                        // slack of the last iteration, written back after the loop
#pragma unroll
  for (int u = 0; u < IPT; ++u) xi_last[u] = T(0);
  auto g_row = [&](int u) -> size_t {                    // global index of the inequality row of item u (recomputed: not kept live)
    return (size_t)(blockIdx.x * PG + item_g(u)) * mg + (item_el(u) / n) * ng + (int)((fl[u] >> F_ROW_SH) & 31u);
  };
#pragma unroll
  for (int u = 0; u < IPT; ++u) {
    const int g = item_g(u), el = item_el(u), t = el / n, i = el - t * n, p = blockIdx.x * PG + g;
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
      int r = -1;
      if (d.g_sel) {
#pragma unroll
        for (int rr = 0; rr < NC; ++rr) if (rr < ng && d.g_col[rr] == i) r = rr;   // static indices: no local copy of the array
      } else if (i < ng) r = i;
      if (r >= 0) {
        const size_t row = (size_t)p * mg + t * ng + r;
        fl[u] |= F_INEQ | ((unsigned)r << F_ROW_SH);
        lo[u] = a.qp.lo[row]; hi[u] = a.qp.hi[row]; yg[u] = a.yg[row];
        if (a.zg_given) zg[u] = a.zg[row];
        else if (a.iters == 0) a.xi[row] = T(0);
        if (a.soft_rows ? (a.soft_rows[row] != 0) : (((d.soft_mask >> r) & 1u) != 0)) fl[u] |= F_SOFT;
      }
    }
  }
  auto put_r = [&](int u) {                              // r = rho_f c - y_f, for both records that read it
    const T r = a.prm.rho_f * cv[u] - yf[u];
    sm[bt[u] + RC::RM + it_i[u]] = r; sm[bn[u] + RC::RP + it_i[u]] = r;
  };
  // z_g^0 = clip(G x^0, lo, hi) unless given (x-space, straight from the problem data); r, s
#pragma unroll
  for (int u = 0; u < IPT; ++u) if (fl[u] & F_VALID) sm[bt[u] + RC::D + it_i[u]] = x[u];
  bar_sync(3, nti);
#pragma unroll
  for (int u = 0; u < IPT; ++u) {
    if (fl[u] & F_INEQ) {
      if (!a.zg_given) {
        T gx;
        if (d.g_sel) gx = x[u];
        else {
          const T* gr = a.qp.G + a.qp.sG * (blockIdx.x * PG + item_g(u)) + ((size_t)(item_el(u) / n) * ng + it_i[u]) * n;
          gx = T(0);
          for (int j = 0; j < n; ++j) gx += gr[j] * sm[bt[u] + RC::D + j];
        }
        zg[u] = tmin(tmax(gx, lo[u]), hi[u]);
      }
      if (!d.g_sel) sm[bt[u] + RC::S + it_i[u]] = a.prm.rho_g * zg[u] - yg[u];
    }
    if (fl[u] & F_DYN) put_r(u);
  }
  bar_sync(3, nti);

#ifdef TMPC_TIMING
  long long t_eta = 0, t_wait = 0, t_proj = 0, t_bar3 = 0;
#endif
#pragma unroll 1
  for (int it = 0; it < a.iters; ++it) {
#ifdef TMPC_TIMING
    const long long c0 = clock64();
#endif
    // a4 in scaled variables: eta~ = X (sigma x - q + G's) + A~^-' r_t + A~^+' r_{t-1}   [+ G~' s for a dense G]   (eq. 51)
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
      if (!(fl[u] & F_VALID)) continue;
      T dd = a.prm.sigma * x[u] - q[u];
      if (d.g_sel && (fl[u] & F_INEQ)) dd += a.prm.rho_g * zg[u] - yg[u];
      sm[bt[u] + RC::D + it_i[u]] = dd;
    }
    group_sync();
    // operand vectors of my stage, once for both rows (natural order; a row's chunk swizzle is undone on the registers)
    auto for_row = [&](int u, const T (&nat)[n], T (&out)[n]) {       // natural order -> chunk order of row it_i[u] (see Rec)
#pragma unroll
      for (int j = 0; j < n; ++j) {
        if constexpr (NC != 8) out[j] = nat[j];
        else if constexpr (sizeof(T) == 4) out[j] = nat[j ^ (4 * u)];
        else out[j] = ((it_i[u] >> 1) & 1) ? nat[j ^ (4 * u) ^ 2] : nat[j ^ (4 * u)];      // fp64: chunks of two, swizzle (row >> 1) & 3
      }
    };
    if constexpr (PAIR) {
      if (fl[0] & F_VALID) {                           // both rows belong to the same (valid or padding) stage
        const int b = bt[0];
        T dnat[n], rm[nx], rp[nx];
        ld_vec<n>(sm + b + RC::D, dnat); ld_vec<nx>(sm + b + RC::RM, rm); ld_vec<nx>(sm + b + RC::RP, rp);
#pragma unroll
        for (int u = 0; u < IPT; ++u) {
          const int i = it_i[u];
          T xr[n], dv[n], am[nx], ap[nx];
          ld_vec<n>(sm + b + RC::SINV + i * n, xr);
          for_row(u, dnat, dv);
#pragma unroll
          for (int k = 0; k < nx; ++k) { am[k] = sm[b + RC::AM + sw(k, i)]; ap[k] = sm[b + RC::AP + sw(k, i)]; }
          T s = dotv<n>(xr, dv) + (dotv<nx>(am, rm) + dotv<nx>(ap, rp));
          if (!d.g_sel) for (int r = 0; r < ng; ++r) s += sm[b + RC::G + r * n + i] * sm[b + RC::S + r];
          sm[b + RC::E1 + i] = s;
        }
      }
    } else {
#pragma unroll
      for (int u = 0; u < IPT; ++u) {
        if (!(fl[u] & F_VALID)) continue;
        const int b = bt[u], i = it_i[u];
        T xr[n], dv[n], am[nx], ap[nx], rm[nx], rp[nx];
        ld_vec<n>(sm + b + RC::SINV + i * n, xr); ld_operand(b, RC::D, i, dv);
#pragma unroll
        for (int k = 0; k < nx; ++k) { am[k] = sm[b + RC::AM + sw(k, i)]; ap[k] = sm[b + RC::AP + sw(k, i)]; }
        ld_vec<nx>(sm + b + RC::RM, rm); ld_vec<nx>(sm + b + RC::RP, rp);
        T s = dotv<n>(xr, dv) + (dotv<nx>(am, rm) + dotv<nx>(ap, rp));
        if (!d.g_sel) for (int r = 0; r < ng; ++r) s += sm[b + RC::G + r * n + i] * sm[b + RC::S + r];
        sm[b + RC::E1 + i] = s;
      }
    }
#ifdef TMPC_TIMING
    const long long c1 = clock64();
#endif
    bar_arrive(1, nt);
    bar_sync(2, nt);
#ifdef TMPC_TIMING
    const long long c2 = clock64();
#endif
    // a7 + a8 on y: z~_f = A~^- y_t + A~^+ y_{t+1}, x~_i = X(:,i)' y_t, z~_g = x~_i or G~ y_t; relaxation (eq. 10),
    // projection (eq. 12-15), duals (eq. 16 / 44-45)
    if constexpr (PAIR) {
      if (fl[0] & F_VALID) {
        const int b = bt[0];
        T yv[n], ybn[n];
        ld_vec<n>(sm + b + RC::E0, yv);
        if (fl[0] & F_DYN) ld_vec<n>(sm + bn[0] + RC::E0, ybn);     // row i0 < n / IPT <= nx is a dynamics row whenever any is
#pragma unroll
        for (int u = 0; u < IPT; ++u) {
          const int i = it_i[u];
          T xc[n];
#pragma unroll
          for (int j = 0; j < n; ++j) xc[j] = sm[b + RC::SINV + sw(j, i)];
          const T xt = dotv<n>(xc, yv);
          if (fl[u] & F_DYN) {
            T am[n], ap[n], ya[n], yb[n];
            ld_vec<n>(sm + b + RC::AM + i * n, am); ld_vec<n>(sm + bn[u] + RC::AP + i * n, ap);
            for_row(u, yv, ya); for_row(u, ybn, yb);
            const T zt = dotv<n>(am, ya) + dotv<n>(ap, yb);
            yf[u] += A.rfa * (zt - cv[u]);
            put_r(u);
          }
          if (fl[u] & F_INEQ) {
            T ztg = xt;
            if (!d.g_sel) { T gr[n]; ld_vec<n>(sm + b + RC::G + i * n, gr); ztg = dotv<n>(gr, yv); }
            const T zh = a.prm.alpha * ztg + A.oma * zg[u];
            const T v = zh + yg[u] * A.inv_rho_g;
            T z, s;
            project_row<T>((fl[u] & F_SOFT) != 0, v, lo[u], hi[u], a.prm.rho_g, A.inv_rg, a.prm.lam, z, s);
            yg[u] += a.prm.rho_g * (zh - z);
            zg[u] = z;
            if (!d.g_sel) sm[b + RC::S + i] = a.prm.rho_g * z - yg[u];
            xi_last[u] = s;
          }
          x[u] = a.prm.alpha * xt + A.oma * x[u];
        }
      }
    } else {
#pragma unroll
      for (int u = 0; u < IPT; ++u) {
        if (!(fl[u] & F_VALID)) continue;
        const int b = bt[u], i = it_i[u];
        T xc[n], yv[n];
#pragma unroll
        for (int j = 0; j < n; ++j) xc[j] = sm[b + RC::SINV + sw(j, i)];
        ld_vec<n>(sm + b + RC::E0, yv);
        const T xt = dotv<n>(xc, yv);
        if (fl[u] & F_DYN) {
          T am[n], ap[n], ya[n], yb[n];
          ld_vec<n>(sm + b + RC::AM + i * n, am); ld_vec<n>(sm + bn[u] + RC::AP + i * n, ap);
          if constexpr (NC == 8 && sizeof(T) == 4) {      // y_t is already in registers (yv): permute instead of reloading
            const bool sw4 = swz_x<T, NC>(i) != 0;
#pragma unroll
            for (int j = 0; j < n; ++j) ya[j] = sw4 ? yv[j ^ 4] : yv[j];
          } else ld_operand(b, RC::E0, i, ya);
          ld_operand(bn[u], RC::E0, i, yb);
          const T zt = dotv<n>(am, ya) + dotv<n>(ap, yb);
          yf[u] += A.rfa * (zt - cv[u]);
          put_r(u);
        }
        if (fl[u] & F_INEQ) {
          T ztg = xt;
          if (!d.g_sel) { T gr[n]; ld_vec<n>(sm + b + RC::G + i * n, gr); ztg = dotv<n>(gr, yv); }
          const T zh = a.prm.alpha * ztg + A.oma * zg[u];
          const T v = zh + yg[u] * A.inv_rho_g;
          T z, s;
          project_row<T>((fl[u] & F_SOFT) != 0, v, lo[u], hi[u], a.prm.rho_g, A.inv_rg, a.prm.lam, z, s);
          yg[u] += a.prm.rho_g * (zh - z);
          zg[u] = z;
          if (!d.g_sel) sm[b + RC::S + i] = a.prm.rho_g * z - yg[u];
          xi_last[u] = s;
        }
        x[u] = a.prm.alpha * xt + A.oma * x[u];
      }
    }
#ifdef TMPC_TIMING
    const long long c3 = clock64();
#endif
    bar_sync(3, nti);
#ifdef TMPC_TIMING
    t_eta += c1 - c0; t_wait += c2 - c1; t_proj += c3 - c2; t_bar3 += clock64() - c3;
#endif
  }
#ifdef TMPC_TIMING
  if (blockIdx.x == 0 && (tid == 32 || tid == nt - 32)) printf("item warp %d: eta %lld wait %lld proj %lld bar3 %lld cycles per iteration\n", tid >> 5, t_eta / a.iters, t_wait / a.iters, t_proj / a.iters, t_bar3 / a.iters);
#endif

  // ---- write back the state
#pragma unroll
  for (int u = 0; u < IPT; ++u) {
    if (!(fl[u] & F_VALID)) continue;
    const int el = item_el(u), t = el / n, i = it_i[u], p = blockIdx.x * PG + item_g(u);
    a.x[(size_t)p * nz + el] = x[u];
    if (fl[u] & F_DYN) a.yf[(size_t)p * mf + (t < N ? nx + t * nx + i : i)] = yf[u];
    if (fl[u] & F_INEQ) { const size_t row = g_row(u); a.zg[row] = zg[u]; a.yg[row] = yg[u]; if (a.iters > 0) a.xi[row] = xi_last[u]; }
  }
}

// ---- a9: residuals (eq. 3) and objective at the iterate in global memory; one CTA per problem
template <typename T>
struct ResidualArgs {
  Dims d; Params<T> prm; QpView<T> qp;
  const T* x; const T* zg; const T* yf; const T* yg; const T* xi;
  T* r_prim; T* r_dual; T* objective; int32_t* status;
  double* partial; int nparts;          // nparts > 1: gridDim.y CTAs per problem write partials, residual_finish_kernel reduces them in a fixed order
  // f1: optional scales of the termination test eq. 4: norm_prim = |(Ax, z)|_inf, norm_dual = |(Px, A'y, q, gamma xi,
  // y_g on soft rows)|_inf, [B] each (single-part launches only), and the activity flags (terminated problems keep their last values)
  T* norm_prim; T* norm_dual;
  const int32_t* active;
};

template <typename T>
__global__ void __launch_bounds__(256) residual_kernel(ResidualArgs<T> a) {
  __shared__ T red[64];
  const Dims& d = a.d;
  const int n = d.n, nx = d.nx, ng = d.ng, N = d.N, nn = n * n, nz = d.nz, mf = d.mf, mg = d.mg;
  const int p = blockIdx.x, nt = blockDim.x * gridDim.y, tid = blockIdx.y * blockDim.x + threadIdx.x;   // parts interleave
  if (a.active && !a.active[p]) return;
  const T gam = a.prm.gamma, lam = a.prm.lam;
  T nrp = T(0), nrd = T(0);
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
    rp = tmax(rp, tabs(cx - c)); nrp = tmax(nrp, tmax(tabs(cx), tabs(c)));
  }
  for (int e = tid; e < mg; e += nt) {
    const int t = e / ng, r = e - t * ng;
    T gx;
    if (d.g_sel) gx = x[t * n + d.g_col[r]];
    else { const T* g = G + ((size_t)t * ng + r) * n; gx = T(0); for (int j = 0; j < n; ++j) gx += g[j] * x[t * n + j]; }
    rp = tmax(rp, tabs(gx - zg[e])); nrp = tmax(nrp, tmax(tabs(gx), tabs(zg[e])));
    if ((d.soft_mask >> r) & 1u) nrd = tmax(nrd, tmax(tabs(gam * xi[e]), tabs(yg[e])));
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
    T g = T(0);                                        // A'y = C'y_f + G'y_g
    if (t == 0 && i < nx) g += yf[i];
    if (t < N) { const T* A_ = Am + (size_t)t * nx * n + i; for (int k = 0; k < nx; ++k) g += A_[k * n] * yf[nx + t * nx + k]; }
    if (t > 0) { const T* A_ = Ap + (size_t)(t - 1) * nx * n + i; for (int k = 0; k < nx; ++k) g += A_[k * n] * yf[nx + (t - 1) * nx + k]; }
    if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) g += yg[t * ng + r]; }
    else { const T* gg = G + (size_t)t * ng * n + i; for (int r = 0; r < ng; ++r) g += gg[r * n] * yg[t * ng + r]; }
    nrd = tmax(nrd, tmax(tabs(px), tmax(tabs(g), tabs(q[e]))));
    rd = tmax(rd, tabs(px + q[e] + g));
    ob += T(0.5) * x[e] * px + q[e] * x[e];
    if (!isfinite(x[e])) bad = 1;
  }
  rp = block_max(rp, red); rd = block_max(rd, red); ob = block_sum(ob, red);
  if (a.norm_prim) { nrp = block_max(nrp, red); nrd = block_max(nrd, red); if (threadIdx.x == 0) { a.norm_prim[p] = nrp; a.norm_dual[p] = nrd; } }
  bad = __syncthreads_or(bad);
  if (threadIdx.x == 0) {
    if (a.nparts > 1) { double* o = a.partial + ((size_t)p * a.nparts + blockIdx.y) * 4; o[0] = (double)rp; o[1] = (double)rd; o[2] = (double)ob; o[3] = bad ? 1.0 : 0.0; return; }
    if (a.r_prim) a.r_prim[p] = rp;
    if (a.r_dual) a.r_dual[p] = rd;
    if (a.objective) a.objective[p] = ob;
    if (a.status && bad) atomicOr(&a.status[p], TMPC_ST_NAN);
  }
}

template <typename T>
__global__ void residual_finish_kernel(ResidualArgs<T> a) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= a.d.B) return;
  double rp = 0, rd = 0, ob = 0; bool bad = false;
  for (int k = 0; k < a.nparts; ++k) { const double* o = a.partial + ((size_t)p * a.nparts + k) * 4; rp = fmax(rp, o[0]); rd = fmax(rd, o[1]); ob += o[2]; bad |= o[3] != 0.0; }
  if (a.r_prim) a.r_prim[p] = (T)rp;
  if (a.r_dual) a.r_dual[p] = (T)rd;
  if (a.objective) a.objective[p] = (T)ob;
  if (a.status && bad) atomicOr(&a.status[p], TMPC_ST_NAN);
}

// ---- f1: the decisions at a scheduled check (eq. 4 and eq. 17), one thread per problem, in double.
struct AdaptParams { int k, last, adapt_rho; double eps_abs, eps_rel, ratio, rho_min, rho_max; };
template <typename T>
__global__ void adapt_kernel(int B, AdaptParams ap, const T* __restrict__ r_prim, const T* __restrict__ r_dual, const T* __restrict__ norm_prim,
                             const T* __restrict__ norm_dual, T* __restrict__ rho_bar, int32_t* __restrict__ active, int32_t* __restrict__ mask,
                             int32_t* __restrict__ iters, int32_t* __restrict__ converged, int32_t* __restrict__ n_active) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= B) return;
  mask[p] = 0;
  if (!active[p]) return;
  iters[p] = ap.k;
  const double rp = (double)r_prim[p], rd = (double)r_dual[p], np_ = (double)norm_prim[p], nd_ = (double)norm_dual[p];
  if (rp <= ap.eps_abs + ap.eps_rel * np_ && rd <= ap.eps_abs + ap.eps_rel * nd_) { active[p] = 0; converged[p] = 1; return; }
  if (ap.last) { active[p] = 0; return; }
  atomicAdd(n_active, 1);
  if (ap.adapt_rho && rd > 0.0 && np_ > 0.0 && nd_ > 0.0) {
    const double rho = (double)rho_bar[p];
    double cand = rho * sqrt((rp / np_) / (rd / nd_));
    cand = fmin(fmax(cand, ap.rho_min), ap.rho_max);
    if (fmax(cand / rho, rho / cand) > ap.ratio) { rho_bar[p] = (T)cand; mask[p] = 1; }
  }
}
template <typename T>
__global__ void adapt_init_kernel(int B, T rho0, T* rho_bar, int32_t* active, int32_t* mask, int32_t* iters, int32_t* converged, int32_t* n_active) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p == 0) *n_active = 0;
  if (p < B) { rho_bar[p] = rho0; active[p] = 1; mask[p] = 0; iters[p] = 0; converged[p] = 0; }
}

}  // namespace tmpc
