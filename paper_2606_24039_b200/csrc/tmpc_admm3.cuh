// tmpc_admm3.cuh — a4..a8 for the RESIDENT class, second generation (round 2): the fused ADMM loop of Alg. 3
// on the twisted block factor of tmpc_factor2.cuh, all iterations in one launch.
//
// What changed against round 1's admm2_kernel, and why (ncu of admm2 at config 2: 62 % of the warp samples wait at a barrier, the
// LSU pipe carries 1435 shared-memory wavefronts per problem-iteration = 52 % of its peak, 23 % of them excess):
//  * TWO lanes per stage instead of four.  Lane h of a stage owns the columns [h n/2, (h+1) n/2) of every block of
//    the stage record, the same rows of the stage variable, and half of the dynamics / inequality rows.  Every matrix
//    access is then a vector load of "my column chunk of row k" (products with a transposed block: A~' r, X' y, G~' s)
//    or of a full row taken "my chunk first, the partner's second" (X d, A~ y, G~ y) — no scalar column loads, every
//    block element is read exactly once per use and no operand vector is loaded by four threads.
//  * the stage vector d = sigma x - q + G's and r = rho_f c - y_f are exchanged between the two lanes of a stage with
//    shuffles; nothing but eta~ and y goes through shared memory between the item warps and the chain warp.
//  * ONE stage-parallel phase per iteration instead of two with a CTA-wide barrier in between: the owner of dynamics
//    block t adds A~^-_t' r_t to its own stage (field E1A) and A~^+_t' r_t to the NEXT stage (field E1B of record t+1),
//    so no thread reads another stage's r; the chain warp consumes eta~ = E1A + E1B.
//  * the records are NOT swizzled: with a record stride of 8 (mod 32) words the eight lanes of a quarter warp (four
//    stages x two halves) hit the eight distinct 16-byte bank groups in every access pattern above, and so do the eight
//    lanes of a chain slot once rows >= n/2 take their two chunks in the opposite order (admm2's 2-way conflict).
//  * the chain warp's loops are unrolled by two with the row / column buffers swapping roles (no register copies inside
//    the dependent chain), and the outward sweep prefetches the next stage's column of B and w one step ahead.
// The named-barrier handshake (1: right-hand side ready, 2: solution ready) is that of admm2.
#pragma once
#include "tmpc_common.cuh"
#include "tmpc_admm.cuh"
#include "tmpc_admm2.cuh"

namespace tmpc {

// ---- shared-memory record of one stage (elements of T), rows stored unswizzled:
//   AM  A~^-_t = A^-_t X_t'          [nx][n]   (zero for t = N)
//   AP  A~^+_{t-1} = A^+_{t-1} X_t'  [nx][n]   (A_init = [I 0] for t = 0: the rows x_0 = x_init are "dynamics block -1",
//                                               owned by the lanes of stage N)
//   E0  y_t [n]      E1A  eta~_t (own part) -> w_t [n]      E1B  eta~_t (part of the block before) [n]
//   LAM -B_t [n][n]  SINV X_t = L_t^{-1} [n][n]
//   G   G~_t = G_t X_t' [ng][n]      (dense G only; s_t = rho_g z_g - y_g lives in the registers of the row owners)
// XG ("X and A~ in global memory", long horizons): the record keeps only what the CHAIN warp reads — y, eta~ / w and -B_t — and the item
// lanes take X_t, A~^-_t, A~^+_t (G~_t) from global memory, from the stage-minor scratch atil_kernel fills (ld_half_g), where they are L2
// hits: the chain is the latency-bound part, the item phases are throughput-bound and tolerate the longer loads.
template <typename T, int NC, int NX, bool XG = false>
struct Rec3 {
  static constexpr int V = 16 / (int)sizeof(T);
  static constexpr int up(int v) { return (v + V - 1) / V * V; }
  static constexpr int AM = 0, AP = AM + (XG ? 0 : up(NX * NC)), E0 = AP + (XG ? 0 : up(NX * NC)), E1A = E0 + up(NC), E1B = E1A + up(NC),
                       LAM = E1B + up(NC), SINV = LAM + up(NC * NC), G = SINV + (XG ? 0 : up(NC * NC));
  // record stride: 32 bytes (mod 128 bytes) for the 16-byte accesses of n = 8 (a quarter warp = four stages x two halves covers
  // the eight bank groups); 24 bytes (mod 128) for the 6-wide rows of n = 6, whose 8-byte pairs and single elements cannot all
  // be conflict free: this residue makes the single-element loads conflict free and the pair loads 2-way (simulated over all
  // residues; 32 bytes gives 4-way and 8-way)
  static constexpr int pad_stride(int r) {
    if (XG) return r;                                      // the item lanes touch only the three vectors of a record: no residue to protect
    constexpr bool SIX32 = NC == 6 && sizeof(T) == 4;      // (double keeps 32 bytes: its pairs are 16-byte loads)
    constexpr int W128 = 128 / (int)sizeof(T), WR = (SIX32 ? 24 : 32) / (int)sizeof(T), STEP = SIX32 ? 2 : V;
    while (r % W128 != WR) r += STEP;
    return r;
  }
};
// Placement of the records of one problem: stages 0..m (the up chain and the middle) at t R; stages m+1..N (the down chain) in REVERSE
// order from `down0`, i.e. stage t at down0 + (N - t) R, so that step k of both chains sits at (k R) and (down0 + k R): with
// down0 = 64 bytes (mod 128) and the second problem of a CTA another 32 bytes off, the four slots of the chain warp read four disjoint
// 8-bank windows at every step, for any record stride (n = 6 and n = 8 alike).
struct Admm3Plan { int R, down0, per_problem; };

template <typename T, int NC, int NX, bool XG = false>
inline Admm3Plan admm3_plan(const Dims& d, int pg) {
  using RC = Rec3<T, NC, NX, XG>;
  Admm3Plan P;
  int R = (d.g_sel || XG) ? RC::G : RC::G + ((d.ng * NC + RC::V - 1) / RC::V) * RC::V;
  P.R = RC::pad_stride(R);
  const int w128 = 128 / (int)sizeof(T), w64 = 64 / (int)sizeof(T), w32 = 32 / (int)sizeof(T), m = d.T / 2;
  int d0 = ((m + 1) * P.R + RC::V - 1) / RC::V * RC::V;
  while (d0 % w128 != w64) d0 += RC::V;
  P.down0 = d0;
  int pp = (d0 + (d.T - 1 - m) * P.R + RC::V - 1) / RC::V * RC::V;
  if (pg == 2) { while (pp % w128 != w32) pp += RC::V; }
  P.per_problem = pp;
  return P;
}
template <typename T, int NC, int NX, bool XG = false>
inline size_t admm3_smem_bytes(const Dims& d, int pg) { return (size_t)admm3_plan<T, NC, NX, XG>(d, pg).per_problem * pg * sizeof(T); }

// Cluster variant (CL): per CTA the records of its half (+ the zero record that stands in for the middle stage in the down CTA), the mailbox of
// the middle exchange and three mbarriers (mid, eta, y).  down0 = 0: each CTA stores its own half from offset 0.
template <typename T, int NC, int NX, bool XG>
inline Admm3Plan admm3_cl_plan(const Dims& d) {
  using RC = Rec3<T, NC, NX, XG>;
  Admm3Plan P;
  P.R = RC::pad_stride((d.g_sel || XG) ? RC::G : RC::G + RC::up(d.ng * NC)); P.down0 = 0;
  const int m = d.T / 2, nrecs = (m + 1 > d.T - m) ? m + 1 : d.T - m;
  P.per_problem = RC::up(nrecs * P.R) + RC::up(NC);      // records + mailbox (zero-filled by the prologue); the mbarriers follow
  return P;
}
template <typename T, int NC, int NX, bool XG>
inline size_t admm3_cl_smem_bytes(const Dims& d) { return (size_t)admm3_cl_plan<T, NC, NX, XG>(d).per_problem * sizeof(T) + 32; }

template <typename T>
struct Admm3Args {
  AdmmArgs<T> a;
  Admm3Plan pl;
  const T* atil;                      // XG only: X, A~^-, A~^+ and (dense G) G~ of every stage in the stage-minor layout atil_kernel writes
  int tpad;                           // ... whose chunk stride is tpad * V elements (tpad = T rounded up to 8 stages)
  T rfa, oma, inv_rho_g, inv_rg;      // rho_f alpha, 1 - alpha, 1 / rho_g, 1 / (rho_g + gamma)
};

// ---- a lane's half of an n-wide row.  Half h holds H = n/2 columns in its LOCAL slot order:
//   n = 8:  slots (0,1,2,3) = columns 4h + (0,1,2,3): one 16-byte load (two for double);
//   n = 6:  slots (0,1,2)   = columns (0,1,2) for h = 0 and (4,5,3) for h = 1: the aligned pair at 4h and the single
//           element at 2 + h, so both halves execute the same two instructions and no select is needed; every per-column
//           array of a lane (state, operand halves, accumulators) lives in this slot order.
template <int NC> __device__ __forceinline__ constexpr int slot_col(int h, int s) { return NC == 6 ? (h ? (s < 2 ? 4 + s : 3) : s) : h * (NC / 2) + s; }
struct HalfOff { int pair, single; };                                         // element offsets of a half inside a row
template <int NC> __device__ __forceinline__ HalfOff half_off(int h) { HalfOff o; o.pair = NC == 6 ? 4 * h : h * (NC / 2); o.single = NC == 6 ? 2 + h : 0; return o; }

//   other even n (n = 12): slots = columns h n/2 + s, loaded in the widest aligned vectors (8 bytes for a 24-byte half, else 16)
template <int NC> __device__ __forceinline__ void ld_half(const float* __restrict__ row, const HalfOff& o, float (&r)[NC / 2]) {
  constexpr int H = NC / 2;
  if constexpr (NC == 6) { const float2 v = *reinterpret_cast<const float2*>(row + o.pair); r[0] = v.x; r[1] = v.y; r[2] = row[o.single]; }
  else if constexpr (H % 4 == 0) {
#pragma unroll
    for (int c = 0; c < H / 4; ++c) { const float4 v = reinterpret_cast<const float4*>(row + o.pair)[c]; r[4 * c] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w; }
  } else {
    static_assert(H % 2 == 0, "half rows of floats in 8-byte vectors");
#pragma unroll
    for (int c = 0; c < H / 2; ++c) { const float2 v = reinterpret_cast<const float2*>(row + o.pair)[c]; r[2 * c] = v.x; r[2 * c + 1] = v.y; }
  }
}
template <int NC> __device__ __forceinline__ void ld_half(const double* __restrict__ row, const HalfOff& o, double (&r)[NC / 2]) {
  constexpr int H = NC / 2;
  if constexpr (NC == 6) { const double2 v = *reinterpret_cast<const double2*>(row + o.pair); r[0] = v.x; r[1] = v.y; r[2] = row[o.single]; }
  else {
    static_assert(H % 2 == 0, "half rows of doubles in 16-byte vectors");
#pragma unroll
    for (int c = 0; c < H / 2; ++c) { const double2 v = reinterpret_cast<const double2*>(row + o.pair)[c]; r[2 * c] = v.x; r[2 * c + 1] = v.y; }
  }
}
template <int NC> __device__ __forceinline__ void st_half(float* __restrict__ row, const HalfOff& o, const float (&r)[NC / 2]) {
  constexpr int H = NC / 2;
  if constexpr (NC == 6) { *reinterpret_cast<float2*>(row + o.pair) = make_float2(r[0], r[1]); row[o.single] = r[2]; }
  else if constexpr (H % 4 == 0) {
#pragma unroll
    for (int c = 0; c < H / 4; ++c) reinterpret_cast<float4*>(row + o.pair)[c] = make_float4(r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
  } else {
#pragma unroll
    for (int c = 0; c < H / 2; ++c) reinterpret_cast<float2*>(row + o.pair)[c] = make_float2(r[2 * c], r[2 * c + 1]);
  }
}
template <int NC> __device__ __forceinline__ void st_half(double* __restrict__ row, const HalfOff& o, const double (&r)[NC / 2]) {
  constexpr int H = NC / 2;
  if constexpr (NC == 6) { *reinterpret_cast<double2*>(row + o.pair) = make_double2(r[0], r[1]); row[o.single] = r[2]; }
  else {
#pragma unroll
    for (int c = 0; c < H / 2; ++c) reinterpret_cast<double2*>(row + o.pair)[c] = make_double2(r[2 * c], r[2 * c + 1]);
  }
}
// acc[s] += m[s] * w for a half (packed FFMA2 for float)
template <int H> __device__ __forceinline__ void axpy_half(float (&acc)[H], const float (&m)[H], float w) {
#pragma unroll
  for (int s = 0; s + 1 < H; s += 2) { const float2 r = __ffma2_rn(make_float2(m[s], m[s + 1]), make_float2(w, w), make_float2(acc[s], acc[s + 1])); acc[s] = r.x; acc[s + 1] = r.y; }
  if constexpr (H % 2) acc[H - 1] = fmaf(m[H - 1], w, acc[H - 1]);
}
template <int H> __device__ __forceinline__ void axpy_half(double (&acc)[H], const double (&m)[H], double w) {
#pragma unroll
  for (int s = 0; s < H; ++s) acc[s] = fma(m[s], w, acc[s]);
}
__device__ __forceinline__ float shfl_x1(float v) { return __shfl_xor_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_x1(double v) { return __shfl_xor_sync(0xffffffffu, v, 1); }
// full-row product: first half of the row with my half of the operand, second half with the partner's
template <typename T, int H> __device__ __forceinline__ T dot2(const T (&a)[H], const T (&x)[H], const T (&b)[H], const T (&y)[H]) {
  return dotv<H>(a, x) + dotv<H>(b, y);
}

// ---- the same half rows from the STAGE-MINOR global scratch of the chain-resident variants (XG): element e of a row lives at
// row + (e / V) cs + e % V with V = 16 / sizeof(T) elements per 16-byte chunk and cs the chunk stride (all stages of a problem side by side), so
// that the lanes of a warp — consecutive stages — read consecutive 16-byte chunks: a warp-wide load is two contiguous runs (one per half)
// instead of 32 scattered half rows (measured: the scattered form ran at one 32-byte sector per cycle and made the stage-parallel phases
// 75 % of an iteration).
template <int NC> __device__ __forceinline__ void ld_half_g(const float* __restrict__ row, const HalfOff& o, float (&r)[NC / 2], int cs) {
  constexpr int H = NC / 2;
  if constexpr (NC == 6) { const float2 v = *reinterpret_cast<const float2*>(row + (o.pair >> 2) * cs); r[0] = v.x; r[1] = v.y; r[2] = row[o.single]; }
  else if constexpr (H % 4 == 0) {
#pragma unroll
    for (int c = 0; c < H / 4; ++c) { const float4 v = *reinterpret_cast<const float4*>(row + ((o.pair >> 2) + c) * cs); r[4 * c] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w; }
  } else {
#pragma unroll
    for (int c = 0; c < H / 2; ++c) { const int e = o.pair + 2 * c; const float2 v = *reinterpret_cast<const float2*>(row + (e >> 2) * cs + (e & 3)); r[2 * c] = v.x; r[2 * c + 1] = v.y; }
  }
}
template <int NC> __device__ __forceinline__ void ld_half_g(const double* __restrict__ row, const HalfOff& o, double (&r)[NC / 2], int cs) {
  constexpr int H = NC / 2;
  if constexpr (NC == 6) { const double2 v = *reinterpret_cast<const double2*>(row + (o.pair >> 1) * cs); r[0] = v.x; r[1] = v.y; r[2] = row[(o.single >> 1) * cs + (o.single & 1)]; }
  else {
#pragma unroll
    for (int c = 0; c < H / 2; ++c) { const double2 v = *reinterpret_cast<const double2*>(row + ((o.pair >> 1) + c) * cs); r[2 * c] = v.x; r[2 * c + 1] = v.y; }
  }
}

// ---- x~ = S^{-1} eta on the scaled variables (tmpc_factor2.cuh): E1A + E1B hold eta~ on entry, E1A holds w on exit, E0
// receives y.  One warp; lanes = (problem, direction, row), 8 lanes per slot.  Every step is: publish my component (STS),
// read the vector back as a broadcast vector load, one row (inward sweep) or column (outward sweep) of -B_t, one dot.
// Row i >= n/2 takes its 16-byte chunks in the opposite order (`swb`; the data is not swizzled) so that the eight rows of a
// slot cover the eight bank groups; the broadcast operand vector is read in the same order.
// ---- CL ("cluster"): one problem on a thread-block CLUSTER of two CTAs, for horizons whose chain share outgrows one SM.  The twisted factor
// splits the work by construction: CTA 0 holds the records of stages 0..m and runs the up chain, CTA 1 holds m+1..N (in reverse order) and runs
// the down chain.  They meet three times per iteration, each time through distributed shared memory and an mbarrier in the RECEIVER's CTA:
//   eta:  the item lanes of the boundary stage write their share of the neighbour's right-hand side (E1B of record m+1 resp. 0) remotely;
//   mid:  the down chain sends its contribution to the middle stage into CTA 0's mailbox, CTA 0 returns y_m into CTA 1's mailbox;
//   y:    each chain tells the neighbour's boundary lanes that its y's are complete (they read y_{m+1} resp. y_0 remotely in the second phase).
// Ordering of the remote fields across iterations (each mbarrier completes one phase per iteration, parity = iteration & 1):
//   * a boundary lane writes the neighbour's E1B for iteration k+1 only after its own second phase of iteration k, which waited for `y` of
//     iteration k, i.e. for the neighbour's chain to have consumed iteration k's right-hand side;
//   * a chain warp starts iteration k+1 (and overwrites its y's, its mailbox partner's contents) only after `eta` of iteration k+1, which the
//     neighbour's boundary lanes send after their second phase of iteration k — their remote reads of y are done, and the neighbour's chain
//     warp, having passed its named barrier 2 of iteration k before those lanes could, is done with both mailboxes;
//   * the first remote access of the kernel comes after the cluster barrier that follows the prologue, the last one before the cluster barrier
//     at exit.
struct ClCtx { int rank; unsigned box, mb_mid, r_box, r_mb_mid, parity; };   // shared-window addresses: my mailbox / mbarrier, the partner's (shared::cluster)
__device__ __forceinline__ unsigned cl_rank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned cl_map(unsigned saddr, unsigned rank) { unsigned r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank)); return r; }
__device__ __forceinline__ void cl_sync() { asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl_mbar_init(unsigned a, unsigned cnt) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(cnt) : "memory"); }
__device__ __forceinline__ void cl_arrive_remote(unsigned ra) { asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(ra) : "memory"); }
__device__ __forceinline__ void cl_wait(unsigned a, unsigned parity) {
  unsigned ok;
  do { asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(a), "r"(parity) : "memory"); } while (!ok);
}
__device__ __forceinline__ void cl_sts(unsigned ra, float v) { asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(ra), "f"(v) : "memory"); }
__device__ __forceinline__ void cl_sts(unsigned ra, double v) { asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(ra), "d"(v) : "memory"); }

template <typename T, int NC, int NX, int PG, bool XG = false, bool CL = false>
__device__ __forceinline__ void chain3_solve(T* sm, int R, int DOWN0, int PP, int T_, int lane, unsigned pmask, const ClCtx cl = ClCtx()) {   // pmask: bit g = problem g of the CTA is live
  constexpr int SL = NC <= 8 ? 8 : 16;                   // lanes per slot (one per row)
  static_assert(NC <= 16 && PG * 2 * SL <= 32, "the chain warp holds (problems x 2 directions) slots of SL lanes");
  static_assert(!CL || PG == 1, "the cluster variant keeps one problem per CTA pair");
  using RC = Rec3<T, NC, NX, XG>;
  constexpr int n = NC;
  constexpr unsigned ES = sizeof(T);
  const unsigned sb = (unsigned)__cvta_generic_to_shared(sm);
  const int N = T_ - 1, m = T_ / 2;
  // Lanes without a chain of their own (rows >= n of a slot, the upper half warp when the CTA holds one problem, a terminated problem)
  // still walk the records of a live-looking slot and load from them — the SAME addresses as that slot's lanes, i.e. pure broadcasts that
  // cost no extra shared-memory wavefront (ncu: parked on the middle record they collided with the working lanes) — but never store.
  const int slot = (lane / SL) % (2 * PG), i8 = lane % SL;
  const int g = PG == 2 ? (slot >> 1) : 0, dir = CL ? cl.rank : (slot & 1);           // CL: every slot mirrors slot 0, which runs this CTA's direction
  const bool live = (CL ? lane < SL : lane < 2 * PG * SL) && i8 < n && ((pmask >> g) & 1u);
  const int ii = i8 < n ? i8 : 0;
  const unsigned swb = (unsigned)swz_x<T, NC>(ii) * ES;                 // chunk ORDER of my row (bytes)
  const int cnt = dir ? T_ - 1 - m : m, t0 = dir ? N : 0;
  const int dRb = R * (int)ES;                           // both chains advance by +R per step (the down half is stored in reverse order)
  auto rec = [&](int t) { return t > m ? DOWN0 + (N - t) * R : t * R; };
  // CL, down CTA: the middle stage lives in the partner; a zero record behind the cnt records of this CTA stands in for it
  const unsigned pb = sb + (unsigned)(g * PP) * ES, bm = pb + (unsigned)((CL && dir) ? cnt * R : rec(m)) * ES;
  constexpr unsigned oE0 = RC::E0 * ES, oE1 = RC::E1A * ES, oE1B = RC::E1B * ES, oLAM = RC::LAM * ES;
  const unsigned me = (unsigned)ii * ES, myrow = oLAM + (unsigned)(ii * n) * ES;
  auto ld_eta = [&](unsigned base) { return lds_1(base + oE1 + me, T(0)) + lds_1(base + oE1B + me, T(0)); };
  unsigned bt = cnt > 0 ? pb + (unsigned)rec(t0) * ES : bm;
  T wv = cnt > 0 ? ld_eta(bt) : T(0);
  T Br[n];
  lds_row<T, NC>(bt + myrow, swb, Br);
  const int cmin = CL ? cnt : T_ - 1 - m;               // = the down chain's length <= the up chain's (m); CL: this CTA's own chain
  const int kmain = cmin > 1 ? ((cmin - 1) & ~1) : 0;   // even: the main loop is unrolled by two
  const int dRa = dRb;
  // Main loop: every active slot is on and none is at its last stage, so no predicates.  Two steps per trip with the row
  // buffers Br / Bn swapping roles (in admm2 the copies Br <- Bn sat in front of the final adds in program order and made
  // the in-order issue wait for the NEXT step's row load inside the dependent chain of THIS step).
#pragma unroll 1
  for (int k = 0; k < kmain; k += 2) {
    T W[n], Bn[n], eta;
    if (live) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    lds_row<T, NC>(bt + oE1, swb, W);
    bt += dRa;
    eta = ld_eta(bt);
    lds_row<T, NC>(bt + myrow, swb, Bn);
    wv = dotv_from<n>(Br, W, eta);
    if (live) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    lds_row<T, NC>(bt + oE1, swb, W);
    bt += dRa;
    eta = ld_eta(bt);
    lds_row<T, NC>(bt + myrow, swb, Br);
    wv = dotv_from<n>(Bn, W, eta);
  }
  const int kend = CL ? cnt : m;
#pragma unroll 1
  for (int k = kmain; k < kend; ++k) {                 // w_next = eta~_next + (-B_t) w_t, with the per-slot end conditions
    const bool on = k < cnt, last = k == cnt - 1;
    if (on && live) sts_1(bt + oE1 + me, wv);
    __syncwarp();
    T W[n];
    lds_row<T, NC>(bt + oE1, swb, W);
    pin_vec<n>(W);
    const unsigned bnext = last ? bm : bt + dRb;
    const T eta = (on && !(last && dir)) ? ld_eta(bnext) : T(0);
    if (on) bt = bnext;
    T Bn[n];
    lds_row<T, NC>(bt + myrow, swb, Bn);               // next step's row (record m holds zeros: harmless)
    const T nw = dotv_from<n>(Br, W, eta);
    if (on) wv = nw;
#pragma unroll
    for (int j = 0; j < n; ++j) Br[j] = Bn[j];
  }
  // middle stage: w_m = eta~_m + both contributions; y_m = w_m
  T wm;
  unsigned bp0 = bm;                                    // where the outward sweep finds the y vector of its first step
  if constexpr (CL) {
    if (dir) {                                          // down chain: contribution -> CTA 0's mailbox; y_m comes back into mine
      if (live) cl_sts(cl.r_box + me, wv);
      cl_arrive_remote(cl.r_mb_mid);
      cl_wait(cl.mb_mid, cl.parity);
      wm = T(0);
      bp0 = cl.box - oE0;
    } else {
      cl_wait(cl.mb_mid, cl.parity);
      wm = wv + lds_1(cl.box + me, T(0));
      if (live) { sts_1(bm + oE1 + me, wm); sts_1(bm + oE0 + me, wm); cl_sts(cl.r_box + me, wm); }
      cl_arrive_remote(cl.r_mb_mid);
    }
  } else {
    wm = wv + __shfl_xor_sync(0xffffffffu, wv, SL);
    if (live) { sts_1(bm + oE1 + me, wm); sts_1(bm + oE0 + me, wm); }
  }
  __syncwarp();
  // outward sweep: y_t = w_t + (-B_t)' y_next.  The column of -B_t and w_t of the NEXT step are loaded while this step's
  // y vector is in flight; two steps per trip with the buffers swapping roles.
  unsigned bc = cnt > 0 ? pb + (unsigned)rec(t0 + (cnt - 1) * (dir ? -1 : 1)) * ES : bm, bp = bp0;
  auto ld_col = [&](unsigned base, T (&col)[n], T& w) {
#pragma unroll
    for (int j = 0; j < n; ++j) col[j] = lds_1(base + oLAM + (unsigned)(j * n) * ES + me, T(0));
    w = lds_1(base + oE1 + me, T(0));
  };
  auto bstep = [&](const T (&col)[n], const T w, T (&coln)[n], T& wn, int k) {
    const bool on = k < cnt;
    T Y[n];
    lds_row<T, NC>(bp + oE0, 0u, Y);
    const unsigned bnx = (on && k > 0) ? bc - dRb : bc;
    ld_col(bnx, coln, wn);
    const T y = dotv_from<n>(col, Y, w);
    if (on) { if (live) sts_1(bc + oE0 + me, y); bp = bc; bc = bnx; }
    __syncwarp();
  };
  T colA[n], colB[n], wA, wB;
  ld_col(bc, colA, wA);
  int k = kend - 1;
#pragma unroll 1
  for (; k >= 1; k -= 2) { bstep(colA, wA, colB, wB, k); bstep(colB, wB, colA, wA, k - 1); }
  if (k == 0) bstep(colA, wA, colB, wB, 0);
}

// Lane map of an item thread: (problem g of the CTA, stage t, half h).  Half h owns the columns / x-rows of its half (slot
// order above), the dynamics rows [h KA, ...) of ITS stage's block (block t for t < N; the rows x_0 = x_init for t = N, whose
// A^+ = [I 0] sits in record 0), and the inequality rows: for a selection G the rows whose column it owns, for a dense G the
// rows 2 s + h.
template <typename T, int NC, int NX, int PG, int MAXT, int MINB, bool XG = false, bool CL = false>
__global__ void __launch_bounds__(MAXT, MINB) admm3_kernel(const __grid_constant__ Admm3Args<T> A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  using RC = Rec3<T, NC, NX, XG>;
  static_assert(NC % 2 == 0, "two lanes per stage own half a row each");
  const AdmmArgs<T>& a = A.a;
  const Dims& d = a.d;
  constexpr int n = NC, nx = NX, nn = NC * NC, H = NC / 2, KA = (NX + 1) / 2;
  const int R = A.pl.R, PP = A.pl.per_problem;
  const int ng = d.ng, N = d.N, T_ = d.T, nz = T_ * n, mf = d.mf, mg = d.mg;
  const int tid = threadIdx.x, nt = blockDim.x, it_tid = tid - 32;
  const int m = T_ / 2;
  const int DOWN0 = A.pl.down0;
  auto rec = [&](int t) { return t > m ? DOWN0 + (N - t) * R : t * R; };
  // CL: CTA `crank` of the pair holds stages [cl_t0, cl_t0 + cl_cnt) of problem blockIdx.x / 2
  const int crank = CL ? (int)cl_rank() : 0, cl_t0 = crank ? m + 1 : 0, cl_cnt = CL ? (crank ? T_ - 1 - m : m + 1) : T_;
  const int pbase = CL ? (int)(blockIdx.x >> 1) : (int)blockIdx.x * PG;
  if constexpr (CL) { if (a.active && !a.active[pbase]) return; }      // a terminated problem (f1): both CTAs of the pair leave before any cluster barrier
  else if (a.active) {                                                 // a CTA whose problems have all terminated leaves before the prologue
    bool any = false;
#pragma unroll
    for (int g = 0; g < PG; ++g) any |= pbase + g < d.B && a.active[pbase + g] != 0;
    if (!any) return;
  }
  const unsigned cl_sb = (unsigned)__cvta_generic_to_shared(sm);
  const unsigned cl_box = cl_sb + (unsigned)(PP - (NC + RC::V - 1) / RC::V * RC::V) * (unsigned)sizeof(T), cl_mb = cl_sb + (unsigned)PP * (unsigned)sizeof(T);   // mailbox; mbarriers mid, eta, y

  // ---- stage 1: X_t, -B_t and the raw constraint blocks of every problem of this CTA into the records (all threads)
#pragma unroll 1
  for (int g = 0; g < PG; ++g) {
    const int p = pbase + g;
    T* P = sm + g * PP;
    for (int e = tid; e < PP; e += nt) P[e] = T(0);
    __syncthreads();
    if (p >= d.B) continue;
    const T* gLam = a.Lam + (size_t)p * T_ * nn;
    const T* gX = a.Sinv + (size_t)p * T_ * nn;
    for (int e = tid; e < cl_cnt * nn; e += nt) {
      const int t = cl_t0 + e / nn, rc = e - (t - cl_t0) * nn;
      const int o = rec(t) + rc;
      if (t != m) P[o + RC::LAM] = -gLam[(size_t)t * nn + rc];
      if constexpr (!XG) P[o + RC::SINV] = gX[(size_t)t * nn + rc];
    }
    if (!XG && !a.kkt_only) {
      const T* gAm = a.qp.Am + (size_t)p * N * nx * n; const T* gAp = a.qp.Ap + (size_t)p * N * nx * n;
      for (int e = tid; e < cl_cnt * nx * n; e += nt) {
        const int t = cl_t0 + e / (nx * n), rc = e - (t - cl_t0) * nx * n, k = rc / n, j = rc - k * n;
        if (t < N) P[rec(t) + RC::AM + rc] = gAm[(size_t)t * nx * n + rc];
        P[rec(t) + RC::AP + rc] = t > 0 ? gAp[(size_t)(t - 1) * nx * n + rc] : (k == j ? T(1) : T(0));      // A_init = [I 0]
      }
      if (!d.g_sel) {
        const T* gG = a.qp.G + a.qp.sG * p;
        for (int e = tid; e < cl_cnt * ng * n; e += nt) { const int t = cl_t0 + e / (ng * n), rc = e - (t - cl_t0) * ng * n; P[rec(t) + RC::G + rc] = gG[(size_t)t * ng * n + rc]; }
      }
    }
  }
  __syncthreads();
  // ---- stage 2: the constraint blocks in the scaled variables, row by row in place: M~[k][j] = sum_{l <= j} M[k][l] X_t[j][l]
  // (A~^-_t = A^-_t X_t', A~^+_{t-1} = A^+_{t-1} X_t', G~_t = G_t X_t'); a thread owns a whole row, so there is no hazard
  if (!XG && !a.kkt_only) {
    const int rows_t = 2 * nx + (d.g_sel ? 0 : ng);       // rows per stage: AM, AP, G
    for (int e = tid; e < PG * cl_cnt * rows_t; e += nt) {
      const int g = e / (cl_cnt * rows_t), r2 = e - g * cl_cnt * rows_t, t = cl_t0 + r2 / rows_t, k = r2 - (t - cl_t0) * rows_t;
      if (pbase + g >= d.B) continue;
      T* rowp = sm + g * PP + rec(t) + (k < nx ? RC::AM + k * n : (k < 2 * nx ? RC::AP + (k - nx) * n : RC::G + (k - 2 * nx) * n));
      const T* X = sm + g * PP + rec(t) + RC::SINV;
      T v[n], o[n];
#pragma unroll
      for (int l = 0; l < n; ++l) v[l] = rowp[l];
#pragma unroll
      for (int j = 0; j < n; ++j) { T acc = T(0);
#pragma unroll
        for (int l = 0; l < n; ++l) if (l <= j) acc += v[l] * X[j * n + l];
        o[j] = acc; }
#pragma unroll
      for (int j = 0; j < n; ++j) rowp[j] = o[j];
    }
    __syncthreads();
  }

  // CL: the three mbarriers of this CTA (mid: the partner's chain warp arrives; eta: the partner's two boundary lanes; y: the partner's chain warp),
  // then a cluster barrier: nobody touches the partner's shared memory before it is set up
  unsigned r_box = 0u, r_mb = 0u;
  if constexpr (CL) {
    if (tid == 0) {
      cl_mbar_init(cl_mb, 32u); cl_mbar_init(cl_mb + 8u, 2u); cl_mbar_init(cl_mb + 16u, 32u);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    r_box = cl_map(cl_box, (unsigned)(crank ^ 1)); r_mb = cl_map(cl_mb, (unsigned)(crank ^ 1));
    cl_sync();
  }

  // ================================================================ chain warp
  if (tid < 32) {
    const int iters = a.kkt_only ? 1 : a.iters;
    unsigned pmask = 0u;
#pragma unroll
    for (int g = 0; g < PG; ++g) { const int p = pbase + g; if (p < d.B && (!a.active || a.active[p])) pmask |= 1u << g; }
#pragma unroll 1
#ifdef TMPC_TIMING
    long long tch = 0; const long long tbeg = clock64();
#endif
    for (int it = 0; it < iters; ++it) {
      bar_sync(1, nt);
#ifdef TMPC_TIMING
      __syncwarp(); const T probe = sm[tid & 7]; const long long c1 = clock64() + (probe == T(12345.678) ? 1 : 0);   // the load makes the deferred barrier block first
#endif
      if constexpr (CL) {
        if (!a.kkt_only) cl_wait(cl_mb + 8u, (unsigned)(it & 1));      // the partner's boundary lanes have delivered their share of my right-hand side
        ClCtx cc; cc.rank = crank; cc.box = cl_box; cc.mb_mid = cl_mb; cc.r_box = r_box; cc.r_mb_mid = r_mb; cc.parity = (unsigned)(it & 1);
        chain3_solve<T, NC, NX, PG, XG, true>(sm, R, A.pl.down0, PP, T_, tid, pmask, cc);
      } else chain3_solve<T, NC, NX, PG, XG>(sm, R, A.pl.down0, PP, T_, tid, pmask);
      __syncwarp();
#ifdef TMPC_TIMING
      tch += clock64() - c1;
#endif
      bar_arrive(2, nt);
      if constexpr (CL) cl_arrive_remote(r_mb + 16u);                  // my y's are complete: the partner's boundary lanes may read across
    }
    if constexpr (CL) cl_sync();                                       // neither CTA leaves while the other may still reach into it
#ifdef TMPC_TIMING
    if ((blockIdx.x == 0 || blockIdx.x == gridDim.x - 1) && tid == 0) printf("cta %d: %lld cycles per iteration, of which chain %lld\n", blockIdx.x, (clock64() - tbeg) / iters, tch / iters);
#endif
    return;
  }

  // ================================================================ item warps
  const int per_p = 2 * cl_cnt;                          // lanes per problem (CL: of this CTA's half)
  const int g = it_tid / per_p, rem = it_tid - g * per_p, t = cl_t0 + (rem >> 1), h = rem & 1, p = pbase + g;
  const bool valid = g < PG && p < d.B && (!a.active || a.active[p]);      // a terminated problem (f1) is left untouched
  const HalfOff mine = half_off<NC>(h), other = half_off<NC>(1 - h);
  const int b = valid ? g * PP + rec(t) : 0, bn = valid ? g * PP + (t < N ? rec(t + 1) : rec(0)) : 0;
  // the record of the next stage (E1B written in the first phase, E0 and A~^+ read): for the boundary stage of a CL half it is the partner's
  const bool cross = CL && valid && (crank ? t == N : t == m);
  T* nbp = sm + bn;
  if constexpr (CL) { if (cross) { unsigned long long ga; asm volatile("mapa.u64 %0, %1, %2;" : "=l"(ga) : "l"((unsigned long long)(sm + bn)), "r"((unsigned)(crank ^ 1))); nbp = reinterpret_cast<T*>(ga); } }
  // the blocks the item lanes read: X_t, A~^-_t (my record) and A~^+_t (the next record) — shared memory, or global memory for XG
  // XG: rows of X, A~^-, A~^+, G~ in that order, row r of stage t at gp + r RS + t V, its 16-byte chunks CS apart (atil_kernel)
  constexpr int VV = RC::V, CCH = (NC + VV - 1) / VV;
  const int CS = XG ? A.tpad * VV : VV, RS = XG ? CCH * CS : n;
  const int arows = n + 2 * nx + (d.g_sel ? 0 : ng);
  const T* gp = XG ? A.atil + (valid ? (size_t)p * arows * RS : 0) : nullptr;
  const int tn = valid ? (t < N ? t + 1 : 0) : 0, tv = valid ? t : 0;
  const T* Xb = XG ? gp + tv * VV : sm + b + RC::SINV;
  const T* AMb = XG ? gp + (size_t)n * RS + tv * VV : sm + b + RC::AM;
  const T* APn = XG ? gp + (size_t)(n + nx) * RS + tn * VV : nbp + RC::AP;
  const T* Gb = XG ? gp + (size_t)(n + 2 * nx) * RS + tv * VV : sm + b + RC::G;
  auto ldh = [&](const T* row, const HalfOff& o, T (&r)[H]) { if constexpr (XG) ld_half_g<NC>(row, o, r, CS); else ld_half<NC>(row, o, r); };

  if (a.kkt_only) {                                      // xt <- S^{-1} eta : eta~ = X eta, solve, x = X' y
    T eo[H], er[H];
#pragma unroll
    for (int s = 0; s < H; ++s) eo[s] = valid ? a.x[(size_t)p * nz + t * n + slot_col<NC>(h, s)] : T(0);
#pragma unroll
    for (int s = 0; s < H; ++s) er[s] = shfl_x1(eo[s]);
    if (valid) {
      T acc[H];
#pragma unroll
      for (int s = 0; s < H; ++s) { T f[H], f2[H]; const T* row = Xb + slot_col<NC>(h, s) * RS; ldh(row, mine, f); ldh(row, other, f2); acc[s] = dot2<T, H>(f, eo, f2, er); }
      st_half<NC>(sm + b + RC::E1A, mine, acc);
    }
    bar_arrive(1, nt);
    bar_sync(2, nt);
    if (valid) {
      T yo[H], yr[H], xt[H];
      ld_half<NC>(sm + b + RC::E0, mine, yo); ld_half<NC>(sm + b + RC::E0, other, yr);
#pragma unroll
      for (int s = 0; s < H; ++s) xt[s] = T(0);
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ldh(Xb + slot_col<NC>(h, jj) * RS, mine, mk); axpy_half<H>(xt, mk, yo[jj]); }
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ldh(Xb + slot_col<NC>(1 - h, jj) * RS, mine, mk); axpy_half<H>(xt, mk, yr[jj]); }
#pragma unroll
      for (int s = 0; s < H; ++s) a.xi[(size_t)p * nz + t * n + slot_col<NC>(h, s)] = xt[s];
    }
    if constexpr (CL) cl_sync();
    return;
  }

  // step sizes: per problem when the adaptive schedule (f1) runs, else the handle's
  const T rho_g = (a.rho_bar && valid) ? a.rho_bar[p] : a.prm.rho_g, rho_f = a.rho_bar ? a.rho_scale * rho_g : a.prm.rho_f;
  const T rfa = a.rho_bar ? rho_f * a.prm.alpha : A.rfa, inv_rho_g = a.rho_bar ? T(1) / rho_g : A.inv_rho_g, inv_rg = a.rho_bar ? T(1) / (rho_g + a.prm.gamma) : A.inv_rg;
  // ---- per-lane state in registers (slot order)
  constexpr unsigned Q_VALID = 1u, Q_SOFT = 2u, Q_ROW_SH = 4;         // inequality slot flags: valid, soft, row index << 4
  T x[H], q[H], zg[H], yg[H], lo[H], hi[H], xi_last[H];
  T yf[KA], cv[KA];
  unsigned qf[H];                                                     // inequality slot s <-> (selection: my column of slot s; dense: row 2 s + h)
  const int k0 = h * KA, nk = valid ? (h ? nx - KA : KA) : 0;         // my dynamics rows k0 .. k0 + nk - 1
  const int k0p = (1 - h) * KA, nkp = valid ? (h ? KA : nx - KA) : 0; // the partner's
#pragma unroll
  for (int s = 0; s < H; ++s) { x[s] = q[s] = zg[s] = yg[s] = lo[s] = hi[s] = xi_last[s] = T(0); qf[s] = 0u; }
#pragma unroll
  for (int s = 0; s < KA; ++s) yf[s] = cv[s] = T(0);
  if (valid) {
#pragma unroll
    for (int s = 0; s < H; ++s) { const size_t el = (size_t)p * nz + t * n + slot_col<NC>(h, s); x[s] = a.x[el]; q[s] = a.qp.q[el]; }
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
        const int col = slot_col<NC>(h, s);
#pragma unroll
        for (int rr = 0; rr < NC; ++rr) if (rr < ng && d.g_col[rr] == col) r = rr;
      } else if (2 * s + h < ng) r = 2 * s + h;
      if (r < 0) continue;
      const size_t row = (size_t)p * mg + t * ng + r;
      if (a.soft_rows && a.soft_rows[row] == 2) continue;      // row switched off (adjoint refinement: inactive rows, and soft-active rows that live in the factor only)
      qf[s] = Q_VALID | ((unsigned)r << Q_ROW_SH);
      lo[s] = a.qp.lo[row]; hi[s] = a.qp.hi[row]; yg[s] = a.yg[row];
      if (a.soft_rows ? (a.soft_rows[row] == 1) : (((d.soft_mask >> r) & 1u) != 0)) qf[s] |= Q_SOFT;
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
    }
  }

#ifdef TMPC_TIMING
  long long tA = 0, tW = 0, tB = 0, qs = clock64();
#endif
#pragma unroll 1
  for (int it = 0; it < a.iters; ++it) {
#ifdef TMPC_TIMING
    if (it > 0) { const long long q0 = clock64(); tB += q0 - qs; qs = q0; }
#endif
    // ---- a4 in scaled variables (eq. 51): eta~_t = X_t (sigma x - q + G's) + A~^-_t' r_t  [+ G~_t' s_t]  -> E1A of my record,
    //      and my block's share of the next stage's right-hand side, A~^+_t' r_t -> E1B of record t+1 (record 0 for t = N)
    T dn[H], dr[H], ro[KA], rr[KA];
#pragma unroll
    for (int s = 0; s < H; ++s) {
      T dd = a.prm.sigma * x[s] - q[s];
      if (d.g_sel && (qf[s] & Q_VALID)) dd += rho_g * zg[s] - yg[s];
      dn[s] = dd;
    }
#pragma unroll
    for (int s = 0; s < KA; ++s) ro[s] = rho_f * cv[s] - yf[s];   // r = rho_f c - y_f of my rows (0 beyond nk: c = y_f = 0)
#pragma unroll
    for (int s = 0; s < H; ++s) dr[s] = shfl_x1(dn[s]);                // the partner's halves
#pragma unroll
    for (int s = 0; s < KA; ++s) rr[s] = shfl_x1(ro[s]);
    T sg[H], sgr[H];
    if (!d.g_sel) {
#pragma unroll
      for (int s = 0; s < H; ++s) sg[s] = (qf[s] & Q_VALID) ? rho_g * zg[s] - yg[s] : T(0);
#pragma unroll
      for (int s = 0; s < H; ++s) sgr[s] = shfl_x1(sg[s]);
    }
    if (valid) {
      T acc[H], accb[H];
#pragma unroll
      for (int s = 0; s < H; ++s) {                    // my rows of X_t: my half first, then the partner's
        T f[H], f2[H];
        const T* row = Xb + slot_col<NC>(h, s) * RS;
        ldh(row, mine, f); ldh(row, other, f2);
        acc[s] = dot2<T, H>(f, dn, f2, dr);
        accb[s] = T(0);
      }
#pragma unroll
      for (int s = 0; s < KA; ++s) {                   // my columns of A~^-_t (my record) and A~^+_t (next record), rows of my block half / the partner's
        T mk[H];
        if (s < nk) {
          ldh(AMb + (k0 + s) * RS, mine, mk); axpy_half<H>(acc, mk, ro[s]);
          ldh(APn + (k0 + s) * RS, mine, mk); axpy_half<H>(accb, mk, ro[s]);
        }
        if (s < nkp) {
          ldh(AMb + (k0p + s) * RS, mine, mk); axpy_half<H>(acc, mk, rr[s]);
          ldh(APn + (k0p + s) * RS, mine, mk); axpy_half<H>(accb, mk, rr[s]);
        }
      }
      if (!d.g_sel) {
#pragma unroll
        for (int s = 0; s < H; ++s) {
          T mk[H];
          if (2 * s + h < ng) { ldh(Gb + (2 * s + h) * RS, mine, mk); axpy_half<H>(acc, mk, sg[s]); }
          if (2 * s + 1 - h < ng) { ldh(Gb + (2 * s + 1 - h) * RS, mine, mk); axpy_half<H>(acc, mk, sgr[s]); }
        }
      }
      st_half<NC>(sm + b + RC::E1A, mine, acc);
      st_half<NC>(nbp + RC::E1B, mine, accb);
      if constexpr (CL) { if (cross) cl_arrive_remote(r_mb + 8u); }
    }
#ifdef TMPC_TIMING
    const long long qa = clock64();
#endif
    bar_arrive(1, nt);
    bar_sync(2, nt);
    if constexpr (CL) { if (cross) cl_wait(cl_mb + 16u, (unsigned)(it & 1)); }   // the partner's chain has finished: y of the stage across the boundary is there
#ifdef TMPC_TIMING
    { const T probe = sm[b + RC::E0]; const long long qb = clock64() + (probe == T(12345.678) ? 1 : 0); tA += qa - qs; tW += qb - qa; qs = qb; }
#endif
    // ---- a7 + a8 on y: x~ = X_t' y_t, z~_f = A~^-_t y_t + A~^+_t y_{t+1}, z~_g = x~_col or G~_t y_t; relaxation (eq. 10),
    // projection (eq. 12-15), duals (eq. 16 / 44-45)
    if (valid) {
      T yo[H], yr[H], xt[H];
      ld_half<NC>(sm + b + RC::E0, mine, yo); ld_half<NC>(sm + b + RC::E0, other, yr);
#pragma unroll
      for (int s = 0; s < H; ++s) xt[s] = T(0);
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ldh(Xb + slot_col<NC>(h, jj) * RS, mine, mk); axpy_half<H>(xt, mk, yo[jj]); }       // rows of my half
#pragma unroll
      for (int jj = 0; jj < H; ++jj) { T mk[H]; ldh(Xb + slot_col<NC>(1 - h, jj) * RS, mine, mk); axpy_half<H>(xt, mk, yr[jj]); }   // rows of the partner's half
      if (nk > 0) {
        T y2o[H], y2r[H];
        ld_half<NC>(nbp + RC::E0, mine, y2o); ld_half<NC>(nbp + RC::E0, other, y2r);
#pragma unroll
        for (int s = 0; s < KA; ++s) if (s < nk) {
          const int k = k0 + s;
          T f[H], f2[H];
          ldh(AMb + k * RS, mine, f); ldh(AMb + k * RS, other, f2);
          T zt = dot2<T, H>(f, yo, f2, yr);
          ldh(APn + k * RS, mine, f); ldh(APn + k * RS, other, f2);
          zt += dot2<T, H>(f, y2o, f2, y2r);
          yf[s] += rfa * (zt - cv[s]);
        }
      }
#pragma unroll
      for (int s = 0; s < H; ++s) {
        if (qf[s] & Q_VALID) {
          T ztg = xt[s];
          if (!d.g_sel) { const T* row = Gb + (int)(qf[s] >> Q_ROW_SH) * RS; T f[H], f2[H]; ldh(row, mine, f); ldh(row, other, f2); ztg = dot2<T, H>(f, yo, f2, yr); }
          const T zh = a.prm.alpha * ztg + A.oma * zg[s];
          const T v = zh + yg[s] * inv_rho_g;
          T z, sl;
          project_row<T>((qf[s] & Q_SOFT) != 0, v, lo[s], hi[s], rho_g, inv_rg, a.prm.lam, z, sl);
          yg[s] += rho_g * (zh - z);
          zg[s] = z;
          xi_last[s] = sl;
        }
        x[s] = a.prm.alpha * xt[s] + A.oma * x[s];
      }
    }
  }

#ifdef TMPC_TIMING
  if (blockIdx.x == 0 && (tid == 32 || tid == 160)) printf("item warp %d: phase A %lld, wait for chain %lld, phase B %lld cycles per iteration\n", tid >> 5, tA / a.iters, tW / a.iters, tB / a.iters);
#endif
  // ---- write back the state
  if (valid) {
#pragma unroll
    for (int s = 0; s < H; ++s) a.x[(size_t)p * nz + t * n + slot_col<NC>(h, s)] = x[s];
#pragma unroll
    for (int s = 0; s < KA; ++s) if (s < nk) a.yf[(size_t)p * mf + (t < N ? nx + t * nx + k0 + s : k0 + s)] = yf[s];
#pragma unroll
    for (int s = 0; s < H; ++s) if (qf[s] & Q_VALID) {
      const size_t row = (size_t)p * mg + t * ng + (qf[s] >> Q_ROW_SH);
      a.zg[row] = zg[s]; a.yg[row] = yg[s]; if (a.iters > 0) a.xi[row] = xi_last[s];
    }
  }
  if constexpr (CL) cl_sync();
}

// ---- XG: what the item lanes read, once per launch of the solve, in the STAGE-MINOR layout of ld_half_g: per problem the rows
//   [0, n)                 X_t                                   (copied from the factor)
//   [n, n + nx)            A~^-_t = A^-_t X_t'                    (zero for t = N)
//   [n + nx, n + 2 nx)     A~^+_{t-1} = A^+_{t-1} X_t'            (A_init = [I 0] for t = 0)
//   [n + 2 nx, .. + ng)    G~_t = G_t X_t'                        (dense G only)
// with M~[k][j] = sum_{l <= j} M[k][l] X_t[j][l] (X_t lower triangular); element j of row r of stage t goes to
// (p rows + r) RS + (j / V) CS + t V + j % V, CS = tpad V, RS = ceil(n / V) CS.  One thread per (problem, row, stage), stage fastest; n <= 16.
template <typename T>
__global__ void __launch_bounds__(128) atil_kernel(const AdmmArgs<T> a, T* __restrict__ atil, int tpad, int rows, const int32_t* __restrict__ mask) {   // rows = n for kkt_only (X only); mask: only the problems whose factor has changed
  const Dims& d = a.d;
  constexpr int V = 16 / (int)sizeof(T);
  const int n = d.n, nx = d.nx, T_ = d.T, N = d.N;
  const int CS = tpad * V, RS = (n + V - 1) / V * CS;
  const int rows_all = n + 2 * nx + (d.g_sel ? 0 : d.ng);
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (long long)d.B * rows * T_) return;
  const int t = (int)(e % T_), r = (int)((e / T_) % rows), p = (int)(e / ((long long)rows * T_));
  if (mask && !mask[p]) return;
  const T* X = a.Sinv + ((size_t)p * T_ + t) * n * n;
  T* out = atil + ((size_t)p * rows_all + r) * RS + (size_t)t * V;
  if (r < n) {                                         // a row of X_t
    for (int j = 0; j < n; ++j) out[(j / V) * CS + j % V] = X[r * n + j];
    return;
  }
  const int k2 = r - n;
  const bool plus = k2 >= nx && k2 < 2 * nx, isg = k2 >= 2 * nx; const int k = isg ? k2 - 2 * nx : (plus ? k2 - nx : k2);
  T v[16];
#pragma unroll
  for (int l = 0; l < 16; ++l) {
    T s = T(0);
    if (l < n) {
      if (isg) s = a.qp.G[a.qp.sG * p + ((size_t)t * d.ng + k) * n + l];
      else if (!plus) { if (t < N) s = a.qp.Am[(((size_t)p * N + t) * nx + k) * n + l]; }
      else s = t > 0 ? a.qp.Ap[(((size_t)p * N + t - 1) * nx + k) * n + l] : (l == k ? T(1) : T(0));
    }
    v[l] = s;
  }
  for (int j = 0; j < n; ++j) {
    T acc = T(0);
#pragma unroll
    for (int l = 0; l < 16; ++l) if (l <= j) acc += v[l] * X[j * n + l];
    out[(j / V) * CS + j % V] = acc;
  }
}

}  // namespace tmpc
