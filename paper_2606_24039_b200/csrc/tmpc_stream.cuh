// tmpc_stream.cuh — a4..a8 for the STREAMED class (config 3: n = 88, 2.8 MB of factor + constraint blocks per problem,
// far beyond shared memory): the fused ADMM loop of Alg. 3 with every matrix block streamed from
// HBM exactly as often as the algorithm needs it (Lambda twice, Sigma^{-1} once, A^-/A^+ once per iteration =
// SURVEY.md 8(d)'s 4.33 MB per problem-iteration at config 3).
//
// One CTA per problem.  Warp 0 is the PRODUCER: it walks the (fully predictable) sequence of blocks of an iteration and
// copies each into a ring of shared-memory slots with one bulk asynchronous copy (cp.async.bulk -> UBLKCP), completion signalled on a 'full' mbarrier per slot; it waits on the
// slot's 'empty' mbarrier before refilling.  The other warps are CONSUMERS: thread i owns row / column i of the
// current block (row-wise vector loads for w = eta - Lambda w, v = Sigma^{-1} w, z~ = A x~; column-wise scalar loads
// for x~ = v - Lambda' x~ and eta += A' r); a quad of lanes shares each row / column.
// The sweep over t that produces x~_t (outward) also applies the stage-local updates (eq. 9-16) and accumulates the
// next right-hand side eta (eq. 51) while A^-_t / A^+_t are resident, so the constraint blocks are read once.
// Factor format: the one-directional block LDL' of factor_kernel (Lam [N][n][n], Sinv [T][n][n]).
#pragma once
#include <cstdlib>
#include "tmpc_common.cuh"
#include "tmpc_admm.cuh"

namespace tmpc {

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_arrive(unsigned bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

struct StreamPlan { int LD, slots, tile_elems, nthreads; size_t smem; };

// row stride of a block in shared memory (elements).  Blocks are copied with ONE bulk copy each (small per-row copies
// are issue-bound: ~50 cycles per cp.async.bulk measured), so rows stay unpadded; with a quad of lanes per row the
// column-wise reads are conflict free for n = 88 and the row-wise vector reads see at most 2-way conflicts.
template <typename T>
__host__ __device__ inline int stream_ld(int n) { return n; }
template <typename T>
__host__ inline StreamPlan stream_plan(const Dims& d, size_t max_smem) {
  StreamPlan P; P.LD = stream_ld<T>(d.n); P.tile_elems = d.n * P.LD;
  const int nc = (4 * (d.n > d.nx ? d.n : d.nx) + 31) / 32 * 32;    // a quad of threads per row
  P.nthreads = 32 + nc;
  const size_t fixed = (size_t)(d.nz + 2 * d.n + 2 * d.nx + 2 * d.ng + 64) * sizeof(T) + 256;   // x~/v, w window, r, s
  const size_t tile = (size_t)P.tile_elems * sizeof(T);
  long s = ((long)max_smem - (long)fixed) / (long)tile;
  const int smax = s > 6 ? 6 : (int)s;
  P.slots = smax;
  // the consumers are latency bound (dependent dots + CTA barriers): co-resident CTAs hide that better than a deep ring
  // (measured at config 3: two CTAs per SM with 2 slots 116 ms, one CTA with 6 slots 144 ms), so take the deepest ring
  // that still lets two CTAs share an SM
  for (int k = smax; k >= 2; --k) if (2 * (fixed + k * tile + 1024) <= (size_t)228 * 1024) { P.slots = k; break; }
  P.smem = fixed + (size_t)(P.slots > 0 ? P.slots : 0) * tile;
  return P;
}

template <typename T>
// g0, chunks: iteration-chunk scheduling (launch_admm): CTA b of a launch runs chunk (g0 + b) / B of problem (g0 + b) % B,
// i.e. iterations [iters k / chunks, iters (k+1) / chunks); chunks = 1, g0 = 0 is the plain one-CTA-per-problem launch.
struct StreamArgs { AdmmArgs<T> a; int LD, slots, tile_elems; T* eta; int g0, chunks; };   // eta: global scratch [B][nz] (right-hand side, L2 resident)

// block sequence of one launch, identical in the producer and the consumers:
//   [eta pass]   t = N-1..0 : A^-_t, A^+_t                         (skipped for kkt_only)
//   iteration:   t = 0..N   : Lambda_{t-1} (t > 0), Sigma^{-1}_t
//                t = N..0   : Lambda_t, A^-_t, A^+_t (t < N; the A blocks skipped for kkt_only)
template <typename T>
__global__ void __launch_bounds__(1024) admm_stream_kernel(const __grid_constant__ StreamArgs<T> S) {
  extern __shared__ __align__(128) unsigned char smem_ring_raw[];   // own name: the other kernels of this translation unit declare theirs 16-byte aligned
  const AdmmArgs<T>& a = S.a;
  const Dims& d = a.d;
  const int n = d.n, nx = d.nx, ng = d.ng, N = d.N, T_ = d.T, nn = n * n, an = nx * n, nz = d.nz, mf = d.mf, mg = d.mg;
  const int LD = S.LD, KS = S.slots, tid = threadIdx.x;
  const int gjob = S.g0 + (int)blockIdx.x, chunk = gjob / d.B, p = gjob - chunk * d.B;
  const int zg_given = chunk > 0 ? 1 : a.zg_given;                   // later chunks resume from the stored state
  if (a.active && !a.active[p]) return;                              // terminated problem (f1): the whole CTA leaves before any barrier is set up
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_ring_raw);            // full[KS], empty[KS]
  T* ring = reinterpret_cast<T*>(smem_ring_raw + 256);
  // Only v / x~ is kept whole in shared memory.  The right-hand side eta lives in global memory (each element is written
  // once and read once per iteration by the SAME thread, prefetched a step ahead), x is updated in place in global
  // memory, and w_t only needs a two-stage window: the small footprint leaves room for a deeper ring / more CTAs.
  T* e1 = ring + (size_t)KS * S.tile_elems;       // v / x~   [nz]
  T* wwin = e1 + nz;                              // w_{t-1}, w_t   [2][n]
  T* rbuf = wwin + 2 * n;                         // r_t [nx]
  T* sbuf = rbuf + 2 * nx;                        // s_t [ng]
  const unsigned bar0 = smem_u32(bars);
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (KS + s); };
  const int ncons = blockDim.x - 32;
  if (tid == 0) {
    for (int s = 0; s < KS; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), ncons); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const T* gLam = a.Lam + (size_t)p * N * nn;
  const T* gSinv = a.Sinv + (size_t)p * T_ * nn;
  const T* gAm = a.kkt_only ? nullptr : a.qp.Am + (size_t)p * N * an;
  const T* gAp = a.kkt_only ? nullptr : a.qp.Ap + (size_t)p * N * an;
  const int iters = a.kkt_only ? 1 : (int)(((long long)a.iters * (chunk + 1)) / S.chunks - ((long long)a.iters * chunk) / S.chunks);

  // ======================================================================= producer warp
  if (tid < 32) {
    int c = 0;                                                          // running tile counter
    auto push = [&](const T* src, int rows) {
      const int s = c % KS; const unsigned ph = (unsigned)(c / KS) & 1u;
      if (c >= KS) mbar_wait(empty_bar(s), ph ^ 1u);
      if (tid == 0) {
        const unsigned bytes = (unsigned)(rows * n) * sizeof(T);
        mbar_expect_tx(full_bar(s), bytes);
        bulk_g2s(smem_u32(ring + (size_t)s * S.tile_elems), src, bytes, full_bar(s));
      }
      __syncwarp();
      ++c;
    };
    if (!a.kkt_only) for (int t = N - 1; t >= 0; --t) { push(gAm + (size_t)t * an, nx); push(gAp + (size_t)t * an, nx); }
    for (int it = 0; it < iters; ++it) {
      for (int t = 0; t < T_; ++t) { if (t > 0) push(gLam + (size_t)(t - 1) * nn, n); push(gSinv + (size_t)t * nn, n); }
      for (int t = N - 1; t >= 0; --t) {
        push(gLam + (size_t)t * nn, n);
        if (!a.kkt_only) { push(gAm + (size_t)t * an, nx); push(gAp + (size_t)t * an, nx); }
      }
    }
    return;
  }

  // ======================================================================= consumer warps
  const int ct = tid - 32, ci = ct >> 2, cq = ct & 3;                   // four threads (a quad of lanes) share row / column ci
  auto cons_bar = [&]() { asm volatile("bar.sync 1, %0;" ::"r"(ncons) : "memory"); };
  int c = 0;
  auto acquire = [&](int ahead) -> const T* { const int cc = c + ahead; const int s = cc % KS; mbar_wait(full_bar(s), (unsigned)(cc / KS) & 1u); return ring + (size_t)s * S.tile_elems; };
  auto release = [&](int count) { for (int k = 0; k < count; ++k) { mbar_arrive(empty_bar(c % KS)); ++c; } };
  auto quad_sum = [&](T v) -> T { v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2); return v; };
  // (M vec)[ci] for a block of `rows` rows: lane cq of the quad takes the 16-byte chunks cq, cq+4, .. of the padded row.
  // Called by every consumer thread (the quad reduction is a full-warp shuffle).
  auto row_dot = [&](const T* M, const T* vec, int rows) -> T {
    const T* row = M + (size_t)(ci < rows ? ci : 0) * LD;
    T acc[2] = {T(0), T(0)};
    if constexpr (sizeof(T) == 4) {                    // explicit 16-byte loads (rows and vectors are 16-byte aligned: n % 4 == 0)
      float2 p2 = make_float2(0.f, 0.f);
      for (int j = cq * 4; j < n; j += 16) {
        const float4 m4 = *reinterpret_cast<const float4*>(row + j), v4 = *reinterpret_cast<const float4*>(vec + j);
        p2 = __ffma2_rn(make_float2(m4.x, m4.y), make_float2(v4.x, v4.y), p2);
        p2 = __ffma2_rn(make_float2(m4.z, m4.w), make_float2(v4.z, v4.w), p2);
      }
      acc[0] = p2.x; acc[1] = p2.y;
    } else {
      for (int j = cq * 2; j < n; j += 8) {
        const double2 m2 = *reinterpret_cast<const double2*>(row + j), v2 = *reinterpret_cast<const double2*>(vec + j);
        acc[0] += m2.x * v2.x; acc[1] += m2.y * v2.y;
      }
    }
    return quad_sum(acc[0] + acc[1]);
  };
  // (M' vec)[ci] for a block of `rows` rows: lane cq takes rows cq, cq+4, ..
  auto col_dot = [&](const T* M, const T* vec, int rows) -> T {
    const int col = ci < n ? ci : 0;
    T acc[2] = {T(0), T(0)};
    int k = cq;
    for (; k + 4 < rows; k += 8) { acc[0] += M[(size_t)k * LD + col] * vec[k]; acc[1] += M[(size_t)(k + 4) * LD + col] * vec[k + 4]; }
    for (; k < rows; k += 4) acc[0] += M[(size_t)k * LD + col] * vec[k];
    return quad_sum(acc[0] + acc[1]);
  };
  const T sigma = a.prm.sigma, rho_g = a.rho_bar ? a.rho_bar[p] : a.prm.rho_g, rho_f = a.rho_bar ? a.rho_scale * rho_g : a.prm.rho_f, alpha = a.prm.alpha;   // per-problem step size under f1
  const T inv_rho_g = T(1) / rho_g, inv_rg = T(1) / (rho_g + a.prm.gamma), lam = a.prm.lam;
  const bool own_x = cq == 0 && ci < n, own_f = cq == 0 && ci < nx, own_g = cq == 0 && ci < ng;
  const size_t gx = (size_t)p * nz, gf = (size_t)p * mf, gg = (size_t)p * mg;
  const T* Gd = (!a.kkt_only && !d.g_sel && ng > 0) ? a.qp.G + a.qp.sG * p : nullptr;
  unsigned gmask = 0u; int gcol = 0;
  if (d.g_sel) for (int r = 0; r < ng; ++r) { if (d.g_col[r] == ci) gmask |= 1u << r; if (r == ci) gcol = d.g_col[r]; }
  // (G_t' s_t)[ci] with s_t in `sv` (shared or computed on the fly from global z_g, y_g)
  auto gts = [&](int t, const T* sv) -> T {
    T acc = T(0);
    if (d.g_sel) { unsigned mk = gmask; while (mk) { const int r = __ffs(mk) - 1; mk &= mk - 1; acc += sv ? sv[r] : rho_g * a.zg[gg + t * ng + r] - a.yg[gg + t * ng + r]; } }
    else for (int r = 0; r < ng; ++r) acc += Gd[((size_t)t * ng + r) * n + ci] * (sv ? sv[r] : rho_g * a.zg[gg + t * ng + r] - a.yg[gg + t * ng + r]);
    return acc;
  };
  auto g_row_dot = [&](int t, const T* vec) -> T {                      // (G_t vec_t)[row ci]
    if (d.g_sel) return vec[t * n + gcol];
    const T* g = Gd + ((size_t)t * ng + ci) * n; T s = T(0);
    for (int j = 0; j < n; ++j) s += g[j] * vec[t * n + j];
    return s;
  };

  T* geta = S.eta + gx;                                                 // my problem's right-hand side (global)
  const T* eta_rd = a.kkt_only ? a.x + gx : geta;                       // tmpc_kkt_solve: eta is the caller's vector
  T* gxs = a.x + gx;                                                    // x, updated in place
  if (!a.kkt_only) {
    if (own_g) for (int t = 0; t < T_; ++t) {
      const size_t row = gg + t * ng + ci;
      if (!zg_given) a.zg[row] = tmin(tmax(g_row_dot(t, gxs), a.qp.lo[row]), a.qp.hi[row]);
      if (!zg_given && a.iters == 0) a.xi[row] = T(0);
    }
    cons_bar();
    __threadfence_block();
    // ---- eta pass: eta = sigma x - q + C'(rho_f c - y_f) + G'(rho_g z_g - y_g)  (eq. 51).  Thread ci carries the
    // partial eta of the stage above in a register until block t has added A^+_t' r_t, then stores it once.
    T pend = own_x ? sigma * gxs[N * n + ci] - a.qp.q[gx + N * n + ci] + gts(N, nullptr) : T(0);
    for (int t = N - 1; t >= 0; --t) {
      if (own_f) rbuf[ci] = rho_f * a.qp.b[((size_t)p * N + t) * nx + ci] - a.yf[gf + nx + t * nx + ci];
      const T base = own_x ? sigma * gxs[t * n + ci] - a.qp.q[gx + t * n + ci] + gts(t, nullptr) : T(0);
      const T* Am = acquire(0); const T* Ap = acquire(1);
      cons_bar();
      const T da = col_dot(Am, rbuf, nx), dp = col_dot(Ap, rbuf, nx);
      if (own_x) { geta[(t + 1) * n + ci] = pend + dp; pend = base + da; }
      release(2);
      cons_bar();
    }
    if (own_f) pend += rho_f * a.qp.x_init[(size_t)p * nx + ci] - a.yf[gf + ci];
    if (own_x) geta[ci] = pend;
  }

  for (int it = 0; it < iters; ++it) {
    const bool lastit = it == iters - 1;
    // ---- forward sweep: w_t = eta_t - Lambda_{t-1} w_{t-1},  v_t = Sigma_t^{-1} w_t                         (eq. 8)
    T eta_nx = own_x ? eta_rd[ci] : T(0);
    for (int t = 0; t < T_; ++t) {
      const T eta_t = eta_nx;
      if (t + 1 < T_ && own_x) eta_nx = eta_rd[(t + 1) * n + ci];       // prefetch
      T* wt = wwin + (t & 1) * n;
      if (t > 0) {
        const T* L = acquire(0);
        const T lw = row_dot(L, wwin + ((t - 1) & 1) * n, n);
        release(1);
        if (own_x) wt[ci] = eta_t - lw;
      } else if (own_x) wt[ci] = eta_t;
      cons_bar();
      const T* Si = acquire(0);
      { const T v = row_dot(Si, wt, n); if (own_x) e1[t * n + ci] = v; }
      release(1);
    }
    cons_bar();
    // ---- outward sweep: x~_t = v_t - Lambda_t' x~_{t+1}, then everything local to stage t and dynamics block t.
    // The per-row state of stage t-1 (x, z_g, y_g, lo, hi, y_f, c, q: global memory, L2 resident) is prefetched into
    // registers while stage t is processed, so no global-load latency sits on the dependent path.
    T pzg = T(0), pyg = T(0), plo = T(0), phi = T(0), pyf = T(0), pc = T(0), pq = T(0), px = T(0);
    auto prefetch_state = [&](int t) {
      if (a.kkt_only || t < 0) return;
      if (own_g) { const size_t row = gg + t * ng + ci; pzg = a.zg[row]; pyg = a.yg[row]; plo = a.qp.lo[row]; phi = a.qp.hi[row]; }
      if (own_f && t < N) { pyf = a.yf[gf + nx + t * nx + ci]; pc = a.qp.b[((size_t)p * N + t) * nx + ci]; }
      if (own_x) { pq = a.qp.q[gx + t * n + ci]; px = gxs[t * n + ci]; }
    };
    prefetch_state(N);
    T pend = T(0);                                     // partial next eta of stage t+1 (see the eta pass)
    for (int t = N; t >= 0; --t) {
      if (t < N) {
        const T* L = acquire(0);
        const T lx = col_dot(L, e1 + (t + 1) * n, n);
        release(1);
        if (own_x) e1[t * n + ci] -= lx;
        cons_bar();
      }
      if (a.kkt_only) continue;
      const T zgo = pzg, ygo = pyg, lo_ = plo, hi_ = phi, yfo = pyf, cval = pc, qv = pq, xo = px;
      prefetch_state(t - 1);
      if (own_g) {                                     // eq. 9-16 on inequality row (t, ci)
        const size_t row = gg + t * ng + ci;
        const T zh = alpha * g_row_dot(t, e1) + (T(1) - alpha) * zgo;
        const T v = zh + ygo * inv_rho_g;
        const bool soft = a.soft_rows ? (a.soft_rows[row] != 0) : (((d.soft_mask >> ci) & 1u) != 0);
        T z, s;
        project_row<T>(soft, v, lo_, hi_, rho_g, inv_rg, lam, z, s);
        const T y = ygo + rho_g * (zh - z);
        a.zg[row] = z; a.yg[row] = y; sbuf[ci] = rho_g * z - y;
        if (lastit) a.xi[row] = s;
      }
      T xn = T(0);
      if (own_x) { xn = alpha * e1[t * n + ci] + (T(1) - alpha) * xo; gxs[t * n + ci] = xn; }
      const T* Am = nullptr; const T* Ap = nullptr;
      if (t < N) {
        Am = acquire(0); Ap = acquire(1);
        const T ztf = row_dot(Am, e1 + t * n, nx) + row_dot(Ap, e1 + (t + 1) * n, nx);
        if (own_f) {
          const T y = yfo + rho_f * alpha * (ztf - cval);
          a.yf[gf + nx + t * nx + ci] = y; rbuf[ci] = rho_f * cval - y;
        }
      }
      cons_bar();
      T da = T(0), dp = T(0);
      if (t < N) { da = col_dot(Am, rbuf, nx); dp = col_dot(Ap, rbuf, nx); }
      if (own_x) {
        if (t < N) geta[(t + 1) * n + ci] = pend + dp;  // stage t+1 is complete
        pend = sigma * xn - qv + gts(t, sbuf) + da;
        if (t == 0) {
          if (own_f) {                                 // rows x_0 = x_init (A_init = [I 0])
            const T xi0 = a.qp.x_init[(size_t)p * nx + ci];
            const T y = a.yf[gf + ci] + rho_f * alpha * (e1[ci] - xi0);
            a.yf[gf + ci] = y; pend += rho_f * xi0 - y;
          }
          geta[ci] = pend;
        }
      }
      if (t < N) release(2);
    }
  }
  cons_bar();
  if (a.kkt_only) { for (int e = ct; e < nz; e += ncons) a.xi[gx + e] = e1[e]; }
}

}  // namespace tmpc
