// tmpc_admm2.cuh — pieces shared by the resident-class kernels: vector loads and packed dot products, explicit shared-state-space
// accesses for the chain warp, named barriers, the residual kernel (a9) and the f1 decision kernels.  The first-generation resident
// kernel that lived here (four lanes per stage, XOR-swizzled records) was replaced by tmpc_admm3.cuh in round 2.
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

// chunk-order offset (in elements) of row `row` of an 8-wide block: rows that would collide on the same banks take their 16-byte
// chunks in a different order (tmpc_admm3.cuh chain3_solve); identity for other n
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
__device__ __forceinline__ void lds_chunk(unsigned a, float& r0, float& r1, float& r2, float& r3) { asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r0), "=f"(r1), "=f"(r2), "=f"(r3) : "r"(a)); }
__device__ __forceinline__ void lds_chunk(unsigned a, double& r0, double& r1) { asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(r0), "=d"(r1) : "r"(a)); }
template <typename T, int NC> __device__ __forceinline__ void lds_row(unsigned a, unsigned swb, T (&r)[NC]) {
  if constexpr (NC == 8 && sizeof(T) == 4) lds_vec8(a + swb, a + 16u - swb, r);     // swb in {0,16}: chunks (0,16) or (16,0), one add each
  else if constexpr (NC == 8) lds_vec8(a + (0u ^ swb), a + (16u ^ swb), a + (32u ^ swb), a + (48u ^ swb), r);
  else if constexpr (NC == 6) lds_vec6(a, r);
  else if constexpr (sizeof(T) == 4) {                  // wider rows (n = 12, ...): 16-byte chunks in natural order
    static_assert(NC % 4 == 0, "float rows in 16-byte chunks");
#pragma unroll
    for (int c = 0; c < NC / 4; ++c) lds_chunk(a + 16u * c, r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
  } else {
    static_assert(NC % 2 == 0, "double rows in 16-byte chunks");
#pragma unroll
    for (int c = 0; c < NC / 2; ++c) lds_chunk(a + 16u * c, r[2 * c], r[2 * c + 1]);
  }
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
