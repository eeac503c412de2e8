// tmpc_api.cu — the C ABI of include/tmpc.h: argument checking, workspace layout, kernel-family dispatch.
// No CPU fallback: every compute entry point needs a CUDA device and returns TMPC_E_CUDA otherwise.
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>
#include "tmpc_common.cuh"
#include "tmpc_factor.cuh"
#include "tmpc_factor2.cuh"
#include "tmpc_factor3.cuh"
#include "tmpc_admm.cuh"
#include "tmpc_admm2.cuh"
#include "tmpc_admm3.cuh"
#include "tmpc_stream.cuh"
#include "tmpc_misc.cuh"
#include "tmpc_backward.cuh"
#include "tmpc_cr.cuh"
#include "tmpc_cr2.cuh"
#include "tmpc_peak.cuh"
#include "tmpc_sqp.cuh"
#include "tmpc_srb.cuh"

using namespace tmpc;

namespace {

constexpr size_t kMaxSmem = 227 * 1024;
inline size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
inline size_t esize(int dtype) { return dtype == TMPC_F64 ? 8 : 4; }

struct Layout {   // byte offsets into the workspace
  size_t Lam, Sinv, atil, eta, fstatus, ad_rho, ad_np, ad_nd, ad_rp, ad_rd, ad_obj, ad_active, ad_mask, ad_iters, ad_conv, ad_count, cls, soft_adj, rhs, w_rows, lo_adj, hi_adj, q_adj, ax, azg, ayf, ayg, axi, zero_xinit, zero_b, res, cr, total;
};

// Cyclic reduction (tmpc_cr.cuh) exists for n = 6 and n = 8 and pays off for a few very long horizons; TMPC_LIN_AUTO picks it
// only there and keeps the sequential families for every other shape.
bool use_cr(const tmpc_config& c) {
  if (c.linsolve == TMPC_LIN_CYCLIC_REDUCTION) return true;
  const int n = c.nx + c.nu;
  if (c.linsolve == TMPC_LIN_AUTO) return c.batch <= 4 && c.N >= 1024 && (n == 6 || n == 8);
  return false;
}

Dims make_dims(const tmpc_config& c) {
  Dims d; memset(&d, 0, sizeof(d));
  d.B = c.batch; d.N = c.N; d.T = c.N + 1; d.nx = c.nx; d.nu = c.nu; d.n = c.nx + c.nu; d.ng = c.ng;
  d.nz = d.T * d.n; d.mf = c.nx + c.N * c.nx; d.mg = d.T * c.ng; d.g_sel = c.g_is_selection;
  for (int r = 0; r < c.ng && r < TMPC_MAX_NG; ++r) { d.g_col[r] = c.g_col[r]; if (c.soft_row[r]) d.soft_mask |= 1u << r; }
  return d;
}

bool plan_xg(const tmpc_config& c);      // the resident kernel keeps X and A~ in global memory (long horizons of n = 12): defined beside fast_plan()

Layout make_layout(const tmpc_config& c) {
  const Dims d = make_dims(c); const size_t es = esize(c.dtype), B = d.B, nn = (size_t)d.n * d.n;
  Layout L; size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  L.Lam = take(B * d.T * nn * es); L.Sinv = take(B * d.T * nn * es); L.eta = take(B * d.nz * es);
  // X, A~ and G~ rows in the stage-minor layout of atil_kernel (16-byte chunks, horizon padded to 8 stages), only for the handles whose plan reads it
  L.atil = take(plan_xg(c) ? B * ((size_t)d.n + 2 * d.nx + (d.g_sel ? 0 : d.ng)) * ((d.n * es + 15) / 16) * (size_t)((d.T + 7) / 8 * 8) * 16 : 0);
  L.fstatus = take(B * sizeof(int32_t));       // per-problem TMPC_ST_PIVOT word of the last tmpc_factor
  // f1 (tmpc_admm_solve_adaptive): per-problem rho_bar, eq. 4 scales, residuals / objective when the caller passes no info, flags, counters
  L.ad_rho = take(B * es); L.ad_np = take(B * es); L.ad_nd = take(B * es); L.ad_rp = take(B * es); L.ad_rd = take(B * es); L.ad_obj = take(B * es);
  L.ad_active = take(B * sizeof(int32_t)); L.ad_mask = take(B * sizeof(int32_t)); L.ad_iters = take(B * sizeof(int32_t)); L.ad_conv = take(B * sizeof(int32_t));
  L.ad_count = take(256);
  L.cls = take(B * d.mg); L.soft_adj = take(B * d.mg);
  L.rhs = take(B * d.nz * es); L.w_rows = take(B * d.mg * es); L.lo_adj = take(B * d.mg * es); L.hi_adj = take(B * d.mg * es);
  L.q_adj = take(B * d.nz * es); L.ax = take(B * d.nz * es); L.azg = take(B * d.mg * es); L.ayf = take(B * d.mf * es);
  L.ayg = take(B * d.mg * es); L.axi = take(B * d.mg * es); L.zero_xinit = take(B * d.nx * es); L.zero_b = take(B * (size_t)d.N * d.nx * es);
  L.res = take(B * 64 * 4 * sizeof(double));
  L.cr = take(use_cr(c) ? cr_workspace_bytes(d, es) : 0);   // cyclic-reduction scratch only for handles that use it
  L.total = o;
  return L;
}

tmpc_status check_cfg(const tmpc_config* c) {
  if (!c) return TMPC_E_BADARG;
  if (c->batch < 1 || c->N < 1 || c->nx < 1 || c->nu < 0 || c->ng < 0) return TMPC_E_DIM;
  if (c->ng > TMPC_MAX_NG) return TMPC_E_DIM;
  if (c->dtype != TMPC_F32 && c->dtype != TMPC_F64) return TMPC_E_BADARG;
  if (!(c->sigma > 0) || !(c->rho_bar > 0) || !(c->rho_eq_scale > 0) || !(c->alpha > 0 && c->alpha < 2)) return TMPC_E_BADARG;
  if (!(c->slack_gamma >= 0) || !(c->slack_lambda >= 0)) return TMPC_E_BADARG;
  if (c->g_is_selection) for (int r = 0; r < c->ng; ++r) if (c->g_col[r] < 0 || c->g_col[r] >= c->nx + c->nu) return TMPC_E_BADARG;
  if (c->model == TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT && (c->nx != 4 || c->nu != 2 || c->ng != 3 || c->g_is_selection)) return TMPC_E_DIM;
  if (c->model == TMPC_MODEL_SRB_HUMANOID_RK4 && (c->nx != 12 || c->nu != 6 || (c->ng > 0 && !c->g_is_selection) || !(c->model_params[0] > 0) ||
                                                 !(c->model_params[4] > 0) || !(c->model_params[5] > 0) || !(c->model_params[6] > 0) || !(c->dt > 0))) return TMPC_E_DIM;
  if (c->model != TMPC_MODEL_NONE && c->model != TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT && c->model != TMPC_MODEL_SRB_HUMANOID_RK4) return TMPC_E_BADARG;
  return TMPC_OK;
}

}  // namespace

struct tmpc_ctx {
  tmpc_config cfg; Dims d; Layout lay; unsigned char* ws; cudaStream_t stream; bool factored; bool cr; bool twisted; int64_t launches;
  // set while tmpc_admm_solve_adaptive runs (f1): per-problem rho_bar, activity flags for the solve kernels, refactor mask for the factor kernels
  const void* cur_rho; const int32_t* cur_active; const int32_t* cur_mask;
  bool bwd_classified;                          // tmpc_backward has left the row classification of its state in the workspace
  cudaStream_t aux[2]; cudaEvent_t ev[3];       // tmpc_admm_solve_host: two sub-batches in flight (copies of one overlap the kernels of the other)
  bool mask_sparse;                             // hint for the masked factor launch: few problems flagged (later rounds of f1)
  bool atil_valid;                              // the stage-minor scratch of the chain-resident variants matches the factor in the workspace
  int32_t* pin_live; cudaEvent_t ad_ev[2];      // tmpc_admm_solve_adaptive: pinned landing slots of the per-round live counts and their events (created on first use)
};

namespace {

template <typename T> QpView<T> view(const tmpc_qp* q) {
  QpView<T> v;
  v.D = (const T*)q->D; v.sD = q->D_bstride; v.E = (const T*)q->E; v.sE = q->E_bstride; v.q = (const T*)q->q;
  v.Am = (const T*)q->Am; v.Ap = (const T*)q->Ap; v.b = (const T*)q->b; v.x_init = (const T*)q->x_init;
  v.G = (const T*)q->G; v.sG = q->G_bstride; v.lo = (const T*)q->lo; v.hi = (const T*)q->hi;
  return v;
}
template <typename T> Params<T> params(const tmpc_config& c) {
  Params<T> p; p.sigma = (T)c.sigma; p.rho_g = (T)c.rho_bar; p.rho_f = (T)(c.rho_eq_scale * c.rho_bar); p.alpha = (T)c.alpha;
  p.gamma = (T)c.slack_gamma; p.lam = (T)c.slack_lambda; return p;
}
inline bool cuda_ok() { return cudaGetLastError() == cudaSuccess; }


// ---- factor launch (a2 + a3)
template <typename T>
tmpc_status launch_factor(tmpc_ctx* h, const tmpc_qp* qp, double w_eq, double w_in, const T* w_rows, int32_t* status) {
  FactorArgs<T> a; a.d = h->d; a.qp = view<T>(qp); a.sigma = h->cfg.sigma; a.w_eq = w_eq; a.w_in = w_in; a.w_rows = w_rows;
  a.rho_bar = w_rows ? nullptr : (const T*)h->cur_rho; a.rho_scale = h->cfg.rho_eq_scale; a.mask = w_rows ? nullptr : h->cur_mask;
  a.Lam = (T*)(h->ws + h->lay.Lam); a.Sinv = (T*)(h->ws + h->lay.Sinv); a.status = status;
  h->atil_valid = false;                                // another factor form takes the workspace
  // small compile-time shapes: the warp-level kernel in its one-directional form (tmpc_factor2.cuh)
  if (h->d.n == 8 && h->d.nx == 6 && h->d.ng <= 8) { factor_tw2_kernel<T, 8, 6, false><<<h->d.B, 32, 0, h->stream>>>(a); h->launches++; return cuda_ok() ? TMPC_OK : TMPC_E_CUDA; }
  if (h->d.n == 6 && h->d.nx == 4 && h->d.ng <= 6) { factor_tw2_kernel<T, 6, 4, false><<<h->d.B, 32, 0, h->stream>>>(a); h->launches++; return cuda_ok() ? TMPC_OK : TMPC_E_CUDA; }
  const int nn = h->d.n * h->d.n;
  {                                      // large blocks: register-tiled products (tmpc_factor3.cuh)
    const int nt8 = f3_ld(h->d.n) / 8; const size_t smem3 = factor3_smem<T>(h->d.n);   // 4 x 4 warps x (3 x 3) tiles of 8 x 8
    if (h->d.n >= 32 && nt8 <= 12 && smem3 <= kMaxSmem) {
      auto k3 = factor3_kernel<T>;
      if (cudaFuncSetAttribute(k3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem3) != cudaSuccess) return TMPC_E_CUDA;
      k3<<<h->d.B, 512, smem3, h->stream>>>(a); h->launches++;
      return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
    }
  }
  int nt = ((nn + 31) / 32) * 32; if (nt > 1024) nt = 1024; if (nt < 32) nt = 32;
  const size_t smem = 3 * (size_t)nn * sizeof(double);
  if (smem > kMaxSmem) return TMPC_E_UNSUPPORTED;
  auto k = factor_kernel<T, double>;
  if (smem > 48 * 1024 && cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return TMPC_E_CUDA;
  k<<<h->d.B, nt, smem, h->stream>>>(a); h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}

// ---- ADMM launch (a4..a9); also serves tmpc_kkt_solve and the REUSE backward mode
template <typename T, int NC, bool RES>
tmpc_status launch_admm_inst(tmpc_ctx* h, const AdmmArgs<T>& a, int nt, size_t smem) {
  auto k = admm_kernel<T, NC, RES>;
  if (smem > 48 * 1024 && cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return TMPC_E_CUDA;
  k<<<h->d.B, nt, smem, h->stream>>>(a); h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}
struct FastPlan { bool ok, xg, cl; int pg, nt, ctas_per_sm; size_t smem; };   // xg: X / A~ in global memory; cl: one problem on a cluster of two CTAs
template <typename T> FastPlan fast_plan(const Dims& d);
template <typename T> tmpc_status launch_resident(tmpc_ctx* h, const AdmmArgs<T>& a, const FastPlan& f);
template <typename T> tmpc_status launch_residual(tmpc_ctx* h, const AdmmArgs<T>& s);
template <typename T>
tmpc_status launch_admm(tmpc_ctx* h, AdmmArgs<T>& a) {
  const Dims& d = h->d;
  if (h->twisted) {                      // the factor in the workspace is the twisted one: only admm3_kernel reads it
    tmpc_status s = launch_resident<T>(h, a, fast_plan<T>(d));
    if (s != TMPC_OK || a.kkt_only) return s;
    return launch_residual<T>(h, a);
  }
  size_t smem_res = admm_smem_elems(d, true) * sizeof(T), smem_str = admm_smem_elems(d, false) * sizeof(T);
  const bool res = smem_res <= kMaxSmem;
  if (!res) {                            // streamed class: bulk-copy ring (tmpc_stream.cuh) when the shape allows it
    const StreamPlan sp = stream_plan<T>(d, kMaxSmem);
    const int V = 16 / (int)sizeof(T);
    if ((d.n * d.n) % V == 0 && (d.nx * d.n) % V == 0 && d.n % V == 0 && 4 * d.ng <= sp.nthreads - 32 && sp.slots >= 2 && sp.nthreads <= 1024) {
      StreamArgs<T> S; S.a = a; S.LD = sp.LD; S.slots = sp.slots; S.tile_elems = sp.tile_elems; S.eta = (T*)(h->ws + h->lay.eta);
      S.g0 = 0; S.chunks = 1;
      auto k = admm_stream_kernel<T>;
      if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sp.smem) != cudaSuccess) return TMPC_E_CUDA;
      // Wave quantisation: a CTA runs at a fixed rate (measured: B = 296 = one full wave of 2 CTAs x 148 SMs takes 44.6 ms,
      // B = 512 takes 87.4 ms, B = 592 89.4 ms), so a partial last wave costs a whole one.  The ADMM state between two
      // iterations is complete in global memory (warm start = resume), hence the solve is cut into `chunks` iteration
      // ranges per problem and the B x chunks jobs, ordered (chunk, problem), are run `cslots` at a time in successive
      // launches: consecutive jobs of a launch are distinct problems and a problem's previous chunk sits >= one launch
      // earlier (B > cslots).  Cost model: launches x iterations per chunk, plus the eta pass each launch repeats.
      int per_sm = 0, dev = 0, sms = 0;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, sp.nthreads, sp.smem) != cudaSuccess || cudaGetDevice(&dev) != cudaSuccess ||
          cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return TMPC_E_CUDA;
      const long long cslots = (long long)per_sm * sms;
      int best_c = 1;
      if (!a.kkt_only && cslots > 0 && d.B > cslots && a.iters >= 32) {
        double best = (double)((d.B + cslots - 1) / cslots) * (a.iters + 0.3);
        for (int c = 2; c <= 8 && a.iters / c >= 16; ++c) {
          const long long rounds = ((long long)d.B * c + cslots - 1) / cslots;
          const double cost = (double)rounds * ((a.iters + c - 1) / c + 0.3);
          if (cost < 0.97 * best) { best = cost; best_c = c; }
        }
      }
      S.chunks = best_c;
      const long long jobs = (long long)d.B * best_c, per = best_c > 1 ? cslots : jobs;
      for (long long g0 = 0; g0 < jobs; g0 += per) {
        S.g0 = (int)g0;
        const long long grid = jobs - g0 < per ? jobs - g0 : per;
        k<<<(unsigned)grid, sp.nthreads, sp.smem, h->stream>>>(S); h->launches++;
      }
      if (!cuda_ok()) return TMPC_E_CUDA;
      return a.kkt_only ? TMPC_OK : launch_residual<T>(h, a);
    }
  }
  if (!res && smem_str > kMaxSmem) return TMPC_E_UNSUPPORTED;
  int nt = ((d.nz + 31) / 32) * 32; if (nt > 1024) nt = 1024; if (nt < 64) nt = 64;
  if (res) {
    if (a.active) {                      // adaptive schedule (f1): the eq. 4 scales come from residual_kernel, not from the in-kernel residuals
      AdmmArgs<T> b = a; b.r_prim = b.r_dual = b.objective = nullptr; b.status = nullptr;
      const tmpc_status s = d.n == 6 ? launch_admm_inst<T, 6, true>(h, b, nt, smem_res) : d.n == 8 ? launch_admm_inst<T, 8, true>(h, b, nt, smem_res)
                                                                                                    : launch_admm_inst<T, 0, true>(h, b, nt, smem_res);
      return s != TMPC_OK ? s : launch_residual<T>(h, a);
    }
    if (d.n == 6) return launch_admm_inst<T, 6, true>(h, a, nt, smem_res);
    if (d.n == 8) return launch_admm_inst<T, 8, true>(h, a, nt, smem_res);
    return launch_admm_inst<T, 0, true>(h, a, nt, smem_res);
  }
  return launch_admm_inst<T, 0, false>(h, a, nt, smem_str);
}

// ---- resident fast path (tmpc_admm3.cuh): eligibility and launch shape
constexpr size_t kSmemPerSM = 228 * 1024;
int sm_count() {
  static int sms = 0;
  if (sms == 0) { int dev = 0; if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) { cudaGetLastError(); sms = 148; } }
  return sms;
}
template <typename T>
FastPlan fast_plan(const Dims& d) {
  FastPlan f; f.ok = false; f.xg = false; f.cl = false; f.pg = 1; f.nt = 0; f.ctas_per_sm = 0; f.smem = 0;
  const bool shape = (d.n == 8 && d.nx == 6) || (d.n == 6 && d.nx == 4) || (d.n == 12 && d.nx == 8);   // (12, 8): the nominal block size of the paper's scaling study (f4)
  if (!shape || d.ng > d.n || d.T < 2) return f;
  if (d.g_sel) for (int r = 0; r < d.ng; ++r) for (int q = 0; q < r; ++q) if (d.g_col[r] == d.g_col[q]) return f;   // one selection row per column
  const size_t s1 = d.n == 8 ? admm3_smem_bytes<T, 8, 6>(d, 1) : d.n == 6 ? admm3_smem_bytes<T, 6, 4>(d, 1) : admm3_smem_bytes<T, 12, 8>(d, 1);
  const size_t s2 = d.n == 8 ? admm3_smem_bytes<T, 8, 6>(d, 2) : d.n == 6 ? admm3_smem_bytes<T, 6, 4>(d, 2) : kMaxSmem + 1;   // n = 12: one problem per CTA (16 chain lanes per slot)
  if (s1 > kMaxSmem) {
    // The full records of one problem do not fit one SM.  In order of preference:
    // (1) (12, 8) block, batch that leaves half of the SMs idle anyway: a CLUSTER of two CTAs per problem (tmpc_admm3.cuh, CL) with full records,
    //     if the two halves fit two SMs — about half the latency per iteration of (2); for batches that fill the GPU (2) is ~8 % faster
    //     (15.9 vs 17.4 ms per 100 iterations at (1024,80,8,4) fp64);
    const int half = d.T / 2 + 1, ntc = 32 + (2 * half + 31) / 32 * 32;
    const bool cl_shape = d.n == 12 && d.T >= 8 && ntc <= 384;
    if (cl_shape && 2 * d.B <= sm_count()) {
      const size_t sr = admm3_cl_smem_bytes<T, 12, 8, false>(d);
      if (sr <= kMaxSmem) { f.ok = true; f.cl = true; f.nt = ntc; f.ctas_per_sm = 1; f.smem = sr; return f; }
    }
    // (2) one CTA per problem with only the chain's share of a record in shared memory (Rec3<.., XG>), the rest from the stage-minor global scratch;
    const size_t sx = d.n == 8 ? admm3_smem_bytes<T, 8, 6, true>(d, 1) : d.n == 6 ? admm3_smem_bytes<T, 6, 4, true>(d, 1) : admm3_smem_bytes<T, 12, 8, true>(d, 1);
    const int ntx = 32 + (2 * d.T + 31) / 32 * 32;
    // (3) (12, 8) block: the cluster pair with the chain's share, when even that does not fit one SM (where it fits, (2) is faster: 37 against
    //     50 us per iteration at (64,160,8,4) fp64).
    const bool one_fits = sx <= kMaxSmem && ntx <= 1024;
    if (cl_shape && !one_fits) {
      const size_t sc = admm3_cl_smem_bytes<T, 12, 8, true>(d);
      if (sc <= kMaxSmem) { f.ok = true; f.xg = true; f.cl = true; f.nt = ntc; f.ctas_per_sm = 1; f.smem = sc; return f; }
    }
    if (!one_fits) return f;
    f.ok = true; f.xg = true; f.pg = 1; f.nt = ntx; f.ctas_per_sm = (int)(kSmemPerSM / (sx + 1024)); f.smem = sx;
    return f;
  }
  const int c1 = (int)(kSmemPerSM / (s1 + 1024)), c2 = s2 <= kMaxSmem ? (int)(kSmemPerSM / (s2 + 1024)) : 0;
  f.pg = (d.B >= 2 && c2 >= 2 && 2 * c2 >= c1) ? 2 : 1;
  const int ipt = d.n / 2;                                 // rows of a stage per item thread (admm3: two lanes per stage)
  auto threads = [&](int pg) { int t = ((pg * d.nz + ipt - 1) / ipt + 31) / 32 * 32; return 32 + (t < 32 ? 32 : t); };   // + the chain warp
  const int tmax = 1024;
  if (threads(f.pg) > tmax) f.pg = 1;
  f.nt = threads(f.pg);
  if (f.nt > tmax) return f;
  f.smem = f.pg == 2 ? s2 : s1; f.ctas_per_sm = f.pg == 2 ? c2 : c1; f.ok = true;
  return f;
}

bool plan_xg(const tmpc_config& c) {
  const Dims d = make_dims(c);
  return c.dtype == TMPC_F64 ? fast_plan<double>(d).xg : fast_plan<float>(d).xg;
}

template <typename T, int NC, int NX, int PG, int MAXT, int MINB, bool XG = false, bool CL = false>
tmpc_status launch_admm3_inst(tmpc_ctx* h, const AdmmArgs<T>& a, const FastPlan& f) {
  auto k = admm3_kernel<T, NC, NX, PG, MAXT, MINB, XG, CL>;
  if (f.smem > 48 * 1024 && cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f.smem) != cudaSuccess) return TMPC_E_CUDA;
  const unsigned grid = (unsigned)((h->d.B + PG - 1) / PG);
  Admm3Args<T> A; A.a = a; A.atil = nullptr;
  if constexpr (CL) A.pl = admm3_cl_plan<T, NC, NX, XG>(h->d); else A.pl = admm3_plan<T, NC, NX, XG>(h->d, PG);
  A.tpad = (h->d.T + 7) / 8 * 8;
  if constexpr (XG) {
    T* atil = (T*)(h->ws + h->lay.atil); A.atil = atil;
    // The scratch depends on the factor and the constraint blocks only: it is rebuilt in full after a full (or adjoint) factorisation, for the
    // re-factored problems after a masked one (f1, SQP: cur_mask still holds the mask that factorisation took), and not at all otherwise.
    const int rows = a.kkt_only ? h->d.n : h->d.n + 2 * h->d.nx + (h->d.g_sel ? 0 : h->d.ng);      // tmpc_kkt_solve needs X only
    const long long work = (long long)h->d.B * rows * h->d.T;
    const bool full = !h->atil_valid;
    if (full || h->cur_mask) { atil_kernel<T><<<(unsigned)((work + 127) / 128), 128, 0, h->stream>>>(a, atil, A.tpad, rows, full ? nullptr : h->cur_mask); h->launches++; }
    if (full && !a.kkt_only) h->atil_valid = true;
  }
  A.rfa = a.prm.rho_f * a.prm.alpha; A.oma = T(1) - a.prm.alpha; A.inv_rho_g = T(1) / a.prm.rho_g; A.inv_rg = T(1) / (a.prm.rho_g + a.prm.gamma);
  if constexpr (CL) {                                   // two CTAs per problem, launched as a cluster
    cudaLaunchConfig_t lc; memset(&lc, 0, sizeof(lc));
    lc.gridDim = dim3(2u * (unsigned)h->d.B); lc.blockDim = dim3((unsigned)f.nt); lc.dynamicSmemBytes = f.smem; lc.stream = h->stream;
    cudaLaunchAttribute at[1]; at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.attrs = at; lc.numAttrs = 1;
    if (cudaLaunchKernelEx(&lc, k, A) != cudaSuccess) { cudaGetLastError(); return TMPC_E_CUDA; }
    h->launches++;
    return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
  }
  k<<<grid, f.nt, f.smem, h->stream>>>(A); h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}
template <typename T, int NC, int NX, int PG>
tmpc_status launch_admm3_shape(tmpc_ctx* h, const AdmmArgs<T>& a, const FastPlan& f) {
  if (f.nt <= 256) {
    // a grid that leaves SMs idle anyway (config 1: one problem) takes the variant without a register cap: the capped ones spill for double
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return TMPC_E_CUDA;
    if ((h->d.B + PG - 1) / PG <= sms) return launch_admm3_inst<T, NC, NX, PG, 256, 1>(h, a, f);
    if constexpr (sizeof(T) == 8) { if (f.nt <= 192 && f.ctas_per_sm == 2) return launch_admm3_inst<T, NC, NX, PG, 192, 2>(h, a, f); }   // 170 registers: no spills for double
    if (f.ctas_per_sm >= 3) return launch_admm3_inst<T, NC, NX, PG, 256, 3>(h, a, f);
    if (f.ctas_per_sm >= 2) return launch_admm3_inst<T, NC, NX, PG, 256, 2>(h, a, f);
    return launch_admm3_inst<T, NC, NX, PG, 256, 1>(h, a, f);
  }
  return launch_admm3_inst<T, NC, NX, PG, 1024, 1>(h, a, f);
}
template <typename T, int NC, int NX>
tmpc_status launch_admm3_xg(tmpc_ctx* h, const AdmmArgs<T>& a, const FastPlan& f) {      // chain-resident variant: thread caps by horizon
  if (f.nt <= 384) return launch_admm3_inst<T, NC, NX, 1, 384, 1, true>(h, a, f);
  if (f.nt <= 704) return launch_admm3_inst<T, NC, NX, 1, 704, 1, true>(h, a, f);
  return launch_admm3_inst<T, NC, NX, 1, 1024, 1, true>(h, a, f);
}
template <typename T>
tmpc_status launch_resident(tmpc_ctx* h, const AdmmArgs<T>& a, const FastPlan& f) {
  const Dims& d = h->d;
  if (f.cl) return f.xg ? launch_admm3_inst<T, 12, 8, 1, 384, 1, true, true>(h, a, f) : launch_admm3_inst<T, 12, 8, 1, 384, 1, false, true>(h, a, f);
  if (f.xg) {
    if (d.n == 12) return launch_admm3_xg<T, 12, 8>(h, a, f);
    if (d.n == 8) return launch_admm3_xg<T, 8, 6>(h, a, f);
    if (d.n == 6) return launch_admm3_xg<T, 6, 4>(h, a, f);
  }
  if (d.n == 8) return f.pg == 2 ? launch_admm3_shape<T, 8, 6, 2>(h, a, f) : launch_admm3_shape<T, 8, 6, 1>(h, a, f);
  if (d.n == 6) return f.pg == 2 ? launch_admm3_shape<T, 6, 4, 2>(h, a, f) : launch_admm3_shape<T, 6, 4, 1>(h, a, f);
  if (d.n == 12) return launch_admm3_shape<T, 12, 8, 1>(h, a, f);
  return TMPC_E_UNSUPPORTED;
}
template <typename T>
tmpc_status launch_factor_tw(tmpc_ctx* h, const tmpc_qp* qp, double w_eq, double w_in, int32_t* status, const T* w_rows = nullptr) {
  FactorArgs<T> a; a.d = h->d; a.qp = view<T>(qp); a.sigma = h->cfg.sigma; a.w_eq = w_eq; a.w_in = w_in; a.w_rows = w_rows;
  a.rho_bar = w_rows ? nullptr : (const T*)h->cur_rho; a.rho_scale = h->cfg.rho_eq_scale; a.mask = w_rows ? nullptr : h->cur_mask;
  if (!a.mask) h->atil_valid = false;                   // every problem's factor changes (a masked factorisation is followed by a masked atil_kernel)
  a.Lam = (T*)(h->ws + h->lay.Lam); a.Sinv = (T*)(h->ws + h->lay.Sinv); a.status = status;
  // Warps per chain (tmpc_factor2.cuh): a launch that cannot fill the GPU lasts as long as ONE problem's chain, so small batches take four (n = 12:
  // eight) warps per chain; MASKED launches after the first check of f1 (typically a few flagged problems, the other CTAs leave at once) and mid-size batches of
  // the (12, 8) block (up to eight per SM) take four warps at four CTAs per SM; everything else keeps one warp per chain, twelve CTAs per SM
  // (measured at B = 1024: n = 12 fp64 475 -> 459 us, but n = 8 config 2 1.05 -> 1.16 ms per step with four warps).
  const int B = h->d.B, sms = sm_count();
  const int wpc = B <= 2 * sms ? ((h->d.n == 12 && B <= sms) ? 8 : 4) : (((a.mask && h->mask_sparse) || (h->d.n == 12 && B <= 8 * sms)) ? 44 : 1);      // 44: four warps, four CTAs per SM
  auto go = [&](auto nc, auto nx) {
    constexpr int NC = decltype(nc)::value, NX = decltype(nx)::value;
    if (wpc == 8) { if constexpr (NC == 12) factor_tw2_kernel<T, NC, NX, true, 8><<<B, 512, 0, h->stream>>>(a); }
    else if (wpc == 4) factor_tw2_kernel<T, NC, NX, true, 4><<<B, 256, 0, h->stream>>>(a);
    else if (wpc == 44) factor_tw2_kernel<T, NC, NX, true, 4, 4><<<B, 256, 0, h->stream>>>(a);
    else factor_tw2_kernel<T, NC, NX, true><<<B, 64, 0, h->stream>>>(a);
  };
  if (h->d.n == 8 && h->d.nx == 6 && h->d.ng <= 8) go(std::integral_constant<int, 8>(), std::integral_constant<int, 6>());
  else if (h->d.n == 6 && h->d.nx == 4 && h->d.ng <= 6) go(std::integral_constant<int, 6>(), std::integral_constant<int, 4>());
  else if (h->d.n == 12 && h->d.nx == 8 && h->d.ng <= 12) go(std::integral_constant<int, 12>(), std::integral_constant<int, 8>());
  else return TMPC_E_UNSUPPORTED;      // fast_plan() only admits the shapes above
  h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}
template <typename T>
tmpc_status launch_residual(tmpc_ctx* h, const AdmmArgs<T>& s) {
  if (!s.r_prim && !s.r_dual && !s.objective && !s.status) return TMPC_OK;
  ResidualArgs<T> r; r.d = h->d; r.prm = s.prm; r.qp = s.qp; r.x = s.x; r.zg = s.zg; r.yf = s.yf; r.yg = s.yg; r.xi = s.xi;
  r.r_prim = s.r_prim; r.r_dual = s.r_dual; r.objective = s.objective; r.status = s.status;
  r.norm_prim = nullptr; r.norm_dual = nullptr; r.active = s.active;
  if (s.active) { r.norm_prim = (T*)(h->ws + h->lay.ad_np); r.norm_dual = (T*)(h->ws + h->lay.ad_nd); }
  int nt = ((h->d.nz + 31) / 32) * 32; if (nt > 256) nt = 256;
  int nparts = 1;                        // few long problems: several CTAs per problem, partials reduced in a fixed order
  if (h->d.B < 64 && !s.active) { nparts = (h->d.nz + 2047) / 2048; if (nparts > 64) nparts = 64; if (nparts < 1) nparts = 1; }
  r.partial = (double*)(h->ws + h->lay.res); r.nparts = nparts;
  residual_kernel<T><<<dim3(h->d.B, nparts), nt, 0, h->stream>>>(r); h->launches++;
  if (nparts > 1) { residual_finish_kernel<T><<<(h->d.B + 63) / 64, 64, 0, h->stream>>>(r); h->launches++; }
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}

template <typename T>
tmpc_status do_factor(tmpc_ctx* h, const tmpc_qp* qp) {
  const double rho_f = h->cfg.rho_eq_scale * h->cfg.rho_bar, rho_g = h->cfg.rho_bar;
  int32_t* fstatus = (int32_t*)(h->ws + h->lay.fstatus);
  if (h->cr) {                           // the cyclic-reduction kernels keep their own per-problem pivot flag and OR it in themselves
    if (cudaMemsetAsync(fstatus, 0, (size_t)h->d.B * sizeof(int32_t), h->stream) != cudaSuccess) return TMPC_E_CUDA;
    return cr_factor<T>(h->d, view<T>(qp), h->cfg.sigma, rho_f, rho_g, h->ws + h->lay.cr, h->stream, &h->launches);
  }
  h->twisted = fast_plan<T>(h->d).ok;
  if (h->twisted) return launch_factor_tw<T>(h, qp, rho_f, rho_g, fstatus);
  return launch_factor<T>(h, qp, rho_f, rho_g, nullptr, fstatus);
}

// info.status[b] <- pivot word of the last tmpc_factor (overwrites whatever the caller's buffer held); the solve kernels OR TMPC_ST_NAN in
__global__ void status_init_kernel(int B, const int32_t* __restrict__ fstatus, int32_t* __restrict__ status) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < B) status[p] = fstatus[p];
}

template <typename T>
tmpc_status do_solve(tmpc_ctx* h, const tmpc_qp* qp, tmpc_state* st, int iters, int flags, tmpc_info* info) {
  if (info && info->status) {
    status_init_kernel<<<(h->d.B + 255) / 256, 256, 0, h->stream>>>(h->d.B, (const int32_t*)(h->ws + h->lay.fstatus), info->status); h->launches++;
    if (!cuda_ok()) return TMPC_E_CUDA;
  }
  if (h->cr) {
    // chunked form (tmpc_cr2.cuh) when the horizon is long enough and one CTA per chunk (+1) is co-resident
    const Dims& d = h->d;
    const int nchunks = (d.T + CR2_CS - 1) / CR2_CS, S = d.N / CR2_CS + 1;
    int dev = 0, sms = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const bool shape = (d.n == 6 && d.nx == 4) || (d.n == 8 && d.nx == 6);
    if (shape && d.T >= 4 * CR2_CS && (long long)(nchunks + 1) * d.B <= sms && 3 * S * d.n + S * d.nx <= 3 * 4096) {
      const size_t smem = (d.n == 6 ? cr2_smem_elems<T, 6, 4>(d.ng, S) : cr2_smem_elems<T, 8, 6>(d.ng, S)) * sizeof(T);
      if (smem <= kMaxSmem) {
        CrAdmmArgs<T> a; memset(&a, 0, sizeof(a));
        a.d = d; a.prm = params<T>(h->cfg); a.qp = view<T>(qp); a.ws = h->ws + h->lay.cr;
        a.x = (T*)st->x; a.zg = (T*)st->zg; a.yf = (T*)st->yf; a.yg = (T*)st->yg; a.xi = (T*)st->xi;
        a.status = info ? info->status : nullptr; a.iters = iters; a.zg_given = (flags & TMPC_SOLVE_ZG_GIVEN) != 0;
        void* kern = d.n == 6 ? (void*)cr2_admm_kernel<T, 6, 4> : (void*)cr2_admm_kernel<T, 8, 6>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return TMPC_E_CUDA;
        int nch = nchunks; void* params_[] = { (void*)&a, (void*)&nch };
        if (cudaLaunchCooperativeKernel(kern, dim3((unsigned)nchunks + 1, (unsigned)d.B), dim3(256), params_, smem, h->stream) != cudaSuccess) { cudaGetLastError(); return TMPC_E_CUDA; }
        h->launches++;
        if (!info) return TMPC_OK;
        AdmmArgs<T> r; memset(&r, 0, sizeof(r));
        r.d = d; r.prm = a.prm; r.qp = a.qp; r.x = a.x; r.zg = a.zg; r.yf = a.yf; r.yg = a.yg; r.xi = a.xi;
        r.r_prim = (T*)info->r_prim; r.r_dual = (T*)info->r_dual; r.objective = (T*)info->objective; r.status = info->status;
        return launch_residual<T>(h, r);
      }
    }
    return cr_admm<T>(h->d, params<T>(h->cfg), view<T>(qp), h->ws + h->lay.cr, (T*)st->x, (T*)st->zg, (T*)st->yf, (T*)st->yg, (T*)st->xi,
                      info ? (T*)info->r_prim : nullptr, info ? (T*)info->r_dual : nullptr, info ? (T*)info->objective : nullptr,
                      info ? info->status : nullptr, iters, (flags & TMPC_SOLVE_ZG_GIVEN) != 0, h->stream, &h->launches);
  }
  AdmmArgs<T> a; memset(&a, 0, sizeof(a));
  a.d = h->d; a.prm = params<T>(h->cfg); a.qp = view<T>(qp);
  a.Lam = (const T*)(h->ws + h->lay.Lam); a.Sinv = (const T*)(h->ws + h->lay.Sinv);
  a.x = (T*)st->x; a.zg = (T*)st->zg; a.yf = (T*)st->yf; a.yg = (T*)st->yg; a.xi = (T*)st->xi;
  if (info) { a.r_prim = (T*)info->r_prim; a.r_dual = (T*)info->r_dual; a.objective = (T*)info->objective; a.status = info->status; }
  a.iters = iters; a.zg_given = (flags & TMPC_SOLVE_ZG_GIVEN) ? 1 : 0;
  a.rho_bar = (const T*)h->cur_rho; a.rho_scale = (T)h->cfg.rho_eq_scale; a.active = h->cur_active;
  return launch_admm<T>(h, a);
}

// ---- f1: Alg. 3 with the adaptive step size (eq. 17) and the termination test (eq. 4).
// Rounds of `check_every` iterations: [solve kernel on the live problems with their own rho_bar] -> [residuals + eq. 4 scales] ->
// [adapt_kernel: terminate / new rho_bar / refactor mask] -> [masked refactor].  The number of live problems comes back to the host
// after every round (4 bytes), so the call returns as soon as every problem has terminated.
// Two pinned ints per handle for the live counts of tmpc_admm_solve_adaptive, handed out round-robin from ONE page-locked page per process
// (cudaHostAlloc costs milliseconds, too much for a handle that lives for one solve; the page is never freed).  512 pairs: more handles than
// that running the adaptive solve at the same time would share landing slots.
int32_t* pinned_pair() {
  static std::mutex mu; static int32_t* pool = nullptr; static unsigned next = 0;
  std::lock_guard<std::mutex> lk(mu);
  if (!pool && cudaHostAlloc((void**)&pool, 1024 * sizeof(int32_t), cudaHostAllocPortable) != cudaSuccess) { cudaGetLastError(); pool = nullptr; return nullptr; }
  return pool + 2 * (next++ % 512u);
}

template <typename T>
tmpc_status do_solve_adaptive(tmpc_ctx* h, const tmpc_qp* qp, tmpc_state* st, const tmpc_adaptive* ad, int flags, tmpc_info* info,
                              int32_t* iters_out, int32_t* conv_out, void* rho_out) {
  const Dims& d = h->d; const Layout& L = h->lay; unsigned char* ws = h->ws;
  if (h->cr) return TMPC_E_UNSUPPORTED;
  T* rho = (T*)(ws + L.ad_rho); int32_t* active = (int32_t*)(ws + L.ad_active); int32_t* mask = (int32_t*)(ws + L.ad_mask);
  int32_t* iters = (int32_t*)(ws + L.ad_iters); int32_t* conv = (int32_t*)(ws + L.ad_conv); int32_t* count = (int32_t*)(ws + L.ad_count);
  tmpc_info li;
  li.r_prim = info && info->r_prim ? info->r_prim : ws + L.ad_rp; li.r_dual = info && info->r_dual ? info->r_dual : ws + L.ad_rd;
  li.objective = info && info->objective ? info->objective : ws + L.ad_obj; li.status = info ? info->status : nullptr;
  const unsigned nb = (unsigned)((d.B + 255) / 256);
  adapt_init_kernel<T><<<nb, 256, 0, h->stream>>>(d.B, (T)h->cfg.rho_bar, rho, active, mask, iters, conv, count); h->launches++;
  if (!cuda_ok()) return TMPC_E_CUDA;
  // The host only needs the live count to stop launching: it reads round r's count AFTER round r + 1 has been enqueued (two counters, two pinned
  // landing slots, two events), so the GPU never idles while the host waits.  A round enqueued after every problem has terminated finds all
  // activity flags clear and changes nothing.
  if (!h->pin_live) { h->pin_live = pinned_pair(); if (!h->pin_live) return TMPC_E_CUDA; }
  for (int e = 0; e < 2; ++e) if (!h->ad_ev[e] && cudaEventCreateWithFlags(&h->ad_ev[e], cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return TMPC_E_CUDA; }
  h->cur_rho = rho; h->cur_active = active; h->cur_mask = mask;
  tmpc_status rc = TMPC_OK;
  int k = 0, f = flags, round = 0;
  while (k < ad->max_iters && rc == TMPC_OK) {
    const int chunk = ad->max_iters - k < ad->check_every ? ad->max_iters - k : ad->check_every;
    rc = do_solve<T>(h, qp, st, chunk, f, &li);          // also runs residual_kernel with the eq. 4 scales (li is never null)
    if (rc != TMPC_OK) break;
    k += chunk; f |= TMPC_SOLVE_ZG_GIVEN;
    int32_t* cnt_r = count + (round & 1);
    if (cudaMemsetAsync(cnt_r, 0, sizeof(int32_t), h->stream) != cudaSuccess) { rc = TMPC_E_CUDA; break; }
    AdaptParams ap; ap.k = k; ap.last = k >= ad->max_iters; ap.adapt_rho = ad->adapt_rho; ap.eps_abs = ad->eps_abs; ap.eps_rel = ad->eps_rel;
    ap.ratio = ad->rho_ratio; ap.rho_min = ad->rho_min; ap.rho_max = ad->rho_max;
    adapt_kernel<T><<<nb, 256, 0, h->stream>>>(d.B, ap, (const T*)li.r_prim, (const T*)li.r_dual, (const T*)(ws + L.ad_np), (const T*)(ws + L.ad_nd), rho, active, mask,
                                              iters, conv, cnt_r); h->launches++;
    if (!cuda_ok() || cudaMemcpyAsync(h->pin_live + (round & 1), cnt_r, sizeof(int32_t), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
        cudaEventRecord(h->ad_ev[round & 1], h->stream) != cudaSuccess) { rc = TMPC_E_CUDA; break; }
    if (round > 0) {                                     // the count of the round before this one
      if (cudaEventSynchronize(h->ad_ev[(round - 1) & 1]) != cudaSuccess) { rc = TMPC_E_CUDA; break; }
      if (h->pin_live[(round - 1) & 1] == 0) break;
    }
    h->mask_sparse = round > 0;                          // the first check re-scales most problems, the later ones a few
    if (ad->adapt_rho && k < ad->max_iters) rc = do_factor<T>(h, qp);          // only the problems whose rho_bar changed (mask)
    ++round;
  }
  h->mask_sparse = false;
  if (rc == TMPC_OK && cudaStreamSynchronize(h->stream) != cudaSuccess) rc = TMPC_E_CUDA;      // the call synchronises (tmpc.h)
  h->cur_rho = nullptr; h->cur_active = nullptr; h->cur_mask = nullptr;
  h->factored = false;                                   // the factor in the workspace now belongs to the per-problem rho_bar values
  if (rc != TMPC_OK) return rc;
  if (iters_out && cudaMemcpyAsync(iters_out, iters, (size_t)d.B * sizeof(int32_t), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  if (conv_out && cudaMemcpyAsync(conv_out, conv, (size_t)d.B * sizeof(int32_t), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  if (rho_out && cudaMemcpyAsync(rho_out, rho, (size_t)d.B * sizeof(T), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  return TMPC_OK;
}

// ---- f2: SQP with linesearch and the eq. 18 stop (Alg. 1, App. D) for the built-in bicycle model.  One linearisation per iteration
// serves both the convergence test of the previous step and the next QP; converged problems are frozen (activity flags of f1).
template <typename T>
tmpc_status do_sqp(tmpc_ctx* h, tmpc_qp* qp, tmpc_state* st, const void* stage_ref, const tmpc_sqp_opts* o, int32_t* iters_out, int32_t* conv_out,
                   void* alpha_log, void* kkt_out) {
  const Dims& d = h->d; const Layout& L = h->lay; unsigned char* ws = h->ws;
  const int model = h->cfg.model;
  if (model != TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT && model != TMPC_MODEL_SRB_HUMANOID_RK4) return TMPC_E_UNSUPPORTED;
  int32_t* active = (int32_t*)(ws + L.ad_active); int32_t* mask = (int32_t*)(ws + L.ad_mask);
  int32_t* iters = (int32_t*)(ws + L.ad_iters); int32_t* conv = (int32_t*)(ws + L.ad_conv); int32_t* count = (int32_t*)(ws + L.ad_count);
  const unsigned nb = (unsigned)((d.B + 255) / 256);
  adapt_init_kernel<T><<<nb, 256, 0, h->stream>>>(d.B, (T)h->cfg.rho_bar, (T*)(ws + L.ad_rho), active, mask, iters, conv, count); h->launches++;
  if (!cuda_ok()) return TMPC_E_CUDA;
  SqpArgs<T> a; memset(&a, 0, sizeof(a));
  a.d = d; a.qp = view<T>(qp); a.Lwb = h->cfg.wheelbase; a.dt = h->cfg.dt; a.gamma = h->cfg.slack_gamma; a.lam = h->cfg.slack_lambda; a.eps_c = o->eps_c; a.eta = o->eta;
  for (int i = 0; i < 13; ++i) a.mp[i] = h->cfg.model_params[i];
  a.n_alpha = o->n_alpha; a.active = active; a.act_rw = active; a.iters = iters; a.converged = conv; a.n_active = count;
  a.ox = (const T*)(ws + L.ax); a.oxi = (const T*)(ws + L.axi); a.oyf = (const T*)(ws + L.ayf); a.oyg = (const T*)(ws + L.ayg);
  a.x = (T*)st->x; a.xi = (T*)st->xi; a.yf = (T*)st->yf; a.yg = (T*)st->yg; a.alpha_log = (T*)alpha_log; a.max_sqp = o->max_sqp; a.kkt = (T*)kkt_out;
  const size_t es = sizeof(T);
  tmpc_status rc = TMPC_OK;
  for (int it = 0; it <= o->max_sqp && rc == TMPC_OK; ++it) {
    rc = tmpc_linearize(h, st->x, stage_ref, qp); if (rc != TMPC_OK) break;
    if (it > 0) {                                         // eq. 18 at the iterate the last step produced
      if (cudaMemsetAsync(count, 0, sizeof(int32_t), h->stream) != cudaSuccess) { rc = TMPC_E_CUDA; break; }
      a.it = it;
      sqp_kkt_kernel<T><<<d.B, 128, 0, h->stream>>>(a); h->launches++;
      int32_t live = 0;
      if (!cuda_ok() || cudaMemcpyAsync(&live, count, sizeof(int32_t), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess ||
          cudaStreamSynchronize(h->stream) != cudaSuccess) { rc = TMPC_E_CUDA; break; }
      if (live == 0 || it == o->max_sqp) break;
    }
    // keep the iterate, solve the QP from it (y carried, z_g re-projected: reading A-26), search along the step
    if (cudaMemcpyAsync(ws + L.ax, st->x, (size_t)d.B * d.nz * es, cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess ||
        cudaMemcpyAsync(ws + L.axi, st->xi, (size_t)d.B * d.mg * es, cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess ||
        cudaMemcpyAsync(ws + L.ayf, st->yf, (size_t)d.B * d.mf * es, cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess ||
        cudaMemcpyAsync(ws + L.ayg, st->yg, (size_t)d.B * d.mg * es, cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) { rc = TMPC_E_CUDA; break; }
    h->cur_active = active; h->cur_mask = active;
    rc = do_factor<T>(h, qp);
    if (rc == TMPC_OK) { h->factored = true; rc = do_solve<T>(h, qp, st, o->admm_iters, 0, nullptr); }
    h->cur_active = nullptr; h->cur_mask = nullptr;
    if (rc != TMPC_OK) break;
    a.it = it;
    if (model == TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT) sqp_linesearch_kernel<T, 1><<<d.B, 32 * (o->n_alpha + 1), 0, h->stream>>>(a);
    else sqp_linesearch_kernel<T, 2><<<d.B, 32 * (o->n_alpha + 1), 0, h->stream>>>(a);
    h->launches++;
    if (!cuda_ok()) rc = TMPC_E_CUDA;
  }
  h->cur_active = nullptr; h->cur_mask = nullptr;
  if (rc != TMPC_OK) return rc;
  if (iters_out && cudaMemcpyAsync(iters_out, iters, (size_t)d.B * sizeof(int32_t), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  if (conv_out && cudaMemcpyAsync(conv_out, conv, (size_t)d.B * sizeof(int32_t), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  return TMPC_OK;
}

template <typename T>
tmpc_status kkt_solve_t(tmpc_handle h, const void* eta, void* xt) {
  AdmmArgs<T> a; memset(&a, 0, sizeof(a));
  a.d = h->d; a.prm = params<T>(h->cfg);
  a.Lam = (const T*)(h->ws + h->lay.Lam); a.Sinv = (const T*)(h->ws + h->lay.Sinv);
  a.x = (T*)eta; a.xi = (T*)xt; a.kkt_only = 1;
  return launch_admm<T>(h, a);
}
}  // namespace

// =================================================================================================== C ABI
extern "C" {

const char* tmpc_status_string(tmpc_status s) {
  switch (s) {
    case TMPC_OK: return "ok";
    case TMPC_E_BADARG: return "bad argument";
    case TMPC_E_DIM: return "bad dimension";
    case TMPC_E_UNSUPPORTED: return "unsupported configuration";
    case TMPC_E_STATE: return "call order: tmpc_factor must precede tmpc_admm_solve / tmpc_backward / tmpc_kkt_solve";
    case TMPC_E_WORKSPACE: return "workspace missing, misaligned or too small";
    case TMPC_E_CUDA: return "CUDA error (or no CUDA device: there is no CPU fallback)";
    case TMPC_E_STATIC_LIMIT: return "problem exceeds the static scratch of tmpc_admm_solve_static (tmpc_workspace_bytes > TMPC_STATIC_SCRATCH_BYTES = 8 MiB)";
  }
  return "unknown";
}

tmpc_status tmpc_workspace_bytes(const tmpc_config* cfg, size_t* bytes) {
  tmpc_status s = check_cfg(cfg); if (s != TMPC_OK) return s;
  if (!bytes) return TMPC_E_BADARG;
  *bytes = make_layout(*cfg).total;
  return TMPC_OK;
}

tmpc_status tmpc_setup(const tmpc_config* cfg, void* workspace, size_t bytes, void* cuda_stream, tmpc_handle* out) {
  tmpc_status s = check_cfg(cfg); if (s != TMPC_OK) return s;
  if (!out) return TMPC_E_BADARG;
  Layout L = make_layout(*cfg);
  if (!workspace || ((uintptr_t)workspace & 255) || bytes < L.total) return TMPC_E_WORKSPACE;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return TMPC_E_CUDA; }
  tmpc_ctx* h = new (std::nothrow) tmpc_ctx;
  if (!h) return TMPC_E_BADARG;
  h->cfg = *cfg; h->d = make_dims(*cfg); h->lay = L; h->ws = (unsigned char*)workspace; h->stream = (cudaStream_t)cuda_stream;
  h->factored = false; h->cr = use_cr(*cfg); h->twisted = false; h->launches = 0;
  h->cur_rho = nullptr; h->cur_active = nullptr; h->cur_mask = nullptr; h->bwd_classified = false;
  h->aux[0] = h->aux[1] = nullptr; h->ev[0] = h->ev[1] = h->ev[2] = nullptr;
  h->pin_live = nullptr; h->ad_ev[0] = h->ad_ev[1] = nullptr; h->atil_valid = false; h->mask_sparse = false;
  // zero buffers of the adjoint QP (x_init = 0, b = 0)
  if (cudaMemsetAsync(h->ws + L.zero_xinit, 0, L.zero_b - L.zero_xinit, h->stream) != cudaSuccess ||
      cudaMemsetAsync(h->ws + L.zero_b, 0, L.cr - L.zero_b, h->stream) != cudaSuccess) { delete h; return TMPC_E_CUDA; }
  if (h->cr) {                           // barrier words of the cyclic-reduction kernels (tmpc_cr.cuh GridBar) start at zero
    const size_t crb = cr_workspace_bytes(h->d, esize(cfg->dtype)), flags = 256 * (size_t)h->d.B + 1024;
    if (cudaMemsetAsync(h->ws + L.cr + crb - flags, 0, flags, h->stream) != cudaSuccess) { delete h; return TMPC_E_CUDA; }
  }
  *out = h;
  return TMPC_OK;
}

tmpc_status tmpc_measure_peak(int32_t what, void* scratch, void* cuda_stream, int32_t reps, double* out) {
  if (what < 0 || what > 3 || !scratch || !out || reps < 1) return TMPC_E_BADARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return TMPC_E_CUDA; }
  return measure_peak(what, (float*)scratch, (cudaStream_t)cuda_stream, reps, out);
}

tmpc_status tmpc_destroy(tmpc_handle h) {
  if (h) {
    for (int k = 0; k < 2; ++k) if (h->aux[k]) cudaStreamDestroy(h->aux[k]);
    for (int k = 0; k < 3; ++k) if (h->ev[k]) cudaEventDestroy(h->ev[k]);
    for (int k = 0; k < 2; ++k) if (h->ad_ev[k]) cudaEventDestroy(h->ad_ev[k]);
  }
  delete h; return TMPC_OK;
}
int64_t tmpc_launch_count(tmpc_handle h) { return h ? h->launches : 0; }

extern "C++" {
template <typename T>
static tmpc_status srb_linearize_launch(tmpc_handle h, const void* xbar, tmpc_qp* qp) {
  SrbArgs<T> a; a.B = h->d.B; a.N = h->d.N; a.dt = (T)h->cfg.dt;
  for (int k = 0; k < 13; ++k) a.mp[k] = (T)h->cfg.model_params[k];
  a.xbar = (const T*)xbar; a.Am = (T*)qp->Am; a.Ap = (T*)qp->Ap; a.b = (T*)qp->b;
  srb_linearize_kernel<T><<<(unsigned)((long long)h->d.B * h->d.N), 32, 0, h->stream>>>(a); h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}
}  // extern "C++"

tmpc_status tmpc_linearize(tmpc_handle h, const void* xbar, const void* stage_ref, tmpc_qp* qp) {
  if (h && h->cfg.model == TMPC_MODEL_SRB_HUMANOID_RK4) {
    if (!xbar || !qp || !qp->Am || !qp->Ap || !qp->b) return TMPC_E_BADARG;
    return h->cfg.dtype == TMPC_F32 ? srb_linearize_launch<float>(h, xbar, qp) : srb_linearize_launch<double>(h, xbar, qp);
  }
  if (!h || !xbar || !stage_ref || !qp || !qp->Am || !qp->Ap || !qp->b || !qp->G || !qp->lo || !qp->hi) return TMPC_E_BADARG;
  if (h->cfg.model != TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT) return TMPC_E_UNSUPPORTED;
  if (qp->G_bstride != (int64_t)h->d.T * 3 * 6 && h->d.B > 1) return TMPC_E_BADARG;
  if (((uintptr_t)qp->Am | (uintptr_t)qp->Ap | (uintptr_t)qp->b | (uintptr_t)qp->G) & 15u) return TMPC_E_BADARG;      // vector stores (tmpc.h)
  const long long total = (long long)h->d.B * h->d.T; const int nt = 128; const unsigned nb = (unsigned)((total + nt - 1) / nt);
  const tmpc_config& c = h->cfg;
  if (c.dtype == TMPC_F32) {
    LinArgs<float> a; a.B = h->d.B; a.N = h->d.N; a.Lwb = (float)c.wheelbase; a.dt = (float)c.dt; a.xbar = (const float*)xbar; a.ref = (const float*)stage_ref;
    for (int k = 0; k < 3; ++k) { a.glo[k] = (float)c.g_lo[k]; a.ghi[k] = (float)c.g_hi[k]; }
    a.Am = (float*)qp->Am; a.Ap = (float*)qp->Ap; a.b = (float*)qp->b; a.G = (float*)qp->G; a.lo = (float*)qp->lo; a.hi = (float*)qp->hi;
    bicycle_linearize_kernel<float><<<nb, nt, 0, h->stream>>>(a);
  } else {
    LinArgs<double> a; a.B = h->d.B; a.N = h->d.N; a.Lwb = c.wheelbase; a.dt = c.dt; a.xbar = (const double*)xbar; a.ref = (const double*)stage_ref;
    for (int k = 0; k < 3; ++k) { a.glo[k] = c.g_lo[k]; a.ghi[k] = c.g_hi[k]; }
    a.Am = (double*)qp->Am; a.Ap = (double*)qp->Ap; a.b = (double*)qp->b; a.G = (double*)qp->G; a.lo = (double*)qp->lo; a.hi = (double*)qp->hi;
    bicycle_linearize_kernel<double><<<nb, nt, 0, h->stream>>>(a);
  }
  h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}

static tmpc_status check_qp(tmpc_handle h, const tmpc_qp* qp) {
  if (!h || !qp || !qp->D || !qp->E || !qp->q || !qp->Am || !qp->Ap || !qp->b || !qp->x_init) return TMPC_E_BADARG;
  if (h->d.ng > 0 && (!qp->lo || !qp->hi)) return TMPC_E_BADARG;
  if (h->d.ng > 0 && !h->cfg.g_is_selection && !qp->G) return TMPC_E_BADARG;
  const void* al[6] = {qp->D, qp->E, qp->Am, qp->Ap, qp->b, qp->G};          // 16-byte aligned (tmpc.h)
  for (int k = 0; k < 6; ++k) if ((uintptr_t)al[k] & 15u) return TMPC_E_BADARG;
  return TMPC_OK;
}

tmpc_status tmpc_factor(tmpc_handle h, const tmpc_qp* qp) {
  tmpc_status s = check_qp(h, qp); if (s != TMPC_OK) return s;
  s = h->cfg.dtype == TMPC_F32 ? do_factor<float>(h, qp) : do_factor<double>(h, qp);
  if (s == TMPC_OK) h->factored = true;
  return s;
}

tmpc_status tmpc_admm_solve(tmpc_handle h, const tmpc_qp* qp, tmpc_state* st, int32_t iters, int32_t flags, tmpc_info* info) {
  tmpc_status s = check_qp(h, qp); if (s != TMPC_OK) return s;
  if (!st || !st->x || !st->zg || !st->yf || !st->yg || !st->xi || iters < 0) return TMPC_E_BADARG;
  if (!h->factored) return TMPC_E_STATE;
  return h->cfg.dtype == TMPC_F32 ? do_solve<float>(h, qp, st, iters, flags, info) : do_solve<double>(h, qp, st, iters, flags, info);
}

tmpc_status tmpc_admm_solve_adaptive(tmpc_handle h, const tmpc_qp* qp, tmpc_state* st, const tmpc_adaptive* ad, int32_t flags, tmpc_info* info,
                                     int32_t* iters_out, int32_t* converged_out, void* rho_out) {
  tmpc_status s = check_qp(h, qp); if (s != TMPC_OK) return s;
  if (!st || !st->x || !st->zg || !st->yf || !st->yg || !st->xi || !ad) return TMPC_E_BADARG;
  if (ad->max_iters < 1 || ad->check_every < 1 || !(ad->eps_abs >= 0) || !(ad->eps_rel >= 0)) return TMPC_E_BADARG;
  if (ad->adapt_rho && (!(ad->rho_ratio >= 1) || !(ad->rho_min > 0) || !(ad->rho_max >= ad->rho_min))) return TMPC_E_BADARG;
  if (!h->factored) return TMPC_E_STATE;
  return h->cfg.dtype == TMPC_F32 ? do_solve_adaptive<float>(h, qp, st, ad, flags, info, iters_out, converged_out, rho_out)
                                  : do_solve_adaptive<double>(h, qp, st, ad, flags, info, iters_out, converged_out, rho_out);
}

tmpc_status tmpc_sqp_solve(tmpc_handle h, tmpc_qp* qp, tmpc_state* st, const void* stage_ref, const tmpc_sqp_opts* o, int32_t* iters_out,
                           int32_t* converged_out, void* alpha_log, void* kkt_out) {
  if (!h || !qp || !st || !o || !st->x || !st->zg || !st->yf || !st->yg || !st->xi) return TMPC_E_BADARG;
  const bool bicycle = h->cfg.model == TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT;      // the bicycle model reads stage_ref and writes dense G rows
  if (bicycle && (!stage_ref || !qp->G)) return TMPC_E_BADARG;
  if (!qp->D || !qp->E || !qp->q || !qp->x_init || !qp->Am || !qp->Ap || !qp->b || !qp->lo || !qp->hi) return TMPC_E_BADARG;
  if (o->max_sqp < 1 || o->admm_iters < 1 || o->n_alpha < 1 || o->n_alpha > SQP_MAX_ALPHA || !(o->eps_c > 0) || !(o->eta > 0 && o->eta < 1)) return TMPC_E_BADARG;
  if (h->cr) return TMPC_E_UNSUPPORTED;
  return h->cfg.dtype == TMPC_F32 ? do_sqp<float>(h, qp, st, stage_ref, o, iters_out, converged_out, alpha_log, kkt_out)
                                  : do_sqp<double>(h, qp, st, stage_ref, o, iters_out, converged_out, alpha_log, kkt_out);
}

tmpc_status tmpc_kkt_solve(tmpc_handle h, const void* eta, void* xt) {
  if (!h || !eta || !xt) return TMPC_E_BADARG;
  if (!h->factored) return TMPC_E_STATE;
  if (h->cr) return h->cfg.dtype == TMPC_F32 ? cr_kkt_solve<float>(h->d, h->ws + h->lay.cr, (const float*)eta, (float*)xt, h->stream, &h->launches)
                                             : cr_kkt_solve<double>(h->d, h->ws + h->lay.cr, (const double*)eta, (double*)xt, h->stream, &h->launches);
  return h->cfg.dtype == TMPC_F32 ? kkt_solve_t<float>(h, eta, xt) : kkt_solve_t<double>(h, eta, xt);
}

}  // extern "C"

// =================================================================================================== backward + host entry
namespace {

template <typename T>
tmpc_status do_backward(tmpc_ctx* h, const tmpc_qp* qp, const tmpc_state* st, const void* dLdx, const void* dLdxi, int mode, int iters, void* dq, void* dxinit) {
  const Dims& d = h->d; const Layout& L = h->lay; unsigned char* ws = h->ws;
  if (h->cr) return TMPC_E_UNSUPPORTED;
  BwdArgs<T> a; memset(&a, 0, sizeof(a));
  h->bwd_classified = true;
  a.d = d; a.qp = view<T>(qp); a.x = (const T*)st->x; a.yg = (const T*)st->yg; a.xi = (const T*)st->xi;
  a.dLdx = (const T*)dLdx; a.dLdxi = (const T*)dLdxi;
  a.eps_abs = (T)h->cfg.eps_active_abs; a.eps_rel = (T)h->cfg.eps_active_rel; a.gamma = (T)h->cfg.slack_gamma; a.sigma = (T)h->cfg.sigma;
  a.rho_adj = sizeof(T) == 8 ? (T)1e6 : (T)1e4;
  a.cls = (int8_t*)(ws + L.cls); a.rhs = (T*)(ws + L.rhs);
  a.dq = (T*)dq; a.dxinit = (T*)dxinit; a.sweeps = iters;
  int ntp = ((d.nz + 31) / 32) * 32; if (ntp > 512) ntp = 512; if (ntp < 64) ntp = 64;
  if (mode == TMPC_BWD_REFACTOR_REFINE && fast_plan<T>(d).ok) {
    // Resident class: the refinement  e <- e + K_reg^{-1}(rhs - K e)  of the active-set system is, term by term, Alg. 3 with alpha = 1 on the
    // equality-constrained adjoint QP  min 1/2 x'(P + gamma G_s'G_s)x - rhs'x  s.t. Cx = 0, G_h x = 0  with rho_f = rho_g = rho_adj:
    //   x+ = S_adj^{-1}(sigma x + rhs - C'y_f - G_h'y_g),  y+ = y + rho_adj A_a x+      (z = 0 on every constraint row)
    // so it runs on the twisted factor and the resident kernel: soft-active rows only weight the factor (gamma), inactive rows are off.
    a.w_rows = (T*)(ws + L.w_rows); a.refine_codes = 1;
    a.lo_adj = (T*)(ws + L.lo_adj); a.hi_adj = (T*)(ws + L.hi_adj); a.soft_adj = (int8_t*)(ws + L.soft_adj); a.q_adj = (T*)(ws + L.q_adj);
    bwd_prepare_kernel<T><<<d.B, ntp, 0, h->stream>>>(a); h->launches++;
    if (!cuda_ok()) return TMPC_E_CUDA;
    tmpc_status s = launch_factor_tw<T>(h, qp, (double)a.rho_adj, 0.0, nullptr, a.w_rows);
    h->factored = false; h->twisted = true;       // the forward factor has been overwritten
    if (s != TMPC_OK) return s;
    if (cudaMemsetAsync(ws + L.ax, 0, L.zero_xinit - L.ax, h->stream) != cudaSuccess) return TMPC_E_CUDA;
    AdmmArgs<T> r; memset(&r, 0, sizeof(r));
    r.d = d; r.prm = params<T>(h->cfg); r.prm.alpha = T(1); r.prm.rho_f = a.rho_adj; r.prm.rho_g = a.rho_adj; r.prm.lam = T(0); r.qp = view<T>(qp);
    r.qp.q = a.q_adj; r.qp.b = (const T*)(ws + L.zero_b); r.qp.x_init = (const T*)(ws + L.zero_xinit); r.qp.lo = a.lo_adj; r.qp.hi = a.hi_adj;
    r.Lam = (const T*)(ws + L.Lam); r.Sinv = (const T*)(ws + L.Sinv);
    r.x = (T*)(ws + L.ax); r.zg = (T*)(ws + L.azg); r.yf = (T*)(ws + L.ayf); r.yg = (T*)(ws + L.ayg); r.xi = (T*)(ws + L.axi);
    r.iters = iters; r.soft_rows = a.soft_adj;
    s = launch_resident<T>(h, r, fast_plan<T>(d));
    h->twisted = false;
    if (s != TMPC_OK) return s;
    const long long tot = (long long)d.B * d.nz;
    bwd_reuse_finish_kernel<T><<<(unsigned)((tot + 255) / 256), 256, 0, h->stream>>>(d.B, d.nz, d.nx, d.mf, r.x, r.yf, (T*)dq, (T*)dxinit); h->launches++;
    return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
  }
  if (mode == TMPC_BWD_REFACTOR_REFINE) {
    a.w_rows = (T*)(ws + L.w_rows);
    bwd_prepare_kernel<T><<<d.B, ntp, 0, h->stream>>>(a); h->launches++;
    if (!cuda_ok()) return TMPC_E_CUDA;
    tmpc_status s = launch_factor<T>(h, qp, (double)a.rho_adj, 0.0, a.w_rows, nullptr);
    h->factored = false; h->twisted = false;   // the forward factor has been overwritten (one-directional form)
    if (s != TMPC_OK) return s;
    a.Lam = (const T*)(ws + L.Lam); a.Sinv = (const T*)(ws + L.Sinv);
    const size_t smem = (3 * (size_t)d.nz + 2 * (size_t)d.mf + 2 * (size_t)d.mg) * sizeof(T);
    if (smem > kMaxSmem) return TMPC_E_UNSUPPORTED;
    int nt = ((d.nz + 31) / 32) * 32; if (nt > 1024) nt = 1024; if (nt < 64) nt = 64;
    auto launch = [&](auto k) -> tmpc_status {
      if (smem > 48 * 1024 && cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return TMPC_E_CUDA;
      k<<<d.B, nt, smem, h->stream>>>(a); h->launches++;
      return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
    };
    if (d.n == 6) return launch(bwd_refine_kernel<T, 6>);
    if (d.n == 8) return launch(bwd_refine_kernel<T, 8>);
    return launch(bwd_refine_kernel<T, 0>);
  }
  // ---- ADMM on the adjoint QP (eq. 67) with the forward factor
  if (!h->factored) return TMPC_E_STATE;
  a.lo_adj = (T*)(ws + L.lo_adj); a.hi_adj = (T*)(ws + L.hi_adj); a.soft_adj = (int8_t*)(ws + L.soft_adj); a.q_adj = (T*)(ws + L.q_adj);
  bwd_prepare_kernel<T><<<d.B, ntp, 0, h->stream>>>(a); h->launches++;
  if (!cuda_ok()) return TMPC_E_CUDA;
  if (cudaMemsetAsync(ws + L.ax, 0, L.zero_xinit - L.ax, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  AdmmArgs<T> s; memset(&s, 0, sizeof(s));
  s.d = d; s.prm = params<T>(h->cfg); s.prm.lam = T(0); s.qp = view<T>(qp);
  s.qp.q = a.q_adj; s.qp.b = (const T*)(ws + L.zero_b); s.qp.x_init = (const T*)(ws + L.zero_xinit); s.qp.lo = a.lo_adj; s.qp.hi = a.hi_adj;
  s.Lam = (const T*)(ws + L.Lam); s.Sinv = (const T*)(ws + L.Sinv);
  s.x = (T*)(ws + L.ax); s.zg = (T*)(ws + L.azg); s.yf = (T*)(ws + L.ayf); s.yg = (T*)(ws + L.ayg); s.xi = (T*)(ws + L.axi);
  s.iters = iters; s.soft_rows = a.soft_adj;
  tmpc_status rc = launch_admm<T>(h, s);
  if (rc != TMPC_OK) return rc;
  const long long tot = (long long)d.B * d.nz;
  bwd_reuse_finish_kernel<T><<<(unsigned)((tot + 255) / 256), 256, 0, h->stream>>>(d.B, d.nz, d.nx, d.mf, s.x, s.yf, (T*)dq, (T*)dxinit); h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}

struct HostPlan { size_t off[20]; size_t bytes[20]; size_t total; };
// order: D E q Am Ap b x_init G lo hi | x zg yf yg xi | r_prim r_dual objective status
HostPlan host_plan(const tmpc_config& c, int64_t sD, int64_t sE, int64_t sG, bool haveG) {
  const Dims d = make_dims(c); const size_t es = esize(c.dtype), B = d.B, nn = (size_t)d.n * d.n;
  HostPlan P; memset(&P, 0, sizeof(P));
  size_t sz[20] = { (sD ? B : 1) * d.T * nn * es, (sE ? B : 1) * d.N * nn * es, B * d.nz * es, B * d.N * d.nx * d.n * es, B * d.N * d.nx * d.n * es,
                    B * d.N * d.nx * es, B * d.nx * es, haveG ? (sG ? B : 1) * (size_t)d.T * d.ng * d.n * es : 0, B * d.mg * es, B * d.mg * es,
                    B * d.nz * es, B * d.mg * es, B * d.mf * es, B * d.mg * es, B * d.mg * es, B * es, B * es, B * es, B * 4, 0 };
  size_t o = 0;
  for (int i = 0; i < 20; ++i) { P.off[i] = o; P.bytes[i] = sz[i]; o = align_up(o + sz[i]); }
  P.total = o;
  return P;
}

}  // namespace

extern "C" {

tmpc_status tmpc_backward(tmpc_handle h, const tmpc_qp* qp, const tmpc_state* st, const void* dL_dx, const void* dL_dxi,
                          int32_t mode, int32_t iters, void* dL_dq, void* dL_dxinit) {
  tmpc_status s = check_qp(h, qp); if (s != TMPC_OK) return s;
  if (!st || !st->x || !st->yg || !st->xi || !dL_dx || !dL_dq || !dL_dxinit || iters < 0) return TMPC_E_BADARG;
  if (mode != TMPC_BWD_REFACTOR_REFINE && mode != TMPC_BWD_ADMM_REUSE_FACTOR) return TMPC_E_BADARG;
  return h->cfg.dtype == TMPC_F32 ? do_backward<float>(h, qp, st, dL_dx, dL_dxi, mode, iters, dL_dq, dL_dxinit)
                                  : do_backward<double>(h, qp, st, dL_dx, dL_dxi, mode, iters, dL_dq, dL_dxinit);
}

tmpc_status tmpc_backward_dgamma(tmpc_handle h, const tmpc_qp* qp, const tmpc_state* st, const void* dL_dq, void* dL_dgamma) {
  tmpc_status s = check_qp(h, qp); if (s != TMPC_OK) return s;
  if (!st || !st->xi || !dL_dq || !dL_dgamma) return TMPC_E_BADARG;
  if (!h->bwd_classified) return TMPC_E_STATE;
  const int8_t* cls = (const int8_t*)(h->ws + h->lay.cls);
  if (h->cfg.dtype == TMPC_F32) bwd_dgamma_kernel<float><<<h->d.B, 256, 0, h->stream>>>(h->d, view<float>(qp), cls, (const float*)st->xi, (const float*)dL_dq, (float*)dL_dgamma);
  else bwd_dgamma_kernel<double><<<h->d.B, 256, 0, h->stream>>>(h->d, view<double>(qp), cls, (const double*)st->xi, (const double*)dL_dq, (double*)dL_dgamma);
  h->launches++;
  return cuda_ok() ? TMPC_OK : TMPC_E_CUDA;
}

tmpc_status tmpc_host_staging_bytes(const tmpc_config* cfg, size_t* bytes) {
  tmpc_status s = check_cfg(cfg); if (s != TMPC_OK) return s;
  if (!bytes) return TMPC_E_BADARG;
  *bytes = host_plan(*cfg, 1, 1, 1, true).total;   // upper bound: nothing shared
  return TMPC_OK;
}

// One sub-batch [p0, p0 + nb) of the host entry on stream `st`: copy in, factor + solve on a handle view of nb problems whose workspace
// is `ws`, copy out.  The staging arrays are indexed by problem, so a sub-batch is a pointer offset into each of them.
static tmpc_status host_sub_batch(tmpc_ctx* h, const HostPlan& P, const tmpc_qp* hq, tmpc_state* hs, tmpc_info* hi_, unsigned char* dv, int iters, int flags,
                                  int p0, int nb, unsigned char* ws, cudaStream_t st, bool copy_shared) {
  const size_t B = h->d.B;
  tmpc_ctx sub = *h; sub.cfg.batch = nb; sub.d.B = nb; sub.lay = make_layout(sub.cfg); sub.ws = ws; sub.stream = st; sub.factored = false; sub.launches = 0;
  const void* src[15] = { hq->D, hq->E, hq->q, hq->Am, hq->Ap, hq->b, hq->x_init, hq->G, hq->lo, hq->hi, hs->x, hs->zg, hs->yf, hs->yg, hs->xi };
  const int64_t bstride[15] = { hq->D_bstride, hq->E_bstride, 1, 1, 1, 1, 1, hq->G_bstride, 1, 1, 1, 1, 1, 1, 1 };
  auto per = [&](int i) { return P.bytes[i] / B; };                       // bytes per problem of a per-problem array
  unsigned char* d_[19];
  for (int i = 0; i < 19; ++i) d_[i] = dv + P.off[i] + ((i < 15 && bstride[i] == 0) ? 0 : (size_t)p0 * (P.bytes[i] / B));
  for (int i = 0; i < 15; ++i) {
    if (!src[i] || !P.bytes[i]) continue;
    if ((i == 11 || i == 14) && !(flags & TMPC_SOLVE_ZG_GIVEN)) continue;      // zg, xi are outputs only
    if (bstride[i] == 0) { if (copy_shared && cudaMemcpyAsync(dv + P.off[i], src[i], P.bytes[i], cudaMemcpyHostToDevice, st) != cudaSuccess) return TMPC_E_CUDA; continue; }
    if (cudaMemcpyAsync(d_[i], (const unsigned char*)src[i] + (size_t)p0 * per(i), (size_t)nb * per(i), cudaMemcpyHostToDevice, st) != cudaSuccess) return TMPC_E_CUDA;
  }
  tmpc_qp dq = *hq;
  dq.D = d_[0]; dq.E = d_[1]; dq.q = d_[2]; dq.Am = d_[3]; dq.Ap = d_[4]; dq.b = d_[5]; dq.x_init = d_[6]; dq.G = hq->G ? d_[7] : nullptr; dq.lo = d_[8]; dq.hi = d_[9];
  tmpc_state ds = { d_[10], d_[11], d_[12], d_[13], d_[14] };
  tmpc_info di = { d_[15], d_[16], d_[17], (int32_t*)d_[18] };
  tmpc_status s = tmpc_factor(&sub, &dq); if (s != TMPC_OK) return s;
  s = tmpc_admm_solve(&sub, &dq, &ds, iters, flags, &di); if (s != TMPC_OK) return s;
  h->launches += sub.launches;
  void* dst[5] = { hs->x, hs->zg, hs->yf, hs->yg, hs->xi };
  for (int i = 0; i < 5; ++i) if (cudaMemcpyAsync((unsigned char*)dst[i] + (size_t)p0 * per(10 + i), d_[10 + i], (size_t)nb * per(10 + i), cudaMemcpyDeviceToHost, st) != cudaSuccess) return TMPC_E_CUDA;
  if (hi_) {
    void* idst[4] = { hi_->r_prim, hi_->r_dual, hi_->objective, hi_->status };
    for (int i = 0; i < 4; ++i) if (idst[i] && cudaMemcpyAsync((unsigned char*)idst[i] + (size_t)p0 * per(15 + i), d_[15 + i], (size_t)nb * per(15 + i), cudaMemcpyDeviceToHost, st) != cudaSuccess) return TMPC_E_CUDA;
  }
  return TMPC_OK;
}

tmpc_status tmpc_admm_solve_host(tmpc_handle h, const tmpc_qp* hq, tmpc_state* hs, int32_t iters, int32_t flags, tmpc_info* hi_, void* staging, size_t staging_bytes) {
  tmpc_status s = check_qp(h, hq); if (s != TMPC_OK) return s;
  if (!hs || !hs->x || !hs->zg || !hs->yf || !hs->yg || !hs->xi || !staging || iters < 0) return TMPC_E_BADARG;
  const HostPlan P = host_plan(h->cfg, hq->D_bstride, hq->E_bstride, hq->G_bstride, hq->G != nullptr);
  if (staging_bytes < P.total || ((uintptr_t)staging & 255)) return TMPC_E_WORKSPACE;
  unsigned char* dv = (unsigned char*)staging;
  h->factored = false;                                    // the workspace is re-laid out per sub-batch below
  // Two sub-batches on two internal streams, so that the host->device copy of the second overlaps the kernels of the first and
  // the device->host copy of the first overlaps the kernels of the second.  Each half gets its own half of the workspace.
  const int B = h->d.B, nb0 = (B + 1) / 2;
  tmpc_config half = h->cfg; half.batch = nb0;
  const size_t half_bytes = make_layout(half).total;
  const bool split = B >= 64 && !h->cr && 2 * half_bytes <= h->lay.total;
  if (!split) {
    s = host_sub_batch(h, P, hq, hs, hi_, dv, iters, flags, 0, B, h->ws, h->stream, true); if (s != TMPC_OK) return s;
    return cudaStreamSynchronize(h->stream) == cudaSuccess ? TMPC_OK : TMPC_E_CUDA;
  }
  for (int k = 0; k < 2; ++k) if (!h->aux[k] && cudaStreamCreateWithFlags(&h->aux[k], cudaStreamNonBlocking) != cudaSuccess) return TMPC_E_CUDA;
  for (int k = 0; k < 3; ++k) if (!h->ev[k] && cudaEventCreateWithFlags(&h->ev[k], cudaEventDisableTiming) != cudaSuccess) return TMPC_E_CUDA;
  // batch-shared arrays (D, E, G with a zero batch stride) go in once on the handle's stream; both sub-batch streams start after them
  {
    const void* ssrc[3] = { hq->D, hq->E, hq->G }; const int sidx[3] = { 0, 1, 7 }; const int64_t sstr[3] = { hq->D_bstride, hq->E_bstride, hq->G_bstride };
    for (int i = 0; i < 3; ++i) if (ssrc[i] && sstr[i] == 0 && P.bytes[sidx[i]] &&
                                    cudaMemcpyAsync(dv + P.off[sidx[i]], ssrc[i], P.bytes[sidx[i]], cudaMemcpyHostToDevice, h->stream) != cudaSuccess) return TMPC_E_CUDA;
  }
  if (cudaEventRecord(h->ev[2], h->stream) != cudaSuccess) return TMPC_E_CUDA;           // order after whatever the caller queued
  for (int k = 0; k < 2; ++k) if (cudaStreamWaitEvent(h->aux[k], h->ev[2], 0) != cudaSuccess) return TMPC_E_CUDA;
  s = host_sub_batch(h, P, hq, hs, hi_, dv, iters, flags, 0, nb0, h->ws, h->aux[0], false); if (s != TMPC_OK) return s;
  if (cudaEventRecord(h->ev[0], h->aux[0]) != cudaSuccess) return TMPC_E_CUDA;
  s = host_sub_batch(h, P, hq, hs, hi_, dv, iters, flags, nb0, B - nb0, h->ws + half_bytes, h->aux[1], false); if (s != TMPC_OK) return s;
  if (cudaEventRecord(h->ev[1], h->aux[1]) != cudaSuccess) return TMPC_E_CUDA;
  for (int k = 0; k < 2; ++k) if (cudaStreamWaitEvent(h->stream, h->ev[k], 0) != cudaSuccess) return TMPC_E_CUDA;
  return cudaStreamSynchronize(h->stream) == cudaSuccess ? TMPC_OK : TMPC_E_CUDA;
}

}  // extern "C"

// =================================================================================================== allocation-free entry
// Scratch of tmpc_admm_solve_static: one array per GPU that loads the library, held until the process exits.  In HOST code the name below is a
// host-side stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_tmpc_static_scratch[TMPC_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kMaxDevices = 64;
unsigned char* g_static_ptr[kMaxDevices] = {};           // device address of g_tmpc_static_scratch on device d (nullptr: not looked up yet)

tmpc_status static_scratch_ptr(unsigned char** out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return TMPC_E_CUDA; }
  if (dev < 0 || dev >= kMaxDevices) return TMPC_E_UNSUPPORTED;
  if (!g_static_ptr[dev]) {                              // (a race between two host threads here stores the same value twice)
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_tmpc_static_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return TMPC_E_CUDA; }
    g_static_ptr[dev] = (unsigned char*)ptr;
  }
  *out = g_static_ptr[dev];
  return TMPC_OK;
}
}  // namespace

extern "C" tmpc_status tmpc_admm_solve_static(const tmpc_config* cfg, const tmpc_qp* qp, tmpc_state* st, int32_t iters, int32_t flags, tmpc_info* info,
                                              void* cuda_stream) {
  tmpc_status s = check_cfg(cfg); if (s != TMPC_OK) return s;
  if (!st || !st->x || !st->zg || !st->yf || !st->yg || !st->xi || iters < 0) return TMPC_E_BADARG;
  if (use_cr(*cfg)) return TMPC_E_UNSUPPORTED;
  const Layout L = make_layout(*cfg);
  if (L.total > (size_t)TMPC_STATIC_SCRATCH_BYTES) return TMPC_E_STATIC_LIMIT;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return TMPC_E_CUDA; }
  unsigned char* ws = nullptr;
  s = static_scratch_ptr(&ws); if (s != TMPC_OK) return s;
  tmpc_ctx c;                                             // a handle on the host stack: nothing is allocated, nothing outlives the call
  c.cfg = *cfg; c.d = make_dims(*cfg); c.lay = L; c.ws = ws; c.stream = (cudaStream_t)cuda_stream;
  c.factored = false; c.cr = false; c.twisted = false; c.launches = 0;
  c.cur_rho = nullptr; c.cur_active = nullptr; c.cur_mask = nullptr; c.bwd_classified = false;
  c.aux[0] = c.aux[1] = nullptr; c.ev[0] = c.ev[1] = c.ev[2] = nullptr; c.pin_live = nullptr; c.ad_ev[0] = c.ad_ev[1] = nullptr; c.atil_valid = false; c.mask_sparse = false;
  s = check_qp(&c, qp); if (s != TMPC_OK) return s;
  // the array keeps the previous call's contents: the per-problem status words must start at zero (the factor kernels overwrite them, this is
  // belt and braces); the factor, the eta scratch of the streamed class and the residual partials are all written before they are read
  if (cudaMemsetAsync(ws + L.fstatus, 0, (size_t)c.d.B * sizeof(int32_t), c.stream) != cudaSuccess) { cudaGetLastError(); return TMPC_E_CUDA; }
  s = c.cfg.dtype == TMPC_F32 ? do_factor<float>(&c, qp) : do_factor<double>(&c, qp);
  if (s != TMPC_OK) return s;
  c.factored = true;
  return c.cfg.dtype == TMPC_F32 ? do_solve<float>(&c, qp, st, iters, flags, info) : do_solve<double>(&c, qp, st, iters, flags, info);
}
