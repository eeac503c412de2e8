// tmpc_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded-per-problem fp64 CPU implementation of what the TurboMPC hot path
// computes (arxiv/paper_2606_24039; citations are /root/reference/PAPER.md lines).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.  It shares
// no code, header, table or helper with paper_2606_24039_b200/csrc (the CUDA path) and neither
// includes the other.  No BLAS/LAPACK/Eigen: scalar loops only, so it can be checked against the
// paper by eye.
//
//   O-1  assemble   P, C, G from the stage blocks (eq. 1, 612-621 eq. 29-31) and
//                   S = P + sigma I + rho_f C'C + rho_g G'G from THOSE matrices, never
//                   from the Theta/Phi block formulas that the CUDA path uses.
//   O-2  factor     hand-written Cholesky S = L L' (jik scalar loops) + two triangular solves.
//                   Storage is a symmetric band of half-bandwidth bw: bw = n_z-1 is the literal dense
//                   matrix (cfg.band = 0); bw = 2n-1 (cfg.band = 1) skips structural zeros only
//                   (reading O-7) and is tested equal to the dense path.
//   O-3  ADMM       Alg. 3 with eq. 8-16, 42-45, 51, in the paper's order.
//   O-4  SQP        fixed-count full-step driver around O-1..O-3 with the bicycle model linearised
//                   by eq. 36-38.
//   f1   adaptive   Alg. 3 with the adaptive step size of eq. 17 and the termination test eq. 4 (admm_adaptive).
//   f2   SQP + linesearch   App. D l1-merit backtracking and the convergence test eq. 18 (sqp_ls_bicycle; sqp_ls_srb for the second model).
//   f3   SRB model  single-rigid-body humanoid dynamics (eq. 68-69) + RK4 and its eq. 36-37 blocks by forward-mode dual numbers.
//   O-5  backward   the definition: dense active-set KKT system eq. 62 / 65 solved by
//                   Gaussian elimination with partial pivoting; dL/dq = -eta_x, dL/dx_init = +eta_f[0:nx].
//
// Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): Theta/Phi block formulas, LQR Riccati, brute-force
// active-set enumeration, projection closed forms and invariants, residual convergence, central finite
// differences for backward (hard-active, soft-active, L1 dead-zone rows, with and without a dL/dxi term) and for the
// bicycle Jacobians, the row classification on hand-built states, the slack terms of r_dual / objective recomputed in
// numpy, every iterate against the un-reduced KKT form eq. 7 (large sigma, alpha != 1), equality rows re-posed as
// two-sided inequality rows (z_f == c), three SQP steps driven by hand, dense == band.  Nothing is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>
#include <limits>

namespace {

typedef std::vector<double> vec;

struct Cfg {              // mirrored field-by-field by oracle/__init__.py (ctypes.Structure)
  int32_t N, nx, nu, ng;
  int32_t band;           // 0: dense storage (bw = n_z-1); 1: banded (bw = 2n-1)
  int32_t g_sel;          // 1: G_t rows are unit vectors e_{g_col[r]} and G == nullptr
  int32_t zg_given;       // 0: z_g^0 = clip(G x^0, lo, hi) (reading A-12); 1: use zg as passed (resume)
  int32_t model;          // 0 none, 1 kinematic bicycle + implicit midpoint (reading A-24)
  double sigma, rho_bar, rho_eq_scale, alpha;
  double gamma, lam;      // gamma_xi and the L1 slack weight lambda (reading A-14)
  double eps_abs, eps_rel;  // active-set classification (reading A-16)
  double wheelbase, dt;   // bicycle
  double g_lo[64], g_hi[64];  // un-shifted bounds of g_t (model != 0)
  int32_t g_col[64];
  uint8_t soft[64];       // per-row delta_xi (reading A-13)
  double model_params[16]; // model 2 (SRB humanoid): mass, g[3], diag(I)[3], foot_L[3], foot_R[3] (world positions)
};

// ---- symmetric band matrix, lower storage: element (i,j), i-bw <= j <= i, at a[i*(bw+1) + (j-i+bw)]
struct Band {
  int n, bw; vec a;
  Band(int n_, int bw_) : n(n_), bw(std::min(bw_, n_ - 1 < 0 ? 0 : n_ - 1)), a((size_t)n_ * (std::min(bw_, n_ - 1 < 0 ? 0 : n_ - 1) + 1), 0.0) {}
  inline double& lo(int i, int j) { return a[(size_t)i * (bw + 1) + (j - i + bw)]; }     // needs j <= i
  inline double get(int i, int j) const { if (j > i) std::swap(i, j); if (i - j > bw) return 0.0; return a[(size_t)i * (bw + 1) + (j - i + bw)]; }
  inline void add_sym(int i, int j, double v) { if (j > i) return; lo(i, j) += v; }      // caller passes both (i,j),(j,i); keep lower
};

// ---- a matrix whose every row is dense on a window of columns [c0, c0+len)  (C and G, eq. 30-31)
struct Rows {
  int m = 0, stride = 0; std::vector<int> c0, len; vec v;
  void init(int m_, int stride_) { m = m_; stride = stride_; c0.assign(m, 0); len.assign(m, 0); v.assign((size_t)m * stride, 0.0); }
  double* row(int r) { return &v[(size_t)r * stride]; }
  const double* row(int r) const { return &v[(size_t)r * stride]; }
  void mul(const vec& x, vec& z) const {           // z = M x
    for (int r = 0; r < m; ++r) { double s = 0; const double* a = row(r); for (int k = 0; k < len[r]; ++k) s += a[k] * x[c0[r] + k]; z[r] = s; }
  }
  void mulT_add(const vec& y, vec& out) const {    // out += M' y
    for (int r = 0; r < m; ++r) { const double* a = row(r); for (int k = 0; k < len[r]; ++k) out[c0[r] + k] += a[k] * y[r]; }
  }
  void add_AtA(Band& S, double w) const {          // S += w M'M   (row by row: w * row' row)
    for (int r = 0; r < m; ++r) { const double* a = row(r);
      for (int i = 0; i < len[r]; ++i) { if (a[i] == 0.0) continue; for (int j = 0; j <= i; ++j) S.lo(c0[r] + i, c0[r] + j) += w * a[i] * a[j]; } }
  }
  void add_AtWA(Band& S, const vec& w) const {     // S += M' diag(w) M
    for (int r = 0; r < m; ++r) { if (w[r] == 0.0) continue; const double* a = row(r);
      for (int i = 0; i < len[r]; ++i) { if (a[i] == 0.0) continue; for (int j = 0; j <= i; ++j) S.lo(c0[r] + i, c0[r] + j) += w[r] * a[i] * a[j]; } }
  }
};

struct QP {               // one problem, assembled per O-1
  int N, T, nx, nu, n, ng, nz, mf, mg;
  Band P; Rows C, G; vec q, c, lo, hi;
  QP(int N_, int nx_, int nu_, int ng_, int bw) : N(N_), T(N_ + 1), nx(nx_), nu(nu_), n(nx_ + nu_), ng(ng_), nz((N_ + 1) * (nx_ + nu_)),
      mf(nx_ + N_ * nx_), mg((N_ + 1) * ng_), P((N_ + 1) * (nx_ + nu_), bw) {}
};

int half_bandwidth(const Cfg& c) { int n = c.nx + c.nu; int nz = (c.N + 1) * n; return c.band ? std::min(2 * n - 1, nz - 1) : nz - 1; }

// O-1.  D [T][n][n], E [N][n][n] (block (t+1,t) of P), q [T][n], Am/Ap [N][nx][n], b [N][nx], x_init [nx],
//       G [T][ng][n] or nullptr with cfg.g_sel, lo/hi [T][ng].
QP assemble(const Cfg& cf, const double* D, const double* E, const double* q, const double* Am, const double* Ap, const double* b,
            const double* x_init, const double* G, const double* lo, const double* hi) {
  QP p(cf.N, cf.nx, cf.nu, cf.ng, half_bandwidth(cf));
  const int n = p.n, nx = p.nx, N = p.N, T = p.T, ng = p.ng;
  for (int t = 0; t < T; ++t)                                    // P: D_t on the diagonal (eq. 29)
    for (int i = 0; i < n; ++i) for (int j = 0; j <= i; ++j) p.P.lo(t * n + i, t * n + j) += D[((size_t)t * n + i) * n + j];   // D_t symmetric by contract: lower part taken
  for (int t = 0; t < N; ++t)                                    // E_t at block (t+1, t)
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) p.P.lo((t + 1) * n + i, t * n + j) += E[((size_t)t * n + i) * n + j];
  p.q.assign(q, q + p.nz);
  p.C.init(p.mf, 2 * n); p.c.assign(p.mf, 0.0);                  // C: eq. 30; rows 0..nx-1: A_init = [I 0], rhs x_init
  for (int i = 0; i < nx; ++i) { p.C.c0[i] = 0; p.C.len[i] = n; p.C.row(i)[i] = 1.0; p.c[i] = x_init[i]; }
  for (int t = 0; t < N; ++t) for (int i = 0; i < nx; ++i) {     // dynamics row: [A_t^- | A_t^+] on stages t, t+1 (eq. 36)
    int r = nx + t * nx + i; p.C.c0[r] = t * n; p.C.len[r] = 2 * n;
    for (int j = 0; j < n; ++j) { p.C.row(r)[j] = Am[((size_t)t * nx + i) * n + j]; p.C.row(r)[n + j] = Ap[((size_t)t * nx + i) * n + j]; }
    p.c[r] = b[(size_t)t * nx + i];
  }
  p.G.init(p.mg, n); p.lo.assign(p.mg, 0.0); p.hi.assign(p.mg, 0.0);   // G: eq. 31, block diagonal
  for (int t = 0; t < T; ++t) for (int r = 0; r < ng; ++r) {
    int row = t * ng + r; p.G.c0[row] = t * n; p.G.len[row] = n;
    if (cf.g_sel) p.G.row(row)[cf.g_col[r]] = 1.0; else for (int j = 0; j < n; ++j) p.G.row(row)[j] = G[((size_t)t * ng + r) * n + j];
    p.lo[row] = lo[(size_t)t * ng + r]; p.hi[row] = hi[(size_t)t * ng + r];
  }
  return p;
}

// S = P + sigma I + C' diag(wf) C + G' diag(wg) G   (PAPER.md:172, 788 with rho = diag(rho_f I, rho_g I))
Band build_S(const QP& p, double sigma, const vec& wf, const vec& wg) {
  Band S = p.P;
  for (int i = 0; i < p.nz; ++i) S.lo(i, i) += sigma;
  p.C.add_AtWA(S, wf); p.G.add_AtWA(S, wg);
  return S;
}

// O-2.  In-place Cholesky of the band (lower factor overwrites S).  Returns the smallest pivot seen (<=0: failure).
double cholesky(Band& S) {
  const int n = S.n, bw = S.bw; double minpiv = std::numeric_limits<double>::infinity();
  for (int j = 0; j < n; ++j) {
    for (int i = j; i <= std::min(n - 1, j + bw); ++i) {
      double s = S.lo(i, j);
      for (int k = std::max(0, i - bw); k < j; ++k) s -= S.lo(i, k) * S.lo(j, k);
      if (i == j) { minpiv = std::min(minpiv, s); S.lo(j, j) = std::sqrt(s); }
      else S.lo(i, j) = s / S.lo(j, j);
    }
  }
  return minpiv;
}
void chol_solve(Band& L, vec& x) {            // x <- (L L')^{-1} x
  const int n = L.n, bw = L.bw;
  for (int i = 0; i < n; ++i) { double s = x[i]; for (int k = std::max(0, i - bw); k < i; ++k) s -= L.lo(i, k) * x[k]; x[i] = s / L.lo(i, i); }
  for (int i = n - 1; i >= 0; --i) { double s = x[i]; for (int k = i + 1; k <= std::min(n - 1, i + bw); ++k) s -= L.lo(k, i) * x[k]; x[i] = s / L.lo(i, i); }
}

void band_mul(const Band& A, const vec& x, vec& y) {   // y = A x (symmetric)
  for (int i = 0; i < A.n; ++i) { double s = 0; for (int j = std::max(0, i - A.bw); j <= std::min(A.n - 1, i + A.bw); ++j) s += A.get(i, j) * x[j]; y[i] = s; }
}

inline double clip(double v, double lo, double hi) { return std::min(std::max(v, lo), hi); }

// O-3 step 5.  Hard row: eq. 13.  Soft row: eq. 15a/15b generalised with the L1 weight lambda (reading A-14);
// lambda = 0 is exactly eq. 15 == the 3-case formula at PAPER.md:836.
inline void project_row(bool soft, double v, double lo, double hi, double rho, double gamma, double lam, double& z, double& xi) {
  if (!soft) { z = clip(v, lo, hi); xi = 0.0; return; }
  double sp = std::max(0.0, (rho * (v - hi) - lam) / (rho + gamma));
  double sm = std::max(0.0, (rho * (lo - v) - lam) / (rho + gamma));
  z = clip(v, lo, hi) + sp - sm; xi = sm - sp;
}

struct Info { double r_prim, r_dual, objective, min_pivot; };

// O-3.  K iterations of Alg. 3.  x [nz], zg [mg], yf [mf], yg [mg], xi [mg] in/out.
// soft_rows (optional, [mg]): per-ROW soft flag replacing the per-row-type mask cf.soft — used for the adjoint QP eq. 67, whose
// soft rows are the soft-ACTIVE rows of one particular solution; the arithmetic is the same.
Info admm(const Cfg& cf, const QP& p, double* x_, double* zg_, double* yf_, double* yg_, double* xi_, int K, const uint8_t* soft_rows = nullptr) {
  auto is_soft = [&](int i) { return soft_rows ? soft_rows[i] != 0 : cf.soft[i % p.ng] != 0; };
  const double rho_g = cf.rho_bar, rho_f = cf.rho_eq_scale * cf.rho_bar, sigma = cf.sigma, alpha = cf.alpha;
  vec x(x_, x_ + p.nz), zg(p.mg), yf(yf_, yf_ + p.mf), yg(yg_, yg_ + p.mg), xi(p.mg, 0.0);
  vec tmp(p.mg);
  if (cf.zg_given) { zg.assign(zg_, zg_ + p.mg); xi.assign(xi_, xi_ + p.mg); }
  else { p.G.mul(x, tmp); for (int i = 0; i < p.mg; ++i) zg[i] = clip(tmp[i], p.lo[i], p.hi[i]); }
  Band L = build_S(p, sigma, vec(p.mf, rho_f), vec(p.mg, rho_g));
  Info info; info.min_pivot = cholesky(L);
  vec eta(p.nz), xt(p.nz), ztf(p.mf), ztg(p.mg), rf(p.mf), rg(p.mg);
  for (int k = 0; k < K; ++k) {
    // 1. eta = sigma x - q + C'(rho_f c - y_f) + G'(rho_g z_g - y_g)              (eq. 51, z_f == c)
    for (int i = 0; i < p.nz; ++i) eta[i] = sigma * x[i] - p.q[i];
    for (int i = 0; i < p.mf; ++i) rf[i] = rho_f * p.c[i] - yf[i];
    for (int i = 0; i < p.mg; ++i) rg[i] = rho_g * zg[i] - yg[i];
    p.C.mulT_add(rf, eta); p.G.mulT_add(rg, eta);
    // 2. x~ = S^{-1} eta (eq. 8);  z~ = A x~ (eq. 9)
    xt = eta; chol_solve(L, xt); p.C.mul(xt, ztf); p.G.mul(xt, ztg);
    // 3. x^{k+1} = alpha x~ + (1-alpha) x^k                                         (eq. 10-11)
    for (int i = 0; i < p.nz; ++i) x[i] = alpha * xt[i] + (1.0 - alpha) * x[i];
    // 4.-6. z^_g, v, projection (eq. 12-15), dual updates (eq. 44-45)
    for (int i = 0; i < p.mg; ++i) {
      double zh = alpha * ztg[i] + (1.0 - alpha) * zg[i];
      double v = zh + yg[i] / rho_g, z, s;
      project_row(is_soft(i), v, p.lo[i], p.hi[i], rho_g, cf.gamma, cf.lam, z, s);
      zg[i] = z; xi[i] = s; yg[i] = yg[i] + rho_g * (zh - z);
    }
    for (int i = 0; i < p.mf; ++i) yf[i] = yf[i] + rho_f * alpha * (ztf[i] - p.c[i]);
  }
  // residuals (eq. 3) and objective at the K-th iterate
  p.C.mul(x, ztf); p.G.mul(x, ztg);
  double rp = 0; for (int i = 0; i < p.mf; ++i) rp = std::max(rp, std::fabs(ztf[i] - p.c[i]));
  for (int i = 0; i < p.mg; ++i) rp = std::max(rp, std::fabs(ztg[i] - zg[i]));
  vec g(p.nz), Px(p.nz); band_mul(p.P, x, Px);
  for (int i = 0; i < p.nz; ++i) g[i] = Px[i] + p.q[i];
  p.C.mulT_add(yf, g); p.G.mulT_add(yg, g);
  double rd = 0; for (int i = 0; i < p.nz; ++i) rd = std::max(rd, std::fabs(g[i]));
  double obj = 0; for (int i = 0; i < p.nz; ++i) obj += 0.5 * x[i] * Px[i] + p.q[i] * x[i];
  for (int i = 0; i < p.mg; ++i) if (is_soft(i) && xi[i] != 0.0) {
    double sg = xi[i] > 0 ? 1.0 : -1.0;
    rd = std::max(rd, std::fabs(cf.gamma * xi[i] + cf.lam * sg + yg[i]));
    obj += cf.lam * std::fabs(xi[i]) + 0.5 * cf.gamma * xi[i] * xi[i];
  }
  info.r_prim = rp; info.r_dual = rd; info.objective = obj;
  std::copy(x.begin(), x.end(), x_); std::copy(zg.begin(), zg.end(), zg_); std::copy(yf.begin(), yf.end(), yf_);
  std::copy(yg.begin(), yg.end(), yg_); std::copy(xi.begin(), xi.end(), xi_);
  return info;
}

// f1: Alg. 3 with the paper's adaptive step size and termination test.
//   * every `check_every` (k_rho^iter: 25) iterations, and at iteration K_max, the residuals (eq. 3) and the
//     scales of eq. 4 are evaluated:  np = |(Ax, z)|_inf with A = [C; G], z = (c, z_g);
//     nd = |(Px, A'y, q, gamma xi, y_g on soft rows)|_inf   (reading A-32: the test is run at the
//     rho schedule's cadence, not after every iteration);
//   * converged  <=>  r_prim <= eps_abs + eps_rel np  and  r_dual <= eps_abs + eps_rel nd   (eq. 4)  ->  stop;
//   * otherwise (eq. 17):  rho_new = clip(rho_bar sqrt((r_prim/np) / (r_dual/nd)), [rho_min, rho_max]),
//     accepted iff max(rho_new/rho_bar, rho_bar/rho_new) > ratio; on acceptance S is re-assembled with the new rho and
//     re-factorised; x, z, y are kept.  A zero denominator (r_dual, np or nd = 0) skips the update.
// log_out (optional, 8 doubles per check): k, r_prim, r_dual, np, nd, rho before, rho after, converged.
struct Adaptive { int32_t max_iters, check_every, adapt_rho, pad; double eps_abs, eps_rel, ratio, rho_min, rho_max; };

int admm_adaptive(const Cfg& cf, const QP& p, const Adaptive& ad, double* x_, double* zg_, double* yf_, double* yg_, double* xi_, double* info_out,
                  double* log_out, int max_log) {
  const double sigma = cf.sigma, alpha = cf.alpha;
  double rho_bar = cf.rho_bar;
  vec x(x_, x_ + p.nz), zg(p.mg), yf(yf_, yf_ + p.mf), yg(yg_, yg_ + p.mg), xi(p.mg, 0.0), tmp(p.mg);
  if (cf.zg_given) { zg.assign(zg_, zg_ + p.mg); xi.assign(xi_, xi_ + p.mg); }
  else { p.G.mul(x, tmp); for (int i = 0; i < p.mg; ++i) zg[i] = clip(tmp[i], p.lo[i], p.hi[i]); }
  double rho_g = rho_bar, rho_f = cf.rho_eq_scale * rho_bar;
  Band L = build_S(p, sigma, vec(p.mf, rho_f), vec(p.mg, rho_g));
  double minpiv = cholesky(L);
  vec eta(p.nz), xt(p.nz), ztf(p.mf), ztg(p.mg), rf(p.mf), rg(p.mg), g(p.nz), Px(p.nz), Aty(p.nz);
  int k = 0, nlog = 0, converged = 0;
  double rp = 0, rd = 0, obj = 0;
  while (k < ad.max_iters && !converged) {
    for (int i = 0; i < p.nz; ++i) eta[i] = sigma * x[i] - p.q[i];
    for (int i = 0; i < p.mf; ++i) rf[i] = rho_f * p.c[i] - yf[i];
    for (int i = 0; i < p.mg; ++i) rg[i] = rho_g * zg[i] - yg[i];
    p.C.mulT_add(rf, eta); p.G.mulT_add(rg, eta);
    xt = eta; chol_solve(L, xt); p.C.mul(xt, ztf); p.G.mul(xt, ztg);
    for (int i = 0; i < p.nz; ++i) x[i] = alpha * xt[i] + (1.0 - alpha) * x[i];
    for (int i = 0; i < p.mg; ++i) {
      double zh = alpha * ztg[i] + (1.0 - alpha) * zg[i];
      double v = zh + yg[i] / rho_g, z, s;
      project_row(cf.soft[i % p.ng] != 0, v, p.lo[i], p.hi[i], rho_g, cf.gamma, cf.lam, z, s);
      zg[i] = z; xi[i] = s; yg[i] = yg[i] + rho_g * (zh - z);
    }
    for (int i = 0; i < p.mf; ++i) yf[i] = yf[i] + rho_f * alpha * (ztf[i] - p.c[i]);
    ++k;
    if (k % ad.check_every != 0 && k != ad.max_iters) continue;
    // residuals (eq. 3) and the scales of eq. 4
    p.C.mul(x, ztf); p.G.mul(x, ztg);
    rp = 0; double np_ = 0;
    for (int i = 0; i < p.mf; ++i) { rp = std::max(rp, std::fabs(ztf[i] - p.c[i])); np_ = std::max(np_, std::max(std::fabs(ztf[i]), std::fabs(p.c[i]))); }
    for (int i = 0; i < p.mg; ++i) { rp = std::max(rp, std::fabs(ztg[i] - zg[i])); np_ = std::max(np_, std::max(std::fabs(ztg[i]), std::fabs(zg[i]))); }
    band_mul(p.P, x, Px);
    std::fill(Aty.begin(), Aty.end(), 0.0); p.C.mulT_add(yf, Aty); p.G.mulT_add(yg, Aty);
    rd = 0; double nd_ = 0; obj = 0;
    for (int i = 0; i < p.nz; ++i) {
      rd = std::max(rd, std::fabs(Px[i] + p.q[i] + Aty[i]));
      nd_ = std::max(nd_, std::max(std::fabs(Px[i]), std::max(std::fabs(Aty[i]), std::fabs(p.q[i]))));
      obj += 0.5 * x[i] * Px[i] + p.q[i] * x[i];
    }
    for (int i = 0; i < p.mg; ++i) if (cf.soft[i % p.ng]) {
      nd_ = std::max(nd_, std::max(std::fabs(cf.gamma * xi[i]), std::fabs(yg[i])));
      if (xi[i] != 0.0) {
        double sg = xi[i] > 0 ? 1.0 : -1.0;
        rd = std::max(rd, std::fabs(cf.gamma * xi[i] + cf.lam * sg + yg[i]));
        obj += cf.lam * std::fabs(xi[i]) + 0.5 * cf.gamma * xi[i] * xi[i];
      }
    }
    converged = (rp <= ad.eps_abs + ad.eps_rel * np_) && (rd <= ad.eps_abs + ad.eps_rel * nd_);
    const double rho_before = rho_bar;
    if (!converged && ad.adapt_rho && k % ad.check_every == 0 && k < ad.max_iters && rd > 0.0 && np_ > 0.0 && nd_ > 0.0) {
      double cand = rho_bar * std::sqrt((rp / np_) / (rd / nd_));
      cand = std::min(std::max(cand, ad.rho_min), ad.rho_max);
      if (std::max(cand / rho_bar, rho_bar / cand) > ad.ratio) {
        rho_bar = cand; rho_g = rho_bar; rho_f = cf.rho_eq_scale * rho_bar;
        L = build_S(p, sigma, vec(p.mf, rho_f), vec(p.mg, rho_g));
        minpiv = std::min(minpiv, cholesky(L));
      }
    }
    if (log_out && nlog < max_log) { double* l = log_out + 8 * nlog++; l[0] = k; l[1] = rp; l[2] = rd; l[3] = np_; l[4] = nd_; l[5] = rho_before; l[6] = rho_bar; l[7] = converged; }
  }
  info_out[0] = rp; info_out[1] = rd; info_out[2] = obj; info_out[3] = minpiv; info_out[4] = k; info_out[5] = rho_bar; info_out[6] = converged; info_out[7] = nlog;
  std::copy(x.begin(), x.end(), x_); std::copy(zg.begin(), zg.end(), zg_); std::copy(yf.begin(), yf.end(), yf_);
  std::copy(yg.begin(), yg.end(), yg_); std::copy(xi.begin(), xi.end(), xi_);
  return minpiv > 0 ? 0 : 1;
}

// dense Gaussian elimination with partial pivoting, A [m][m] row-major, rhs in/out.  Returns min |pivot|.
double gauss_solve(vec& A, vec& rhs, int m) {
  double minpiv = std::numeric_limits<double>::infinity();
  for (int k = 0; k < m; ++k) {
    int piv = k; double best = std::fabs(A[(size_t)k * m + k]);
    for (int i = k + 1; i < m; ++i) { double a = std::fabs(A[(size_t)i * m + k]); if (a > best) { best = a; piv = i; } }
    minpiv = std::min(minpiv, best);
    if (best == 0.0) return 0.0;
    if (piv != k) { for (int j = 0; j < m; ++j) std::swap(A[(size_t)k * m + j], A[(size_t)piv * m + j]); std::swap(rhs[k], rhs[piv]); }
    double d = A[(size_t)k * m + k];
    for (int i = k + 1; i < m; ++i) { double f = A[(size_t)i * m + k] / d; if (f == 0.0) continue;
      for (int j = k; j < m; ++j) A[(size_t)i * m + j] -= f * A[(size_t)k * m + j]; rhs[i] -= f * rhs[k]; }
  }
  for (int i = m - 1; i >= 0; --i) { double s = rhs[i]; for (int j = i + 1; j < m; ++j) s -= A[(size_t)i * m + j] * rhs[j]; rhs[i] = s / A[(size_t)i * m + i]; }
  return minpiv;
}

// Row classification (readings A-16): 0 inactive, 1 hard-active, 2 soft-active.
void classify(const Cfg& cf, const QP& p, const double* x, const double* yg, const double* xi, std::vector<int>& cls) {
  vec xv(x, x + p.nz), gx(p.mg); p.G.mul(xv, gx);
  double ymax = 0; for (int i = 0; i < p.mg; ++i) ymax = std::max(ymax, std::fabs(yg[i]));
  const double eps_y = cf.eps_abs + cf.eps_rel * ymax;
  cls.assign(p.mg, 0);
  for (int i = 0; i < p.mg; ++i) {
    bool soft = cf.soft[i % p.ng] != 0;
    if (soft && std::fabs(xi[i]) > cf.eps_abs) { cls[i] = 2; continue; }
    if (std::fabs(yg[i]) > eps_y) { cls[i] = 1; continue; }
    double dl = gx[i] - p.lo[i], du = p.hi[i] - gx[i];
    bool near_lo = std::isfinite(p.lo[i]) && dl <= cf.eps_abs + cf.eps_rel * std::fabs(p.lo[i]);
    bool near_hi = std::isfinite(p.hi[i]) && du <= cf.eps_abs + cf.eps_rel * std::fabs(p.hi[i]);
    if (near_lo || near_hi) cls[i] = 1;
  }
}

// O-5.  Backward by the definition (eq. 62 / 65).  Returns min |pivot| of the elimination.
// dgamma (optional): dL/dgamma_xi of eq. 66 in the signed slack: the only explicit dependence of the KKT conditions on gamma
// is the stationarity row gamma xi + lam sgn(xi) + y_g = 0 of the soft-active rows, so dL/dgamma = -xi_s' eta_xi with eta_xi = -G_s eta_x (eq. 64),
// i.e. dL/dgamma = sum_{soft-active i} xi_i (G eta_x)_i.
double backward(const Cfg& cf, const QP& p, const double* x, const double* yg, const double* xi, const double* dLdx, const double* dLdxi,
                double* dq, double* dxinit, int* n_hard, int* n_soft, double* dgamma = nullptr) {
  std::vector<int> cls; classify(cf, p, x, yg, xi, cls);
  std::vector<int> hard; int ns = 0;
  for (int i = 0; i < p.mg; ++i) { if (cls[i] == 1) hard.push_back(i); if (cls[i] == 2) ++ns; }
  const int nh = (int)hard.size(), m = p.nz + p.mf + nh;
  vec K((size_t)m * m, 0.0), rhs(m, 0.0);
  for (int i = 0; i < p.nz; ++i) for (int j = std::max(0, i - p.P.bw); j <= std::min(p.nz - 1, i + p.P.bw); ++j) K[(size_t)i * m + j] = p.P.get(i, j);
  for (int i = 0; i < p.nz; ++i) rhs[i] = dLdx[i];
  // + gamma G_s' G_s ;  rhs -= G_s' dL/dxi_s  (eq. 65).  dLdxi is the gradient w.r.t. the SIGNED slack xi of the OCP / of Alg. 3
  // (lo <= Gx + xi <= hi), i.e. the `xi` this solver returns.  App. E writes the active rows as
  // g_A + S xi_A = 0 with S = sign(xi) (eq. 54), which is the same row Gx + xi = bound in the variable xi_A = S xi = |xi|;
  // eq. 65's right-hand side -G_s' S dL/dxi_A then equals -G_s' S (S dL/dxi) = -G_s' dL/dxi  (reading A-31,
  // pinned by central finite differences in tests/test_oracle_pins.py).
  for (int r = 0; r < p.mg; ++r) if (cls[r] == 2) {
    const double* a = p.G.row(r); int c0 = p.G.c0[r];
    for (int i = 0; i < p.G.len[r]; ++i) for (int j = 0; j < p.G.len[r]; ++j) K[(size_t)(c0 + i) * m + c0 + j] += cf.gamma * a[i] * a[j];
    if (dLdxi) for (int i = 0; i < p.G.len[r]; ++i) rhs[c0 + i] -= a[i] * dLdxi[r];
  }
  for (int r = 0; r < p.mf; ++r) { const double* a = p.C.row(r); for (int k = 0; k < p.C.len[r]; ++k) { K[(size_t)(p.nz + r) * m + p.C.c0[r] + k] = a[k]; K[(size_t)(p.C.c0[r] + k) * m + p.nz + r] = a[k]; } }
  for (int h = 0; h < nh; ++h) { int r = hard[h]; const double* a = p.G.row(r); for (int k = 0; k < p.G.len[r]; ++k) { K[(size_t)(p.nz + p.mf + h) * m + p.G.c0[r] + k] = a[k]; K[(size_t)(p.G.c0[r] + k) * m + p.nz + p.mf + h] = a[k]; } }
  double piv = gauss_solve(K, rhs, m);
  for (int i = 0; i < p.nz; ++i) dq[i] = -rhs[i];                 // dL/dq = -eta_x         (eq. 59, dF/dq = [I;0;0])
  for (int i = 0; i < p.nx; ++i) dxinit[i] = rhs[p.nz + i];       // dL/dx_init = +eta_f[0:nx] (dF/dx_init = -I on init rows)
  if (dgamma) {
    double s = 0;
    for (int r = 0; r < p.mg; ++r) if (cls[r] == 2) { const double* a = p.G.row(r); double ge = 0; for (int k = 0; k < p.G.len[r]; ++k) ge += a[k] * rhs[p.G.c0[r] + k];
      // the adjoint of the eliminated slack also carries the upstream dL/dxi: gamma eta_xi + eta_yg = dL/dxi, G eta_x + eta_xi = 0 (eq. 60 rows 2, 4)
      s += xi[r] * ge; }
    *dgamma = s;
  }
  *n_hard = nh; *n_soft = ns;
  return piv;
}

// ---- kinematic bicycle, implicit midpoint (reading A-24).  v = (px, py, psi, vel, a, delta).
// residual f_k = x_k + dt F((x_k + x_{k+1})/2, u_k) - x_{k+1},  F = (v cos psi, v sin psi, v/L tan delta, a)
void bicycle_residual(double Lwb, double dt, const double* vk, const double* vk1, double* f) {
  double psi = 0.5 * (vk[2] + vk1[2]), vel = 0.5 * (vk[3] + vk1[3]), a = vk[4], del = vk[5];
  double F[4] = { vel * std::cos(psi), vel * std::sin(psi), vel / Lwb * std::tan(del), a };
  for (int i = 0; i < 4; ++i) f[i] = vk[i] + dt * F[i] - vk1[i];
}
// eq. 36-38 for the bicycle: Am = df/dv_k, Ap = df/dv_{k+1}, b = Am v_k + Ap v_{k+1} - f (eq. 37);
// g_t(v) = (a, delta, lateral error e = -sin(psi_ref)(px - px_ref) + cos(psi_ref)(py - py_ref)) is linear in v,
// so G_t is its constant Jacobian and the shifted bounds (eq. 38) are g_lo - g(v) + G v = g_lo + G_lat . p_ref on row 2.
void bicycle_linearize(const Cfg& cf, const double* xbar, const double* ref, double* Am, double* Ap, double* b, double* G, double* lo, double* hi) {
  const int N = cf.N, n = 6, nx = 4; const double dt = cf.dt, L = cf.wheelbase;
  for (int t = 0; t < N; ++t) {
    const double* vk = xbar + (size_t)t * n; const double* vk1 = vk + n;
    double psi = 0.5 * (vk[2] + vk1[2]), vel = 0.5 * (vk[3] + vk1[3]), del = vk[5];
    double Fx[4][4] = {{0, 0, -vel * std::sin(psi), std::cos(psi)}, {0, 0, vel * std::cos(psi), std::sin(psi)}, {0, 0, 0, std::tan(del) / L}, {0, 0, 0, 0}};
    double Fu[4][2] = {{0, 0}, {0, 0}, {0, vel / (L * std::cos(del) * std::cos(del))}, {1, 0}};
    double* am = Am + (size_t)t * nx * n; double* ap = Ap + (size_t)t * nx * n;
    for (int i = 0; i < nx; ++i) {
      for (int j = 0; j < nx; ++j) { am[i * n + j] = (i == j ? 1.0 : 0.0) + 0.5 * dt * Fx[i][j]; ap[i * n + j] = (i == j ? -1.0 : 0.0) + 0.5 * dt * Fx[i][j]; }
      for (int j = 0; j < 2; ++j) { am[i * n + nx + j] = dt * Fu[i][j]; ap[i * n + nx + j] = 0.0; }
    }
    double f[4]; bicycle_residual(L, dt, vk, vk1, f);
    for (int i = 0; i < nx; ++i) { double s = -f[i]; for (int j = 0; j < n; ++j) s += am[i * n + j] * vk[j] + ap[i * n + j] * vk1[j]; b[(size_t)t * nx + i] = s; }
  }
  for (int t = 0; t <= N; ++t) {
    const double* r = ref + (size_t)t * n; double* g = G + (size_t)t * 3 * n;
    for (int k = 0; k < 3 * n; ++k) g[k] = 0.0;
    g[0 * n + 4] = 1.0; g[1 * n + 5] = 1.0; g[2 * n + 0] = -std::sin(r[2]); g[2 * n + 1] = std::cos(r[2]);
    double off = g[2 * n + 0] * r[0] + g[2 * n + 1] * r[1];
    for (int k = 0; k < 3; ++k) { double o = (k == 2) ? off : 0.0; lo[(size_t)t * 3 + k] = cf.g_lo[k] + o; hi[(size_t)t * 3 + k] = cf.g_hi[k] + o; }
  }
}

// ---- f3: single-rigid-body humanoid model (eq. 68-69), RK4 with step cf.dt: x = (p, Theta = (roll, pitch, yaw), v, omega),
// u = (f_L, f_R) world-frame foot forces.  Readings (A-38): I = diag(model_params[4..6]) in the body frame; the contact vectors are
// r_i = foot_i - p with fixed world foot positions (model_params[7..12]); the torque r x f enters eq. 68d as printed (no frame change).
// Written once as a template over the scalar type so that the SAME lines give values (double) and exact directional derivatives (Dual).
struct Dual { double v, d; };
inline Dual operator+(Dual a, Dual b) { return {a.v + b.v, a.d + b.d}; }
inline Dual operator-(Dual a, Dual b) { return {a.v - b.v, a.d - b.d}; }
inline Dual operator*(Dual a, Dual b) { return {a.v * b.v, a.d * b.v + a.v * b.d}; }
inline Dual operator/(Dual a, Dual b) { return {a.v / b.v, (a.d * b.v - a.v * b.d) / (b.v * b.v)}; }
inline Dual operator*(double a, Dual b) { return {a * b.v, a * b.d}; }
inline Dual operator+(Dual a, double b) { return {a.v + b, a.d}; }
inline Dual operator-(double a, Dual b) { return {a - b.v, -b.d}; }
inline Dual dsin(Dual a) { return {std::sin(a.v), std::cos(a.v) * a.d}; }
inline Dual dcos(Dual a) { return {std::cos(a.v), -std::sin(a.v) * a.d}; }
inline double dsin(double a) { return std::sin(a); }
inline double dcos(double a) { return std::cos(a); }

template <typename S>
void srb_xdot(const double* mp, const S* x, const S* u, S* xd) {       // eq. 68a-d with T(Theta) of eq. 69
  const double mass = mp[0];
  const S phi = x[3], th = x[4];
  const S sp = dsin(phi), cp = dcos(phi), st = dsin(th), ct = dcos(th), tt = st / ct;
  for (int i = 0; i < 3; ++i) xd[i] = x[6 + i];                          // p' = v
  const S w0 = x[9], w1 = x[10], w2 = x[11];
  xd[3] = w0 + sp * tt * w1 + cp * tt * w2;                              // Theta' = T(Theta) omega
  xd[4] = cp * w1 - sp * w2;
  xd[5] = sp / ct * w1 + cp / ct * w2;
  for (int i = 0; i < 3; ++i) xd[6 + i] = (1.0 / mass) * (u[i] + u[3 + i]) + mp[1 + i];     // v' = (f_L + f_R)/m + g
  S tau[3];
  for (int i = 0; i < 3; ++i) tau[i] = 0.0 * w0;
  for (int f = 0; f < 2; ++f) {                                          // r x f, r = foot - p
    S r[3]; for (int i = 0; i < 3; ++i) r[i] = mp[7 + 3 * f + i] - x[i];
    const S* F = u + 3 * f;
    tau[0] = tau[0] + (r[1] * F[2] - r[2] * F[1]); tau[1] = tau[1] + (r[2] * F[0] - r[0] * F[2]); tau[2] = tau[2] + (r[0] * F[1] - r[1] * F[0]);
  }
  const S Iw0 = mp[4] * w0, Iw1 = mp[5] * w1, Iw2 = mp[6] * w2;          // omega x (I omega)
  xd[9] = (1.0 / mp[4]) * (tau[0] - (w1 * Iw2 - w2 * Iw1));
  xd[10] = (1.0 / mp[5]) * (tau[1] - (w2 * Iw0 - w0 * Iw2));
  xd[11] = (1.0 / mp[6]) * (tau[2] - (w0 * Iw1 - w1 * Iw0));
}
template <typename S>
void srb_rk4(const double* mp, double dt, const S* x, const S* u, S* xn) {   // classical RK4: x+ = x + dt/6 (k1 + 2 k2 + 2 k3 + k4)
  S k1[12], k2[12], k3[12], k4[12], xt[12];
  srb_xdot(mp, x, u, k1);
  for (int i = 0; i < 12; ++i) xt[i] = x[i] + (0.5 * dt) * k1[i];
  srb_xdot(mp, xt, u, k2);
  for (int i = 0; i < 12; ++i) xt[i] = x[i] + (0.5 * dt) * k2[i];
  srb_xdot(mp, xt, u, k3);
  for (int i = 0; i < 12; ++i) xt[i] = x[i] + dt * k3[i];
  srb_xdot(mp, xt, u, k4);
  for (int i = 0; i < 12; ++i) xn[i] = x[i] + (dt / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
}
// eq. 36-37 for f_k(v_k, v_{k+1}) = Phi(x_k, u_k) - x_{k+1}: Am = [dPhi/dx dPhi/du] (one Dual sweep per column), Ap = [-I 0], b = Am v_k + Ap v_{k+1} - f_k
void srb_linearize(const Cfg& cf, const double* xbar, double* Am, double* Ap, double* b) {
  const int N = cf.N, n = 18, nx = 12;
  for (int t = 0; t < N; ++t) {
    const double* vk = xbar + (size_t)t * n; const double* vk1 = vk + n;
    double* am = Am + (size_t)t * nx * n; double* ap = Ap + (size_t)t * nx * n;
    for (int j = 0; j < n; ++j) {
      Dual xd[12], ud[6], out[12];
      for (int i = 0; i < 12; ++i) xd[i] = {vk[i], i == j ? 1.0 : 0.0};
      for (int i = 0; i < 6; ++i) ud[i] = {vk[12 + i], 12 + i == j ? 1.0 : 0.0};
      srb_rk4<Dual>(cf.model_params, cf.dt, xd, ud, out);
      for (int i = 0; i < nx; ++i) am[i * n + j] = out[i].d;
    }
    for (int i = 0; i < nx; ++i) for (int j = 0; j < n; ++j) ap[i * n + j] = (i == j) ? -1.0 : 0.0;
    double phi[12]; srb_rk4<double>(cf.model_params, cf.dt, vk, vk + 12, phi);
    for (int i = 0; i < nx; ++i) {
      double sacc = -(phi[i] - vk1[i]);
      for (int j = 0; j < n; ++j) sacc += am[i * n + j] * vk[j] + ap[i * n + j] * vk1[j];
      b[(size_t)t * nx + i] = sacc;
    }
  }
}

// ---- f2: SQP with the l1-merit backtracking linesearch of App. D and the convergence test eq. 18
// (PAPER.md:305-314), for the bicycle model.  Readings (A-34..A-37):
//   x~ = (x, xi); l(x~) = 1/2 x'Px + q'x + sum_soft (lam |xi| + gamma/2 xi^2); f(x~) = (x_0 - x_init ; f_k(v_k, v_{k+1}));
//   g(x~) = G x + xi on soft rows, G x on hard rows (g is linear for this model, so the shifted bounds of eq. 38 are exact);
//   c1 = |f|_1 + |[g - hi]_+|_1 + |[lo - g]_+|_1;  dl = (Px + q)'dx + sum_soft (lam s_i + gamma xi_i) dxi_i with s_i = sgn(xi_i), or
//   sgn(dxi_i) where xi_i = 0 (one-sided derivative of |.|);  mu = max(0, dl / (1/2 max(c1, eps_c)));  D_mu = dl - mu c1;
//   candidates alpha_j = 2^-j, j = 0..J-1: the largest with phi(x~ + alpha d) <= phi(x~) + eta alpha D_mu, else the one with the smallest phi;
//   (x, xi, y_f, y_g) <- (x, xi, y_f, y_g) + alpha ((x*, xi*, y_f*, y_g*) - (x, xi, y_f, y_g)).
//   eq. 18 at the new iterate, with the Jacobians re-linearised there: |Px + q + C'y_f + G'y_g|_inf, |f|_inf, max bound violation, all <= eps_c.
struct SqpOpt { int32_t max_sqp, admm_iters, n_alpha, pad; double eps_c, eta; };

double merit_parts(const Cfg& c, const Band& P, const vec& q, const double* x_init, const double* x, const double* xi, const double* G, const double* lo,
                   const double* hi, double* cost_out, double* finf_out, double* ginf_out) {
  const int N = c.N, T = N + 1, n = 6, nx = 4, ng = 3, nz = T * n;
  vec xv(x, x + nz), Px(nz); band_mul(P, xv, Px);
  double cost = 0; for (int i = 0; i < nz; ++i) cost += 0.5 * x[i] * Px[i] + q[i] * x[i];
  double c1 = 0, finf = 0, ginf = 0, f[4];
  for (int i = 0; i < nx; ++i) { double r = x[i] - x_init[i]; c1 += std::fabs(r); finf = std::max(finf, std::fabs(r)); }
  for (int t = 0; t < N; ++t) { bicycle_residual(c.wheelbase, c.dt, x + (size_t)t * n, x + (size_t)(t + 1) * n, f); for (int i = 0; i < 4; ++i) { c1 += std::fabs(f[i]); finf = std::max(finf, std::fabs(f[i])); } }
  for (int t = 0; t < T; ++t) for (int r = 0; r < ng; ++r) {
    const int e = t * ng + r; double g = 0; for (int j = 0; j < n; ++j) g += G[(size_t)e * n + j] * x[t * n + j];
    if (c.soft[r]) { g += xi[e]; cost += c.lam * std::fabs(xi[e]) + 0.5 * c.gamma * xi[e] * xi[e]; }
    double v = std::max(0.0, g - hi[e]) + std::max(0.0, lo[e] - g);
    c1 += v; ginf = std::max(ginf, v);
  }
  *cost_out = cost; if (finf_out) *finf_out = finf; if (ginf_out) *ginf_out = ginf;
  return c1;
}

// log_out (optional): 10 doubles per SQP iteration: alpha, mu, phi0, phi(alpha), c1, dl, armijo-accepted flag, then eq. 18 after the step: stat, |f|_inf, viol
int sqp_ls_bicycle(const Cfg& cf_in, const SqpOpt& op, const double* D, const double* E, const double* q_, const double* x_init, const double* ref, double* xbar,
                   double* zg, double* yf, double* yg, double* xi, double* info_out, double* log_out) {
  Cfg c = cf_in; c.g_sel = 0; c.zg_given = 0;
  const int N = c.N, T = N + 1, n = 6, nx = 4, ng = 3, nz = T * n, mf = nx + N * nx, mg = T * ng;
  vec Am((size_t)N * nx * n), Ap((size_t)N * nx * n), b((size_t)N * nx), G((size_t)T * ng * n), lo(mg), hi(mg), q(q_, q_ + nz);
  vec xs(nz), zs(mg), yfs(mf), ygs(mg), xis(mg), xc(nz), xic(mg), g(nz), Px(nz);
  int fail = 0, it = 0, converged = 0;
  double stat = 0, finf = 0, ginf = 0;
  for (it = 0; it < op.max_sqp && !converged; ) {
    bicycle_linearize(c, xbar, ref, Am.data(), Ap.data(), b.data(), G.data(), lo.data(), hi.data());
    QP p = assemble(c, D, E, q.data(), Am.data(), Ap.data(), b.data(), x_init, G.data(), lo.data(), hi.data());
    // QP solve (Alg. 3) warm-started at (xbar, y); the solution goes to (xs, xis, yfs, ygs)
    std::copy(xbar, xbar + nz, xs.begin()); std::copy(yf, yf + mf, yfs.begin()); std::copy(yg, yg + mg, ygs.begin());
    double inf4[4]; Info ai = admm(c, p, xs.data(), zs.data(), yfs.data(), ygs.data(), xis.data(), op.admm_iters); (void)inf4;
    if (!(ai.min_pivot > 0)) fail = 1;
    // linesearch (App. D)
    double cost0, c1 = merit_parts(c, p.P, q, x_init, xbar, xi, G.data(), lo.data(), hi.data(), &cost0, nullptr, nullptr);
    vec xb(xbar, xbar + nz); band_mul(p.P, xb, Px);
    double dl = 0; for (int i = 0; i < nz; ++i) dl += (Px[i] + q[i]) * (xs[i] - xbar[i]);
    for (int e = 0; e < mg; ++e) if (c.soft[e % ng]) { double dxi = xis[e] - xi[e]; double sg = xi[e] > 0 ? 1.0 : (xi[e] < 0 ? -1.0 : (dxi > 0 ? 1.0 : (dxi < 0 ? -1.0 : 0.0))); dl += (c.lam * sg + c.gamma * xi[e]) * dxi; }
    const double mu = std::max(0.0, dl / (0.5 * std::max(c1, op.eps_c))), phi0 = cost0 + mu * c1, Dmu = dl - mu * c1;
    double alpha = 0, best_phi = std::numeric_limits<double>::infinity(), best_alpha = 1.0, phi_a = 0; int accepted = 0;
    for (int j = 0; j < op.n_alpha && !accepted; ++j) {
      const double a = std::ldexp(1.0, -j);
      for (int i = 0; i < nz; ++i) xc[i] = xbar[i] + a * (xs[i] - xbar[i]);
      for (int e = 0; e < mg; ++e) xic[e] = xi[e] + a * (xis[e] - xi[e]);
      double costa, c1a = merit_parts(c, p.P, q, x_init, xc.data(), xic.data(), G.data(), lo.data(), hi.data(), &costa, nullptr, nullptr);
      const double phi = costa + mu * c1a;
      if (phi < best_phi) { best_phi = phi; best_alpha = a; }
      if (phi <= phi0 + op.eta * a * Dmu) { alpha = a; phi_a = phi; accepted = 1; }
    }
    if (!accepted) { alpha = best_alpha; phi_a = best_phi; }
    for (int i = 0; i < nz; ++i) xbar[i] += alpha * (xs[i] - xbar[i]);
    for (int e = 0; e < mg; ++e) { xi[e] += alpha * (xis[e] - xi[e]); yg[e] += alpha * (ygs[e] - yg[e]); zg[e] = zs[e]; }
    for (int e = 0; e < mf; ++e) yf[e] += alpha * (yfs[e] - yf[e]);
    ++it;
    // eq. 18 at the new iterate (Jacobians re-linearised there)
    bicycle_linearize(c, xbar, ref, Am.data(), Ap.data(), b.data(), G.data(), lo.data(), hi.data());
    QP pn = assemble(c, D, E, q.data(), Am.data(), Ap.data(), b.data(), x_init, G.data(), lo.data(), hi.data());
    vec xn(xbar, xbar + nz), yfv(yf, yf + mf), ygv(yg, yg + mg); band_mul(pn.P, xn, Px);
    for (int i = 0; i < nz; ++i) g[i] = Px[i] + q[i];
    pn.C.mulT_add(yfv, g); pn.G.mulT_add(ygv, g);
    stat = 0; for (int i = 0; i < nz; ++i) stat = std::max(stat, std::fabs(g[i]));
    double cdummy; merit_parts(c, pn.P, q, x_init, xbar, xi, G.data(), lo.data(), hi.data(), &cdummy, &finf, &ginf);
    converged = stat <= op.eps_c && finf <= op.eps_c && ginf <= op.eps_c;
    if (log_out) { double* l = log_out + 10 * (it - 1); l[0] = alpha; l[1] = mu; l[2] = phi0; l[3] = phi_a; l[4] = c1; l[5] = dl; l[6] = accepted; l[7] = stat; l[8] = finf; l[9] = ginf; }
  }
  info_out[0] = it; info_out[1] = converged; info_out[2] = stat; info_out[3] = finf; info_out[4] = ginf;
  return fail;
}

// ---- f2 for the SRB humanoid model (second built-in model): the same App. D linesearch and eq. 18 test as sqp_ls_bicycle, with
//   f(x~) = (x_0 - x_init ; Phi(x_k, u_k) - x_{k+1}) (RK4 of eq. 68), g(x~) = the selected components of v_t (+ xi on soft rows) against the
//   caller's constant bounds (eq. 70d).  Kept apart from the bicycle routine so that its pinned arithmetic is not touched.
double merit_parts_srb(const Cfg& c, const Band& P, const vec& q, const double* x_init, const double* x, const double* xi, const double* lo,
                       const double* hi, double* cost_out, double* finf_out, double* ginf_out) {
  const int N = c.N, T = N + 1, n = 18, nx = 12, ng = c.ng, nz = T * n;
  vec xv(x, x + nz), Px(nz); band_mul(P, xv, Px);
  double cost = 0; for (int i = 0; i < nz; ++i) cost += 0.5 * x[i] * Px[i] + q[i] * x[i];
  double c1 = 0, finf = 0, ginf = 0, phi[12];
  for (int i = 0; i < nx; ++i) { double r = x[i] - x_init[i]; c1 += std::fabs(r); finf = std::max(finf, std::fabs(r)); }
  for (int t = 0; t < N; ++t) {
    const double* vk = x + (size_t)t * n; const double* vk1 = vk + n;
    srb_rk4<double>(c.model_params, c.dt, vk, vk + 12, phi);
    for (int i = 0; i < nx; ++i) { const double f = phi[i] - vk1[i]; c1 += std::fabs(f); finf = std::max(finf, std::fabs(f)); }
  }
  for (int t = 0; t < T; ++t) for (int r = 0; r < ng; ++r) {
    const int e = t * ng + r; double g = x[t * n + c.g_col[r]];
    if (c.soft[r]) { g += xi[e]; cost += c.lam * std::fabs(xi[e]) + 0.5 * c.gamma * xi[e] * xi[e]; }
    double v = std::max(0.0, g - hi[e]) + std::max(0.0, lo[e] - g);
    c1 += v; ginf = std::max(ginf, v);
  }
  *cost_out = cost; if (finf_out) *finf_out = finf; if (ginf_out) *ginf_out = ginf;
  return c1;
}

// log_out as in sqp_ls_bicycle
int sqp_ls_srb(const Cfg& cf_in, const SqpOpt& op, const double* D, const double* E, const double* q_, const double* x_init, const double* lo, const double* hi,
               double* xbar, double* zg, double* yf, double* yg, double* xi, double* info_out, double* log_out) {
  Cfg c = cf_in; c.g_sel = 1; c.zg_given = 0;
  const int N = c.N, T = N + 1, n = 18, nx = 12, ng = c.ng, nz = T * n, mf = nx + N * nx, mg = T * ng;
  vec Am((size_t)N * nx * n), Ap((size_t)N * nx * n), b((size_t)N * nx), q(q_, q_ + nz);
  vec xs(nz), zs(mg), yfs(mf), ygs(mg), xis(mg), xc(nz), xic(mg), g(nz), Px(nz);
  int fail = 0, it = 0, converged = 0;
  double stat = 0, finf = 0, ginf = 0;
  for (it = 0; it < op.max_sqp && !converged; ) {
    srb_linearize(c, xbar, Am.data(), Ap.data(), b.data());
    QP p = assemble(c, D, E, q.data(), Am.data(), Ap.data(), b.data(), x_init, nullptr, lo, hi);
    std::copy(xbar, xbar + nz, xs.begin()); std::copy(yf, yf + mf, yfs.begin()); std::copy(yg, yg + mg, ygs.begin());
    Info ai = admm(c, p, xs.data(), zs.data(), yfs.data(), ygs.data(), xis.data(), op.admm_iters);
    if (!(ai.min_pivot > 0)) fail = 1;
    double cost0, c1 = merit_parts_srb(c, p.P, q, x_init, xbar, xi, lo, hi, &cost0, nullptr, nullptr);
    vec xb(xbar, xbar + nz); band_mul(p.P, xb, Px);
    double dl = 0; for (int i = 0; i < nz; ++i) dl += (Px[i] + q[i]) * (xs[i] - xbar[i]);
    for (int e = 0; e < mg; ++e) if (c.soft[e % ng]) { double dxi = xis[e] - xi[e]; double sg = xi[e] > 0 ? 1.0 : (xi[e] < 0 ? -1.0 : (dxi > 0 ? 1.0 : (dxi < 0 ? -1.0 : 0.0))); dl += (c.lam * sg + c.gamma * xi[e]) * dxi; }
    const double mu = std::max(0.0, dl / (0.5 * std::max(c1, op.eps_c))), phi0 = cost0 + mu * c1, Dmu = dl - mu * c1;
    double alpha = 0, best_phi = std::numeric_limits<double>::infinity(), best_alpha = 1.0, phi_a = 0; int accepted = 0;
    for (int j = 0; j < op.n_alpha && !accepted; ++j) {
      const double a = std::ldexp(1.0, -j);
      for (int i = 0; i < nz; ++i) xc[i] = xbar[i] + a * (xs[i] - xbar[i]);
      for (int e = 0; e < mg; ++e) xic[e] = xi[e] + a * (xis[e] - xi[e]);
      double costa, c1a = merit_parts_srb(c, p.P, q, x_init, xc.data(), xic.data(), lo, hi, &costa, nullptr, nullptr);
      const double phi = costa + mu * c1a;
      if (phi < best_phi) { best_phi = phi; best_alpha = a; }
      if (phi <= phi0 + op.eta * a * Dmu) { alpha = a; phi_a = phi; accepted = 1; }
    }
    if (!accepted) { alpha = best_alpha; phi_a = best_phi; }
    for (int i = 0; i < nz; ++i) xbar[i] += alpha * (xs[i] - xbar[i]);
    for (int e = 0; e < mg; ++e) { xi[e] += alpha * (xis[e] - xi[e]); yg[e] += alpha * (ygs[e] - yg[e]); zg[e] = zs[e]; }
    for (int e = 0; e < mf; ++e) yf[e] += alpha * (yfs[e] - yf[e]);
    ++it;
    srb_linearize(c, xbar, Am.data(), Ap.data(), b.data());
    QP pn = assemble(c, D, E, q.data(), Am.data(), Ap.data(), b.data(), x_init, nullptr, lo, hi);
    vec xn(xbar, xbar + nz), yfv(yf, yf + mf), ygv(yg, yg + mg); band_mul(pn.P, xn, Px);
    for (int i = 0; i < nz; ++i) g[i] = Px[i] + q[i];
    pn.C.mulT_add(yfv, g); pn.G.mulT_add(ygv, g);
    stat = 0; for (int i = 0; i < nz; ++i) stat = std::max(stat, std::fabs(g[i]));
    double cdummy; merit_parts_srb(c, pn.P, q, x_init, xbar, xi, lo, hi, &cdummy, &finf, &ginf);
    converged = stat <= op.eps_c && finf <= op.eps_c && ginf <= op.eps_c;
    if (log_out) { double* l = log_out + 10 * (it - 1); l[0] = alpha; l[1] = mu; l[2] = phi0; l[3] = phi_a; l[4] = c1; l[5] = dl; l[6] = accepted; l[7] = stat; l[8] = finf; l[9] = ginf; }
  }
  info_out[0] = it; info_out[1] = converged; info_out[2] = stat; info_out[3] = finf; info_out[4] = ginf;
  return fail;
}

}  // namespace

extern "C" {

// Dense S [nz][nz] (full symmetric) for the Theta/Phi pin.
int orc_assemble_S(const Cfg* cf, const double* D, const double* E, const double* Am, const double* Ap, const double* G, double* S_out) {
  int n = cf->nx + cf->nu, nz = (cf->N + 1) * n, T = cf->N + 1;
  vec q(nz, 0.0), b((size_t)cf->N * cf->nx, 0.0), xi(cf->nx, 0.0), lo((size_t)T * cf->ng, 0.0);
  QP p = assemble(*cf, D, E, q.data(), Am, Ap, b.data(), xi.data(), G, lo.data(), lo.data());
  Band S = build_S(p, cf->sigma, vec(p.mf, cf->rho_eq_scale * cf->rho_bar), vec(p.mg, cf->rho_bar));
  for (int i = 0; i < nz; ++i) for (int j = 0; j < nz; ++j) S_out[(size_t)i * nz + j] = S.get(i, j);
  return 0;
}

// x~ = S^{-1} eta by O-2 (pin for the block factor, the solves and the cyclic reduction).  Returns 0, or 1 on a non-positive pivot.
int orc_solve_S(const Cfg* cf, const double* D, const double* E, const double* Am, const double* Ap, const double* G, const double* eta, double* xt) {
  int n = cf->nx + cf->nu, nz = (cf->N + 1) * n, T = cf->N + 1;
  vec q(nz, 0.0), b((size_t)cf->N * cf->nx, 0.0), xi(cf->nx, 0.0), lo((size_t)T * cf->ng, 0.0);
  QP p = assemble(*cf, D, E, q.data(), Am, Ap, b.data(), xi.data(), G, lo.data(), lo.data());
  Band L = build_S(p, cf->sigma, vec(p.mf, cf->rho_eq_scale * cf->rho_bar), vec(p.mg, cf->rho_bar));
  double piv = cholesky(L); vec x(eta, eta + nz); chol_solve(L, x); std::copy(x.begin(), x.end(), xt);
  return piv > 0 ? 0 : 1;
}

void orc_project(int soft, double v, double lo, double hi, double rho, double gamma, double lam, double* z, double* xi) { project_row(soft != 0, v, lo, hi, rho, gamma, lam, *z, *xi); }

// One problem, K iterations of Alg. 3.  info_out[4] = r_prim, r_dual, objective, min Cholesky pivot.
int orc_admm(const Cfg* cf, const double* D, const double* E, const double* q, const double* Am, const double* Ap, const double* b, const double* x_init,
             const double* G, const double* lo, const double* hi, double* x, double* zg, double* yf, double* yg, double* xi, int K, double* info_out) {
  QP p = assemble(*cf, D, E, q, Am, Ap, b, x_init, G, lo, hi);
  Info i = admm(*cf, p, x, zg, yf, yg, xi, K);
  info_out[0] = i.r_prim; info_out[1] = i.r_dual; info_out[2] = i.objective; info_out[3] = i.min_pivot;
  return i.min_pivot > 0 ? 0 : 1;
}

// One problem with a per-row soft flag array soft_rows [mg] (adjoint QP, eq. 67).
int orc_admm_rows(const Cfg* cf, const double* D, const double* E, const double* q, const double* Am, const double* Ap, const double* b, const double* x_init,
                  const double* G, const double* lo, const double* hi, const uint8_t* soft_rows, double* x, double* zg, double* yf, double* yg, double* xi, int K,
                  double* info_out) {
  QP p = assemble(*cf, D, E, q, Am, Ap, b, x_init, G, lo, hi);
  Info i = admm(*cf, p, x, zg, yf, yg, xi, K, soft_rows);
  info_out[0] = i.r_prim; info_out[1] = i.r_dual; info_out[2] = i.objective; info_out[3] = i.min_pivot;
  return i.min_pivot > 0 ? 0 : 1;
}

// Batch of independent problems spread over nthreads std::threads (each problem stays single-threaded).  Strides in elements; 0 = shared.
int orc_admm_batch(const Cfg* cf, int B, int nthreads, const double* D, int64_t sD, const double* E, int64_t sE, const double* q, const double* Am,
                   const double* Ap, const double* b, const double* x_init, const double* G, int64_t sG, const double* lo, const double* hi,
                   double* x, double* zg, double* yf, double* yg, double* xi, int K, double* info_out) {
  const int n = cf->nx + cf->nu, T = cf->N + 1, nz = T * n, mf = cf->nx + cf->N * cf->nx, mg = T * cf->ng;
  std::vector<int> fail(std::max(1, nthreads), 0);
  auto work = [&](int tid) {
    for (int p = tid; p < B; p += nthreads)
      fail[tid] |= orc_admm(cf, D + sD * p, E + sE * p, q + (size_t)nz * p, Am + (size_t)cf->N * cf->nx * n * p, Ap + (size_t)cf->N * cf->nx * n * p,
                            b + (size_t)cf->N * cf->nx * p, x_init + (size_t)cf->nx * p, G ? G + sG * p : nullptr, lo + (size_t)mg * p, hi + (size_t)mg * p,
                            x + (size_t)nz * p, zg + (size_t)mg * p, yf + (size_t)mf * p, yg + (size_t)mg * p, xi + (size_t)mg * p, K, info_out + 4 * (size_t)p);
  };
  if (nthreads <= 1) { nthreads = 1; work(0); }
  else { std::vector<std::thread> th; for (int t = 0; t < nthreads; ++t) th.emplace_back(work, t); for (auto& t : th) t.join(); }
  int f = 0; for (int v : fail) f |= v; return f;
}

// O-5 for one problem.  counts_out[2] = #hard-active, #soft-active.  Returns 0, or 2 when the KKT system is (numerically) singular (reading A-18).
int orc_backward(const Cfg* cf, const double* D, const double* E, const double* q, const double* Am, const double* Ap, const double* b, const double* x_init,
                 const double* G, const double* lo, const double* hi, const double* x, const double* yg, const double* xi, const double* dLdx,
                 const double* dLdxi, double* dq, double* dxinit, int* counts_out, double* dgamma_out) {
  Cfg c = *cf;
  QP p = assemble(c, D, E, q, Am, Ap, b, x_init, G, lo, hi);
  double piv = backward(c, p, x, yg, xi, dLdx, dLdxi, dq, dxinit, &counts_out[0], &counts_out[1], dgamma_out);
  return piv > 1e-12 ? 0 : 2;
}

int orc_classify(const Cfg* cf, const double* D, const double* E, const double* q, const double* Am, const double* Ap, const double* b, const double* x_init,
                 const double* G, const double* lo, const double* hi, const double* x, const double* yg, const double* xi, int32_t* cls_out) {
  QP p = assemble(*cf, D, E, q, Am, Ap, b, x_init, G, lo, hi);
  std::vector<int> cls; classify(*cf, p, x, yg, xi, cls); for (int i = 0; i < p.mg; ++i) cls_out[i] = cls[i];
  return 0;
}

void orc_bicycle_residual(const Cfg* cf, const double* vk, const double* vk1, double* f) { bicycle_residual(cf->wheelbase, cf->dt, vk, vk1, f); }
void orc_bicycle_linearize(const Cfg* cf, const double* xbar, const double* ref, double* Am, double* Ap, double* b, double* G, double* lo, double* hi) {
  bicycle_linearize(*cf, xbar, ref, Am, Ap, b, G, lo, hi);
}

// O-4.  n_sqp x (linearise at xbar -> K ADMM iterations warm-started with x^0 = xbar, y carried, z_g re-projected -> full step), reading A-26.
// xbar [T][n] in/out (final iterate), yf/yg in/out, xi/zg out.  fnorm_out[n_sqp+1]: ||f(xbar)||_inf before each step and after the last.
int orc_sqp_bicycle(const Cfg* cf, const double* D, const double* E, const double* q, const double* x_init, const double* ref, double* xbar, double* zg,
                    double* yf, double* yg, double* xi, int n_sqp, int K, double* info_out, double* fnorm_out) {
  const int N = cf->N, T = N + 1, n = 6, nx = 4, ng = 3;
  vec Am((size_t)N * nx * n), Ap((size_t)N * nx * n), b((size_t)N * nx), G((size_t)T * ng * n), lo((size_t)T * ng), hi((size_t)T * ng);
  Cfg c = *cf; c.g_sel = 0; c.zg_given = 0; int fail = 0;
  auto fnorm = [&]() { double m = 0, f[4]; for (int t = 0; t < N; ++t) { bicycle_residual(c.wheelbase, c.dt, xbar + (size_t)t * n, xbar + (size_t)(t + 1) * n, f); for (int i = 0; i < 4; ++i) m = std::max(m, std::fabs(f[i])); } return m; };
  for (int s = 0; s < n_sqp; ++s) {
    if (fnorm_out) fnorm_out[s] = fnorm();
    bicycle_linearize(c, xbar, ref, Am.data(), Ap.data(), b.data(), G.data(), lo.data(), hi.data());
    fail |= orc_admm(&c, D, E, q, Am.data(), Ap.data(), b.data(), x_init, G.data(), lo.data(), hi.data(), xbar, zg, yf, yg, xi, K, info_out);
  }
  if (fnorm_out) fnorm_out[n_sqp] = fnorm();
  return fail;
}

int orc_sqp_bicycle_batch(const Cfg* cf, int B, int nthreads, const double* D, const double* E, const double* q, const double* x_init, const double* ref,
                          double* xbar, double* zg, double* yf, double* yg, double* xi, int n_sqp, int K, double* info_out) {
  const int T = cf->N + 1, n = 6, nz = T * n, mf = 4 + cf->N * 4, mg = T * 3;
  std::vector<int> fail(std::max(1, nthreads), 0);
  auto work = [&](int tid) {
    for (int p = tid; p < B; p += nthreads)
      fail[tid] |= orc_sqp_bicycle(cf, D, E, q + (size_t)nz * p, x_init + (size_t)4 * p, ref + (size_t)nz * p, xbar + (size_t)nz * p, zg + (size_t)mg * p,
                                   yf + (size_t)mf * p, yg + (size_t)mg * p, xi + (size_t)mg * p, n_sqp, K, info_out + 4 * (size_t)p, nullptr);
  };
  if (nthreads <= 1) { nthreads = 1; work(0); }
  else { std::vector<std::thread> th; for (int t = 0; t < nthreads; ++t) th.emplace_back(work, t); for (auto& t : th) t.join(); }
  int f = 0; for (int v : fail) f |= v; return f;
}

// f1: one problem, adaptive rho + termination.  info_out[8] = r_prim, r_dual, objective, min pivot, iterations, final rho_bar, converged, #log rows.
int orc_admm_adaptive(const Cfg* cf, const Adaptive* ad, const double* D, const double* E, const double* q, const double* Am, const double* Ap, const double* b,
                      const double* x_init, const double* G, const double* lo, const double* hi, double* x, double* zg, double* yf, double* yg, double* xi,
                      double* info_out, double* log_out, int max_log) {
  QP p = assemble(*cf, D, E, q, Am, Ap, b, x_init, G, lo, hi);
  return admm_adaptive(*cf, p, *ad, x, zg, yf, yg, xi, info_out, log_out, max_log);
}
int orc_sizeof_adaptive() { return (int)sizeof(Adaptive); }

// f2 for one problem.  info_out[5] = SQP iterations, converged, eq. 18 quantities (stationarity, |f|_inf, bound violation); log_out [max_sqp][10].
int orc_sqp_ls_bicycle(const Cfg* cf, const SqpOpt* op, const double* D, const double* E, const double* q, const double* x_init, const double* ref, double* xbar,
                       double* zg, double* yf, double* yg, double* xi, double* info_out, double* log_out) {
  return sqp_ls_bicycle(*cf, *op, D, E, q, x_init, ref, xbar, zg, yf, yg, xi, info_out, log_out);
}
int orc_sizeof_sqpopt() { return (int)sizeof(SqpOpt); }

// f3: SRB humanoid model.  orc_srb_step: x+ = Phi(x, u) (RK4 of eq. 68); orc_srb_linearize: eq. 36-37 blocks; orc_sqp_srb: the fixed-count full-step
// SQP driver of O-4 (reading A-26) around them, inequality rows = selection rows with the caller's constant bounds (eq. 70d).
void orc_srb_step(const Cfg* cf, const double* x, const double* u, double* xn) { srb_rk4<double>(cf->model_params, cf->dt, x, u, xn); }
void orc_srb_linearize(const Cfg* cf, const double* xbar, double* Am, double* Ap, double* b) { srb_linearize(*cf, xbar, Am, Ap, b); }
int orc_sqp_srb(const Cfg* cf, const double* D, const double* E, const double* q, const double* x_init, const double* lo, const double* hi, double* xbar,
                double* zg, double* yf, double* yg, double* xi, int n_sqp, int K, double* info_out) {
  const int N = cf->N, n = 18, nx = 12;
  vec Am((size_t)N * nx * n), Ap((size_t)N * nx * n), b((size_t)N * nx);
  Cfg c = *cf; c.g_sel = 1; c.zg_given = 0; int fail = 0;
  for (int s = 0; s < n_sqp; ++s) {
    srb_linearize(c, xbar, Am.data(), Ap.data(), b.data());
    fail |= orc_admm(&c, D, E, q, Am.data(), Ap.data(), b.data(), x_init, nullptr, lo, hi, xbar, zg, yf, yg, xi, K, info_out);
  }
  return fail;
}

int orc_sqp_ls_srb(const Cfg* cf, const SqpOpt* op, const double* D, const double* E, const double* q, const double* x_init, const double* lo, const double* hi,
                   double* xbar, double* zg, double* yf, double* yg, double* xi, double* info_out, double* log_out) {
  return sqp_ls_srb(*cf, *op, D, E, q, x_init, lo, hi, xbar, zg, yf, yg, xi, info_out, log_out);
}

int orc_sizeof_cfg() { return (int)sizeof(Cfg); }

}  // extern "C"
