// tmpc_sqp.cuh — f2: the SQP outer loop of Alg. 1 around the ADMM solve for the two built-in models (MODEL = 1: kinematic
// bicycle, implicit midpoint, dense G rows; MODEL = 2: SRB humanoid, RK4, f_k = Phi(x_k, u_k) - x_{k+1}, selection rows with constant bounds):
// l1-merit backtracking linesearch with the step-size candidates evaluated in parallel (App. D) and the
// convergence test eq. 18.  Readings A-34..A-37 of DESIGN.md:
//   x~ = (x, xi);  l(x~) = 1/2 x'Px + q'x + sum_soft (lam |xi| + gamma/2 xi^2);  f(x~) = (x_0 - x_init ; f_k(v_k, v_{k+1}));
//   g(x~) = G x + xi on soft rows (g is linear for this model, the shifted bounds of eq. 38 are exact);
//   c1 = |f|_1 + |[g - hi]_+|_1 + |[lo - g]_+|_1;  dl = (Px + q)'dx + sum_soft (lam s + gamma xi) dxi, s = sgn(xi) or sgn(dxi) at xi = 0;
//   mu = max(0, dl / (1/2 max(c1, eps_c)));  D_mu = dl - mu c1;  alpha_j = 2^-j: the largest with phi(alpha) <= phi(0) + eta alpha D_mu,
//   else the one with the smallest phi;  (x, xi, y_f, y_g) += alpha ((x*, xi*, y_f*, y_g*) - (x, xi, y_f, y_g)).
// All sums and decisions are taken in double, in a fixed order (warp j owns candidate j, lanes stride over the stages,
// shuffle tree), so a run is reproducible.
#pragma once
#include "tmpc_common.cuh"
#include "tmpc_srb.cuh"

namespace tmpc {

constexpr int SQP_MAX_ALPHA = 15;      // candidates alpha = 2^0 .. 2^-(n_alpha-1); one warp each plus one for the current point

template <typename T>
struct SqpArgs {
  Dims d; QpView<T> qp;
  double Lwb, dt, gamma, lam, eps_c, eta;
  double mp[13];                                               // SRB model parameters (tmpc_config.model_params)
  int n_alpha, it;
  const int32_t* active;
  const T* ox; const T* oxi; const T* oyf; const T* oyg;      // iterate before the QP solve  [B][nz], [B][mg], [B][mf], [B][mg]
  T* x; T* xi; T* yf; T* yg;                                   // in: QP solution (x*, xi*, y*); out: the new iterate
  T* alpha_log; int max_sqp;                                   // optional [B][max_sqp]
  // eq. 18
  T* kkt;                                                      // [B][3]: stationarity, |f|_inf, bound violation
  int32_t* act_rw; int32_t* iters; int32_t* converged; int32_t* n_active;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// implicit-midpoint residual of the kinematic bicycle (reading A-24), double
__device__ __forceinline__ void bicycle_res(double Lwb, double dt, const double* vk, const double* vk1, double* f) {
  const double psi = 0.5 * (vk[2] + vk1[2]), vel = 0.5 * (vk[3] + vk1[3]);
  double sn, cs; sincos(psi, &sn, &cs);
  f[0] = vk[0] + dt * vel * cs - vk1[0]; f[1] = vk[1] + dt * vel * sn - vk1[1];
  f[2] = vk[2] + dt * vel / Lwb * tan(vk[5]) - vk1[2]; f[3] = vk[3] + dt * vk[4] - vk1[3];
}

// Phi(x, u) - x_next of the SRB model in double: the RK4 step of tmpc_srb.cuh on Fwd<double> numbers with zero derivative parts
__device__ __forceinline__ void srb_res(const double* mp, double dt, const double* vk, const double* vk1, double* f) {
  Fwd<double> x[12], u[6], k1[12], k2[12], k3[12], k4[12], xt[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) x[i] = {vk[i], 0.0};
#pragma unroll
  for (int i = 0; i < 6; ++i) u[i] = {vk[12 + i], 0.0};
  srb_rhs<double>(mp, x, u, k1);
#pragma unroll
  for (int i = 0; i < 12; ++i) xt[i] = x[i] + scale(0.5 * dt, k1[i]);
  srb_rhs<double>(mp, xt, u, k2);
#pragma unroll
  for (int i = 0; i < 12; ++i) xt[i] = x[i] + scale(0.5 * dt, k2[i]);
  srb_rhs<double>(mp, xt, u, k3);
#pragma unroll
  for (int i = 0; i < 12; ++i) xt[i] = x[i] + scale(dt, k3[i]);
  srb_rhs<double>(mp, xt, u, k4);
#pragma unroll
  for (int i = 0; i < 12; ++i) f[i] = (x[i] + scale(dt / 6.0, k1[i] + scale(2.0, k2[i]) + scale(2.0, k3[i]) + k4[i])).v - vk1[i];
}

// grid = B, block = 32 (n_alpha + 1): warp j < n_alpha evaluates the merit parts at alpha = 2^-j, warp n_alpha at alpha = 0 (plus dl)
template <typename T, int MODEL>
__global__ void __launch_bounds__(32 * (SQP_MAX_ALPHA + 1)) sqp_linesearch_kernel(SqpArgs<T> a) {
  __shared__ double s_cost[SQP_MAX_ALPHA + 1], s_c1[SQP_MAX_ALPHA + 1], s_dl, s_alpha;
  const Dims& d = a.d;
  const int p = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nA = a.n_alpha;
  if (a.active && !a.active[p]) return;
  constexpr int n = MODEL == 1 ? 6 : 18, nx = MODEL == 1 ? 4 : 12;
  const int ng = MODEL == 1 ? 3 : d.ng;
  const int N = d.N, T_ = d.T, nz = d.nz, mg = d.mg, mf = d.mf, nn = n * n;
  const T* ox = a.ox + (size_t)p * nz; const T* sx = a.x + (size_t)p * nz;
  const T* oxi = a.oxi + (size_t)p * mg; const T* sxi = a.xi + (size_t)p * mg;
  const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p; const T* q = a.qp.q + (size_t)p * nz;
  const T* G = MODEL == 1 ? a.qp.G + a.qp.sG * p : nullptr; const T* lo = a.qp.lo + (size_t)p * mg; const T* hi = a.qp.hi + (size_t)p * mg;
  const double al = warp < nA ? ldexp(1.0, -warp) : 0.0;
  double cost = 0, c1 = 0, dl = 0;
  for (int t = lane; t < T_; t += 32) {
    double v[n], v1[n], dx[n];
#pragma unroll
    for (int i = 0; i < n; ++i) { const double o = (double)ox[t * n + i]; dx[i] = (double)sx[t * n + i] - o; v[i] = o + al * dx[i]; }
    if (t < N) {
#pragma unroll
      for (int i = 0; i < n; ++i) { const double o = (double)ox[(t + 1) * n + i]; v1[i] = o + al * ((double)sx[(t + 1) * n + i] - o); }
    }
    // cost: 1/2 v'D_t v + q_t'v + v_{t+1}'E_t v_t ;  gradient (alpha = 0 warp): g_t = D_t v_t + E_{t-1} v_{t-1} + E_t' v_{t+1} + q_t
    double gq[n];
#pragma unroll
    for (int i = 0; i < n; ++i) { double s = 0;
#pragma unroll
      for (int j = 0; j < n; ++j) s += (double)Dp[(size_t)t * nn + i * n + j] * v[j];
      cost += 0.5 * v[i] * s + (double)q[t * n + i] * v[i]; gq[i] = s + (double)q[t * n + i]; }
    if (t < N) {
#pragma unroll
      for (int i = 0; i < n; ++i) { double s = 0;
#pragma unroll
        for (int j = 0; j < n; ++j) s += (double)Ep[(size_t)t * nn + i * n + j] * v[j];
        cost += v1[i] * s; }
    }
    if (warp == nA) {                                  // dl = (Px + q)' dx at the current point
      if (t < N) {
#pragma unroll
        for (int i = 0; i < n; ++i) { double s = 0;
#pragma unroll
          for (int j = 0; j < n; ++j) s += (double)Ep[(size_t)t * nn + j * n + i] * v1[j];
          gq[i] += s; }
      }
      if (t > 0) {
#pragma unroll
        for (int i = 0; i < n; ++i) { double s = 0;
#pragma unroll
          for (int j = 0; j < n; ++j) s += (double)Ep[(size_t)(t - 1) * nn + i * n + j] * (double)ox[(t - 1) * n + j];
          gq[i] += s; }
      }
#pragma unroll
      for (int i = 0; i < n; ++i) dl += gq[i] * dx[i];
    }
    // equality residuals
    if (t == 0) {
#pragma unroll
      for (int i = 0; i < nx; ++i) c1 += fabs(v[i] - (double)a.qp.x_init[(size_t)p * nx + i]);
    }
    if (t < N) {
      if constexpr (MODEL == 1) { double f[4]; bicycle_res(a.Lwb, a.dt, v, v1, f); c1 += fabs(f[0]) + fabs(f[1]) + fabs(f[2]) + fabs(f[3]); }
      else { double f[12]; srb_res(a.mp, a.dt, v, v1, f);
#pragma unroll
        for (int i = 0; i < 12; ++i) c1 += fabs(f[i]); }
    }
    // inequality rows with their slack
    for (int r = 0; r < ng; ++r) {
      const int e = t * ng + r;
      double g = 0;
      if constexpr (MODEL == 1) {
#pragma unroll
        for (int j = 0; j < n; ++j) g += (double)G[(size_t)e * n + j] * v[j];
      } else {
        const int col = d.g_col[r];
#pragma unroll
        for (int j = 0; j < n; ++j) if (j == col) g = v[j];
      }
      if ((d.soft_mask >> r) & 1u) {
        const double xo = (double)oxi[e], dxi = (double)sxi[e] - xo, xc = xo + al * dxi;
        g += xc; cost += a.lam * fabs(xc) + 0.5 * a.gamma * xc * xc;
        if (warp == nA) { const double sg = xo > 0 ? 1.0 : (xo < 0 ? -1.0 : (dxi > 0 ? 1.0 : (dxi < 0 ? -1.0 : 0.0))); dl += (a.lam * sg + a.gamma * xo) * dxi; }
      }
      c1 += fmax(0.0, g - (double)hi[e]) + fmax(0.0, (double)lo[e] - g);
    }
  }
  cost = warp_sum(cost); c1 = warp_sum(c1); dl = warp_sum(dl);
  if (lane == 0) { s_cost[warp] = cost; s_c1[warp] = c1; if (warp == nA) s_dl = dl; }
  __syncthreads();
  if (threadIdx.x == 0) {
    const double c10 = s_c1[nA], mu = fmax(0.0, s_dl / (0.5 * fmax(c10, a.eps_c))), phi0 = s_cost[nA] + mu * c10, Dmu = s_dl - mu * c10;
    double alpha = 0.0, best = INFINITY, best_a = 1.0; bool acc = false;
    for (int j = 0; j < nA && !acc; ++j) {
      const double aj = ldexp(1.0, -j), phi = s_cost[j] + mu * s_c1[j];
      if (phi < best) { best = phi; best_a = aj; }
      if (phi <= phi0 + a.eta * aj * Dmu) { alpha = aj; acc = true; }
    }
    if (!acc) alpha = best_a;
    s_alpha = alpha;
    if (a.alpha_log) a.alpha_log[(size_t)p * a.max_sqp + a.it] = (T)alpha;
  }
  __syncthreads();
  const double alpha = s_alpha;
  T* X = a.x + (size_t)p * nz; T* XI = a.xi + (size_t)p * mg; T* YF = a.yf + (size_t)p * mf; T* YG = a.yg + (size_t)p * mg;
  const T* oyf = a.oyf + (size_t)p * mf; const T* oyg = a.oyg + (size_t)p * mg;
  for (int e = threadIdx.x; e < nz; e += blockDim.x) { const double o = (double)ox[e]; X[e] = (T)(o + alpha * ((double)X[e] - o)); }
  for (int e = threadIdx.x; e < mg; e += blockDim.x) {
    const double o = (double)oxi[e]; XI[e] = (T)(o + alpha * ((double)XI[e] - o));
    const double y = (double)oyg[e]; YG[e] = (T)(y + alpha * ((double)YG[e] - y));
  }
  for (int e = threadIdx.x; e < mf; e += blockDim.x) { const double y = (double)oyf[e]; YF[e] = (T)(y + alpha * ((double)YF[e] - y)); }
}

// eq. 18 at the iterate (x, xi, y) with the blocks linearised THERE (so C x - c = f(x) exactly, eq. 37): one CTA of 128 threads per problem
template <typename T>
__global__ void __launch_bounds__(128) sqp_kkt_kernel(SqpArgs<T> a) {
  __shared__ double red[3][4];
  const Dims& d = a.d;
  const int p = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  if (!a.act_rw[p]) return;
  const int n = d.n, nx = d.nx, ng = d.ng;
  const int N = d.N, nz = d.nz, mg = d.mg, mf = d.mf, nn = n * n;
  const T* x = a.x + (size_t)p * nz; const T* xi = a.xi + (size_t)p * mg; const T* yf = a.yf + (size_t)p * mf; const T* yg = a.yg + (size_t)p * mg;
  const T* Dp = a.qp.D + a.qp.sD * p; const T* Ep = a.qp.E + a.qp.sE * p; const T* q = a.qp.q + (size_t)p * nz;
  const T* Am = a.qp.Am + (size_t)p * N * nx * n; const T* Ap = a.qp.Ap + (size_t)p * N * nx * n; const T* bb = a.qp.b + (size_t)p * N * nx;
  const T* G = d.g_sel ? nullptr : a.qp.G + a.qp.sG * p; const T* lo = a.qp.lo + (size_t)p * mg; const T* hi = a.qp.hi + (size_t)p * mg;
  double stat = 0, finf = 0, ginf = 0;
  for (int e = tid; e < nz; e += nt) {
    const int t = e / n, i = e - t * n;
    double g = (double)q[e];
    for (int j = 0; j < n; ++j) g += (double)Dp[(size_t)t * nn + i * n + j] * (double)x[t * n + j];
    if (t > 0) for (int j = 0; j < n; ++j) g += (double)Ep[(size_t)(t - 1) * nn + i * n + j] * (double)x[(t - 1) * n + j];
    if (t < N) for (int j = 0; j < n; ++j) g += (double)Ep[(size_t)t * nn + j * n + i] * (double)x[(t + 1) * n + j];
    if (t == 0 && i < nx) g += (double)yf[i];
    if (t < N) for (int k = 0; k < nx; ++k) g += (double)Am[((size_t)t * nx + k) * n + i] * (double)yf[nx + t * nx + k];
    if (t > 0) for (int k = 0; k < nx; ++k) g += (double)Ap[((size_t)(t - 1) * nx + k) * n + i] * (double)yf[nx + (t - 1) * nx + k];
    if (d.g_sel) { for (int r = 0; r < ng; ++r) if (d.g_col[r] == i) g += (double)yg[t * ng + r]; }
    else for (int r = 0; r < ng; ++r) g += (double)G[((size_t)t * ng + r) * n + i] * (double)yg[t * ng + r];
    stat = fmax(stat, fabs(g));
  }
  for (int e = tid; e < mf; e += nt) {
    double r;
    if (e < nx) r = (double)x[e] - (double)a.qp.x_init[(size_t)p * nx + e];
    else {
      const int t = (e - nx) / nx, k = (e - nx) - t * nx;
      r = -(double)bb[e - nx];
      for (int j = 0; j < n; ++j) r += (double)Am[((size_t)t * nx + k) * n + j] * (double)x[t * n + j] + (double)Ap[((size_t)t * nx + k) * n + j] * (double)x[(t + 1) * n + j];
    }
    finf = fmax(finf, fabs(r));
  }
  for (int e = tid; e < mg; e += nt) {
    const int t = e / ng, r = e - t * ng;
    double g = ((d.soft_mask >> r) & 1u) ? (double)xi[e] : 0.0;
    if (d.g_sel) g += (double)x[t * n + d.g_col[r]];
    else for (int j = 0; j < n; ++j) g += (double)G[(size_t)e * n + j] * (double)x[t * n + j];
    ginf = fmax(ginf, fmax(0.0, g - (double)hi[e]) + fmax(0.0, (double)lo[e] - g));
  }
  stat = warp_max(stat); finf = warp_max(finf); ginf = warp_max(ginf);
  if ((tid & 31) == 0) { red[0][tid >> 5] = stat; red[1][tid >> 5] = finf; red[2][tid >> 5] = ginf; }
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < (nt >> 5); ++w) { stat = fmax(stat, red[0][w]); finf = fmax(finf, red[1][w]); ginf = fmax(ginf, red[2][w]); }
    if (a.kkt) { a.kkt[(size_t)p * 3] = (T)stat; a.kkt[(size_t)p * 3 + 1] = (T)finf; a.kkt[(size_t)p * 3 + 2] = (T)ginf; }
    a.iters[p] = a.it;
    if (stat <= a.eps_c && finf <= a.eps_c && ginf <= a.eps_c) { a.act_rw[p] = 0; a.converged[p] = 1; }
    else atomicAdd(a.n_active, 1);
  }
}

}  // namespace tmpc
