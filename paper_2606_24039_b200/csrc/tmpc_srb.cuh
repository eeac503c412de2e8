// tmpc_srb.cuh — a1 for the second built-in model (f3): single-rigid-body humanoid dynamics (eq. 68-69) integrated with
// classical RK4, x = (p, Theta = (roll, pitch, yaw), v, omega) in R^12, u = (f_L, f_R) in R^6 (world-frame foot forces).
//   f_k(v_k, v_{k+1}) = Phi(x_k, u_k) - x_{k+1}:   A^-_k = [dPhi/dx dPhi/du],  A^+_k = [-I 0],  b_k = A^- v_k + A^+ v_{k+1} - f_k  (eq. 36-37).
// The Jacobian comes from forward-mode differentiation of the integrator itself: thread (problem, stage, j) pushes the seed e_j through the
// four RK4 stages with a (value, derivative) pair type and gets column j of A^-; thread j = 18 evaluates Phi and, after a CTA barrier, b.
// Readings (A-38): I = diag(mp[4..6]) (body frame), contact vectors r_i = foot_i - p with fixed world foot positions mp[7..12],
// the torque r x f enters eq. 68d as printed.  mp[0] = mass, mp[1..3] = g.
#pragma once
#include "tmpc_common.cuh"

namespace tmpc {

template <typename T> struct Fwd { T v, d; };            // value and one directional derivative
template <typename T> __device__ __forceinline__ Fwd<T> operator+(Fwd<T> a, Fwd<T> b) { return {a.v + b.v, a.d + b.d}; }
template <typename T> __device__ __forceinline__ Fwd<T> operator-(Fwd<T> a, Fwd<T> b) { return {a.v - b.v, a.d - b.d}; }
template <typename T> __device__ __forceinline__ Fwd<T> operator*(Fwd<T> a, Fwd<T> b) { return {a.v * b.v, a.d * b.v + a.v * b.d}; }
template <typename T> __device__ __forceinline__ Fwd<T> scale(T s, Fwd<T> a) { return {s * a.v, s * a.d}; }
template <typename T> __device__ __forceinline__ Fwd<T> recip(Fwd<T> a) { const T r = T(1) / a.v; return {r, -a.d * r * r}; }

template <typename T>
__device__ void srb_rhs(const T* __restrict__ mp, const Fwd<T>* x, const Fwd<T>* u, Fwd<T>* xd) {
  T sp, cp, st, ct;
  if constexpr (sizeof(T) == 8) { sincos(x[3].v, &sp, &cp); sincos(x[4].v, &st, &ct); } else { sincosf(x[3].v, &sp, &cp); sincosf(x[4].v, &st, &ct); }
  const Fwd<T> Sp{sp, cp * x[3].d}, Cp{cp, -sp * x[3].d}, St{st, ct * x[4].d}, Ct{ct, -st * x[4].d};
  const Fwd<T> iCt = recip(Ct), Tt = St * iCt;
#pragma unroll
  for (int i = 0; i < 3; ++i) xd[i] = x[6 + i];
  const Fwd<T> w0 = x[9], w1 = x[10], w2 = x[11];
  xd[3] = w0 + Sp * Tt * w1 + Cp * Tt * w2;              // eq. 69, row by row
  xd[4] = Cp * w1 - Sp * w2;
  xd[5] = Sp * iCt * w1 + Cp * iCt * w2;
  const T im = T(1) / mp[0];
#pragma unroll
  for (int i = 0; i < 3; ++i) { xd[6 + i] = scale(im, u[i] + u[3 + i]); xd[6 + i].v += mp[1 + i]; }
  Fwd<T> tau[3] = {{T(0), T(0)}, {T(0), T(0)}, {T(0), T(0)}};
#pragma unroll
  for (int f = 0; f < 2; ++f) {
    Fwd<T> r[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) r[i] = {mp[7 + 3 * f + i] - x[i].v, -x[i].d};
    const Fwd<T>* F = u + 3 * f;
    tau[0] = tau[0] + (r[1] * F[2] - r[2] * F[1]); tau[1] = tau[1] + (r[2] * F[0] - r[0] * F[2]); tau[2] = tau[2] + (r[0] * F[1] - r[1] * F[0]);
  }
  const Fwd<T> Iw0 = scale(mp[4], w0), Iw1 = scale(mp[5], w1), Iw2 = scale(mp[6], w2);
  xd[9] = scale(T(1) / mp[4], tau[0] - (w1 * Iw2 - w2 * Iw1));
  xd[10] = scale(T(1) / mp[5], tau[1] - (w2 * Iw0 - w0 * Iw2));
  xd[11] = scale(T(1) / mp[6], tau[2] - (w0 * Iw1 - w1 * Iw0));
}

template <typename T>
struct SrbArgs { int B, N; T dt; T mp[13]; const T* xbar; T* Am; T* Ap; T* b; };

// grid = B * N CTAs (one per dynamics block), block = 32 threads: lanes 0..17 = seed columns, lane 18 = the value Phi(v_k)
template <typename T>
__global__ void __launch_bounds__(32) srb_linearize_kernel(SrbArgs<T> a) {
  constexpr int n = 18, nx = 12;
  __shared__ T sA[nx * n], sPhi[nx];
  const long long blk = blockIdx.x;
  const int p = (int)(blk / a.N), t = (int)(blk - (long long)p * a.N), j = threadIdx.x;
  const T* vk = a.xbar + ((size_t)p * (a.N + 1) + t) * n; const T* vk1 = vk + n;
  if (j <= n) {
    Fwd<T> x[12], u[6], k1[12], k2[12], k3[12], k4[12], xt[12];
#pragma unroll
    for (int i = 0; i < 12; ++i) x[i] = {vk[i], i == j ? T(1) : T(0)};
#pragma unroll
    for (int i = 0; i < 6; ++i) u[i] = {vk[12 + i], 12 + i == j ? T(1) : T(0)};
    const T dt = a.dt;
    srb_rhs<T>(a.mp, x, u, k1);
#pragma unroll
    for (int i = 0; i < 12; ++i) xt[i] = x[i] + scale(T(0.5) * dt, k1[i]);
    srb_rhs<T>(a.mp, xt, u, k2);
#pragma unroll
    for (int i = 0; i < 12; ++i) xt[i] = x[i] + scale(T(0.5) * dt, k2[i]);
    srb_rhs<T>(a.mp, xt, u, k3);
#pragma unroll
    for (int i = 0; i < 12; ++i) xt[i] = x[i] + scale(dt, k3[i]);
    srb_rhs<T>(a.mp, xt, u, k4);
#pragma unroll
    for (int i = 0; i < 12; ++i) {
      const Fwd<T> o = x[i] + scale(dt / T(6), k1[i] + scale(T(2), k2[i]) + scale(T(2), k3[i]) + k4[i]);
      if (j < n) sA[i * n + j] = o.d; else sPhi[i] = o.v;
    }
  }
  __syncthreads();
  T* am = a.Am + ((size_t)p * a.N + t) * nx * n; T* ap = a.Ap + ((size_t)p * a.N + t) * nx * n;
  for (int e = threadIdx.x; e < nx * n; e += 32) { am[e] = sA[e]; ap[e] = (e / n == e % n) ? T(-1) : T(0); }
  if (threadIdx.x < nx) {                                // b_i = sum_j Am[i][j] v_k[j] - x_{k+1,i} - (Phi_i - x_{k+1,i})
    const int i = threadIdx.x;
    T s = -sPhi[i];
    for (int c = 0; c < n; ++c) s += sA[i * n + c] * vk[c];
    (void)vk1;
    a.b[((size_t)p * a.N + t) * nx + i] = s;
  }
}

}  // namespace tmpc
