// tmpc_misc.cuh — a1 (linearise, eq. 36-38) and a10 (backward: classification, adjoint data, KKT refinement).
#pragma once
#include "tmpc_common.cuh"
#include "tmpc_admm.cuh"

namespace tmpc {

__device__ __forceinline__ void tsincos(float a, float* s, float* c) { sincosf(a, s, c); }
__device__ __forceinline__ void tsincos(double a, double* s, double* c) { sincos(a, s, c); }
__device__ __forceinline__ float ttan(float a) { return tanf(a); }
__device__ __forceinline__ double ttan(double a) { return tan(a); }

// ---------------------------------------------------------------------------------------------------------------
// a1.  Kinematic bicycle, implicit midpoint (reading A-24):  v = (px, py, psi, vel, a, delta),
//   f_k = x_k + dt F((x_k + x_{k+1})/2, u_k) - x_{k+1},  F = (vel cos psi, vel sin psi, vel/L tan delta, a).
//   A^-_k = [I + dt/2 F_x , dt F_u],  A^+_k = [-I + dt/2 F_x , 0],  b_k = A^- v_k + A^+ v_{k+1} - f_k   (eq. 36-37).
//   g_t = (a, delta, e_lat),  e_lat = -sin(psi_ref)(px - px_ref) + cos(psi_ref)(py - py_ref): linear, so G_t is constant
//   and the shifted bounds (eq. 38) are g_lo + G_t . p_ref on the lateral row.
// One thread per (problem, stage).
template <typename T>
struct LinArgs {
  int B, N; T Lwb, dt; const T* xbar; const T* ref; T glo[3], ghi[3];
  T* Am; T* Ap; T* b; T* G; T* lo; T* hi;
};

// contiguous run of CNT elements in 16-byte stores (dst 16-byte aligned, CNT a multiple of 16 / sizeof(T)) or 8-byte stores for floats
template <int CNT> __device__ __forceinline__ void store_run16(float* dst, const float* v) {
#pragma unroll
  for (int c = 0; c < CNT / 4; ++c) reinterpret_cast<float4*>(dst)[c] = make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
}
template <int CNT> __device__ __forceinline__ void store_run16(double* dst, const double* v) {
#pragma unroll
  for (int c = 0; c < CNT / 2; ++c) reinterpret_cast<double2*>(dst)[c] = make_double2(v[2 * c], v[2 * c + 1]);
}
template <int CNT> __device__ __forceinline__ void store_run8(float* dst, const float* v) {      // 8-byte aligned run of floats
#pragma unroll
  for (int c = 0; c < CNT / 2; ++c) reinterpret_cast<float2*>(dst)[c] = make_float2(v[2 * c], v[2 * c + 1]);
}
template <int CNT> __device__ __forceinline__ void store_run8(double* dst, const double* v) {
#pragma unroll
  for (int c = 0; c < CNT; ++c) dst[c] = v[c];
}

template <typename T>
__global__ void bicycle_linearize_kernel(LinArgs<T> a) {
  const int T_ = a.N + 1, n = 6, nx = 4;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)a.B * T_) return;
  const int p = (int)(gid / T_), t = (int)(gid - (long long)p * T_);
  const T* r = a.ref + ((size_t)p * T_ + t) * n;
  T* g = a.G + ((size_t)p * T_ + t) * 3 * n;
  T sr, cr; tsincos(r[2], &sr, &cr);
  {                                                      // the three G rows of a stage are 72 / 144 contiguous bytes: vector stores
    T gv[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) gv[k] = T(0);
    gv[4] = T(1); gv[n + 5] = T(1); gv[2 * n] = -sr; gv[2 * n + 1] = cr;
    store_run8<18>(g, gv);
  }
  const T off = -sr * r[0] + cr * r[1];
  T* lo = a.lo + ((size_t)p * T_ + t) * 3; T* hi = a.hi + ((size_t)p * T_ + t) * 3;
  lo[0] = a.glo[0]; lo[1] = a.glo[1]; lo[2] = a.glo[2] + off;
  hi[0] = a.ghi[0]; hi[1] = a.ghi[1]; hi[2] = a.ghi[2] + off;
  if (t >= a.N) return;
  const T* vk = a.xbar + ((size_t)p * T_ + t) * n; const T* vk1 = vk + n;
  const T dt = a.dt, h = T(0.5) * dt;
  const T psi = T(0.5) * (vk[2] + vk1[2]), vel = T(0.5) * (vk[3] + vk1[3]), acc = vk[4], del = vk[5];
  T s, c; tsincos(psi, &s, &c);
  const T td = ttan(del), iL = T(1) / a.Lwb;
  // F_x columns psi (2) and vel (3) only; F_u: d(psi_dot)/d(delta) = vel / (L cos^2 delta) = vel (1 + tan^2) / L, d(v_dot)/da = 1
  const T Fx02 = -vel * s, Fx03 = c, Fx12 = vel * c, Fx13 = s, Fx23 = td * iL;
  const T Fu21 = vel * (T(1) + td * td) * iL;
  T am[4][6], ap[4][6];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 6; ++j) { am[i][j] = (i == j) ? T(1) : T(0); ap[i][j] = (i == j) ? T(-1) : T(0); }
  am[0][2] += h * Fx02; am[0][3] += h * Fx03; am[1][2] += h * Fx12; am[1][3] += h * Fx13; am[2][3] += h * Fx23;
  ap[0][2] += h * Fx02; ap[0][3] += h * Fx03; ap[1][2] += h * Fx12; ap[1][3] += h * Fx13; ap[2][3] += h * Fx23;
  am[2][5] = dt * Fu21; am[3][4] = dt;
  const T F[4] = {vel * c, vel * s, vel * iL * td, acc};
  T* Am = a.Am + ((size_t)p * a.N + t) * nx * n; T* Ap = a.Ap + ((size_t)p * a.N + t) * nx * n; T* b = a.b + ((size_t)p * a.N + t) * nx;
  T bv[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    T sb = -(vk[i] + dt * F[i] - vk1[i]);
#pragma unroll
    for (int j = 0; j < 6; ++j) sb += am[i][j] * vk[j] + ap[i][j] * vk1[j];
    bv[i] = sb;
  }
  store_run16<24>(Am, &am[0][0]); store_run16<24>(Ap, &ap[0][0]); store_run16<4>(b, bv);      // 96 / 192 and 16 / 32 contiguous bytes per block
}

}  // namespace tmpc
