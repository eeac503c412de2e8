// tmpc_common.cuh — shared argument structs and small device helpers of the CUDA path.
// Product code: shares nothing with oracle/ (the CPU oracle is test infrastructure).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/tmpc.h"

namespace tmpc {

// Problem data as the kernels see it (device pointers in the working dtype T; strides in elements).
template <typename T>
struct QpView {
  const T* D; int64_t sD;      // [B|1][T][n][n]
  const T* E; int64_t sE;      // [B|1][N][n][n]
  const T* q;                  // [B][T][n]
  const T* Am; const T* Ap;    // [B][N][nx][n]
  const T* b;                  // [B][N][nx]
  const T* x_init;             // [B][nx]
  const T* G; int64_t sG;      // [B|1][T][ng][n] or null (selection)
  const T* lo; const T* hi;    // [B][T][ng]
};

struct Dims {
  int B, N, T, nx, nu, n, ng, nz, mf, mg;
  int g_sel;
  int g_col[TMPC_MAX_NG];
  unsigned soft_mask;          // bit r = row r is soft
};

template <typename T>
struct Params {                // scalars of Alg. 3 in the working dtype
  T sigma, rho_f, rho_g, alpha, gamma, lam;
};

__device__ __forceinline__ float tmin(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double tmin(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float tmax(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double tmax(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float tabs(float a) { return fabsf(a); }
__device__ __forceinline__ double tabs(double a) { return fabs(a); }

// eq. 13 (hard rows) and eq. 15a/15b generalised with the L1 weight lambda (soft rows; lambda = 0 is eq. 15):
//   s+ = max(0, (rho (v - hi) - lam)/(rho + gamma)),  s- = max(0, (rho (lo - v) - lam)/(rho + gamma)),
//   z = clip(v, lo, hi) + s+ - s-,  xi = s- - s+.
template <typename T>
__device__ __forceinline__ void project_row(bool soft, T v, T lo, T hi, T rho, T inv_rho_gamma, T lam, T& z, T& xi) {
  T c = tmin(tmax(v, lo), hi);
  if (!soft) { z = c; xi = T(0); return; }
  T sp = tmax(T(0), (rho * (v - hi) - lam) * inv_rho_gamma);
  T sm = tmax(T(0), (rho * (lo - v) - lam) * inv_rho_gamma);
  z = c + sp - sm; xi = sm - sp;
}

// block-wide max reduction through shared memory (scratch: >= 32 elements); result valid in every thread.
template <typename T>
__device__ T block_max(T v, T* scratch) {
  for (int o = 16; o > 0; o >>= 1) v = tmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (l == 0) scratch[w] = v;
  __syncthreads();
  T r = scratch[0];
  for (int k = 1; k < nw; ++k) r = tmax(r, scratch[k]);
  return r;
}
template <typename T>
__device__ T block_sum(T v, T* scratch) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (l == 0) scratch[w] = v;
  __syncthreads();
  T r = scratch[0];
  for (int k = 1; k < nw; ++k) r += scratch[k];   // fixed order: deterministic
  return r;
}

}  // namespace tmpc
