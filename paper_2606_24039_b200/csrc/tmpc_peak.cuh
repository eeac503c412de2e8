// tmpc_peak.cuh — micro-benchmarks that MEASURE the roofline denominators bench.py reports against (SURVEY.md 8(d):
// "FP32/FP64 FMA peaks are not in MEASURED_PEAKS.json and must be measured by the builder"): dependent-chain-free FMA
// loops for the plain FP32 (FFMA and packed FFMA2) and FP64 (DFMA) pipes and a conflict-free LDS.128 loop for the
// shared-memory bandwidth that bounds the stage-parallel phases of the resident class.
// Diagnostic entry point: tmpc_measure_peak (include/tmpc.h).  Not on the hot path.
#pragma once
#include "tmpc_common.cuh"

namespace tmpc {

constexpr int PEAK_ITERS = 2048;     // loop trips per thread
constexpr int PEAK_ACC = 12;         // independent accumulators per thread (covers the 4-cycle FMA latency with 2+ warps per scheduler)

// what = 0: FFMA2 (two fp32 FMAs per instruction), 1: FFMA, 2: DFMA.  Every thread keeps PEAK_ACC independent chains.
template <int WHAT>
__global__ void __launch_bounds__(512) fma_peak_kernel(float seed, float* sink) {
  if constexpr (WHAT == 0) {
    float2 acc[PEAK_ACC];
#pragma unroll
    for (int k = 0; k < PEAK_ACC; ++k) acc[k] = make_float2(seed + k, seed - k);
    const float2 m = make_float2(1.f + seed * 1e-7f, 1.f - seed * 1e-7f), c = make_float2(seed * 1e-7f, -seed * 1e-7f);   // run-time operands: the 3-register form
#pragma unroll 1
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
      for (int k = 0; k < PEAK_ACC; ++k) acc[k] = __ffma2_rn(acc[k], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PEAK_ACC; ++k) s += acc[k].x + acc[k].y;
    if (s == 12345.678f) sink[0] = s;
  } else if constexpr (WHAT == 1) {
    float acc[2 * PEAK_ACC];
#pragma unroll
    for (int k = 0; k < 2 * PEAK_ACC; ++k) acc[k] = seed + k;
    const float m = 1.f + seed * 1e-7f, c = seed * 1e-7f;
#pragma unroll 1
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
      for (int k = 0; k < 2 * PEAK_ACC; ++k) acc[k] = fmaf(acc[k], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 2 * PEAK_ACC; ++k) s += acc[k];
    if (s == 12345.678f) sink[0] = s;
  } else {
    double acc[PEAK_ACC];
#pragma unroll
    for (int k = 0; k < PEAK_ACC; ++k) acc[k] = (double)seed + k;
    const double m = 1.0 + (double)seed * 1e-7, c = (double)seed * 1e-7;
#pragma unroll 1
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
      for (int k = 0; k < PEAK_ACC; ++k) acc[k] = fma(acc[k], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PEAK_ACC; ++k) s += acc[k];
    if (s == 12345.678) sink[0] = (float)s;
  }
}
// flops one thread of fma_peak_kernel executes
__host__ __device__ constexpr double fma_peak_flops_per_thread(int what) {
  return what == 0 ? 2.0 * 2 * PEAK_ACC * PEAK_ITERS : what == 1 ? 2.0 * 2 * PEAK_ACC * PEAK_ITERS : 2.0 * PEAK_ACC * PEAK_ITERS;
}

// Conflict-free 16-byte shared-memory loads: lane l reads the float4 at (l + 32 j) mod 2048, 8 loads in flight per trip.
constexpr int LDS_ITERS = 1024, LDS_UNROLL = 8;
__global__ void __launch_bounds__(512) lds_peak_kernel(float* sink) {
  __shared__ float4 buf[2048];
  for (int e = threadIdx.x; e < 2048; e += blockDim.x) buf[e] = make_float4((float)e, 1.f, 2.f, 3.f);
  __syncthreads();
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  unsigned idx = threadIdx.x;
#pragma unroll 1
  for (int it = 0; it < LDS_ITERS; ++it) {
#pragma unroll
    for (int j = 0; j < LDS_UNROLL; ++j) {
      const float4 v = buf[(idx + 32u * j) & 2047u];
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    idx += 32u * LDS_UNROLL;
  }
  if (acc.x + acc.y + acc.z + acc.w == 12345.678f) sink[0] = acc.x;
}

// Runs `what` (0 FFMA2, 1 FFMA, 2 DFMA: result in TFLOP/s; 3 LDS.128: result in GB/s) `reps` times on `stream`, timed with CUDA events
// (best repetition after one warm-up), at the clocks found.
inline tmpc_status measure_peak(int what, float* scratch, cudaStream_t stream, int reps, double* out) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return TMPC_E_CUDA;
  const int nt = 512, grid = sms * 4 * 8;              // 4 resident CTAs of 512 threads per SM, 8 waves
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return TMPC_E_CUDA;
  double best = 0.0;
  for (int r = 0; r <= reps; ++r) {
    cudaEventRecord(e0, stream);
    if (what == 0) fma_peak_kernel<0><<<grid, nt, 0, stream>>>(1.0f, scratch);
    else if (what == 1) fma_peak_kernel<1><<<grid, nt, 0, stream>>>(1.0f, scratch);
    else if (what == 2) fma_peak_kernel<2><<<grid, nt, 0, stream>>>(1.0f, scratch);
    else lds_peak_kernel<<<grid, nt, 0, stream>>>(scratch);
    cudaEventRecord(e1, stream);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); cudaGetLastError(); return TMPC_E_CUDA; }
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    if (r == 0 || ms <= 0.f) continue;               // warm-up
    const double units = what == 3 ? 16.0 * LDS_ITERS * LDS_UNROLL * (double)nt * grid / 1e9       // GB
                                   : fma_peak_flops_per_thread(what) * (double)nt * grid / 1e12;    // TFLOP
    const double rate = units / (ms * 1e-3);
    if (rate > best) best = rate;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *out = best;
  return best > 0.0 ? TMPC_OK : TMPC_E_CUDA;
}

}  // namespace tmpc
