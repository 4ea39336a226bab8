// xc_peak.cu -- FP64 pipe microbenchmarks behind xc_measure_fp64_peak (include/xc_b200.h).
//
// MEASURED_PEAKS.json holds HBM and bf16 peaks only; the roofline of the batch kernel's contractions
// needs the FP64 rate of this very GPU.  Two register-resident kernels with no memory traffic:
//   kind 0: DFMA    -- 8 independent fma chains per thread
//   kind 1: DMMA    -- 8 independent mma.sync.m8n8k4.f64 accumulator pairs per warp (DMMA.8x8x4 SASS)
// Timed with CUDA events on the caller's stream; the best of `reps` launches is returned.
#include <cuda_runtime.h>

#include <algorithm>

#include "../../include/xc_b200.h"

namespace {

__global__ void __launch_bounds__(256) k_peak_dfma(int iters, double seed, double* out) {
  double a[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) a[k] = seed * (threadIdx.x + k + 1);
  const double m = 1.0 - 1e-9 * seed, c = 1e-9 * seed;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = fma(a[k], m, c);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += a[k];
  if (s == 123.456) out[0] = s;   // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) k_peak_dmma(int iters, double seed, double* out) {
  double c0[8], c1[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { c0[k] = 0.0; c1[k] = 0.0; }
  const double a = seed * 1e-3 * (threadIdx.x & 31), b = seed * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c0[k]), "+d"(c1[k])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += c0[k] + c1[k];
  if (s == 123.456) out[0] = s;
}

}  // namespace

extern "C" int xc_measure_fp64_peak(int32_t kind, int32_t device, int32_t reps, double* tflops, double* sm_clock_mhz_est) {
  if (!tflops || kind < 0 || kind > 1 || reps < 1) return XC_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return XC_ECUDA;
  if (cudaSetDevice(device) != cudaSuccess) return XC_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return XC_ECUDA;
  double* d = nullptr;
  if (cudaMalloc((void**)&d, 8) != cudaSuccess) return XC_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 1 << 15, threads = 256, blocks = prop.multiProcessorCount * 8;
  // flops per launch
  const double flops = kind == 0 ? 2.0 * 8 * (double)iters * threads * blocks
                                 : 512.0 * 8 * (double)iters * (threads / 32) * blocks;
  float best = 1e30f;
  for (int r = 0; r < reps + 1; ++r) {   // first launch = warm-up
    cudaEventRecord(e0, 0);
    if (kind == 0) k_peak_dfma<<<blocks, threads>>>(iters, 1.0 + r, d);
    else k_peak_dmma<<<blocks, threads>>>(iters, 1.0 + r, d);
    cudaEventRecord(e1, 0);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return XC_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0) best = std::min(best, ms);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d);
  *tflops = flops / (best * 1e-3) * 1e-12;
  // clock implied by the nominal 64 FP64 FMA / clk / SM of the datasheet (diagnostic only)
  if (sm_clock_mhz_est) *sm_clock_mhz_est = *tflops * 1e12 / (2.0 * 64.0 * prop.multiProcessorCount) * 1e-6;
  return cudaGetLastError() == cudaSuccess ? XC_OK : XC_ECUDA;
}
