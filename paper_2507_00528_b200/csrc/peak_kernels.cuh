// peak_kernels.cuh -- FP32 FMA microbenchmark: the measured denominator of the plain-ALU roofline.
// Every thread runs PEAK_CHAINS independent FMA chains (no memory traffic in the loop), all SMs, 2048 threads per SM:
// flops = threads x iterations x PEAK_CHAINS x 2.  The result is stored only under a condition that never holds, which
// keeps the arithmetic alive without a store in the timed loop.
#pragma once
#include <cuda_runtime.h>

#define PEAK_CHAINS 16
#define PEAK_UNROLL 8

__global__ void __launch_bounds__(256) k_ffma_peak(int iters, float a, float b, float *__restrict__ sink) {
  float x[PEAK_CHAINS];
#pragma unroll
  for (int c = 0; c < PEAK_CHAINS; ++c) x[c] = (float)(threadIdx.x + c) * 1e-3f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u)
#pragma unroll
      for (int c = 0; c < PEAK_CHAINS; ++c) x[c] = fmaf(x[c], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < PEAK_CHAINS; ++c) s += x[c];
  if (s == 123456.789f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
