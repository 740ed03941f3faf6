// FP64 peak calibration: MEASURED_PEAKS.json has HBM and bf16 only, so the denominator of the
// FP64 roofline is measured on the device the library runs on: register-resident loops of independent DMMA.8x8x4
// (mma.sync m8n8k4 f64) and of plain DFMA, no memory traffic.
#pragma once
#include "common.cuh"

namespace ctqmc {

__global__ void __launch_bounds__(256) peak_dmma_kernel(int iters, double* sink) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = 0.0;
  const double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) dmma884(c[2 * i], c[2 * i + 1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) peak_dfma_kernel(int iters, double* sink) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) c[i] = threadIdx.x * 1e-3 + i;
  const double a = 1.0 + 1e-9, b = 1e-12;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = fma(c[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += c[i];
  if (s == 123.456) sink[0] = s;
}

}  // namespace ctqmc
