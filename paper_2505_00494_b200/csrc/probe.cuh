// FP64 issue-rate probes: the roofline denominators of DESIGN.md section 6.
// Register-resident chains, no memory traffic: what the FP64 pipes can sustain
// at the clocks the board actually runs at.
#pragma once
#include <cuda_runtime.h>

namespace qk {

__global__ void probe_dfma_kernel(double* out, int iters, double s) {
  double acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = threadIdx.x * 0.001 + i;
  double x = s, y = 1.0 - s * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = fma(acc[i], y, x);
  }
  double t = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) t += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = t;
}

__global__ void probe_dmma_kernel(double* out, int iters, double s) {
  double c[8][2];
#pragma unroll
  for (int i = 0; i < 8; i++) { c[i][0] = i; c[i][1] = threadIdx.x; }
  double a = s, b = 1.0 + s;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double t = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) t += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = t;
}

}  // namespace qk
