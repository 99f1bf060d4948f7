// probe.cuh -- peak probes used by bench.py (FP64 DFMA rate, HBM streaming read)
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
#pragma once
#include "common.cuh"

namespace {

// ------------------------------------------------------------------ probes
__global__ void __launch_bounds__(256) fp64_probe_kernel(double* out, int iters, double seed) {
  double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999, c = 1e-9;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) out[0] = s;     // never true; keeps the chain alive
}
// The same with three FRESH vector-register operands per DFMA (no constant, uniform or reused operand): on B200 this
// issues every 3 cycles per SM sub-partition instead of 2 (register-file read bandwidth), i.e. 2/3 of the nominal peak.
__global__ void __launch_bounds__(256) fp64_probe3_kernel(double* out, int iters, const double* in) {
  double a[6], y[6], z[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) { a[i] = in[threadIdx.x + i]; y[i] = in[threadIdx.x + 8 + i]; z[i] = in[threadIdx.x + 16 + i]; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 6; ++i) a[i] = fma(a[i], y[i], z[i]);
  }
  double s = a[0] + a[1] + a[2] + a[3] + a[4] + a[5];
  if (s == 123.456) out[0] = s;
}
__global__ void __launch_bounds__(256) hbm_probe_kernel(const double2* in, int64_t n, double* out) {
  double acc = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double2 v = __ldcs(in + i);
    acc += v.x + v.y;
  }
  if (acc == 123.456) out[0] = acc;
}


}  // namespace
