// loglike.cuh -- stage (d): streaming reduction of Eq. 8 + fixed-order final sum
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
#pragma once
#include "common.cuh"

namespace {

// ------------------------------------------------------------------ (d) likelihood reduction
struct LikeArgs {
  const double2* H;        // [2*K][Nf] complex (row pitch Nf)
  const double2* D;        // [2][Nf]
  const double* w;         // [Nf] 1/S_n or 0
  double* partial;         // [K_total][n_part], this chunk starts at row k0
  int k0, K;
  int64_t Nf;
  int n_part;              // partial sums per walker = tiles * LL_WARPS
};

__global__ void __launch_bounds__(LL_THREADS) loglike_kernel(LikeArgs a) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t base = (int64_t)blockIdx.x * LL_TILE + threadIdx.x;
  double2 dI[LL_BINS_PER_THREAD], dII[LL_BINS_PER_THREAD];
  double wt[LL_BINS_PER_THREAD];
#pragma unroll
  for (int b = 0; b < LL_BINS_PER_THREAD; ++b) {
    const int64_t m = base + (int64_t)b * LL_THREADS;
    const bool in = m < a.Nf;
    dI[b] = in ? __ldg(a.D + m) : make_double2(0.0, 0.0);
    dII[b] = in ? __ldg(a.D + a.Nf + m) : make_double2(0.0, 0.0);
    wt[b] = in ? __ldg(a.w + m) : 0.0;
  }
  for (int kl = 0; kl < a.K; ++kl) {
    const double2* HI = a.H + (size_t)(2 * kl) * a.Nf;
    const double2* HII = HI + a.Nf;
    double2 hI[LL_BINS_PER_THREAD], hII[LL_BINS_PER_THREAD];
#pragma unroll
    for (int b = 0; b < LL_BINS_PER_THREAD; ++b) {
      const int64_t m = base + (int64_t)b * LL_THREADS;
      const bool in = m < a.Nf;
      hI[b] = in ? __ldcs(HI + m) : make_double2(0.0, 0.0);
      hII[b] = in ? __ldcs(HII + m) : make_double2(0.0, 0.0);
    }
    double acc = 0.0;
#pragma unroll
    for (int b = 0; b < LL_BINS_PER_THREAD; ++b) {
      const double ar = dI[b].x - hI[b].x, ai = dI[b].y - hI[b].y;
      const double br = dII[b].x - hII[b].x, bi = dII[b].y - hII[b].y;
      const double pw = fma(ar, ar, ai * ai) + fma(br, br, bi * bi);
      acc = fma(wt[b], pw, acc);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane == 0) a.partial[(size_t)(a.k0 + kl) * a.n_part + (size_t)blockIdx.x * LL_WARPS + warp] = acc;
  }
}

// fixed-order final sum: one warp per walker, lane-strided partial sums then a shuffle tree
__global__ void loglike_final_kernel(const double* partial, int n_part, int K, double scale, const int32_t* status,
                                     double* logL, int32_t* status_out) {
  const int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (k >= K) return;
  const double* p = partial + (size_t)k * n_part;
  double acc = 0.0;
  for (int i = lane; i < n_part; i += 32) acc += p[i];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if (lane == 0) {
    const int32_t st = status[k];
    logL[k] = (st & (EMRI_ST_BADPARAM | EMRI_ST_DELAY | EMRI_ST_STATE)) ? -INFINITY : -scale * acc;
    if (status_out) status_out[k] = st;
  }
}

__global__ void copy_status_kernel(const int32_t* in, int32_t* out, int K) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < K) out[k] = in[k];
}

}  // namespace
