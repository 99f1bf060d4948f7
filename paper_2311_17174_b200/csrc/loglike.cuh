// loglike.cuh -- stage (d): streaming reduction of Eq. 8 + fixed-order final sum, and the
// pack / unpack kernels of the two-channels-in-one-complex-transform layout.
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
//
// Layout: the synthesis writes z[i] = h_I[i] + i h_II[i] (one complex128 per sample), stage
// (c) is ONE complex transform Z = DFT(z) per walker, and since h_I, h_II are real
//     H_I[m]  = (Z[m] + conj Z[N-m]) / 2,      H_II[m] = (Z[m] - conj Z[N-m]) / (2i),     m = 0..N/2
// (indices mod N).  The reduction reads Z[m] and Z[N-m] together, so every element of Z is read exactly once and
// the real-to-complex pre/post passes of a D2Z transform are never run.
#pragma once
#include "common.cuh"

namespace {

constexpr int LL_THREADS = 256;
constexpr int LL_WARPS = LL_THREADS / 32;
constexpr int LL_GROUP = 8;          // walkers per CTA (one accumulator each per thread)
constexpr int LL_RANGE = 8192;       // bins per CTA

DEVINL void split_channels(const double2 zm, const double2 zn, double2& HI, double2& HII) {
  HI = make_double2(0.5 * (zm.x + zn.x), 0.5 * (zm.y - zn.y));
  HII = make_double2(0.5 * (zm.y + zn.y), 0.5 * (zn.x - zm.x));
}

struct LikeArgs {
  const double2* Z;        // [K][N] complex, transform of h_I + i h_II
  const double2* D;        // [2][Nf] data spectrum, channel I then II
  const double* w;         // [Nf] 1/S_n or 0
  double* partial;         // [K_total][n_part], this chunk starts at row k0
  int k0, K;
  int64_t N, Nf;
  int n_part;              // partial sums per walker = number of bin ranges
  const double* fcoef;     // [K_total][6] {a1,a2,a3,b1,b2,b3} of Eq. 7's power series (kFdep only), row k0 + walker
  double x_per_bin;        // (1/(N dt)) / f_*
  double f_per_bin;        // 1/(N dt)
};

// grid (bin ranges, walker groups).  Each thread owns bins m = range_begin + tid + 256 j and LL_GROUP walkers:
// the 2 LL_GROUP loads of Z are issued together (memory-level parallelism), D and w come from L2.
//
// kFdep: frequency-dependent propagation (Eq. 7; reading D11): every walker's spectrum is multiplied
// per bin by G = exp(-Dm(f)) exp(-2 pi i f tau(f)), Dm = sum a_n x^n, tau = sum b_n x^n, x = f/f_*, n = 1..3, before
// the residual is taken -- "such frequency-dependent terms need to act upon a tabulated waveform in frequency space".
template <bool kFdep>
__global__ void __launch_bounds__(LL_THREADS) loglike_kernel(LikeArgs a) {
  __shared__ double s_fc[LL_GROUP][6];
  if (kFdep) {
    if (threadIdx.x < LL_GROUP * 6) {
      const int g = threadIdx.x / 6, c = threadIdx.x - 6 * g;
      const int kk = min((int)blockIdx.y * LL_GROUP + g, a.K - 1);
      s_fc[g][c] = a.fcoef[(size_t)(a.k0 + kk) * 6 + c];
    }
    __syncthreads();
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int kg0 = blockIdx.y * LL_GROUP;
  const int64_t m_begin = (int64_t)blockIdx.x * LL_RANGE;
  const int64_t m_end = min(a.Nf, m_begin + (int64_t)LL_RANGE);
  const double2* zrow[LL_GROUP];
  double acc[LL_GROUP];
#pragma unroll
  for (int g = 0; g < LL_GROUP; ++g) {
    const int kk = min(kg0 + g, a.K - 1);
    zrow[g] = a.Z + (size_t)kk * a.N;
    acc[g] = 0.0;
  }
  for (int64_t m = m_begin + threadIdx.x; m < m_end; m += LL_THREADS) {
    const int64_t mn = (m == 0) ? 0 : a.N - m;
    double2 zm[LL_GROUP], zn[LL_GROUP];
#pragma unroll
    for (int g = 0; g < LL_GROUP; ++g) { zm[g] = __ldcs(zrow[g] + m); zn[g] = __ldcs(zrow[g] + mn); }
    const double2 dI = __ldg(a.D + m), dII = __ldg(a.D + a.Nf + m);
    const double wt = __ldg(a.w + m);
#pragma unroll
    for (int g = 0; g < LL_GROUP; ++g) {
      double2 HI, HII;
      split_channels(zm[g], zn[g], HI, HII);
      if (kFdep) {
        const double x = (double)m * a.x_per_bin, f = (double)m * a.f_per_bin;
        const double Dm = x * fma(x, fma(x, s_fc[g][2], s_fc[g][1]), s_fc[g][0]);
        const double tau = x * fma(x, fma(x, s_fc[g][5], s_fc[g][4]), s_fc[g][3]);
        const double amp = exp(-Dm);
        double sn, cs;
        sincospi(-2.0 * (f * tau), &sn, &cs);
        const double gr = amp * cs, gi = amp * sn;
        HI = make_double2(fma(gr, HI.x, -gi * HI.y), fma(gr, HI.y, gi * HI.x));
        HII = make_double2(fma(gr, HII.x, -gi * HII.y), fma(gr, HII.y, gi * HII.x));
      }
      const double ar = dI.x - HI.x, ai = dI.y - HI.y, br = dII.x - HII.x, bi = dII.y - HII.y;
      const double pw = fma(ar, ar, ai * ai) + fma(br, br, bi * bi);
      acc[g] = fma(wt, pw, acc[g]);
    }
  }
  __shared__ double s_acc[LL_WARPS][LL_GROUP];
#pragma unroll
  for (int g = 0; g < LL_GROUP; ++g) {
    double v = acc[g];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) s_acc[warp][g] = v;
  }
  __syncthreads();
  if (threadIdx.x < LL_GROUP && kg0 + (int)threadIdx.x < a.K) {
    double v = 0.0;
#pragma unroll
    for (int wq = 0; wq < LL_WARPS; ++wq) v += s_acc[wq][threadIdx.x];
    a.partial[(size_t)(a.k0 + kg0 + threadIdx.x) * a.n_part + blockIdx.x] = v;
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

// Z[K][N] -> spectra[K][2][Nf] (emri_waveform_fft, emri_data_fft: off the hot path)
__global__ void __launch_bounds__(256) unpack_spectrum_kernel(const double2* Z, double2* out, int K, int64_t N, int64_t Nf) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)K * Nf) return;
  const int k = (int)(idx / Nf);
  const int64_t m = idx - (int64_t)k * Nf;
  const double2* z = Z + (size_t)k * N;
  double2 HI, HII;
  split_channels(z[m], z[m == 0 ? 0 : N - m], HI, HII);
  out[((size_t)k * 2) * Nf + m] = HI;
  out[((size_t)k * 2 + 1) * Nf + m] = HII;
}

// two real series -> one complex series z = a + i b
__global__ void __launch_bounds__(256) pack_complex_kernel(const double* a, const double* b, double2* z, int64_t N) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < N) z[i] = make_double2(a[i], b[i]);
}

}  // namespace
