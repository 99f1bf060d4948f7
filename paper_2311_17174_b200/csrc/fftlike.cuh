// fftlike.cuh -- stages (c)+(d) fused: the LAST pass of the transform and the reduction of Eq. 8
// in one kernel, so that the spectrum is never written back nor read again (PAPER.md:43,
// :134: waveform and FFT are one GPU stage).
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
//
// N = N1 N2 (powers of two; N1 = 1024 for N >= 2^20 -- the length cuFFT's strided kernel is fastest at, measured -- and
// N2 = N / N1 <= 4096).  With i = N2 i1 + i2 and m = m1 + N1 m2,
//     Z[m1 + N1 m2] = sum_{i2} W_N^{i2 m1} W_N2^{i2 m2}  [ sum_{i1} z[N2 i1 + i2] W_N1^{i1 m1} ].
//   pass A  the bracket: N2 strided transforms of length N1 per walker.  The synthesis writes the chunk walker-interleaved,
//           z[i1][k][i2], so ONE strided batched cuFFT plan (stride K_c N2, distance 1, batch K_c N2) does all walkers of a
//           chunk in place: Y[m1][k][i2].  (The one vendor call.)
//   pass B  this file: one row (m1, k) of N2 contiguous elements per group of N2/16 threads: load, multiply by the
//           twiddle W_N^{i2 m1}, N2-point transform (radix-16 stages in registers, padded shared-memory exchanges in
//           between, last stage radix N2/256 or 16), and the outputs Z[m1 + N1 m2] go straight from registers into Eq. 8.
//
// Eq. 8 without pairing.  With a = Z[m], b = conj Z[N-m] the two channels are H_I = (a+b)/2, H_II = (a-b)/(2i), and
//     |D_I - H_I|^2 + |D_II - H_II|^2 = |D_I|^2 + |D_II|^2 - 2 Re(a P + b Q) + (|a|^2 + |b|^2)/2,
//     P = (conj D_I - i conj D_II)/2,  Q = (conj D_I + i conj D_II)/2,
// which is a sum over single elements of Z: logL = -(2 dt/N) [ C_D + sum_j ( alpha_j |Z_j|^2 - 2 Re(Z_j gamma_j) ) ],
// alpha_j = w_m / 2, gamma_m = w_m P_m, gamma_{N-m} = w_m conj(Q_m) (the self-paired bins m = 0, N/2 carry both halves),
// C_D = sum_m w_m (|D_I|^2 + |D_II|^2).  like_weights_kernel builds alpha, gamma (in pass-B order) and C_D from the
// caller's data spectrum once per call; every partial sum has a fixed place and order (bitwise reproducible).
#pragma once
#include "common.cuh"

namespace {

constexpr int FB_THREADS = 256;           // threads per CTA of the pass-B kernel
constexpr int FB_EPT = 16;                // elements per thread
constexpr int FB_ELEMS = FB_THREADS * FB_EPT;   // elements per CTA pass = 4096: 4096 / N2 rows at once

DEVINL double2 cmul(const double2 a, const double2 b) {
  return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}

// (a - b) * W_16^Q with the trivial cases folded at compile time
template <int Q>
DEVINL double2 sub_twiddle16(const double2 a, const double2 b) {
  const double dx = a.x - b.x, dy = a.y - b.y;
  if (Q == 0) return make_double2(dx, dy);
  if (Q == 4) return make_double2(dy, -dx);                       // * (-i)
  if (Q == 2) return make_double2(0.70710678118654757274 * (dx + dy), 0.70710678118654757274 * (dy - dx));
  if (Q == 6) return make_double2(0.70710678118654757274 * (dy - dx), -0.70710678118654757274 * (dx + dy));
  constexpr double c = (Q == 1) ? 0.92387953251128673848 : (Q == 3) ? 0.38268343236508978178
                     : (Q == 5) ? -0.38268343236508978178 : -0.92387953251128673848;
  constexpr double s = (Q == 1) ? -0.38268343236508978178 : (Q == 3) ? -0.92387953251128673848
                     : (Q == 5) ? -0.92387953251128673848 : -0.38268343236508978178;
  return make_double2(fma(dx, c, -dy * s), fma(dx, s, dy * c));
}

// one decimation-in-frequency level on registers: blocks of 2 HALF, twiddle W_{2 HALF}^i = W_16^{i 8 / HALF}
template <int R, int HALF, int I = 0>
struct DifLevel {
  DEVINL static void run(double2* v) {
    if constexpr (I < R / 2) {
      constexpr int blk = I / HALF, i = I % HALF, lo = blk * 2 * HALF + i, hi = lo + HALF;
      const double2 a = v[lo], b = v[hi];
      v[lo] = make_double2(a.x + b.x, a.y + b.y);
      v[hi] = sub_twiddle16<(i * 8) / HALF>(a, b);
      DifLevel<R, HALF, I + 1>::run(v);
    }
  }
};
// forward DFT of R = 2, 4, 8, 16 points in registers; the result of index q is left at position bitrev_R(q)
template <int R>
DEVINL void fft_regs(double2* v) {
  if constexpr (R >= 16) DifLevel<R, 8>::run(v);
  if constexpr (R >= 8) DifLevel<R, 4>::run(v);
  if constexpr (R >= 4) DifLevel<R, 2>::run(v);
  DifLevel<R, 1>::run(v);
}
template <int R>
__host__ __device__ constexpr int bitrev(int q) {
  int r = 0;
  for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (q & 1); q >>= 1; }
  return r;
}

DEVINL int fb_pad(int a) { return a + (a >> 4); }      // one element of padding per 16: conflict-free exchanges

struct FftLikeArgs {
  const double2* Y;        // [N1][K][N2] after pass A
  const double2* twid;     // [256 + N2]: W_256^{k t} at [16 t + k] (second radix-16 stage), then W_N2^{jj t} at
                           // [t NSL + jj] (last stage) -- both transposed so that consecutive threads read consecutive entries
  const double2* twA;      // [N / 1024] W_N^{1024 q}: with twB the inter-pass twiddle W_N^q = twA[q >> 10] twB[q & 1023]
  const double2* twB;      // [1024] W_N^q
  const double* alpha;     // [N1][N2] alpha of element (m1, m2), pass-B order
  const double2* gamma;    // [N1][N2]
  double* partial;         // [K_total][n_part]; this chunk's walker kl at row k0 + kl, entry m1
  int k0, K, n_part;
  int N1;
  int64_t N;
};

// LOG2L = log2 N2 in {8 .. 12}.  CTA pass = FB_ELEMS / N2 consecutive rows of Y (same m1 for a chunk size that is a
// multiple of that; any chunk size works, the row's (m1, k) are recomputed per row).
template <int LOG2L>
__global__ void __launch_bounds__(FB_THREADS, 2) fft_like_kernel(FftLikeArgs a) {
  constexpr int L = 1 << LOG2L, T = L / FB_EPT;                 // threads per row
  constexpr int ROWS = FB_ELEMS / L;                            // rows per CTA pass
  constexpr int NFULL = (LOG2L - 1) / 4;                        // radix-16 stages that end in shared memory
  constexpr int RL = L >> (4 * NFULL);                          // radix of the last stage (16, 2, 4)
  constexpr int U = FB_EPT / RL;                                // last-stage transforms per thread
  constexpr int NSL = L / RL;                                   // their stride
  extern __shared__ __align__(16) unsigned char fb_smem[];
  double2* s_tw2 = reinterpret_cast<double2*>(fb_smem);                      // [16][16]
  double2* s_tw = s_tw2 + 256;                                               // [RL][NSL]
  double2* s_x = s_tw + L;                                                   // [ROWS][L + L/16]
  __shared__ double s_red[FB_THREADS / 32];
  const int tid = threadIdx.x, row_in = tid / T, j = tid % T;
  for (int q = tid; q < 256 + L; q += FB_THREADS) s_tw2[q] = a.twid[q];
  double2* x = s_x + (size_t)row_in * (L + L / 16);
  const int64_t n_rows = (int64_t)a.N1 * a.K;
  __syncthreads();
  for (int64_t r0 = (int64_t)blockIdx.x * ROWS; r0 < n_rows; r0 += (int64_t)gridDim.x * ROWS) {
    const int64_t r = r0 + row_in;
    const bool live = r < n_rows;
    const int m1 = live ? (int)(r / a.K) : 0, kl = live ? (int)(r - (int64_t)m1 * a.K) : 0;
    double2 v[FB_EPT];
    // ---- load (streaming: each element of Y is read exactly once) and inter-pass twiddle W_N^{c m1}, c = j + t T
    {
      const double2* src = a.Y + (size_t)r * L + j;
#pragma unroll
      for (int t = 0; t < FB_EPT; ++t) v[t] = live ? __ldcs(src + t * T) : make_double2(0.0, 0.0);
      // W_N^{j m1} and W_N^{T m1} from the two-level table (exactly rounded entries, one complex product)
      const int64_t q0 = ((int64_t)j * m1) & (a.N - 1), q1 = ((int64_t)T * m1) & (a.N - 1);
      double2 w = cmul(__ldg(a.twA + (q0 >> 10)), __ldg(a.twB + (q0 & 1023)));
      const double2 ws = cmul(__ldg(a.twA + (q1 >> 10)), __ldg(a.twB + (q1 & 1023)));
      // running product: 15 complex multiplications, < 2e-15 relative on the last factor
#pragma unroll
      for (int t = 0; t < FB_EPT; ++t) {
        v[t] = cmul(v[t], w);
        w = cmul(w, ws);
      }
    }
    // ---- radix-16 stages ending in shared memory (Stockham autosort)
#pragma unroll
    for (int s = 0; s < NFULL; ++s) {
      const int Ns = 1 << (4 * s);
      const int k = j & (Ns - 1);
      if (s > 0) {
#pragma unroll
        for (int t = 0; t < FB_EPT; ++t) v[t] = x[fb_pad(j + t * T)];
        // twiddle W_{16 Ns}^{k t}: Ns = 16 here (at most two such stages), table [t][k]
#pragma unroll
        for (int t = 1; t < FB_EPT; ++t) v[t] = cmul(v[t], s_tw2[16 * t + k]);
        __syncthreads();                       // every thread holds its inputs: the buffer may be overwritten
      }
      fft_regs<16>(v);
      const int base = (j - k) * 16 + k;
#pragma unroll
      for (int t = 0; t < FB_EPT; ++t) x[fb_pad(base + t * Ns)] = v[bitrev<16>(t)];
      __syncthreads();
    }
    // ---- last stage in registers, outputs m2 = jj + t NSL go straight into Eq. 8
    double acc = 0.0;
    const double* al = a.alpha + (size_t)m1 * L;
    const double2* ga = a.gamma + (size_t)m1 * L;
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int jj = j + u * T;
      double2 q[RL];
#pragma unroll
      for (int t = 0; t < RL; ++t) q[t] = x[fb_pad(jj + t * NSL)];
#pragma unroll
      for (int t = 1; t < RL; ++t) q[t] = cmul(q[t], s_tw[t * NSL + jj]);
      fft_regs<RL>(q);
#pragma unroll
      for (int t = 0; t < RL; ++t) {
        const double2 z = q[bitrev<RL>(t)];
        const int m2 = jj + t * NSL;
        const double alp = __ldg(al + m2);
        const double2 g = __ldg(ga + m2);
        acc = fma(alp, fma(z.x, z.x, z.y * z.y), acc);
        acc = fma(-2.0, fma(z.x, g.x, -z.y * g.y), acc);
      }
    }
    __syncthreads();                           // the exchange buffer is free for the next pass
    // ---- fixed-order sum over the row's T threads: shuffle tree inside a warp, then across the row's warps
    if (T >= 32) {
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
      if ((tid & 31) == 0) s_red[tid >> 5] = acc;
      __syncthreads();
      if (j == 0 && live) {
        double sum = 0.0;
#pragma unroll
        for (int wq = 0; wq < T / 32; ++wq) sum += s_red[row_in * (T / 32) + wq];
        a.partial[(size_t)(a.k0 + kl) * a.n_part + m1] = sum;
      }
      __syncthreads();
    } else {
#pragma unroll
      for (int off = T / 2; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
      if (j == 0 && live) a.partial[(size_t)(a.k0 + kl) * a.n_part + m1] = acc;
    }
  }
}

// alpha, gamma (pass-B order: element j = m1 + N1 m2 at m1 N2 + m2) and the partial sums of C_D, from the data spectrum
// D[2][Nf] and the weights w[Nf].  One thread per bin m = 0..N/2; block b writes cd_part[b].
__global__ void __launch_bounds__(256) like_weights_kernel(const double2* __restrict__ D, const double* __restrict__ w,
                                                           int64_t N, int64_t Nf, int N1, int log2N1, int N2,
                                                           double* __restrict__ alpha, double2* __restrict__ gamma,
                                                           double* __restrict__ cd_part) {
  const int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double cd = 0.0;
  if (m < Nf) {
    const double wt = w[m];
    const double2 dI = D[m], dII = D[Nf + m];
    cd = wt * (fma(dI.x, dI.x, dI.y * dI.y) + fma(dII.x, dII.x, dII.y * dII.y));
    // P = (conj D_I - i conj D_II)/2,  conj Q = (D_I - i D_II)/2
    const double2 P = make_double2(0.5 * (dI.x - dII.y), 0.5 * (-dI.y - dII.x));
    const double2 cQ = make_double2(0.5 * (dI.x + dII.y), 0.5 * (dI.y - dII.x));
    const int64_t jn = (m == 0) ? 0 : N - m;
    const int64_t pa = (m & (N1 - 1)) * N2 + (m >> log2N1), pb = (jn & (N1 - 1)) * N2 + (jn >> log2N1);
    if (jn == m) {            // m = 0 or N/2: the element pairs with itself
      alpha[pa] = wt;
      gamma[pa] = make_double2(wt * (P.x + cQ.x), wt * (P.y + cQ.y));
    } else {
      alpha[pa] = 0.5 * wt; gamma[pa] = make_double2(wt * P.x, wt * P.y);
      alpha[pb] = 0.5 * wt; gamma[pb] = make_double2(wt * cQ.x, wt * cQ.y);
    }
  }
  __shared__ double s[8];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) cd += __shfl_xor_sync(0xffffffffu, cd, off);
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = cd;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) t += s[q];
    cd_part[blockIdx.x] = t;
  }
}

// fixed-order final sum of the fused path: logL_k = -scale (C_D + sum_m1 partial[k][m1]); one warp per walker
__global__ void fftlike_final_kernel(const double* partial, int n_part, const double* cd_part, int n_cd, int K, double scale,
                                     const int32_t* status, double* logL, int32_t* status_out) {
  const int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (k >= K) return;
  const double* p = partial + (size_t)k * n_part;
  double acc = 0.0, cd = 0.0;
  for (int i = lane; i < n_part; i += 32) acc += p[i];
  for (int i = lane; i < n_cd; i += 32) cd += cd_part[i];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    acc += __shfl_xor_sync(0xffffffffu, acc, off);
    cd += __shfl_xor_sync(0xffffffffu, cd, off);
  }
  if (lane == 0) {
    const int32_t st = status[k];
    logL[k] = (st & (EMRI_ST_BADPARAM | EMRI_ST_DELAY | EMRI_ST_STATE)) ? -INFINITY : -scale * (cd + acc);
    if (status_out) status_out[k] = st;
  }
}

}  // namespace
