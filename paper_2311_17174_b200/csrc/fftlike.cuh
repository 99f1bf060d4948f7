// fftlike.cuh -- stages (c)+(d) fused: BOTH passes of the transform and the reduction of Eq. 8
// in one persistent kernel of this library, so that the spectrum is never written back nor read again
// (waveform and FFT are one GPU stage).
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
//
// N = N1 N2 (powers of two, N1 in 256 .. 1024, N2 in 256 .. 4096; N1 = 512 at one year of samples).  With i = N2 i1 + i2
// and m = m1 + N1 m2,
//     Z[m1 + N1 m2] = sum_{i2} W_N^{i2 m1} W_N2^{i2 m2}  [ sum_{i1} z[N2 i1 + i2] W_N1^{i1 m1} ].
//   pass A  the bracket: N2 strided transforms of length N1 per walker, read from the chunk z[k][N] the synthesis wrote
//           (natural layout): a ticket is 4096/N1 adjacent columns (128-byte segments at N1 = 512); the result goes to
//           a second buffer as Y[k][m1][i2] (per walker N1 rows of N2: pass A's stores stay within 32 MB per ticket).
//   pass B  one row (m1, k) of N2 contiguous elements per group of N2/16 threads: load, multiply by the twiddle
//           W_N^{i2 m1}, N2-point transform, and the outputs Z[m1 + N1 m2] go straight from registers into Eq. 8.
// Both passes: 16 elements per thread, radix-16 stages in registers, padded shared-memory exchanges in between
// (Stockham autosort), last stage radix L/256 (or 16).
//
// Eq. 8 without pairing, on the residual itself.  Z = DFT(h_I + i h_II) holds Z[m] = H_I[m] + i H_II[m] and
// Z[N-m] = conj H_I[m] + i conj H_II[m].  Pack the data the same way, ZD[m] = D_I[m] + i D_II[m],
// ZD[N-m] = conj D_I[m] + i conj D_II[m]; with R = D - H per channel, ZD[m] - Z[m] = R_I + i R_II and
// ZD[N-m] - Z[N-m] = conj R_I + i conj R_II, whose squared moduli add up to 2 (|R_I|^2 + |R_II|^2) (the cross terms
// cancel).  Hence a sum over single elements of Z:
//     logL = -(2 dt/N) [ C_self + sum_j alpha_j |Z_j - ZD_j|^2 ],   alpha_m = alpha_{N-m} = w_m / 2.
// The self-paired bins m = 0, N/2 take alpha = w_m and ZD = Re D_I + i Re D_II; what the definition adds there for data
// whose DC / Nyquist entries are not real, w_m (Im D_I^2 + Im D_II^2), is the constant C_self (0 for the transform of a
// real series).  No <d|d> - 2<d|h> + <h|h> cancellation: at the injection every term is a small square and logL -> 0
// like the plain path's.  like_weights_kernel builds alpha, ZD (in pass-B order) and C_self from the caller's data
// spectrum once per call; every partial sum has a fixed place and order (bitwise reproducible).
#pragma once
#include "common.cuh"

namespace {

constexpr int FB_THREADS = 256;           // threads per CTA
constexpr int FB_EPT = 16;                // elements per thread
constexpr int FB_ELEMS = FB_THREADS * FB_EPT;   // elements per ticket = 4096

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

// Pass B ticket: ROWS = FB_ELEMS / N2 consecutive rows (m1, k) of Y[K][N1][N2] in the order r = m1 K + k (the K walkers of
// a row m1 share its weights), starting at r0.
// LOG2L = log2 N2 in {8 .. 12}.  Y is read with ld.global.cg (it was written by other CTAs of the same launch); the last
// stage's twiddles `tw_last` [N2] and the weights come from global memory through L1.  s_tw3: three-level table of the
// inter-pass twiddle in shared memory, W_N^q = t0[q & 127] t1[(q >> 7) & 127] t2[q >> 14].  Ends with the exchange
// buffer still in use by slower threads: the caller's next barrier frees it.
template <int LOG2L>
DEVINL void passB_rows(const double2* __restrict__ Ybuf, int64_t r0, int64_t n_rows, int K, int64_t N,
                       const double2* s_tw3, const double2* s_tw2,
                       const double2* __restrict__ tw_last, double2* s_x, double* s_red, const double* __restrict__ alpha,
                       const double2* __restrict__ gamma, double* __restrict__ partial, int k_first, int n_part) {
  constexpr int L = 1 << LOG2L, T = L / FB_EPT;                 // threads per row
  constexpr int NFULL = (LOG2L - 1) / 4;                        // radix-16 stages that end in shared memory
  constexpr int RL = L >> (4 * NFULL);                          // radix of the last stage (16, 2, 4, 8)
  constexpr int U = FB_EPT / RL;                                // last-stage transforms per thread
  constexpr int NSL = L / RL;                                   // their stride
  const int tid = threadIdx.x, row_in = tid / T, j = tid % T;
  double2* x = s_x + (size_t)row_in * (L + L / 16);
  const int64_t r = r0 + row_in;
  const bool live = r < n_rows;
  const int m1 = live ? (int)(r / K) : 0, kl = live ? (int)(r - (int64_t)m1 * K) : 0;
  double2 v[FB_EPT];
  // ---- load (each element of Y is read exactly once) and inter-pass twiddle W_N^{c m1}, c = j + t T
  {
    const int N1 = (int)(n_rows / K);
    const double2* src = Ybuf + ((size_t)kl * N1 + m1) * L + j;      // Y[k][m1][i2]
#pragma unroll
    for (int t = 0; t < FB_EPT; ++t)
      v[t] = live ? __ldcg(src + t * T) : make_double2(0.0, 0.0);
    // W_N^{j m1} and W_N^{T m1} from the three-level table (exactly rounded entries, two complex products)
    const int64_t q0 = ((int64_t)j * m1) & (N - 1), q1 = ((int64_t)T * m1) & (N - 1);
    double2 w = cmul(cmul(s_tw3[q0 & 127], s_tw3[128 + ((q0 >> 7) & 127)]), s_tw3[256 + (q0 >> 14)]);
    const double2 ws = cmul(cmul(s_tw3[q1 & 127], s_tw3[128 + ((q1 >> 7) & 127)]), s_tw3[256 + (q1 >> 14)]);
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
  const double* al = alpha + (size_t)m1 * L;
  const double2* ga = gamma + (size_t)m1 * L;
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int jj = j + u * T;
    double2 q[RL];
#pragma unroll
    for (int t = 0; t < RL; ++t) q[t] = x[fb_pad(jj + t * NSL)];
#pragma unroll
    for (int t = 1; t < RL; ++t) q[t] = cmul(q[t], __ldg(tw_last + t * NSL + jj));
    fft_regs<RL>(q);
#pragma unroll
    for (int t = 0; t < RL; ++t) {
      const double2 z = q[bitrev<RL>(t)];
      const int m2 = jj + t * NSL;
      const double alp = __ldg(al + m2);
      const double2 g = __ldg(ga + m2);                       // packed data spectrum ZD at this element
      const double rx = z.x - g.x, ry = z.y - g.y;
      acc = fma(alp, fma(rx, rx, ry * ry), acc);
    }
  }
  // ---- fixed-order sum over the row's T threads: shuffle tree inside a warp, then across the row's warps
  // (no barrier of its own frees the exchange buffer or s_red: the one that releases the ticket follows)
  if (T >= 32) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if ((tid & 31) == 0) s_red[tid >> 5] = acc;
    __syncthreads();
    if (j == 0 && live) {
      double sum = 0.0;
#pragma unroll
      for (int wq = 0; wq < T / 32; ++wq) sum += s_red[row_in * (T / 32) + wq];
      partial[(size_t)(k_first + kl) * n_part + m1] = sum;
    }
  } else {
#pragma unroll
    for (int off = T / 2; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (j == 0 && live) partial[(size_t)(k_first + kl) * n_part + m1] = acc;
  }
}

// ---- The kernel.  Pass A of the chunk writes the second buffer, pass B reads it back and feeds Eq. 8.  One persistent
// kernel runs both as a dataflow: CTAs pop tickets (4096 elements each) from ONE counter, first the `items` tickets of
// pass A, then the `items` tickets of pass B.  A pass-B ticket waits until every pass-A ticket is done; those are SMALLER
// tickets, which running CTAs hold, so the schedule cannot deadlock whatever the number of resident CTAs.
// (Round 2 also measured splitting the chunk into groups of g walkers with a two-slot ring, A(q+1) interleaved with B(q):
// on B200 at configs[3] the larger the group the faster -- the weights of a row m1 are shared by all walkers and stay in
// L1/L2, and keeping the intermediate of a small group inside the 126 MB L2 gained nothing because the kernel is bound by
// instruction latency, not by HBM -- so only the single-group schedule is kept; DESIGN.md section 6c has the numbers.)
struct Fft2Args {
  const double2* z;        // [kc][N] chunk, natural layout
  double2* ring;           // [kc][N] intermediate Y[k][m1][i2]
  const double2* twid1;    // [256 + N1] stage twiddles of pass A (same construction as twid2)
  const double2* twid2;    // [256 + N2] of pass B
  const double2* tw3;      // [512] inter-pass twiddle in three levels: W_N^q, W_N^{128 q} (q < 128), W_N^{16384 q} (q < 256)
  const double* alpha;
  const double2* gamma;
  double* partial;
  unsigned* ctr;           // [0] ticket counter, [1] tickets of pass A done; zeroed before the launch
  int k0, kc, n_part, N1, N2;
  unsigned items;          // tickets per pass = kc N / 4096
  int64_t N;
};

DEVINL void fft2_wait(const unsigned* ctr, unsigned target) {
  if (threadIdx.x == 0) {
    unsigned v;
    for (;;) {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if (v >= target) break;
      __nanosleep(64);
    }
  }
  __syncthreads();
}
// end of a ticket: every thread's global stores and shared-memory reads precede the barrier; thread 0 then releases the
// ticket (`done` may be NULL) and publishes the next one
DEVINL void fft2_finish(unsigned* done, unsigned* s_ticket, unsigned next_tk) {
  __syncthreads();
  if (threadIdx.x == 0) {
    if (done) { __threadfence(); atomicAdd(done, 1u); }
    *s_ticket = next_tk;
  }
  __syncthreads();
}

// Pass A ticket: COLS adjacent columns (col0 ..) of one walker: N1-point transforms along i1 (stride N2), output row m1
// of the group's ring slot.  Lanes run over the columns first, so a warp touches 32 / COLS segments of COLS x 16 B.
template <int LOG2L>
DEVINL void passA_cols(const double2* __restrict__ zk, double2* __restrict__ Yslot, int gq, int kl, int col0, int N2,
                       const double2* s_tw2, const double2* __restrict__ tw_last, double2* s_x) {
  constexpr int L = 1 << LOG2L, T = L / FB_EPT, COLS = FB_ELEMS / L;
  constexpr int NFULL = (LOG2L - 1) / 4, RL = L >> (4 * NFULL), U = FB_EPT / RL, NSL = L / RL;
  constexpr int XS = L + L / 16 + (COLS >= 8 ? 1 : 8 / COLS);   // column stride: the COLS lanes of a quarter-warp hit different banks
  const int tid = threadIdx.x, c = tid % COLS, j = tid / COLS;
  double2* x = s_x + (size_t)c * XS;
  double2 v[FB_EPT];
  {
    const double2* src = zk + (size_t)j * N2 + col0 + c;
#pragma unroll
    for (int t = 0; t < FB_EPT; ++t) v[t] = __ldcs(src + (size_t)t * T * N2);
  }
#pragma unroll
  for (int s = 0; s < NFULL; ++s) {
    const int Ns = 1 << (4 * s);
    const int k = j & (Ns - 1);
    if (s > 0) {
#pragma unroll
      for (int t = 0; t < FB_EPT; ++t) v[t] = x[fb_pad(j + t * T)];
#pragma unroll
      for (int t = 1; t < FB_EPT; ++t) v[t] = cmul(v[t], s_tw2[16 * t + k]);
      __syncthreads();
    }
    fft_regs<16>(v);
    const int base = (j - k) * 16 + k;
#pragma unroll
    for (int t = 0; t < FB_EPT; ++t) x[fb_pad(base + t * Ns)] = v[bitrev<16>(t)];
    __syncthreads();
  }
#pragma unroll
  for (int u = 0; u < U; ++u) {
    const int jj = j + u * T;
    double2 q[RL];
#pragma unroll
    for (int t = 0; t < RL; ++t) q[t] = x[fb_pad(jj + t * NSL)];
#pragma unroll
    for (int t = 1; t < RL; ++t) q[t] = cmul(q[t], __ldg(tw_last + t * NSL + jj));
    fft_regs<RL>(q);
#pragma unroll
    for (int t = 0; t < RL; ++t) {
      const int m1 = jj + t * NSL;
      Yslot[((size_t)kl * L + m1) * N2 + col0 + c] = q[bitrev<RL>(t)];      // Y[k][m1][i2], L = N1
    }
  }
}                                            // (the barrier that releases the ticket frees the exchange buffer)

template <int LG1, int LG2>
__global__ void __launch_bounds__(FB_THREADS, 2) fft2_like_kernel(Fft2Args a) {
  constexpr int COLS = FB_ELEMS >> LG1, ROWS = FB_ELEMS >> LG2;
  extern __shared__ __align__(16) unsigned char fb_smem[];
  double2* s_tw2 = reinterpret_cast<double2*>(fb_smem);                      // [16][16] W_256^{k t}
  double2* s_tw3 = s_tw2 + 256;                                              // [512] inter-pass twiddle levels
  double2* s_x = s_tw3 + 512;                                                // exchange buffer of either pass
  __shared__ double s_red[FB_THREADS / 32];
  __shared__ unsigned s_ticket;
  for (int q = threadIdx.x; q < 256; q += FB_THREADS) s_tw2[q] = a.twid2[q];
  for (int q = threadIdx.x; q < 512; q += FB_THREADS) s_tw3[q] = a.tw3[q];
  const unsigned total = 2u * a.items;
  // thread 0 draws the NEXT ticket while the current one is being worked on (the round trip of the atomic is off the
  // critical path); a CTA thus holds two tickets, which keeps the no-deadlock argument: the smallest unfinished ticket
  // is running, or held by a CTA whose running ticket is smaller still
  unsigned next_tk = 0;
  if (threadIdx.x == 0) next_tk = atomicAdd(a.ctr, 1u);
  if (threadIdx.x == 0) s_ticket = next_tk;
  __syncthreads();
  for (;;) {
    const unsigned tk = s_ticket;
    if (tk >= total) break;
    if (threadIdx.x == 0) next_tk = atomicAdd(a.ctr, 1u);
    // ticket order: the `items` tickets of pass A, then the `items` tickets of pass B
    const int kind = tk >= a.items ? 1 : 0;
    const unsigned idx = tk - (kind ? a.items : 0u);
    if (kind == 0) {
      const int cbs = a.N2 / COLS;
      const int kl = (int)idx / cbs, cb = (int)idx - kl * cbs;
      passA_cols<LG1>(a.z + (size_t)kl * a.N, a.ring, a.kc, kl, cb * COLS, a.N2, s_tw2, a.twid1 + 256, s_x);
      fft2_finish(a.ctr + 1, &s_ticket, next_tk);
    } else {
      fft2_wait(a.ctr + 1, a.items);
      passB_rows<LG2>(a.ring, (int64_t)idx * ROWS, (int64_t)a.N1 * a.kc, a.kc, a.N, s_tw3, s_tw2, a.twid2 + 256, s_x,
                      s_red, a.alpha, a.gamma, a.partial, a.k0, a.n_part);
      fft2_finish(nullptr, &s_ticket, next_tk);
    }
  }
}

// alpha and the packed data spectrum ZD (`gamma`; pass-B order: element j = m1 + N1 m2 at m1 N2 + m2) and the partial
// sums of C_self, from the data spectrum D[2][Nf] and the weights w[Nf].  One thread per bin m = 0..N/2; block b writes
// cd_part[b].
__global__ void __launch_bounds__(256) like_weights_kernel(const double2* __restrict__ D, const double* __restrict__ w,
                                                           int64_t N, int64_t Nf, int N1, int log2N1, int N2,
                                                           double* __restrict__ alpha, double2* __restrict__ gamma,
                                                           double* __restrict__ cd_part) {
  const int64_t m = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double cd = 0.0;
  if (m < Nf) {
    const double wt = w[m];
    const double2 dI = D[m], dII = D[Nf + m];
    const int64_t jn = (m == 0) ? 0 : N - m;
    const int64_t pa = (m & (N1 - 1)) * N2 + (m >> log2N1), pb = (jn & (N1 - 1)) * N2 + (jn >> log2N1);
    if (jn == m) {            // m = 0 or N/2: the element pairs with itself; Z is H_I + i H_II with both real
      alpha[pa] = wt;
      gamma[pa] = make_double2(dI.x, dII.x);
      cd = wt * fma(dI.y, dI.y, dII.y * dII.y);               // 0 for the transform of a real series
    } else {
      alpha[pa] = 0.5 * wt; gamma[pa] = make_double2(dI.x - dII.y, dI.y + dII.x);      // D_I + i D_II
      alpha[pb] = 0.5 * wt; gamma[pb] = make_double2(dI.x + dII.y, dII.x - dI.y);      // conj D_I + i conj D_II
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

// fixed-order final sum of the fused path: logL_k = -scale (C_self + sum_m1 partial[k][m1]); one warp per walker
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
