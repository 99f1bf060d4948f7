// loglike_static.cu -- emri_spectra_loglike_static (include/emri.h): Eq. 8 for callers that cannot
// allocate device memory.
//
// Who needs this.  Every other likelihood call of the library goes through an emri_plan, and a plan gets its workspace
// from cudaMalloc.  That is not open to everybody:
//   - a process that has handed the whole GPU to one memory pool at start-up (a framework's caching allocator, a
//     sampler that pre-partitions the card between chains) has nothing left for a second allocator to take;
//   - a client with a fixed memory quota (MPS limits, a container's share of the card) may be refused at any time;
//   - a latency-critical host thread must not call cudaMalloc / cudaFree at all, because both synchronise the whole
//     device and stall every other stream while they run.
// Such a caller already holds the model spectra (emri_waveform_fft wrote them into ITS buffer) and only needs the
// noise-weighted residual sum.  The two-pass reduction below needs one piece of memory beyond its inputs and its output,
// the per-(walker, bin-range) partial sums; here that memory is a fixed array that is part of the library image itself.
//
// What it costs.  EMRI_STATIC_SCRATCH_DOUBLES doubles (512 KiB) of device memory on every GPU that loads the library, from
// the moment the library's module is loaded on that GPU until the process exits, whether or not this entry point is used.
//
// Self-contained on purpose: array, address look-up, kernels and entry point live in this one file and share nothing
// with the plan-based path in emri.cu (which is unchanged).
#include <cuda_runtime.h>
#include <cmath>
#include <cstdint>
#include <mutex>
#include "../../include/emri.h"

// The scratch array.  In HOST code the name `g_static_partials` is only a handle for the runtime's symbol table, not a
// device address: passing it to a kernel would hand the kernel a host-side address.  Host code must translate it with
// cudaGetSymbolAddress (scratch_of_current_device below); device code could name it directly, but the kernels take the
// translated pointer as an argument so that there is exactly one way the address reaches them.
static __device__ __align__(256) double g_static_partials[EMRI_STATIC_SCRATCH_DOUBLES];

namespace {

constexpr int SL_THREADS = 256;
constexpr int SL_WARPS = SL_THREADS / 32;
constexpr int SL_GROUP = 8;                          // walkers per CTA, one accumulator each per thread
constexpr int SL_RANGE = EMRI_STATIC_BINS_PER_PART;  // bins per CTA = bins per partial sum
constexpr int SL_MAX_DEVICES = 64;

std::mutex g_mu;
double* g_scratch_addr[SL_MAX_DEVICES];  // device address of g_static_partials on device d; nullptr = not looked up yet
int g_last_cuda_error = 0;               // raw cudaError_t of the last failing runtime call (under g_mu)

// Set-up, once per device, with that device current: ask the runtime where the array lives ON THIS DEVICE (every device
// that loads the module has its own copy at its own address).  The look-up may make the runtime load the library's module
// on the device, which is why the first call per device belongs before any stream capture the caller plans.
int scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  std::lock_guard<std::mutex> lk(g_mu);
  if (e != cudaSuccess) { g_last_cuda_error = (int)e; return EMRI_ECUDA; }
  if (dev < 0 || dev >= SL_MAX_DEVICES) return EMRI_EINVAL;
  if (!g_scratch_addr[dev]) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_static_partials);
    if (e != cudaSuccess || !ptr) { g_last_cuda_error = (int)e; return EMRI_ECUDA; }
    g_scratch_addr[dev] = static_cast<double*>(ptr);
  }
  *out = g_scratch_addr[dev];
  return EMRI_OK;
}

// First pass.  grid (bin ranges, walker groups): CTA (x, y) sums w_m (|D_I - H_I|^2 + |D_II - H_II|^2) over the bins
// m in [x SL_RANGE, (x+1) SL_RANGE) for walkers 8y .. 8y+7 and writes one partial per walker.  A variant of
// loglike_kernel (loglike.cuh) that reads the two channel spectra as emri_waveform_fft stores them instead of the
// packed transform, and derives the weight from the PSD in place (same masking rule as emri_plan_create).
// Every cell partial[k][x], k < K, x < n_part, is WRITTEN here before the second pass reads it, so whatever an earlier
// call left in the array is never seen and nothing has to be cleared.
__global__ void __launch_bounds__(SL_THREADS)
spectra_loglike_static_kernel(const double2* __restrict__ H, const double2* __restrict__ D, const double* __restrict__ psd,
                              double* __restrict__ partial, int K, int64_t Nf, int n_part) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int kg0 = blockIdx.y * SL_GROUP;
  const int64_t m_begin = (int64_t)blockIdx.x * SL_RANGE;
  const int64_t m_end = m_begin + SL_RANGE < Nf ? m_begin + SL_RANGE : Nf;
  const double2* row[SL_GROUP];
  double acc[SL_GROUP];
#pragma unroll
  for (int g = 0; g < SL_GROUP; ++g) {
    const int kk = kg0 + g < K ? kg0 + g : K - 1;  // the ragged last group re-reads walker K-1 and drops the result
    row[g] = H + (size_t)kk * 2 * Nf;
    acc[g] = 0.0;
  }
  for (int64_t m = m_begin + threadIdx.x; m < m_end; m += SL_THREADS) {
    double2 hI[SL_GROUP], hII[SL_GROUP];
#pragma unroll
    for (int g = 0; g < SL_GROUP; ++g) { hI[g] = __ldcs(row[g] + m); hII[g] = __ldcs(row[g] + Nf + m); }
    const double2 dI = __ldg(D + m), dII = __ldg(D + Nf + m);
    const double s = __ldg(psd + m);
    const double wt = (s > 0.0 && isfinite(s)) ? 1.0 / s : 0.0;
#pragma unroll
    for (int g = 0; g < SL_GROUP; ++g) {
      const double ar = dI.x - hI[g].x, ai = dI.y - hI[g].y, br = dII.x - hII[g].x, bi = dII.y - hII[g].y;
      const double pw = fma(ar, ar, ai * ai) + fma(br, br, bi * bi);
      acc[g] = fma(wt, pw, acc[g]);
    }
  }
  __shared__ double s_acc[SL_WARPS][SL_GROUP];
#pragma unroll
  for (int g = 0; g < SL_GROUP; ++g) {
    double v = acc[g];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) s_acc[warp][g] = v;
  }
  __syncthreads();
  if (threadIdx.x < SL_GROUP && kg0 + (int)threadIdx.x < K) {
    double v = 0.0;
#pragma unroll
    for (int wq = 0; wq < SL_WARPS; ++wq) v += s_acc[wq][threadIdx.x];
    partial[(size_t)(kg0 + threadIdx.x) * n_part + blockIdx.x] = v;
  }
}

// Second pass, fixed order (no atomics, so the result is reproducible bit for bit): one warp per walker.
__global__ void spectra_loglike_static_final_kernel(const double* __restrict__ partial, int n_part, int K, double scale,
                                                    double* __restrict__ logL) {
  const int k = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (k >= K) return;
  const double* p = partial + (size_t)k * n_part;
  double acc = 0.0;
  for (int i = lane; i < n_part; i += 32) acc += p[i];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
  if (lane == 0) logL[k] = -scale * acc;
}

}  // namespace

extern "C" int64_t emri_static_scratch_need(int K, int64_t N) {
  if (K < 1 || N < 4 || (N & 1)) return -1;
  const int64_t Nf = N / 2 + 1;
  return (int64_t)K * ((Nf + SL_RANGE - 1) / SL_RANGE);
}

extern "C" int emri_static_last_cuda_error(void) {
  std::lock_guard<std::mutex> lk(g_mu);
  return g_last_cuda_error;
}

extern "C" int emri_spectra_loglike_static(const double* spectra, int K, int64_t N, double dt, const double* data_fft,
                                           const double* psd, double* logL, void* cuda_stream) {
  // argument and size checks first: none of them touches the CUDA runtime
  if (!spectra || !data_fft || !psd || !logL || K < 1 || N < 4 || (N & 1) || !(dt > 0.0) || !std::isfinite(dt))
    return EMRI_EINVAL;
  const int64_t need = emri_static_scratch_need(K, N);
  if (need > (int64_t)EMRI_STATIC_SCRATCH_DOUBLES) return EMRI_ELIMIT;
  const int64_t Nf = N / 2 + 1;
  const int n_part = (int)((Nf + SL_RANGE - 1) / SL_RANGE);
  if ((K + SL_GROUP - 1) / SL_GROUP > 65535) return EMRI_ELIMIT;  // grid.y; unreachable below the scratch limit

  double* partial = nullptr;
  if (int rc = scratch_of_current_device(&partial)) return rc;

  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const dim3 grid((unsigned)n_part, (unsigned)((K + SL_GROUP - 1) / SL_GROUP));
  spectra_loglike_static_kernel<<<grid, SL_THREADS, 0, s>>>(reinterpret_cast<const double2*>(spectra),
                                                            reinterpret_cast<const double2*>(data_fft), psd, partial, K, Nf,
                                                            n_part);
  spectra_loglike_static_final_kernel<<<(K + 3) / 4, 128, 0, s>>>(partial, n_part, K, 2.0 * dt / (double)N, logL);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    std::lock_guard<std::mutex> lk(g_mu);
    g_last_cuda_error = (int)e;
    return EMRI_ECUDA;
  }
  return EMRI_OK;
}
