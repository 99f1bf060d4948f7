// emri.cu -- sm_100a implementation of include/emri.h (the hot path of EMRI_MC, arXiv 2311.17174).
//
// Host side of the library: plan, workspace, stage sequencing, cuFFT.  Stages:
//   (a) orbit.cuh    per-walker scalars (Eq. 6) and the fixed-step RK4 integration of Eq. 1
//                     on the coarse grid, evaluated parallel in time (multiple shooting)
//   (b) synth.cuh    persistent CTAs over (walker, unit of 256-sample tiles): cubic-Hermite orbit, Peters-Mathews
//                    harmonic sum n = 1..n_max (Eq. 2), LISA response,
//                    propagation factors (Eqs. 4-6); writes z = h_I + i h_II
//   (c) cufftExecZ2Z one in-place complex transform per walker carries both channels, the one vendor call
//   (d) loglike.cuh  streaming reduction of Eq. 8 on the packed spectrum (+ Eq. 7's factor) and the
//                    fixed-order final sum
// Nothing here is shared with oracle/ (which is test infrastructure).  FP64 throughout.
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>
#include <vector>

#include "../../include/emri.h"

#include "common.cuh"
#include "orbit.cuh"
#include "orbit_dp5.cuh"
#include "synth.cuh"
#include "loglike.cuh"
#include "fftlike.cuh"
#include "stretch.cuh"

// =================================================================== host side
struct emri_plan {
  int64_t N = 0, Nf = 0, Nc = 0, Nn = 0;
  double dt = 0;
  int n_max = 0, K_max = 0, S = 256, logS = 8, chunk = 0;
  double H0 = 67.4, Om = 0.315;
  int device = 0, sm_count = 148, synth_grid = 0;
  size_t synth_smem = 0;
  // device buffers
  double* d_w = nullptr;
  double* d_wc = nullptr;
  double* d_nodes = nullptr;
  double* d_hbuf = nullptr;
  double* d_partial = nullptr;
  double4* d_base = nullptr;      // Taylor coefficients of the harmonic brackets in e^2 (synth.cuh)
  double* d_gtab = nullptr;       // n (n/2)^{n-2} / (n-2)!: bracket scale of the Bessel path (n_max > 48)
  double2* d_nodeaux = nullptr;
  int32_t* d_jpl = nullptr;
  int32_t* d_status = nullptr;
  // adaptive embedded pair (orbit_dp5.cuh): emri_plan_set_integrator
  int integrator = 0, dp_cap = 0;
  bool orbit_ran = false;                    // stage (a) has run since the last change of integrator / schedule
  double dp_rtol = 1e-12, dp_atol[5] = {1e-12, 1e-21, 1e-12, 1e-17, 1e-12};
  double* d_dpsteps = nullptr;
  int32_t* d_dpn = nullptr; int32_t* d_dpstop = nullptr; int32_t* d_dpbad = nullptr; int32_t* d_dpzero = nullptr;
  // multiple-shooting orbit (orbit.cuh): segment records, per-walker mode / tail start / post-plunge row
  int orbit_mode = 1, anchor_end = 0, seg_L = 0, seg_P = 0, unit_tiles_override = 0, unit_tiles_cap = 8;
  int synth_debug = 0;                       // emri_plan_set_synth_debug
  double series_tol = 1e-14;                 // emri_plan_set_series_tolerance (reading D8)
  int launches = 0;                          // kernels of this library enqueued by the last hot call
  // CUDA graphs of emri_loglike (one per distinct argument set, a few kept): the 13-27 launches of a call become one
  struct GraphEntry {
    const void *params, *data, *logL, *status, *fcoef;
    int K; double fstar; cudaGraphExec_t exec; int launches, n_chunks; uint64_t used;
  };
  std::vector<GraphEntry> graphs;
  bool graphs_on = true;
  cudaStream_t s_cap = nullptr;              // capture stream (the caller's may be the legacy stream, which cannot capture)
  int64_t graph_captures = 0, graph_replays = 0;
  uint64_t graph_clock = 0;
  unsigned long long* d_counts = nullptr;    // [SYN_COUNTS] path counters of stage (b), zeroed at the start of every call
  double* d_seg = nullptr;
  double* d_plrow = nullptr;
  int32_t* d_mode = nullptr;
  int32_t* d_pclamp = nullptr;
  // host-variant staging
  double* d_params = nullptr;
  double* d_data = nullptr;
  double* d_logL = nullptr;
  bool data_loaded = false;
  // stretch move scratch
  double* d_Y = nullptr; double* d_z = nullptr; double* d_lnu = nullptr; double* d_logLY = nullptr;
  int32_t* d_inbox = nullptr; int32_t* d_partner = nullptr;
  // fused transform + reduction (fftlike.cuh): N = N1 N2; available for N = 2^16 .. 2^22
  bool fused_ok = false;
  bool fused_on = true;                // false: full cuFFT transform + loglike_kernel
  int N1 = 0, N2 = 0, log2N1 = 0, log2N2 = 0, n_cd = 0;
  double2* d_ring = nullptr;           // [chunk][N] pass-A output
  unsigned* d_fft2ctr = nullptr;       // ticket and completion counters of fft2_like_kernel
  double2* d_twid1 = nullptr;          // stage twiddles of pass A (length N1)
  double2* d_tw3 = nullptr;            // three-level inter-pass twiddle of fft2_like_kernel
  double2* d_twid = nullptr;
  double* d_alpha = nullptr;
  double2* d_gamma = nullptr;
  double* d_cdpart = nullptr;
  // cuFFT
  std::map<int, cufftHandle> fft;
  void* d_fftwork = nullptr;
  size_t fftwork_bytes = 0;
  // copy stream of emri_loglike_host: the data spectrum is uploaded while stages (a)-(c) run
  cudaStream_t s_copy = nullptr;
  cudaEvent_t ev_call = nullptr, ev_data = nullptr;
  cudaEvent_t wait_before_like = nullptr;     // set for the duration of one loglike_impl call
  // timings
  bool timing = false;
  std::vector<cudaEvent_t> ev;
  int ev_used = 0;
  int n_chunks_last = 0;
  bool had_like = false;
  int last_err = 0;
  int64_t bytes = 0;
  int n_part = 0;
};

namespace {

#define CK(call)                                        \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) { p->last_err = (int)e_; return EMRI_ECUDA; } \
  } while (0)
#define CKF(call)                                       \
  do {                                                  \
    cufftResult r_ = (call);                            \
    if (r_ != CUFFT_SUCCESS) { p->last_err = (int)r_; return EMRI_ECUFFT; } \
  } while (0)

// EMRI_DEBUG_SYNC=1 in the environment synchronises after every kernel of stage (a) and names the one that failed
int debug_sync(emri_plan* p, cudaStream_t s, const char* what) {
  static const bool on = std::getenv("EMRI_DEBUG_SYNC") != nullptr;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess && on) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) {
    p->last_err = (int)e;
    if (on) std::fprintf(stderr, "[emri] %s failed: %s\n", what, cudaGetErrorString(e));
    return EMRI_ECUDA;
  }
  return EMRI_OK;
}
#define DBG(what) do { int rc_ = debug_sync(p, s, what); if (rc_) return rc_; } while (0)

// every setting that changes what a call enqueues invalidates the captured graphs
void drop_graphs(emri_plan* p) {
  for (auto& g : p->graphs) cudaGraphExecDestroy(g.exec);
  p->graphs.clear();
}

template <class T> int dev_alloc(emri_plan* p, T** ptr, size_t count) {
  if (*ptr) { cudaFree(*ptr); *ptr = nullptr; }
  if (count == 0) return EMRI_OK;
  cudaError_t e = cudaMalloc((void**)ptr, count * sizeof(T));
  if (e != cudaSuccess) { p->last_err = (int)e; *ptr = nullptr; cudaGetLastError(); return EMRI_ENOMEM; }
  p->bytes += (int64_t)(count * sizeof(T));
  return EMRI_OK;
}

// Taylor coefficients in w = e^2 of the three harmonic brackets (synth.cuh), in long double.
// With J_k(n e) = (n e/2)^k s_k(w), s_k(w) = sum_m sigma(k,m) w^m, sigma(k,m) = (-n^2/4)^m / (m! (m+k)!):
//   n >= 2:  n [J_{n-2} - 2e J_{n-1} + (2/n) J_n + 2e J_{n+1} - J_{n+2}] = e^{n-2} PA_n(w)   etc.
//   n == 1:  the same brackets with J_{-1} = -J_1 carry e^{+1}.
void build_base_table(int n_max, std::vector<double4>& base) {
  base.assign((size_t)(n_max + 1) * BASE_M, make_double4(0.0, 0.0, 0.0, 0.0));
  std::vector<long double> fact(2 * BASE_M + EMRI_NMAX_CAP + 8);
  fact[0] = 1.0L;
  for (size_t i = 1; i < fact.size(); ++i) fact[i] = fact[i - 1] * (long double)i;
  for (int n = 1; n <= n_max; ++n) {
    const long double nn = n, y = -0.25L * nn * nn;
    auto sigma = [&](int k, int m) -> long double {
      if (m < 0) return 0.0L;
      return powl(y, (long double)m) / (fact[m] * fact[m + k]);
    };
    for (int m = 0; m < BASE_M; ++m) {
      long double pa, pb, pc;
      if (n == 1) {
        pa = 0.5L * sigma(1, m) - 2.0L * sigma(0, m) + 0.5L * sigma(2, m - 1) - 0.125L * sigma(3, m - 1);
        pb = -1.5L * sigma(1, m) + 0.125L * sigma(3, m - 1);
        pc = 0.5L * sigma(1, m);
      } else {
        const long double pref = powl(0.5L * nn, (long double)(n - 2));          // (n/2)^{n-2}
        const long double n2 = nn * nn, n3 = n2 * nn, n4 = n2 * n2;
        pa = nn * pref * (sigma(n - 2, m) - nn * sigma(n - 1, m - 1) + 0.5L * nn * sigma(n, m - 1) +
                          0.25L * n3 * sigma(n + 1, m - 2) - 0.0625L * n4 * sigma(n + 2, m - 2));
        pb = nn * pref * (sigma(n - 2, m) - 0.5L * n2 * sigma(n, m - 1) + 0.0625L * n4 * sigma(n + 2, m - 2));
        pc = pref * 0.25L * n2 * sigma(n, m - 1);
      }
      base[(size_t)n * BASE_M + m] = make_double4((double)pa, (double)pb, (double)pc, 0.0);
    }
  }
}

int alloc_workspace(emri_plan* p) {
  int rc;
  p->Nc = (p->N + p->S - 1) / p->S;
  p->Nn = p->Nc + 3;
  if ((rc = dev_alloc(p, &p->d_nodes, (size_t)p->K_max * p->Nn * NODE_STRIDE))) return rc;
  if ((rc = dev_alloc(p, &p->d_nodeaux, (size_t)p->K_max * p->Nn))) return rc;
  // segments of the parallel-in-time orbit: L = power of two nearest sqrt(n_steps / 2) (cost ~ P + 2 L steps)
  const int64_t n_steps = p->Nc + 1;
  int lg = (int)std::floor(0.5 * std::log2(0.5 * (double)n_steps) + 0.5);
  if (lg < 2) lg = 2;
  // orbit_correct_kernel keeps 96 B per segment in shared memory: at most 2048 segments (192 KB)
  while (((n_steps + (1 << lg) - 1) >> lg) > 2048) ++lg;
  p->seg_L = 1 << lg;
  p->seg_P = (int)((n_steps + p->seg_L - 1) / p->seg_L);
  if (cudaFuncSetAttribute(orbit_correct_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           std::max(48 * 1024, p->seg_P * 12 * (int)sizeof(double))) != cudaSuccess) {
    p->last_err = (int)cudaGetLastError();
    return EMRI_ECUDA;
  }
  if ((rc = dev_alloc(p, &p->d_seg, (size_t)p->K_max * p->seg_P * SEG_STRIDE))) return rc;
  return EMRI_OK;
}

int get_fft(emri_plan* p, int batch, cufftHandle* out);
cudaError_t fft2_set_smem();
// (Re)allocates the chunk buffer and creates, up front, every cuFFT plan the hot calls of a full ensemble need: a full
// chunk, the ragged last chunk of K_max walkers, and the single transform of emri_data_fft.  The work area is sized by
// the largest of them (the full chunk), so a later call with another ragged K only builds its plan object on first use
// and never allocates or synchronises (include/emri.h: "only ENQUEUES").
int alloc_chunk(emri_plan* p) {
  int rc;
  if ((rc = dev_alloc(p, &p->d_hbuf, (size_t)2 * p->chunk * p->N))) return rc;      // z = h_I + i h_II, [chunk][N] complex
  if (p->fused_ok) {
    if ((rc = dev_alloc(p, &p->d_ring, (size_t)p->chunk * p->N))) return rc;          // pass A -> pass B intermediate
    if ((rc = dev_alloc(p, &p->d_fft2ctr, (size_t)2))) return rc;                       // ticket counter, pass-A tickets done
  }
  for (auto& kv : p->fft) cufftDestroy(kv.second);
  p->fft.clear();
  cufftHandle h;
  if ((rc = get_fft(p, p->chunk, &h))) return rc;
  if (p->K_max % p->chunk) { if ((rc = get_fft(p, p->K_max % p->chunk, &h))) return rc; }
  if ((rc = get_fft(p, 1, &h))) return rc;
  return EMRI_OK;
}

int get_fft(emri_plan* p, int batch, cufftHandle* out) {
  auto it = p->fft.find(batch);
  if (it != p->fft.end()) { *out = it->second; return EMRI_OK; }
  cufftHandle h;
  CKF(cufftCreate(&h));
  CKF(cufftSetAutoAllocation(h, 0));
  long long n[1] = {(long long)p->N};
  long long embed[1] = {(long long)p->N};
  size_t ws = 0;
  // one complex transform per walker carries both real channels (loglike.cuh)
  cufftResult r = cufftMakePlanMany64(h, 1, n, embed, 1, (long long)p->N, embed, 1, (long long)p->N, CUFFT_Z2Z,
                                      (long long)batch, &ws);
  if (r != CUFFT_SUCCESS) { p->last_err = (int)r; cufftDestroy(h); return EMRI_ECUFFT; }
  if (ws > p->fftwork_bytes) {
    // grow the shared work area; every cached plan is re-pointed at it.  Reached from alloc_chunk (plan creation,
    // emri_plan_set_chunk) only: the full chunk is planned first and no smaller batch is expected to need more.  Should
    // cuFFT ever ask for more for a smaller batch, the captured graphs still hold the old work-area pointer: drop them
    drop_graphs(p);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { p->last_err = (int)e; cufftDestroy(h); return EMRI_ECUDA; }
    if (p->d_fftwork) { cudaFree(p->d_fftwork); p->bytes -= (int64_t)p->fftwork_bytes; p->d_fftwork = nullptr; }
    e = cudaMalloc(&p->d_fftwork, ws);
    if (e != cudaSuccess) { p->last_err = (int)e; p->fftwork_bytes = 0; cufftDestroy(h); cudaGetLastError(); return EMRI_ENOMEM; }
    p->fftwork_bytes = ws;
    p->bytes += (int64_t)ws;
    for (auto& kv : p->fft) cufftSetWorkArea(kv.second, p->d_fftwork);
  }
  if (p->d_fftwork) CKF(cufftSetWorkArea(h, p->d_fftwork));
  p->fft[batch] = h;
  *out = h;
  return EMRI_OK;
}

cudaEvent_t next_event(emri_plan* p) {
  if (p->ev_used == (int)p->ev.size()) {
    cudaEvent_t e;
    cudaEventCreate(&e);
    p->ev.push_back(e);
  }
  return p->ev[p->ev_used++];
}
void mark(emri_plan* p, cudaStream_t s) {
  if (p->timing) cudaEventRecord(next_event(p), s);
}

int run_orbit(emri_plan* p, const double* params, int K, cudaStream_t s) {
  p->launches = 0;
  p->orbit_ran = true;     // (a graph replay re-runs what a capture enqueued here under the same settings)
  CK(cudaMemsetAsync(p->d_counts, 0, SYN_COUNTS * sizeof(unsigned long long), s));
  OrbitArgs a;
  a.params = params; a.K = K; a.N = p->N; a.dt = p->dt; a.S = p->S; a.Nc = p->Nc; a.Nn = p->Nn; a.n_max = p->n_max;
  a.tH = kMpcMetre / (p->H0 * 1000.0); a.Om = p->Om; a.anchor_end = p->anchor_end;
  a.wc = p->d_wc; a.nodes = p->d_nodes; a.jpl = p->d_jpl; a.status = p->d_status; a.nodeaux = p->d_nodeaux;
  const unsigned aux_grid = (unsigned)(((int64_t)K * p->Nn + 127) / 128);
  if (p->integrator == 1) {
    // the paper's own kind of integrator: adaptive embedded pair, dense output sampled at the coarse nodes
    Dp5Args d;
    d.o = a; d.rtol = p->dp_rtol;
    for (int q = 0; q < 5; ++q) d.atol[q] = p->dp_atol[q];
    d.steps = p->d_dpsteps; d.nsteps = p->d_dpn; d.stop = p->d_dpstop; d.first_bad = p->d_dpbad; d.zero_flag = p->d_dpzero;
    d.cap_long = p->dp_cap;
    orbit_dp5_kernel<<<(K + 31) / 32, 32, 0, s>>>(d);
    DBG("orbit_dp5_kernel");
    orbit_dp5_nodes_kernel<<<aux_grid, 128, 0, s>>>(d);
    DBG("orbit_dp5_nodes_kernel");
    orbit_dp5_finish_kernel<<<aux_grid, 128, 0, s>>>(d);
    p->launches += 3;
    CK(cudaGetLastError());
    return EMRI_OK;
  }
  if (p->orbit_mode == 0) {
    // reference schedule: the whole recursion in one thread per walker
    orbit_kernel<<<(K + 31) / 32, 32, 0, s>>>(a);
    orbit_aux_kernel<<<aux_grid, 128, 0, s>>>(a);
    p->launches += 2;
    CK(cudaGetLastError());
    return EMRI_OK;
  }
  ShootArgs sa;
  sa.o = a; sa.L = p->seg_L; sa.P = p->seg_P; sa.n_steps = p->Nc + 1;
  sa.seg = p->d_seg; sa.mode = p->d_mode; sa.pclamp = p->d_pclamp; sa.plrow = p->d_plrow;
  sa.round = 0; sa.last_round = 0;
  orbit_init_kernel<<<(K + 31) / 32, 64, 0, s>>>(sa);      // two warps per 32 walkers
  DBG("orbit_init_kernel");
  p->launches += 1 + 2 * 3 + 2;
  const int n_rounds = 3;
  for (int r = 0; r < n_rounds; ++r) {
    sa.round = r; sa.last_round = (r == n_rounds - 1);
    const int64_t threads = (int64_t)K * sa.P;
    orbit_sweep_kernel<<<dim3((unsigned)((threads + 63) / 64), r == 0 ? 3 : 1), 64, 0, s>>>(sa);
    DBG("orbit_sweep_kernel");
    orbit_correct_kernel<<<K, 32, (size_t)sa.P * 12 * sizeof(double), s>>>(sa);
    DBG("orbit_correct_kernel");
  }
  orbit_tail_kernel<<<(K + 31) / 32, 32, 0, s>>>(sa);
  DBG("orbit_tail_kernel");
  orbit_fixup_kernel<<<aux_grid, 128, 0, s>>>(sa);      // + the per-node amplitude pair (orbit_aux_kernel's work)
  CK(cudaGetLastError());
  return EMRI_OK;
}

int run_synth(emri_plan* p, int k0, int K, double* outI, double* outII, int64_t pitch, double* outZ, cudaStream_t s) {
  SynthArgs a;
  a.wc = p->d_wc; a.nodes = p->d_nodes; a.nodeaux = p->d_nodeaux; a.jpl = p->d_jpl; a.status = p->d_status;
  a.base = p->d_base; a.tol = p->series_tol;
  a.gtab = p->d_gtab; a.bessel = p->n_max > 48 ? 1 : 0;
  a.cbrt_thr = (p->synth_debug & 2) ? -1.0 : 4e-3;
  a.force_base = (p->synth_debug & 1) ? 1 : 0;
  a.counts = p->d_counts;
  a.k0 = k0; a.K = K; a.N = p->N; a.dt = p->dt; a.S = p->S; a.logS = p->logS; a.Nn = p->Nn; a.n_max = p->n_max;
  a.outI = outI; a.outII = outII; a.pitch = pitch; a.outZ = reinterpret_cast<double2*>(outZ);
  a.tiles_per_walker = (p->N + TILE - 1) / TILE;
  // tiles per unit: 16 measured best on B200 with the per-unit order selection (8: 2-3 % slower, 4: 8 %); fewer only while
  // there is not one unit per resident CTA (tiny calls: one re-expansion per tile makes the producer warp the bottleneck,
  // configs[0]: 39 us at 1 tile per unit, 33 at 2 or 4)
  int ut = UNIT_TILES_MAX;
  while (ut > 1 && (int64_t)K * ((a.tiles_per_walker + ut - 1) / ut) < (int64_t)p->synth_grid) ut >>= 1;
  if (p->unit_tiles_override > 0) ut = p->unit_tiles_override;
  a.unit_tiles = ut;
  a.unit_tiles_cap = p->unit_tiles_cap;
  a.units_per_walker = (a.tiles_per_walker + ut - 1) / ut;
  int64_t total = (int64_t)K * a.units_per_walker;
  int grid = (int)std::min<int64_t>(total, p->synth_grid);
  // S >= 256: every tile lies inside one coarse interval and the producer warp stages its cubics (the default)
  if (a.bessel) {
    if (p->S >= TILE) synth_kernel<true, true><<<grid, SYNTH_BLOCK, p->synth_smem, s>>>(a);
    else synth_kernel<false, true><<<grid, SYNTH_BLOCK, p->synth_smem, s>>>(a);
  } else {
    if (p->S >= TILE) synth_kernel<true, false><<<grid, SYNTH_BLOCK, p->synth_smem, s>>>(a);
    else synth_kernel<false, false><<<grid, SYNTH_BLOCK, p->synth_smem, s>>>(a);
  }
  p->launches += 1;
  CK(cudaGetLastError());
  return EMRI_OK;
}

int fft_chunk(emri_plan* p, int kc, double* z, cudaStream_t s) {
  cufftHandle h;
  int rc = get_fft(p, kc, &h);
  if (rc) return rc;
  CKF(cufftSetStream(h, s));
  CKF(cufftExecZ2Z(h, reinterpret_cast<cufftDoubleComplex*>(z), reinterpret_cast<cufftDoubleComplex*>(z), CUFFT_FORWARD));
  return EMRI_OK;
}

int run_like(emri_plan* p, int k0, int K, const double* Z, const double* data_fft, const double* fcoef, double fstar,
             cudaStream_t s) {
  LikeArgs a;
  a.Z = reinterpret_cast<const double2*>(Z);
  a.D = reinterpret_cast<const double2*>(data_fft);
  a.w = p->d_w; a.partial = p->d_partial; a.k0 = k0; a.K = K; a.N = p->N; a.Nf = p->Nf; a.n_part = p->n_part;
  a.fcoef = fcoef;
  a.f_per_bin = 1.0 / ((double)p->N * p->dt);
  a.x_per_bin = fcoef ? a.f_per_bin / fstar : 0.0;
  dim3 grid((unsigned)p->n_part, (unsigned)((K + LL_GROUP - 1) / LL_GROUP));
  if (fcoef) loglike_kernel<true><<<grid, LL_THREADS, 0, s>>>(a);
  else loglike_kernel<false><<<grid, LL_THREADS, 0, s>>>(a);
  p->launches += 1;
  CK(cudaGetLastError());
  return EMRI_OK;
}

// both transform passes + Eq. 8 of a chunk in its natural layout z[kc][N] (fftlike.cuh: fft2_like_kernel)
constexpr size_t FFT2_SMEM = ((size_t)256 + 512 + FB_ELEMS + FB_ELEMS / 16 + 16) * sizeof(double2);
template <int LG1>
cudaError_t fft2_set_smem_row() {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(fft2_like_kernel<LG1, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT2_SMEM))) return e;
  if ((e = cudaFuncSetAttribute(fft2_like_kernel<LG1, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT2_SMEM))) return e;
  if ((e = cudaFuncSetAttribute(fft2_like_kernel<LG1, 10>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT2_SMEM))) return e;
  if ((e = cudaFuncSetAttribute(fft2_like_kernel<LG1, 11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT2_SMEM))) return e;
  return cudaFuncSetAttribute(fft2_like_kernel<LG1, 12>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT2_SMEM);
}
cudaError_t fft2_set_smem() {
  cudaError_t e;
  if ((e = fft2_set_smem_row<8>())) return e;
  if ((e = fft2_set_smem_row<9>())) return e;
  return fft2_set_smem_row<10>();
}
template <int LG1>
void fft2_launch_row(int lg2, int grid, cudaStream_t s, const Fft2Args& a) {
  switch (lg2) {
    case 8: fft2_like_kernel<LG1, 8><<<grid, FB_THREADS, FFT2_SMEM, s>>>(a); break;
    case 9: fft2_like_kernel<LG1, 9><<<grid, FB_THREADS, FFT2_SMEM, s>>>(a); break;
    case 10: fft2_like_kernel<LG1, 10><<<grid, FB_THREADS, FFT2_SMEM, s>>>(a); break;
    case 11: fft2_like_kernel<LG1, 11><<<grid, FB_THREADS, FFT2_SMEM, s>>>(a); break;
    default: fft2_like_kernel<LG1, 12><<<grid, FB_THREADS, FFT2_SMEM, s>>>(a); break;
  }
}
int run_fft2_like(emri_plan* p, int k0, int kc, const double* z, cudaStream_t s) {
  Fft2Args a;
  a.z = reinterpret_cast<const double2*>(z); a.ring = p->d_ring; a.twid1 = p->d_twid1; a.twid2 = p->d_twid;
  a.tw3 = p->d_tw3; a.alpha = p->d_alpha; a.gamma = p->d_gamma; a.partial = p->d_partial; a.ctr = p->d_fft2ctr;
  a.k0 = k0; a.kc = kc; a.n_part = p->N1; a.N1 = p->N1; a.N2 = p->N2;
  a.N = p->N; a.items = (unsigned)(((int64_t)kc * p->N) / FB_ELEMS);
  CK(cudaMemsetAsync(p->d_fft2ctr, 0, (size_t)2 * sizeof(unsigned), s));
  const int64_t total = (int64_t)2 * a.items;
  const int grid = (int)std::min<int64_t>(total, (int64_t)p->sm_count * 2);
  if (p->log2N1 == 8) fft2_launch_row<8>(p->log2N2, grid, s, a);
  else if (p->log2N1 == 9) fft2_launch_row<9>(p->log2N2, grid, s, a);
  else fft2_launch_row<10>(p->log2N2, grid, s, a);
  p->launches += 1;
  CK(cudaGetLastError());
  return EMRI_OK;
}

bool valid_call(const emri_plan* p, const void* params, int K) { return p && params && K >= 1 && K <= p->K_max; }

}  // namespace

extern "C" {

const char* emri_strerror(int code) {
  switch (code) {
    case EMRI_OK: return "success";
    case EMRI_EINVAL: return "invalid argument";
    case EMRI_ENOMEM: return "out of memory";
    case EMRI_ECUDA: return "CUDA runtime error (see emri_plan_last_cuda_error)";
    case EMRI_ECUFFT: return "cuFFT error (see emri_plan_last_cuda_error)";
    case EMRI_ELIMIT: return "problem larger than the built-in scratch array (EMRI_STATIC_SCRATCH_DOUBLES)";
    default: return "unknown error code";
  }
}

int emri_plan_create(emri_plan** out, int64_t N, double dt, int n_max, int K_max, const double* psd) {
  if (!out) return EMRI_EINVAL;
  *out = nullptr;
  if (N < 4 || (N & 1) || !(dt > 0.0) || !std::isfinite(dt) || n_max < 1 || n_max > EMRI_NMAX_CAP || K_max < 1)
    return EMRI_EINVAL;
  emri_plan* p = new (std::nothrow) emri_plan;
  if (!p) return EMRI_ENOMEM;
  p->N = N; p->Nf = N / 2 + 1; p->dt = dt; p->n_max = n_max; p->K_max = K_max;
  p->chunk = K_max < 128 ? K_max : 128;
  int rc = EMRI_OK;
  auto fail = [&](int code) { int le = p->last_err; emri_plan_destroy(p); (void)le; return code; };
  if (cudaGetDevice(&p->device) != cudaSuccess) return fail(EMRI_ECUDA);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) return fail(EMRI_ECUDA);
  p->sm_count = prop.multiProcessorCount;

  // weights w_m = 1/S_n(f_m), 0 where masked
  std::vector<double> w((size_t)p->Nf, 0.0);
  if (psd)
    for (int64_t m = 0; m < p->Nf; ++m) w[m] = (psd[m] > 0.0 && std::isfinite(psd[m])) ? 1.0 / psd[m] : 0.0;
  std::vector<double4> base;
  build_base_table(n_max, base);

  if ((rc = dev_alloc(p, &p->d_w, (size_t)p->Nf))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_wc, (size_t)K_max * WC_STRIDE))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_jpl, (size_t)K_max))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_status, (size_t)K_max))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_mode, (size_t)K_max))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_pclamp, (size_t)K_max))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_plrow, (size_t)K_max * NODE_STRIDE))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_base, base.size()))) return fail(rc);
  {
    // bracket scale of the Bessel path: n (n/2)^{n-2} / (n-2)! as a running product in long double
    std::vector<double> g((size_t)n_max + 1, 1.0);
    for (int n = 2; n <= n_max; ++n) {
      long double v = (long double)n;
      for (int i = 1; i <= n - 2; ++i) v *= 0.5L * (long double)n / (long double)i;
      g[n] = (double)v;
    }
    if ((rc = dev_alloc(p, &p->d_gtab, g.size()))) return fail(rc);
    if (cudaMemcpy(p->d_gtab, g.data(), g.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess) return fail(EMRI_ECUDA);
  }
  p->n_part = (int)((p->Nf + LL_RANGE - 1) / LL_RANGE);
  // fused transform + reduction (fftlike.cuh): N = 2^16 .. 2^22 = N1 N2
  std::vector<double2> twid;
  if ((N & (N - 1)) == 0 && N >= (1 << 16) && N <= (1 << 22)) {
    int lg = 0;
    while (((int64_t)1 << lg) < N) ++lg;
    // split N = N1 N2 (N1 in 256 .. 1024, N2 in 256 .. 4096): N1 = 512 at one year of samples -- a pass-A ticket is then
    // 8 adjacent columns (128-byte segments) and a pass-B ticket one 4096-point row (measured best on B200)
    p->log2N1 = lg <= 19 ? 8 : (lg <= 21 ? 9 : 10);
    p->log2N2 = lg - p->log2N1;
    p->N2 = 1 << p->log2N2; p->N1 = 1 << p->log2N1;
    p->fused_ok = true;
    p->n_cd = (int)((p->Nf + 255) / 256);
    // stage twiddles of an L-point pass, transposed (fftlike.cuh): W_256^{k t} at [16 t + k], W_L^{jj t} at [256 + t NSL + jj]
    auto stage_twiddles = [](int log2L, std::vector<double2>& tw) {
      const long double tp = -2.0L * 3.14159265358979323846264338327950288L;
      const int L = 1 << log2L, nfull = (log2L - 1) / 4, RL = L >> (4 * nfull), NSL = L / RL;
      tw.resize((size_t)256 + L);
      for (int t = 0; t < 16; ++t)
        for (int k = 0; k < 16; ++k) {
          const long double ang = tp * (long double)(k * t) / 256.0L;
          tw[16 * t + k] = make_double2((double)cosl(ang), (double)sinl(ang));
        }
      for (int t = 0; t < RL; ++t)
        for (int jj = 0; jj < NSL; ++jj) {
          const long double ang = tp * (long double)(((int64_t)jj * t) % L) / (long double)L;
          tw[256 + (size_t)t * NSL + jj] = make_double2((double)cosl(ang), (double)sinl(ang));
        }
    };
    stage_twiddles(p->log2N2, twid);
    {
      std::vector<double2> tw1;
      stage_twiddles(p->log2N1, tw1);
      if ((rc = dev_alloc(p, &p->d_twid1, tw1.size()))) return fail(rc);
      if (cudaMemcpy(p->d_twid1, tw1.data(), tw1.size() * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(EMRI_ECUDA);
    }
    if ((rc = dev_alloc(p, &p->d_twid, twid.size()))) return fail(rc);
    if ((rc = dev_alloc(p, &p->d_alpha, (size_t)N))) return fail(rc);
    if ((rc = dev_alloc(p, &p->d_gamma, (size_t)N))) return fail(rc);
    if ((rc = dev_alloc(p, &p->d_cdpart, (size_t)p->n_cd))) return fail(rc);
    if (cudaMemcpy(p->d_twid, twid.data(), twid.size() * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess)
      return fail(EMRI_ECUDA);
    {
      // three-level table of the inter-pass twiddle: W_N^q, W_N^{128 q} (q < 128), W_N^{16384 q} (q < 256)
      const long double tp = -2.0L * 3.14159265358979323846264338327950288L;
      std::vector<double2> t3(512, make_double2(1.0, 0.0));
      for (int q = 0; q < 512; ++q) {
        const int64_t e = q < 128 ? q : (q < 256 ? (int64_t)128 * (q - 128) : (int64_t)16384 * (q - 256));
        if (e >= N) continue;
        const long double ang = tp * (long double)e / (long double)N;
        t3[q] = make_double2((double)cosl(ang), (double)sinl(ang));
      }
      if ((rc = dev_alloc(p, &p->d_tw3, t3.size()))) return fail(rc);
      if (cudaMemcpy(p->d_tw3, t3.data(), t3.size() * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess) return fail(EMRI_ECUDA);
    }
    if (fft2_set_smem() != cudaSuccess) return fail(EMRI_ECUDA);
  }
  if ((rc = dev_alloc(p, &p->d_partial, (size_t)K_max * std::max(p->n_part, p->N1)))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_params, (size_t)K_max * EMRI_NPAR))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_data, (size_t)4 * p->Nf))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_logL, (size_t)K_max))) return fail(rc);
  // scratch of emri_stretch_step: K/2 <= K_max proposal rows
  const size_t H = (size_t)K_max;
  if ((rc = dev_alloc(p, &p->d_counts, (size_t)SYN_COUNTS))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_Y, H * EMRI_NPAR))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_z, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_lnu, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_logLY, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_inbox, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_partner, H))) return fail(rc);
  if ((rc = alloc_workspace(p))) return fail(rc);
  if ((rc = alloc_chunk(p))) return fail(rc);
  if (cudaMemcpy(p->d_w, w.data(), w.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(p->d_base, base.data(), base.size() * sizeof(double4), cudaMemcpyHostToDevice) != cudaSuccess)
    return fail(EMRI_ECUDA);

  // persistent grid for the synthesis kernel: resident CTAs per SM x SM count
  p->unit_tiles_cap = UNIT_TILES_MAX;
  p->synth_smem = synth_smem_doubles(n_max, p->unit_tiles_cap) * sizeof(double);
  int per_sm = 0, per_sm_direct = 0;
  if (n_max > 48) {
    if (cudaFuncSetAttribute(synth_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->synth_smem) != cudaSuccess ||
        cudaFuncSetAttribute(synth_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->synth_smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, synth_kernel<true, true>, SYNTH_BLOCK, p->synth_smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_direct, synth_kernel<false, true>, SYNTH_BLOCK, p->synth_smem) != cudaSuccess)
      return fail(EMRI_ECUDA);
  } else {
    if (cudaFuncSetAttribute(synth_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->synth_smem) != cudaSuccess ||
        cudaFuncSetAttribute(synth_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->synth_smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, synth_kernel<true, false>, SYNTH_BLOCK, p->synth_smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_direct, synth_kernel<false, false>, SYNTH_BLOCK, p->synth_smem) != cudaSuccess)
      return fail(EMRI_ECUDA);
  }
  if (per_sm < 1 || per_sm_direct < 1) return fail(EMRI_ECUDA);
  per_sm = std::min(per_sm, per_sm_direct);
  p->synth_grid = per_sm * p->sm_count;
  if (cudaStreamCreateWithFlags(&p->s_cap, cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&p->s_copy, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->ev_call, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&p->ev_data, cudaEventDisableTiming) != cudaSuccess)
    return fail(EMRI_ECUDA);
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(EMRI_ECUDA);
  *out = p;
  return EMRI_OK;
}

int emri_plan_destroy(emri_plan* p) {
  if (!p) return EMRI_EINVAL;
  cudaDeviceSynchronize();
  for (auto& kv : p->fft) cufftDestroy(kv.second);
  for (auto e : p->ev) cudaEventDestroy(e);
  if (p->ev_call) cudaEventDestroy(p->ev_call);
  if (p->ev_data) cudaEventDestroy(p->ev_data);
  drop_graphs(p);
  if (p->s_cap) cudaStreamDestroy(p->s_cap);
  if (p->s_copy) cudaStreamDestroy(p->s_copy);
  void* ptrs[] = {p->d_w, p->d_wc, p->d_nodes, p->d_hbuf, p->d_partial, p->d_base, p->d_nodeaux, p->d_jpl, p->d_status,
                  p->d_params, p->d_data, p->d_logL, p->d_Y, p->d_z, p->d_lnu, p->d_logLY, p->d_inbox,
                  p->d_partner, p->d_fftwork, p->d_seg, p->d_plrow, p->d_mode, p->d_pclamp, p->d_counts,
                  p->d_twid, p->d_twid1, p->d_tw3, p->d_ring, p->d_fft2ctr, p->d_alpha, p->d_gamma, p->d_cdpart, p->d_gtab, p->d_dpsteps, p->d_dpn, p->d_dpstop,
                  p->d_dpbad, p->d_dpzero};
  for (void* q : ptrs) if (q) cudaFree(q);
  delete p;
  return EMRI_OK;
}

int emri_plan_set_cosmology(emri_plan* p, double H0, double Om) {
  if (!p || !(H0 > 0.0) || !(Om > 0.0) || !(Om <= 1.0) || !std::isfinite(H0)) return EMRI_EINVAL;
  drop_graphs(p);
  p->H0 = H0; p->Om = Om;
  return EMRI_OK;
}

int emri_plan_set_coarse_stride(emri_plan* p, int S) {
  if (!p || S < 2 || S > 65536 || (S & (S - 1))) return EMRI_EINVAL;
  drop_graphs(p);
  CK(cudaDeviceSynchronize());
  p->S = S;
  p->logS = 0;
  while ((1 << p->logS) < S) ++p->logS;
  if (p->d_nodes) p->bytes -= (int64_t)((size_t)p->K_max * p->Nn * NODE_STRIDE * sizeof(double));
  if (p->d_seg) p->bytes -= (int64_t)((size_t)p->K_max * p->seg_P * SEG_STRIDE * sizeof(double));
  if (p->d_nodeaux) p->bytes -= (int64_t)((size_t)p->K_max * p->Nn * sizeof(double2));
  return alloc_workspace(p);
}

int emri_plan_set_orbit_schedule(emri_plan* p, int schedule) {
  if (!p || (schedule != 0 && schedule != 1)) return EMRI_EINVAL;
  drop_graphs(p);
  p->orbit_mode = schedule;
  p->orbit_ran = false;
  return EMRI_OK;
}

int emri_plan_set_anchor(emri_plan* p, int at_lso) {
  if (!p || (at_lso != 0 && at_lso != 1)) return EMRI_EINVAL;
  drop_graphs(p);
  p->anchor_end = at_lso;
  return EMRI_OK;
}

int emri_plan_orbit_report(emri_plan* p, int K, int32_t* modes) {
  if (!p || !modes || K < 1 || K > p->K_max) return EMRI_EINVAL;
  // d_mode is written by the parallel-in-time RK4 schedule only: refuse to hand out leftovers of another configuration
  if (p->integrator != 0 || p->orbit_mode != 1 || !p->orbit_ran) return EMRI_EINVAL;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpy(modes, p->d_mode, (size_t)K * sizeof(int32_t), cudaMemcpyDeviceToHost));
  return EMRI_OK;
}

int emri_plan_synth_report(emri_plan* p, int64_t counts[16]) {
  if (!p || !counts) return EMRI_EINVAL;
  CK(cudaDeviceSynchronize());
  unsigned long long h[SYN_COUNTS];
  CK(cudaMemcpy(h, p->d_counts, sizeof(h), cudaMemcpyDeviceToHost));
  for (int i = 0; i < 16; ++i) counts[i] = i < SYN_COUNTS ? (int64_t)h[i] : 0;
  return EMRI_OK;
}

int emri_plan_set_integrator(emri_plan* p, int kind, double rtol, const double* atol, int max_steps) {
  if (!p || (kind != 0 && kind != 1)) return EMRI_EINVAL;
  drop_graphs(p);
  p->orbit_ran = false;
  if (kind == 0) { p->integrator = 0; return EMRI_OK; }
  if (!(rtol > 0.0) || !std::isfinite(rtol) || !atol || max_steps < 16) return EMRI_EINVAL;
  for (int q = 0; q < 5; ++q) if (!(atol[q] >= 0.0) || !std::isfinite(atol[q])) return EMRI_EINVAL;
  CK(cudaDeviceSynchronize());
  int rc;
  if (max_steps != p->dp_cap || !p->d_dpsteps) {
    if (p->d_dpsteps) p->bytes -= (int64_t)((size_t)p->K_max * (p->dp_cap + DP_SHORT) * DP_REC * sizeof(double));
    p->dp_cap = max_steps;
    if ((rc = dev_alloc(p, &p->d_dpsteps, (size_t)p->K_max * (p->dp_cap + DP_SHORT) * DP_REC))) { p->dp_cap = 0; return rc; }
  }
  if (!p->d_dpn) {
    if ((rc = dev_alloc(p, &p->d_dpn, (size_t)2 * p->K_max))) return rc;
    if ((rc = dev_alloc(p, &p->d_dpstop, (size_t)2 * p->K_max))) return rc;
    if ((rc = dev_alloc(p, &p->d_dpbad, (size_t)p->K_max))) return rc;
    if ((rc = dev_alloc(p, &p->d_dpzero, (size_t)p->K_max))) return rc;
  }
  p->dp_rtol = rtol;
  for (int q = 0; q < 5; ++q) p->dp_atol[q] = atol[q];
  p->integrator = 1;
  return EMRI_OK;
}

int emri_plan_orbit_steps(emri_plan* p, int k, int branch, int max_out, double* t, double* h, double* y, int32_t* info) {
  if (!p || p->integrator != 1 || !p->orbit_ran || k < 0 || k >= p->K_max || (branch != 0 && branch != 1) || max_out < 0 || !info)
    return EMRI_EINVAL;
  CK(cudaDeviceSynchronize());
  int32_t n[2], st[2];
  CK(cudaMemcpy(n, p->d_dpn + 2 * k, sizeof(n), cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(st, p->d_dpstop + 2 * k, sizeof(st), cudaMemcpyDeviceToHost));
  info[0] = n[branch]; info[1] = st[branch];
  const bool is_long = (branch == 0) != (p->anchor_end != 0);
  const size_t base = ((size_t)k * (p->dp_cap + DP_SHORT) + (is_long ? 0 : p->dp_cap)) * DP_REC;
  const int cnt = std::min(max_out, (int)n[branch]);
  std::vector<double> rec((size_t)cnt * DP_REC);
  if (cnt > 0) CK(cudaMemcpy(rec.data(), p->d_dpsteps + base, rec.size() * sizeof(double), cudaMemcpyDeviceToHost));
  for (int i = 0; i < cnt; ++i) {
    if (t) t[i] = rec[(size_t)i * DP_REC];
    if (h) h[i] = rec[(size_t)i * DP_REC + 1];
    if (y) for (int q = 0; q < 5; ++q) y[5 * i + q] = rec[(size_t)i * DP_REC + 2 + q];
  }
  return EMRI_OK;
}

int emri_plan_set_unit_tiles(emri_plan* p, int tiles) {
  if (!p || tiles < 0 || tiles > UNIT_TILES_MAX || (tiles & (tiles - 1))) return EMRI_EINVAL;
  drop_graphs(p);
  p->unit_tiles_override = tiles;
  return EMRI_OK;
}

int emri_plan_set_transform(emri_plan* p, int fused) {
  if (!p || (fused != 0 && fused != 1)) return EMRI_EINVAL;
  drop_graphs(p);
  p->fused_on = fused != 0;
  return EMRI_OK;
}

int emri_plan_transform_is_fused(const emri_plan* p) { return (p && p->fused_ok && p->fused_on) ? 1 : 0; }

int emri_plan_set_series_tolerance(emri_plan* p, double tol) {
  if (!p || !(tol >= 1e-17) || !(tol <= 1e-10)) return EMRI_EINVAL;
  drop_graphs(p);
  p->series_tol = tol;
  return EMRI_OK;
}

int emri_plan_set_synth_debug(emri_plan* p, int flags) {
  if (!p || flags < 0 || flags > 3) return EMRI_EINVAL;
  drop_graphs(p);
  p->synth_debug = flags;
  return EMRI_OK;
}

int emri_plan_set_chunk(emri_plan* p, int c) {
  if (!p || c < 1) return EMRI_EINVAL;
  drop_graphs(p);
  if (c > p->K_max) c = p->K_max;
  CK(cudaDeviceSynchronize());
  if (p->d_hbuf) p->bytes -= (int64_t)((size_t)2 * p->chunk * p->N * sizeof(double));
  if (p->d_ring) p->bytes -= (int64_t)((size_t)p->chunk * p->N * sizeof(double2) + (size_t)2 * sizeof(unsigned));
  p->chunk = c;
  return alloc_chunk(p);
}

int64_t emri_plan_num_nodes(const emri_plan* p) { return p ? p->Nn : 0; }

int emri_orbit(emri_plan* p, const double* params, int K, double* nodes, int32_t* status, void* stream) {
  if (!valid_call(p, params, K) || !nodes) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  int rc = run_orbit(p, params, K, s);
  if (rc) return rc;
  CK(cudaMemcpyAsync(nodes, p->d_nodes, (size_t)K * p->Nn * NODE_STRIDE * sizeof(double), cudaMemcpyDeviceToDevice, s));
  if (status) {
    copy_status_kernel<<<(K + 127) / 128, 128, 0, s>>>(p->d_status, status, K);
    CK(cudaGetLastError());
  }
  return EMRI_OK;
}

int emri_waveform(emri_plan* p, const double* params, int K, double* h_I, double* h_II, int32_t* status, void* stream) {
  if (!valid_call(p, params, K) || !h_I || !h_II) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  p->ev_used = 0; p->n_chunks_last = 1; p->had_like = false;
  mark(p, s);
  int rc = run_orbit(p, params, K, s);
  if (rc) return rc;
  mark(p, s);
  mark(p, s);
  if ((rc = run_synth(p, 0, K, h_I, h_II, p->N, nullptr, s))) return rc;
  mark(p, s);
  mark(p, s);
  mark(p, s);
  if (status) {
    copy_status_kernel<<<(K + 127) / 128, 128, 0, s>>>(p->d_status, status, K);
    CK(cudaGetLastError());
  }
  return EMRI_OK;
}

int emri_waveform_fft(emri_plan* p, const double* params, int K, double* spectra, int32_t* status, void* stream) {
  if (!valid_call(p, params, K) || !spectra) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  p->ev_used = 0; p->had_like = false;
  mark(p, s);
  int rc = run_orbit(p, params, K, s);
  if (rc) return rc;
  mark(p, s);
  int nch = 0;
  for (int k0 = 0; k0 < K; k0 += p->chunk, ++nch) {
    const int kc = std::min(p->chunk, K - k0);
    mark(p, s);
    if ((rc = run_synth(p, k0, kc, nullptr, nullptr, 0, p->d_hbuf, s))) return rc;
    mark(p, s);
    if ((rc = fft_chunk(p, kc, p->d_hbuf, s))) return rc;
    {
      const int64_t tot = (int64_t)kc * p->Nf;
      unpack_spectrum_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(
          reinterpret_cast<const double2*>(p->d_hbuf), reinterpret_cast<double2*>(spectra) + (size_t)k0 * 2 * p->Nf, kc, p->N, p->Nf);
      CK(cudaGetLastError());
    }
    mark(p, s);
    mark(p, s);
  }
  p->n_chunks_last = nch;
  if (status) {
    copy_status_kernel<<<(K + 127) / 128, 128, 0, s>>>(p->d_status, status, K);
    CK(cudaGetLastError());
  }
  return EMRI_OK;
}

int emri_data_fft(emri_plan* p, const double* d_I, const double* d_II, double* data_fft, void* stream) {
  if (!p || !d_I || !d_II || !data_fft) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  pack_complex_kernel<<<(unsigned)((p->N + 255) / 256), 256, 0, s>>>(d_I, d_II, reinterpret_cast<double2*>(p->d_hbuf), p->N);
  CK(cudaGetLastError());
  int rc = fft_chunk(p, 1, p->d_hbuf, s);
  if (rc) return rc;
  unpack_spectrum_kernel<<<(unsigned)((p->Nf + 255) / 256), 256, 0, s>>>(reinterpret_cast<const double2*>(p->d_hbuf),
                                                                         reinterpret_cast<double2*>(data_fft), 1, p->N, p->Nf);
  CK(cudaGetLastError());
  return EMRI_OK;
}

static int loglike_enqueue(emri_plan* p, const double* params, int K, const double* fcoef, double fstar, const double* data_fft,
                           double* logL, int32_t* status, cudaStream_t s);

// emri_loglike / emri_loglike_fdep: replay the CUDA graph of this argument set if the plan holds one, else capture it (on
// the plan's own stream: the caller's may be the legacy default stream) and launch it into the caller's stream.  Plain
// enqueueing when graphs are off, stage timings are on, the call is the host variant's (it waits on the copy stream), or
// capture fails for any reason.
static int loglike_impl(emri_plan* p, const double* params, int K, const double* fcoef, double fstar, const double* data_fft,
                        double* logL, int32_t* status, void* stream) {
  if (!valid_call(p, params, K) || !data_fft || !logL) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  static const bool dbg = std::getenv("EMRI_DEBUG_SYNC") != nullptr;
  if (!p->graphs_on || p->timing || p->wait_before_like || dbg || !p->s_cap)
    return loglike_enqueue(p, params, K, fcoef, fstar, data_fft, logL, status, s);
  for (auto& g : p->graphs)
    if (g.params == params && g.data == data_fft && g.logL == logL && g.status == status && g.fcoef == fcoef && g.K == K &&
        g.fstar == fstar) {
      CK(cudaGraphLaunch(g.exec, s));
      g.used = ++p->graph_clock;
      p->launches = g.launches; p->n_chunks_last = g.n_chunks; p->had_like = true; p->ev_used = 0;
      ++p->graph_replays;
      return EMRI_OK;
    }
  // every cuFFT plan the call needs must exist before the capture starts (plan creation cannot be captured)
  {
    const bool fused = p->fused_ok && p->fused_on && !fcoef;
    cufftHandle h;
    int rc;
    for (int k0 = 0; k0 < K && !fused; k0 += p->chunk) {
      const int kc = std::min(p->chunk, K - k0);
      if ((rc = get_fft(p, kc, &h))) return rc;
    }
  }
  cudaGraph_t graph = nullptr;
  if (cudaStreamBeginCapture(p->s_cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    return loglike_enqueue(p, params, K, fcoef, fstar, data_fft, logL, status, s);
  }
  const int rc = loglike_enqueue(p, params, K, fcoef, fstar, data_fft, logL, status, p->s_cap);
  const cudaError_t ec = cudaStreamEndCapture(p->s_cap, &graph);
  cudaGraphExec_t exec = nullptr;
  if (rc != EMRI_OK || ec != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    if (rc != EMRI_OK) return rc;
    return loglike_enqueue(p, params, K, fcoef, fstar, data_fft, logL, status, s);
  }
  cudaGraphDestroy(graph);
  if (p->graphs.size() >= 8) {            // keep a few: evict the least recently used
    size_t lru = 0;
    for (size_t i = 1; i < p->graphs.size(); ++i) if (p->graphs[i].used < p->graphs[lru].used) lru = i;
    cudaGraphExecDestroy(p->graphs[lru].exec);
    p->graphs.erase(p->graphs.begin() + (long)lru);
  }
  p->graphs.push_back({params, data_fft, logL, status, fcoef, K, fstar, exec, p->launches, p->n_chunks_last, ++p->graph_clock});
  ++p->graph_captures;
  CK(cudaGraphLaunch(exec, s));
  return EMRI_OK;
}

static int loglike_enqueue(emri_plan* p, const double* params, int K, const double* fcoef, double fstar, const double* data_fft,
                           double* logL, int32_t* status, cudaStream_t s) {
  p->ev_used = 0; p->had_like = true;
  mark(p, s);
  int rc = run_orbit(p, params, K, s);
  if (rc) return rc;
  mark(p, s);
  int nch = 0;
  const double scale = 2.0 * p->dt / (double)p->N;
  if (p->fused_ok && p->fused_on && !fcoef) {
    // fused path (fftlike.cuh): ONE kernel of this library does both transform passes and Eq. 8
    for (int k0 = 0; k0 < K; k0 += p->chunk, ++nch) {
      const int kc = std::min(p->chunk, K - k0);
      mark(p, s);
      if ((rc = run_synth(p, k0, kc, nullptr, nullptr, 0, p->d_hbuf, s))) return rc;
      mark(p, s);
      mark(p, s);
      if (nch == 0) {
        // the weights of Eq. 8 in pass-B order, from the caller's data spectrum (the only reader of data_fft)
        if (p->wait_before_like) { CK(cudaStreamWaitEvent(s, p->wait_before_like, 0)); p->wait_before_like = nullptr; }
        like_weights_kernel<<<p->n_cd, 256, 0, s>>>(reinterpret_cast<const double2*>(data_fft), p->d_w, p->N, p->Nf, p->N1,
                                                    p->log2N1, p->N2, p->d_alpha, p->d_gamma, p->d_cdpart);
        p->launches += 1;
        CK(cudaGetLastError());
      }
      if ((rc = run_fft2_like(p, k0, kc, p->d_hbuf, s))) return rc;
      mark(p, s);
    }
    p->n_chunks_last = nch;
    fftlike_final_kernel<<<(K + 3) / 4, 128, 0, s>>>(p->d_partial, p->N1, p->d_cdpart, p->n_cd, K, scale, p->d_status, logL,
                                                     status);
    p->launches += 1;
    CK(cudaGetLastError());
    return EMRI_OK;
  }
  for (int k0 = 0; k0 < K; k0 += p->chunk, ++nch) {
    const int kc = std::min(p->chunk, K - k0);
    mark(p, s);
    if ((rc = run_synth(p, k0, kc, nullptr, nullptr, 0, p->d_hbuf, s))) return rc;
    mark(p, s);
    if ((rc = fft_chunk(p, kc, p->d_hbuf, s))) return rc;
    mark(p, s);
    if (p->wait_before_like) { CK(cudaStreamWaitEvent(s, p->wait_before_like, 0)); p->wait_before_like = nullptr; }
    if ((rc = run_like(p, k0, kc, p->d_hbuf, data_fft, fcoef, fstar, s))) return rc;
    mark(p, s);
  }
  p->n_chunks_last = nch;
  loglike_final_kernel<<<(K + 3) / 4, 128, 0, s>>>(p->d_partial, p->n_part, K, scale, p->d_status, logL, status);
  p->launches += 1;
  CK(cudaGetLastError());
  return EMRI_OK;
}

int emri_loglike(emri_plan* p, const double* params, int K, const double* data_fft, double* logL, int32_t* status,
                 void* stream) {
  return loglike_impl(p, params, K, nullptr, 1.0, data_fft, logL, status, stream);
}

int emri_loglike_fdep(emri_plan* p, const double* params, int K, const double* fcoef, double f_star, const double* data_fft,
                      double* logL, int32_t* status, void* stream) {
  if (!fcoef || !(f_star > 0.0) || !std::isfinite(f_star)) return EMRI_EINVAL;
  return loglike_impl(p, params, K, fcoef, f_star, data_fft, logL, status, stream);
}

int emri_loglike_host(emri_plan* p, const double* params, int K, const double* data_fft, double* logL, int32_t* status,
                      void* stream) {
  if (!valid_call(p, params, K) || !logL) return EMRI_EINVAL;
  if (!data_fft && !p->data_loaded) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaMemcpyAsync(p->d_params, params, (size_t)K * EMRI_NPAR * sizeof(double), cudaMemcpyHostToDevice, s));
  if (data_fft) {
    // upload on the copy stream, ordered after everything already enqueued on s (an earlier reader of d_data);
    // the reduction kernel, the only reader, waits for it -- the orbit, synthesis and transform do not
    CK(cudaEventRecord(p->ev_call, s));
    CK(cudaStreamWaitEvent(p->s_copy, p->ev_call, 0));
    CK(cudaMemcpyAsync(p->d_data, data_fft, (size_t)4 * p->Nf * sizeof(double), cudaMemcpyHostToDevice, p->s_copy));
    CK(cudaEventRecord(p->ev_data, p->s_copy));
    p->wait_before_like = p->ev_data;
    p->data_loaded = true;
  }
  int rc = emri_loglike(p, p->d_params, K, p->d_data, p->d_logL, nullptr, stream);
  p->wait_before_like = nullptr;
  if (rc) return rc;
  CK(cudaMemcpyAsync(logL, p->d_logL, (size_t)K * sizeof(double), cudaMemcpyDeviceToHost, s));
  if (status) CK(cudaMemcpyAsync(status, p->d_status, (size_t)K * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return EMRI_OK;
}

int emri_plan_set_graphs(emri_plan* p, int on) {
  if (!p || (on != 0 && on != 1)) return EMRI_EINVAL;
  p->graphs_on = on != 0;
  if (!on) drop_graphs(p);
  return EMRI_OK;
}

int emri_plan_graph_stats(const emri_plan* p, int64_t out[2]) {
  if (!p || !out) return EMRI_EINVAL;
  out[0] = p->graph_captures; out[1] = p->graph_replays;
  return EMRI_OK;
}

int emri_plan_enable_timings(emri_plan* p, int on) {
  if (!p) return EMRI_EINVAL;
  p->timing = on != 0;
  p->ev_used = 0;
  return EMRI_OK;
}

int emri_plan_get_timings(emri_plan* p, double ms[4]) {
  if (!p || !ms) return EMRI_EINVAL;
  ms[0] = ms[1] = ms[2] = ms[3] = 0.0;
  if (!p->timing || p->ev_used < 2) return EMRI_OK;
  CK(cudaEventSynchronize(p->ev[p->ev_used - 1]));
  float t = 0.f;
  CK(cudaEventElapsedTime(&t, p->ev[0], p->ev[1]));
  ms[0] = t;
  for (int c = 0; c < p->n_chunks_last; ++c) {
    const int b = 2 + 4 * c;
    if (b + 3 >= p->ev_used) break;
    CK(cudaEventElapsedTime(&t, p->ev[b], p->ev[b + 1])); ms[1] += t;
    CK(cudaEventElapsedTime(&t, p->ev[b + 1], p->ev[b + 2])); ms[2] += t;
    CK(cudaEventElapsedTime(&t, p->ev[b + 2], p->ev[b + 3])); ms[3] += t;
  }
  return EMRI_OK;
}

int emri_plan_last_cuda_error(const emri_plan* p) { return p ? p->last_err : 0; }
int emri_plan_last_launch_count(const emri_plan* p) { return p ? p->launches : 0; }
int64_t emri_plan_workspace_bytes(const emri_plan* p) { return p ? p->bytes : 0; }

int emri_stretch_step(emri_plan* p, double* X, double* logL, int K, const double* data_fft, const double* lo,
                      const double* hi, double a_stretch, uint64_t seed, int64_t step, int half, int32_t* accepted,
                      double* log_buf, void* stream) {
  if (!p || !X || !logL || !data_fft || !lo || !hi || K < 2 || (K & 1) || K / 2 > p->K_max || !(a_stretch > 1.0) ||
      (half != 0 && half != 1))
    return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  StretchArgs a;
  a.X = X; a.logL = logL; a.K = K; a.lo = lo; a.hi = hi; a.a = a_stretch; a.seed = seed; a.step = step; a.half = half;
  a.Y = p->d_Y; a.zbuf = p->d_z; a.lnu = p->d_lnu; a.inbox = p->d_inbox; a.partner = p->d_partner; a.logLY = p->d_logLY;
  a.accepted = accepted; a.log_buf = log_buf;
  const int H = K / 2;
  stretch_propose_kernel<<<(H + 127) / 128, 128, 0, s>>>(a);
  CK(cudaGetLastError());
  int rc = emri_loglike(p, p->d_Y, H, data_fft, p->d_logLY, nullptr, stream);
  if (rc) return rc;
  stretch_accept_kernel<<<(H + 127) / 128, 128, 0, s>>>(a);
  CK(cudaGetLastError());
  return EMRI_OK;
}

}  // extern "C"

