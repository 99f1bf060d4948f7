/* emri.h -- C ABI of the B200-native (sm_100a) hot path of EMRI_MC (arXiv 2311.17174).
 *
 * The library evaluates, for a whole MCMC ensemble of K walkers at once (PAPER.md:57, :122, :146:
 * "a matrix (n_walkers x n_dim) ... computed in a vectorised manner"), the Analytic-Kludge EMRI
 * waveform (Eqs. 1-2), its projection on the two LISA channels,
 * the modified-gravity propagation factors (Eqs. 4-6), its discrete Fourier
 * transform and the noise-weighted Gaussian log-likelihood (PAPER.md:112-116,
 * Eq. 8).  The equations the paper defers to Barack & Cutler 2004 and Peters & Mathews 1963 are
 * restated in DESIGN.md section 3.
 *
 * Conventions
 *  - "DEV" pointers are CUDA device pointers on the plan's device, "HOST" pointers are host memory.
 *    The caller owns every pointer it passes; the plan owns its workspace.
 *  - Every call that takes `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default
 *    stream) only ENQUEUES work on that stream and returns; it never synchronises.  Results are
 *    valid after the stream reaches the end of the enqueued work.  The *_host variants copy with
 *    cudaMemcpyAsync on the same stream and DO synchronise the stream before returning.
 *  - One plan must not be used from two streams concurrently (the workspace is shared).
 *  - All functions return EMRI_OK (0) or a negative error code; they never throw or exit.
 *  - EMRI_DEBUG_SYNC=1 in the environment makes stage (a) synchronise after each of its kernels and name on stderr
 *    the one that failed (debugging aid; off by default).
 *
 * Parameter row, P = EMRI_NPAR = 17 doubles per walker, row-major params[K][17]
 * (first three are M, mu, S/M^2 as PAPER.md:149 prescribes):
 *    0 M      central mass, detector frame [Msun]     9  theta_S  source colatitude [rad]
 *    1 mu     small mass [Msun]                       10 phi_S    source azimuth    [rad]
 *    2 a      spin S/M^2, |a| <= 1                    11 theta_K  spin colatitude   [rad]
 *    3 e0     eccentricity at t = 0, [0,1)            12 phi_K    spin azimuth      [rad]
 *    4 nu0    orbital frequency at t = 0 [Hz]         13 D_L      EM luminosity distance [Gpc]
 *    5 Phi0   mean anomaly at t = 0 [rad]             14 Xi0      Eq. 6
 *    6 gam0   gamma~ at t = 0 [rad]                   15 n_Xi     Eq. 6
 *    7 alp0   alpha at t = 0 [rad]                    16 delta_T  c_T - 1 (GW speed excess)
 *    8 lambda angle between L and S [rad]
 *
 * Per-walker status bits (not errors; written to `status[K]` when it is not NULL):
 *    1 EMRI_ST_BADPARAM  non-finite or out-of-domain parameter (M, mu, D_L, nu0 <= 0, e0 not in
 *                        [0,1), |a| > 1, Xi(z) <= 0)
 *    2 EMRI_ST_PLUNGE    nu reached nu_LSO(e) inside the window; the waveform is
 *                        zero from the first plunged coarse node on; logL uses the truncated wave
 *    4 EMRI_ST_DELAY     |Delta T| exceeds one coarse interval (the guard)
 *    8 EMRI_ST_STATE     e left [0,1) or the state became non-finite during the integration
 * For bits 1, 4, 8 the waveform rows are zero and logL = -inf.
 */
#ifndef EMRI_H
#define EMRI_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EMRI_NPAR 17
#define EMRI_NMAX_CAP 128 /* largest n_max a plan accepts */

enum {
  EMRI_OK = 0,
  EMRI_EINVAL = -1, /* bad argument (NULL pointer, K > K_max, N odd or < 4, n_max out of range ...) */
  EMRI_ENOMEM = -2, /* host or device allocation failed */
  EMRI_ECUDA = -3,  /* a CUDA runtime call failed; see emri_plan_last_cuda_error */
  EMRI_ECUFFT = -4, /* a cuFFT call failed; see emri_plan_last_cuda_error */
  EMRI_ELIMIT = -5  /* the problem is larger than the library's built-in scratch array (emri_spectra_loglike_static) */
};

enum { EMRI_ST_BADPARAM = 1, EMRI_ST_PLUNGE = 2, EMRI_ST_DELAY = 4, EMRI_ST_STATE = 8 };

typedef struct emri_plan emri_plan;

/* Static description of an error code. */
const char* emri_strerror(int code);

/* Create a plan for N samples at spacing dt [s], harmonics n = 1..n_max (Eq. 2), at
 * most K_max walkers per call.  psd: HOST, N/2+1 values of the one-sided noise PSD S_n(f_m) [1/Hz]
 * at f_m = m/(N dt) (Eq. 8's S_noise); entries that are <= 0, NaN or +inf mask
 * their bin (weight 0); pass +inf at m = 0 and m = N/2 to exclude DC and Nyquist.  psd may be NULL
 * (all weights 0; only emri_waveform / emri_data_fft are then meaningful).
 * Requirements: N even, N >= 4; dt > 0; 1 <= n_max <= EMRI_NMAX_CAP; K_max >= 1.
 * Uses the current CUDA device; synchronises it.  Defaults: flat LambdaCDM H0 = 67.4 km/s/Mpc,
 * Omega_m = 0.315 (the paper's dL() leaves the cosmology open); coarse stride
 * S = 256 samples. */
int emri_plan_create(emri_plan** out, int64_t N, double dt, int n_max, int K_max, const double* psd);

/* Free everything the plan owns (synchronises the device). */
int emri_plan_destroy(emri_plan* p);

/* Background cosmology behind z(D_L) and the look-back time. */
int emri_plan_set_cosmology(emri_plan* p, double H0_km_s_Mpc, double Omega_m);

/* Coarse-grid stride S in samples (power of two, 2 <= S <= 65536): the RK4 step of the orbital
 * ODEs (Eq. 1) is S*dt.  Reallocates the orbit workspace; synchronises. */
int emri_plan_set_coarse_stride(emri_plan* p, int S);

/* How stage (a) is scheduled on the device.  1 (default): parallel in time -- multiple shooting
 * over segments of the coarse grid with a Newton correction and verification, which reproduces the
 * sequential RK4 recursion to ~1e-18 relative in (nu, e).  0: the plain
 * sequential recursion, one thread per walker (latency-bound; kept as the in-library reference of
 * the schedule and used by the tests).  Both evaluate the same scheme (S3). */
int emri_plan_set_orbit_schedule(emri_plan* p, int schedule);

/* Which integrator stage (a) uses.  kind 0 (default): the fixed-step RK4 of BASELINE.json's north_star (the two schedules
 * above).  kind 1: the paper's own kind of integrator ("standard ODE methods, such as the 7th-order
 * Runge-Kutta scheme", :133 solve_ivp, :157; reading D14) -- an embedded Runge-Kutta pair with per-walker step
 * control and dense output on the device: Dormand-Prince 5(4), the step-size controller solve_ivp uses (error norm = rms
 * over the five components of err / (atol + rtol max(|Y|, |Y_new|)), angles counted in unwrapped cycles), Shampine's
 * continuous extension.  The dense output is sampled at the coarse nodes (value; slope = right-hand side at the node;
 * unwrapped increment), so every later stage is unchanged.  rtol > 0; atol: HOST [5] for (Phi [cycles], nu [Hz],
 * gamma~ [cycles], e, alpha [cycles]); max_steps: accepted steps kept per walker (>= 16; a walker that needs more gets
 * EMRI_ST_STATE).  Allocates K_max (max_steps + 64) 256 B of step records; synchronises.  Works with both anchors. */
int emri_plan_set_integrator(emri_plan* p, int kind, double rtol, const double* atol, int max_steps);

/* Diagnostics of the last adaptive orbit (kind 1): the accepted steps of walker k's branch (0: forward from the anchor,
 * 1: backward).  t, h: HOST [max_out] start and signed size of each step; y: HOST [max_out][5] state at the start (angles
 * wrapped, cycles), any of them may be NULL; info: HOST int32 [2] = {steps taken, 0 / EMRI_ST_PLUNGE / EMRI_ST_STATE why
 * the branch ended early}.  Synchronises.  EMRI_EINVAL unless the adaptive integrator is selected and stage (a) has run since
 * it was selected. */
int emri_plan_orbit_steps(emri_plan* p, int k, int branch, int max_out, double* t, double* h, double* y, int32_t* info);

/* Where the orbital state of the parameter row is given.  0 (default): at the first sample, t = 0, integrated forward.
 * 1: the paper's own convention ("initial conditions at the LSO ... integrated backwards"): the row's
 * e0, Phi0, gam0, alp0 are the values AT PLUNGE, placed at the last coarse node t = ceil(N/S) S dt (the end of the window),
 * nu there is nu_LSO(e0) = ((1-e0^2)/(6+2 e0))^{3/2} / (2 pi M) (column nu0 is ignored but must be positive), and the
 * same fixed-step RK4 runs backwards.  Nothing plunges inside the window; if e leaves [0,1) on the way back the
 * walker gets EMRI_ST_STATE (zero rows, logL = -inf).  Applies to every later call of the plan. */
int emri_plan_set_anchor(emri_plan* p, int at_lso);

/* Diagnostics of the last parallel-in-time orbit evaluation: modes[k] (HOST int32 [K]) is 1 if
 * walker k's segments were all verified after a Newton round, 2 if a sequential tail was needed
 * from the first unverified boundary, 3 if its node rows are zero (invalid parameters, plunge at
 * t = 0, bad guard step).  Synchronises the device.  EMRI_EINVAL unless the plan is on the fixed-step integrator with
 * schedule 1 and stage (a) has run since that was last set (the modes of another configuration would be leftovers). */
int emri_plan_orbit_report(emri_plan* p, int K, int32_t* modes);

/* Diagnostics of stage (b) over the last emri_waveform / emri_waveform_fft / emri_loglike* call (all chunks):
 * which evaluation path the data selected.  counts (HOST int64 [16]):
 *   [0] units (one walker x up to 16 tiles of 256 samples) synthesised, [1..8] of them by the local order kept in the
 *   re-summed harmonic series (first harmonic range), [9] units that fell back to the base series in e^2 (local order 8 still significant),
 *   [10] samples whose amplitude (2 pi M nu)^{2/3} took the cube root instead of the Taylor series about the coarse
 *   node (|nu/nu_j - 1| > 4e-3), [11] units of walkers with a fatal status (zero-filled), [12] sum over units of the harmonics evaluated (the last
 *   harmonic with a term above the truncation threshold, <= n_max), [13] of those, the harmonics of the first order range,
 *   [14] sum over units of the second range's order, [15] 0.
 * Synchronises the device. */
int emri_plan_synth_report(emri_plan* p, int64_t counts[16]);

/* How emri_loglike runs stages (c)+(d).  1 (default where available: N a power of two, 2^16 <= N <= 2^22): fused -- ONE
 * persistent kernel of this library does both passes of the transform, N = N1 N2 (N1-point transforms down the columns of
 * the chunk the synthesis wrote, then N2 <= 4096 points per row, in registers and shared memory) and feeds the outputs of
 * the last pass straight into Eq. 8, so the spectrum is never written back nor read again and cuFFT is not on the path
 * (DESIGN.md section 6c).  Needs a second chunk-sized buffer.  0: the full cuFFT transform followed by
 * the streaming reduction kernel (also used for every other N and by emri_loglike_fdep).  Both give logL within the parity
 * tolerance of each other (not bit-identical: the fused path sums alpha_j |Z_j - ZD_j|^2 over the single elements of the
 * packed transform, the same squared residuals in another order; both give logL = 0 at a noise-free injection).
 * emri_plan_transform_is_fused reports what the next emri_loglike will do. */
int emri_plan_set_transform(emri_plan* p, int fused);
int emri_plan_transform_is_fused(const emri_plan* p);

/* CUDA graphs.  1 (default): emri_loglike / emri_loglike_fdep (and the likelihood inside emri_stretch_step) capture their
 * whole kernel sequence -- orbit, synthesis, transform, reduction, 13 to 30 launches -- into a CUDA graph the first time an
 * argument set (pointers, K) is seen and replay it afterwards: one launch per call, which is what the small ensembles of
 * the paper's own run shape (8 walkers) are bound by.  The plan keeps the graphs of the last 8 argument
 * sets; any emri_plan_set_* call drops them.  Not used while stage timings are enabled nor by emri_loglike_host.
 * 0: every call enqueues its kernels one by one.  Results are identical bit for bit.
 * emri_plan_graph_stats: out[0] = graphs captured, out[1] = calls served by a replay, since plan creation. */
int emri_plan_set_graphs(emri_plan* p, int on);
int emri_plan_graph_stats(const emri_plan* p, int64_t out[2]);

/* Truncation of the harmonic series of stage (b) (readings D8 and D13): a term of a re-summed
 * bracket series, or a whole overtone, is dropped where it stays below tol x the largest harmonic of its unit (one walker,
 * 4096 samples), so the waveform carries a relative truncation error of at most ~n_max tol / 4.  Default 1e-14: a hundredth
 * of the rounding noise the path has anyway (the phases are ~1e5 cycles known to 1e-16 relative: 1e-12 of max |h|, measured
 * against the oracle), so the default is indistinguishable from 1e-16 in every parity figure.  1e-17 <= tol <= 1e-10; each
 * decade buys about 3.5 % of the synthesis time at n_max = 30 (measured on B200). */
int emri_plan_set_series_tolerance(emri_plan* p, double tol);

/* Test hook: force the data-selected slow paths of stage (b) for every later call.  flags bit 0: every unit evaluates
 * the base series in e^2; bit 1: every sample takes the cube-root amplitude.  0 restores the defaults.  Results must
 * not change beyond rounding (tests/test_gpu_paths.py). */
int emri_plan_set_synth_debug(emri_plan* p, int flags);

/* Test hook: tiles (of 256 samples) per synthesis unit, the stretch of one walker over which stage (b) re-expands the
 * harmonic series and picks its order.  0 (default): chosen per call -- 16, fewer while a small call would otherwise leave
 * CTAs idle.  1, 2, 4, 8 or 16 fixes it for every later call, so that a test can put a short, strongly chirping series
 * into 16-tile units and reach the base-series fallback (tests/test_gpu_paths.py).  Results must not change beyond
 * rounding. */
int emri_plan_set_unit_tiles(emri_plan* p, int tiles);

/* Number of walkers processed per internal chunk (bounds the workspace: chunk*N complex128 for z = h_I + i h_II
 * plus the second buffer of the fused transform and the cuFFT work area).  Default min(K_max, 128).  Reallocates,
 * re-creates the cuFFT plans (full chunk, ragged last chunk of K_max, single transform) and their shared work area;
 * synchronises. */
int emri_plan_set_chunk(emri_plan* p, int walkers_per_chunk);

/* Stage (a): coarse orbit of Eq. 1 by fixed-step RK4 (S3).
 * params: DEV [K][17].  nodes: DEV, K * n_nodes * 16 doubles, n_nodes = ceil(N/S) + 3 (node j at
 * row j+1, j = -1 .. ceil(N/S)+1); each node row is
 *   {Phi_c, nu, gam_c, e, alp_c,  d/dt of those five,  increment of those five over [j, j+1], 0}
 * with the three angles in cycles wrapped to [0,1) and their increments unwrapped.
 * status: DEV [K] or NULL.  Mainly for stage-wise parity tests. */
int emri_orbit(emri_plan* p, const double* params, int K, double* nodes, int32_t* status,
               void* cuda_stream);
int64_t emri_plan_num_nodes(const emri_plan* p);

/* Stages (a)+(b): observed strain of both LISA channels, h_alpha(t_i), i = 0..N-1, t_i = i dt
 * (Eq. 2 with the response of PAPER.md:79/:118 and the factors of Eqs. 4-6 folded in).
 * params: DEV [K][17]; h_I, h_II: DEV [K][N] each (row k = walker k); status: DEV [K] or NULL. */
int emri_waveform(emri_plan* p, const double* params, int K, double* h_I, double* h_II,
                  int32_t* status, void* cuda_stream);

/* Stages (a)+(b)+(c): un-normalised forward DFT  H[m] = sum_i h[i] exp(-2 pi i i m / N),
 * m = 0..N/2.  spectra: DEV [K][2][N/2+1] complex128 (re, im interleaved),
 * channel I then II.  For stage-wise parity tests and for building data. */
int emri_waveform_fft(emri_plan* p, const double* params, int K, double* spectra, int32_t* status,
                      void* cuda_stream);

/* Transform a measured / mock time series of both channels into the `data_fft` argument of
 * emri_loglike (the paper's h[theta_0](f)).  d_I, d_II: DEV [N] each;
 * data_fft: DEV [2][N/2+1] complex128, same convention as emri_waveform_fft. */
int emri_data_fft(emri_plan* p, const double* d_I, const double* d_II, double* data_fft,
                  void* cuda_stream);

/* Stages (a)..(d): Gaussian log-likelihood of Eq. 8 for every walker,
 *   logL[k] = -(1/2) <d - h_k | d - h_k> = -(2 dt / N) sum_{chan} sum_m |D[m] - H_k[m]|^2 / S_n(f_m)
 * over the unmasked bins.  params: DEV [K][17], K <= K_max; data_fft: DEV [2][N/2+1] complex128;
 * logL: DEV [K]; status: DEV [K] or NULL. */
int emri_loglike(emri_plan* p, const double* params, int K, const double* data_fft, double* logL,
                 int32_t* status, void* cuda_stream);

/* emri_loglike with the frequency-dependent propagation of Eq. 7 (alpha_M = F(z,f), alpha_T = G(z,f),
 * "a power series expansion sum_n a_n(z) (f/f_*)^n ... such frequency-dependent terms need to act upon a tabulated
 * waveform in frequency space"; get_damping(), get_modified_speed()).  Every walker's spectrum is
 * multiplied per bin, inside the reduction kernel, by
 *     G_k(f) = exp(-Dm_k(f)) exp(-2 pi i f tau_k(f)),   Dm_k = sum_{n=1..3} a_{k,n} (f/f_*)^n,  tau_k = sum_{n=1..3} b_{k,n} (f/f_*)^n [s]
 * (the integrated friction and delay series of Eqs. 4-5; the n = 0 terms are Xi(z) and Delta T of the parameter row)
 * and logL[k] = -(2 dt/N) sum |D - G_k H_k|^2 / S_n.   fcoef: DEV [K][6] rows {a1,a2,a3,b1,b2,b3}; f_star > 0 [Hz].
 * All-zero rows reproduce emri_loglike bit for bit up to the factor G = 1 (exp(0), cos(0)). */
int emri_loglike_fdep(emri_plan* p, const double* params, int K, const double* fcoef, double f_star,
                      const double* data_fft, double* logL, int32_t* status, void* cuda_stream);

/* Same as emri_loglike with HOST buffers: copies params (and data_fft, unless it is NULL, in which
 * case the data uploaded by the previous non-NULL call is reused) to the device, runs the path,
 * copies logL and status back and synchronises the stream.  This is the end-to-end entry point
 * bench.py times as "e2e". */
int emri_loglike_host(emri_plan* p, const double* params, int K, const double* data_fft,
                      double* logL, int32_t* status, void* cuda_stream);

/* Device milliseconds of stages (a) orbit, (b) synthesis, (c) cuFFT, (d) likelihood reduction of
 * the last emri_loglike / emri_waveform(_fft) call, summed over chunks.  Timing events are only
 * recorded after emri_plan_enable_timings(p, 1).  Synchronises on the recorded events. */
int emri_plan_enable_timings(emri_plan* p, int on);
int emri_plan_get_timings(emri_plan* p, double ms[4]);

/* Raw cudaError_t / cufftResult of the last failing CUDA / cuFFT call on this plan (0 if none). */
int emri_plan_last_cuda_error(const emri_plan* p);

/* Number of kernels of THIS library the last emri_orbit / emri_waveform(_fft) / emri_loglike* call enqueued (the status
 * copy of emri_orbit / emri_waveform and cuFFT's own kernels are not counted).  bench.py reports it as `gpu_launches`. */
int emri_plan_last_launch_count(const emri_plan* p);

/* Bytes of device memory the plan currently owns. */
int64_t emri_plan_workspace_bytes(const emri_plan* p);

/* ---- ensemble sampler step (BASELINE.json configs[4]; emcee's affine-invariant
 * stretch move [Goodman & Weare], run on the device so that parameters and logL never visit the
 * host).  Walkers are split in two fixed halves; `emri_stretch_step` updates half `half` (0 or 1)
 * given the other:  for walker k in the active half, partner j uniform in the other half,
 * z = ((a-1) u + 1)^2 / a, Y = X_j + z (X_k - X_j), accept iff
 * ln u' < (P_free - 1) ln z + lnp(Y) - lnp(X_k), lnp = logL + uniform box prior.
 * Random numbers: Philox4x32-10 keyed by `seed`, counter (step, half, walker).
 *   X: DEV [K][17] in/out; logL: DEV [K] in/out (must hold logL of X on entry; use
 *   emri_loglike first); lo, hi: DEV [17] box prior (a column with lo == hi is held fixed and
 *   does not count in P_free); accepted: DEV int32 [K] or NULL, set to 1/0 for the active half;
 *   log_buf: DEV [K/2][EMRI_NPAR+4] doubles or NULL: per active walker {proposal[17], z, ln u',
 *   logL(Y), partner} for the teacher-forced parity protocol. K must be even, K/2 <= K_max (the plan's proposal
 *   scratch holds K_max rows). */
int emri_stretch_step(emri_plan* p, double* X, double* logL, int K, const double* data_fft,
                      const double* lo, const double* hi, double a_stretch, uint64_t seed,
                      int64_t step, int half, int32_t* accepted, double* log_buf,
                      void* cuda_stream);

/* ---- Eq. 8 without any device allocation (csrc/loglike_static.cu)
 *
 * For callers that cannot allocate device memory and therefore cannot own an emri_plan (a plan cudaMallocs its
 * workspace): a process that gave the whole card to one memory pool at start-up, a client running under a fixed memory
 * quota that may refuse the request, or a latency-critical host thread that must keep clear of cudaMalloc / cudaFree
 * because both synchronise the entire device and stall every other stream.  Such a caller keeps the model spectra in a
 * buffer of its own (layout of emri_waveform_fft) and gets the noise-weighted residual sum of PAPER.md:112-116 from
 *
 *   logL[k] = -(2 dt / N) sum_{chan I,II} sum_{m=0..N/2} |data_fft[chan][m] - spectra[k][chan][m]|^2 / psd[m]
 *
 * spectra: DEV [K][2][N/2+1] complex128; data_fft: DEV [2][N/2+1] complex128; psd: DEV [N/2+1] one-sided S_n(f_m), masked
 * exactly as in emri_plan_create (an entry that is <= 0, NaN or +inf gives its bin weight 0); logL: DEV [K].  The caller
 * owns all four and nothing else is touched except the scratch described next.  No per-walker status enters: a walker
 * whose rows are all zero gets -(1/2)<d|d>, not -inf.  Enqueues two kernels on cuda_stream and returns without
 * synchronising.  The call itself performs no cudaMalloc, cudaFree or other allocating call, ever.
 *
 * Scratch and its limit.  The per-(walker, bin range) partial sums of the two-pass reduction live in an array that is part
 * of the library image: EMRI_STATIC_SCRATCH_DOUBLES doubles = 512 KiB, held by every GPU on which the library is loaded
 * until the process exits.  One partial covers EMRI_STATIC_BINS_PER_PART bins, so the call needs
 * emri_static_scratch_need(K, N) = K ceil((N/2+1)/8192) doubles (K <= 508 at N = 2^21, K <= 13107 at N = 2^16) and returns
 * EMRI_ELIMIT, before touching the CUDA runtime, when that exceeds the array.  Split a larger ensemble into several
 * calls on ONE stream.
 *
 * Sharing.  There is one array per GPU and every call on that GPU uses it from offset 0.  Calls that may overlap on the
 * device (different streams, different host threads without ordering between their streams) race on it and give
 * wrong logL; calls on one stream are ordered and safe.  The array keeps the previous call's partials; that is harmless
 * because the first kernel writes every cell the second one reads, so nothing needs to start at zero.
 *
 * First call on a device.  With that device current, the first call looks up the array's device address
 * (cudaGetSymbolAddress) and remembers it; this can make the runtime load the library's kernels onto the device.  Make
 * that first call during start-up, before any stream capture you intend to do.  Later calls on the same device only
 * launch.  The stream must belong to the current device.
 *
 * Errors: EMRI_EINVAL (NULL pointer, K < 1, N odd or < 4, dt <= 0, device ordinal >= 64), EMRI_ELIMIT (see above),
 * EMRI_ECUDA (a runtime call or launch failed; emri_static_last_cuda_error() returns the raw cudaError_t of the last
 * such failure in this process). */
#define EMRI_STATIC_SCRATCH_DOUBLES 65536
#define EMRI_STATIC_BINS_PER_PART 8192
int emri_spectra_loglike_static(const double* spectra, int K, int64_t N, double dt, const double* data_fft,
                                const double* psd, double* logL, void* cuda_stream);
int64_t emri_static_scratch_need(int K, int64_t N); /* doubles of scratch a (K, N) call needs; -1 for invalid K, N */
int emri_static_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* EMRI_H */
