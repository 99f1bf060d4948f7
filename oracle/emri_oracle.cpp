// emri_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, single-translation-unit CPU implementation of what the EMRI_MC hot path
// computes (arXiv 2311.17174, /root/reference/PAPER.md), written from the paper and from the
// equations SURVEY.md section 8(c) restates out of the literature the paper defers to
// (Barack & Cutler 2004 = "BC", ref. [1] at PAPER.md:187; Peters & Mathews 1963, ref. [45] at
// PAPER.md:234).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this library.  It shares no code, header, table or helper with
// the CUDA path under paper_2311_17174_b200/csrc/.
//
// What it is: the algorithm step by step (S0..S7 of SURVEY.md 8(c)), in the paper's order:
//   S0 constants / units           PAPER.md:73  (cgs units -> geometric units, seconds)
//   S1 per-walker scalars          PAPER.md:144-145, Eq. 6 (:97), Eq. 4-5 (:88-93)
//   S2 AK orbital right-hand side  PAPER.md:69-73 (Eq. 1), BC Eqs. 27-31
//   S3 fixed-step RK4 on a coarse grid, angles in cycles   BASELINE.json north_star (a)
//   S4 cubic Hermite interpolation                          BASELINE.json north_star (b)
//   S5 Peters-Mathews harmonic sum + LISA response + propagation factors
//                                  PAPER.md:75-79 (Eq. 2), :118, Eq. 4-6 (:88-97)
//   S6 un-normalised forward DFT
//   S7 Gaussian log-likelihood     PAPER.md:112-116 (Eq. 8)
//   S3' (next row f-3, reading D14) the paper's own kind of integrator instead of S3: an embedded Runge-Kutta pair with
//       per-walker step control and dense output ("standard ODE methods ... Runge-Kutta scheme", solve_ivp; PAPER.md:120,
//       :133) -- Dormand-Prince 5(4) with Hairer's step-size controller and Shampine's continuous extension, whose
//       dense output is sampled at the coarse nodes; S4..S7 are unchanged
// No blocking, fusion or reordering beyond what those passages state.  Bessel functions are the
// ascending power series (the definition); cos(n Phi) is called directly for every n.
//
// Precision: the scalar type is `real` (double by default; -DEMRI_ORACLE_LONG_DOUBLE builds the
// same file in 80-bit long double for conditioning diagnostics, same C ABI with double I/O).
// Two places deliberately spend extra precision so that the oracle, not the GPU, is the accurate
// side: (1) the RK4 state update of nu and e is Kahan-compensated (a rounding error in nu at one
// node would otherwise be carried to every later node and grow linearly in the phase, DESIGN.md
// reading D3); (2) the cube root is taken in long double and rounded once; (3) the likelihood sum
// is accumulated in long double.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): see the table in DESIGN.md section 5.
// Functions whose fidelity to BC's printed coefficients cannot be pinned here (the article is
// not in the container) are marked "fidelity: literature only" -- this cannot break GPU parity.
//
// Build:  g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC emri_oracle.cpp -o libemri_oracle.so
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>

#ifdef EMRI_ORACLE_LONG_DOUBLE
typedef long double real;
#else
typedef double real;
#endif

namespace {

// ---------------------------------------------------------------- S0 constants
const real kPi = (real)3.14159265358979323846264338327950288L;
const real kTwoPi = 2 * kPi;
const real kMsunSec = (real)4.925490947e-6L;     // G Msun / c^3  [s]
const real kGpcSec = (real)1.0292712503e17L;     // Gpc / c       [s]
const real kAuSec = (real)499.004783836L;        // AU / c = R    [s]
const real kYearSec = (real)31557600.0L;         // Julian year   [s]
const real kMpcMetre = (real)3.0856775814913673e22L;
const real kCLight = (real)299792458.0L;         // m/s

enum { P_M = 0, P_MU, P_A, P_E0, P_NU0, P_PHI0, P_GAM0, P_ALP0, P_LAM, P_THS, P_PHS, P_THK,
       P_PHK, P_DL, P_XI0, P_NXI, P_DELT, NPAR = 17 };

enum { ST_BADPARAM = 1, ST_PLUNGE = 2, ST_DELAY = 4, ST_STATE = 8 };

struct Cosmo { real H0_km_s_Mpc; real Om; };

real frac(real x) { return x - std::floor(x); }
// cube root taken in long double and rounded once: glibc's double cbrt is only faithful (~1 ulp),
// and because its argument drifts slowly its error is systematic from step to step, which biases
// gamma~ by ~1e-11 cycles over a year (reading D3)
real cbrt_r(real x) { return (real)cbrtl((long double)x); }

// ---------------------------------------------------------------- S1 cosmology
real Ez(real z, const Cosmo& c) {
  real a = 1 + z;
  return std::sqrt(c.Om * a * a * a + (1 - c.Om));
}
// composite Simpson, 1024 panels, of g on [0, z]
template <class G> real simpson(G g, real z) {
  const int n = 1024;
  real h = z / n, s = g((real)0) + g(z);
  for (int i = 1; i < n; ++i) s += g(i * h) * ((i & 1) ? 4 : 2);
  return s * h / 3;
}
real hubble_time_sec(const Cosmo& c) { return kMpcMetre / (c.H0_km_s_Mpc * 1000); }
// EM luminosity distance in seconds (d_L / c)
real dL_sec(real z, const Cosmo& c) {
  return (1 + z) * hubble_time_sec(c) * simpson([&](real x) { return 1 / Ez(x, c); }, z);
}
real lookback_sec(real z, const Cosmo& c) {
  return hubble_time_sec(c) * simpson([&](real x) { return 1 / ((1 + x) * Ez(x, c)); }, z);
}
// solve d_L(z) = D for z by bisection on [0, 20]
real z_of_dL(real D_sec, const Cosmo& c) {
  real lo = 0, hi = 20;
  for (int it = 0; it < 200; ++it) {
    real mid = (lo + hi) / 2;
    if (mid == lo || mid == hi) break;
    if (dL_sec(mid, c) < D_sec) lo = mid; else hi = mid;
  }
  return (lo + hi) / 2;
}
// Eq. 6
real Xi_of_z(real Xi0, real nXi, real z) { return Xi0 + (1 - Xi0) * std::pow(1 + z, -nXi); }

// ---------------------------------------------------------------- per-walker constant block
struct Walker {
  real Ms, mus, a, clam, slam;      // masses in seconds, spin, cos/sin lambda
  real thS, phS, thK, phK;          // fixed angles [rad]
  real Ds, z, Xi, amp;              // distance [s], redshift, Xi(z), amplitude scale mu/(Xi D)
  real dT;                          // arrival delay Delta T [s] (reading R9)
  real p0[5];                       // initial state (Phi_c, nu, gam_c, e, alp_c), angles in cycles
  int status;
};

Walker make_walker(const double* p, const Cosmo& c) {
  Walker w;
  std::memset(&w, 0, sizeof w);
  bool ok = true;
  for (int i = 0; i < NPAR; ++i) ok = ok && std::isfinite(p[i]);
  ok = ok && p[P_M] > 0 && p[P_MU] > 0 && p[P_DL] > 0 && p[P_E0] >= 0 && p[P_E0] < 1 &&
       std::fabs(p[P_A]) <= 1 && p[P_NU0] > 0;
  if (!ok) { w.status = ST_BADPARAM; return w; }
  w.Ms = (real)p[P_M] * kMsunSec;
  w.mus = (real)p[P_MU] * kMsunSec;
  w.a = p[P_A];
  w.clam = std::cos((real)p[P_LAM]);
  w.slam = std::sin((real)p[P_LAM]);
  w.thS = p[P_THS]; w.phS = p[P_PHS]; w.thK = p[P_THK]; w.phK = p[P_PHK];
  w.Ds = (real)p[P_DL] * kGpcSec;
  w.z = z_of_dL(w.Ds, c);
  w.Xi = Xi_of_z(p[P_XI0], p[P_NXI], w.z);
  if (!(w.Xi > 0) || !std::isfinite((double)w.Xi)) { w.status = ST_BADPARAM; return w; }
  w.amp = w.mus / (w.Xi * w.Ds);                       // d_GW = Xi d_EM, Eq. 5
  w.dT = -(real)p[P_DELT] * lookback_sec(w.z, c);      // reading R9
  w.p0[0] = frac((real)p[P_PHI0] / kTwoPi);
  w.p0[1] = p[P_NU0];
  w.p0[2] = frac((real)p[P_GAM0] / kTwoPi);
  w.p0[3] = p[P_E0];
  w.p0[4] = frac((real)p[P_ALP0] / kTwoPi);
  return w;
}

// ---------------------------------------------------------------- S2 right-hand side (BC 27-31)
// State y = (Phi_c, nu, gam_c, e, alp_c); the three angles are in CYCLES, so their rates are the
// BC rates divided by 2 pi.  pn_mask: bit 0 keeps the 1PN (x^{2/3}) terms, bit 1 keeps the
// spin-orbit terms; 3 = the full model.  Masks other than 3 exist only for the closed-form pins.
// Higher-order numerical coefficients: fidelity literature only (SURVEY 8(c) pin table).
void rhs(const Walker& w, const real y[5], int pn_mask, real f[5]) {
  const real nu = y[1], e = y[3];
  const real x = kTwoPi * w.Ms * nu;          // 2 pi M nu
  const real cb = cbrt_r(x);
  const real u = (pn_mask & 1) ? cb * cb : (real)0;    // x^{2/3}, the 1PN parameter
  const real u0 = cb * cb;
  const real sp = (pn_mask & 2) ? w.a * w.clam : (real)0;  // (S/M^2) cos(lambda)
  const real e2 = e * e, e4 = e2 * e2, e6 = e4 * e2;
  const real q = 1 - e2;
  const real sq = std::sqrt(q);
  const real x113 = x * x * x * u0;            // x^{11/3}
  const real x83 = x * x * u0;                 // x^{8/3}
  // Phi' = 2 pi nu
  f[0] = nu;
  // nu'
  {
    real t0 = (1 + (real)73 / 24 * e2 + (real)37 / 96 * e4) * q;
    real t1 = u * ((real)1273 / 336 - (real)2561 / 224 * e2 - (real)3885 / 128 * e4 -
                   (real)13147 / 5376 * e6);
    real t2 = x * sp / sq * ((real)73 / 12 + (real)1211 / 24 * e2 + (real)3143 / 96 * e4 +
                             (real)65 / 64 * e6);
    real q92 = q * q * q * q * sq;             // q^{9/2}
    f[1] = (real)96 / (10 * kPi) * (w.mus / (w.Ms * w.Ms * w.Ms)) * x113 / q92 * (t0 + t1 - t2);
  }
  // gamma~' / 2 pi
  {
    real uq = u / q;
    f[2] = 3 * nu * u0 / q * (1 + uq * (26 - 15 * e2) / 4) - 6 * nu * sp * x / (q * sq);
  }
  // e'
  {
    real q72 = q * q * q * sq;
    real t0 = (304 + 121 * e2) * q * (1 + 12 * u);
    real t1 = u * ((real)8 * 16705 + (real)12 * 9082 * e2 - 25211 * e4) / 56;
    real t2 = sp * x113 / (q * q * q * q) *
              ((real)1364 / 5 + (real)5032 / 15 * e2 + (real)263 / 10 * e4);
    f[3] = -(e / 15) * (w.mus / (w.Ms * w.Ms)) * x83 / q72 * (t0 - t1) +
           e * (w.mus / (w.Ms * w.Ms)) * t2;
  }
  // alpha' / 2 pi
  f[4] = (pn_mask & 2) ? 2 * nu * w.a * x / (q * sq) : (real)0;
}

// PAPER.md:120  nu_LSO = c^3/(2 pi G M) ((1-e^2)/(6+2e))^{3/2}
real nu_lso(real Ms, real e) {
  real r = (1 - e * e) / (6 + 2 * e);
  return r * std::sqrt(r) / (kTwoPi * Ms);
}

// ---------------------------------------------------------------- S3 coarse RK4 orbit
struct Orbit {
  int64_t Nc;            // number of coarse intervals covering the N samples
  int G;                 // guard intervals each side (1)
  int64_t Nn;            // nodes = Nc + 1 + 2G, node j lives at index j + G
  real Delta;            // coarse step [s]
  int64_t jpl;           // first plunged node (node index j), or Nn if none
  std::vector<real> val[5], slope[5], inc[5];   // inc[q][j+G] = unwrapped increment over interval j
  int status;
};

bool state_ok(const real y[5]) {
  for (int q = 0; q < 5; ++q) if (!std::isfinite((double)y[q])) return false;
  return y[3] >= 0 && y[3] < 1 && y[1] > 0;
}

// one classical RK4 step of size h from y; returns the unwrapped increment d[5]
void rk4_increment(const Walker& w, const real y[5], real h, int pn_mask, real d[5], real k1[5]) {
  real k2[5], k3[5], k4[5], t[5];
  rhs(w, y, pn_mask, k1);
  for (int q = 0; q < 5; ++q) t[q] = y[q] + (h / 2) * k1[q];
  rhs(w, t, pn_mask, k2);
  for (int q = 0; q < 5; ++q) t[q] = y[q] + (h / 2) * k2[q];
  rhs(w, t, pn_mask, k3);
  for (int q = 0; q < 5; ++q) t[q] = y[q] + h * k3[q];
  rhs(w, t, pn_mask, k4);
  for (int q = 0; q < 5; ++q) d[q] = (h / 6) * (k1[q] + 2 * k2[q] + 2 * k3[q] + k4[q]);
}

// The paper's own initial-condition convention ("initial conditions at the LSO ... integrated
// backwards", nu_LSO = c^3/(2 pi G M) ((1-e^2)/(6+2e))^{3/2}; reading D12 of DESIGN.md): the parameter row's
// (e, Phi, gamma~, alpha) are the values AT PLUNGE, placed at the last coarse node t_A = Nc*Delta (the end of the window),
// nu there is nu_LSO(e_LSO) (column nu0 is ignored), and the same fixed-step RK4 runs backwards, node Nc -> node -1.
// The interval increments are stored in forward time (inc[j] = y_{j+1} - y_j); one forward step gives the guard node
// Nc+1.  Nothing plunges inside the window by construction; a bad state (e leaving [0,1)) sets ST_STATE.
Orbit integrate_orbit_from_lso(const Walker& w, int64_t N, real dt, int S, int pn_mask) {
  Orbit o;
  o.G = 1;
  o.Nc = (N + S - 1) / S;
  o.Nn = o.Nc + 1 + 2 * o.G;
  o.Delta = S * dt;
  o.jpl = o.Nn;
  o.status = w.status;
  for (int q = 0; q < 5; ++q) {
    o.val[q].assign(o.Nn, 0);
    o.slope[q].assign(o.Nn, 0);
    o.inc[q].assign(o.Nn, 0);
  }
  if (w.status & ST_BADPARAM) return o;
  const int G = o.G;
  real y[5], d[5], k1[5];
  for (int q = 0; q < 5; ++q) y[q] = w.p0[q];
  y[1] = nu_lso(w.Ms, y[3]);
  auto fail = [&]() {
    for (int q = 0; q < 5; ++q) {
      std::fill(o.val[q].begin(), o.val[q].end(), (real)0);
      std::fill(o.slope[q].begin(), o.slope[q].end(), (real)0);
      std::fill(o.inc[q].begin(), o.inc[q].end(), (real)0);
    }
    o.status |= ST_STATE;
    return o;
  };
  // forward guard step: node Nc+1 = anchor advanced by +Delta
  {
    rk4_increment(w, y, o.Delta, pn_mask, d, k1);
    real yp[5];
    for (int q = 0; q < 5; ++q) yp[q] = y[q] + d[q];
    yp[0] = frac(yp[0]); yp[2] = frac(yp[2]); yp[4] = frac(yp[4]);
    if (!state_ok(yp)) return fail();
    real kp[5];
    rhs(w, yp, pn_mask, kp);
    const int64_t jj = o.Nc + 1 + G;
    for (int q = 0; q < 5; ++q) { o.val[q][jj] = yp[q]; o.slope[q][jj] = kp[q]; o.inc[q][jj] = 0; }
    for (int q = 0; q < 5; ++q) o.inc[q][o.Nc + G] = d[q];
  }
  // backward sweep; nu and e carry a Kahan compensation term
  real comp_nu = 0, comp_e = 0;
  for (int64_t j = o.Nc; j >= -G; --j) {
    const int64_t jj = j + G;
    if (j == -G) {                 // last node: one extra slope evaluation
      rhs(w, y, pn_mask, k1);
      for (int q = 0; q < 5; ++q) { o.val[q][jj] = y[q]; o.slope[q][jj] = k1[q]; }
      break;
    }
    rk4_increment(w, y, -o.Delta, pn_mask, d, k1);
    for (int q = 0; q < 5; ++q) { o.val[q][jj] = y[q]; o.slope[q][jj] = k1[q]; o.inc[q][jj - 1] = -d[q]; }
    real yn[5];
    yn[0] = frac(y[0] + d[0]);
    yn[2] = frac(y[2] + d[2]);
    yn[4] = frac(y[4] + d[4]);
    { real a = d[1] - comp_nu, t = y[1] + a; comp_nu = (t - y[1]) - a; yn[1] = t; }
    { real a = d[3] - comp_e, t = y[3] + a; comp_e = (t - y[3]) - a; yn[3] = t; }
    if (!state_ok(yn)) return fail();
    for (int q = 0; q < 5; ++q) y[q] = yn[q];
  }
  return o;
}

// ---------------------------------------------------------------- S3' adaptive embedded pair with dense output (f-3, D14)
// Dormand & Prince 1980, RK5(4)7M: c, a_ij, b (5th order, = the 7th row: first-same-as-last), e = b - b^ (4th order
// embedded), and the coefficients of Shampine's 4th-order continuous extension,
//     y(t_n + theta h) = y_n + h sum_i K_i sum_{j=0..3} P_ij theta^{j+1}.
const real DP_C[6] = {0, (real)1 / 5, (real)3 / 10, (real)4 / 5, (real)8 / 9, 1};
const real DP_A[6][5] = {
    {0, 0, 0, 0, 0},
    {(real)1 / 5, 0, 0, 0, 0},
    {(real)3 / 40, (real)9 / 40, 0, 0, 0},
    {(real)44 / 45, (real)-56 / 15, (real)32 / 9, 0, 0},
    {(real)19372 / 6561, (real)-25360 / 2187, (real)64448 / 6561, (real)-212 / 729, 0},
    {(real)9017 / 3168, (real)-355 / 33, (real)46732 / 5247, (real)49 / 176, (real)-5103 / 18656}};
const real DP_B[6] = {(real)35 / 384, 0, (real)500 / 1113, (real)125 / 192, (real)-2187 / 6784, (real)11 / 84};
const real DP_E[7] = {(real)-71 / 57600, 0, (real)71 / 16695, (real)-71 / 1920, (real)17253 / 339200, (real)-22 / 525,
                      (real)1 / 40};
const real DP_P[7][4] = {
    {1, (real)-8048581381.0L / 2820520608.0L, (real)8663915743.0L / 2820520608.0L, (real)-12715105075.0L / 11282082432.0L},
    {0, 0, 0, 0},
    {0, (real)131558114200.0L / 32700410799.0L, (real)-68118460800.0L / 10900136933.0L, (real)87487479700.0L / 32700410799.0L},
    {0, (real)-1754552775.0L / 470086768.0L, (real)14199869525.0L / 1410260304.0L, (real)-10690763975.0L / 1880347072.0L},
    {0, (real)127303824393.0L / 49829197408.0L, (real)-318862633887.0L / 49829197408.0L,
     (real)701980252875.0L / 199316789632.0L},
    {0, (real)-282668133.0L / 205662961.0L, (real)2019193451.0L / 616988883.0L, (real)-1453857185.0L / 822651844.0L},
    {0, (real)40617522.0L / 29380423.0L, (real)-110615467.0L / 29380423.0L, (real)69997945.0L / 29380423.0L}};

struct Dp5Step {
  real t, h;          // start of the step and its signed size
  real y[5];          // state at t: angles (0, 2, 4) in cycles wrapped to [0, 1), nu, e
  real turns[3];      // whole cycles removed from the three angles so far (enters the error scale only)
  real Q[5][4];       // dense output: y(t + theta h) = y + sum_j Q[q][j] theta^{j+1}  (already multiplied by h)
  real D[5];          // the step's own increment h sum_i b_i K_i (unwrapped); Q(1) equals it up to the rounding of P
  real err;           // the controller's error norm of this step (also evaluated, but not acted on, for a forced step)
};
struct Dp5Branch {
  std::vector<Dp5Step> steps;
  real t_end;         // where the branch stops (the bound, or the end of the step after which the state is unusable)
  int stop;           // 0 reached the bound; ST_PLUNGE / ST_STATE: stopped early after an accepted step
};

real rms5(const real v[5]) {
  real s = 0;
  for (int q = 0; q < 5; ++q) s += v[q] * v[q];
  return std::sqrt(s / 5);
}

// Integrate dY/dt = f(Y) from (t0, y0) to t_bound with Dormand-Prince 5(4) and the step-size controller of Hairer,
// Norsett & Wanner (Solving ODEs I, sec. II.4), in the form SciPy's solve_ivp(method="RK45") uses it (the paper's
// integrator is solve_ivp): error norm = rms over the components of err_q / (atol_q + rtol max(|Y_q|,
// |Y_q,new|)); accepted when < 1; new step = h min(10, 0.9 err^{-1/5}) (at most h after a rejection); rejected: h max(0.2,
// 0.9 err^{-1/5}); first step from the two-evaluation estimate of the same section; the last step is cut to land on the
// bound.  |Y| is the UNWRAPPED angle (turns + fraction) so that the scale is what an integration in plain cycles sees,
// while the state itself is kept wrapped (only frac matters downstream, D2).  stop_at_plunge: forward integration of a
// walker given at t = 0 ends after the first accepted step whose end state is past nu_LSO(e) (reading R8).
// forced (may be NULL): n_forced prescribed step sizes taken one after the other instead of the controller's -- the
// teacher-forced half of the parity protocol (D14): at tolerances near rounding the error estimate is dominated
// by rounding noise, so two correct implementations choose different steps; given the SAME steps they must agree.
Dp5Branch dp5_integrate(const Walker& w, const real y0[5], real t0, real t_bound, real rtol, const real atol[5], int pn_mask,
                        bool stop_at_plunge, const double* forced = nullptr, int64_t n_forced = 0) {
  Dp5Branch br;
  br.t_end = t0; br.stop = 0;
  const real dir = (t_bound >= t0) ? 1 : -1;
  if (t_bound == t0) return br;
  real t = t0, y[5], turns[3] = {0, 0, 0}, f[5];
  for (int q = 0; q < 5; ++q) y[q] = y0[q];
  rhs(w, y, pn_mask, f);
  auto unwrapped = [&](const real yy[5], const real tt[3], int q) -> real {
    return (q == 0) ? tt[0] + yy[0] : (q == 2) ? tt[1] + yy[2] : (q == 4) ? tt[2] + yy[4] : yy[q];
  };
  // first step
  real h_abs;
  {
    const real interval = std::fabs(t_bound - t0);
    real sc[5], v0[5], v1[5];
    for (int q = 0; q < 5; ++q) { sc[q] = atol[q] + std::fabs(unwrapped(y, turns, q)) * rtol; v0[q] = unwrapped(y, turns, q) / sc[q]; v1[q] = f[q] / sc[q]; }
    const real d0 = rms5(v0), d1 = rms5(v1);
    real h0 = (d0 < (real)1e-5 || d1 < (real)1e-5) ? (real)1e-6 : (real)0.01 * d0 / d1;
    if (h0 > interval) h0 = interval;
    real y1[5], f1[5], v2[5];
    for (int q = 0; q < 5; ++q) y1[q] = y[q] + h0 * dir * f[q];
    rhs(w, y1, pn_mask, f1);
    for (int q = 0; q < 5; ++q) v2[q] = (f1[q] - f[q]) / sc[q];
    const real d2 = rms5(v2) / h0;
    const real dm = d1 > d2 ? d1 : d2;
    real h1 = (d1 <= (real)1e-15 && d2 <= (real)1e-15) ? std::max((real)1e-6, h0 * (real)1e-3)
                                                       : std::pow((real)0.01 / dm, (real)1 / 5);
    h_abs = std::min(std::min(100 * h0, h1), interval);
  }
  const real expo = (real)-1 / 5;
  for (int n_steps = 0; forced ? n_steps < n_forced : t != t_bound; ++n_steps) {
    if (n_steps >= 1000000) { br.stop = ST_STATE; break; }
    const real min_step = 10 * std::fabs(std::nextafter(t, dir * std::numeric_limits<real>::infinity()) - t);
    if (h_abs < min_step) h_abs = min_step;
    bool rejected = false;
    real K[7][5], y_new[5], h = 0, t_new = t, err_acc = 0;
    for (;;) {
      if (h_abs < min_step && !forced) { br.stop = ST_STATE; br.t_end = t; return br; }
      h = h_abs * dir;
      t_new = t + h;
      if (dir * (t_new - t_bound) > 0) t_new = t_bound;
      h = t_new - t;
      if (forced) { h = (real)forced[n_steps]; t_new = t + h; }
      h_abs = std::fabs(h);
      for (int q = 0; q < 5; ++q) K[0][q] = f[q];
      for (int s = 1; s < 6; ++s) {
        real ys[5];
        for (int q = 0; q < 5; ++q) {
          real dy = 0;
          for (int j = 0; j < s; ++j) dy += DP_A[s][j] * K[j][q];
          ys[q] = y[q] + dy * h;
        }
        rhs(w, ys, pn_mask, K[s]);
      }
      for (int q = 0; q < 5; ++q) {
        real dy = 0;
        for (int j = 0; j < 6; ++j) dy += DP_B[j] * K[j][q];
        y_new[q] = y[q] + h * dy;
      }
      rhs(w, y_new, pn_mask, K[6]);
      real en[5];
      for (int q = 0; q < 5; ++q) {
        real e = 0;
        for (int j = 0; j < 7; ++j) e += DP_E[j] * K[j][q];
        // |Y_new| unwrapped = |Y| + increment for the angles
        const real Yo = unwrapped(y, turns, q), Yn = (q == 1 || q == 3) ? y_new[q] : Yo + (y_new[q] - y[q]);
        const real sc = atol[q] + std::max(std::fabs(Yo), std::fabs(Yn)) * rtol;
        en[q] = e * h / sc;
      }
      const real err = rms5(en);
      err_acc = err;
      if (forced) break;
      if (err < 1) {
        real factor = (err == 0) ? (real)10 : std::min((real)10, (real)0.9 * std::pow(err, expo));
        if (rejected && factor > 1) factor = 1;
        h_abs *= factor;
        break;
      }
      h_abs *= std::max((real)0.2, (real)0.9 * std::pow(err, expo));
      rejected = true;
    }
    // record the accepted step with its dense output
    Dp5Step st;
    st.t = t; st.h = h; st.err = err_acc;
    for (int q = 0; q < 5; ++q) st.y[q] = y[q];
    for (int a = 0; a < 3; ++a) st.turns[a] = turns[a];
    for (int q = 0; q < 5; ++q)
      for (int j = 0; j < 4; ++j) {
        real c = 0;
        for (int i = 0; i < 7; ++i) c += K[i][q] * DP_P[i][j];
        st.Q[q][j] = h * c;
      }
    for (int q = 0; q < 5; ++q) st.D[q] = y_new[q] - y[q];
    br.steps.push_back(st);
    // advance; the angles are wrapped and the whole cycles remembered
    for (int q = 0; q < 5; ++q) y[q] = y_new[q];
    for (int a = 0; a < 3; ++a) {
      const int q = 2 * a;
      const real fl = std::floor(y[q]);
      turns[a] += fl; y[q] -= fl;
    }
    for (int q = 0; q < 5; ++q) f[q] = K[6][q];
    t = t_new;
    br.t_end = t;
    if (!state_ok(y)) { br.stop = ST_STATE; break; }
    if (stop_at_plunge && !(y[1] < nu_lso(w.Ms, y[3]))) { br.stop = ST_PLUNGE; break; }
  }
  return br;
}

// dense output of step st at fraction theta: offset from st.y (unwrapped for the angles)
void dp5_offset(const Dp5Step& st, real theta, real off[5]) {
  for (int q = 0; q < 5; ++q) off[q] = theta * (st.Q[q][0] + theta * (st.Q[q][1] + theta * (st.Q[q][2] + theta * st.Q[q][3])));
}

// The coarse orbit (same node table as S3) sampled from the dense output of the adaptive integration: from the anchor
// (t = 0 forward convention, or the last node in the LSO convention) one branch runs forward to node Nc + 1 and one
// backward to node -1.  Node values are y_n + offset(theta) (angles wrapped), node slopes the right-hand side AT the node,
// interval increments the unwrapped offset differences, pieced together step by step so that no large number is ever
// differenced.  Between nodes S4's cubic Hermite is kept: at the default stride its truncation error is below the rounding of
// the phases (D3), so sampling the dense output at every sample instead would change nothing above 1e-14 cycles.
Orbit integrate_orbit_adaptive(const Walker& w, int64_t N, real dt, int S, int pn_mask, int anchor, real rtol, const real atol[5],
                               const double* forced_fwd = nullptr, int64_t n_fwd = 0, const double* forced_bwd = nullptr,
                               int64_t n_bwd = 0) {
  Orbit o;
  o.G = 1;
  o.Nc = (N + S - 1) / S;
  o.Nn = o.Nc + 1 + 2 * o.G;
  o.Delta = S * dt;
  o.jpl = o.Nn;
  o.status = w.status;
  for (int q = 0; q < 5; ++q) { o.val[q].assign(o.Nn, 0); o.slope[q].assign(o.Nn, 0); o.inc[q].assign(o.Nn, 0); }
  if (w.status & ST_BADPARAM) return o;
  const int G = o.G;
  real y0[5];
  for (int q = 0; q < 5; ++q) y0[q] = w.p0[q];
  const int64_t ja = anchor ? o.Nc : 0;                 // anchor node
  if (anchor) y0[1] = nu_lso(w.Ms, y0[3]);
  else if (!(y0[1] < nu_lso(w.Ms, y0[3]))) { o.status |= ST_PLUNGE; o.jpl = 0; return o; }
  const real ta = (real)ja * o.Delta;
  Dp5Branch fwd = dp5_integrate(w, y0, ta, (real)(o.Nc + G) * o.Delta, rtol, atol, pn_mask, !anchor, forced_fwd, n_fwd);
  Dp5Branch bwd = dp5_integrate(w, y0, ta, (real)(-G) * o.Delta, rtol, atol, pn_mask, false, forced_bwd, n_bwd);
  auto zero_all = [&](int bit) {
    for (int q = 0; q < 5; ++q) {
      std::fill(o.val[q].begin(), o.val[q].end(), (real)0);
      std::fill(o.slope[q].begin(), o.slope[q].end(), (real)0);
      std::fill(o.inc[q].begin(), o.inc[q].end(), (real)0);
    }
    o.status |= bit;
    return o;
  };
  if (bwd.stop || (anchor && fwd.stop)) return zero_all(ST_STATE);          // the guard side / the LSO convention must be clean
  if (fwd.stop == ST_STATE && fwd.steps.empty()) return zero_all(ST_STATE);
  // position of node j in its branch: step index and theta
  struct Pos { const Dp5Branch* br; int64_t n; real theta; bool ok; };
  auto locate = [&](int64_t j, int64_t hint, const Dp5Branch& br) -> Pos {
    const real tj = (real)j * o.Delta;
    const real dir = (br.steps.empty() || br.steps[0].h >= 0) ? 1 : -1;
    if (br.steps.empty() || dir * (tj - br.t_end) > 0) return Pos{&br, 0, 0, false};
    int64_t n = hint;
    while (n + 1 < (int64_t)br.steps.size() && dir * (tj - (br.steps[n].t + br.steps[n].h)) > 0) ++n;
    return Pos{&br, n, (tj - br.steps[n].t) / br.steps[n].h, true};
  };
  auto node_state = [&](const Pos& p, real y[5]) {
    real off[5];
    const Dp5Step& st = p.br->steps[p.n];
    dp5_offset(st, p.theta, off);
    for (int q = 0; q < 5; ++q) y[q] = st.y[q] + off[q];
    y[0] = frac(y[0]); y[2] = frac(y[2]); y[4] = frac(y[4]);
  };
  // unwrapped change from position a to position b, b not before a in the branch's own order
  auto change = [&](const Pos& a, const Pos& b, real d[5]) {
    real oa[5], ob[5];
    dp5_offset(a.br->steps[a.n], a.theta, oa);
    dp5_offset(b.br->steps[b.n], b.theta, ob);
    if (a.n == b.n) { for (int q = 0; q < 5; ++q) d[q] = ob[q] - oa[q]; return; }
    // whole steps contribute their own increments D (what the state actually advanced by), so that the pieces add up
    // to value(b) - value(a) exactly; every term is at most a step's increment in size
    for (int q = 0; q < 5; ++q) d[q] = a.br->steps[a.n].D[q] - oa[q];
    for (int64_t i = a.n + 1; i < b.n; ++i)
      for (int q = 0; q < 5; ++q) d[q] += a.br->steps[i].D[q];
    for (int q = 0; q < 5; ++q) d[q] += ob[q];
  };
  // forward side: nodes ja .. Nc + G in time order
  {
    int64_t hint = 0;
    Pos prev{&fwd, 0, 0, false};
    for (int64_t j = ja; j <= o.Nc + G; ++j) {
      const int64_t jj = j + G;
      Pos p = locate(j, hint, fwd);
      real y[5];
      bool bad = !p.ok;
      if (p.ok) {
        node_state(p, y);
        if (!state_ok(y)) { bad = true; o.status |= ST_STATE; }
        else if (!anchor && !(y[1] < nu_lso(w.Ms, y[3]))) { bad = true; o.status |= ST_PLUNGE; }
      } else {
        o.status |= (fwd.stop == ST_STATE) ? ST_STATE : ST_PLUNGE;
      }
      if (bad) {
        if (anchor) return zero_all(ST_STATE);
        o.jpl = j;
        // nodes from j_pl on are copies of node j_pl - 1 with zero increments (as S3); the interval before them too
        for (int64_t m = j; m <= o.Nc + G; ++m)
          for (int q = 0; q < 5; ++q) {
            o.val[q][m + G] = (j > ja) ? o.val[q][jj - 1] : (real)0;
            o.slope[q][m + G] = (j > ja) ? o.slope[q][jj - 1] : (real)0;
            o.inc[q][m + G] = 0;
          }
        if (j > ja) for (int q = 0; q < 5; ++q) o.inc[q][jj - 1] = 0;
        break;
      }
      real f[5];
      rhs(w, y, pn_mask, f);
      for (int q = 0; q < 5; ++q) { o.val[q][jj] = y[q]; o.slope[q][jj] = f[q]; }
      if (j > ja) {
        real d[5];
        change(prev, p, d);
        for (int q = 0; q < 5; ++q) o.inc[q][jj - 1] = d[q];
      }
      prev = p; hint = p.n;
    }
  }
  // backward side: nodes ja - 1 .. -G, in the branch's order (decreasing time); increments are stored in forward time
  {
    int64_t hint = 0;
    Pos prev{&bwd, 0, 0, true};                       // the anchor node itself: step 0, theta 0
    if (bwd.steps.empty()) return zero_all(ST_STATE);
    for (int64_t j = ja - 1; j >= -G; --j) {
      const int64_t jj = j + G;
      Pos p = locate(j, hint, bwd);
      if (!p.ok) return zero_all(ST_STATE);
      real y[5], f[5], d[5];
      node_state(p, y);
      if (!state_ok(y)) return zero_all(ST_STATE);
      rhs(w, y, pn_mask, f);
      for (int q = 0; q < 5; ++q) { o.val[q][jj] = y[q]; o.slope[q][jj] = f[q]; }
      change(prev, p, d);                              // from node j + 1 to node j
      for (int q = 0; q < 5; ++q) o.inc[q][jj] = -d[q];
      prev = p; hint = p.n;
    }
  }
  return o;
}

// anchor: 0 = the parameter row is the state at the first sample (forward), 1 = at plunge, at the last coarse node (D12)
// adaptive: NULL = the fixed-step RK4 of S3; else {rtol, atol[5], n_fwd, n_bwd, forced steps ...} of the embedded pair of S3'
Orbit integrate_orbit(const Walker& w, int64_t N, real dt, int S, int pn_mask, int anchor, const double* adaptive) {
  if (adaptive) {
    real at[5];
    for (int q = 0; q < 5; ++q) at[q] = (real)adaptive[1 + q];
    // adaptive[6], adaptive[7]: numbers of prescribed steps of the forward / backward branch (0: the controller decides),
    // followed by the step sizes themselves
    const int64_t nf = (int64_t)adaptive[6], nb = (int64_t)adaptive[7];
    return integrate_orbit_adaptive(w, N, dt, S, pn_mask, anchor, (real)adaptive[0], at, nf ? adaptive + 8 : nullptr, nf,
                                    nb ? adaptive + 8 + nf : nullptr, nb);
  }
  if (anchor) return integrate_orbit_from_lso(w, N, dt, S, pn_mask);
  Orbit o;
  o.G = 1;
  o.Nc = (N + S - 1) / S;
  o.Nn = o.Nc + 1 + 2 * o.G;
  o.Delta = S * dt;
  o.jpl = o.Nn;    // "no plunge" sentinel (node index space j + G)
  o.status = w.status;
  for (int q = 0; q < 5; ++q) {
    o.val[q].assign(o.Nn, 0);
    o.slope[q].assign(o.Nn, 0);
    o.inc[q].assign(o.Nn, 0);
  }
  if (w.status & ST_BADPARAM) return o;
  const int G = o.G;
  real y[5], d[5], k1[5];
  for (int q = 0; q < 5; ++q) y[q] = w.p0[q];
  // node 0: already plunged at the first sample?
  if (!(y[1] < nu_lso(w.Ms, y[3]))) { o.status |= ST_PLUNGE; o.jpl = 0; return o; }
  // backward guard step: node -1 = node 0 advanced by -Delta
  {
    rk4_increment(w, y, -o.Delta, pn_mask, d, k1);
    real ym[5];
    for (int q = 0; q < 5; ++q) ym[q] = y[q] + d[q];
    ym[0] = frac(ym[0]); ym[2] = frac(ym[2]); ym[4] = frac(ym[4]);
    if (!state_ok(ym)) { o.status |= ST_STATE; return o; }
    real km[5];
    rhs(w, ym, pn_mask, km);
    for (int q = 0; q < 5; ++q) {
      o.val[q][0] = ym[q];
      o.slope[q][0] = km[q];
      o.inc[q][0] = -d[q];       // increment over interval -1, taken forward in time
    }
  }
  // forward sweep; nu and e carry a Kahan compensation term (header, D3)
  real comp_nu = 0, comp_e = 0;
  for (int64_t j = 0; j <= o.Nc + G; ++j) {
    const int64_t jj = j + G;
    if (j == o.Nc + G) {           // last node: one extra slope evaluation
      rhs(w, y, pn_mask, k1);
      for (int q = 0; q < 5; ++q) { o.val[q][jj] = y[q]; o.slope[q][jj] = k1[q]; }
      break;
    }
    rk4_increment(w, y, o.Delta, pn_mask, d, k1);
    for (int q = 0; q < 5; ++q) { o.val[q][jj] = y[q]; o.slope[q][jj] = k1[q]; o.inc[q][jj] = d[q]; }
    real yn[5];
    yn[0] = frac(y[0] + d[0]);
    yn[2] = frac(y[2] + d[2]);
    yn[4] = frac(y[4] + d[4]);
    { real a = d[1] - comp_nu, t = y[1] + a; comp_nu = (t - y[1]) - a; yn[1] = t; }
    { real a = d[3] - comp_e, t = y[3] + a; comp_e = (t - y[3]) - a; yn[3] = t; }
    bool ok = state_ok(yn);
    bool plunged = ok && !(yn[1] < nu_lso(w.Ms, yn[3]));
    if (!ok || plunged) {
      o.status |= ok ? ST_PLUNGE : ST_STATE;
      o.jpl = j + 1;
      // nodes from j_pl on are copies of node j_pl - 1; their increments are zero
      for (int64_t m = j + 1; m <= o.Nc + G; ++m)
        for (int q = 0; q < 5; ++q) {
          o.val[q][m + G] = o.val[q][jj];
          o.slope[q][m + G] = o.slope[q][jj];
          o.inc[q][m + G] = 0;
        }
      return o;
    }
    for (int q = 0; q < 5; ++q) y[q] = yn[q];
  }
  return o;
}

// ---------------------------------------------------------------- S4 cubic Hermite
// Split the source time t' = i dt - dT into coarse interval j and fraction s in [0,1) without
// cancellation (reading D4): j0 = i / S, s0 = (i mod S)/S exactly, then shift by
// sigma = dT/Delta, |sigma| < 1.
void split_time(int64_t i, int S, real sigma, int64_t* j, real* s) {
  int64_t j0 = i / S;
  real s0 = (real)(i % S) / (real)S;
  real ss = s0 - sigma;
  if (ss < 0) { ss += 1; j0 -= 1; }
  else if (ss >= 1) { ss -= 1; j0 += 1; }
  *j = j0; *s = ss;
}
real hermite(const Orbit& o, int q, int64_t j, real s) {
  const int64_t jj = j + o.G;
  real s2 = s * s, s3 = s2 * s;
  return o.val[q][jj] + (3 * s2 - 2 * s3) * o.inc[q][jj] +
         o.Delta * ((s3 - 2 * s2 + s) * o.slope[q][jj] + (s3 - s2) * o.slope[q][jj + 1]);
}

// ---------------------------------------------------------------- S5.6 Bessel J_k(x), power series
// J_k(x) = sum_m (-1)^m (x/2)^{2m+k} / (m! (m+k)!), summed until the term is below 1e-18 of the
// sum; J_{-k} = (-1)^k J_k.
real bessel_j(int k, real x) {
  if (k < 0) { real v = bessel_j(-k, x); return (k & 1) ? -v : v; }
  real hx = x / 2;
  real term = 1;
  for (int i = 1; i <= k; ++i) term *= hx / i;        // (x/2)^k / k!
  real sum = term;
  real y = hx * hx;
  for (int m = 1; m < 500; ++m) {
    term *= -y / ((real)m * (real)(m + k));
    sum += term;
    if (std::fabs(term) <= (real)1e-18L * std::fabs(sum)) break;
  }
  return sum;
}

// brackets of a_n, b_n, c_n (BC Eqs. 7-9 / Peters-Mathews), x = n e
struct Brackets { real Ba, Bb, Bc; };
Brackets brackets(int n, real e) {
  real x = n * e;
  real Jm2 = bessel_j(n - 2, x), Jm1 = bessel_j(n - 1, x), J0 = bessel_j(n, x),
       Jp1 = bessel_j(n + 1, x), Jp2 = bessel_j(n + 2, x);
  Brackets b;
  b.Ba = Jm2 - 2 * e * Jm1 + ((real)2 / n) * J0 + 2 * e * Jp1 - Jp2;
  b.Bb = std::sqrt(1 - e * e) * (Jm2 - 2 * J0 + Jp2);
  b.Bc = J0;
  return b;
}

// ---------------------------------------------------------------- S5.2/3/7 geometry
struct Geometry {
  real cthL, sthL, phL;       // orbital-plane normal L^ (BC 19-21)
  real Ln, Sn;                // L^.n^, S^.n^
  real sinb, cosb, beta;      // BC 22-24
  real cthd, phid, psi;       // detector-frame angles (BC 17-18, Cutler 1998)
  real Npsi, Dpsi;
};
// alpha [rad] at source time; phibar [rad] = 2 pi t_i / T_yr at detector time (R5: phibar0 = 0,
// alphabar0 = 0)
Geometry geometry(const Walker& w, real alpha, real phibar) {
  Geometry g;
  const real cS = std::cos(w.thS), sS = std::sin(w.thS), cK = std::cos(w.thK), sK = std::sin(w.thK);
  const real cl = w.clam, sl = w.slam, ca = std::cos(alpha), sa = std::sin(alpha);
  // BC 19-21
  g.cthL = cK * cl + sK * sl * ca;
  real Lx = sK * std::cos(w.phK) * cl - std::cos(w.phK) * cK * sl * ca + std::sin(w.phK) * sl * sa;
  real Ly = sK * std::sin(w.phK) * cl - std::sin(w.phK) * cK * sl * ca - std::cos(w.phK) * sl * sa;
  g.sthL = std::sqrt(Lx * Lx + Ly * Ly);
  g.phL = std::atan2(Ly, Lx);
  g.Ln = cS * g.cthL + sS * g.sthL * std::cos(w.phS - g.phL);
  g.Sn = cS * cK + sS * sK * std::cos(w.phS - w.phK);
  // BC 22-24
  real den = sl * std::sqrt(1 - g.Ln * g.Ln);
  real nSxL = sS * std::sin(w.phK - w.phS) * sl * ca + (g.Sn * cK - cS) / sK * sl * sa;
  g.sinb = (cl * g.Ln - g.Sn) / den;
  g.cosb = nSxL / den;
  g.beta = std::atan2(g.sinb, g.cosb);
  // BC 17-18 (Cutler 1998), detector time
  real dph = phibar - w.phS;
  g.cthd = cS / 2 - std::sqrt((real)3) / 2 * sS * std::cos(dph);
  g.phid = phibar + std::atan2(std::sqrt((real)3) * cS + sS * std::cos(dph), 2 * sS * std::sin(dph));
  const real r3 = std::sqrt((real)3) / 2;
  g.Npsi = g.cthL / 2 - r3 * g.sthL * std::cos(phibar - g.phL) -
           g.cthd * (g.cthL * cS + g.sthL * sS * std::cos(g.phL - w.phS));
  g.Dpsi = g.sthL * sS * std::sin(g.phL - w.phS) / 2 -
           r3 * std::cos(phibar) * (g.cthL * sS * std::sin(w.phS) - cS * g.sthL * std::sin(g.phL)) -
           r3 * std::sin(phibar) * (cS * g.sthL * std::cos(g.phL) - g.cthL * sS * std::cos(w.phS));
  g.psi = std::atan2(g.Npsi, g.Dpsi);
  return g;
}
// BC 15-16
void antenna(real cthd, real phid, real psi, real F[4]) {
  real h = (1 + cthd * cthd) / 2;
  real c2p = std::cos(2 * phid), s2p = std::sin(2 * phid), c2s = std::cos(2 * psi), s2s = std::sin(2 * psi);
  F[0] = h * c2p * c2s - cthd * s2p * s2s;   // F_I^+
  F[1] = h * c2p * s2s + cthd * s2p * c2s;   // F_I^x
  F[2] = h * s2p * c2s + cthd * c2p * s2s;   // F_II^+
  F[3] = h * s2p * s2s - cthd * c2p * c2s;   // F_II^x
}

// ---------------------------------------------------------------- S5 one sample
// returns h_I, h_II at sample i; also the polarisation amplitudes for the e=0 pin
void sample(const Walker& w, const Orbit& o, int S, real dt, int n_max, int64_t i, real* hI, real* hII,
            real* Aplus, real* Across) {
  *hI = 0; *hII = 0;
  if (Aplus) { *Aplus = 0; *Across = 0; }
  if (o.status & (ST_BADPARAM | ST_DELAY | ST_STATE)) return;
  int64_t j; real s;
  split_time(i, S, w.dT / o.Delta, &j, &s);
  if (j + 1 >= o.jpl) return;                       // R8: zero from the first plunged node on
  // S4: orbit at the source time
  real Phic = hermite(o, 0, j, s), nu = hermite(o, 1, j, s), gamc = hermite(o, 2, j, s),
       e = hermite(o, 3, j, s), alpc = hermite(o, 4, j, s);
  real t_i = (real)i * dt;
  real phibar = kTwoPi * frac(t_i / kYearSec);      // S5.1
  Geometry g = geometry(w, kTwoPi * alpc, phibar);  // S5.2, S5.3, S5.7
  real gam = kTwoPi * gamc + g.beta;                // gamma = gamma~ + beta
  // S5.4 Doppler, in cycles: Phi_tot/2pi = Phi_c + nu R sin(thS) cos(phibar - phS)
  real Phitc = frac(Phic + nu * kAuSec * std::sin(w.thS) * std::cos(phibar - w.phS));
  // S5.5 amplitude (with Eq. 4-6 folded in)
  real cb = cbrt_r(kTwoPi * w.Ms * nu);
  real A = cb * cb * w.amp;
  // S5.6 harmonics
  real c2g = std::cos(2 * gam), s2g = std::sin(2 * gam);
  real Ap = 0, Ax = 0;
  for (int n = 1; n <= n_max; ++n) {
    Brackets b = brackets(n, e);
    real ph = kTwoPi * frac(n * Phitc);
    real cn = std::cos(ph), sn = std::sin(ph);
    real an = -n * A * b.Ba * cn;
    real bn = -n * A * b.Bb * sn;
    real cc = 2 * A * b.Bc * cn;
    Ap += -(1 + g.Ln * g.Ln) * (an * c2g - bn * s2g) + (1 - g.Ln * g.Ln) * cc;
    Ax += 2 * g.Ln * (bn * c2g + an * s2g);
  }
  real F[4];
  antenna(g.cthd, g.phid, g.psi, F);                // S5.8
  const real r3 = std::sqrt((real)3) / 2;
  *hI = r3 * (F[0] * Ap + F[1] * Ax);               // S5.9
  *hII = r3 * (F[2] * Ap + F[3] * Ax);
  if (Aplus) { *Aplus = Ap; *Across = Ax; }
}

int finish_status(const Walker& w, const Orbit& o) {
  int st = o.status;
  if (!(st & ST_BADPARAM) && !(std::fabs(w.dT) <= o.Delta)) st |= ST_DELAY;   // R20
  return st;
}

// ---------------------------------------------------------------- S6 radix-2 FFT
// iterative decimation-in-time complex FFT, twiddles from a direct sin/cos of every angle
void fft_c(std::vector<real>& re, std::vector<real>& im) {
  const size_t n = re.size();
  for (size_t i = 1, j = 0; i < n; ++i) {
    size_t bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) { std::swap(re[i], re[j]); std::swap(im[i], im[j]); }
  }
  for (size_t len = 2; len <= n; len <<= 1) {
    const size_t half = len >> 1;
    for (size_t k = 0; k < half; ++k) {
      real ang = -kTwoPi * (real)k / (real)len;
      real wr = std::cos(ang), wi = std::sin(ang);
      for (size_t i = k; i < n; i += len) {
        size_t m = i + half;
        real tr = re[m] * wr - im[m] * wi, ti = re[m] * wi + im[m] * wr;
        re[m] = re[i] - tr; im[m] = im[i] - ti;
        re[i] += tr; im[i] += ti;
      }
    }
  }
}

}  // namespace

// =================================================================== C ABI (double I/O)
extern "C" {

// `anchor` argument of the orbit / waveform entry points: 0 = the parameter row is the state at the first sample;
// 1 = at plunge, at the last coarse node (reading D12).  An explicit argument: no process-wide state.

int emri_o_real_bits(void) { return (int)std::numeric_limits<real>::digits; }

double emri_o_bessel_j(int k, double x) { return (double)bessel_j(k, (real)x); }

// out[0..2] = bracket of a_n, bracket of b_n including sqrt(1-e^2), J_n(ne)
void emri_o_brackets(int n, double e, double* out) {
  Brackets b = brackets(n, (real)e);
  out[0] = (double)b.Ba; out[1] = (double)b.Bb; out[2] = (double)b.Bc;
}

double emri_o_nu_lso(double M_msun, double e) { return (double)nu_lso((real)M_msun * kMsunSec, (real)e); }

// cosmology: out = {z, lookback time [s], d_L(z) recomputed [s]}
void emri_o_cosmology(double DL_gpc, double H0, double Om, double* out) {
  Cosmo c{(real)H0, (real)Om};
  real z = z_of_dL((real)DL_gpc * kGpcSec, c);
  out[0] = (double)z; out[1] = (double)lookback_sec(z, c); out[2] = (double)dL_sec(z, c);
}
double emri_o_dL_sec(double z, double H0, double Om) { Cosmo c{(real)H0, (real)Om}; return (double)dL_sec((real)z, c); }
double emri_o_xi(double Xi0, double nXi, double z) { return (double)Xi_of_z(Xi0, nXi, z); }

// per-walker scalars: out = {Ms, mus, Ds, z, Xi, amp, dT, status}
void emri_o_walker_scalars(const double* params, double H0, double Om, double* out) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  out[0] = (double)w.Ms; out[1] = (double)w.mus; out[2] = (double)w.Ds; out[3] = (double)w.z;
  out[4] = (double)w.Xi; out[5] = (double)w.amp; out[6] = (double)w.dT; out[7] = w.status;
}

// right-hand side at state y (angles in cycles) for a parameter row; f = d(state)/dt
void emri_o_rhs(const double* params, const double* y, int pn_mask, double* f) {
  Cosmo c{(real)67.4, (real)0.315};
  Walker w = make_walker(params, c);
  real yy[5], ff[5];
  for (int q = 0; q < 5; ++q) yy[q] = y[q];
  rhs(w, yy, pn_mask, ff);
  for (int q = 0; q < 5; ++q) f[q] = (double)ff[q];
}

// coarse orbit.  Outputs (each may be NULL): val, slope, inc are [5][Nn] row-major with
// Nn = ceil(N/S) + 3, node j at column j+1; info = {Nn, jpl (node index j, or Nn if none), status}
int emri_o_orbit(const double* params, int64_t N, double dt, int S, int pn_mask, double H0, double Om,
                 double* val, double* slope, double* inc, int64_t* info, int anchor, const double* adaptive) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  Orbit o = integrate_orbit(w, N, (real)dt, S, pn_mask, anchor, adaptive);
  for (int q = 0; q < 5; ++q)
    for (int64_t m = 0; m < o.Nn; ++m) {
      if (val) val[q * o.Nn + m] = (double)o.val[q][m];
      if (slope) slope[q * o.Nn + m] = (double)o.slope[q][m];
      if (inc) inc[q * o.Nn + m] = (double)o.inc[q][m];
    }
  if (info) { info[0] = o.Nn; info[1] = o.jpl; info[2] = finish_status(w, o); }
  return 0;
}

// orbit interpolated at sample indices idx[0..n_idx): out[5][n_idx] (angles in cycles, unwrapped
// relative to the wrapped node value)
int emri_o_orbit_at(const double* params, int64_t N, double dt, int S, int pn_mask, double H0, double Om,
                    const int64_t* idx, int64_t n_idx, double* out, int anchor, const double* adaptive) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  Orbit o = integrate_orbit(w, N, (real)dt, S, pn_mask, anchor, adaptive);
  for (int64_t m = 0; m < n_idx; ++m) {
    int64_t j; real s;
    split_time(idx[m], S, w.dT / o.Delta, &j, &s);
    for (int q = 0; q < 5; ++q) out[q * n_idx + m] = (double)hermite(o, q, j, s);
  }
  return 0;
}

// S3' for the pins: the accepted steps of the adaptive integration from the parameter row's state at t = 0 to t_end (either
// sign).  Returns the number of steps (at most max_steps are written): t[n], h[n], y[n][5] (angles wrapped), turns[n][3],
// Q[n][5][4]; info = {stop bit, t reached}.
int64_t emri_o_dp5_steps(const double* params, double t_end, double rtol, const double* atol, int pn_mask, double H0, double Om,
                         int stop_at_plunge, int64_t max_steps, double* t, double* h, double* y, double* turns, double* Q,
                         double* info) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  real at[5];
  for (int q = 0; q < 5; ++q) at[q] = (real)atol[q];
  Dp5Branch br = dp5_integrate(w, w.p0, 0, (real)t_end, (real)rtol, at, pn_mask, stop_at_plunge != 0);
  const int64_t n = (int64_t)br.steps.size();
  for (int64_t i = 0; i < n && i < max_steps; ++i) {
    const Dp5Step& st = br.steps[i];
    t[i] = (double)st.t; h[i] = (double)st.h;
    for (int q = 0; q < 5; ++q) y[5 * i + q] = (double)st.y[q];
    for (int a = 0; a < 3; ++a) turns[3 * i + a] = (double)st.turns[a];
    for (int q = 0; q < 5; ++q) for (int j = 0; j < 4; ++j) Q[(5 * i + q) * 4 + j] = (double)st.Q[q][j];
  }
  if (info) { info[0] = br.stop; info[1] = (double)br.t_end; }
  return n;
}

// S3', validity half of the teacher-forced protocol (D14): the controller's error norm, as THIS implementation
// evaluates it, of every step of a prescribed sequence h[0..n) taken from the parameter row's state at t = 0 (steps of
// either sign, all of one sign).  A step another implementation accepted must have norm < 1 here, and where the norm is
// above rounding the next step it chose must be h min(10, 0.9 norm^{-1/5}) (or smaller, after a rejection).
// Returns the number of norms written.
int64_t emri_o_dp5_forced_errors(const double* params, double rtol, const double* atol, int pn_mask, double H0, double Om,
                                 const double* h, int64_t n, double* err) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  real at[5];
  for (int q = 0; q < 5; ++q) at[q] = (real)atol[q];
  real t_end = 0;
  for (int64_t i = 0; i < n; ++i) t_end += (real)h[i];
  if (n < 1 || t_end == 0) return 0;
  Dp5Branch br = dp5_integrate(w, w.p0, 0, t_end, (real)rtol, at, pn_mask, false, h, n);
  const int64_t m = (int64_t)br.steps.size();
  for (int64_t i = 0; i < m; ++i) err[i] = (double)br.steps[i].err;
  return m;
}

// Hermite basis check: interpolate a caller-supplied single interval
double emri_o_hermite1(double y0, double inc, double m0, double m1, double Delta, double s) {
  Orbit o; o.G = 0; o.Delta = Delta;
  for (int q = 0; q < 5; ++q) { o.val[q] = {(real)y0, 0}; o.inc[q] = {(real)inc, 0}; o.slope[q] = {(real)m0, (real)m1}; }
  return (double)hermite(o, 0, 0, (real)s);
}

// geometry at (alpha [rad], phibar [rad]); out = {cthL, sthL, phL, Ln, Sn, sinb, cosb, beta, cthd,
// phid, psi, Npsi, Dpsi}
void emri_o_geometry(const double* params, double alpha, double phibar, double* out) {
  Cosmo c{(real)67.4, (real)0.315};
  Walker w = make_walker(params, c);
  Geometry g = geometry(w, (real)alpha, (real)phibar);
  real v[13] = {g.cthL, g.sthL, g.phL, g.Ln, g.Sn, g.sinb, g.cosb, g.beta, g.cthd, g.phid, g.psi, g.Npsi, g.Dpsi};
  for (int i = 0; i < 13; ++i) out[i] = (double)v[i];
}
void emri_o_antenna(double cthd, double phid, double psi, double* F) {
  real f[4]; antenna((real)cthd, (real)phid, (real)psi, f);
  for (int i = 0; i < 4; ++i) F[i] = (double)f[i];
}

// waveform at selected sample indices (idx == NULL: all samples 0..N-1, n_idx = N).
// hI, hII: [n_idx]; Apl, Acr (may be NULL): polarisation amplitudes A+, Ax.  Returns status bits.
int emri_o_waveform(const double* params, int64_t N, double dt, int n_max, int S, double H0, double Om,
                    const int64_t* idx, int64_t n_idx, double* hI, double* hII, double* Apl, double* Acr, int anchor,
                    const double* adaptive) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  Orbit o = integrate_orbit(w, N, (real)dt, S, 3, anchor, adaptive);
  o.status = finish_status(w, o);
  for (int64_t m = 0; m < n_idx; ++m) {
    int64_t i = idx ? idx[m] : m;
    real a, b, ap, ax;
    sample(w, o, S, (real)dt, n_max, i, &a, &b, &ap, &ax);
    hI[m] = (double)a; hII[m] = (double)b;
    if (Apl) { Apl[m] = (double)ap; Acr[m] = (double)ax; }
  }
  return o.status;
}

// batch of K walkers, all samples, OpenMP over walkers only.  h: [K][2][N] (channel I then II),
// status: [K]
int emri_o_waveform_batch(const double* params, int K, int64_t N, double dt, int n_max, int S, double H0,
                          double Om, double* h, int32_t* status, int anchor, const double* adaptive) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int k = 0; k < K; ++k)
    status[k] = emri_o_waveform(params + (size_t)k * NPAR, N, dt, n_max, S, H0, Om, nullptr, N,
                                h + (size_t)k * 2 * N, h + (size_t)k * 2 * N + N, nullptr, nullptr, anchor, adaptive);
  return 0;
}

// S6: H[m] = sum_i h[i] exp(-2 pi i i m / N), m = 0..N/2; N a power of two.  H interleaved re,im.
int emri_o_rfft(const double* h, int64_t N, double* H) {
  if (N < 1 || (N & (N - 1))) return -1;
  std::vector<real> re(N), im(N, 0);
  for (int64_t i = 0; i < N; ++i) re[i] = h[i];
  fft_c(re, im);
  for (int64_t m = 0; m <= N / 2; ++m) { H[2 * m] = (double)re[m]; H[2 * m + 1] = (double)im[m]; }
  return 0;
}
// naive O(N^2) DFT of the same convention, any N (for the brute-force pin)
void emri_o_dft_naive(const double* h, int64_t N, double* H) {
  for (int64_t m = 0; m <= N / 2; ++m) {
    long double sr = 0, si = 0;
    for (int64_t i = 0; i < N; ++i) {
      long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)((i * m) % N) / (long double)N;
      sr += h[i] * cosl(ang); si += h[i] * sinl(ang);
    }
    H[2 * m] = (double)sr; H[2 * m + 1] = (double)si;
  }
}

// S7: logL = -(2 dt / N) sum_{chan} sum_{m: w_m>0} |D[m]-H[m]|^2 / S_n(f_m); bins whose psd is
// <= 0, NaN or +inf are masked.  D, H: [2][N/2+1] complex interleaved; psd: [N/2+1].
double emri_o_loglike(const double* H, const double* D, const double* psd, int64_t N, double dt) {
  const int64_t Nf = N / 2 + 1;
  long double acc = 0;
  for (int ch = 0; ch < 2; ++ch)
    for (int64_t m = 0; m < Nf; ++m) {
      double s = psd[m];
      if (!(s > 0) || !std::isfinite(s)) continue;
      long double dr = (long double)D[2 * (ch * Nf + m)] - (long double)H[2 * (ch * Nf + m)];
      long double di = (long double)D[2 * (ch * Nf + m) + 1] - (long double)H[2 * (ch * Nf + m) + 1];
      acc += (dr * dr + di * di) / (long double)s;
    }
  return (double)(-(2.0L * (long double)dt / (long double)N) * acc);
}

// <a|b> = 4 Re sum_chan sum_m conj(a~) b~ / S_n df with a~ = dt A[m]: = (4 dt / N) Re sum conj(A) B / S
// Frequency-dependent propagation (Eq. 7: alpha_M = F(z,f), alpha_T = G(z,f), "an example includes a
// power series expansion sum_n a_n(z) (f/f_*)^n ... such frequency-dependent terms need to act upon a tabulated
// waveform in frequency space"; get_damping(), get_modified_speed() at PAPER.md:143).  Reading D11 of DESIGN.md: by
// Eq. 4-5 a frequency-dependent friction multiplies the spectrum by exp(-Dm(f)) and a frequency-dependent speed
// delays it by tau(f), i.e. multiplies it by exp(-2 pi i f tau(f)) (k -> 2 pi f), with the integrated power series
//   Dm(f) = sum_{n=1..3} a_n (f/f_*)^n,      tau(f) = sum_{n=1..3} b_n (f/f_*)^n  [s],     fcoef = {a1,a2,a3,b1,b2,b3}.
// The n = 0 terms are the frequency-independent Xi(z) and Delta T already inside the waveform.
//   logL = -(2 dt/N) sum_ch sum_m |D[m] - G[m] H[m]|^2 / S_n(f_m),   G[m] = exp(-Dm(f_m)) exp(-2 pi i f_m tau(f_m)).
double emri_o_loglike_fdep(const double* H, const double* D, const double* psd, int64_t N, double dt, const double* fcoef,
                           double fstar) {
  const int64_t Nf = N / 2 + 1;
  const long double twopi = 6.283185307179586476925286766559L;
  long double acc = 0;
  for (int ch = 0; ch < 2; ++ch)
    for (int64_t m = 0; m < Nf; ++m) {
      double s = psd[m];
      if (!(s > 0) || !std::isfinite(s)) continue;
      const long double f = (long double)m / ((long double)N * (long double)dt);
      const long double x = f / (long double)fstar;
      const long double Dm = fcoef[0] * x + fcoef[1] * x * x + fcoef[2] * x * x * x;
      const long double tau = fcoef[3] * x + fcoef[4] * x * x + fcoef[5] * x * x * x;
      const long double g = expl(-Dm), ph = -twopi * f * tau;
      const long double gr = g * cosl(ph), gi = g * sinl(ph);
      const long double hr = H[2 * (ch * Nf + m)], hi = H[2 * (ch * Nf + m) + 1];
      const long double dr = (long double)D[2 * (ch * Nf + m)] - (gr * hr - gi * hi);
      const long double di = (long double)D[2 * (ch * Nf + m) + 1] - (gr * hi + gi * hr);
      acc += (dr * dr + di * di) / (long double)s;
    }
  return (double)(-(2.0L * (long double)dt / (long double)N) * acc);
}

double emri_o_inner(const double* A, const double* B, const double* psd, int64_t N, double dt) {
  const int64_t Nf = N / 2 + 1;
  long double acc = 0;
  for (int ch = 0; ch < 2; ++ch)
    for (int64_t m = 0; m < Nf; ++m) {
      double s = psd[m];
      if (!(s > 0) || !std::isfinite(s)) continue;
      size_t o = 2 * (ch * Nf + m);
      acc += ((long double)A[o] * B[o] + (long double)A[o + 1] * B[o + 1]) / (long double)s;
    }
  return (double)((4.0L * (long double)dt / (long double)N) * acc);
}

// whole path for K walkers: waveform -> rfft -> logL against data D ([2][N/2+1] complex).
// status-1/4/8 walkers get -inf.  spectra (may be NULL): [K][2][N/2+1] complex out.
int emri_o_loglike_batch(const double* params, int K, int64_t N, double dt, int n_max, int S, double H0,
                         double Om, const double* D, const double* psd, double* logL, int32_t* status,
                         double* spectra, int anchor, const double* adaptive) {
  const int64_t Nf = N / 2 + 1;
  int rc = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int k = 0; k < K; ++k) {
    std::vector<double> h(2 * (size_t)N), H(4 * (size_t)Nf);
    int st = emri_o_waveform(params + (size_t)k * NPAR, N, dt, n_max, S, H0, Om, nullptr, N, h.data(),
                             h.data() + N, nullptr, nullptr, anchor, adaptive);
    if (emri_o_rfft(h.data(), N, H.data()) || emri_o_rfft(h.data() + N, N, H.data() + 2 * Nf)) {
#pragma omp atomic write
      rc = -1;
    }
    if (status) status[k] = st;
    logL[k] = (st & (ST_BADPARAM | ST_DELAY | ST_STATE)) ? -std::numeric_limits<double>::infinity()
                                                         : emri_o_loglike(H.data(), D, psd, N, dt);
    if (spectra) std::memcpy(spectra + (size_t)k * 4 * Nf, H.data(), sizeof(double) * 4 * Nf);
  }
  return rc;
}

}  // extern "C"
