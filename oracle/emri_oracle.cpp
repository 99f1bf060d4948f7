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

// anchor: 0 = the parameter row is the state at the first sample (forward), 1 = at plunge, at the last coarse node (D12)
Orbit integrate_orbit(const Walker& w, int64_t N, real dt, int S, int pn_mask, int anchor) {
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
                 double* val, double* slope, double* inc, int64_t* info, int anchor) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  Orbit o = integrate_orbit(w, N, (real)dt, S, pn_mask, anchor);
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
                    const int64_t* idx, int64_t n_idx, double* out, int anchor) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  Orbit o = integrate_orbit(w, N, (real)dt, S, pn_mask, anchor);
  for (int64_t m = 0; m < n_idx; ++m) {
    int64_t j; real s;
    split_time(idx[m], S, w.dT / o.Delta, &j, &s);
    for (int q = 0; q < 5; ++q) out[q * n_idx + m] = (double)hermite(o, q, j, s);
  }
  return 0;
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
                    const int64_t* idx, int64_t n_idx, double* hI, double* hII, double* Apl, double* Acr, int anchor) {
  Cosmo c{(real)H0, (real)Om};
  Walker w = make_walker(params, c);
  Orbit o = integrate_orbit(w, N, (real)dt, S, 3, anchor);
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
                          double Om, double* h, int32_t* status, int anchor) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int k = 0; k < K; ++k)
    status[k] = emri_o_waveform(params + (size_t)k * NPAR, N, dt, n_max, S, H0, Om, nullptr, N,
                                h + (size_t)k * 2 * N, h + (size_t)k * 2 * N + N, nullptr, nullptr, anchor);
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
                         double* spectra, int anchor) {
  const int64_t Nf = N / 2 + 1;
  int rc = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int k = 0; k < K; ++k) {
    std::vector<double> h(2 * (size_t)N), H(4 * (size_t)Nf);
    int st = emri_o_waveform(params + (size_t)k * NPAR, N, dt, n_max, S, H0, Om, nullptr, N, h.data(),
                             h.data() + N, nullptr, nullptr, anchor);
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
