// emri.cu -- sm_100a implementation of include/emri.h (the hot path of EMRI_MC, arXiv 2311.17174).
//
// Stages:
//   (a) orbit_kernel      one thread per walker: per-walker scalars (Eq. 6) and the
//                         fixed-step RK4 integration of Eq. 1 on the coarse grid
//   (b) synth_kernel      persistent CTAs over (walker, 256-sample tile): cubic-Hermite orbit,
//                         Peters-Mathews harmonic sum n = 1..n_max (Eq. 2), LISA response
//                         (PAPER.md:79, :118), propagation factors (Eqs. 4-6)
//   (c) cufftExecD2Z      batched in-place real-to-complex transform, the one vendor call
//   (d) loglike_kernel    streaming reduction of Eq. 8 + fixed-order final sum
// Nothing here is shared with oracle/ (which is test infrastructure).  FP64 throughout.
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <vector>

#include "../../include/emri.h"

namespace {

// ------------------------------------------------------------------ constants (S0)
constexpr double kPi = 3.14159265358979323846;
constexpr double kTwoPi = 6.28318530717958647692;
constexpr double kMsunSec = 4.925490947e-6;
constexpr double kGpcSec = 1.0292712503e17;
constexpr double kAuSec = 499.004783836;
constexpr double kYearSec = 31557600.0;
constexpr double kMpcMetre = 3.0856775814913673e22;
constexpr double kSqrt3 = 1.7320508075688772935;
constexpr double kHalfSqrt3 = 0.86602540378443864676;

constexpr int NODE_STRIDE = 16;   // doubles per coarse node: 5 values, 5 slopes, 5 increments, 1 spare
constexpr int WC_STRIDE = 48;     // doubles of per-walker constants
constexpr int MCAP = 48;          // largest number of Bessel series terms kept per (n, order)
constexpr int NCOEF = 12;         // per-harmonic constants
constexpr int SYNTH_THREADS = 128;
constexpr int TILE = 2 * SYNTH_THREADS;   // samples per tile (2 per thread)
constexpr int LL_THREADS = 256;
constexpr int LL_BINS_PER_THREAD = 4;
constexpr int LL_TILE = LL_THREADS * LL_BINS_PER_THREAD;
constexpr int LL_WARPS = LL_THREADS / 32;

// per-walker constant block
enum {
  WC_TWOPIMS = 0, WC_CNU, WC_CE, WC_A, WC_SP, WC_AMP, WC_DT, WC_SIGMA, WC_DOP,
  WC_CPHS, WC_SPHS, WC_CS, WC_SS, WC_LN0, WC_LN1, WC_LN2, WC_CL, WC_SN, WC_B1, WC_B2,
  WC_A0X, WC_A0Y, WC_A0Z, WC_A1X, WC_A1Y, WC_A1Z, WC_A2X, WC_A2Y,
  WC_Z, WC_XI, WC_EMAX, WC_COUNT
};
static_assert(WC_COUNT <= WC_STRIDE, "constant block too small");

enum { P_M = 0, P_MU, P_A, P_E0, P_NU0, P_PHI0, P_GAM0, P_ALP0, P_LAM, P_THS, P_PHS, P_THK, P_PHK,
       P_DL, P_XI0, P_NXI, P_DELT };

#define DEVINL __device__ __forceinline__

DEVINL double frac(double x) { return x - floor(x); }

// cube root polished by one Newton step on an exactly computed residual: CUDA's cbrt is faithful
// (1 ulp) and, for a slowly drifting argument, its error is systematic from step to step, which
// would bias gamma~ over ~1e4 steps (reading D3)
DEVINL double cbrt_polished(double x) {
  double c = cbrt(x);
  double p = c * c;
  double ep = fma(c, c, -p);
  double r = fma(-p, c, x) - ep * c;
  return fma(r, (double)__frcp_rn((float)(3.0 * p)), c);
}

// ------------------------------------------------------------------ (a0) cosmology, per walker
// 16-point Gauss-Legendre on panels of width <= 0.75 in z.
__constant__ double c_glx[8] = {0.0950125098376374401853193, 0.2816035507792589132304605,
                                0.4580167776572273863424194, 0.6178762444026437484466718,
                                0.7554044083550030338951012, 0.8656312023878317438804679,
                                0.9445750230732325760779884, 0.9894009349916499325961542};
__constant__ double c_glw[8] = {0.1894506104550684962853967, 0.1826034150449235888667637,
                                0.1691565193950025381893121, 0.1495959888165767320815017,
                                0.1246289712555338720524763, 0.0951585116824927848099251,
                                0.0622535239386478928628438, 0.0271524594117540948517806};

DEVINL double Ez(double z, double Om) {
  double a = 1.0 + z;
  return sqrt(fma(Om * a, a * a, 1.0 - Om));
}
// I1 = int_0^z dz'/E, I2 = int_0^z dz'/((1+z')E)
DEVINL void cosmo_integrals(double z, double Om, double* I1, double* I2) {
  int np = (int)ceil(z / 0.75);
  if (np < 1) np = 1;
  double h = z / np, s1 = 0.0, s2 = 0.0;
  for (int p = 0; p < np; ++p) {
    double mid = (p + 0.5) * h;
    for (int i = 0; i < 8; ++i) {
      double dx = 0.5 * h * c_glx[i];
      double za = mid - dx, zb = mid + dx;
      double fa = 1.0 / Ez(za, Om), fb = 1.0 / Ez(zb, Om);
      s1 += c_glw[i] * (fa + fb);
      s2 += c_glw[i] * (fa / (1.0 + za) + fb / (1.0 + zb));
    }
  }
  *I1 = 0.5 * h * s1;
  *I2 = 0.5 * h * s2;
}
// solve (1+z) tH I1(z) = D for z in [0, 20]: safeguarded Newton
DEVINL double z_of_dL(double D, double tH, double Om) {
  double lo = 0.0, hi = 20.0;
  double z = fmin(D / tH, 1.0);
  for (int it = 0; it < 60; ++it) {
    double I1, I2;
    cosmo_integrals(z, Om, &I1, &I2);
    double f = (1.0 + z) * tH * I1 - D;
    if (f > 0.0) hi = z; else lo = z;
    double fp = tH * (I1 + (1.0 + z) / Ez(z, Om));
    double zn = z - f / fp;
    if (!(zn > lo && zn < hi)) zn = 0.5 * (lo + hi);
    if (fabs(zn - z) <= 4e-16 * fmax(zn, 1e-300)) { z = zn; break; }
    z = zn;
  }
  return z;
}

// ------------------------------------------------------------------ (a1) right-hand side, BC Eqs. 27-31
struct OrbitConst { double twoPiMs, Cnu, Ce, a, sp; };

// rates of (nu, gam_c, e, alp_c); Phi_c' = nu.  Angles in cycles (reading D2).
DEVINL void rhs(const OrbitConst& w, double nu, double e, double* fnu, double* fgam, double* fe, double* falp) {
  const double x = w.twoPiMs * nu;
  const double cb = cbrt_polished(x);
  const double u = cb * cb;
  const double e2 = e * e;
  const double q = 1.0 - e2;
  const double rq = 1.0 / q;
  const double sq = sqrt(q);
  const double rsq = sq * rq;          // q^{-1/2}
  const double x2 = x * x;
  const double x83 = x2 * u, x113 = x83 * x;
  const double rq2 = rq * rq;
  // nu'
  {
    double t0 = fma(e2, fma(e2, 37.0 / 96.0, 73.0 / 24.0), 1.0) * q;
    double t1 = u * fma(e2, fma(e2, fma(e2, -13147.0 / 5376.0, -3885.0 / 128.0), -2561.0 / 224.0), 1273.0 / 336.0);
    double t2 = x * w.sp * rsq * fma(e2, fma(e2, fma(e2, 65.0 / 64.0, 3143.0 / 96.0), 1211.0 / 24.0), 73.0 / 12.0);
    *fnu = w.Cnu * x113 * (rq2 * rq2 * rsq) * (t0 + t1 - t2);
  }
  // gamma~'/2pi
  {
    double uq = u * rq;
    *fgam = 3.0 * nu * uq * fma(uq, 0.25 * fma(e2, -15.0, 26.0), 1.0) - 6.0 * nu * w.sp * x * (rq * rsq);
  }
  // e'
  {
    double t0 = fma(e2, 121.0, 304.0) * q * fma(u, 12.0, 1.0);
    double t1 = u * fma(e2, fma(e2, -25211.0, 12.0 * 9082.0), 8.0 * 16705.0) * (1.0 / 56.0);
    double t2 = w.sp * x113 * (rq2 * rq2) * fma(e2, fma(e2, 263.0 / 10.0, 5032.0 / 15.0), 1364.0 / 5.0);
    *fe = e * w.Ce * (t2 - (1.0 / 15.0) * x83 * (rq2 * rq * rsq) * (t0 - t1));
  }
  *falp = 2.0 * nu * w.a * x * (rq * rsq);
}

DEVINL bool plunged(const OrbitConst& w, double nu, double e) {
  // nu >= nu_LSO(e) = ((1-e^2)/(6+2e))^{3/2} / (2 pi M), division- and root-free
  double x = w.twoPiMs * nu, q = 1.0 - e * e, d = 6.0 + 2.0 * e;
  return !(x * x * d * d * d < q * q * q);
}

struct RkOut { double d[5]; double k1[5]; };

DEVINL void rk4_increment(const OrbitConst& w, const double y[5], double h, RkOut& o) {
  double k2[5], k3[5], k4[5];
  o.k1[0] = y[1];
  rhs(w, y[1], y[3], &o.k1[1], &o.k1[2], &o.k1[3], &o.k1[4]);
  double hh = 0.5 * h;
  double nu = fma(hh, o.k1[1], y[1]), e = fma(hh, o.k1[3], y[3]);
  k2[0] = nu;
  rhs(w, nu, e, &k2[1], &k2[2], &k2[3], &k2[4]);
  nu = fma(hh, k2[1], y[1]); e = fma(hh, k2[3], y[3]);
  k3[0] = nu;
  rhs(w, nu, e, &k3[1], &k3[2], &k3[3], &k3[4]);
  nu = fma(h, k3[1], y[1]); e = fma(h, k3[3], y[3]);
  k4[0] = nu;
  rhs(w, nu, e, &k4[1], &k4[2], &k4[3], &k4[4]);
#pragma unroll
  for (int q = 0; q < 5; ++q) o.d[q] = (h / 6.0) * (o.k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
}

struct OrbitArgs {
  const double* params;   // [K][17]
  int K;
  int64_t N;
  double dt;
  int S;
  int64_t Nc, Nn;
  int n_max;
  double tH, Om;          // Hubble time [s], Omega_m
  double* wc;             // [K][WC_STRIDE]
  double* nodes;          // [K][Nn][NODE_STRIDE]
  int32_t* jpl;           // [K] first plunged node (index j), Nn if none
  int32_t* status;        // [K]
  uint8_t* mterms;        // [K][EMRI_NMAX_CAP+1] Bessel series lengths per harmonic
};

DEVINL void store_node(double* row, const double y[5], const double k1[5], const double d[5]) {
  double2* r = reinterpret_cast<double2*>(row);
  r[0] = make_double2(y[0], y[1]);
  r[1] = make_double2(y[2], y[3]);
  r[2] = make_double2(y[4], k1[0]);
  r[3] = make_double2(k1[1], k1[2]);
  r[4] = make_double2(k1[3], k1[4]);
  r[5] = make_double2(d[0], d[1]);
  r[6] = make_double2(d[2], d[3]);
  r[7] = make_double2(d[4], 0.0);
}

__global__ void __launch_bounds__(32) orbit_kernel(OrbitArgs a) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= a.K) return;
  const double* p = a.params + (size_t)k * EMRI_NPAR;
  double* wc = a.wc + (size_t)k * WC_STRIDE;
  double* nodes = a.nodes + (size_t)k * a.Nn * NODE_STRIDE;
  const double Delta = a.S * a.dt;
  int status = 0;
  int32_t jpl = (int32_t)a.Nn;

  // ---- (a0) validity and per-walker scalars
  bool ok = true;
#pragma unroll
  for (int i = 0; i < EMRI_NPAR; ++i) ok = ok && isfinite(p[i]);
  ok = ok && p[P_M] > 0.0 && p[P_MU] > 0.0 && p[P_DL] > 0.0 && p[P_E0] >= 0.0 && p[P_E0] < 1.0 &&
       fabs(p[P_A]) <= 1.0 && p[P_NU0] > 0.0;
  double Xi = 1.0, z = 0.0, dT = 0.0, amp = 0.0;
  const double Ms = p[P_M] * kMsunSec, mus = p[P_MU] * kMsunSec;
  if (ok) {
    const double Ds = p[P_DL] * kGpcSec;
    z = z_of_dL(Ds, a.tH, a.Om);
    Xi = p[P_XI0] + (1.0 - p[P_XI0]) * pow(1.0 + z, -p[P_NXI]);     // Eq. 6
    ok = (Xi > 0.0) && isfinite(Xi);
    if (ok) {
      double I1, I2;
      cosmo_integrals(z, a.Om, &I1, &I2);
      dT = -p[P_DELT] * (a.tH * I2);                                 // reading R9
      amp = mus / (Xi * Ds);                                         // d_GW = Xi d_EM (Eq. 5)
    }
  }
  if (!ok) status |= EMRI_ST_BADPARAM;

  OrbitConst oc;
  oc.twoPiMs = kTwoPi * Ms;
  oc.Cnu = 96.0 / (10.0 * kPi) * (mus / (Ms * Ms * Ms));
  oc.Ce = mus / (Ms * Ms);
  oc.a = p[P_A];
  double sl, cl;
  sincos(p[P_LAM], &sl, &cl);
  oc.sp = p[P_A] * cl;
  {
    double sS, cS, sK, cK, sphS, cphS, sphK, cphK;
    sincos(p[P_THS], &sS, &cS);
    sincos(p[P_THK], &sK, &cK);
    sincos(p[P_PHS], &sphS, &cphS);
    sincos(p[P_PHK], &sphK, &cphK);
    // L^(alpha) = A0 + A1 cos(alpha) + A2 sin(alpha)   (BC Eqs. 19-21)
    const double A0x = sK * cphK * cl, A0y = sK * sphK * cl, A0z = cK * cl;
    const double A1x = -cphK * cK * sl, A1y = -sphK * cK * sl, A1z = sK * sl;
    const double A2x = sphK * sl, A2y = -cphK * sl;
    const double nx = sS * cphS, ny = sS * sphS, nz = cS;
    const double Sn = cS * cK + sS * sK * (cphS * cphK + sphS * sphK);
    wc[WC_TWOPIMS] = oc.twoPiMs; wc[WC_CNU] = oc.Cnu; wc[WC_CE] = oc.Ce; wc[WC_A] = oc.a; wc[WC_SP] = oc.sp;
    wc[WC_AMP] = amp; wc[WC_DT] = dT; wc[WC_SIGMA] = dT / Delta; wc[WC_DOP] = kAuSec * sS;
    wc[WC_CPHS] = cphS; wc[WC_SPHS] = sphS; wc[WC_CS] = cS; wc[WC_SS] = sS;
    wc[WC_LN0] = A0x * nx + A0y * ny + A0z * nz;
    wc[WC_LN1] = A1x * nx + A1y * ny + A1z * nz;
    wc[WC_LN2] = A2x * nx + A2y * ny;
    wc[WC_CL] = cl; wc[WC_SN] = Sn;
    wc[WC_B1] = sS * (sphK * cphS - cphK * sphS) * sl;               // sin(thS) sin(phK - phS) sin(lam)
    wc[WC_B2] = (Sn * cK - cS) / sK * sl;
    wc[WC_A0X] = A0x; wc[WC_A0Y] = A0y; wc[WC_A0Z] = A0z;
    wc[WC_A1X] = A1x; wc[WC_A1Y] = A1y; wc[WC_A1Z] = A1z;
    wc[WC_A2X] = A2x; wc[WC_A2Y] = A2y;
    wc[WC_Z] = z; wc[WC_XI] = Xi;
  }
  if (ok && !(fabs(dT) <= Delta)) status |= EMRI_ST_DELAY;          // reading R20

  // ---- (a1) RK4 on the coarse grid
  double y[5] = {frac(p[P_PHI0] / kTwoPi), p[P_NU0], frac(p[P_GAM0] / kTwoPi), p[P_E0], frac(p[P_ALP0] / kTwoPi)};
  double emax = ok ? y[3] : 0.0;
  const double zero5[5] = {0, 0, 0, 0, 0};
  bool run = ok;
  if (run && plunged(oc, y[1], y[3])) { status |= EMRI_ST_PLUNGE; jpl = 0; run = false; }
  if (!run) {
    for (int64_t m = 0; m < a.Nn; ++m) store_node(nodes + m * NODE_STRIDE, zero5, zero5, zero5);
  } else {
    RkOut r;
    // backward guard step: node -1
    rk4_increment(oc, y, -Delta, r);
    double ym[5] = {frac(y[0] + r.d[0]), y[1] + r.d[1], frac(y[2] + r.d[2]), y[3] + r.d[3], frac(y[4] + r.d[4])};
    bool okm = isfinite(ym[0]) && isfinite(ym[1]) && isfinite(ym[2]) && isfinite(ym[3]) && isfinite(ym[4]) &&
               ym[3] >= 0.0 && ym[3] < 1.0 && ym[1] > 0.0;
    if (!okm) {
      status |= EMRI_ST_STATE;
      for (int64_t m = 0; m < a.Nn; ++m) store_node(nodes + m * NODE_STRIDE, zero5, zero5, zero5);
    } else {
      double km[5], dm[5];
      km[0] = ym[1];
      rhs(oc, ym[1], ym[3], &km[1], &km[2], &km[3], &km[4]);
#pragma unroll
      for (int q = 0; q < 5; ++q) dm[q] = -r.d[q];
      store_node(nodes, ym, km, dm);
      emax = fmax(emax, ym[3]);
      // forward sweep; nu and e are Kahan-compensated (reading D3)
      double comp_nu = 0.0, comp_e = 0.0;
      const int64_t last = a.Nc + 1;          // node index j of the last node (G = 1)
      for (int64_t j = 0; j <= last; ++j) {
        double* row = nodes + (j + 1) * NODE_STRIDE;
        if (j == last) {
          double k1[5];
          k1[0] = y[1];
          rhs(oc, y[1], y[3], &k1[1], &k1[2], &k1[3], &k1[4]);
          store_node(row, y, k1, zero5);
          break;
        }
        rk4_increment(oc, y, Delta, r);
        store_node(row, y, r.k1, r.d);
        double yn[5];
        yn[0] = frac(y[0] + r.d[0]);
        yn[2] = frac(y[2] + r.d[2]);
        yn[4] = frac(y[4] + r.d[4]);
        { double t = r.d[1] - comp_nu, s = y[1] + t; comp_nu = (s - y[1]) - t; yn[1] = s; }
        { double t = r.d[3] - comp_e, s = y[3] + t; comp_e = (s - y[3]) - t; yn[3] = s; }
        bool okn = isfinite(yn[0]) && isfinite(yn[1]) && isfinite(yn[2]) && isfinite(yn[3]) && isfinite(yn[4]) &&
                   yn[3] >= 0.0 && yn[3] < 1.0 && yn[1] > 0.0;
        bool pl = okn && plunged(oc, yn[1], yn[3]);
        if (!okn || pl) {
          status |= okn ? EMRI_ST_PLUNGE : EMRI_ST_STATE;
          jpl = (int32_t)(j + 1);
          // nodes from j_pl on are copies of node j_pl - 1 with zero increments
          for (int64_t m = j + 1; m <= last; ++m) store_node(nodes + (m + 1) * NODE_STRIDE, y, r.k1, zero5);
          break;
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) y[q] = yn[q];
      }
    }
  }
  wc[WC_EMAX] = emax;
  a.jpl[k] = jpl;
  a.status[k] = status;
  // Bessel series lengths: smallest M with prod_{i<=M} y/(i(i+n+1)) < 2^-58, y = (n emax/2)^2
  uint8_t* mt = a.mterms + (size_t)k * (EMRI_NMAX_CAP + 1);
  for (int n = 1; n <= a.n_max; ++n) {
    double yy = 0.25 * n * n * emax * emax, term = 1.0;
    int M = 1;
    while (M < MCAP) {
      term *= yy / ((double)M * (double)(M + n + 1));
      ++M;                      // M coefficients cover powers 0..M-1; `term` is the size of power M-1
      if (term < 3.5e-18) break;
    }
    mt[n] = (uint8_t)M;
  }
}

// ------------------------------------------------------------------ (b) synthesis
struct SynthArgs {
  const double* wc;
  const double* nodes;
  const int32_t* jpl;
  const int32_t* status;
  const uint8_t* mterms;
  const double2* series;   // [n_max+1][MCAP] {coef for order n+1, coef for order n+2} in powers of e^2
  const double* ncoef;     // [n_max+1][NCOEF]
  int k0, K;               // walkers k0 .. k0+K-1
  int64_t N;
  double dt;
  int S, logS;
  int64_t Nn;
  int n_max;
  double* outI;            // row of walker k0+i at outI + i*pitch
  double* outII;
  int64_t pitch;
  int64_t tiles_per_walker;
};

struct Sample {
  double e2, e4, c1, s1;     // e^2, e^4, cos/sin of Phi_tot
  double cn, sn;             // cos/sin(n Phi_tot)
  double Sa, Sb, Sc;
};

// cubic Hermite of the five orbital quantities at fraction s of interval j (node row jj = j+1)
DEVINL void hermite5(const double* __restrict__ nodes, int64_t jj, double s, double Delta, double out[5]) {
  const double2* r0 = reinterpret_cast<const double2*>(nodes + jj * NODE_STRIDE);
  const double2* r1 = r0 + NODE_STRIDE / 2;
  double2 v01 = __ldg(r0), v23 = __ldg(r0 + 1), v4m0 = __ldg(r0 + 2), m12 = __ldg(r0 + 3), m34 = __ldg(r0 + 4),
          d01 = __ldg(r0 + 5), d23 = __ldg(r0 + 6), d4 = __ldg(r0 + 7);
  double2 n4m0 = __ldg(r1 + 2), n12 = __ldg(r1 + 3), n34 = __ldg(r1 + 4);
  const double s2 = s * s, s3 = s2 * s;
  const double b = 3.0 * s2 - 2.0 * s3;
  const double c0 = Delta * (s3 - 2.0 * s2 + s), c1 = Delta * (s3 - s2);
  out[0] = v01.x + fma(b, d01.x, fma(c0, v4m0.y, c1 * n4m0.y));
  out[1] = v01.y + fma(b, d01.y, fma(c0, m12.x, c1 * n12.x));
  out[2] = v23.x + fma(b, d23.x, fma(c0, m12.y, c1 * n12.y));
  out[3] = v23.y + fma(b, d23.y, fma(c0, m34.x, c1 * n34.x));
  out[4] = v4m0.x + fma(b, d4.x, fma(c0, m34.y, c1 * n34.y));
}

struct Projection { double FIp, FIx, FIIp, FIIx, c2g, s2g, sq, A, Ln, e; };

// everything of one sample that does not depend on the harmonic index
DEVINL void sample_setup(const double* __restrict__ w, const double* __restrict__ nodes, int64_t i, int S, int logS,
                         double dt, int32_t jpl, bool* live, Sample* sm, Projection* pr) {
  // source-time split (reading D4)
  int64_t j = i >> logS;
  double s = (double)(i & (S - 1)) * (1.0 / (double)S) - w[WC_SIGMA];
  if (s < 0.0) { s += 1.0; j -= 1; } else if (s >= 1.0) { s -= 1.0; j += 1; }
  *live = (j + 1 < (int64_t)jpl);
  double orb[5];
  hermite5(nodes, j + 1, s, S * dt, orb);
  const double Phic = orb[0], nu = orb[1], gamc = orb[2], e = orb[3], alpc = orb[4];
  double sa, ca, s2gt, c2gt, spb, cpb;
  sincospi(2.0 * alpc, &sa, &ca);
  sincospi(4.0 * gamc, &s2gt, &c2gt);
  sincospi(2.0 * frac(((double)i * dt) / kYearSec), &spb, &cpb);
  // orbital-plane normal and its projections (BC 19-21)
  const double Lx = fma(w[WC_A2X], sa, fma(w[WC_A1X], ca, w[WC_A0X]));
  const double Ly = fma(w[WC_A2Y], sa, fma(w[WC_A1Y], ca, w[WC_A0Y]));
  const double Lz = fma(w[WC_A1Z], ca, w[WC_A0Z]);
  const double Ln = fma(w[WC_LN2], sa, fma(w[WC_LN1], ca, w[WC_LN0]));
  // beta (BC 22-24): tan(beta) = Ns/Nc
  const double Ns = fma(w[WC_CL], Ln, -w[WC_SN]);
  const double Nc = fma(w[WC_B2], sa, w[WC_B1] * ca);
  const double den_b = fma(Nc, Nc, Ns * Ns);
  // detector time quantities
  const double cphS = w[WC_CPHS], sphS = w[WC_SPHS], cS = w[WC_CS], sS = w[WC_SS];
  const double cd = fma(cpb, cphS, spb * sphS), sd = fma(spb, cphS, -cpb * sphS);
  const double cthd = fma(-kHalfSqrt3 * sS, cd, 0.5 * cS);
  const double Pq = fma(sS, cd, kSqrt3 * cS), Qq = 2.0 * sS * sd;
  const double den_a = fma(Pq, Pq, Qq * Qq);
  const double Npsi = fma(-cthd, Ln, fma(-kHalfSqrt3, fma(Lx, cpb, Ly * spb), 0.5 * Lz));
  const double Dpsi = 0.5 * sS * fma(Ly, cphS, -Lx * sphS)
                      - kHalfSqrt3 * (cpb * fma(Lz * sS, sphS, -cS * Ly) + spb * fma(cS, Lx, -Lz * sS * cphS));
  const double den_p = fma(Npsi, Npsi, Dpsi * Dpsi);
  // one division for the three normalisations
  const double bp = den_b * den_p;
  const double inv = 1.0 / (bp * den_a);
  const double ib = (den_b > 0.0) ? inv * (den_a * den_p) : 0.0;
  const double ia = inv * bp;
  const double ip = (den_p > 0.0) ? inv * (den_a * den_b) : 0.0;
  double c2b = fma(Nc, Nc, -Ns * Ns) * ib, s2b = 2.0 * Ns * Nc * ib;
  if (!(den_b > 0.0)) { c2b = 1.0; s2b = 0.0; }                     // reading R16: beta = 0
  const double c2a = fma(Qq, Qq, -Pq * Pq) * ia, s2a = 2.0 * Pq * Qq * ia;
  double c2s = fma(Dpsi, Dpsi, -Npsi * Npsi) * ip, s2s = 2.0 * Npsi * Dpsi * ip;
  if (!(den_p > 0.0)) { c2s = 1.0; s2s = 0.0; }
  const double c2g = fma(c2gt, c2b, -s2gt * s2b), s2g = fma(s2gt, c2b, c2gt * s2b);
  const double c2pb = fma(cpb, cpb, -spb * spb), s2pb = 2.0 * cpb * spb;
  const double c2p = fma(c2pb, c2a, -s2pb * s2a), s2p = fma(s2pb, c2a, c2pb * s2a);
  const double hh = 0.5 * fma(cthd, cthd, 1.0);
  pr->FIp = fma(hh * c2p, c2s, -cthd * s2p * s2s);
  pr->FIx = fma(hh * c2p, s2s, cthd * s2p * c2s);
  pr->FIIp = fma(hh * s2p, c2s, cthd * c2p * s2s);
  pr->FIIx = fma(hh * s2p, s2s, -cthd * c2p * c2s);
  // amplitude A = (2 pi M nu)^{2/3} mu / (Xi D)   (BC 10 with Eqs. 4-6 folded in)
  const double cb = cbrt(w[WC_TWOPIMS] * nu);
  pr->A = cb * cb * w[WC_AMP];
  pr->Ln = Ln;
  pr->sq = sqrt(fma(-e, e, 1.0));
  pr->c2g = c2g; pr->s2g = s2g; pr->e = e;
  // Doppler-shifted phase in cycles (BC 25)
  const double Phit = frac(fma(nu * w[WC_DOP], cd, Phic));
  sincospi(2.0 * Phit, &sm->s1, &sm->c1);
  sm->e2 = e * e;
  sm->e4 = sm->e2 * sm->e2;
  sm->cn = sm->c1; sm->sn = sm->s1;
  sm->Sa = 0.0; sm->Sb = 0.0; sm->Sc = 0.0;
}

DEVINL void sample_finish(const Sample& sm, const Projection& pr, bool live, double* hI, double* hII) {
  const double Ln2 = pr.Ln * pr.Ln;
  const double sb = pr.sq * sm.Sb;
  // A+ = A {(1+Ln^2)(c2g Sa - s2g sq Sb) + 2 (1-Ln^2) Sc},  Ax = -2 A Ln (sq Sb c2g + Sa s2g)   (BC 7-9 summed over n)
  const double Ap = pr.A * fma(1.0 + Ln2, fma(pr.c2g, sm.Sa, -pr.s2g * sb), 2.0 * (1.0 - Ln2) * sm.Sc);
  const double Ax = -2.0 * pr.A * pr.Ln * fma(sb, pr.c2g, sm.Sa * pr.s2g);
  *hI = live ? kHalfSqrt3 * fma(pr.FIp, Ap, pr.FIx * Ax) : 0.0;
  *hII = live ? kHalfSqrt3 * fma(pr.FIIp, Ap, pr.FIIx * Ax) : 0.0;
}

__global__ void __launch_bounds__(SYNTH_THREADS, 4) synth_kernel(SynthArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* s_series = reinterpret_cast<double2*>(smem_raw);                         // [(n_max+1)*MCAP]
  double* s_ncoef = reinterpret_cast<double*>(s_series + (size_t)(a.n_max + 1) * MCAP);   // [(n_max+1)*NCOEF]
  double* s_wc = s_ncoef + (size_t)(a.n_max + 1) * NCOEF;                           // [WC_STRIDE]
  __shared__ uint8_t s_mt[EMRI_NMAX_CAP + 1];

  for (int i = threadIdx.x; i < (a.n_max + 1) * MCAP; i += blockDim.x) s_series[i] = a.series[i];
  for (int i = threadIdx.x; i < (a.n_max + 1) * NCOEF; i += blockDim.x) s_ncoef[i] = a.ncoef[i];

  const int64_t total = (int64_t)a.K * a.tiles_per_walker;
  int cur_k = -1;
  for (int64_t t = blockIdx.x; t < total; t += gridDim.x) {
    const int kl = (int)(t / a.tiles_per_walker);
    const int64_t tile = t - (int64_t)kl * a.tiles_per_walker;
    const int k = a.k0 + kl;
    if (k != cur_k) {
      __syncthreads();
      if (threadIdx.x < WC_STRIDE) s_wc[threadIdx.x] = a.wc[(size_t)k * WC_STRIDE + threadIdx.x];
      if (threadIdx.x <= EMRI_NMAX_CAP) s_mt[threadIdx.x] = a.mterms[(size_t)k * (EMRI_NMAX_CAP + 1) + threadIdx.x];
      cur_k = k;
      __syncthreads();
    }
    const int64_t i0 = tile * TILE + 2 * threadIdx.x;
    if (i0 >= a.N) continue;
    double* oI = a.outI + (size_t)kl * a.pitch + i0;
    double* oII = a.outII + (size_t)kl * a.pitch + i0;
    const int32_t st = a.status[k];
    if (st & (EMRI_ST_BADPARAM | EMRI_ST_DELAY | EMRI_ST_STATE)) {
      *reinterpret_cast<double2*>(oI) = make_double2(0.0, 0.0);
      *reinterpret_cast<double2*>(oII) = make_double2(0.0, 0.0);
      continue;
    }
    const double* nodes = a.nodes + (size_t)k * a.Nn * NODE_STRIDE;
    const int32_t jpl = a.jpl[k];
    Sample A, B;
    Projection pa, pb;
    bool la, lb;
    sample_setup(s_wc, nodes, i0, a.S, a.logS, a.dt, jpl, &la, &A, &pa);
    sample_setup(s_wc, nodes, i0 + 1, a.S, a.logS, a.dt, jpl, &lb, &B, &pb);

    // ---- harmonic n = 1 (brackets odd in e; J_{-1} = -J_1)
    {
      const int M = s_mt[1];
      const double2* tab = s_series + MCAP;
      double2 c = tab[M - 1];
      double j2a = c.x, j3a = c.y, j2b = c.x, j3b = c.y;     // scaled J_2, J_3
      for (int m = M - 2; m >= 0; --m) {
        c = tab[m];
        j2a = fma(j2a, A.e2, c.x); j3a = fma(j3a, A.e2, c.y);
        j2b = fma(j2b, B.e2, c.x); j3b = fma(j3b, B.e2, c.y);
      }
      const double* kc = s_ncoef + NCOEF;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        Sample& s = h ? B : A;
        const double e = h ? pb.e : pa.e;
        const double j2 = h ? j2b : j2a, j3 = h ? j3b : j3a;
        const double j1 = fma(-s.e2 * kc[8], j3, j2);
        const double j0 = fma(-s.e2 * kc[9], j2, j1);
        const double ba = fma(s.e2, fma(-1.0 / 48.0, j3, 0.25 * j2), fma(0.5, j1, -2.0 * j0));
        const double bb = fma(s.e2 * (1.0 / 48.0), j3, -1.5 * j1);
        const double tc = e * s.cn, ts = e * s.sn;
        s.Sa = ba * tc; s.Sb = bb * ts; s.Sc = 0.5 * j1 * tc;
        const double cn = fma(s.cn, s.c1, -s.sn * s.s1), sn = fma(s.sn, s.c1, s.cn * s.s1);
        s.cn = cn; s.sn = sn;
      }
    }
    // ---- harmonics n = 2 .. n_max
    double ta = 1.0, tb = 1.0;     // t'_n = (n e/2)^{n-2}/(n-2)!
    for (int n = 2; n <= a.n_max; ++n) {
      const int M = s_mt[n];
      const double2* tab = s_series + n * MCAP;
      double2 c = tab[M - 1];
      double p1a = c.x, p2a = c.y, p1b = c.x, p2b = c.y;     // scaled J_{n+1}, J_{n+2}
      for (int m = M - 2; m >= 0; --m) {
        c = tab[m];
        p1a = fma(p1a, A.e2, c.x); p2a = fma(p2a, A.e2, c.y);
        p1b = fma(p1b, B.e2, c.x); p2b = fma(p2b, B.e2, c.y);
      }
      const double* kc = s_ncoef + n * NCOEF;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        Sample& s = h ? B : A;
        const double p1 = h ? p1b : p1a, p2 = h ? p2b : p2a;
        double& t = h ? tb : ta;
        const double j0 = fma(-s.e2 * kc[8], p2, p1);        // scaled J_n
        const double jm1 = fma(-s.e2 * kc[9], p1, j0);       // scaled J_{n-1}
        const double jm2 = fma(-s.e2 * kc[10], j0, jm1);     // scaled J_{n-2}
        const double ba = fma(s.e4, fma(kc[4], p2, kc[3] * p1), fma(s.e2, fma(kc[2], j0, kc[1] * jm1), kc[0] * jm2));
        const double bb = fma(s.e4 * kc[6], p2, fma(s.e2 * kc[5], j0, kc[0] * jm2));
        const double bc = s.e2 * kc[7] * j0;
        const double tc = t * s.cn, ts = t * s.sn;
        s.Sa = fma(ba, tc, s.Sa); s.Sb = fma(bb, ts, s.Sb); s.Sc = fma(bc, tc, s.Sc);
        const double cn = fma(s.cn, s.c1, -s.sn * s.s1), sn = fma(s.sn, s.c1, s.cn * s.s1);
        s.cn = cn; s.sn = sn;
        t *= (h ? pb.e : pa.e) * kc[11];
      }
    }
    double hIa, hIIa, hIb, hIIb;
    sample_finish(A, pa, la, &hIa, &hIIa);
    sample_finish(B, pb, lb, &hIb, &hIIb);
    *reinterpret_cast<double2*>(oI) = make_double2(hIa, hIb);
    *reinterpret_cast<double2*>(oII) = make_double2(hIIa, hIIb);
  }
}

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

// ------------------------------------------------------------------ stretch move (configs[4])
DEVINL uint32_t mulhilo(uint32_t a, uint32_t b, uint32_t* hi) {
  uint64_t p = (uint64_t)a * b;
  *hi = (uint32_t)(p >> 32);
  return (uint32_t)p;
}
// Philox4x32-10 (Salmon et al. 2011)
DEVINL void philox4x32(uint32_t c[4], uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0, hi1;
    uint32_t lo0 = mulhilo(0xD2511F53u, c[0], &hi0);
    uint32_t lo1 = mulhilo(0xCD9E8D57u, c[2], &hi1);
    uint32_t n0 = hi1 ^ c[1] ^ k0, n1 = lo1, n2 = hi0 ^ c[3] ^ k1, n3 = lo0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
}
DEVINL double u53(uint32_t hi, uint32_t lo) {      // uniform in (0,1): (53-bit integer + 0.5) / 2^53
  uint64_t v = (((uint64_t)hi << 32) | lo) >> 11;
  return ((double)v + 0.5) * (1.0 / 9007199254740992.0);
}

struct StretchArgs {
  double* X; double* logL; int K;
  const double* lo; const double* hi;
  double a; uint64_t seed; int64_t step; int half;
  double* Y;        // [K/2][17] proposals
  double* zbuf;     // [K/2] z
  double* lnu;      // [K/2] ln u'
  int32_t* inbox;   // [K/2]
  int32_t* partner; // [K/2]
  const double* logLY;
  int32_t* accepted;
  double* log_buf;
};

__global__ void stretch_propose_kernel(StretchArgs s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int H = s.K / 2;
  if (i >= H) return;
  const int k = s.half * H + i, ob = (1 - s.half) * H;
  uint32_t c[4] = {(uint32_t)s.step, (uint32_t)((uint64_t)s.step >> 32), (uint32_t)(2 * i + s.half), 0u};
  philox4x32(c, (uint32_t)s.seed, (uint32_t)(s.seed >> 32));
  const double u1 = u53(c[0], c[1]), u2 = u53(c[2], c[3]);
  uint32_t c2[4] = {(uint32_t)s.step, (uint32_t)((uint64_t)s.step >> 32), (uint32_t)(2 * i + s.half), 1u};
  philox4x32(c2, (uint32_t)s.seed, (uint32_t)(s.seed >> 32));
  const double u3 = u53(c2[0], c2[1]);
  int j = ob + min((int)(u1 * H), H - 1);
  const double sz = fma(s.a - 1.0, u2, 1.0);
  const double z = sz * sz / s.a;
  bool in = true;
  for (int q = 0; q < EMRI_NPAR; ++q) {
    const double xk = s.X[(size_t)k * EMRI_NPAR + q], xj = s.X[(size_t)j * EMRI_NPAR + q];
    const bool fixed = !(s.lo[q] < s.hi[q]);
    const double y = fixed ? xk : fma(z, xk - xj, xj);
    s.Y[(size_t)i * EMRI_NPAR + q] = y;
    in = in && (fixed || (y >= s.lo[q] && y <= s.hi[q]));
  }
  s.zbuf[i] = z; s.lnu[i] = log(u3); s.inbox[i] = in ? 1 : 0; s.partner[i] = j;
}

__global__ void stretch_accept_kernel(StretchArgs s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int H = s.K / 2;
  if (i >= H) return;
  const int k = s.half * H + i;
  int nfree = 0;
  for (int q = 0; q < EMRI_NPAR; ++q) nfree += (s.lo[q] < s.hi[q]) ? 1 : 0;
  const double lY = s.inbox[i] ? s.logLY[i] : -INFINITY;
  const double lnq = (double)(nfree - 1) * log(s.zbuf[i]) + lY - s.logL[k];
  const bool acc = isfinite(lY) && (s.lnu[i] < lnq);
  if (s.log_buf) {
    double* lb = s.log_buf + (size_t)i * (EMRI_NPAR + 4);
    for (int q = 0; q < EMRI_NPAR; ++q) lb[q] = s.Y[(size_t)i * EMRI_NPAR + q];
    lb[EMRI_NPAR] = s.zbuf[i]; lb[EMRI_NPAR + 1] = s.lnu[i]; lb[EMRI_NPAR + 2] = lY; lb[EMRI_NPAR + 3] = (double)s.partner[i];
  }
  if (acc) {
    for (int q = 0; q < EMRI_NPAR; ++q) s.X[(size_t)k * EMRI_NPAR + q] = s.Y[(size_t)i * EMRI_NPAR + q];
    s.logL[k] = lY;
  }
  if (s.accepted) s.accepted[k] = acc ? 1 : 0;
}

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
__global__ void __launch_bounds__(256) hbm_probe_kernel(const double2* in, int64_t n, double* out) {
  double acc = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double2 v = __ldcs(in + i);
    acc += v.x + v.y;
  }
  if (acc == 123.456) out[0] = acc;
}

}  // namespace

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
  double2* d_series = nullptr;
  double* d_ncoef = nullptr;
  int32_t* d_jpl = nullptr;
  int32_t* d_status = nullptr;
  uint8_t* d_mterms = nullptr;
  // host-variant staging
  double* d_params = nullptr;
  double* d_data = nullptr;
  double* d_logL = nullptr;
  bool data_loaded = false;
  // stretch move scratch
  double* d_Y = nullptr; double* d_z = nullptr; double* d_lnu = nullptr; double* d_logLY = nullptr;
  int32_t* d_inbox = nullptr; int32_t* d_partner = nullptr;
  // cuFFT
  std::map<int, cufftHandle> fft;
  void* d_fftwork = nullptr;
  size_t fftwork_bytes = 0;
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

template <class T> int dev_alloc(emri_plan* p, T** ptr, size_t count) {
  if (*ptr) { cudaFree(*ptr); *ptr = nullptr; }
  if (count == 0) return EMRI_OK;
  cudaError_t e = cudaMalloc((void**)ptr, count * sizeof(T));
  if (e != cudaSuccess) { p->last_err = (int)e; *ptr = nullptr; cudaGetLastError(); return EMRI_ENOMEM; }
  p->bytes += (int64_t)(count * sizeof(T));
  return EMRI_OK;
}

// Bessel series and per-harmonic constants, built in long double
void build_tables(int n_max, std::vector<double2>& series, std::vector<double>& ncoef) {
  series.assign((size_t)(n_max + 1) * MCAP, make_double2(0.0, 0.0));
  ncoef.assign((size_t)(n_max + 1) * NCOEF, 0.0);
  for (int n = 1; n <= n_max; ++n) {
    // scaled Bessel function Jhat_k(n e) = sum_m (-n^2/4)^m / (m! (k+1)_m) (e^2)^m, k = n+1 and n+2
    long double y = -0.25L * n * n;
    long double c1 = 1.0L, c2 = 1.0L;
    for (int m = 0; m < MCAP; ++m) {
      if (m > 0) {
        c1 *= y / ((long double)m * (long double)(m + n + 1));
        c2 *= y / ((long double)m * (long double)(m + n + 2));
      }
      series[(size_t)n * MCAP + m] = make_double2((double)c1, (double)c2);
    }
    double* kc = &ncoef[(size_t)n * NCOEF];
    long double nn = n;
    kc[8] = (double)(nn * nn / (4.0L * (nn + 1) * (nn + 2)));        // J_n     from J_{n+1}, J_{n+2}
    kc[9] = (double)(nn * nn / (4.0L * nn * (nn + 1)));              // J_{n-1} from J_n, J_{n+1}
    if (n >= 2) {
      long double r1 = nn / (2 * (nn - 1)), r2 = nn / (2 * nn), r3 = nn / (2 * (nn + 1)), r4 = nn / (2 * (nn + 2));
      kc[0] = (double)nn;
      kc[1] = (double)(-2 * nn * r1);
      kc[2] = (double)(2 * r1 * r2);
      kc[3] = (double)(2 * nn * r1 * r2 * r3);
      kc[4] = (double)(-nn * r1 * r2 * r3 * r4);
      kc[5] = (double)(-2 * nn * r1 * r2);
      kc[6] = (double)(nn * r1 * r2 * r3 * r4);
      kc[7] = (double)(r1 * r2);
      kc[10] = (double)(nn * nn / (4.0L * (nn - 1) * nn));           // J_{n-2} from J_{n-1}, J_n
      kc[11] = (double)(0.5L * powl((nn + 1) / nn, (long double)(n - 2)) * (nn + 1) / (nn - 1));   // t'_{n+1}/(e t'_n)
    }
  }
}

int alloc_workspace(emri_plan* p) {
  int rc;
  p->Nc = (p->N + p->S - 1) / p->S;
  p->Nn = p->Nc + 3;
  if ((rc = dev_alloc(p, &p->d_nodes, (size_t)p->K_max * p->Nn * NODE_STRIDE))) return rc;
  return EMRI_OK;
}

int alloc_chunk(emri_plan* p) {
  int rc;
  if ((rc = dev_alloc(p, &p->d_hbuf, (size_t)2 * p->chunk * (p->N + 2)))) return rc;
  for (auto& kv : p->fft) cufftDestroy(kv.second);
  p->fft.clear();
  return EMRI_OK;
}

int get_fft(emri_plan* p, int batch, cufftHandle* out) {
  auto it = p->fft.find(batch);
  if (it != p->fft.end()) { *out = it->second; return EMRI_OK; }
  cufftHandle h;
  CKF(cufftCreate(&h));
  CKF(cufftSetAutoAllocation(h, 0));
  long long n[1] = {(long long)p->N};
  long long inembed[1] = {(long long)p->N + 2}, onembed[1] = {(long long)p->N / 2 + 1};
  size_t ws = 0;
  cufftResult r = cufftMakePlanMany64(h, 1, n, inembed, 1, (long long)p->N + 2, onembed, 1, (long long)p->N / 2 + 1,
                                      CUFFT_D2Z, (long long)batch, &ws);
  if (r != CUFFT_SUCCESS) { p->last_err = (int)r; cufftDestroy(h); return EMRI_ECUFFT; }
  if (ws > p->fftwork_bytes) {
    // grow the shared work area; every cached plan is re-pointed at it
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
  OrbitArgs a;
  a.params = params; a.K = K; a.N = p->N; a.dt = p->dt; a.S = p->S; a.Nc = p->Nc; a.Nn = p->Nn; a.n_max = p->n_max;
  a.tH = kMpcMetre / (p->H0 * 1000.0); a.Om = p->Om;
  a.wc = p->d_wc; a.nodes = p->d_nodes; a.jpl = p->d_jpl; a.status = p->d_status; a.mterms = p->d_mterms;
  orbit_kernel<<<(K + 31) / 32, 32, 0, s>>>(a);
  CK(cudaGetLastError());
  return EMRI_OK;
}

int run_synth(emri_plan* p, int k0, int K, double* outI, double* outII, int64_t pitch, cudaStream_t s) {
  SynthArgs a;
  a.wc = p->d_wc; a.nodes = p->d_nodes; a.jpl = p->d_jpl; a.status = p->d_status; a.mterms = p->d_mterms;
  a.series = p->d_series; a.ncoef = p->d_ncoef;
  a.k0 = k0; a.K = K; a.N = p->N; a.dt = p->dt; a.S = p->S; a.logS = p->logS; a.Nn = p->Nn; a.n_max = p->n_max;
  a.outI = outI; a.outII = outII; a.pitch = pitch;
  a.tiles_per_walker = (p->N + TILE - 1) / TILE;
  int64_t total = (int64_t)K * a.tiles_per_walker;
  int grid = (int)std::min<int64_t>(total, p->synth_grid);
  synth_kernel<<<grid, SYNTH_THREADS, p->synth_smem, s>>>(a);
  CK(cudaGetLastError());
  return EMRI_OK;
}

int run_like(emri_plan* p, int k0, int K, const double* H, const double* data_fft, cudaStream_t s) {
  LikeArgs a;
  a.H = reinterpret_cast<const double2*>(H);
  a.D = reinterpret_cast<const double2*>(data_fft);
  a.w = p->d_w; a.partial = p->d_partial; a.k0 = k0; a.K = K; a.Nf = p->Nf; a.n_part = p->n_part;
  int grid = (int)((p->Nf + LL_TILE - 1) / LL_TILE);
  loglike_kernel<<<grid, LL_THREADS, 0, s>>>(a);
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
  std::vector<double2> series;
  std::vector<double> ncoef;
  build_tables(n_max, series, ncoef);

  if ((rc = dev_alloc(p, &p->d_w, (size_t)p->Nf))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_wc, (size_t)K_max * WC_STRIDE))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_jpl, (size_t)K_max))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_status, (size_t)K_max))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_mterms, (size_t)K_max * (EMRI_NMAX_CAP + 1)))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_series, series.size()))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_ncoef, ncoef.size()))) return fail(rc);
  p->n_part = (int)((p->Nf + LL_TILE - 1) / LL_TILE) * LL_WARPS;
  if ((rc = dev_alloc(p, &p->d_partial, (size_t)K_max * p->n_part))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_params, (size_t)K_max * EMRI_NPAR))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_data, (size_t)4 * p->Nf))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_logL, (size_t)K_max))) return fail(rc);
  const size_t H = (size_t)(K_max + 1) / 2 + 1;
  if ((rc = dev_alloc(p, &p->d_Y, H * EMRI_NPAR))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_z, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_lnu, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_logLY, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_inbox, H))) return fail(rc);
  if ((rc = dev_alloc(p, &p->d_partner, H))) return fail(rc);
  if ((rc = alloc_workspace(p))) return fail(rc);
  if ((rc = alloc_chunk(p))) return fail(rc);
  if (cudaMemcpy(p->d_w, w.data(), w.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(p->d_series, series.data(), series.size() * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(p->d_ncoef, ncoef.data(), ncoef.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess)
    return fail(EMRI_ECUDA);

  // persistent grid for the synthesis kernel: resident CTAs per SM x SM count
  p->synth_smem = (size_t)(n_max + 1) * MCAP * sizeof(double2) + (size_t)(n_max + 1) * NCOEF * sizeof(double) +
                  WC_STRIDE * sizeof(double);
  if (cudaFuncSetAttribute(synth_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->synth_smem) != cudaSuccess)
    return fail(EMRI_ECUDA);
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, synth_kernel, SYNTH_THREADS, p->synth_smem) != cudaSuccess ||
      per_sm < 1)
    return fail(EMRI_ECUDA);
  p->synth_grid = per_sm * p->sm_count;
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(EMRI_ECUDA);
  *out = p;
  return EMRI_OK;
}

int emri_plan_destroy(emri_plan* p) {
  if (!p) return EMRI_EINVAL;
  cudaDeviceSynchronize();
  for (auto& kv : p->fft) cufftDestroy(kv.second);
  for (auto e : p->ev) cudaEventDestroy(e);
  void* ptrs[] = {p->d_w, p->d_wc, p->d_nodes, p->d_hbuf, p->d_partial, p->d_series, p->d_ncoef, p->d_jpl, p->d_status,
                  p->d_mterms, p->d_params, p->d_data, p->d_logL, p->d_Y, p->d_z, p->d_lnu, p->d_logLY, p->d_inbox,
                  p->d_partner, p->d_fftwork};
  for (void* q : ptrs) if (q) cudaFree(q);
  delete p;
  return EMRI_OK;
}

int emri_plan_set_cosmology(emri_plan* p, double H0, double Om) {
  if (!p || !(H0 > 0.0) || !(Om > 0.0) || !(Om <= 1.0) || !std::isfinite(H0)) return EMRI_EINVAL;
  p->H0 = H0; p->Om = Om;
  return EMRI_OK;
}

int emri_plan_set_coarse_stride(emri_plan* p, int S) {
  if (!p || S < 2 || S > 65536 || (S & (S - 1))) return EMRI_EINVAL;
  CK(cudaDeviceSynchronize());
  p->S = S;
  p->logS = 0;
  while ((1 << p->logS) < S) ++p->logS;
  if (p->d_nodes) p->bytes -= (int64_t)((size_t)p->K_max * p->Nn * NODE_STRIDE * sizeof(double));
  return alloc_workspace(p);
}

int emri_plan_set_chunk(emri_plan* p, int c) {
  if (!p || c < 1) return EMRI_EINVAL;
  if (c > p->K_max) c = p->K_max;
  CK(cudaDeviceSynchronize());
  if (p->d_hbuf) p->bytes -= (int64_t)((size_t)2 * p->chunk * (p->N + 2) * sizeof(double));
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
  if ((rc = run_synth(p, 0, K, h_I, h_II, p->N, s))) return rc;
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
    double* rows = spectra + (size_t)k0 * 2 * (p->N + 2);
    mark(p, s);
    if ((rc = run_synth(p, k0, kc, rows, rows + (p->N + 2), 2 * (p->N + 2), s))) return rc;
    mark(p, s);
    cufftHandle h;
    if ((rc = get_fft(p, 2 * kc, &h))) return rc;
    CKF(cufftSetStream(h, s));
    CKF(cufftExecD2Z(h, rows, reinterpret_cast<cufftDoubleComplex*>(rows)));
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
  CK(cudaMemcpyAsync(data_fft, d_I, (size_t)p->N * sizeof(double), cudaMemcpyDeviceToDevice, s));
  CK(cudaMemcpyAsync(data_fft + (p->N + 2), d_II, (size_t)p->N * sizeof(double), cudaMemcpyDeviceToDevice, s));
  cufftHandle h;
  int rc = get_fft(p, 2, &h);
  if (rc) return rc;
  CKF(cufftSetStream(h, s));
  CKF(cufftExecD2Z(h, data_fft, reinterpret_cast<cufftDoubleComplex*>(data_fft)));
  return EMRI_OK;
}

int emri_loglike(emri_plan* p, const double* params, int K, const double* data_fft, double* logL, int32_t* status,
                 void* stream) {
  if (!valid_call(p, params, K) || !data_fft || !logL) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  p->ev_used = 0; p->had_like = true;
  mark(p, s);
  int rc = run_orbit(p, params, K, s);
  if (rc) return rc;
  mark(p, s);
  int nch = 0;
  for (int k0 = 0; k0 < K; k0 += p->chunk, ++nch) {
    const int kc = std::min(p->chunk, K - k0);
    mark(p, s);
    if ((rc = run_synth(p, k0, kc, p->d_hbuf, p->d_hbuf + (p->N + 2), 2 * (p->N + 2), s))) return rc;
    mark(p, s);
    cufftHandle h;
    if ((rc = get_fft(p, 2 * kc, &h))) return rc;
    CKF(cufftSetStream(h, s));
    CKF(cufftExecD2Z(h, p->d_hbuf, reinterpret_cast<cufftDoubleComplex*>(p->d_hbuf)));
    mark(p, s);
    if ((rc = run_like(p, k0, kc, p->d_hbuf, data_fft, s))) return rc;
    mark(p, s);
  }
  p->n_chunks_last = nch;
  const double scale = 2.0 * p->dt / (double)p->N;
  loglike_final_kernel<<<(K + 3) / 4, 128, 0, s>>>(p->d_partial, p->n_part, K, scale, p->d_status, logL, status);
  CK(cudaGetLastError());
  return EMRI_OK;
}

int emri_loglike_host(emri_plan* p, const double* params, int K, const double* data_fft, double* logL, int32_t* status,
                      void* stream) {
  if (!valid_call(p, params, K) || !logL) return EMRI_EINVAL;
  if (!data_fft && !p->data_loaded) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CK(cudaMemcpyAsync(p->d_params, params, (size_t)K * EMRI_NPAR * sizeof(double), cudaMemcpyHostToDevice, s));
  if (data_fft) {
    CK(cudaMemcpyAsync(p->d_data, data_fft, (size_t)4 * p->Nf * sizeof(double), cudaMemcpyHostToDevice, s));
    p->data_loaded = true;
  }
  int rc = emri_loglike(p, p->d_params, K, p->d_data, p->d_logL, nullptr, stream);
  if (rc) return rc;
  CK(cudaMemcpyAsync(logL, p->d_logL, (size_t)K * sizeof(double), cudaMemcpyDeviceToHost, s));
  if (status) CK(cudaMemcpyAsync(status, p->d_status, (size_t)K * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
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

int emri_probe_fp64_peak(double* tflops, void* stream) {
  if (!tflops) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return EMRI_ECUDA;
  double* d = nullptr;
  if (cudaMalloc(&d, 8) != cudaSuccess) return EMRI_ENOMEM;
  const int iters = 4096, blocks = sms * 8;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  fp64_probe_kernel<<<blocks, 256, 0, s>>>(d, 64, 1.0);      // warm-up
  double best = 0.0;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, s);
    fp64_probe_kernel<<<blocks, 256, 0, s>>>(d, iters, 1.0);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return EMRI_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    double fl = 2.0 * 64.0 * (double)iters * 256.0 * (double)blocks;
    best = std::max(best, fl / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d);
  *tflops = best;
  return EMRI_OK;
}

int emri_probe_hbm_read(int64_t bytes, double* gbs, void* stream) {
  if (!gbs || bytes < (1 << 20)) return EMRI_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return EMRI_ECUDA;
  double2* buf = nullptr;
  double* d = nullptr;
  const int64_t n = bytes / 16;
  if (cudaMalloc(&buf, (size_t)n * 16) != cudaSuccess) { cudaGetLastError(); return EMRI_ENOMEM; }
  if (cudaMalloc(&d, 8) != cudaSuccess) { cudaFree(buf); return EMRI_ENOMEM; }
  cudaMemsetAsync(buf, 0, (size_t)n * 16, s);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  hbm_probe_kernel<<<sms * 8, 256, 0, s>>>(buf, n, d);
  double best = 0.0;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, s);
    hbm_probe_kernel<<<sms * 8, 256, 0, s>>>(buf, n, d);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(buf); cudaFree(d); return EMRI_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    best = std::max(best, (double)n * 16.0 / (ms * 1e-3) * 1e-9);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(buf); cudaFree(d);
  *gbs = best;
  return EMRI_OK;
}

}  // extern "C"
