// orbit.cuh -- stage (a): per-walker scalars (Eq. 6) and the fixed-step RK4 integration of Eq. 1
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
#pragma once
#include "common.cuh"

namespace {

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
  // f(z) = d_L(z) - D is increasing and convex, so Newton converges monotonically from above after the first step
  // (quadratically: ~6 steps).  The convergence test comes BEFORE the bracket safeguard: a converged step lands on
  // the bracket's edge, and bisecting there would throw the iterate away.
  double lo = 0.0, hi = 20.0;
  double z = fmin(D / tH, 1.0);
  for (int it = 0; it < 60; ++it) {
    double I1, I2;
    cosmo_integrals(z, Om, &I1, &I2);
    const double f = (1.0 + z) * tH * I1 - D;
    const double fp = tH * (I1 + (1.0 + z) / Ez(z, Om));
    double zn = z - f / fp;
    if (fabs(zn - z) <= 2e-15 * fmax(fabs(zn), 1e-300)) { z = zn; break; }
    if (f > 0.0) hi = z; else lo = z;
    if (!(zn >= lo && zn <= hi)) zn = 0.5 * (lo + hi);
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
  int anchor_end;         // 0: the parameter row is the state at t = 0; 1: at plunge, at the last coarse node (reading D12)
  double* wc;             // [K][WC_STRIDE]
  double* nodes;          // [K][Nn][NODE_STRIDE]
  int32_t* jpl;           // [K] first plunged node (index j), Nn if none
  int32_t* status;        // [K]
  double2* nodeaux;       // [K][Nn] {(2 pi M nu_j)^{2/3} mu/(Xi D), 1/nu_j} for the amplitude of stage (b)
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

// Recursion node r (0 = where the parameters are given) -> node row.  Forward: node j = r, row r + 1.  Anchored at the
// LSO: node j = Nc - r, row Nc + 1 - r, and the step is -Delta.  A row holds the value and slope at its node and the
// increment over the interval [j, j+1] in FORWARD time: forward, that is the step leaving the node (one row write);
// backward, it is minus the step that ARRIVED at the node, so value + slope and the increment are written separately.
DEVINL int64_t row_of(const OrbitArgs& a, int64_t r) { return a.anchor_end ? a.Nc + 1 - r : r + 1; }
DEVINL void store_value_slope(double* row, const double y[5], const double k1[5]) {
  double2* q = reinterpret_cast<double2*>(row);
  q[0] = make_double2(y[0], y[1]);
  q[1] = make_double2(y[2], y[3]);
  q[2] = make_double2(y[4], k1[0]);
  q[3] = make_double2(k1[1], k1[2]);
  q[4] = make_double2(k1[3], k1[4]);
}
DEVINL void store_increment(double* row, const double d[5], double sign) {
  double2* q = reinterpret_cast<double2*>(row);
  q[5] = make_double2(sign * d[0], sign * d[1]);
  q[6] = make_double2(sign * d[2], sign * d[3]);
  q[7] = make_double2(sign * d[4], 0.0);
}
// node rows of recursion step r -> r + 1 with increment d taken from state y (slope k1)
DEVINL void store_step(const OrbitArgs& a, double* nodes, int64_t r, const double y[5], const double k1[5], const double d[5]) {
  if (!a.anchor_end) {
    store_node(nodes + row_of(a, r) * NODE_STRIDE, y, k1, d);
  } else {
    store_value_slope(nodes + row_of(a, r) * NODE_STRIDE, y, k1);
    store_increment(nodes + row_of(a, r + 1) * NODE_STRIDE, d, -1.0);
  }
}
// the last recursion node: value and slope; forward it has no interval after it
DEVINL void store_last(const OrbitArgs& a, double* nodes, int64_t r, const double y[5], const double k1[5]) {
  const double zero5[5] = {0, 0, 0, 0, 0};
  if (!a.anchor_end) store_node(nodes + row_of(a, r) * NODE_STRIDE, y, k1, zero5);
  else store_value_slope(nodes + row_of(a, r) * NODE_STRIDE, y, k1);
}
// nu_LSO(e) = ((1-e^2)/(6+2e))^{3/2} / (2 pi M)
DEVINL double nu_lso(double twoPiMs, double e) {
  const double t = (1.0 - e * e) / (6.0 + 2.0 * e);
  return t * sqrt(t) / twoPiMs;
}

// (a0) validity, per-walker scalars and the constant block of walker k.
// Returns true when the parameters are in the domain; *status gets BADPARAM / DELAY bits.
DEVINL bool walker_prologue(const OrbitArgs& a, const double* __restrict__ p, double* __restrict__ wc, OrbitConst& oc,
                            int& status) {
  const double Delta = a.S * a.dt;
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
    // lambda = 0 exactly: L^ = S^, beta's atan2 arguments vanish identically (reading R16: beta = 0).  Its numerator
    // cl L^.n^ - S^.n^ would be left at rounding noise by the two different summation orders, so it is made exactly 0
    if (sl == 0.0) { wc[WC_CL] = 0.0; wc[WC_SN] = 0.0; }
    wc[WC_B1] = sS * (sphK * cphS - cphK * sphS) * sl;               // sin(thS) sin(phK - phS) sin(lam)
    wc[WC_B2] = (sS * cK * (cphS * cphK + sphS * sphK) - cS * sK) * sl;   // (Sn cK - cS)/sK sl without the division by sin(thK)
    wc[WC_A0X] = A0x; wc[WC_A0Y] = A0y; wc[WC_A0Z] = A0z;
    wc[WC_A1X] = A1x; wc[WC_A1Y] = A1y; wc[WC_A1Z] = A1z;
    wc[WC_A2X] = A2x; wc[WC_A2Y] = A2y;
    wc[WC_Z] = z; wc[WC_XI] = Xi;
  }
  if (ok && !(fabs(dT) <= Delta)) status |= EMRI_ST_DELAY;          // reading R20

  return ok;
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

  OrbitConst oc;
  const bool ok = walker_prologue(a, p, wc, oc, status);

  // ---- (a1) RK4 on the coarse grid, in the direction of the recursion (forward from t = 0, or backward from the LSO)
  double y[5] = {frac(p[P_PHI0] / kTwoPi), p[P_NU0], frac(p[P_GAM0] / kTwoPi), p[P_E0], frac(p[P_ALP0] / kTwoPi)};
  if (a.anchor_end) y[1] = nu_lso(oc.twoPiMs, y[3]);
  const double h = (a.anchor_end ? -1.0 : 1.0) * Delta;
  double emax = ok ? y[3] : 0.0;
  const double zero5[5] = {0, 0, 0, 0, 0};
  bool run = ok;
  if (run && !a.anchor_end && plunged(oc, y[1], y[3])) { status |= EMRI_ST_PLUNGE; jpl = 0; run = false; }
  if (run) {
    RkOut r;
    // guard step against the direction of the recursion
    rk4_increment(oc, y, -h, r);
    double ym[5] = {frac(y[0] + r.d[0]), y[1] + r.d[1], frac(y[2] + r.d[2]), y[3] + r.d[3], frac(y[4] + r.d[4])};
    bool okm = isfinite(ym[0]) && isfinite(ym[1]) && isfinite(ym[2]) && isfinite(ym[3]) && isfinite(ym[4]) &&
               ym[3] >= 0.0 && ym[3] < 1.0 && ym[1] > 0.0;
    if (!okm) {
      status |= EMRI_ST_STATE;
      run = false;
    } else {
      double km[5], dm[5];
      km[0] = ym[1];
      rhs(oc, ym[1], ym[3], &km[1], &km[2], &km[3], &km[4]);
      if (!a.anchor_end) {
#pragma unroll
        for (int q = 0; q < 5; ++q) dm[q] = -r.d[q];
        store_node(nodes, ym, km, dm);
      } else {
        store_node(nodes + (a.Nc + 2) * NODE_STRIDE, ym, km, zero5);
        store_increment(nodes + (a.Nc + 1) * NODE_STRIDE, r.d, 1.0);
      }
      emax = fmax(emax, ym[3]);
      // sweep; nu and e are Kahan-compensated (reading D3)
      double comp_nu = 0.0, comp_e = 0.0;
      const int64_t last = a.Nc + 1;          // recursion index of the last node (G = 1)
      for (int64_t j = 0; j <= last; ++j) {
        if (j == last) {
          double k1[5];
          k1[0] = y[1];
          rhs(oc, y[1], y[3], &k1[1], &k1[2], &k1[3], &k1[4]);
          store_last(a, nodes, j, y, k1);
          break;
        }
        rk4_increment(oc, y, h, r);
        store_step(a, nodes, j, y, r.k1, r.d);
        double yn[5];
        yn[0] = frac(y[0] + r.d[0]);
        yn[2] = frac(y[2] + r.d[2]);
        yn[4] = frac(y[4] + r.d[4]);
        { double t = r.d[1] - comp_nu, s = y[1] + t; comp_nu = (s - y[1]) - t; yn[1] = s; }
        { double t = r.d[3] - comp_e, s = y[3] + t; comp_e = (s - y[3]) - t; yn[3] = s; }
        bool okn = isfinite(yn[0]) && isfinite(yn[1]) && isfinite(yn[2]) && isfinite(yn[3]) && isfinite(yn[4]) &&
                   yn[3] >= 0.0 && yn[3] < 1.0 && yn[1] > 0.0;
        bool pl = okn && !a.anchor_end && plunged(oc, yn[1], yn[3]);
        if (!okn || pl) {
          status |= okn ? EMRI_ST_PLUNGE : EMRI_ST_STATE;
          if (a.anchor_end) { run = false; break; }      // anchored at the LSO a bad state invalidates the walker
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
  if (!run) {
    for (int64_t m = 0; m < a.Nn; ++m) store_node(nodes + m * NODE_STRIDE, zero5, zero5, zero5);
  }
  wc[WC_EMAX] = emax;
  a.jpl[k] = jpl;
  a.status[k] = status;
}

// ==================================================================== (a1) parallel-in-time evaluation
// The RK4 recursion of S3 is sequential in the node index, so with one thread per walker stage (a)
// is a latency-bound chain (N_c x 4 right-hand sides back to back) that costs as much as the whole
// synthesis at K = 64.  The (nu, e) pair is a closed autonomous 2-d subsystem and Phi, gamma~, alpha
// are quadratures along it, so the SAME discrete trajectory is obtained by multiple shooting:
//   1. orbit_init_kernel     per walker: scalars, guard node, and a COARSE sweep (one RK4 step of
//                            L*Delta per segment) giving a guess U_p of (nu, e) at every L-th node;
//   2. orbit_sweep_kernel    one thread per (walker, segment): the L fine RK4 steps of the scheme
//                            from U_p, storing the node rows; in round 0 two more threads per segment
//                            start from U_p + eps e_i (finite-difference Jacobian J_p of the segment map);
//   3. orbit_correct_kernel  per walker: defects D_{p+1} = F(U_p) - U_{p+1} in compensated arithmetic,
//                            Newton (chord) correction d_{p+1} = D_{p+1} + J_p d_p, U_p += d_p;
//   4. sweep again; the defects are then ~1e-19 nu (quadratic convergence), far below the rounding
//      of the sequential recursion itself; boundaries whose defect exceeds 4e-17 nu are re-corrected
//      once more and whatever is still unverified is integrated sequentially by orbit_tail_kernel
//      from the last verified boundary (so the result never depends on convergence);
//   5. orbit_fixup_kernel    adds the per-segment angle offsets (prefix sum of the wrapped segment
//                            totals), writes the post-plunge copies.
// nu and e are carried as Kahan pairs (value, compensation) exactly as in the sequential kernel, so
// a segment boundary is matched in ~double-double precision.  (DESIGN.md section 6a.)
constexpr int SEG_STRIDE = 32;
enum {
  SG_NU = 0, SG_CNU, SG_E, SG_CE,                 // start of the segment (Kahan pairs)
  SG_ENU, SG_ECNU, SG_EE, SG_ECE,                 // end of the base sweep
  SG_P1NU, SG_P1CNU, SG_P1E, SG_P1CE,             // end of the sweep started at nu + eps1
  SG_P2NU, SG_P2CNU, SG_P2E, SG_P2CE,             // end of the sweep started at e + eps2
  SG_EPS1, SG_EPS2,
  SG_J00, SG_J01, SG_J10, SG_J11,                 // d(end nu, end e)/d(start nu, start e)
  SG_T0, SG_T1, SG_T2,                            // wrapped angle totals of the segment (local end angles)
  SG_O0, SG_O1, SG_O2,                            // angle offsets of the segment (cycles)
  SG_STOP, SG_KIND, SG_EMAX,                      // first bad node j (0 = none), its status bit, max e
  SG_COUNT
};
static_assert(SG_COUNT <= SEG_STRIDE, "segment record too small");
enum { OM_ACTIVE = 0, OM_CONVERGED = 1, OM_TAIL = 2, OM_ZERO = 3, OM_DONE = 4 };

// The part of the prologue the recursion itself needs (validity of the orbital parameters and the constants of the
// right-hand side); the rest -- z(D_L), Xi, Delta T, the geometry block -- is walker_prologue's and can run beside it.
DEVINL bool orbit_const_only(const double* __restrict__ p, OrbitConst& oc) {
  bool ok = true;
#pragma unroll
  for (int i = 0; i < EMRI_NPAR; ++i) ok = ok && isfinite(p[i]);
  ok = ok && p[P_M] > 0.0 && p[P_MU] > 0.0 && p[P_DL] > 0.0 && p[P_E0] >= 0.0 && p[P_E0] < 1.0 &&
       fabs(p[P_A]) <= 1.0 && p[P_NU0] > 0.0;
  const double Ms = p[P_M] * kMsunSec, mus = p[P_MU] * kMsunSec;
  oc.twoPiMs = kTwoPi * Ms;
  oc.Cnu = 96.0 / (10.0 * kPi) * (mus / (Ms * Ms * Ms));
  oc.Ce = mus / (Ms * Ms);
  oc.a = p[P_A];
  double sl, cl;
  sincos(p[P_LAM], &sl, &cl);
  oc.sp = p[P_A] * cl;
  return ok;
}

struct ShootArgs {
  OrbitArgs o;
  int L, P;               // fine steps per segment, number of segments
  int64_t n_steps;        // forward steps = index of the last node = Nc + 1
  double* seg;            // [K][P][SEG_STRIDE]
  int32_t* mode;          // [K] OM_*
  int32_t* pclamp;        // [K] last segment index whose offset applies (tail start)
  double* plrow;          // [K][NODE_STRIDE] row copied to the nodes from j_pl on
  int round, last_round;
};

// rates of (nu, e) only: the part of rhs() on the sequential critical path
DEVINL void rhs_nue(const OrbitConst& w, double nu, double e, double* fnu, double* fe) {
  const double x = w.twoPiMs * nu;
  const double cb = cbrt_polished(x);
  const double u = cb * cb;
  const double e2 = e * e;
  const double q = 1.0 - e2;
  const double rq = 1.0 / q;
  const double sq = sqrt(q);
  const double rsq = sq * rq;
  const double x2 = x * x;
  const double x83 = x2 * u, x113 = x83 * x;
  const double rq2 = rq * rq;
  {
    double t0 = fma(e2, fma(e2, 37.0 / 96.0, 73.0 / 24.0), 1.0) * q;
    double t1 = u * fma(e2, fma(e2, fma(e2, -13147.0 / 5376.0, -3885.0 / 128.0), -2561.0 / 224.0), 1273.0 / 336.0);
    double t2 = x * w.sp * rsq * fma(e2, fma(e2, fma(e2, 65.0 / 64.0, 3143.0 / 96.0), 1211.0 / 24.0), 73.0 / 12.0);
    *fnu = w.Cnu * x113 * (rq2 * rq2 * rsq) * (t0 + t1 - t2);
  }
  {
    double t0 = fma(e2, 121.0, 304.0) * q * fma(u, 12.0, 1.0);
    double t1 = u * fma(e2, fma(e2, -25211.0, 12.0 * 9082.0), 8.0 * 16705.0) * (1.0 / 56.0);
    double t2 = w.sp * x113 * (rq2 * rq2) * fma(e2, fma(e2, 263.0 / 10.0, 5032.0 / 15.0), 1364.0 / 5.0);
    *fe = e * w.Ce * (t2 - (1.0 / 15.0) * x83 * (rq2 * rq * rsq) * (t0 - t1));
  }
}

DEVINL void rk4_nue(const OrbitConst& w, double nu, double e, double h, double* dnu, double* de) {
  double k1n, k1e, k2n, k2e, k3n, k3e, k4n, k4e;
  rhs_nue(w, nu, e, &k1n, &k1e);
  const double hh = 0.5 * h;
  rhs_nue(w, fma(hh, k1n, nu), fma(hh, k1e, e), &k2n, &k2e);
  rhs_nue(w, fma(hh, k2n, nu), fma(hh, k2e, e), &k3n, &k3e);
  rhs_nue(w, fma(h, k3n, nu), fma(h, k3e, e), &k4n, &k4e);
  *dnu = (h / 6.0) * (k1n + 2.0 * k2n + 2.0 * k3n + k4n);
  *de = (h / 6.0) * (k1e + 2.0 * k2e + 2.0 * k3e + k4e);
}

DEVINL void kahan_add(double& y, double& comp, double d) {
  const double t = d - comp, s = y + t;
  comp = (s - y) - t;
  y = s;
}

DEVINL bool state_ok(double p0, double nu, double p2, double e, double p4) {
  return isfinite(p0) && isfinite(nu) && isfinite(p2) && isfinite(e) && isfinite(p4) && e >= 0.0 && e < 1.0 && nu > 0.0;
}

DEVINL void load_orbit_const(const double* __restrict__ wc, OrbitConst& oc) {
  oc.twoPiMs = wc[WC_TWOPIMS]; oc.Cnu = wc[WC_CNU]; oc.Ce = wc[WC_CE]; oc.a = wc[WC_A]; oc.sp = wc[WC_SP];
}

// ---- 1. per walker: prologue, guard node, coarse sweep
__global__ void __launch_bounds__(64) orbit_init_kernel(ShootArgs s) {
  // Two warps per 32 walkers.  Warp 1 runs the full prologue (z(D_L), Xi, Delta T, the geometry block: walker_prologue);
  // warp 0 needs only the constants of the right-hand side for the guard step and the coarse sweep, so the two chains of
  // dependent arithmetic run side by side instead of one after the other (59 -> 33 us at K = 8).
  __shared__ int s_status[32];
  __shared__ int s_ok[32];
  const OrbitArgs& a = s.o;
  const int lane = threadIdx.x & 31;
  const int k = blockIdx.x * 32 + lane;
  const bool live = k < a.K;
  const double* p = a.params + (size_t)(live ? k : 0) * EMRI_NPAR;
  double* wc = a.wc + (size_t)(live ? k : 0) * WC_STRIDE;
  if (threadIdx.x >= 32) {
    if (live) {
      int st = 0;
      OrbitConst oc1;
      const bool ok1 = walker_prologue(a, p, wc, oc1, st);
      s_status[lane] = st;
      s_ok[lane] = ok1 ? 1 : 0;
    }
    __syncthreads();
    return;
  }
  double* nodes = a.nodes + (size_t)(live ? k : 0) * a.Nn * NODE_STRIDE;
  double* seg = s.seg + (size_t)(live ? k : 0) * s.P * SEG_STRIDE;
  const double Delta = a.S * a.dt;
  int status = 0;
  OrbitConst oc;
  const bool ok = live && orbit_const_only(p, oc);
  double y[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (ok) {
    y[0] = frac(p[P_PHI0] / kTwoPi); y[1] = p[P_NU0]; y[2] = frac(p[P_GAM0] / kTwoPi); y[3] = p[P_E0];
    y[4] = frac(p[P_ALP0] / kTwoPi);
    if (a.anchor_end) y[1] = nu_lso(oc.twoPiMs, y[3]);
  }
  const double dir = a.anchor_end ? -1.0 : 1.0;
  int mode = OM_ACTIVE;
  int32_t jpl = (int32_t)a.Nn;
  double emax = ok ? y[3] : 0.0;
  if (!ok) mode = OM_ZERO;
  else if (!a.anchor_end && plunged(oc, y[1], y[3])) { status |= EMRI_ST_PLUNGE; jpl = 0; mode = OM_ZERO; }
  if (mode == OM_ACTIVE) {
    // guard step against the direction of the recursion: node -1 (row 0) forward, node Nc+1 (row Nc+2) at the LSO
    RkOut r;
    rk4_increment(oc, y, -dir * Delta, r);
    double ym[5] = {frac(y[0] + r.d[0]), y[1] + r.d[1], frac(y[2] + r.d[2]), y[3] + r.d[3], frac(y[4] + r.d[4])};
    if (!state_ok(ym[0], ym[1], ym[2], ym[3], ym[4])) {
      status |= EMRI_ST_STATE;
      mode = OM_ZERO;
    } else {
      double km[5], dm[5];
      km[0] = ym[1];
      rhs(oc, ym[1], ym[3], &km[1], &km[2], &km[3], &km[4]);
      if (!a.anchor_end) {
#pragma unroll
        for (int q = 0; q < 5; ++q) dm[q] = -r.d[q];
        store_node(nodes, ym, km, dm);
      } else {
        const double zero5[5] = {0, 0, 0, 0, 0};
        store_node(nodes + (a.Nc + 2) * NODE_STRIDE, ym, km, zero5);
        store_increment(nodes + (a.Nc + 1) * NODE_STRIDE, r.d, 1.0);      // interval [Nc, Nc+1]
      }
      emax = fmax(emax, ym[3]);
    }
  }
  if (mode == OM_ACTIVE) {
    // coarse sweep: one RK4 step of L*Delta per segment
    const double H = dir * (double)s.L * Delta;
    double nu = y[1], e = y[3];
    for (int pp = 0; pp < s.P; ++pp) {
      double* sg = seg + (size_t)pp * SEG_STRIDE;
      sg[SG_NU] = nu; sg[SG_CNU] = 0.0; sg[SG_E] = e; sg[SG_CE] = 0.0;
      if (pp + 1 < s.P) {
        double dn, de;
        rk4_nue(oc, nu, e, H, &dn, &de);
        nu += dn; e += de;
      }
    }
  }
  __syncthreads();                            // warp 1's verdict on the remaining parameters (Xi(z) > 0) and its status bits
  if (!live) return;
  if (!s_ok[lane]) { mode = OM_ZERO; status = s_status[lane]; jpl = (int32_t)a.Nn; emax = 0.0; }
  else status |= s_status[lane];
  wc[WC_EMAX] = emax;
  a.jpl[k] = jpl;
  a.status[k] = status;
  s.mode[k] = mode;
  s.pclamp[k] = s.P - 1;
}

// ---- 2. one thread per (variant, walker, segment): the fine steps of the segment
__global__ void __launch_bounds__(64) orbit_sweep_kernel(ShootArgs s) {
  const OrbitArgs& a = s.o;
  // blockIdx.y = variant (0: the scheme itself; 1, 2 in round 0: the perturbed copies for the Jacobian), so that no warp
  // mixes the two code paths (a warp straddling variants ran them one after the other: 56 instead of 34 us at K = 8)
  const int64_t r0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t per_v = (int64_t)a.K * s.P;
  if (r0 >= per_v) return;
  const int v = (int)blockIdx.y;
  const int k = (int)(r0 / s.P), pp = (int)(r0 - (int64_t)k * s.P);
  if (s.mode[k] != OM_ACTIVE) return;
  double* sg = s.seg + ((size_t)k * s.P + pp) * SEG_STRIDE;
  OrbitConst oc;
  load_orbit_const(a.wc + (size_t)k * WC_STRIDE, oc);
  const double Delta = (a.anchor_end ? -1.0 : 1.0) * (a.S * a.dt);      // signed step of the recursion
  const int64_t j0 = (int64_t)pp * s.L;
  const int nst = (int)((s.n_steps - j0 < (int64_t)s.L) ? (s.n_steps - j0) : (int64_t)s.L);
  double nu = sg[SG_NU], cnu = sg[SG_CNU], e = sg[SG_E], ce = sg[SG_CE];
  if (v != 0) {
    // perturbed start for the finite-difference Jacobian (nu, e part of the scheme only)
    if (v == 1) { const double t = nu + 1e-8 * nu; sg[SG_EPS1] = t - nu; nu = t; }
    else { const double t = e + 1e-8 * fmax(e, 1e-3); sg[SG_EPS2] = t - e; e = t; }
    for (int i = 0; i < nst; ++i) {
      double dn, de;
      rk4_nue(oc, nu, e, Delta, &dn, &de);
      kahan_add(nu, cnu, dn);
      kahan_add(e, ce, de);
    }
    double* out = sg + (v == 1 ? SG_P1NU : SG_P2NU);
    out[0] = nu; out[1] = cnu; out[2] = e; out[3] = ce;
    return;
  }
  // base sweep: full right-hand side, node rows stored with LOCAL angles (segment 0: the initial angles)
  double* nodes = a.nodes + (size_t)k * a.Nn * NODE_STRIDE;
  double ang0 = 0.0, ang1 = 0.0, ang2 = 0.0;
  if (pp == 0) {
    const double* p = a.params + (size_t)k * EMRI_NPAR;
    ang0 = frac(p[P_PHI0] / kTwoPi); ang1 = frac(p[P_GAM0] / kTwoPi); ang2 = frac(p[P_ALP0] / kTwoPi);
  }
  double emax = e;
  int64_t stop = 0;
  int kind = 0;
  RkOut r;
  for (int i = 0; i < nst; ++i) {
    const int64_t j = j0 + i;
    const double y[5] = {ang0, nu, ang1, e, ang2};
    rk4_increment(oc, y, Delta, r);
    store_step(a, nodes, j, y, r.k1, r.d);
    const double n0 = frac(ang0 + r.d[0]), n2 = frac(ang1 + r.d[2]), n4 = frac(ang2 + r.d[4]);
    double nn = nu, nc = cnu, en = e, ec = ce;
    kahan_add(nn, nc, r.d[1]);
    kahan_add(en, ec, r.d[3]);
    const bool okn = state_ok(n0, nn, n2, en, n4);
    if (!okn || (!a.anchor_end && plunged(oc, nn, en))) { stop = j + 1; kind = okn ? EMRI_ST_PLUNGE : EMRI_ST_STATE; break; }
    ang0 = n0; ang1 = n2; ang2 = n4; nu = nn; cnu = nc; e = en; ce = ec;
    emax = fmax(emax, e);
  }
  if (stop == 0 && j0 + nst == s.n_steps) {
    // last node of the grid: value and slope, no increment
    const double y[5] = {ang0, nu, ang1, e, ang2};
    double k1[5];
    k1[0] = nu;
    rhs(oc, nu, e, &k1[1], &k1[2], &k1[3], &k1[4]);
    store_last(a, nodes, s.n_steps, y, k1);
  }
  sg[SG_ENU] = nu; sg[SG_ECNU] = cnu; sg[SG_EE] = e; sg[SG_ECE] = ce;
  sg[SG_T0] = ang0; sg[SG_T1] = ang1; sg[SG_T2] = ang2;
  sg[SG_STOP] = (double)stop; sg[SG_KIND] = (double)kind; sg[SG_EMAX] = emax;
}

// ---- 3. per walker (one warp): defects, verification, Newton correction or finalisation
__global__ void __launch_bounds__(32) orbit_correct_kernel(ShootArgs s) {
  extern __shared__ double sm_c[];          // [P][CS]: D_nu, D_e, J00, J01, J10, J11, stop, finite, tol_nu, tol_e, d_nu, d_e
  constexpr int CS = 12;
  const OrbitArgs& a = s.o;
  const int k = blockIdx.x, lane = threadIdx.x;
  if (s.mode[k] != OM_ACTIVE) return;
  double* seg = s.seg + (size_t)k * s.P * SEG_STRIDE;
  const int P = s.P;
  // boundary b = p+1 between segment p and p+1: defect of segment p's end against segment p+1's start
  for (int p = lane; p < P; p += 32) {
    double* sg = seg + (size_t)p * SEG_STRIDE;
    double* o = sm_c + (size_t)p * CS;
    if (s.round == 0) {
      const double dn1 = (sg[SG_P1NU] - sg[SG_ENU]) - (sg[SG_P1CNU] - sg[SG_ECNU]);
      const double de1 = (sg[SG_P1E] - sg[SG_EE]) - (sg[SG_P1CE] - sg[SG_ECE]);
      const double dn2 = (sg[SG_P2NU] - sg[SG_ENU]) - (sg[SG_P2CNU] - sg[SG_ECNU]);
      const double de2 = (sg[SG_P2E] - sg[SG_EE]) - (sg[SG_P2CE] - sg[SG_ECE]);
      sg[SG_J00] = dn1 / sg[SG_EPS1]; sg[SG_J10] = de1 / sg[SG_EPS1];
      sg[SG_J01] = dn2 / sg[SG_EPS2]; sg[SG_J11] = de2 / sg[SG_EPS2];
    }
    o[2] = sg[SG_J00]; o[3] = sg[SG_J01]; o[4] = sg[SG_J10]; o[5] = sg[SG_J11];
    o[6] = sg[SG_STOP];
    double Dn = 0.0, De = 0.0;
    if (p + 1 < P) {
      const double* nx = sg + SEG_STRIDE;
      Dn = (sg[SG_ENU] - nx[SG_NU]) - (sg[SG_ECNU] - nx[SG_CNU]);
      De = (sg[SG_EE] - nx[SG_E]) - (sg[SG_ECE] - nx[SG_CE]);
    }
    o[0] = Dn; o[1] = De;
    o[8] = 4e-17 * fabs(sg[SG_ENU]); o[9] = 4e-17 * fabs(sg[SG_EE]);      // verification tolerance of boundary p+1
    o[10] = 0.0; o[11] = 0.0;              // correction of THIS segment's start (set by the scan below)
    o[7] = (isfinite(Dn) && isfinite(De) && isfinite(o[2]) && isfinite(o[3]) && isfinite(o[4]) && isfinite(o[5])) ? 1.0 : 0.0;
  }
  __syncwarp();
  __shared__ int sh_first_bad, sh_stop_seg, sh_converged;
  if (lane == 0) {
    // scan the boundaries in order; a segment's result is trusted only if every boundary before it is verified
    int first_bad = -1, stop_seg = -1;
    double dn = 0.0, de = 0.0;
    for (int p = 0; p < P; ++p) {
      double* o = sm_c + (size_t)p * CS;
      if (o[6] != 0.0) { if (first_bad < 0) stop_seg = p; break; }
      if (p + 1 == P) break;
      const bool small = (o[7] != 0.0) && fabs(o[0]) <= o[8] && fabs(o[1]) <= o[9];
      if (!small && first_bad < 0) first_bad = p + 1;
      if (o[7] != 0.0) {
        const double nn = o[0] + fma(o[2], dn, o[3] * de), ne = o[1] + fma(o[4], dn, o[5] * de);
        dn = nn; de = ne;
      } else { dn = 0.0; de = 0.0; }
      o[CS + 10] = dn; o[CS + 11] = de;      // correction of segment p+1's start (the scan touches shared memory only)
    }
    sh_first_bad = first_bad; sh_stop_seg = stop_seg;
    sh_converged = (first_bad < 0) ? 1 : 0;
  }
  __syncwarp();
  const int first_bad = sh_first_bad, stop_seg = sh_stop_seg;
  if (!sh_converged && !s.last_round) {
    // Newton (chord) update of the segment starts, in compensated form
    for (int p = 1 + lane; p < P; p += 32) {
      double* sg = seg + (size_t)p * SEG_STRIDE;
      const double dn = sm_c[(size_t)p * CS + 10], de = sm_c[(size_t)p * CS + 11];
      if (isfinite(dn) && isfinite(de)) {
        const double yn = sg[SG_NU] + dn; sg[SG_CNU] += (yn - sg[SG_NU]) - dn; sg[SG_NU] = yn;
        const double ye = sg[SG_E] + de; sg[SG_CE] += (ye - sg[SG_E]) - de; sg[SG_E] = ye;
      }
    }
    return;
  }
  // finalise: everything before `lim` is verified; a verified stop ends the orbit, an unverified
  // boundary (last round only) hands the rest to orbit_tail_kernel
  if (lane == 0) {
    const int lim = (first_bad >= 0) ? first_bad : ((stop_seg >= 0) ? stop_seg + 1 : P);   // segments [0, lim) are final
    double o0 = 0.0, o1 = 0.0, o2 = 0.0, emax = a.wc[(size_t)k * WC_STRIDE + WC_EMAX];
    for (int p = 0; p < lim; ++p) {
      double* sg = seg + (size_t)p * SEG_STRIDE;
      const double t0 = sg[SG_T0], t1 = sg[SG_T1], t2 = sg[SG_T2];
      sg[SG_O0] = o0; sg[SG_O1] = o1; sg[SG_O2] = o2;
      emax = fmax(emax, sg[SG_EMAX]);
      if (p == 0) { o0 = t0; o1 = t1; o2 = t2; }
      else { o0 = frac(o0 + t0); o1 = frac(o1 + t1); o2 = frac(o2 + t2); }
    }
    a.wc[(size_t)k * WC_STRIDE + WC_EMAX] = emax;
    if (first_bad >= 0) {
      // tail: continue sequentially from the (verified) end of segment first_bad-1
      double* sg = seg + (size_t)first_bad * SEG_STRIDE;
      const double* pv = sg - SEG_STRIDE;
      sg[SG_NU] = pv[SG_ENU]; sg[SG_CNU] = pv[SG_ECNU]; sg[SG_E] = pv[SG_EE]; sg[SG_CE] = pv[SG_ECE];
      sg[SG_O0] = o0; sg[SG_O1] = o1; sg[SG_O2] = o2;
      s.pclamp[k] = first_bad;
      s.mode[k] = OM_TAIL;
    } else {
      s.pclamp[k] = P - 1;
      if (stop_seg >= 0 && a.anchor_end) {
        // anchored at the LSO nothing plunges; a bad state (e leaving [0,1)) invalidates the walker
        a.status[k] |= EMRI_ST_STATE;
        s.mode[k] = OM_ZERO;
        return;
      }
      if (stop_seg >= 0) {
        const double* sg = seg + (size_t)stop_seg * SEG_STRIDE;
        const int64_t jst = (int64_t)sg[SG_STOP];
        a.jpl[k] = (int32_t)jst;
        a.status[k] |= (int)sg[SG_KIND];
        // row copied to the nodes from j_pl on: node j_pl - 1 (global angles), zero increments
        const double* src = a.nodes + ((size_t)k * a.Nn + jst) * NODE_STRIDE;    // row of node jst-1
        double* dst = s.plrow + (size_t)k * NODE_STRIDE;
        for (int q = 0; q < NODE_STRIDE; ++q) dst[q] = (q < 10) ? src[q] : 0.0;
        dst[0] = (stop_seg == 0) ? src[0] : frac(src[0] + sg[SG_O0]);
        dst[2] = (stop_seg == 0) ? src[2] : frac(src[2] + sg[SG_O1]);
        dst[4] = (stop_seg == 0) ? src[4] : frac(src[4] + sg[SG_O2]);
      }
      s.mode[k] = OM_CONVERGED;
    }
  }
}

// ---- 4. sequential continuation from the last verified boundary (only walkers in OM_TAIL)
__global__ void __launch_bounds__(32) orbit_tail_kernel(ShootArgs s) {
  const OrbitArgs& a = s.o;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= a.K || s.mode[k] != OM_TAIL) return;
  const int pb = s.pclamp[k];
  double* sg = s.seg + ((size_t)k * s.P + pb) * SEG_STRIDE;
  double* nodes = a.nodes + (size_t)k * a.Nn * NODE_STRIDE;
  OrbitConst oc;
  load_orbit_const(a.wc + (size_t)k * WC_STRIDE, oc);
  const double Delta = (a.anchor_end ? -1.0 : 1.0) * (a.S * a.dt);      // signed step of the recursion
  double nu = sg[SG_NU], cnu = sg[SG_CNU], e = sg[SG_E], ce = sg[SG_CE];
  double ang0 = 0.0, ang1 = 0.0, ang2 = 0.0;       // local to the tail; orbit_fixup_kernel adds the offset
  double emax = fmax(a.wc[(size_t)k * WC_STRIDE + WC_EMAX], e);
  RkOut r;
  for (int64_t j = (int64_t)pb * s.L; j <= s.n_steps; ++j) {
    const double y[5] = {ang0, nu, ang1, e, ang2};
    if (j == s.n_steps) {
      double k1[5];
      k1[0] = nu;
      rhs(oc, nu, e, &k1[1], &k1[2], &k1[3], &k1[4]);
      store_last(a, nodes, j, y, k1);
      break;
    }
    rk4_increment(oc, y, Delta, r);
    store_step(a, nodes, j, y, r.k1, r.d);
    const double n0 = frac(ang0 + r.d[0]), n2 = frac(ang1 + r.d[2]), n4 = frac(ang2 + r.d[4]);
    double nn = nu, nc = cnu, en = e, ec = ce;
    kahan_add(nn, nc, r.d[1]);
    kahan_add(en, ec, r.d[3]);
    const bool okn = state_ok(n0, nn, n2, en, n4);
    if (!okn || (!a.anchor_end && plunged(oc, nn, en))) {
      a.status[k] |= okn ? EMRI_ST_PLUNGE : EMRI_ST_STATE;
      if (a.anchor_end) { s.mode[k] = OM_ZERO; break; }       // anchored at the LSO a bad state invalidates the walker
      a.jpl[k] = (int32_t)(j + 1);
      double* dst = s.plrow + (size_t)k * NODE_STRIDE;
      dst[0] = frac(ang0 + sg[SG_O0]); dst[1] = nu; dst[2] = frac(ang1 + sg[SG_O1]); dst[3] = e; dst[4] = frac(ang2 + sg[SG_O2]);
      for (int q = 0; q < 5; ++q) { dst[5 + q] = r.k1[q]; dst[10 + q] = 0.0; }
      dst[15] = 0.0;
      break;
    }
    ang0 = n0; ang1 = n2; ang2 = n4; nu = nn; cnu = nc; e = en; ce = ec;
    emax = fmax(emax, e);
  }
  a.wc[(size_t)k * WC_STRIDE + WC_EMAX] = emax;
}

// per-node amplitude data for stage (b): {(2 pi M nu_j)^{2/3} mu/(Xi D), 1/nu_j}
DEVINL double2 node_aux(const double* __restrict__ wc, double nu) {
  if (!(nu > 0.0) || !isfinite(nu)) return make_double2(0.0, 0.0);
  const double cb = cbrt(wc[WC_TWOPIMS] * nu);
  return make_double2(cb * cb * wc[WC_AMP], 1.0 / nu);
}

// ---- 5. node-parallel: global angles, post-plunge copies, zero rows, and the node's amplitude pair
__global__ void __launch_bounds__(128) orbit_fixup_kernel(ShootArgs s) {
  const OrbitArgs& a = s.o;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= a.Nn * a.K) return;
  const int k = (int)(idx / a.Nn);
  const int64_t m = idx - (int64_t)k * a.Nn;
  const int mode = s.mode[k];
  const double* wc = a.wc + (size_t)k * WC_STRIDE;
  double2* row = reinterpret_cast<double2*>(a.nodes + ((size_t)k * a.Nn + m) * NODE_STRIDE);
  if (mode == OM_ZERO) {
#pragma unroll
    for (int q = 0; q < NODE_STRIDE / 2; ++q) row[q] = make_double2(0.0, 0.0);
    a.nodeaux[idx] = make_double2(0.0, 0.0);
    return;
  }
  // recursion index of this row's node: forward r = j = m - 1 (row 0 is the guard node, global angles already);
  // anchored at the LSO r = Nc - j = Nc + 1 - m (row Nc + 2 is the guard node)
  const int64_t r = a.anchor_end ? a.Nc + 1 - m : m - 1;
  const int32_t jpl = a.jpl[k];
  if (r >= 0 && !a.anchor_end && r >= (int64_t)jpl) {
    const double2* src = reinterpret_cast<const double2*>(s.plrow + (size_t)k * NODE_STRIDE);
#pragma unroll
    for (int q = 0; q < NODE_STRIDE / 2; ++q) row[q] = src[q];
    a.nodeaux[idx] = node_aux(wc, src[0].y);
    return;
  }
  double2 v01 = row[0];
  a.nodeaux[idx] = node_aux(wc, v01.y);
  if (r < 0) return;
  int64_t p = r / s.L;
  const int pc = s.pclamp[k];
  if (p > pc) p = pc;
  if (p == 0) return;
  const double* sg = s.seg + ((size_t)k * s.P + p) * SEG_STRIDE;
  double2 v23 = row[1], v4 = row[2];
  v01.x = frac(v01.x + sg[SG_O0]);
  v23.x = frac(v23.x + sg[SG_O1]);
  v4.x = frac(v4.x + sg[SG_O2]);
  row[0] = v01; row[1] = v23; row[2] = v4;
}

// ---- node-parallel (sequential schedule; the parallel one does this in orbit_fixup_kernel): amplitude pair per node
__global__ void __launch_bounds__(128) orbit_aux_kernel(OrbitArgs a) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= a.Nn * a.K) return;
  const int k = (int)(idx / a.Nn);
  a.nodeaux[idx] = node_aux(a.wc + (size_t)k * WC_STRIDE, a.nodes[(size_t)idx * NODE_STRIDE + 1]);
}

}  // namespace
