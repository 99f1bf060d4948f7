// synth.cuh -- stage (b): cubic-Hermite orbit, Peters-Mathews harmonic sum (Eq. 2), LISA response
// (PAPER.md:79, :118), propagation factors (Eqs. 4-6).
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
//
// What is evaluated per (walker, sample) is S4 + S5 of DESIGN.md section 3.  How:
//
//  * Harmonic brackets as power series in w = e^2.  With J_k(ne) = (ne/2)^k s_k(w),
//    s_k(w) = sum_m (-n^2 w/4)^m / (m! (m+k)!), the three brackets of BC Eqs. 7-9 are
//        n [J_{n-2} - 2e J_{n-1} + (2/n) J_n + 2e J_{n+1} - J_{n+2}] = e^{n-2} PA_n(w)
//        n [J_{n-2} - 2 J_n + J_{n+2}]                              = e^{n-2} PB_n(w)
//        J_n                                                        = e^{n-2} PC_n(w)      (n >= 2; n = 1: e^{+1})
//    with entire functions PA_n, PB_n, PC_n whose Taylor coefficients are tabulated on the host in long double
//    (build_base_table in emri.cu).  The factor e^{n-2} rides on the rotation that advances cos/sin(n Phi), so one
//    harmonic costs three Horner evaluations, three accumulations and one scaled rotation.  Well defined at e = 0.
//  * Per unit (one walker, UNIT_TILES tiles of 256 samples) e^2 moves by ~1e-6, so the CTA first RE-EXPANDS the three
//    series about the unit's mid-point w0 (Horner shift, orders 0..MLOC-1, in shared memory) and every sample then
//    evaluates the short local series in x = w - w0.  The number of local orders kept per harmonic is the smallest that
//    leaves a relative truncation < tol (1e-14 by default, reading D8); if order MLOC-1 is still significant the unit falls back to the
//    base series (same loop, global table).  This is a rigorous re-summation, not an interpolation of amplitudes.
//  * Everything of a sample that does not depend on n (Hermite, geometry, antenna patterns, phases, amplitude) is
//    folded into six numbers a_I, b_I, c_I, a_II, b_II, c_II with h_alpha = a S_a + b S_b + c S_c, parked in shared
//    memory during the harmonic loop to keep the loop at few registers.
#pragma once
#include "common.cuh"

namespace {

constexpr int SYNTH_THREADS = 128;        // consumer threads per CTA
constexpr int SYNTH_BLOCK = SYNTH_THREADS + 32;   // + one producer warp
constexpr int TILE = 2 * SYNTH_THREADS;   // samples per tile (2 adjacent samples per thread)
constexpr int UNIT_TILES_MAX = 16;        // tiles per unit (one re-expansion per unit), chosen per launch
constexpr int MLOC = 7;                   // local expansion orders 0..6 are computed ...
constexpr int MKEEP = 6;                  // ... and a unit keeps at most 6 of them (order 6 still significant: base-series fallback)
constexpr int HREC = 22;                  // doubles per harmonic record of the local table: orders 6..0 x {PA, PB, PC} + 1 pad
constexpr int HERM = 26;                  // doubles per staged interval record (cubics of the 5 orbit functions + amplitude data)
#ifndef SYNTH_MINBLOCKS
#define SYNTH_MINBLOCKS 4
#endif
constexpr int BASE_M = 48;                // Taylor coefficients kept per harmonic in the base table

struct SynthArgs {
  const double* wc;
  const double* nodes;
  const double2* nodeaux;  // [K][Nn] {(2 pi M nu_j)^{2/3} mu/(Xi D), 1/nu_j}
  const int32_t* jpl;
  const int32_t* status;
  const double4* base;     // [n_max+1][BASE_M] Taylor coefficients {PA, PB, PC, 0} in w = e^2
  const double* gtab;      // [n_max+1] n (n/2)^{n-2} / (n-2)!  (n >= 2): scale of the brackets in the Bessel path
  int bessel;              // 1: local series from Bessel recurrences (plans with n_max > 48, where the base series in e^2
                           // would cancel); 0: from the tabulated base series
  int k0, K;               // walkers k0 .. k0+K-1
  int64_t N;
  double dt;
  int S, logS;
  int64_t Nn;
  int n_max;
  double* outI;            // separate channels: row of walker k0+i at outI + i*pitch (used when outZ == NULL)
  double* outII;
  int64_t pitch;
  double2* outZ;           // interleaved z = h_I + i h_II, row of walker k0+i at outZ + i*N
  int unit_tiles, unit_tiles_cap;   // tiles per unit of this launch; the plan's maximum (sizes the staging area)
  int64_t tiles_per_walker, units_per_walker;
  double tol;              // relative truncation of the harmonic series
  double cbrt_thr;         // |nu/nu_j - 1| above which the amplitude takes the cube root (4e-3; < 0 forces the branch)
  int force_base;          // diagnostics: every unit takes the base-series fallback
  unsigned long long* counts;   // [SYN_COUNTS] path counters of the call (emri_plan_synth_report)
};

// counters: [0] units, [1..8] units by local order of their first harmonic range, [9] units on the base-series fallback,
// [10] samples whose amplitude took the cube-root branch, [11] units of walkers with a fatal status (zero-filled),
// [12] sum over units of the harmonics evaluated (n2), [13] of those in the first range (n1), [14] sum of the second
// range's order
constexpr int SYN_COUNTS = 16;
enum { SYC_UNITS = 0, SYC_BASE = 9, SYC_CBRT = 10, SYC_SKIP = 11, SYC_NEVAL = 12, SYC_NFIRST = 13, SYC_M2 = 14 };

// FP64 literals of the per-sample code whose low word is not zero.  As immediates ptxas builds each of them with two
// UMOV / IMAD.MOV per use (~100 issue slots per thread and tile, measured); as entries of a __constant__ array with
// literal indices they are constant-bank operands of the DFMA / DMUL itself.
enum { KC_ZSCALE = 0, KC_S7, KC_S5, KC_S3, KC_C6, KC_C4, KC_A4, KC_A3, KC_A2, KC_A1, KC_A0, KC_HSQRT3, KC_SQRT3, KC_COUNT };
__constant__ double kC[KC_COUNT] = {
    kTwoPi / 128.0, -1.0 / 5040.0, 1.0 / 120.0, -1.0 / 6.0, -1.0 / 720.0, 1.0 / 24.0,
    14.0 / 729.0, -7.0 / 243.0, 4.0 / 81.0, -1.0 / 9.0, 2.0 / 3.0, kHalfSqrt3, kSqrt3};

constexpr int SC_TAB = 128;               // entries of the shared cos/sin table (one per 1/128 cycle)
constexpr int SC_REP = 8;                 // replicas of every entry, one per lane & 7

// cos/sin(2 pi x) for x in cycles (|x| < 2^40): nearest table angle (round-to-nearest by the 1.5*2^52 trick, so the
// remainder is exact) and a Taylor rotation by the remainder |z| <= pi/128 (sin to z^7, cos to z^6: < 4e-18).
// The table is replicated 8 times, entry k of replica r at double2 index 8 k + r, and lane l reads replica l & 7: the
// eight lanes of a quarter-warp then always hit eight different 16-byte bank groups, so the 128-bit lookup takes its
// minimum of four wavefronts whatever the angles are (the single 1024-entry table cost ~9).
DEVINL void sincos_cycles(const double2* __restrict__ tab_lane, double x, double& sn, double& cs) {
  const double magic = 6755399441055744.0;
  const double t = fma(x, (double)SC_TAB, magic);
  const int k = __double2loint(t) & (SC_TAB - 1);
  const double r = fma(x, (double)SC_TAB, -(t - magic));
  static_assert(SC_TAB == 128, "kC[KC_ZSCALE] is 2 pi / 128");
  const double z = r * kC[KC_ZSCALE];
  const double z2 = z * z;
  const double sz = fma(z * z2, fma(z2, fma(z2, kC[KC_S7], kC[KC_S5]), kC[KC_S3]), z);
  const double cz = fma(z2, fma(z2, fma(z2, kC[KC_C6], kC[KC_C4]), -0.5), 1.0);
  const double2 e = tab_lane[k * SC_REP];
  cs = fma(e.x, cz, -e.y * sz);
  sn = fma(e.y, cz, e.x * sz);
}

// 1/x to ~1 ulp without the IEEE slow path: hardware seed (2^-23) and two Newton steps
DEVINL double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  r = fma(r, fma(-x, r, 1.0), r);
  r = fma(r, fma(-x, r, 1.0), r);
  return r;
}

struct SampleOut {
  double x, ec, es, C2, S2;     // w - w0;  e cos/sin(Phi_tot);  cos/sin(2 Phi_tot)
};

// Orbit functions of one sample (S4): cubic Hermite of (Phi_c, nu, gam_c, e, alp_c) at the source time, and the data of
// the amplitude series.
struct OrbitAt {
  double Phic, nu, dnu, gamc, e, alpc;
  double Aj, inv_nuj, amp;      // amplitude at the interval's first node (0 when the interval is past plunge), 1/nu_j, mu/(Xi D)
};

// Direct path (S < 256: a tile spans several coarse intervals): integer time split (reading D4), the two node rows from
// global memory (L1-resident, uniform over most of the warp), Hermite basis.
DEVINL void orbit_at_direct(const double* __restrict__ w, const double* __restrict__ nodes, const double2* __restrict__ aux,
                            int64_t i, int S, int logS, double invS, double Delta, int32_t jpl, OrbitAt& o) {
  int64_t j = i >> logS;
  double s = (double)(i & (S - 1)) * invS - w[WC_SIGMA];
  if (s < 0.0) { s += 1.0; j -= 1; } else if (s >= 1.0) { s -= 1.0; j += 1; }
  const bool live = (j + 1 < (int64_t)jpl);
  const double2* r0 = reinterpret_cast<const double2*>(nodes + (j + 1) * NODE_STRIDE);
  const double2* r1 = r0 + NODE_STRIDE / 2;
  const double2 v01 = __ldg(r0), v23 = __ldg(r0 + 1), v4m0 = __ldg(r0 + 2), m12 = __ldg(r0 + 3), m34 = __ldg(r0 + 4),
                d01 = __ldg(r0 + 5), d23 = __ldg(r0 + 6), d4 = __ldg(r0 + 7);
  const double2 n4m0 = __ldg(r1 + 2), n12 = __ldg(r1 + 3), n34 = __ldg(r1 + 4);
  const double2 ax = __ldg(aux + (j + 1));
  const double s2 = s * s, s3 = s2 * s;
  const double hb = fma(-2.0, s3, 3.0 * s2);
  const double h0 = Delta * (s3 - 2.0 * s2 + s), h1 = Delta * (s3 - s2);
  o.Phic = v01.x + fma(hb, d01.x, fma(h0, v4m0.y, h1 * n4m0.y));
  o.dnu = fma(hb, d01.y, fma(h0, m12.x, h1 * n12.x));
  o.nu = v01.y + o.dnu;
  o.gamc = v23.x + fma(hb, d23.x, fma(h0, m12.y, h1 * n12.y));
  o.e = v23.y + fma(hb, d23.y, fma(h0, m34.x, h1 * n34.x));
  o.alpc = v4m0.x + fma(hb, d4.x, fma(h0, m34.y, h1 * n34.y));
  o.Aj = live ? ax.x : 0.0; o.inv_nuj = ax.y; o.amp = live ? w[WC_AMP] : 0.0;
}

// Staged path (S >= 256, the default): the producer warp has turned the (at most two) coarse intervals a tile touches
// into cubics in s, y(s) = c0 + s (c1 + s (c2 + s c3)), in shared memory (stage_intervals).  `loc_s` = (i mod S)/S.
DEVINL void orbit_at_staged(const double* __restrict__ w, const double2* __restrict__ herm, double loc_s, OrbitAt& o) {
  double s = loc_s - w[WC_SIGMA];
  int sel = 0;
  if (s < 0.0) { s += 1.0; sel = HERM / 2; } else if (s >= 1.0) { s -= 1.0; sel = HERM / 2; }
  const double2* h = herm + sel;
  const double2 p01 = h[0], p23 = h[1], n01 = h[2], n23 = h[3], g01 = h[4], g23 = h[5], e01 = h[6], e23 = h[7],
                a01 = h[8], a23 = h[9], ax = h[10];
  o.Phic = fma(s, fma(s, fma(s, p23.y, p23.x), p01.y), p01.x);
  o.dnu = s * fma(s, fma(s, n23.y, n23.x), n01.y);
  o.nu = n01.x + o.dnu;
  o.gamc = fma(s, fma(s, fma(s, g23.y, g23.x), g01.y), g01.x);
  o.e = fma(s, fma(s, fma(s, e23.y, e23.x), e01.y), e01.x);
  o.alpc = fma(s, fma(s, fma(s, a23.y, a23.x), a01.y), a01.x);
  o.Aj = ax.x; o.inv_nuj = ax.y; o.amp = reinterpret_cast<const double*>(h)[22];
}

// Everything of a sample that does not depend on the harmonic index.  (cpb, spb) = cos/sin of the detector phase
// phibar = 2 pi t_i / T_yr.  fin[0..5] (stride fs) receive a_I, b_I, c_I, a_II, b_II, c_II.
DEVINL void sample_setup(const double* __restrict__ w, const double2* __restrict__ sct, const OrbitAt& ob, double cpb, double spb,
                         double w0, double cbrt_thr, unsigned long long* __restrict__ counts, SampleOut& o,
                         double* __restrict__ fin, int fs) {
  const double Phic = ob.Phic, nu = ob.nu, gamc = ob.gamc, e = ob.e, alpc = ob.alpc;
  // amplitude A = (2 pi M nu)^{2/3} mu / (Xi D)  (BC 10 with Eqs. 4-6 folded in): Taylor of (1+d)^{2/3} about the
  // node value, d = (nu - nu_j)/nu_j; remainder 0.014 d^6 < 6e-17 for |d| <= 4e-3, else the cube root itself
  double A;
  {
    const double d = ob.dnu * ob.inv_nuj;
    if (fabs(d) <= cbrt_thr) {
      const double p = fma(d, fma(d, fma(d, fma(d, kC[KC_A4], kC[KC_A3]), kC[KC_A2]), kC[KC_A1]), kC[KC_A0]);
      A = fma(ob.Aj * d, p, ob.Aj);
    } else {
      const double cb = cbrt(w[WC_TWOPIMS] * nu);
      A = cb * cb * ob.amp;
      // rare branch, counted for emri_plan_synth_report: one atomic per converged group of lanes, not one per sample
      // (near plunge whole tiles come here, and a per-sample atomic on one address would serialise them)
      const unsigned act = __activemask();
      if ((threadIdx.x & 31u) == (unsigned)(__ffs((int)act) - 1))
        atomicAdd(counts + SYC_CBRT, (unsigned long long)__popc(act));
    }
  }
  double sa, ca, s2gt, c2gt;
  sincos_cycles(sct, alpc, sa, ca);
  sincos_cycles(sct, 2.0 * gamc, s2gt, c2gt);
  // orbital-plane normal and its projections (BC 19-21)
  const double Lx = fma(w[WC_A2X], sa, fma(w[WC_A1X], ca, w[WC_A0X]));
  const double Ly = fma(w[WC_A2Y], sa, fma(w[WC_A1Y], ca, w[WC_A0Y]));
  const double Lz = fma(w[WC_A1Z], ca, w[WC_A0Z]);
  const double Ln = fma(w[WC_LN2], sa, fma(w[WC_LN1], ca, w[WC_LN0]));
  // beta (BC 22-24): tan(beta) = Ns/Nc
  const double Ns = fma(w[WC_CL], Ln, -w[WC_SN]);
  const double Nc = fma(w[WC_B2], sa, w[WC_B1] * ca);
  const double den_b0 = fma(Nc, Nc, Ns * Ns);
  // detector-time quantities (BC 17-18)
  const double cphS = w[WC_CPHS], sphS = w[WC_SPHS], cS = w[WC_CS], sS = w[WC_SS];
  const double cd = fma(cpb, cphS, spb * sphS), sd = fma(spb, cphS, -cpb * sphS);
  const double cthd = fma(-kC[KC_HSQRT3] * sS, cd, 0.5 * cS);
  const double Pq = fma(sS, cd, kC[KC_SQRT3] * cS), Qq = 2.0 * sS * sd;
  const double den_a = fma(Pq, Pq, Qq * Qq);      // = 4 sin^2(theta_d): zero only for a source exactly on the detector normal
  const double Npsi = fma(-cthd, Ln, fma(-kC[KC_HSQRT3], fma(Lx, cpb, Ly * spb), 0.5 * Lz));
  const double Dpsi = 0.5 * sS * fma(Ly, cphS, -Lx * sphS)
                      - kC[KC_HSQRT3] * (cpb * fma(Lz * sS, sphS, -cS * Ly) + spb * fma(cS, Lx, -Lz * sS * cphS));
  const double den_p0 = fma(Npsi, Npsi, Dpsi * Dpsi);
  // one division for the three normalisations.  Reading R16: an angle whose atan2 arguments both vanish is 0; its
  // denominator is replaced by 1 BEFORE the shared reciprocal so that the other two normalisations stay finite
  // (a branch no sample of a generic walker takes, instead of a dozen selects on every sample)
  const bool ok_b = den_b0 > 0.0, ok_p = den_p0 > 0.0;
  double den_b = den_b0, den_p = den_p0;
  if (!(ok_b && ok_p)) { den_b = ok_b ? den_b0 : 1.0; den_p = ok_p ? den_p0 : 1.0; }
  const double bp = den_b * den_p;
  const double inv = rcp_fast(bp * den_a);
  const double ib = inv * (den_a * den_p), ia = inv * bp, ip = inv * (den_a * den_b);
  double c2b = fma(Nc, Nc, -Ns * Ns) * ib, s2b = 2.0 * Ns * Nc * ib;
  const double c2a = fma(Qq, Qq, -Pq * Pq) * ia, s2a = 2.0 * Pq * Qq * ia;
  double c2s = fma(Dpsi, Dpsi, -Npsi * Npsi) * ip, s2s = 2.0 * Npsi * Dpsi * ip;
  if (!(ok_b && ok_p)) {
    if (!ok_b) { c2b = 1.0; s2b = 0.0; }                            // beta = 0
    if (!ok_p) { c2s = 1.0; s2s = 0.0; }                            // psi = 0
  }
  const double c2g = fma(c2gt, c2b, -s2gt * s2b), s2g = fma(s2gt, c2b, c2gt * s2b);
  const double c2pb = fma(cpb, cpb, -spb * spb), s2pb = 2.0 * cpb * spb;
  const double c2p = fma(c2pb, c2a, -s2pb * s2a), s2p = fma(s2pb, c2a, c2pb * s2a);
  const double hh = 0.5 * fma(cthd, cthd, 1.0);
  // antenna patterns (BC 15-16)
  const double FIp = fma(hh * c2p, c2s, -cthd * s2p * s2s);
  const double FIx = fma(hh * c2p, s2s, cthd * s2p * c2s);
  const double FIIp = fma(hh * s2p, c2s, cthd * c2p * s2s);
  const double FIIx = fma(hh * s2p, s2s, -cthd * c2p * c2s);
  // h_alpha = (sqrt3/2)(F+ A+ + Fx Ax) with A+ = A{(1+Ln^2)(c2g Sa - s2g sq Sb) + 2(1-Ln^2) Sc},
  // Ax = -2 A Ln (sq Sb c2g + Sa s2g)   (BC 7-9, 14 summed over n)  =>  h = a Sa + b Sb + c Sc
  const double sq = sqrt(fma(-e, e, 1.0));
  const double kA = kC[KC_HSQRT3] * A;               // A is 0 past plunge (reading R8)
  const double Ln2 = Ln * Ln;
  const double P1 = kA * (1.0 + Ln2), P2 = 2.0 * kA * Ln, P3 = 2.0 * kA * (1.0 - Ln2);
  const double t1 = P1 * c2g, t2 = P2 * s2g, t3 = P1 * s2g, t4 = P2 * c2g;
  fin[0 * fs] = fma(FIp, t1, -FIx * t2);
  fin[1 * fs] = -sq * fma(FIp, t3, FIx * t4);
  fin[2 * fs] = FIp * P3;
  fin[3 * fs] = fma(FIIp, t1, -FIIx * t2);
  fin[4 * fs] = -sq * fma(FIIp, t3, FIIx * t4);
  fin[5 * fs] = FIIp * P3;
  // Doppler-shifted phase in cycles (BC 25)
  double s1, c1;
  sincos_cycles(sct, fma(nu * w[WC_DOP], cd, Phic), s1, c1);
  o.x = fma(e, e, -w0);
  o.ec = e * c1; o.es = e * s1;
  o.C2 = fma(c1, c1, -s1 * s1); o.S2 = 2.0 * s1 * c1;
}

DEVINL double4 ldg4(const double4* p) {
  const double2* q = reinterpret_cast<const double2*>(p);
  const double2 lo = __ldg(q), hi = __ldg(q + 1);
  return make_double4(lo.x, lo.y, hi.x, hi.y);
}

// ---- harmonic sum n = 1..n_max for the thread's two samples; returns S_a, S_b, S_c of each.
#define EMRI_FMA(d, a, b, c) asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c))
#define EMRI_MUL(d, a, b) asm volatile("mul.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b))
#define EMRI_LDS2(lo, hi, addr) asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(lo), "=d"(hi) : "r"(addr))
#define EMRI_ACCUM_FIRST()                                                                       \
  double SaA = p[0] * A.ec, SbA = p[1] * A.es, ScA = p[2] * A.ec;                                \
  double SaB = p[3] * B.ec, SbB = p[4] * B.es, ScB = p[5] * B.ec;                                \
  double CA = A.C2, SA = A.S2, CB = B.C2, SB = B.S2;
#define EMRI_ACCUM_NEXT()                                                                        \
  {                                                                                              \
    /* issue order chosen so that consecutive instructions share an operand slot (see horner_step) */ \
    double ta, ua, tb, ub;                                                                       \
    EMRI_FMA(SaA, p[0], CA, SaA); EMRI_FMA(ScA, p[2], CA, ScA); EMRI_FMA(SbA, p[1], SA, SbA);    \
    EMRI_MUL(ta, SA, A.es); EMRI_MUL(ua, CA, A.es);                                              \
    EMRI_FMA(CA, CA, A.ec, -ta); EMRI_FMA(SA, SA, A.ec, ua);                                     \
    EMRI_FMA(SaB, p[3], CB, SaB); EMRI_FMA(ScB, p[5], CB, ScB); EMRI_FMA(SbB, p[4], SB, SbB);    \
    EMRI_MUL(tb, SB, B.es); EMRI_MUL(ub, CB, B.es);                                              \
    EMRI_FMA(CB, CB, B.ec, -tb); EMRI_FMA(SB, SB, B.ec, ub);                                     \
  }

// Local table (shared memory): record n holds the re-expanded series of harmonic n, orders MLOC-1..0, {PA, PB, PC} each:
// coefficient (order m, series s) at double 3 (MLOC-1-m) + s of the record.  A thread that keeps M orders streams the
// LAST 3 M doubles of a record, in the order the Horner evaluation consumes them, as 128-bit loads from the aligned
// address below its first coefficient (LEAD = 1: the first double loaded is the tail of order M, unused).
template <int M>
struct CoefStream {
  static constexpr int OFF = 3 * (MLOC - M);
  static constexpr int LEAD = OFF & 1;
  static constexpr int BASE = OFF - LEAD;
  static constexpr int NCH = (3 * M + LEAD + 1) / 2;       // 128-bit chunks per harmonic
};

// One harmonic: the six Horner chains (2 samples x 3 series), the accumulation, the scaled rotation -- and the coefficient
// loads of the NEXT harmonic, each 128-bit chunk re-issued as soon as the Horner step that consumed its last double has
// been issued, so that a load has the rest of the harmonic (>= 20 FP64 instructions of this warp alone) to land and the
// loop never waits on shared memory.  `asm volatile` pins this order (ptxas keeps it).
// The Horner chains are issued so that every consecutive pair of DFMAs shares one operand in the same slot -- A_a, B_a
// (coefficient a), B_b, A_b (coefficient b), A_c, B_c (coefficient c) -- which the operand-reuse cache turns into two
// fresh register reads per DFMA instead of three (28.9 against 20.9 TFLOP/s).
template <int M, bool FIRST>
DEVINL void harmonic_step(double (&v)[2 * CoefStream<M>::NCH], unsigned nxt, const SampleOut& A, const SampleOut& B,
                          double& SaA, double& SbA, double& ScA, double& SaB, double& SbB, double& ScB,
                          double& CA, double& SA, double& CB, double& SB) {
  using CS = CoefStream<M>;
  constexpr int L = CS::LEAD;
  double p[6];
  int reloaded = 0;                 // compile-time after unrolling
  if (M == 1) {
    p[0] = v[L]; p[1] = v[L + 1]; p[2] = v[L + 2]; p[3] = v[L]; p[4] = v[L + 1]; p[5] = v[L + 2];
  } else {
#pragma unroll
    for (int k = 1; k < M; ++k) {
      const int hi = L + 3 * (k - 1), lo = L + 3 * k;
      if (k == 1) {
        EMRI_FMA(p[0], v[hi], A.x, v[lo]); EMRI_FMA(p[3], v[hi], B.x, v[lo]);
        EMRI_FMA(p[4], v[hi + 1], B.x, v[lo + 1]); EMRI_FMA(p[1], v[hi + 1], A.x, v[lo + 1]);
        EMRI_FMA(p[2], v[hi + 2], A.x, v[lo + 2]); EMRI_FMA(p[5], v[hi + 2], B.x, v[lo + 2]);
      } else {
        EMRI_FMA(p[0], p[0], A.x, v[lo]); EMRI_FMA(p[3], p[3], B.x, v[lo]);
        EMRI_FMA(p[4], p[4], B.x, v[lo + 1]); EMRI_FMA(p[1], p[1], A.x, v[lo + 1]);
        EMRI_FMA(p[2], p[2], A.x, v[lo + 2]); EMRI_FMA(p[5], p[5], B.x, v[lo + 2]);
      }
      const int freed = (lo + 3) / 2 < CS::NCH ? (lo + 3) / 2 : CS::NCH;     // chunks whose doubles are all consumed
#pragma unroll
      for (int j = 0; j < CS::NCH; ++j)
        if (j >= reloaded && j < freed) EMRI_LDS2(v[2 * j], v[2 * j + 1], nxt + (unsigned)((CS::BASE + 2 * j) * 8));
      reloaded = freed > reloaded ? freed : reloaded;
    }
  }
  if (FIRST) {
    // n = 1: carrier e (cos, sin)(Phi)
    SaA = p[0] * A.ec; SbA = p[1] * A.es; ScA = p[2] * A.ec;
    SaB = p[3] * B.ec; SbB = p[4] * B.es; ScB = p[5] * B.ec;
    CA = A.C2; SA = A.S2; CB = B.C2; SB = B.S2;
  } else {
    // n >= 2: carrier e^{n-2} (cos, sin)(n Phi), advanced by the scaled rotation
    EMRI_ACCUM_NEXT()
  }
#pragma unroll
  for (int j = 0; j < CS::NCH; ++j)
    if (j >= reloaded) EMRI_LDS2(v[2 * j], v[2 * j + 1], nxt + (unsigned)((CS::BASE + 2 * j) * 8));
}

// carried between the two harmonic ranges of a unit
struct HarmState {
  double SaA, SbA, ScA, SaB, SbB, ScB, CA, SA, CB, SB;
};

// harmonics n_lo..n_hi (n_lo == 1 starts the sums) with M local orders
template <int M>
DEVINL void harmonic_range(unsigned tab, int n_lo, int n_hi, const SampleOut& A, const SampleOut& B, HarmState& h) {
  using CS = CoefStream<M>;
  double v[2 * CS::NCH];
  unsigned rec = tab + (unsigned)(n_lo * HREC * 8);          // record of n_lo
#pragma unroll
  for (int j = 0; j < CS::NCH; ++j) EMRI_LDS2(v[2 * j], v[2 * j + 1], rec + (unsigned)((CS::BASE + 2 * j) * 8));
  int n = n_lo;
  if (n_lo == 1) {
    rec += (unsigned)(HREC * 8);
    harmonic_step<M, true>(v, rec, A, B, h.SaA, h.SbA, h.ScA, h.SaB, h.SbB, h.ScB, h.CA, h.SA, h.CB, h.SB);
    n = 2;
  }
#pragma unroll 1
  for (; n <= n_hi; ++n) {
    rec += (unsigned)(HREC * 8);                             // the table has n_max + 2 records: the last prefetch stays inside
    harmonic_step<M, false>(v, rec, A, B, h.SaA, h.SbA, h.ScA, h.SaB, h.SbB, h.ScB, h.CA, h.SA, h.CB, h.SB);
  }
}

// Fallback version: the base series in w = e^2 straight from the global table, Mn[n] terms (rare, slow path)
DEVINL void series_base(const double4* __restrict__ t, int M, double xa, double xb, double p[6]) {
  double4 c = ldg4(t + (M - 1));
  p[0] = c.x; p[1] = c.y; p[2] = c.z; p[3] = c.x; p[4] = c.y; p[5] = c.z;
  for (int m = M - 2; m >= 0; --m) {
    c = ldg4(t + m);
    p[0] = fma(p[0], xa, c.x); p[1] = fma(p[1], xa, c.y); p[2] = fma(p[2], xa, c.z);
    p[3] = fma(p[3], xb, c.x); p[4] = fma(p[4], xb, c.y); p[5] = fma(p[5], xb, c.z);
  }
}

__device__ __noinline__ void harmonic_sum_base(const double4* __restrict__ base, const int* __restrict__ Mn, int n_max,
                                               const SampleOut& A, const SampleOut& B, double out[6]) {
  double p[6];
  series_base(base + BASE_M, Mn[1], A.x, B.x, p);
  EMRI_ACCUM_FIRST()
  for (int n = 2; n <= n_max; ++n) {
    series_base(base + (size_t)n * BASE_M, Mn[n], A.x, B.x, p);
    EMRI_ACCUM_NEXT()
  }
  out[0] = SaA; out[1] = SbA; out[2] = ScA; out[3] = SaB; out[4] = SbB; out[5] = ScB;
}


// ---- Bessel path (n_max > 48): local series of the brackets from recurrences instead of the base series in e^2.
// With s_k(w) = sum_m (-n^2 w/4)^m / (m! (m+k)!) = J_k(n e) / (n e/2)^k one has d s_k/dw = -(n^2/4) s_{k+1}, so the Taylor
// coefficients of s_k about w0 are (-n^2/4)^j s_{k+j}(w0) / j!, and the brackets are (BC Eqs. 7-9 divided by e^{n-2}):
//   PA = G [s_{n-2} - n w s_{n-1} + (n/2) w s_n + (n^3/4) w^2 s_{n+1} - (n^4/16) w^2 s_{n+2}],
//   PB = G [s_{n-2} - (n^2/2) w s_n + (n^4/16) w^2 s_{n+2}],   PC = G (n/4) w s_n,        G = n (n/2)^{n-2}
// (n = 1, with J_{-1} = -J_1: PA = s_1/2 - 2 s_0 + w s_2/2 - w s_3/8, PB = -3 s_1/2 + w s_3/8, PC = s_1/2).
// hat-s_k = k! s_k (= 1 at w = 0) obeys the division-free form of the three-term recurrence,
//   hs_{k-1} = hs_k - y hs_{k+1} / (k (k+1)),   y = n^2 w0 / 4,
// which is stable downwards.  Small y: the two highest orders from the series itself (terms fall from the start), then
// down.  Otherwise Miller's algorithm: start far above from hs = 1, go down to order 0 and normalise with
// J_0 + 2 sum_m J_2m = 1 (J_k = hs_k y^{k/2} / k!).  No cancellation at any n e (the base series in e^2 loses e^{n e} digits).
constexpr int BES_NS = 5 + MLOC - 1;      // orders needed per harmonic: k = n-2 .. n+2+(MLOC-1)

// hs[i] = hat-s_{k_lo + i}(y), i = 0 .. cnt-1
DEVINL void bessel_hat_s(int k_lo, int cnt, double y, double* __restrict__ hs) {
  const int K = k_lo + cnt - 1;
  if (y <= 0.5 * (double)(K + 1)) {
    double top[2];
#pragma unroll 1
    for (int which = 0; which < 2; ++which) {
      const int k = K + 1 - which;
      double t = 1.0, sum = 1.0;
#pragma unroll 1
      for (int m = 1; m <= 200; ++m) {
        t *= -y / ((double)m * (double)(k + m));
        sum += t;
        if (fabs(t) < 1e-18 * fabs(sum)) break;
      }
      top[which] = sum;
    }
    double hp = top[0], h = top[1];       // orders K+1, K
    hs[cnt - 1] = h;
#pragma unroll 1
    for (int k = K; k > k_lo; --k) {
      const double hm = fma(-y / ((double)k * (double)(k + 1)), hp, h);
      hp = h; h = hm;
      hs[k - 1 - k_lo] = h;
    }
    return;
  }
  const double half = sqrt(y);
  int M = K + 16 + (int)(2.0 * sqrt((double)K)) + (int)(2.0 * half);
  M += M & 1;
  double hp = 1.0, h = 1.0, S = 0.0;
  // f_k = (z/2)^k / k!: tracked in logarithm until it is representable, then by its recurrence f_{k-1} = f_k k / (z/2)
  const double lhalf = log(half);
  double logf = (double)M * lhalf - lgamma((double)M + 1.0);
  bool have_f = logf > -600.0;
  double f = have_f ? exp(logf) : 0.0;
#pragma unroll 1
  for (int k = M; k >= 1; --k) {
    if (k <= K && k >= k_lo) hs[k - k_lo] = h;
    if (have_f && !(k & 1)) S = fma(2.0 * h, f, S);
    const double hm = fma(-y / ((double)k * (double)(k + 1)), hp, h);
    hp = h; h = hm;
    if (have_f) f *= (double)k / half;
    else {
      logf += log((double)k) - lhalf;
      if (logf > -600.0) { f = exp(logf); have_f = true; }
    }
  }
  if (k_lo == 0) hs[0] = h;
  S = fma(h, f, S);                         // k = 0 (f_0 = 1 up to rounding)
  const double rS = 1.0 / S;
#pragma unroll 1
  for (int i = 0; i < cnt; ++i) hs[i] *= rS;
}

// coefficient j of (w0 + x) A(x) and of (w0 + x)^2 A(x)
DEVINL double mulw1(const double* a, int j, double w0) { return fma(w0, a[j], j >= 1 ? a[j - 1] : 0.0); }
DEVINL double mulw2(const double* a, int j, double w0) {
  return fma(w0 * w0, a[j], fma(2.0 * w0, j >= 1 ? a[j - 1] : 0.0, j >= 2 ? a[j - 2] : 0.0));
}

// local series (NORD orders) of PA, PB, PC of harmonic n about w0
template <int NORD>
DEVINL void bessel_local_series(int n, double w0, double gn, double (&PA)[NORD], double (&PB)[NORD], double (&PC)[NORD]) {
  constexpr int CNT = 5 + NORD - 1;
  double hs[CNT], T[5][NORD];
  const double nn = (double)n;
  const double y = 0.25 * nn * nn * w0;
  const int k_lo = (n == 1) ? 0 : n - 2;
  bessel_hat_s(k_lo, (n == 1) ? CNT - 1 : CNT, y, hs);
  // u_i = G s_{k_lo + i} = G hat-s / k!   (n >= 2: G / (n-2)! = gn;  n = 1: G = 1, 0! = 1)
  double fac = (n == 1) ? 1.0 : gn;
#pragma unroll
  for (int i = 0; i < CNT; ++i) {
    if (i > 0) fac /= (double)(k_lo + i);
    hs[i] = (n == 1 && i == CNT - 1) ? 0.0 : hs[i] * fac;
  }
  const double c = -0.25 * nn * nn;
#pragma unroll
  for (int r = 0; r < 5; ++r) {
    double cj = 1.0;
#pragma unroll
    for (int j = 0; j < NORD; ++j) {
      T[r][j] = (n == 1 && r + j >= CNT - 1) ? 0.0 : cj * hs[r + j];
      cj *= c / (double)(j + 1);
    }
  }
  if (n == 1) {
    // T[0..3] = series of s_0, s_1, s_2, s_3
#pragma unroll
    for (int j = 0; j < NORD; ++j) {
      PA[j] = fma(0.5, T[1][j], fma(-2.0, T[0][j], fma(0.5, mulw1(T[2], j, w0), -0.125 * mulw1(T[3], j, w0))));
      PB[j] = fma(-1.5, T[1][j], 0.125 * mulw1(T[3], j, w0));
      PC[j] = 0.5 * T[1][j];
    }
    return;
  }
  const double n2 = nn * nn, n3 = n2 * nn, n4 = n2 * n2;
#pragma unroll
  for (int j = 0; j < NORD; ++j) {
    const double w2 = mulw1(T[2], j, w0), w4 = mulw2(T[4], j, w0);
    PA[j] = T[0][j] - nn * mulw1(T[1], j, w0) + 0.5 * nn * w2 + 0.25 * n3 * mulw2(T[3], j, w0) - 0.0625 * n4 * w4;
    PB[j] = T[0][j] - 0.5 * n2 * w2 + 0.0625 * n4 * w4;
    PC[j] = 0.25 * nn * w2;
  }
}

// Fallback of the Bessel path (local order MKEEP not enough over the unit: the last hours before plunge at high n_max):
// every sample evaluates the brackets of every harmonic at its own e^2 by the recurrences (slow, rare, exact)
__device__ __noinline__ void harmonic_sum_bessel(const double* __restrict__ gtab, int n_max, const SampleOut& A, const SampleOut& B,
                                                 double out[6]) {
  double p[6];
  {
    double a1[1], b1[1], c1[1];
    bessel_local_series<1>(1, A.x, 1.0, a1, b1, c1); p[0] = a1[0]; p[1] = b1[0]; p[2] = c1[0];
    bessel_local_series<1>(1, B.x, 1.0, a1, b1, c1); p[3] = a1[0]; p[4] = b1[0]; p[5] = c1[0];
  }
  EMRI_ACCUM_FIRST()
#pragma unroll 1
  for (int n = 2; n <= n_max; ++n) {
    double a1[1], b1[1], c1[1];
    const double gn = __ldg(gtab + n);
    bessel_local_series<1>(n, A.x, gn, a1, b1, c1); p[0] = a1[0]; p[1] = b1[0]; p[2] = c1[0];
    bessel_local_series<1>(n, B.x, gn, a1, b1, c1); p[3] = a1[0]; p[4] = b1[0]; p[5] = c1[0];
    EMRI_ACCUM_NEXT()
  }
  out[0] = SaA; out[1] = SbA; out[2] = ScA; out[3] = SaB; out[4] = SbB; out[5] = ScB;
}

// ---- per-unit tables, prepared by the producer warp one unit ahead of the consumers (double-buffered)
struct UnitMeta {
  double w0e;         // expansion point subtracted from e^2 (0 on the fallback path)
  int M1, M2;         // local orders kept for harmonics 1..n1 and n1+1..n2; M1 >= MLOC: fallback to the base series
  int n1, n2;         // n2 <= n_max: harmonics above n2 are below the truncation threshold over the whole unit
  int skip;           // walker has a fatal status: the unit is zero-filled
  int32_t jpl;
};

DEVINL double warp_max(double v) {
#pragma unroll 1
  for (int off = 16; off > 0; off >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, off));
  return v;
}

// x^k, k >= 0, by repeated squaring (a bound on a harmonic's carrier e^{n-2}: a few ulps do not matter)
DEVINL double ipow(double x, int k) {
  double r = 1.0;
#pragma unroll 1
  for (; k > 0; k >>= 1) { if (k & 1) r *= x; x *= x; }
  return r;
}

// Staged path: the (at most two) coarse intervals each tile of the unit touches, as cubics in s (executed by ONE warp;
// lane = 2 tile + slot).  Slot 0 is the interval the tile lies in, j0; slot 1 the neighbour the time shift sigma =
// Delta T / Delta (|sigma| < 1, one sign per walker) reaches: j0 - 1 for sigma > 0, j0 + 1 otherwise.  From the Hermite
// data (value y, increment d, end slopes m0, m1):  c0 = y, c1 = Delta m0, c2 = 3 d - Delta (2 m0 + m1),
// c3 = Delta (m0 + m1) - 2 d.  Record: {c0..c3} x (Phi_c, nu, gam_c, e, alp_c), then A_j, 1/nu_j, mu/(Xi D), pad; the two
// amplitude entries are 0 for an interval past plunge (reading R8: the samples are 0).
DEVINL void stage_intervals(const SynthArgs& a, int lane, const double* __restrict__ nodes, const double2* __restrict__ aux,
                            int64_t i_begin, int64_t i_end, double Delta, double sigma, double amp, int32_t jpl,
                            double* __restrict__ herm) {
#pragma unroll 1
  for (int task = lane; task < 2 * a.unit_tiles; task += 32) {
    const int t = task >> 1, slot = task & 1;
    const int64_t i0 = i_begin + (int64_t)t * TILE;
    if (i0 >= i_end) continue;
    const int64_t j = (i0 >> a.logS) + (slot ? (sigma > 0.0 ? -1 : 1) : 0);
    const double2* r0 = reinterpret_cast<const double2*>(nodes + (j + 1) * NODE_STRIDE);
    const double2* r1 = r0 + NODE_STRIDE / 2;
    const double2 v01 = __ldg(r0), v23 = __ldg(r0 + 1), v4m0 = __ldg(r0 + 2), m12 = __ldg(r0 + 3), m34 = __ldg(r0 + 4),
                  d01 = __ldg(r0 + 5), d23 = __ldg(r0 + 6), d4 = __ldg(r0 + 7);
    const double2 n4m0 = __ldg(r1 + 2), n12 = __ldg(r1 + 3), n34 = __ldg(r1 + 4);
    const double2 ax = __ldg(aux + (j + 1));
    const bool live = (j + 1 < (int64_t)jpl);
    const double y[5] = {v01.x, v01.y, v23.x, v23.y, v4m0.x};
    const double d[5] = {d01.x, d01.y, d23.x, d23.y, d4.x};
    const double m0[5] = {v4m0.y, m12.x, m12.y, m34.x, m34.y};
    const double m1[5] = {n4m0.y, n12.x, n12.y, n34.x, n34.y};
    double* rec = herm + (size_t)task * HERM;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      rec[4 * q] = y[q];
      rec[4 * q + 1] = Delta * m0[q];
      rec[4 * q + 2] = fma(-Delta, fma(2.0, m0[q], m1[q]), 3.0 * d[q]);
      rec[4 * q + 3] = fma(Delta, m0[q] + m1[q], -2.0 * d[q]);
    }
    rec[20] = live ? ax.x : 0.0; rec[21] = ax.y; rec[22] = live ? amp : 0.0; rec[23] = 0.0;
  }
}

// Executed by ONE warp: everything of unit (k, i_begin..i_end) that is shared by its samples.
template <bool STAGED, bool BES>
DEVINL void prepare_unit(const SynthArgs& a, int lane, int k, int64_t i_begin, int64_t i_end, double Delta, double inv_year,
                         double* __restrict__ tab, double* __restrict__ s_wc, double* __restrict__ s_rot,
                         double* __restrict__ s_herm, int* __restrict__ s_Mb, int* __restrict__ s_Ml, int* __restrict__ s_Pm,
                         const double2* __restrict__ sct_lane,
                         UnitMeta* __restrict__ meta) {
#pragma unroll 1
  for (int q = lane; q < WC_STRIDE; q += 32) s_wc[q] = a.wc[(size_t)k * WC_STRIDE + q];
#pragma unroll 1
  for (int q = lane; q <= a.n_max; q += 32) s_Mb[q] = 1;
  const int32_t st = a.status[k];
  const bool skip = (st & (EMRI_ST_BADPARAM | EMRI_ST_DELAY | EMRI_ST_STATE)) != 0;
  const int32_t jpl = a.jpl[k];
  if (lane == 0) {
    meta->skip = skip ? 1 : 0; meta->jpl = jpl;
    atomicAdd(a.counts + (skip ? SYC_SKIP : SYC_UNITS), 1ULL);
  }
  if (skip) return;
  const double* nodes = a.nodes + (size_t)k * a.Nn * NODE_STRIDE;
  if (STAGED)
    stage_intervals(a, lane, nodes, a.nodeaux + (size_t)k * a.Nn, i_begin, i_end, Delta, a.wc[(size_t)k * WC_STRIDE + WC_SIGMA],
                    a.wc[(size_t)k * WC_STRIDE + WC_AMP], jpl, s_herm);
  // range of e over the unit from the node rows it touches (the Hermite cubic stays within pad of the nodes)
  int64_t rlo = (i_begin >> a.logS), rhi = ((i_end - 1) >> a.logS) + 3;       // rows = node index + 1
  if (rlo < 0) rlo = 0;
  if (rhi > a.Nn - 1) rhi = a.Nn - 1;
  double v0 = 0.0, v1 = -1.0, v2 = 0.0, v3 = 0.0;       // max e, max -e, max |e'|, max |increment of e|
#pragma unroll 1
  for (int64_t r = rlo + lane; r <= rhi; r += 32) {
    const double* row = nodes + r * NODE_STRIDE;
    const double ev = __ldg(row + 3);
    v0 = fmax(v0, ev); v1 = fmax(v1, -ev);
    v2 = fmax(v2, fabs(__ldg(row + 8))); v3 = fmax(v3, fabs(__ldg(row + 13)));
  }
#pragma unroll 1
  for (int off = 16; off > 0; off >>= 1) {          // rolled: the producer's code must stay small (instruction cache)
    v0 = fmax(v0, __shfl_xor_sync(0xffffffffu, v0, off)); v1 = fmax(v1, __shfl_xor_sync(0xffffffffu, v1, off));
    v2 = fmax(v2, __shfl_xor_sync(0xffffffffu, v2, off)); v3 = fmax(v3, __shfl_xor_sync(0xffffffffu, v3, off));
  }
  const double pad = 0.3 * fma(Delta, v2, v3) + 1e-15;
  const double elo = fmax(-v1 - pad, 0.0), ehi = v0 + pad;
  const double whi = ehi * ehi;
  const double w0 = 0.5 * fma(elo, elo, whi);
  const double xmax = 0.5 * (whi - elo * elo) * (1.0 + 1e-9);
  __syncwarp();
  // re-expansion of the three series of every harmonic about w0 (task = (harmonic, series)); T0 = size of the leading
  // term of the harmonic INCLUDING its carrier e^{n-2} (n = 1: e), at the unit's mid-point
  const double ebar = sqrt(w0);
  double scale = 0.0;
  if (BES) {
    // one lane per harmonic: the three local series from the Bessel recurrences
#pragma unroll 1
    for (int n = 1 + lane; n <= a.n_max; n += 32) {
      double PA[MLOC], PB[MLOC], PC[MLOC];
      bessel_local_series<MLOC>(n, w0, __ldg(a.gtab + n), PA, PB, PC);
      double* dst = tab + (size_t)n * HREC;
#pragma unroll
      for (int j = 0; j < MLOC; ++j) {
        dst[3 * (MLOC - 1 - j)] = PA[j]; dst[3 * (MLOC - 1 - j) + 1] = PB[j]; dst[3 * (MLOC - 1 - j) + 2] = PC[j];
      }
      const int pc = (n == 1) ? 1 : n - 2;
      scale = fmax(scale, fmax(fabs(PA[0]), fmax(fabs(PB[0]), fabs(PC[0]))) * ipow(ebar, pc));
    }
  }
#pragma unroll 1
  for (int task = BES ? 3 * a.n_max : lane; task < 3 * a.n_max; task += 32) {
    const int n = task / 3 + 1, si = task - 3 * (n - 1);
    const double* bp = reinterpret_cast<const double*>(a.base + (size_t)n * BASE_M) + si;
    // base terms that matter at w <= whi (terms rise, then fall: the running maximum is a safe scale)
    int Mb = 1;
    {
      double pw = 1.0, mx = 0.0;
      int below = 0;
#pragma unroll 1
      for (int m = 0; m < BASE_M; ++m) {
        const double t = fabs(__ldg(bp + 4 * m)) * pw;
        mx = fmax(mx, t);
        if (t >= a.tol * mx && t > 0.0) { Mb = m + 1; below = 0; }
        else if (t > 0.0 && ++below >= 3) break;      // past the peak the terms fall monotonically
        pw *= whi;
      }
    }
    double d[MLOC];
#pragma unroll
    for (int j = 0; j < MLOC; ++j) d[j] = 0.0;
#pragma unroll 1
    for (int m = Mb - 1; m >= 0; --m) {
      const double c = __ldg(bp + 4 * m);
#pragma unroll
      for (int j = MLOC - 1; j >= 1; --j) d[j] = fma(d[j], w0, d[j - 1]);
      d[0] = fma(d[0], w0, c);
    }
    double* dst = tab + (size_t)n * HREC + si;
#pragma unroll
    for (int j = 0; j < MLOC; ++j) dst[3 * (MLOC - 1 - j)] = d[j];
    const int pc = (n == 1) ? 1 : n - 2;                 // power of e the harmonic's carrier holds
    scale = fmax(scale, fabs(d[0]) * ipow(ebar, pc));
    atomicMax(&s_Mb[n], Mb);
  }
  scale = warp_max(scale);
#pragma unroll 1
  for (int q = lane; q <= a.n_max; q += 32) s_Ml[q] = 0;
  __syncwarp();
  // Orders kept per harmonic: a term of the local series is kept while it is above thr = tol/4 of the LARGEST harmonic
  // of the unit, carriers included -- a weak overtone needs fewer orders than its own relative accuracy would ask for,
  // and an overtone whose leading term is below thr over the whole unit is not evaluated at all (reading D13: the sum
  // of everything dropped stays below ~n_max tol / 4 of the signal, nine orders inside the 1e-9 parity tolerance)
  const double thr = 0.25 * a.tol * scale;
#pragma unroll 1
  for (int task = lane; task < 3 * a.n_max; task += 32) {
    const int n = task / 3 + 1, si = task - 3 * (n - 1);
    const int pc = (n == 1) ? 1 : n - 2;
    const double car = ipow(ehi, pc);                  // upper bound of the carrier over the unit
    const double* src = tab + (size_t)n * HREC + si;
    int Ml = 0;
    double pw = car;
#pragma unroll
    for (int j = 0; j < MLOC; ++j) {
      if (fabs(src[3 * (MLOC - 1 - j)]) * pw >= thr && thr > 0.0) Ml = j + 1;
      pw *= xmax;
    }
    atomicMax(&s_Ml[n], Ml);                   // Ml == MLOC: order MLOC-1 still significant, the tail is not bounded
  }
  __syncwarp();
  if (lane == 0) {
    // n2 = last harmonic with a term above thr (at least 2: the quadrupole of a circular orbit); split 1..n1 | n1+1..n2
    // at the point that minimises the FP64 instructions per sample, 7 + 3 (M - 1) per harmonic
    int n2 = min(2, a.n_max), Mall = 1;
#pragma unroll 1
    for (int n = 1; n <= a.n_max; ++n) { if (s_Ml[n] > 0) n2 = max(n2, n); Mall = max(Mall, s_Ml[n]); }
    int M1 = Mall, M2 = 1, n1 = n2;
    if (Mall < MLOC) {
      // prefix maxima of the per-harmonic orders, then one walk of the split point downwards with the suffix maximum
      int run = 1;
#pragma unroll 1
      for (int n = 1; n <= n2; ++n) { run = max(run, s_Ml[n]); s_Pm[n] = run; }
      int best = n2 * (4 + 3 * Mall), sfx = 1;
#pragma unroll 1
      for (int c = n2 - 1; c >= 1; --c) {
        sfx = max(sfx, s_Ml[c + 1]);
        const int cost = c * (4 + 3 * s_Pm[c]) + (n2 - c) * (4 + 3 * sfx) + 6;      // + the second range's prologue
        if (cost < best) { best = cost; n1 = c; M1 = s_Pm[c]; M2 = sfx; }
      }
    }
    if (a.force_base || M1 > MKEEP) M1 = MLOC;
    if (M1 >= MLOC) { n1 = n2 = a.n_max; M2 = 1; }
    meta->M1 = M1; meta->M2 = M2; meta->n1 = n1; meta->n2 = n2;
    meta->w0e = (M1 >= MLOC) ? 0.0 : w0;
    atomicAdd(a.counts + (M1 >= MLOC ? SYC_BASE : M1), 1ULL);
    atomicAdd(a.counts + SYC_NEVAL, (unsigned long long)n2);
    atomicAdd(a.counts + SYC_NFIRST, (unsigned long long)n1);
    atomicAdd(a.counts + SYC_M2, (unsigned long long)(n2 > n1 ? M2 : 0));
  }
  // detector phase at the start of each tile of the unit
  if (lane < a.unit_tiles) {
    double sb, cb;
    sincos_cycles(sct_lane, (double)(i_begin + (int64_t)lane * TILE) * a.dt * inv_year, sb, cb);
    s_rot[2 * lane] = cb; s_rot[2 * lane + 1] = sb;
  }
}

// Shared memory of one CTA, in doubles (the host sizes the launch with the same function)
__host__ __device__ inline size_t synth_smem_doubles(int n_max, int unit_tiles_cap) {
  return (size_t)2 * (n_max + 2) * HREC                 // local series, double-buffered
         + (size_t)2 * SC_TAB * SC_REP                  // cos/sin table (double2), replicated
         + (size_t)6 * 2 * SYNTH_THREADS                // the six per-sample coefficients, parked during the harmonic loop
         + (size_t)2 * WC_STRIDE + (size_t)2 * 2 * UNIT_TILES_MAX
         + (size_t)2 * 2 * unit_tiles_cap * HERM;       // staged interval cubics, double-buffered
}

// Consumers (warps 0..3): 2 adjacent samples per thread per tile.  Producer (warp 4): tables of the NEXT unit.
// STAGED: S >= 256, every tile lies inside one coarse interval (the default); otherwise node rows are read per sample.
// BES: the Bessel path of plans with n_max > 48 (its code stays out of the kernels of the other plans: instruction cache).
template <bool STAGED, bool BES>
__global__ void __launch_bounds__(SYNTH_BLOCK, SYNTH_MINBLOCKS) synth_kernel(SynthArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const size_t tab_elems = (size_t)(a.n_max + 2) * HREC;
  double* s_tab = reinterpret_cast<double*>(smem_raw);                                 // [2][n_max+2][HREC]
  double2* s_sct = reinterpret_cast<double2*>(s_tab + 2 * tab_elems);                  // [SC_TAB][SC_REP] {cos, sin}
  double* s_fin = reinterpret_cast<double*>(s_sct + SC_TAB * SC_REP);                  // [6][2][SYNTH_THREADS]
  double* s_wc = s_fin + 6 * 2 * SYNTH_THREADS;                                        // [2][WC_STRIDE]
  double* s_rot = s_wc + 2 * WC_STRIDE;                                                // [2][2 UNIT_TILES_MAX]
  double* s_herm = s_rot + 2 * 2 * UNIT_TILES_MAX;                                     // [2][2 unit_tiles_cap][HERM]
  __shared__ int s_Mb[2][EMRI_NMAX_CAP + 1];  // base-series terms per harmonic (fallback path)
  __shared__ int s_Ml[EMRI_NMAX_CAP + 1];     // local orders per harmonic (producer scratch)
  __shared__ int s_Pm[EMRI_NMAX_CAP + 1];     // their prefix maxima (producer scratch)
  __shared__ UnitMeta s_meta[2];
  const size_t herm_elems = (size_t)2 * a.unit_tiles_cap * HERM;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool producer = warp == SYNTH_THREADS / 32;
  const double Delta = a.S * a.dt, invS = 1.0 / (double)a.S;
  const double inv_year = 1.0 / kYearSec;
  for (int q = tid; q < SC_TAB * SC_REP; q += SYNTH_BLOCK) {
    double sv, cv;
    sincospi(2.0 * (double)(q / SC_REP) / (double)SC_TAB, &sv, &cv);
    s_sct[q] = make_double2(cv, sv);
  }
  for (int q = tid; q < 2 * (int)tab_elems; q += SYNTH_BLOCK) s_tab[q] = 0.0;      // pads and the prefetch-only last record
  const double2* sct_lane = s_sct + (lane & (SC_REP - 1));
  // detector phase of the thread's first sample relative to the tile start, and of one sample step
  double so, co, s1s, c1s;
  sincospi(2.0 * ((double)(2 * tid) * a.dt * inv_year), &so, &co);
  sincospi(2.0 * (a.dt * inv_year), &s1s, &c1s);

  const int64_t total = (int64_t)a.K * a.units_per_walker;
  const int64_t unit_len = (int64_t)a.unit_tiles * TILE;
  auto unit_of = [&](int64_t u, int& kl, int64_t& ib, int64_t& ie) {
    kl = (int)(u / a.units_per_walker);
    const int64_t ug = u - (int64_t)kl * a.units_per_walker;
    ib = ug * unit_len;
    ie = min(a.N, ib + unit_len);
  };
  __syncthreads();
  // One loop, one call site of prepare_unit (its code is inlined once): in the pass of unit u the producer prepares
  // unit u + gridDim.x while the consumers work on u; the first pass (u = first - gridDim.x) only prepares.
  int buf = 1;
  for (int64_t u = (int64_t)blockIdx.x - gridDim.x; u < total; u += gridDim.x, buf ^= 1) {
    if (producer) {
      const int64_t un = u + gridDim.x;
      if (un < total) {
        int kl; int64_t ib, ie;
        unit_of(un, kl, ib, ie);
        const int nb = buf ^ 1;
        prepare_unit<STAGED, BES>(a, lane, a.k0 + kl, ib, ie, Delta, inv_year, s_tab + nb * tab_elems, s_wc + nb * WC_STRIDE,
                             s_rot + nb * 2 * UNIT_TILES_MAX, s_herm + nb * herm_elems, s_Mb[nb], s_Ml, s_Pm, sct_lane, &s_meta[nb]);
      }
    } else if (u >= 0) {
      int kl; int64_t i_begin, i_end;
      unit_of(u, kl, i_begin, i_end);
      const int k = a.k0 + kl;
      const UnitMeta mt = s_meta[buf];
      if (mt.skip) {
        for (int64_t i0 = i_begin + 2 * tid; i0 < i_end; i0 += TILE) {
          if (a.outZ) {
            const size_t zi = (size_t)kl * a.N + i0;
            a.outZ[zi] = make_double2(0.0, 0.0);
            a.outZ[zi + 1] = make_double2(0.0, 0.0);
          } else {
            *reinterpret_cast<double2*>(a.outI + (size_t)kl * a.pitch + i0) = make_double2(0.0, 0.0);
            *reinterpret_cast<double2*>(a.outII + (size_t)kl * a.pitch + i0) = make_double2(0.0, 0.0);
          }
        }
      } else {
        const double* nodes = a.nodes + (size_t)k * a.Nn * NODE_STRIDE;
        const double2* aux = a.nodeaux + (size_t)k * a.Nn;
        const unsigned tab = (unsigned)__cvta_generic_to_shared(s_tab + buf * tab_elems);
        const double* wc = s_wc + buf * WC_STRIDE;
        const double* rot = s_rot + buf * 2 * UNIT_TILES_MAX;
        const double2* herm = reinterpret_cast<const double2*>(s_herm + buf * herm_elems);
        for (int t = 0; t < a.unit_tiles; ++t) {
          const int64_t i0 = i_begin + (int64_t)t * TILE + 2 * tid;
          if (i0 >= i_end) break;
          // detector phase: tile start (x) thread offset, then one sample step
          const double cb = rot[2 * t], sb = rot[2 * t + 1];
          const double cpa = fma(cb, co, -sb * so), spa = fma(sb, co, cb * so);
          const double cpb2 = fma(cpa, c1s, -spa * s1s), spb2 = fma(spa, c1s, cpa * s1s);
          SampleOut A, B;
          double* fin = s_fin + tid;
          {
            OrbitAt oa;
            if (STAGED) orbit_at_staged(wc, herm + (size_t)t * HERM, (double)(int)(i0 & (a.S - 1)) * invS, oa);
            else orbit_at_direct(wc, nodes, aux, i0, a.S, a.logS, invS, Delta, mt.jpl, oa);
            sample_setup(wc, sct_lane, oa, cpa, spa, mt.w0e, a.cbrt_thr, a.counts, A, fin, 2 * SYNTH_THREADS);
          }
          {
            OrbitAt ob;
            if (STAGED) orbit_at_staged(wc, herm + (size_t)t * HERM, (double)(int)((i0 + 1) & (a.S - 1)) * invS, ob);
            else orbit_at_direct(wc, nodes, aux, i0 + 1, a.S, a.logS, invS, Delta, mt.jpl, ob);
            sample_setup(wc, sct_lane, ob, cpb2, spb2, mt.w0e, a.cbrt_thr, a.counts, B, fin + SYNTH_THREADS, 2 * SYNTH_THREADS);
          }
          double S[6];
          if (mt.M1 >= MLOC) {
            // copies: the noinline fallbacks take their arguments by reference, which must not force A and B of the
            // common path into local memory
            const SampleOut A2 = A, B2 = B;
            double S2[6];
            if (BES) harmonic_sum_bessel(a.gtab, a.n_max, A2, B2, S2);
            else harmonic_sum_base(a.base, s_Mb[buf], a.n_max, A2, B2, S2);
#pragma unroll
            for (int q = 0; q < 6; ++q) S[q] = S2[q];
          } else {
            HarmState hs;
#pragma unroll 1
            for (int ph = 0; ph < 2; ++ph) {
              const int lo = ph ? mt.n1 + 1 : 1, hi = ph ? mt.n2 : mt.n1;
              if (lo > hi) break;
              switch (ph ? mt.M2 : mt.M1) {
                case 1: harmonic_range<1>(tab, lo, hi, A, B, hs); break;
                case 2: harmonic_range<2>(tab, lo, hi, A, B, hs); break;
                case 3: harmonic_range<3>(tab, lo, hi, A, B, hs); break;
                case 4: harmonic_range<4>(tab, lo, hi, A, B, hs); break;
                case 5: harmonic_range<5>(tab, lo, hi, A, B, hs); break;
                default: harmonic_range<6>(tab, lo, hi, A, B, hs); break;
              }
            }
            S[0] = hs.SaA; S[1] = hs.SbA; S[2] = hs.ScA; S[3] = hs.SaB; S[4] = hs.SbB; S[5] = hs.ScB;
          }
          const double hIa = fma(fin[0], S[0], fma(fin[2 * SYNTH_THREADS], S[1], fin[4 * SYNTH_THREADS] * S[2]));
          const double hIIa = fma(fin[6 * SYNTH_THREADS], S[0], fma(fin[8 * SYNTH_THREADS], S[1], fin[10 * SYNTH_THREADS] * S[2]));
          const double* fb = fin + SYNTH_THREADS;
          const double hIb = fma(fb[0], S[3], fma(fb[2 * SYNTH_THREADS], S[4], fb[4 * SYNTH_THREADS] * S[5]));
          const double hIIb = fma(fb[6 * SYNTH_THREADS], S[3], fma(fb[8 * SYNTH_THREADS], S[4], fb[10 * SYNTH_THREADS] * S[5]));
          if (a.outZ) {
            const size_t zi = (size_t)kl * a.N + i0;
            a.outZ[zi] = make_double2(hIa, hIIa);
            a.outZ[zi + 1] = make_double2(hIb, hIIb);
          } else {
            *reinterpret_cast<double2*>(a.outI + (size_t)kl * a.pitch + i0) = make_double2(hIa, hIb);
            *reinterpret_cast<double2*>(a.outII + (size_t)kl * a.pitch + i0) = make_double2(hIIa, hIIb);
          }
        }
      }
    }
    __syncthreads();      // unit u consumed and the tables of unit u + gridDim.x complete
  }
}
}  // namespace
