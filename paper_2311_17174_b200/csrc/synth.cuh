// synth.cuh -- stage (b): cubic-Hermite orbit, Peters-Mathews harmonic sum (Eq. 2), LISA response, propagation factors (Eqs. 4-6)
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
#pragma once
#include "common.cuh"

namespace {

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

}  // namespace
