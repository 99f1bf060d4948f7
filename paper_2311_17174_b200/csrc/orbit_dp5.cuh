// orbit_dp5.cuh -- stage (a) with the paper's own kind of integrator (next row f-3, reading D14): an embedded
// Runge-Kutta pair with per-walker step control and dense output on the device.  PAPER.md:120 "standard ODE methods, such
// as the 7th-order Runge-Kutta scheme", :133 solve_ivp, :157 "an important computational overhead ... the ODE solver".
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
//
// Scheme: Dormand-Prince 5(4) (RK5(4)7M, first-same-as-last), the step-size controller of Hairer, Norsett & Wanner (sec.
// II.4) in the form SciPy's solve_ivp uses (error norm = rms of err_q / (atol_q + rtol max(|Y_q|, |Y_q,new|)), factor
// 0.9 err^{-1/5} clipped to [0.2, 10], no growth after a rejection, first step from the two-evaluation estimate), and
// Shampine's 4th-order continuous extension.  The three angles are kept wrapped to [0, 1) cycles (reading D2) and the whole
// cycles removed are remembered for the error scale only.
//   orbit_dp5_kernel        one thread per walker: prologue (a0), then the two branches from the anchor (forward to node
//                           Nc+1, backward to node -1), every accepted step recorded with its dense-output polynomial;
//   orbit_dp5_nodes_kernel  one thread per (walker, coarse node): binary search of the step that holds the node, value from
//                           the dense output, slope = right-hand side AT the node, unwrapped increment to the next node pieced
//                           together step by step; first plunged / unusable node by atomicMin;
//   orbit_dp5_finish_kernel post-plunge copies, zero rows, status bits, the per-node amplitude pair.
// The node table is the one the fixed-step scheme produces, so stages (b)-(d) are unchanged: between nodes S4's cubic
// Hermite stays (its truncation error at the default stride is below the rounding of the phases).
#pragma once
#include "common.cuh"
#include "orbit.cuh"

namespace {

constexpr int DP_REC = 32;        // doubles per recorded step: t, h, y[5], D[5], Q[5][4]
constexpr int DP_SHORT = 64;      // capacity of the short branch (one coarse interval from the anchor)

struct Dp5Args {
  OrbitArgs o;
  double rtol, atol[5];
  double* steps;          // [K][cap_long + DP_SHORT][DP_REC]: the long branch first, then the short one
  int32_t* nsteps;        // [K][2] accepted steps of the {forward, backward} branch
  int32_t* stop;          // [K][2] 0 / EMRI_ST_PLUNGE / EMRI_ST_STATE: why the branch ended early
  int32_t* first_bad;     // [K] 4 * (first unusable node index j + 1) + {0 plunge, 1 state}; INT_MAX if none
  int32_t* zero_flag;     // [K] != 0: the walker's rows are zero (guard side or LSO convention hit a bad state)
  int cap_long;
};

DEVINL double* dp5_branch_base(const Dp5Args& a, int k, int branch) {
  // forward convention: the forward branch is the long one; LSO convention: the backward one
  const bool is_long = (branch == 0) != (a.o.anchor_end != 0);
  return a.steps + ((size_t)k * (a.cap_long + DP_SHORT) + (is_long ? 0 : a.cap_long)) * DP_REC;
}
DEVINL int dp5_branch_cap(const Dp5Args& a, int branch) {
  return ((branch == 0) != (a.o.anchor_end != 0)) ? a.cap_long : DP_SHORT;
}

DEVINL double rms5(const double v[5]) {
  return sqrt((v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + v[3] * v[3] + v[4] * v[4]) / 5.0);
}

// one branch from (t0, y0) to t_bound; returns the stop code
__device__ __noinline__ int dp5_branch(const OrbitConst& oc, const double y0[5], double t0, double t_bound, double rtol,
                                       const double atol[5], bool stop_at_plunge, double* __restrict__ rec, int cap,
                                       int32_t* __restrict__ n_out) {
  // Dormand & Prince 1980, RK5(4)7M
  const double A21 = 1.0 / 5, A31 = 3.0 / 40, A32 = 9.0 / 40, A41 = 44.0 / 45, A42 = -56.0 / 15, A43 = 32.0 / 9,
               A51 = 19372.0 / 6561, A52 = -25360.0 / 2187, A53 = 64448.0 / 6561, A54 = -212.0 / 729,
               A61 = 9017.0 / 3168, A62 = -355.0 / 33, A63 = 46732.0 / 5247, A64 = 49.0 / 176, A65 = -5103.0 / 18656;
  const double B1 = 35.0 / 384, B3 = 500.0 / 1113, B4 = 125.0 / 192, B5 = -2187.0 / 6784, B6 = 11.0 / 84;
  const double E1 = -71.0 / 57600, E3 = 71.0 / 16695, E4 = -71.0 / 1920, E5 = 17253.0 / 339200, E6 = -22.0 / 525, E7 = 1.0 / 40;
  // Shampine's continuous extension, P[i][j] (row 2 is zero)
  const double P[7][4] = {
      {1.0, -8048581381.0 / 2820520608.0, 8663915743.0 / 2820520608.0, -12715105075.0 / 11282082432.0},
      {0.0, 0.0, 0.0, 0.0},
      {0.0, 131558114200.0 / 32700410799.0, -68118460800.0 / 10900136933.0, 87487479700.0 / 32700410799.0},
      {0.0, -1754552775.0 / 470086768.0, 14199869525.0 / 1410260304.0, -10690763975.0 / 1880347072.0},
      {0.0, 127303824393.0 / 49829197408.0, -318862633887.0 / 49829197408.0, 701980252875.0 / 199316789632.0},
      {0.0, -282668133.0 / 205662961.0, 2019193451.0 / 616988883.0, -1453857185.0 / 822651844.0},
      {0.0, 40617522.0 / 29380423.0, -110615467.0 / 29380423.0, 69997945.0 / 29380423.0}};
  int n = 0, stop = 0;
  *n_out = 0;
  if (t_bound == t0) return 0;
  const double dir = (t_bound >= t0) ? 1.0 : -1.0;
  double t = t0, y[5], turns[3] = {0.0, 0.0, 0.0}, f[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) y[q] = y0[q];
  f[0] = y[1];
  rhs(oc, y[1], y[3], &f[1], &f[2], &f[3], &f[4]);
  auto unwrapped = [&](const double* yy, int q) -> double {
    return (q == 0) ? turns[0] + yy[0] : (q == 2) ? turns[1] + yy[2] : (q == 4) ? turns[2] + yy[4] : yy[q];
  };
  double h_abs;
  {
    const double interval = fabs(t_bound - t0);
    double sc[5], v0[5], v1[5], y1[5], f1[5], v2[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      sc[q] = atol[q] + fabs(unwrapped(y, q)) * rtol;
      v0[q] = unwrapped(y, q) / sc[q]; v1[q] = f[q] / sc[q];
    }
    const double d0 = rms5(v0), d1 = rms5(v1);
    double h0 = (d0 < 1e-5 || d1 < 1e-5) ? 1e-6 : 0.01 * d0 / d1;
    h0 = fmin(h0, interval);
#pragma unroll
    for (int q = 0; q < 5; ++q) y1[q] = y[q] + h0 * dir * f[q];
    f1[0] = y1[1];
    rhs(oc, y1[1], y1[3], &f1[1], &f1[2], &f1[3], &f1[4]);
#pragma unroll
    for (int q = 0; q < 5; ++q) v2[q] = (f1[q] - f[q]) / sc[q];
    const double d2 = rms5(v2) / h0;
    const double h1 = (d1 <= 1e-15 && d2 <= 1e-15) ? fmax(1e-6, h0 * 1e-3) : pow(0.01 / fmax(d1, d2), 0.2);
    h_abs = fmin(fmin(100.0 * h0, h1), interval);
  }
  while (t != t_bound) {
    if (n >= cap) { stop = EMRI_ST_STATE; break; }
    const double min_step = 10.0 * fabs(nextafter(t, dir * INFINITY) - t);
    if (h_abs < min_step) h_abs = min_step;
    bool rejected = false, failed = false;
    double K[7][5], y_new[5], h = 0.0, t_new = t;
    for (;;) {
      if (h_abs < min_step) { failed = true; break; }
      h = h_abs * dir;
      t_new = t + h;
      if (dir * (t_new - t_bound) > 0.0) t_new = t_bound;
      h = t_new - t;
      h_abs = fabs(h);
#pragma unroll
      for (int q = 0; q < 5; ++q) K[0][q] = f[q];
      double ys[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) ys[q] = y[q] + (A21 * K[0][q]) * h;
      K[1][0] = ys[1]; rhs(oc, ys[1], ys[3], &K[1][1], &K[1][2], &K[1][3], &K[1][4]);
#pragma unroll
      for (int q = 0; q < 5; ++q) ys[q] = y[q] + (A31 * K[0][q] + A32 * K[1][q]) * h;
      K[2][0] = ys[1]; rhs(oc, ys[1], ys[3], &K[2][1], &K[2][2], &K[2][3], &K[2][4]);
#pragma unroll
      for (int q = 0; q < 5; ++q) ys[q] = y[q] + (A41 * K[0][q] + A42 * K[1][q] + A43 * K[2][q]) * h;
      K[3][0] = ys[1]; rhs(oc, ys[1], ys[3], &K[3][1], &K[3][2], &K[3][3], &K[3][4]);
#pragma unroll
      for (int q = 0; q < 5; ++q) ys[q] = y[q] + (A51 * K[0][q] + A52 * K[1][q] + A53 * K[2][q] + A54 * K[3][q]) * h;
      K[4][0] = ys[1]; rhs(oc, ys[1], ys[3], &K[4][1], &K[4][2], &K[4][3], &K[4][4]);
#pragma unroll
      for (int q = 0; q < 5; ++q)
        ys[q] = y[q] + (A61 * K[0][q] + A62 * K[1][q] + A63 * K[2][q] + A64 * K[3][q] + A65 * K[4][q]) * h;
      K[5][0] = ys[1]; rhs(oc, ys[1], ys[3], &K[5][1], &K[5][2], &K[5][3], &K[5][4]);
#pragma unroll
      for (int q = 0; q < 5; ++q)
        y_new[q] = y[q] + h * (B1 * K[0][q] + B3 * K[2][q] + B4 * K[3][q] + B5 * K[4][q] + B6 * K[5][q]);
      K[6][0] = y_new[1]; rhs(oc, y_new[1], y_new[3], &K[6][1], &K[6][2], &K[6][3], &K[6][4]);
      double en[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const double e = E1 * K[0][q] + E3 * K[2][q] + E4 * K[3][q] + E5 * K[4][q] + E6 * K[5][q] + E7 * K[6][q];
        const double Yo = unwrapped(y, q), Yn = (q == 1 || q == 3) ? y_new[q] : Yo + (y_new[q] - y[q]);
        en[q] = e * h / (atol[q] + fmax(fabs(Yo), fabs(Yn)) * rtol);
      }
      const double err = rms5(en);
      if (err < 1.0) {
        double factor = (err == 0.0) ? 10.0 : fmin(10.0, 0.9 * pow(err, -0.2));
        if (rejected && factor > 1.0) factor = 1.0;
        h_abs *= factor;
        break;
      }
      h_abs *= fmax(0.2, 0.9 * pow(err, -0.2));
      rejected = true;
    }
    if (failed) { stop = EMRI_ST_STATE; break; }
    // record: t, h, y[5], D[5], Q[5][4]
    double* r = rec + (size_t)n * DP_REC;
    r[0] = t; r[1] = h;
#pragma unroll
    for (int q = 0; q < 5; ++q) { r[2 + q] = y[q]; r[7 + q] = y_new[q] - y[q]; }
#pragma unroll
    for (int q = 0; q < 5; ++q)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        double c = 0.0;
#pragma unroll
        for (int i = 0; i < 7; ++i) c += K[i][q] * P[i][j];
        r[12 + 4 * q + j] = h * c;
      }
    ++n;
#pragma unroll
    for (int q = 0; q < 5; ++q) { y[q] = y_new[q]; f[q] = K[6][q]; }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double fl = floor(y[2 * a]);
      turns[a] += fl; y[2 * a] -= fl;
    }
    t = t_new;
    if (!state_ok(y[0], y[1], y[2], y[3], y[4])) { stop = EMRI_ST_STATE; break; }
    if (stop_at_plunge && plunged(oc, y[1], y[3])) { stop = EMRI_ST_PLUNGE; break; }
  }
  *n_out = n;
  return stop;
}

__global__ void __launch_bounds__(32) orbit_dp5_kernel(Dp5Args a) {
  const OrbitArgs& o = a.o;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= o.K) return;
  const double* p = o.params + (size_t)k * EMRI_NPAR;
  double* wc = o.wc + (size_t)k * WC_STRIDE;
  const double Delta = o.S * o.dt;
  int status = 0;
  OrbitConst oc;
  const bool ok = walker_prologue(o, p, wc, oc, status);
  double y0[5] = {frac(p[P_PHI0] / kTwoPi), p[P_NU0], frac(p[P_GAM0] / kTwoPi), p[P_E0], frac(p[P_ALP0] / kTwoPi)};
  if (o.anchor_end) y0[1] = nu_lso(oc.twoPiMs, y0[3]);
  int zero = ok ? 0 : 1;
  int32_t jpl = (int32_t)o.Nn;
  a.nsteps[2 * k] = 0; a.nsteps[2 * k + 1] = 0; a.stop[2 * k] = 0; a.stop[2 * k + 1] = 0;
  a.first_bad[k] = 0x7fffffff;
  if (ok && !o.anchor_end && plunged(oc, y0[1], y0[3])) { status |= EMRI_ST_PLUNGE; jpl = 0; zero = 1; }
  if (!zero) {
    const double ta = o.anchor_end ? (double)o.Nc * Delta : 0.0;
    int32_t n0 = 0, n1 = 0;
    const int s0 = dp5_branch(oc, y0, ta, (double)(o.Nc + 1) * Delta, a.rtol, a.atol, !o.anchor_end, dp5_branch_base(a, k, 0),
                              dp5_branch_cap(a, 0), &n0);
    const int s1 = dp5_branch(oc, y0, ta, -Delta, a.rtol, a.atol, false, dp5_branch_base(a, k, 1), dp5_branch_cap(a, 1), &n1);
    a.nsteps[2 * k] = n0; a.nsteps[2 * k + 1] = n1; a.stop[2 * k] = s0; a.stop[2 * k + 1] = s1;
    // the guard side and the LSO convention must be clean; a forward branch that died before its first step too
    if (s1 || n1 == 0 || (o.anchor_end && s0) || (s0 == EMRI_ST_STATE && n0 == 0)) { status |= EMRI_ST_STATE; zero = 1; }
  }
  wc[WC_EMAX] = 0.0;
  o.jpl[k] = jpl;
  o.status[k] = status;
  a.zero_flag[k] = zero;
}

struct Dp5Pos { const double* rec; int n; double theta; bool ok; };

// position of time tj in a branch of n steps: the first step whose end is not before tj (in the branch's direction)
DEVINL Dp5Pos dp5_locate(const double* __restrict__ rec, int n, double tj) {
  Dp5Pos p{rec, 0, 0.0, false};
  if (n == 0) return p;
  const double dir = (rec[1] >= 0.0) ? 1.0 : -1.0;
  const double* last = rec + (size_t)(n - 1) * DP_REC;
  if (dir * (tj - (last[0] + last[1])) > 0.0) return p;
  int lo = 0, hi = n - 1;                 // smallest i with dir (tj - end_i) <= 0
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    const double* r = rec + (size_t)mid * DP_REC;
    if (dir * (tj - (r[0] + r[1])) > 0.0) lo = mid + 1; else hi = mid;
  }
  const double* r = rec + (size_t)lo * DP_REC;
  p.n = lo; p.theta = (tj - r[0]) / r[1]; p.ok = true;
  return p;
}
DEVINL void dp5_offset(const double* __restrict__ r, double th, double off[5]) {
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const double* Q = r + 12 + 4 * q;
    off[q] = th * (Q[0] + th * (Q[1] + th * (Q[2] + th * Q[3])));
  }
}
// unwrapped change from position a to position b (b not before a in the branch's own order)
DEVINL void dp5_change(const Dp5Pos& a, const Dp5Pos& b, double d[5]) {
  double oa[5], ob[5];
  dp5_offset(a.rec + (size_t)a.n * DP_REC, a.theta, oa);
  dp5_offset(b.rec + (size_t)b.n * DP_REC, b.theta, ob);
  if (a.n == b.n) {
#pragma unroll
    for (int q = 0; q < 5; ++q) d[q] = ob[q] - oa[q];
    return;
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) d[q] = a.rec[(size_t)a.n * DP_REC + 7 + q] - oa[q];
  for (int i = a.n + 1; i < b.n; ++i)
#pragma unroll
    for (int q = 0; q < 5; ++q) d[q] += a.rec[(size_t)i * DP_REC + 7 + q];
#pragma unroll
  for (int q = 0; q < 5; ++q) d[q] += ob[q];
}

__global__ void __launch_bounds__(128) orbit_dp5_nodes_kernel(Dp5Args a) {
  const OrbitArgs& o = a.o;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= o.Nn * o.K) return;
  const int k = (int)(idx / o.Nn);
  const int64_t m = idx - (int64_t)k * o.Nn;
  if (a.zero_flag[k]) return;
  const int64_t j = m - 1, ja = o.anchor_end ? o.Nc : 0;
  const double Delta = o.S * o.dt;
  double* row = o.nodes + ((size_t)k * o.Nn + m) * NODE_STRIDE;
  OrbitConst oc;
  load_orbit_const(o.wc + (size_t)k * WC_STRIDE, oc);
  const bool fwd_side = j >= ja;
  const int br = fwd_side ? 0 : 1;
  const double* rec = dp5_branch_base(a, k, br);
  const int n = a.nsteps[2 * k + br];
  const Dp5Pos p = dp5_locate(rec, n, (double)j * Delta);
  double y[5] = {0, 0, 0, 0, 0}, f[5] = {0, 0, 0, 0, 0}, d[5] = {0, 0, 0, 0, 0};
  int bad = -1;           // -1 usable, 0 plunge, 1 state
  if (!p.ok) {
    bad = (a.stop[2 * k + br] == EMRI_ST_STATE) ? 1 : 0;
  } else {
    double off[5];
    const double* r = rec + (size_t)p.n * DP_REC;
    dp5_offset(r, p.theta, off);
#pragma unroll
    for (int q = 0; q < 5; ++q) y[q] = r[2 + q] + off[q];
    y[0] = frac(y[0]); y[2] = frac(y[2]); y[4] = frac(y[4]);
    if (!state_ok(y[0], y[1], y[2], y[3], y[4])) bad = 1;
    else if (!o.anchor_end && fwd_side && plunged(oc, y[1], y[3])) bad = 0;
  }
  if (bad >= 0) {
    if (fwd_side && !o.anchor_end) atomicMin(a.first_bad + k, (int32_t)(4 * (j + 1) + bad));
    else a.zero_flag[k] = 2;                                  // guard side / LSO convention: the walker is invalid
  } else {
    f[0] = y[1];
    rhs(oc, y[1], y[3], &f[1], &f[2], &f[3], &f[4]);
    // increment over [t_j, t_j+1] (forward time)
    if (fwd_side) {
      if (j < o.Nc + 1) {
        const Dp5Pos pn = dp5_locate(rec, n, (double)(j + 1) * Delta);
        if (pn.ok) dp5_change(p, pn, d);
      }
    } else {
      Dp5Pos pn = (j + 1 == ja) ? Dp5Pos{rec, 0, 0.0, true} : dp5_locate(rec, n, (double)(j + 1) * Delta);
      if (pn.ok) {
        dp5_change(pn, p, d);
#pragma unroll
        for (int q = 0; q < 5; ++q) d[q] = -d[q];
      }
    }
  }
  store_node(row, y, f, d);
}

__global__ void __launch_bounds__(128) orbit_dp5_finish_kernel(Dp5Args a) {
  const OrbitArgs& o = a.o;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= o.Nn * o.K) return;
  const int k = (int)(idx / o.Nn);
  const int64_t m = idx - (int64_t)k * o.Nn;
  double2* row = reinterpret_cast<double2*>(o.nodes + ((size_t)k * o.Nn + m) * NODE_STRIDE);
  const double* wc = o.wc + (size_t)k * WC_STRIDE;
  const int zero = a.zero_flag[k];
  if (zero) {
#pragma unroll
    for (int q = 0; q < NODE_STRIDE / 2; ++q) row[q] = make_double2(0.0, 0.0);
    o.nodeaux[idx] = make_double2(0.0, 0.0);
    if (m == 0 && zero == 2) o.status[k] |= EMRI_ST_STATE;
    return;
  }
  const int32_t fb = a.first_bad[k];
  if (fb != 0x7fffffff) {
    const int64_t jpl = (fb >> 2) - 1;                       // first unusable node
    if (m == 0) { o.jpl[k] = (int32_t)jpl; o.status[k] |= (fb & 1) ? EMRI_ST_STATE : EMRI_ST_PLUNGE; }
    const int64_t j = m - 1;
    if (j >= jpl) {
      // copies of node j_pl - 1 (value and slope), zero increments -- as the fixed-step scheme (reading R8)
      const double2* src = reinterpret_cast<const double2*>(o.nodes + ((size_t)k * o.Nn + jpl) * NODE_STRIDE);   // row of j_pl - 1
      const double2 s0 = src[0], s1 = src[1], s2 = src[2], s3 = src[3], s4 = src[4];
      row[0] = s0; row[1] = s1; row[2] = s2; row[3] = s3; row[4] = s4;
      row[5] = make_double2(0.0, 0.0); row[6] = make_double2(0.0, 0.0); row[7] = make_double2(0.0, 0.0);
      o.nodeaux[idx] = node_aux(wc, s0.y);
      return;
    }
    if (j == jpl - 1) { row[5] = make_double2(0.0, 0.0); row[6] = make_double2(0.0, 0.0); row[7] = make_double2(0.0, 0.0); }
  }
  o.nodeaux[idx] = node_aux(wc, row[0].y);
}

}  // namespace
