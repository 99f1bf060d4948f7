// common.cuh -- constants (S0), layout sizes and small device helpers
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cmath>
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

}  // namespace
