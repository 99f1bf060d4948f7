// stretch.cuh -- affine-invariant stretch move on the device (BASELINE.json configs[4])
// Part of the sm_100a implementation of include/emri.h; included by emri.cu (one translation unit).
#pragma once
#include "common.cuh"

namespace {

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

}  // namespace
