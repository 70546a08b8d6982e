// math64.cuh -- branch-free FP64 elementary functions for the fused re-weighting kernel.
//
// The hot loop is bound by the FP64 pipe, and libdevice's exp/log/division
// carry range checks and slow paths the bounded arguments of this path never take.  These versions
// keep the FP64 instruction count low and move table look-ups and exponent arithmetic to the
// shared-memory and integer pipes.  Accuracy (measured by tests/test_gpu_math.py against libdevice):
// relative error <= ~4e-16 for rcp/rsqrt, <= ~3e-15 for exp, absolute <= ~4e-16 for log on [1, 2^k).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gwc {

constexpr double MAGIC52 = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to an integer in the low word

struct MathTables {
  double2 logtab[64];  // (1/c_j, ln c_j), c_j = 1 + (j+0.5)/64
  double exptab[32];   // 2^(j/32)
};

__device__ __forceinline__ double rcp_seed(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
__device__ __forceinline__ double rsqrt_seed(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}

// 1/x for normal positive x (no zero/inf/denormal handling): MUFU seed, one cubic + one quadratic Newton step.
__device__ __forceinline__ double rcp_fast(double x) {
  double y = rcp_seed(x);
  double e = fma(-x, y, 1.0);
  double t = fma(e, e, e);
  y = fma(y, t, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}

// x^-1/2 for normal positive x: MUFU seed, two Newton steps (second-order in e with the 3/8 e^2 term).
__device__ __forceinline__ double rsqrt_fast(double a) {
  double y = rsqrt_seed(a);
  double ay = a * y;
  double e = fma(-ay, y, 1.0);               // 1 - a y^2
  double t = fma(0.375, e, 0.5) * e;         // e/2 + 3 e^2 / 8
  y = fma(y, t, y);
  ay = a * y;
  e = fma(-ay, y, 1.0);
  return fma(y, 0.5 * e, y);
}

// exp(a) for a in about [-700, 700].  32-entry 2^(j/32) table in shared memory, degree-5 polynomial on
// |r| <= ln2/64, exponent added with integer arithmetic.  CLAMP: arguments below -700 (and -inf) return
// e^-700 (~1e-304); without it the caller guarantees the range.
template <bool CLAMP>
__device__ __forceinline__ double exp_fast(double a, const double* __restrict__ exptab) {
  if (CLAMP) a = fmax(a, -700.0);
  const double K = 46.166241308446828384;          // 32 / ln 2
  const double L_HI = 2.16608493924982901946e-02;  // ln2/32 (rounded)
  const double L_LO = 7.24702129326968612006e-19;  // ln2/32 - L_HI
  double t = fma(a, K, MAGIC52);
  int n = __double2loint(t);
  double nd = t - MAGIC52;
  double r = fma(nd, -L_HI, a);
  r = fma(nd, -L_LO, r);
  double T = exptab[n & 31];
  double p = fma(r, 8.3333333333333332e-03, 4.1666666666666664e-02);
  p = fma(p, r, 1.6666666666666666e-01);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  double s = T * r;
  double v = fma(s, p, T);
  int hi = __double2hiint(v) + ((n >> 5) << 20);
  return __hiloint2double(hi, __double2loint(v));
}

// ln(x) for normal positive x.  64-entry (1/c, ln c) table on the top mantissa bits, degree-6 log1p series.
__device__ __forceinline__ double log_fast(double x, const double2* __restrict__ logtab) {
  int hi = __double2hiint(x), lo = __double2loint(x);
  int e = (hi >> 20) - 1023;
  int j = (hi >> 14) & 63;
  double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
  double2 tc = logtab[j];
  double r = fma(m, tc.x, -1.0);
  double r2 = r * r;
  double p = fma(r, -1.6666666666666666e-01, 0.2);
  p = fma(p, r, -0.25);
  p = fma(p, r, 3.3333333333333331e-01);
  p = fma(p, r, -0.5);
  double l1p = fma(r2, p, r);
  double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - 4503601774854144.0;  // (double)e, 2^52 + 2^31
  return fma(ed, 6.93147180559945286227e-01, tc.y + l1p);
}

// Fill the tables (any block size >= 96 threads; caller synchronises before use).
__device__ __forceinline__ void init_math_tables(MathTables& mt, int tid) {
  if (tid < 64) {
    double c = 1.0 + (tid + 0.5) * (1.0 / 64.0);
    double rc = 1.0 / c;
    mt.logtab[tid] = make_double2(rc, -log(rc));  // -ln(rc): consistent with the rounded reciprocal
  } else if (tid < 96) {
    mt.exptab[tid - 64] = exp2((tid - 64) * (1.0 / 32.0));
  }
}

}  // namespace gwc
