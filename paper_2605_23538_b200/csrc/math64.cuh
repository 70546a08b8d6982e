// math64.cuh -- branch-free FP64 elementary functions for the fused re-weighting kernel.
//
// The hot loop is bound by the FP64 pipe, and libdevice's exp/log/division
// carry range checks and slow paths the bounded arguments of this path never take.  These versions
// keep the FP64 instruction count low and move table look-ups and exponent arithmetic to the
// shared-memory and integer pipes.  Polynomial coefficients live in constant memory so that the
// FP64 instructions read them as c[bank][offset] operands (a 64-bit literal would cost two register
// moves per use).  Accuracy (tests/test_gpu_parity.py::test_math_functions, against torch's fp64):
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

// coefficient block (constant bank operands of the DFMAs)
enum : int {
  K_MAGIC = 0,  // 1.5 * 2^52
  K_EXP_K,      // 32 / ln 2
  K_EXP_NLHI,   // -(ln2/32 rounded)
  K_EXP_NLLO,   // -(ln2/32 - hi)
  K_EXP_C5,     // 1/120
  K_EXP_C4,     // 1/24
  K_EXP_C3,     // 1/6
  K_LOG_C5,     // -1/6
  K_LOG_C4,     // 1/5
  K_LOG_C2,     // 1/3
  K_LN2,
  K_EBIAS,      // 2^52 + 2^31: bias of the int -> double exponent conversion
  K_COUNT
};
static __constant__ double KM[K_COUNT] = {
    6755399441055744.0,
    46.166241308446828384,
    -2.16608493924982901946e-02,
    -7.24702129326968612006e-19,
    8.3333333333333332e-03,
    4.1666666666666664e-02,
    1.6666666666666666e-01,
    -1.6666666666666666e-01,
    0.2,
    3.3333333333333331e-01,
    6.93147180559945286227e-01,
    4503601774854144.0,
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
  if (CLAMP) {
    // a = max(a, -700) on the integer pipe: for negative doubles the high word grows with the magnitude
    // (-700.0 = 0xC085E000'00000000); also maps -inf to -700
    const int ahi = __double2hiint(a);
    const bool low = (unsigned)ahi > 0xC085E000u;
    a = __hiloint2double(low ? (int)0xC085E000u : ahi, low ? 0 : __double2loint(a));
  }
  double t = fma(a, KM[K_EXP_K], KM[K_MAGIC]);
  int n = __double2loint(t);
  double nd = t - KM[K_MAGIC];
  double r = fma(nd, KM[K_EXP_NLHI], a);
  r = fma(nd, KM[K_EXP_NLLO], r);
  double T = *reinterpret_cast<const double*>(reinterpret_cast<const char*>(exptab) + ((n << 3) & 0xf8));
  double p = fma(r, KM[K_EXP_C5], KM[K_EXP_C4]);
  p = fma(p, r, KM[K_EXP_C3]);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  double s = T * r;
  double v = fma(s, p, T);
  int hi = (n & ~31) * 32768 + __double2hiint(v);  // exponent += n >> 5
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
  double p = fma(r, KM[K_LOG_C5], KM[K_LOG_C4]);
  p = fma(p, r, -0.25);
  p = fma(p, r, KM[K_LOG_C2]);
  p = fma(p, r, -0.5);
  double l1p = fma(r2, p, r);
  double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - KM[K_EBIAS];  // (double)e
  return fma(ed, KM[K_LN2], tc.y + l1p);
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
