// math64.cuh -- branch-free FP64 elementary functions for the fused re-weighting kernel.
//
// The hot loop is bound by the FP64 pipe, and libdevice's exp/log/division
// carry range checks and slow paths the bounded arguments of this path never take.  These versions
// keep the FP64 instruction count low and move table look-ups and exponent arithmetic to the
// shared-memory and integer pipes.  Polynomial coefficients live in constant memory so that the
// FP64 instructions read them as c[bank][offset] operands (a 64-bit literal would cost two register
// moves per use).  Accuracy (tests/test_gpu_parity.py::test_math_functions, against torch's fp64):
// relative error <= ~4e-16 for rcp/rsqrt, <= 1.6e-13 for exp (cubic on a 256-entry table), absolute <= 1.8e-13 for log
// (quartic on a 128-entry table): the accuracy budget of DESIGN.md section 5, 5000 times inside the 1e-9 parity bar.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gwc {

constexpr double MAGIC52 = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to an integer in the low word

constexpr int LOG_N = 128;   // entries of the log table (top 7 mantissa bits)
constexpr int EXP_N = 256;   // entries of the 2^(j/EXP_N) table
// The tables are replicated so that a look-up with random indices never meets a bank conflict: a 64-bit shared
// load is served half a warp at a time, so 16 copies (lane & 15 picks one, a row of 16 doubles = the 32 banks) make
// every half-warp conflict-free; a 128-bit load is served a quarter warp at a time, so 8 copies of the double2.
constexpr int EXP_REP = 16;
constexpr int LOG_REP = 8;
struct MathTables {
  double2 logtab[LOG_N * LOG_REP];  // [j][lane & 7]:  (1/c_j, ln c_j), c_j = 1 + (j+0.5)/LOG_N     (16 KB)
  double exptab[EXP_N * EXP_REP];   // [j][lane & 15]: 2^(j/EXP_N)                                    (32 KB)
};

// coefficient block (constant bank operands of the DFMAs)
enum : int {
  K_MAGIC = 0,  // 1.5 * 2^52
  K_EXP_K,      // 256 / ln 2
  K_EXP_NL,     // -(ln2/256), rounded to nearest (the product with n is exact inside the fma)
  K_EXP_C3,     // 1/6
  K_LOG_C2,     // 1/3
  K_LN2,
  K_EBIAS,      // 2^52 + 2^31: bias of the int -> double exponent conversion
  K_COUNT
};
static __constant__ double KM[K_COUNT] = {
    6755399441055744.0,
    369.32993046757462707,
    -2.70760617406228627433e-03,
    1.6666666666666666e-01,
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

// 1/x for normal positive x (no zero/inf/denormal handling): MUFU seed (relative error <= 2^-20, measured on
// B200) and one cubic step y (1 + e + e^2), e = 1 - x y: remaining error e^3 < 1e-18, then rounding.
__device__ __forceinline__ double rcp_fast(double x) {
  double y = rcp_seed(x);
  double e = fma(-x, y, 1.0);
  double t = fma(e, e, e);
  return fma(y, t, y);
}

// x^-1/2 for normal positive x: MUFU seed (|1 - a y^2| <= 2^-19, measured) and one cubic step
// y (1 + e/2 + 3 e^2/8), e = 1 - a y^2: remaining error 5 e^3/16 < 3e-18, then rounding.
__device__ __forceinline__ double rsqrt_fast(double a) {
  double y = rsqrt_seed(a);
  double ay = a * y;
  double e = fma(-ay, y, 1.0);
  double t = fma(0.375, e, 0.5) * e;
  return fma(y, t, y);
}

// exp(a) for a in about [-700, 700].  256-entry 2^(j/256) table in shared memory, cubic on |r| <= ln2/512
// (truncation r^4/24 <= 1.4e-13 relative), exponent added with integer arithmetic: 7 FP64 instructions.  The
// reduction uses one constant: n * (ln2/256) is exact inside the fma, and the constant's own rounding moves r by
// n * 2e-19 (<= 5e-14 at |a| = 700).  CLAMP: arguments below -700 (and -inf) return e^-700 (~1e-304); without
// it the caller guarantees the range.
// `exptab` is the calling lane's copy: MathTables::exptab + (lane & 15).
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
  double r = fma(nd, KM[K_EXP_NL], a);
  double T = *reinterpret_cast<const double*>(reinterpret_cast<const char*>(exptab) + ((n << 7) & (8 * EXP_REP * (EXP_N - 1))));
  double p = fma(r, KM[K_EXP_C3], 0.5);
  p = fma(p, r, 1.0);
  double s = T * r;
  double v = fma(s, p, T);
  int hi = (n & ~(EXP_N - 1)) * (1048576 / EXP_N) + __double2hiint(v);  // exponent += n >> 8
  return __hiloint2double(hi, __double2loint(v));
}

// ln(x) for normal positive x.  128-entry (1/c, ln c) table on the top mantissa bits, degree-4 log1p series on
// |r| <= 1/256 (truncation r^5/5 <= 1.8e-13 absolute): 8 FP64 instructions.  `logtab` is the calling lane's copy:
// MathTables::logtab + (lane & 7).
__device__ __forceinline__ double log_fast(double x, const double2* __restrict__ logtab) {
  int hi = __double2hiint(x), lo = __double2loint(x);
  int e = (hi >> 20) - 1023;
  int j = (hi >> 13) & (LOG_N - 1);
  double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
  double2 tc = logtab[j * LOG_REP];
  double r = fma(m, tc.x, -1.0);
  double r2 = r * r;
  double p = fma(r, -0.25, KM[K_LOG_C2]);
  p = fma(p, r, -0.5);
  double l1p = fma(r2, p, r);
  double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - KM[K_EBIAS];  // (double)e
  return fma(ed, KM[K_LN2], tc.y + l1p);
}

// Fill the tables (any block size; caller synchronises before use).
__device__ __forceinline__ void init_math_tables(MathTables& mt, int tid, int nthreads) {
  for (int i = tid; i < LOG_N; i += nthreads) {
    double c = 1.0 + (i + 0.5) * (1.0 / LOG_N);
    double rc = 1.0 / c;
    const double2 v = make_double2(rc, -log(rc));  // -ln(rc): consistent with the rounded reciprocal
#pragma unroll
    for (int r = 0; r < LOG_REP; ++r) mt.logtab[i * LOG_REP + r] = v;
  }
  for (int i = tid; i < EXP_N; i += nthreads) {
    const double v = exp2(i * (1.0 / EXP_N));
#pragma unroll
    for (int r = 0; r < EXP_REP; ++r) mt.exptab[i * EXP_REP + r] = v;
  }
}

}  // namespace gwc
