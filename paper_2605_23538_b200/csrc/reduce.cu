// reduce.cu -- the small kernels around the fused re-weighting kernel:
//   per-sample preparation (theta-independent logs and the per-segment shift), work grouping,
//   A4 (log L_i, N_eff of Eq. 8, n_live), the injection combine (log xi, Eq. 4),
//   A6 (log L = sum_i log L_i - N log xi, Eq. 3), the all-sky mean,
//   and two measurement helpers (FP64 issue-rate probe, accuracy self-test of math64.cuh).
#include <math_constants.h>

#include "gwc_internal.h"
#include "math64.cuh"

namespace gwc {

namespace {

constexpr int PREP_THREADS = 256;

// One CTA per segment.  Pass 1: shift = max_k(-ln pi_k - ln m1z_k) over valid samples.  Pass 2: write
//   dLc = d_L (NaN marks a dead sample), L1 = ln m1z, Q = ln(m2z/m1z), P = -ln pi - ln m1z - shift.
__global__ void __launch_bounds__(PREP_THREADS) prep_kernel(const int64_t* __restrict__ seg_off,
                                                             const double* __restrict__ dL,
                                                             const double* __restrict__ m1z,
                                                             const double* __restrict__ m2z,
                                                             const double* __restrict__ lprior,
                                                             const int32_t* __restrict__ row, int64_t n_rows,
                                                             double* __restrict__ dLc, double* __restrict__ L1,
                                                             double* __restrict__ Q, double* __restrict__ P,
                                                             double* __restrict__ seg_shift) {
  __shared__ double red[PREP_THREADS / 32];
  __shared__ double s_shift;
  const int seg = blockIdx.x, tid = threadIdx.x;
  const int64_t s0 = seg_off[seg], s1 = seg_off[seg + 1];
  double mx = -CUDART_INF;
  for (int64_t k = s0 + tid; k < s1; k += PREP_THREADS) {
    const double d = dL[k], a = m1z[k], b = m2z[k];
    const double lp = lprior ? lprior[k] : 2.0 * log(d);
    bool ok = isfinite(d) && isfinite(a) && isfinite(b) && isfinite(lp) && d > 0.0 && a > 0.0 && b > 0.0 && b <= a;
    if (row) ok = ok && ((unsigned)row[k] < (unsigned)n_rows) && row[k] >= 0;
    if (ok) mx = fmax(mx, -lp - log(a));
  }
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((tid & 31) == 0) red[tid >> 5] = mx;
  __syncthreads();
  if (tid == 0) {
    double m = red[0];
    for (int i = 1; i < PREP_THREADS / 32; ++i) m = fmax(m, red[i]);
    if (!(m > -CUDART_INF)) m = 0.0;  // no valid sample
    s_shift = m;
    seg_shift[seg] = m;
  }
  __syncthreads();
  const double shift = s_shift;
  for (int64_t k = s0 + tid; k < s1; k += PREP_THREADS) {
    const double d = dL[k], a = m1z[k], b = m2z[k];
    const double lp = lprior ? lprior[k] : 2.0 * log(d);
    bool ok = isfinite(d) && isfinite(a) && isfinite(b) && isfinite(lp) && d > 0.0 && a > 0.0 && b > 0.0 && b <= a;
    if (row) ok = ok && ((unsigned)row[k] < (unsigned)n_rows) && row[k] >= 0;
    const double la = ok ? log(a) : 0.0;
    dLc[k] = ok ? d : CUDART_NAN;
    L1[k] = la;
    Q[k] = ok ? log(b / a) : 0.0;
    P[k] = ok ? (-lp - la) - shift : 0.0;
  }
}

// group g = segments whose first sample lies in [g*target, (g+1)*target): binary search per group
__global__ void make_groups_kernel(const int64_t* __restrict__ seg_off, int64_t n_seg, int64_t target, int n_groups,
                                   int32_t* __restrict__ group_off) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g > n_groups) return;
  if (g == n_groups) { group_off[g] = (int32_t)n_seg; return; }
  const int64_t key = (int64_t)g * target;
  int64_t lo = 0, hi = n_seg;  // first segment with seg_off[s] >= key
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (seg_off[mid] < key) lo = mid + 1; else hi = mid;
  }
  group_off[g] = (int32_t)lo;
}

__global__ void uniform_segments_kernel(int64_t n, int64_t seg, int64_t n_seg, int64_t* seg_off) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i > n_seg) return;
  const int64_t v = i * seg;
  seg_off[i] = v < n ? v : n;
}

// longest segment (single block; d_out must hold 0 before the launch)
__global__ void max_segment_kernel(const int64_t* __restrict__ seg_off, int64_t n_seg, int64_t* __restrict__ d_out) {
  long long m = 0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n_seg; i += (int64_t)gridDim.x * blockDim.x) {
    const long long l = seg_off[i + 1] - seg_off[i];
    m = l > m ? l : m;
  }
  atomicMax(reinterpret_cast<long long*>(d_out), m);
}

__global__ void finalize_events_kernel(const double* __restrict__ part_w, const int32_t* __restrict__ part_n,
                                       const int64_t* __restrict__ seg_off, const double* __restrict__ seg_shift,
                                       const double* __restrict__ tvalid, int64_t n_theta, int64_t n_events,
                                       double* __restrict__ logL, double* __restrict__ neff,
                                       int64_t* __restrict__ nlive, int* __restrict__ flag) {
  const int64_t o = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (o >= n_theta * n_events) return;
  const int64_t t = o / n_events, i = o - t * n_events;
  const double valid = tvalid[t];
  const double sw = part_w[2 * o], sw2 = part_w[2 * o + 1];
  const int32_t n = part_n[o];
  const int64_t S = seg_off[i + 1] - seg_off[i];
  double l, ne;
  if (valid != valid) {
    l = CUDART_NAN;
    ne = CUDART_NAN;
  } else if (n > 0 && !(sw >= RANGE_MIN_SUM)) {
    // every live weight lies more than 300 nats below the segment's reference (a log_pe_prior of enormous spread):
    // the linear-domain sums have left their range (gwc.h, "Range"; R23)
    l = CUDART_NAN;
    ne = CUDART_NAN;
    atomicOr(flag, FLAG_RANGE);
  } else if (sw > 0.0) {
    l = (log(sw) + seg_shift[i]) - log((double)S);
    ne = sw * sw / sw2;
  } else {
    l = -CUDART_INF;
    ne = 0.0;
  }
  logL[o] = l;
  if (neff) neff[o] = ne;
  if (nlive) nlive[o] = (valid != valid) ? 0 : (int64_t)n;
}

// one thread per theta: log-sum-exp over the injection segments (each has its own shift), fixed order
__global__ void finalize_inj_kernel(const double* __restrict__ part_w, const int32_t* __restrict__ part_n,
                                    const double* __restrict__ seg_shift, const double* __restrict__ tvalid,
                                    int64_t n_theta, int64_t n_seg, double n_draw, double* __restrict__ logxi,
                                    double* __restrict__ neff, int* __restrict__ flag) {
  // one warp per theta: a lane takes the segments lane, lane + 32, .. in order, then a butterfly (a fixed order: the
  // one-theta calls of a sampler spent a fifth of their time in the serial form of this loop)
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int64_t t = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  if (t >= n_theta) return;   // (whole warps)
  const double valid = tvalid[t];
  if (valid != valid) {
    if (lane == 0) {
      logxi[t] = CUDART_NAN;
      if (neff) neff[t] = CUDART_NAN;
    }
    return;
  }
  const double* pw = part_w + 2 * t * n_seg;
  const int32_t* pn = part_n + t * n_seg;
  // A segment whose live weights all lie below e^-300 of its own reference has left the range of its linear-domain
  // sums (gwc.h, "Range").  Its computed sum is still an UPPER bound of its true sum (weights are clamped from below,
  // never raised above their value), so shift + ln(sum) bounds what it can add to xi.  When that bound lies 60 nats
  // (e^-60 = 9e-27) under the largest in-range segment, the segment is left out: it cannot move log xi or N_eff
  // in the last bit, however many such segments there are.  Otherwise, or with no segment in range, the theta's
  // outputs are NaN and FLAG_RANGE is raised.
  constexpr double NEGLIGIBLE = 60.0;
  double smax = -CUDART_INF;   // largest shift of the in-range segments
  double lin = -CUDART_INF;    // largest ln(segment sum) + shift of the in-range segments
  double lout = -CUDART_INF;   // largest bound of an out-of-range live segment
  for (int64_t s = lane; s < n_seg; s += 32) {
    const double w = pw[2 * s];
    if (w >= RANGE_MIN_SUM) {
      smax = fmax(smax, seg_shift[s]);
      lin = fmax(lin, seg_shift[s] + log(w));
    } else if (pn[s] > 0) {
      lout = fmax(lout, seg_shift[s] + (w > 0.0 ? log(w) : -690.0));
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    smax = fmax(smax, __shfl_xor_sync(FULL, smax, o));
    lin = fmax(lin, __shfl_xor_sync(FULL, lin, o));
    lout = fmax(lout, __shfl_xor_sync(FULL, lout, o));
  }
  if (lout > -CUDART_INF && !(lout <= lin - NEGLIGIBLE)) {  // (lin = -inf: no segment in range)
    if (lane == 0) {
      logxi[t] = CUDART_NAN;
      if (neff) neff[t] = CUDART_NAN;
      atomicOr(flag, FLAG_RANGE);
    }
    return;
  }
  if (!(smax > -CUDART_INF)) {
    if (lane == 0) {
      logxi[t] = -CUDART_INF;
      if (neff) neff[t] = 0.0;
    }
    return;
  }
  double a = 0.0, b = 0.0;
  for (int64_t s = lane; s < n_seg; s += 32) {
    if (!(pw[2 * s] >= RANGE_MIN_SUM)) continue;   // no live injection, or left out as negligible (above)
    const double e = exp(seg_shift[s] - smax);
    a = fma(pw[2 * s], e, a);
    b = fma(pw[2 * s + 1], e * e, b);
  }
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(FULL, a, o);
    b += __shfl_xor_sync(FULL, b, o);
  }
  if (lane == 0) {
    logxi[t] = (log(a) + smax) - log(n_draw);
    if (neff) neff[t] = a * a / b;
  }
}

constexpr int TOT_THREADS = 128;
// one CTA per theta: strided partial sums, fixed-order tree
__global__ void __launch_bounds__(TOT_THREADS) combine_total_kernel(const double* __restrict__ logL,
                                                                     const double* __restrict__ logxi,
                                                                     int64_t n_events, double* __restrict__ total) {
  __shared__ double red[TOT_THREADS];
  const int64_t t = blockIdx.x;
  const int tid = threadIdx.x;
  double s = 0.0;
  for (int64_t i = tid; i < n_events; i += TOT_THREADS) s += logL[t * n_events + i];
  red[tid] = s;
  __syncthreads();
  for (int o = TOT_THREADS / 2; o > 0; o >>= 1) {
    if (tid < o) red[tid] += red[tid + o];
    __syncthreads();
  }
  if (tid == 0) {
    const double sum = red[0], x = logxi[t];
    double r;
    if (sum != sum || x != x) r = CUDART_NAN;
    else if (sum == -CUDART_INF || x == -CUDART_INF) r = -CUDART_INF;
    else r = sum - (double)n_events * x;
    total[t] = r;
  }
}

// ---- event / injection sharding: the pieces of R ranks -> log L(theta), in rank order ----
// One theta.  S_r = sum of log L_i over rank r's events, x_r = log xi_r and N_r = N_eff,r over rank r's injections
// (computed with the GLOBAL n_draw, so xi = sum_r xi_r; with S1_r = xi_r and S2_r = xi_r^2 / N_r the effective
// number of the whole set is (sum S1)^2 / sum S2).  NaN in any piece -> NaN; -inf stays -inf, never NaN.
__host__ __device__ inline void combine_sharded_one(const double* sum_parts, const double* logxi_parts,
                                                    const double* neff_parts, int n_parts, int64_t stride,
                                                    double n_events_total, double* total, double* logxi, double* neff) {
  const double INF = 1.0 / 0.0;
  double S = 0.0, m = -INF;
  bool nan = false;
  for (int r = 0; r < n_parts; ++r) {
    const double sr = sum_parts[r * stride], xr = logxi_parts[r * stride];
    nan = nan || sr != sr || xr != xr;
    S += sr;
    m = xr > m ? xr : m;
  }
  double lx, ne;
  if (nan) {
    lx = ne = S = INF - INF;
  } else if (!(m > -INF)) {
    lx = -INF;
    ne = 0.0;
  } else {
    double s1 = 0.0, s2 = 0.0;
    for (int r = 0; r < n_parts; ++r) {
      const double e = exp(logxi_parts[r * stride] - m);   // xi_r relative to the largest piece (0 for -inf)
      const double nr = neff_parts ? neff_parts[r * stride] : 0.0;
      s1 += e;
      if (nr > 0.0) s2 += e * e / nr;
    }
    lx = m + log(s1);
    ne = s2 > 0.0 ? s1 * s1 / s2 : 0.0;
  }
  double tot;
  if (nan) tot = INF - INF;
  else if (S == -INF || lx == -INF) tot = -INF;
  else tot = S - n_events_total * lx;
  if (total) *total = tot;
  if (logxi) *logxi = lx;
  if (neff) *neff = ne;
}
__global__ void combine_sharded_kernel(const double* __restrict__ sum_parts, const double* __restrict__ logxi_parts,
                                       const double* __restrict__ neff_parts, int n_parts, int64_t n_theta,
                                       double n_events_total, double* __restrict__ total, double* __restrict__ logxi,
                                       double* __restrict__ neff) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= n_theta) return;
  combine_sharded_one(sum_parts + t, logxi_parts + t, neff_parts ? neff_parts + t : nullptr, n_parts, n_theta,
                      n_events_total, total ? total + t : nullptr, logxi ? logxi + t : nullptr,
                      neff ? neff + t : nullptr);
}

constexpr int AS_ROWS = 512;  // rows per partial block of the all-sky mean
template <typename LosT>
__global__ void allsky_partial_kernel(const LosT* __restrict__ table, int64_t n_rows, int n_z,
                                      double* __restrict__ scratch) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_z) return;
  const int64_t r0 = (int64_t)blockIdx.y * AS_ROWS, r1 = min(n_rows, r0 + AS_ROWS);
  double s = 0.0;
  for (int64_t r = r0; r < r1; ++r) s += (double)table[r * n_z + b];
  scratch[(int64_t)blockIdx.y * n_z + b] = s;
}
__global__ void allsky_final_kernel(const double* __restrict__ scratch, int64_t n_parts, int64_t n_rows, int n_z,
                                    double* __restrict__ allsky) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_z) return;
  double s = 0.0;
  for (int64_t p = 0; p < n_parts; ++p) s += scratch[p * n_z + b];
  allsky[b] = s / (double)n_rows;
}

constexpr int PROBE_THREADS = 512;
constexpr int PROBE_CHAINS = 8;
__global__ void __launch_bounds__(PROBE_THREADS) probe_fp64_kernel(int64_t iters, double* sink) {
  double a[PROBE_CHAINS];
  const double m = 1.0 + 1e-9 * threadIdx.x, c = 1e-12 * blockIdx.x;
#pragma unroll
  for (int i = 0; i < PROBE_CHAINS; ++i) a[i] = 0.5 + i;
  for (int64_t it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < PROBE_CHAINS; ++i) a[i] = fma(a[i], m, c);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < PROBE_CHAINS; ++i) s += a[i];
  if (s == 12345.678) sink[0] = s;  // keeps the chains alive
}

__global__ void math_selftest_kernel(int which, int64_t n, const double* __restrict__ in, double* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char selftest_smem[];
  MathTables& mt = *reinterpret_cast<MathTables*>(selftest_smem);
  init_math_tables(mt, threadIdx.x, blockDim.x);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = in[i];
  double y;
  switch (which) {
    case 0: y = exp_fast<true>(x, mt.exptab + (lane & (EXP_REP - 1))); break;
    case 1: y = log_fast(x, mt.logtab + (lane & (LOG_REP - 1))); break;
    case 2: y = rcp_fast(x); break;
    case 3: y = rsqrt_fast(x); break;
    default: y = exp_fast<false>(x, mt.exptab + (lane & (EXP_REP - 1))); break;
  }
  out[i] = y;
}

// int32 counts [n_theta][n] -> int64 (0 for a theta outside the domain)
__global__ void widen_i32_kernel(const int32_t* __restrict__ in, const double* __restrict__ tvalid, int64_t n_theta,
                                 int64_t n, int64_t* __restrict__ out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n_theta * n) return;
  const int64_t t = i / n;
  out[i] = tvalid[t] == 1.0 ? (int64_t)in[i] : 0;
}

inline int ok() { return cudaGetLastError() == cudaSuccess ? 1 : -1; }

}  // namespace

int launch_prep_samples(int64_t n, int64_t n_seg, const int64_t* seg_off, const double* dL, const double* m1z,
                        const double* m2z, const double* lprior, const int32_t* row, int64_t n_rows, double* dLc,
                        double* L1, double* Q, double* P, double* seg_shift, cudaStream_t s) {
  (void)n;
  if (n_seg <= 0) return 0;
  prep_kernel<<<(unsigned)n_seg, PREP_THREADS, 0, s>>>(seg_off, dL, m1z, m2z, lprior, row, n_rows, dLc, L1, Q, P,
                                                       seg_shift);
  return ok();
}

// Heaviest group first (longest-processing-time order of the work items): order[rank] = group, rank = the number of
// groups with more samples (ties in group order, so equal groups keep the group-major order that keeps a group's LOS
// rows in L2).  Catalogues whose groups are all within 25 % of the mean are left in catalogue order; a ragged one no
// longer ends a launch on its heaviest items.
__global__ void __launch_bounds__(256) order_groups_kernel(const int64_t* __restrict__ seg_off,
                                                           const int32_t* __restrict__ group_off, int n_groups,
                                                           int32_t* __restrict__ order) {
  extern __shared__ int64_t s_w[];   // every group's samples (each CTA loads them all; n_groups <= 8192)
  for (int h = threadIdx.x; h < n_groups; h += blockDim.x) s_w[h] = seg_off[group_off[h + 1]] - seg_off[group_off[h]];
  __syncthreads();
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n_groups) return;
  const int64_t w = s_w[g];
  int rank = 0;
  int64_t wmax = 0;
  for (int h = 0; h < n_groups; ++h) {
    const int64_t wh = s_w[h];
    rank += (wh > w || (wh == w && h < g)) ? 1 : 0;
    wmax = wh > wmax ? wh : wmax;
  }
  // (groups that are all about the same size stay in catalogue order)
  const int64_t n = seg_off[group_off[n_groups]] - seg_off[group_off[0]];
  const bool ragged = wmax * 4 * n_groups > 5 * n;   // heaviest group > 1.25 x the mean
  order[ragged ? rank : g] = g;
}
__global__ void identity_order_kernel(int n_groups, int32_t* __restrict__ order) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g < n_groups) order[g] = g;
}

// group_off [n_groups + 1], group_order [n_groups]; uniform = segments of equal length (the injections): no ordering
int launch_make_groups(const int64_t* seg_off, int64_t n_seg, int64_t target, int n_groups, int32_t* group_off,
                       int32_t* group_order, bool uniform, cudaStream_t s) {
  make_groups_kernel<<<(n_groups + 1 + 127) / 128, 128, 0, s>>>(seg_off, n_seg, target, n_groups, group_off);
  if (!uniform && n_groups <= 8192) {
    cudaFuncSetAttribute(order_groups_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 8);   // (per device)
    order_groups_kernel<<<(n_groups + 255) / 256, 256, (size_t)n_groups * sizeof(int64_t), s>>>(seg_off, group_off, n_groups,
                                                                                             group_order);
  } else {
    identity_order_kernel<<<(n_groups + 127) / 128, 128, 0, s>>>(n_groups, group_order);
  }
  return cudaGetLastError() == cudaSuccess ? 2 : -1;
}

int launch_max_segment(const int64_t* seg_off, int64_t n_seg, int64_t* d_out, cudaStream_t s) {
  if (cudaMemsetAsync(d_out, 0, sizeof(int64_t), s) != cudaSuccess) return -1;
  if (n_seg <= 0) return 0;
  int64_t blocks = (n_seg + 255) / 256;
  if (blocks > 1024) blocks = 1024;
  max_segment_kernel<<<(unsigned)blocks, 256, 0, s>>>(seg_off, n_seg, d_out);
  return ok();
}

int launch_uniform_segments(int64_t n, int64_t seg, int64_t n_seg, int64_t* seg_off, cudaStream_t s) {
  uniform_segments_kernel<<<(unsigned)((n_seg + 1 + 127) / 128), 128, 0, s>>>(n, seg, n_seg, seg_off);
  return ok();
}

int launch_finalize_events(const double* part_w, const int32_t* part_n, const int64_t* seg_off, const double* seg_shift,
                           const double* tvalid, int64_t n_theta, int64_t n_events, double* logL,
                           double* neff, int64_t* nlive, int* d_flag, cudaStream_t s) {
  const int64_t n = n_theta * n_events;
  if (n <= 0) return 0;
  finalize_events_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(part_w, part_n, seg_off, seg_shift, tvalid,
                                                                     n_theta, n_events, logL, neff, nlive, d_flag);
  return ok();
}

int launch_finalize_inj(const double* part_w, const int32_t* part_n, const double* seg_shift, const double* tvalid,
                        int64_t n_theta, int64_t n_seg, double n_draw, double* logxi, double* neff, int* d_flag,
                        cudaStream_t s) {
  if (n_theta <= 0) return 0;
  finalize_inj_kernel<<<(unsigned)((n_theta * 32 + 127) / 128), 128, 0, s>>>(part_w, part_n, seg_shift, tvalid, n_theta,
                                                                        n_seg, n_draw, logxi, neff, d_flag);
  return ok();
}

int launch_widen_i32(const int32_t* in, const double* tvalid, int64_t n_theta, int64_t n, int64_t* out,
                     cudaStream_t s) {
  const int64_t m = n_theta * n;
  if (m <= 0) return 0;
  widen_i32_kernel<<<(unsigned)((m + 255) / 256), 256, 0, s>>>(in, tvalid, n_theta, n, out);
  return ok();
}

int launch_combine_total(const double* logL, const double* logxi, int64_t n_theta, int64_t n_events, double* total,
                         cudaStream_t s) {
  if (n_theta <= 0) return 0;
  combine_total_kernel<<<(unsigned)n_theta, TOT_THREADS, 0, s>>>(logL, logxi, n_events, total);
  return ok();
}

int launch_combine_sharded(const double* sum_parts, const double* logxi_parts, const double* neff_parts, int n_parts,
                           int64_t n_theta, int64_t n_events_total, double* total, double* logxi, double* neff,
                           cudaStream_t s) {
  if (n_theta <= 0) return 0;
  combine_sharded_kernel<<<(unsigned)((n_theta + 127) / 128), 128, 0, s>>>(sum_parts, logxi_parts, neff_parts, n_parts,
                                                                          n_theta, (double)n_events_total, total, logxi,
                                                                          neff);
  return ok();
}
void combine_sharded_host(const double* sum_parts, const double* logxi_parts, const double* neff_parts, int n_parts,
                          int64_t n_theta, int64_t n_events_total, double* total, double* logxi, double* neff) {
  for (int64_t t = 0; t < n_theta; ++t)
    combine_sharded_one(sum_parts + t, logxi_parts + t, neff_parts ? neff_parts + t : nullptr, n_parts, n_theta,
                        (double)n_events_total, total ? total + t : nullptr, logxi ? logxi + t : nullptr,
                        neff ? neff + t : nullptr);
}

size_t allsky_scratch_doubles(int64_t n_rows, int n_z) {
  return (size_t)((n_rows + AS_ROWS - 1) / AS_ROWS) * (size_t)n_z;
}

int launch_allsky(const void* table, gwc_prec prec, int64_t n_rows, int n_z, double* scratch, double* allsky,
                  cudaStream_t s) {
  const int64_t n_parts = (n_rows + AS_ROWS - 1) / AS_ROWS;
  dim3 grid((n_z + 127) / 128, (unsigned)n_parts);
  if (prec == GWC_F64)
    allsky_partial_kernel<double><<<grid, 128, 0, s>>>((const double*)table, n_rows, n_z, scratch);
  else
    allsky_partial_kernel<float><<<grid, 128, 0, s>>>((const float*)table, n_rows, n_z, scratch);
  if (ok() < 0) return -1;
  allsky_final_kernel<<<(n_z + 127) / 128, 128, 0, s>>>(scratch, n_parts, n_rows, n_z, allsky);
  return ok() < 0 ? -1 : 2;
}

int launch_probe_fp64(int64_t iters, int n_blocks, double* d_sink, cudaStream_t s, double* n_instr) {
  probe_fp64_kernel<<<n_blocks, PROBE_THREADS, 0, s>>>(iters, d_sink);
  *n_instr = (double)iters * 8.0 * PROBE_CHAINS * PROBE_THREADS * (double)n_blocks;
  return ok();
}

int launch_math_selftest(int which, int64_t n, const double* d_in, double* d_out, cudaStream_t s) {
  if (n <= 0) return 0;
  if (cudaFuncSetAttribute(math_selftest_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(MathTables)) !=
      cudaSuccess)
    return -1;
  math_selftest_kernel<<<(unsigned)((n + 255) / 256), 256, sizeof(MathTables), s>>>(which, n, d_in, d_out);
  return ok();
}

}  // namespace gwc
