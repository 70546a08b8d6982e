// kde.cu -- NEXT row 1: the paper's own numerator, a kernel density estimate in redshift per sky
// pixel (Eq. 5-7; bandwidth Eq. D1; 256-node grid).
//
// For pixel j of event i (a maximal run of equal sample_row, R25) and one theta (readings R26-R30):
//   v_k  = p(m1, m2 | theta) / (J pi_PE)        Eq. 7's weight without the redshift prior
//   h_j  = 1.06 sigma_j n_j^(-1/5)              sigma_j: v-weighted standard deviation of the z_k, n_j: live samples
//   f_j(z) = sum_k v_k N(z; z_k, h_j)            Eq. 6
//   I_j  = trapezoid over the G-node grid on [0, z_max] of f_j(z) p_los(z | row_j) psi(z)/(1+z)
//   L_i  = (1/S_i) sum_j I_j   over the pixels with n_j >= 2, sigma_j > 0, N_eff,j >= neff_min (Eq. 8)
//
// Mapping (round 2).  Work units are (chunk, theta), chunk-major, handed to the resident warps
// of a persistent grid: a chunk is a run of whole pixels of one event of about KDE_CHUNK = 1024 samples (the table is
// theta-independent, built per call by the kde_chunk_* kernels), so long events spread over many warps and a warp's
// scratch slice stays L2-resident.  Per-theta values and the prior weights on the grid are computed once per call by
// kde_theta_prep_kernel.  A warp first computes (z_k, v_k) of its chunk, 32 samples at a time with every lane busy,
// into its scratch slice; then it takes the chunk 32 samples at a time whatever the pixel boundaries: segmented warp
// scans give sum v, sum v d, sum v d^2, sum v^2 (d = z minus the pixel's first live redshift: the shifted one-pass
// variance) at every pixel's last sample, a run left open by one row is carried to the next, and the pixels that pass
// (n >= 2, variance > 0, N_eff) go through the KDE one after the other.  The KDE pass factorises the Gaussian on the
// uniform grid: a half-warp lane covers 16 consecutive nodes around a centre c, and with q_c = (z_c - z_k)/(h sqrt 2),
// beta = dz/(h sqrt 2) the value at node c + o is E P^o C_o, E = exp(-q_c^2), P = exp(-2 beta q_c),
// C_o = exp(-o^2 beta^2): two exponentials and one reciprocal per (sample, lane) give 16 Gaussians; the two half-warps
// take alternate samples, two samples per step.  Pixels whose bandwidth is below half a grid step take a direct path
// (one exponential per node).  The per-chunk partial sums (relative to e^shift of the event) are combined in chunk
// order by kde_combine_kernel.  Everything is FP64, with math64.cuh's exp / ln / rcp / rsqrt; all sums run in a fixed
// order (bitwise reproducible).  Measured: 4.81 FP64 instructions per Gaussian evaluation (profiles/r02f).
#include <math_constants.h>

#include "gwc_internal.h"
#include "math64.cuh"

namespace gwc {

namespace {

constexpr int KDE_THREADS = 256;
constexpr int KDE_WARPS = KDE_THREADS / 32;
constexpr int KDE_NPL = 8;            // grid nodes per lane: G <= 256
constexpr double KDE_BETA_MAX = 1.5;  // fast path of the KDE pass: grid step <= 1.5 h sqrt(2)
constexpr double C_KMS_KDE = 299792.458;

struct KdeParams {
  int model;                // gwc_mass_model
  const Node64* ftab;       // MULTIPEAK: [n_theta][MF_PITCH] table of |F|(m1) over the smoothing window
  const double* theta;      // [n_theta][npar]: the copy gwc_build_cosmo took (the tables belong to it)
  const void* tab;          // [n_theta][Mp] Node64 | Node32
  const double* tconst;     // [n_theta][nconst_of(model)] (umax, 1/du; MULTIPEAK: N1, C(top), n_g,low)
  const double* tvalid;     // [n_theta] 1.0, or NaN: outside the domain / changed since the build
  int64_t n_theta, n_events;
  int M, Mp;
  double tab_zq;
  const int64_t* ev_off;    // [n_events+1]
  const double *dL, *m1z, *m2z, *lprior;   // lprior may be NULL (2 ln d_L)
  const int32_t* row;
  const double* seg_shift;  // [n_events] reference of the linear-domain sums (prep_kernel)
  const void* los;          // [n_rows][n_z]
  int64_t n_rows;
  int n_z;
  double los_zmax;
  int n_grid;
  double neff_min;
  int bw_rule;              // gwc_bw_rule: Scott (D1), Silverman (D2), biweight as printed (D3), biweight in Scott's rule
  double2* scr;             // [resident warps][scr_stride]: (z_k, v_k) of the event a warp is working on (v < 0: dead)
  int64_t scr_stride;       // >= the longest event
  double* logL;             // [n_theta][n_events]
  int64_t* npass;           // [n_theta][n_events] or NULL
  int64_t* nused;           // [n_theta][n_events] or NULL: live samples of the contributing pixels
  int* flag;                // sticky device flag word (written by -DGWC_CHECKED builds only)
  // Work units are (chunk, theta): a chunk is a run of whole pixels of one event, about KDE_CHUNK samples long
  // (theta-independent; kde_chunk_* kernels).  Chunks keep the (z, v) scratch slice of a warp small enough to stay in
  // L2 and split the long events of a ragged catalogue over many warps.
  const struct ThetaK* thk; // [n_theta] per-theta values (kde_theta_prep_kernel)
  const struct NodeW* gw;   // [n_theta][32 * KDE_NPL] prior weights at the grid nodes
  int64_t n_chunks;
  const int64_t *chunk_start, *chunk_end;   // [n_chunks]
  const int32_t* chunk_event;               // [n_chunks]
  const int64_t* chunk_off;                 // [n_events + 1] chunks of each event
  double* part_e;           // [n_theta][n_chunks] sum of I_j over the chunk's contributing pixels, relative to e^shift
  int32_t* part_np;         // [n_theta][n_chunks] contributing pixels
  int64_t* part_nu;         // [n_theta][n_chunks] their live samples
};

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// per-theta values a warp keeps while it walks an event
struct ThetaK {
  double h0c, umax, invdu, mmin, mmax, alpha, beta, mu, sigma;
  double a_pl, a_g;      // (1 - lambda) n_pl  and  lambda n_g / (sigma sqrt(2 pi))
  double bp1, mminb;     // beta + 1, mmin^(beta+1)
  double Om, OL, cH;     // c / H0
  // MULTIPEAK (R33-R36): a_pl, a_g (the high peak) and a_gl carry 1/N1
  bool mp;
  double a_gl, mul, sigl, dm, fidx, ctop, topb;   // topb = (mmin + dm)^(beta+1)
  const Node64* ftab;
};

__device__ __forceinline__ void node_pair(const Node64* t, int m, double& z0, double& d0, double& z1, double& d1,
                                          double) {
  z0 = t[m].z; d0 = t[m].d; z1 = t[m + 1].z; d1 = t[m + 1].d;
}
__device__ __forceinline__ void node_pair(const Node32* t, int m, double& z0, double& d0, double& z1, double& d1,
                                          double zq) {
  z0 = (double)t[m].zq * zq; d0 = (double)t[m].d * zq; z1 = (double)t[m + 1].zq * zq; d1 = (double)t[m + 1].d * zq;
}

// z_k and v_k of one sample relative to e^shift (v < 0: dead): DESIGN.md section 3 without p_los and the rate term.
// `scale` = exp(-l_pi - shift) (for the default prior exp(-shift) / d_L^2, no logarithm at all).  Powers and the
// Gaussian go through math64.cuh's exp / ln (2e-13), like the fused kernel.
template <typename NodeT, bool MP>
__device__ __forceinline__ double sample_v(const ThetaK& K, const NodeT* tab, int M, double zq, double dL, double m1z,
                                           double m2z, double scale, int32_t row, int64_t n_rows, double los_zmax,
                                           const double2* logtab, const double* exptab, double& z_out) {
  z_out = 0.0;
  if (!(isfinite(dL) && isfinite(m1z) && isfinite(m2z) && isfinite(scale))) return -1.0;
  if (!(dL > 0.0 && m1z > 0.0 && m2z > 0.0)) return -1.0;
  if (row < 0 || (int64_t)row >= n_rows) return -1.0;
  const double u = dL * K.h0c;
  if (!(u < K.umax)) return -1.0;
  const double t = u * K.invdu;
  int m = (int)floor(t);
  m = m > M - 2 ? M - 2 : m;
  const double f = t - (double)m;
  double z0, d0, z1, d1;
  node_pair(tab, m, z0, d0, z1, d1, zq);
  const double dl = z1 - z0, sd = d0 + d1;
  const double c3 = fma(-2.0, dl, sd), c2 = fma(3.0, dl, -(sd + d0));
  const double z = fma(f, fma(f, fma(f, c3, c2), d0), z0);
  if (!(z < los_zmax)) return -1.0;
  const double x = 1.0 + z;
  const double rx = rcp_fast(x);
  const double m1 = m1z * rx, m2 = m2z * rx;
  if (!(m1 > K.mmin && m1 <= K.mmax && m2 >= K.mmin && m2z <= m1z)) return -1.0;
  const double lm1 = log_fast(m1, logtab), lm2 = log_fast(m2 <= m1 ? m2 : m1, logtab);
  const double y = (m1 - K.mu) / K.sigma;
  double p1 = K.a_pl * exp_fast<true>(-K.alpha * lm1, exptab) + K.a_g * exp_fast<true>(-0.5 * y * y, exptab);
  double p2;
  if (MP) {
    // p(m1) p(m2 | m1) = [mix(m1) S(m1) / N1] [m2^beta S(m2) / C(m1)]; inside the smoothing window
    // C(m1) = S(m1) m1^(beta+1) |F|(m1) / |beta+1| from the table (S(m1) cancels), above it elementary
    const double yl = (m1 - K.mul) / K.sigl;
    p1 += K.a_gl * exp_fast<true>(-0.5 * yl * yl, exptab);
    const double m1p = m1 - K.mmin, m2p = m2 - K.mmin;
    double S2 = 1.0;
    if (m2p < K.dm) {
      const double E = K.dm * fma(2.0, m2p, -K.dm) * rcp_fast(m2p * (m2p - K.dm));
      if (!(E <= 250.0)) return -1.0;   // a smoothing factor below e^-250 is zero (R35)
      S2 = 1.0 / (1.0 + exp_fast<true>(E, exptab));
    }
    const double num2 = exp_fast<true>(K.beta * lm2, exptab) * S2;
    const double m1b = exp_fast<true>(K.bp1 * lm1, exptab);
    if (m1p < K.dm) {
      const double t = m1p * K.fidx;
      int k = (int)floor(t);
      k = k < 0 ? 0 : (k > MF_NODES - 2 ? MF_NODES - 2 : k);
      const double f = t - (double)k;
      const Node64 a = K.ftab[k], b = K.ftab[k + 1];
      const double dl = b.z - a.z, sd = a.d + b.d;
      const double c3 = fma(-2.0, dl, sd), c2 = fma(3.0, dl, -(sd + a.d));
      const double F = fma(f, fma(f, fma(f, c3, c2), a.d), a.z);
      p2 = num2 * fabs(K.bp1) / (m1b * F);
    } else {
      p2 = num2 / ((m1b - K.topb) / K.bp1 + K.ctop);
    }
  } else {
    p2 = K.bp1 * exp_fast<true>(K.beta * lm2, exptab) / (exp_fast<true>(K.bp1 * lm1, exptab) - K.mminb);
  }
  if (!(p1 > 0.0) || !(p2 > 0.0) || !(p2 < CUDART_INF)) return -1.0;
  const double rE = rsqrt_fast(fma(K.Om * x * x, x, K.OL));
  const double J = x * x * K.cH * (u * rx + x * rE);
  z_out = z;
  const double v = p1 * p2 * scale / J;
  return v >= 0.0 ? v : -1.0;   // (NaN from a degenerate theta: dead)
}

// ---- order statistics of a pixel's live redshifts (Silverman's rule, Eq. D2; biweight midvariance, Eq. D3-D4) -------
// The value a sample enters the selection with: its redshift, or its absolute deviation from a centre (for the MAD).
struct KeyZ {
  __device__ __forceinline__ double operator()(double z) const { return z; }
};
struct KeyAbsDev {
  double centre;
  __device__ __forceinline__ double operator()(double z) const { return fabs(z - centre); }
};

// k-th smallest (0-based) key of the live samples of scr[r0..r1): bisection on the bit pattern (non-negative doubles
// order like their bits), one counting pass per bit; exact, every lane returns the same value.
template <typename Key>
__device__ double kth_live(const double2* scr, int64_t r0, int64_t r1, int64_t k, Key key, int lane) {
  unsigned long long prefix = 0;
  for (int bit = 62; bit >= 0; --bit) {
    const unsigned long long cand = prefix | (1ull << bit);
    int cnt = 0;
    for (int64_t c0 = r0; c0 < r1; c0 += 32) {
      const int64_t i = c0 + lane;
      if (i < r1) {
        const double2 zv = scr[i];
        cnt += (zv.y >= 0.0 && (unsigned long long)__double_as_longlong(key(zv.x)) < cand) ? 1 : 0;
      }
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if ((int64_t)cnt <= k) prefix = cand;
  }
  return __longlong_as_double((long long)prefix);
}

// the order statistic after x = the k-th one: x again when it is repeated, else the smallest live key above it
template <typename Key>
__device__ double next_live(const double2* scr, int64_t r0, int64_t r1, int64_t k, double x, Key key, int lane) {
  int le = 0;
  double up = CUDART_INF;
  for (int64_t c0 = r0; c0 < r1; c0 += 32) {
    const int64_t i = c0 + lane;
    if (i < r1) {
      const double2 zv = scr[i];
      if (zv.y >= 0.0) {
        const double v = key(zv.x);
        le += v <= x ? 1 : 0;
        up = v > x ? fmin(up, v) : up;
      }
    }
  }
  le = __reduce_add_sync(0xffffffffu, le);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) up = fmin(up, __shfl_xor_sync(0xffffffffu, up, o));
  return (int64_t)le >= k + 2 ? x : up;
}

// q-quantile of the n live keys by linear interpolation between the order statistics at q (n - 1)
template <typename Key>
__device__ double live_quantile(const double2* scr, int64_t r0, int64_t r1, int64_t n, double q, Key key, int lane) {
  const double pos = q * (double)(n - 1);
  const int64_t lo = (int64_t)floor(pos);
  if (lo >= n - 1) return kth_live(scr, r0, r1, n - 1, key, lane);
  const double f = pos - (double)lo;
  const double x0 = kth_live(scr, r0, r1, lo, key, lane);
  const double x1 = next_live(scr, r0, r1, lo, x0, key, lane);
  return __dadd_rn(x0, __dmul_rn(f, x1 - x0));   // (no contraction: the same bits as the plain statement)
}

// Biweight midvariance of the n live redshifts of a pixel, Eq. D3-D4 (R37); NaN when the
// MAD or the denominator is zero.
__device__ double live_biweight(const double2* scr, int64_t r0, int64_t r1, int64_t n, int lane) {
  const double Q = live_quantile(scr, r0, r1, n, 0.5, KeyZ(), lane);
  KeyAbsDev dev;
  dev.centre = Q;
  const double mad = live_quantile(scr, r0, r1, n, 0.5, dev, lane);
  if (!(mad > 0.0)) return CUDART_NAN;
  const double s9 = 9.0 * mad;
  double num = 0.0, den = 0.0;
  for (int64_t c0 = r0; c0 < r1; c0 += 32) {
    const int64_t i = c0 + lane;
    if (i < r1) {
      const double2 zv = scr[i];
      const double d = zv.x - Q, u = d / s9;
      if (zv.y >= 0.0 && fabs(u) < 1.0) {
        const double a = 1.0 - u * u, a2 = a * a;
        num += d * d * a2 * a2;
        den += a * (1.0 - 5.0 * u * u);
      }
    }
  }
  num = wsum(num);
  den = wsum(den);
  return den != 0.0 ? (double)n * num / (den * den) : CUDART_NAN;
}

// Grid node i (< KDE_NPL) of a lane in the prior stage: half-warp lane l16 = lane & 15 owns the 16 consecutive nodes
// 16 l16 .. 16 l16 + 15, of which the lower half-warp keeps the first eight and the upper one the last eight.
__device__ __forceinline__ int kde_node(int lane, int i) { return 16 * (lane & 15) + KDE_NPL * (lane >> 4) + i; }

// The KDE of one pixel on the grid times the prior, Eq. 5-6: returns this lane's share of
// I_j = sum_g c_g R(z_g) p_los(z_g | row) sum_k v_k N(z_g; z_k, h)  (the caller adds the lanes' shares of all pixels
// and reduces once per event).  s_w: per-node prior weights of this theta, [i][lane] pairs (w0, w1) =
// c_g R(z_g) (1 - f_g, f_g) for the two LOS nodes around z_g, g = kde_node(lane, i); s_b: the LOS bin b_g.
struct NodeW { double w0, w1; };
template <typename LosT>
__device__ __forceinline__ double kde_pixel(const double2* __restrict__ scr, int64_t r0, int64_t r1, double h,
                                            int32_t prow, const KdeParams& p, double dzg, const NodeW* s_w,
                                            const int* s_b, const double* exptab, int lane) {
  const unsigned FULL = 0xffffffffu;
  // the LOS nodes this lane needs (8 consecutive grid nodes = a few cache lines of the row) are pulled into L1 now:
  // the latency hides behind the sample loop, and no register is held across it
  const LosT* lrow = reinterpret_cast<const LosT*>(p.los) + (size_t)prow * (size_t)p.n_z;
#pragma unroll
  for (int i = 0; i < KDE_NPL; i += 2) asm volatile("prefetch.global.L1 [%0];" ::"l"(lrow + s_b[i * 32 + lane]));
  asm volatile("prefetch.global.L1 [%0];" ::"l"(lrow + s_b[(KDE_NPL - 1) * 32 + lane] + 1));
  const double invh = rcp_fast(h);
  const double norm = invh * 0.39894228040143267794;   // 1 / (h sqrt(2 pi))
  const double sinvh = invh * 0.70710678118654752440;  // so that the exponent is -(q')^2
  const double beta = dzg * sinvh;   // grid step in units of h sqrt(2)
  const int l16 = lane & 15, up = lane >> 4;
  double mine[KDE_NPL];   // f_j at this lane's eight nodes
  if (beta <= KDE_BETA_MAX) {
    // Fast path (the grid resolves the kernel: h >= dz / 2.1).  The two half-warps take alternate samples; inside a
    // half-warp lane l16 covers the 16 CONSECUTIVE nodes g = 16 l16 + s.  With q_c = (16 l16 + 8) beta - z_k / (h sqrt 2)
    // the exponent at node s is
    //   -(q_c + o beta)^2 = -q_c^2 - 2 o beta q_c - o^2 beta^2,   o = s - 8,
    // so N(z_g; z_k, h) = E P^o C_o with E = exp(-q_c^2), P = exp(-2 beta q_c) and the per-pixel constants
    // C_o = exp(-o^2 beta^2), which leave the sum over samples: two exponentials and a reciprocal per
    // (sample, lane) for 16 Gaussians, the other nodes by multiplication (every intermediate E P^o is a Gaussian
    // value <= 1).  q_c is clamped to +-(12.5 + 8 beta): beyond it every node of the lane is below e^-156 of the
    // sample's own peak, and inside the clamp all arguments stay within the range of exp_fast.
    double acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = 0.0;
    const double qL = (double)(16 * l16 + 8) * beta;
    const int hiQc = __double2hiint(12.5 + 8.0 * beta);   // the clamp compares high words (2^-20 below the limit)
    const double g2 = -2.0 * beta;
    for (int64_t c0 = r0; c0 < r1; c0 += 32) {
      const int64_t k = c0 + lane;
      double zs = 0.0, a = 0.0;   // z_k / (h sqrt 2), v_k / (h sqrt(2 pi))
      if (k < r1) {
        const double2 zv = scr[k];
        a = zv.y >= 0.0 ? zv.y * norm : 0.0;
        zs = zv.x * sinvh;
      }
      const int cnt = (int)min((int64_t)32, r1 - c0);
      auto step = [&](int j) {
        const double zj = __shfl_sync(FULL, zs, j), aj = __shfl_sync(FULL, a, j);
        double qc = qL - zj;
        {
          const int hi = __double2hiint(qc);
          const bool far = (hi & 0x7fffffff) >= hiQc;
          qc = __hiloint2double(far ? ((hi & (int)0x80000000) | hiQc) : hi, far ? 0 : __double2loint(qc));
        }
        const double E = exp_fast<false>(-qc * qc, exptab);
        const double P = exp_fast<false>(g2 * qc, exptab);
        const double Pi = rcp_fast(P);
        const double P2 = P * P, Pi2 = Pi * Pi;
        const double u1 = E * P, u2 = E * P2, u3 = u1 * P2, u4 = u2 * P2, u5 = u3 * P2, u6 = u4 * P2, u7 = u5 * P2;
        const double d1 = E * Pi, d2 = E * Pi2, d3 = d1 * Pi2, d4 = d2 * Pi2, d5 = d3 * Pi2, d6 = d4 * Pi2,
                     d7 = d5 * Pi2, d8 = d6 * Pi2;
        acc[0] = fma(aj, d8, acc[0]);
        acc[1] = fma(aj, d7, acc[1]);
        acc[2] = fma(aj, d6, acc[2]);
        acc[3] = fma(aj, d5, acc[3]);
        acc[4] = fma(aj, d4, acc[4]);
        acc[5] = fma(aj, d3, acc[5]);
        acc[6] = fma(aj, d2, acc[6]);
        acc[7] = fma(aj, d1, acc[7]);
        acc[8] = fma(aj, E, acc[8]);
        acc[9] = fma(aj, u1, acc[9]);
        acc[10] = fma(aj, u2, acc[10]);
        acc[11] = fma(aj, u3, acc[11]);
        acc[12] = fma(aj, u4, acc[12]);
        acc[13] = fma(aj, u5, acc[13]);
        acc[14] = fma(aj, u6, acc[14]);
        acc[15] = fma(aj, u7, acc[15]);
      };
      // two samples per half-warp and step (two independent chains); a slot past the end holds a = 0
      for (int j = up; j - up < cnt; j += 4) {
        step(j);
        step((j + 2) & 31);
      }
    }
    // the halves exchange what the other one keeps; C_o = c1^(o^2), c1 = exp(-beta^2)
    const double c1 = exp_fast<false>(-beta * beta, exptab), cs = c1 * c1;   // (2e-13; its 64th power: 1e-11)
    double C[9];
    C[0] = 1.0;
    double t = c1;
#pragma unroll
    for (int o = 1; o <= 8; ++o) {
      C[o] = C[o - 1] * t;   // c1^(o^2): ratios c1^(2o-1)
      t *= cs;
    }
#pragma unroll
    for (int i = 0; i < KDE_NPL; ++i) {
      const double send = up ? acc[i] : acc[KDE_NPL + i];
      const double keep = up ? acc[KDE_NPL + i] : acc[i];
      mine[i] = (keep + __shfl_xor_sync(FULL, send, 16)) * (up ? C[i] : C[KDE_NPL - i]);
    }
  } else {
    // narrow kernels (h < dz / 2.1, a degenerate pixel): every Gaussian by its own exponential
#pragma unroll
    for (int i = 0; i < KDE_NPL; ++i) mine[i] = 0.0;
    for (int64_t c0 = r0; c0 < r1; c0 += 32) {
      const int64_t k = c0 + lane;
      double zs = 0.0, a = 0.0;
      if (k < r1) {
        const double2 zv = scr[k];
        a = zv.y >= 0.0 ? zv.y * norm : 0.0;
        zs = zv.x * sinvh;
      }
      const int cnt = (int)min((int64_t)32, r1 - c0);
      for (int j = 0; j < cnt; ++j) {
        const double zj = __shfl_sync(FULL, zs, j), aj = __shfl_sync(FULL, a, j);
#pragma unroll
        for (int i = 0; i < KDE_NPL; ++i) {
          const double q = fma((double)kde_node(lane, i), beta, -zj);
          const double g2 = q * q;   // a kernel value below e^-700 is zero (R38)
          mine[i] = fma(g2 > 700.0 ? 0.0 : aj, exp_fast<true>(-g2, exptab), mine[i]);
        }
      }
    }
  }
  // prior at the lane's nodes: p_los(z_g | row) by the table's linear interpolation, times c_g R(z_g)
  double part = 0.0;
#pragma unroll
  for (int i = 0; i < KDE_NPL; ++i) {
    const NodeW w = s_w[i * 32 + lane];
    const int b = s_b[i * 32 + lane];
    GWC_DEV_CHECK(p.flag, b >= 0 && b <= p.n_z - 2 && prow >= 0 && (int64_t)prow < p.n_rows, FLAG_CHK_KDE);
    part = fma(mine[i], fma((double)lrow[b + 1], w.w1, (double)lrow[b] * w.w0), part);
  }
  return part;
}

#ifndef GWC_KDE_CHUNK
#define GWC_KDE_CHUNK 1024
#endif
constexpr int KDE_CHUNK = GWC_KDE_CHUNK;   // target samples per chunk (a pixel is never split)

// ---- chunks: runs of whole pixels of one event, cut at the first pixel start at or after every KDE_CHUNK samples ----
// An event whose offsets do not ascend inside [0, n_samples] gets no chunk (nothing of it is read or written later) and
// raises *bad, which the host turns into GWC_ERR_SHAPE: with every event inside the sample list and disjoint from its
// neighbours the chunk count stays below kde_chunk_bound, the size of the chunk tables.
__global__ void kde_chunk_count_kernel(const int64_t* __restrict__ ev_off, int64_t n_events, int64_t n_samples,
                                       int64_t* __restrict__ cnt, int64_t* __restrict__ bad) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n_events) return;
  const int64_t s0 = ev_off[i], s1 = ev_off[i + 1];
  const bool ok = s0 >= 0 && s0 <= s1 && s1 <= n_samples;
  cnt[i] = ok ? (s1 - s0 + KDE_CHUNK - 1) / KDE_CHUNK : 0;
  if (!ok) *bad = 1;
}
// exclusive scan in order (single CTA); off[n] = total
__global__ void kde_chunk_scan_kernel(const int64_t* __restrict__ cnt, int64_t n, int64_t* __restrict__ off) {
  __shared__ long long part[256];
  __shared__ long long carry;
  const int tid = threadIdx.x;
  if (tid == 0) carry = 0;
  __syncthreads();
  for (int64_t base = 0; base <= n; base += 256) {
    const int64_t i = base + tid;
    part[tid] = i < n ? cnt[i] : 0;
    __syncthreads();
    if (tid == 0) {
      long long run = carry;
      for (int j = 0; j < 256; ++j) {
        const long long v = part[j];
        part[j] = run;
        run += v;
      }
      carry = run;
    }
    __syncthreads();
    if (i <= n) off[i] = part[tid];
    __syncthreads();
  }
}
// first pixel start at or after position k of the event [s0, s1) (s1 when there is none)
__device__ __forceinline__ int64_t next_pixel_start(const int32_t* __restrict__ row, int64_t s0, int64_t s1, int64_t k) {
  if (k <= s0) return s0;
  while (k < s1 && row[k] == row[k - 1]) ++k;
  return k < s1 ? k : s1;
}
__global__ void kde_chunk_bounds_kernel(const int64_t* __restrict__ ev_off, int64_t n_events,
                                        const int64_t* __restrict__ chunk_off, const int32_t* __restrict__ row,
                                        int64_t* __restrict__ c_start, int64_t* __restrict__ c_end,
                                        int32_t* __restrict__ c_event, int64_t* __restrict__ max_len,
                                        int64_t nc_max) {
  const int64_t ev = blockIdx.x;
  const int64_t s0 = ev_off[ev], s1 = ev_off[ev + 1];
  const int64_t c0 = chunk_off[ev], nc = chunk_off[ev + 1] - c0;
  long long mx = 0;
  for (int64_t c = threadIdx.x; c < nc && c0 + c < nc_max; c += blockDim.x) {
    const int64_t a = next_pixel_start(row, s0, s1, s0 + c * KDE_CHUNK);
    const int64_t b = c + 1 < nc ? next_pixel_start(row, s0, s1, s0 + (c + 1) * KDE_CHUNK) : s1;
    c_start[c0 + c] = a;
    c_end[c0 + c] = b;
    c_event[c0 + c] = (int32_t)ev;
    mx = b - a > mx ? b - a : mx;
  }
  if (mx > 0) atomicMax(reinterpret_cast<long long*>(max_len), mx);
}

// ---- per-theta values and prior weights, once per call (one warp per theta) ----
template <bool MP>
__global__ void __launch_bounds__(32) kde_theta_prep_kernel(const KdeParams p, ThetaK* __restrict__ thk,
                                                            NodeW* __restrict__ gw) {
  const int64_t t = blockIdx.x;
  const int lane = threadIdx.x;
  const int G = p.n_grid;
  const double dzg = p.los_zmax / (G - 1);
  const double dzl = p.los_zmax / (p.n_z - 1);
  const double* th = p.theta + t * (MP ? GWC_NPAR_MULTIPEAK : GWC_NPAR);
  const double* tcr = p.tconst + t * nconst_of(MP ? 1 : 0);
  ThetaK K;
  {
    const double H0 = th[0], alpha = th[2], beta = th[3], mmin = th[4], mmax = th[5], mu = th[6], sigma = th[7],
                 lam = th[8];
    K.h0c = H0 / C_KMS_KDE;
    K.cH = C_KMS_KDE / H0;
    K.umax = tcr[C_UMAX];
    K.invdu = tcr[C_INVDU];
    K.mmin = mmin; K.mmax = mmax; K.alpha = alpha; K.beta = beta; K.mu = mu; K.sigma = sigma;
    const double n_pl = (1.0 - alpha) / (pow(mmax, 1.0 - alpha) - pow(mmin, 1.0 - alpha));
    const double rs2 = 1.0 / (sigma * 1.41421356237309504880);
    const double n_g = 1.0 / (0.5 * (erf((mmax - mu) * rs2) - erf((mmin - mu) * rs2)));
    K.a_pl = (1.0 - lam) * n_pl;
    K.a_g = lam * n_g / (sigma * 2.50662827463100050242);
    K.bp1 = beta + 1.0;
    K.mminb = pow(mmin, beta + 1.0);
    K.Om = th[1];
    K.OL = 1.0 - th[1];
    K.mp = MP;
    K.a_gl = 0.0; K.mul = 0.0; K.sigl = 1.0; K.dm = 0.0; K.fidx = 0.0; K.ctop = 0.0; K.topb = K.mminb; K.ftab = nullptr;
    if (MP) {
      const double dm = th[12], laml = th[15], iN1 = 1.0 / tcr[C_N1];
      K.a_pl *= iN1;
      K.a_g *= (1.0 - laml) * iN1;
      K.a_gl = lam * laml * tcr[C_NGL] / (th[14] * 2.50662827463100050242) * iN1;
      K.mul = th[13]; K.sigl = th[14]; K.dm = dm; K.fidx = tcr[C_FIDX]; K.ctop = tcr[C_CTOP];
      K.topb = pow(mmin + dm, beta + 1.0);
      K.ftab = p.ftab + (size_t)t * MF_PITCH;
    }
  }
  if (lane == 0) thk[t] = K;
  // prior weights at the grid nodes: c_g psi(z_g) / (1 + z_g) (trapezoid weight, reading R4) split over the two LOS
  // nodes around z_g (the table's own linear interpolation, R10); stored [i][lane] for node kde_node(lane, i)
  const double gam = th[9], kap = th[10], zp = th[11];
  const double psi0 = 1.0 + pow(1.0 + zp, -(gam + kap));
#pragma unroll 1
  for (int i = 0; i < KDE_NPL; ++i) {
    const int g = kde_node(lane, i);
    const double zg = fmin(g * dzg, p.los_zmax);
    const double tz = zg / dzl;
    int b = (int)floor(tz);
    b = b > p.n_z - 2 ? p.n_z - 2 : b;
    const double fz = tz - (double)b;
    const double x = 1.0 + g * dzg;
    const double psi = psi0 * pow(x, gam) / (1.0 + pow(x / (1.0 + zp), gam + kap));
    const double c = (g == 0 || g == G - 1) ? 0.5 * dzg : dzg;
    const double w = g < G ? c * psi / x : 0.0;
    NodeW nw;
    nw.w0 = w * (1.0 - fz);
    nw.w1 = w * fz;
    gw[(size_t)t * (32 * KDE_NPL) + i * 32 + lane] = nw;
  }
}

template <typename NodeT, typename LosT, bool MP>
__global__ void __launch_bounds__(KDE_THREADS, 2) kde_kernel(const KdeParams p) {
  extern __shared__ __align__(16) unsigned char kde_smem[];
  MathTables& mt = *reinterpret_cast<MathTables*>(kde_smem);
  // the LOS bin of every grid node
  int* s_b = reinterpret_cast<int*>(kde_smem + sizeof(MathTables));
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  init_math_tables(mt, tid, KDE_THREADS);
  __syncthreads();
  const double* exptab = mt.exptab + (lane & (EXP_REP - 1));
  const double2* logtab = mt.logtab + (lane & (LOG_REP - 1));
  const unsigned FULL = 0xffffffffu;
  const int G = p.n_grid;
  const double dzg = p.los_zmax / (G - 1);
  const double dzl = p.los_zmax / (p.n_z - 1);
  const int64_t n_units = p.n_theta * p.n_chunks;
  if (tid < 32 * KDE_NPL) {   // LOS bin of grid node g = kde_node(l, i), stored at [i][l]
    const int l = tid & 31, i = tid >> 5, g = kde_node(l, i);
    const double zg = fmin(g * dzg, p.los_zmax);
    int b = (int)floor(zg / dzl);
    b = b > p.n_z - 2 ? p.n_z - 2 : b;
    s_b[i * 32 + l] = b;
  }
  __syncthreads();

  for (int64_t unit = (int64_t)blockIdx.x * KDE_WARPS + warp; unit < n_units; unit += (int64_t)gridDim.x * KDE_WARPS) {
    const int64_t chunk = unit / p.n_theta, t = unit - chunk * p.n_theta;   // chunk-major: a CTA's warps share samples
    const int64_t ev = p.chunk_event[chunk];
    const int64_t s0 = p.chunk_start[chunk], s1 = p.chunk_end[chunk];
    const size_t o = (size_t)t * (size_t)p.n_chunks + (size_t)chunk;
    if (!(p.tvalid[t] == 1.0) || s1 <= s0) {   // (an invalid theta gets its NaN in the combine)
      if (lane == 0) {
        p.part_e[o] = 0.0;
        p.part_np[o] = 0;
        p.part_nu[o] = 0;
      }
      continue;
    }
    const ThetaK K = p.thk[t];
    const NodeW* s_w = p.gw + (size_t)t * (32 * KDE_NPL);
    __syncwarp();
    const NodeT* tab = reinterpret_cast<const NodeT*>(p.tab) + (size_t)t * p.Mp;
    const double shift = p.seg_shift[ev];
    const double eshift = exp(-shift);
    // ---- (z_k, v_k) of every sample of the event, relative to e^shift ----
    double2* scr = p.scr + ((size_t)blockIdx.x * KDE_WARPS + warp) * (size_t)p.scr_stride - s0;   // indexed by sample
    for (int64_t c0 = s0; c0 < s1; c0 += 32) {
      const int64_t k = c0 + lane;
      if (k < s1) {
        double z;
        const double d = p.dL[k];
        const double lp = p.lprior ? p.lprior[k] : 0.0;
        const double scale = !p.lprior ? eshift / (d * d)
                                       : (isfinite(lp) ? exp_fast<true>(-lp - shift, exptab) : CUDART_NAN);
        const double v = sample_v<NodeT, MP>(K, tab, p.M, p.tab_zq, d, p.m1z[k], p.m2z[k], scale, p.row[k], p.n_rows, p.los_zmax,
                                  logtab, exptab, z);
        GWC_DEV_CHECK(p.flag, k - s0 >= 0 && k - s0 < p.scr_stride, FLAG_CHK_KDE);
        scr[k] = make_double2(z, v);
      }
    }
    __syncwarp();
    double esum = 0.0;   // this lane's share of the sum over the contributing pixels of I_j, relative to e^shift
    int np = 0;
    int64_t nu = 0;
    // ---- per-pixel statistics, 32 samples at a time whatever the pixel boundaries (lanes = samples): segmented warp
    // scans of sum v, sum v d, sum v d^2, sum v^2 with d = z - K, K = the pixel's first live redshift (the shifted
    // one-pass form of the weighted variance: identical samples give exactly 0, and K lies inside the pixel's own
    // spread, so the subtraction loses a few ulp at most); the run a row leaves open is carried to the next row.
    // Pixels end at `tail` lanes: those that pass (n >= 2, N_eff, var > 0) go through the KDE one after the other.
    double cV = 0.0, cVd = 0.0, cVdd = 0.0, cQ = 0.0, cK = 0.0;   // the open run (warp-uniform)
    int cn = 0, clen = 0;
    bool cHasK = false;
    for (int64_t c0 = s0; c0 < s1; c0 += 32) {
      const int64_t k = c0 + lane;
      const bool in = k < s1;
      const int32_t r = in ? p.row[k] : 0;
      const bool head = in && (k == s0 || p.row[k - 1] != r);
      const bool tail = in && (k + 1 >= s1 || p.row[k + 1] != r);
      const double2 zv = in ? scr[k] : make_double2(0.0, -1.0);
      const bool live = zv.y >= 0.0;
      const double v = live ? zv.y : 0.0, z = zv.x;
      const unsigned hall = __ballot_sync(FULL, head), lm = __ballot_sync(FULL, live);
      const unsigned le = 0xffffffffu >> (31 - lane);
      const unsigned hm = hall & le;
      const bool open_left = hm == 0;                       // this lane's run began before the row
      const int first = open_left ? 0 : 31 - __clz(hm);     // first lane of the run inside the row
      const unsigned runm = le & (0xffffffffu << first);    // lanes of the run up to this one
      const unsigned lrun = lm & runm;
      double K = __shfl_sync(FULL, z, lrun ? __ffs(lrun) - 1 : lane);
      if (open_left && cHasK) K = cK;
      const double dz = z - K;
      double V = v, Vd = v * dz, Vdd = v * dz * dz, Q = v * v;
      const int reach = lane - first;
      const int maxd = __reduce_max_sync(FULL, in ? reach : 0);
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        if (o > maxd) break;   // warp-uniform
        const double tV = __shfl_up_sync(FULL, V, o), tVd = __shfl_up_sync(FULL, Vd, o);
        const double tVdd = __shfl_up_sync(FULL, Vdd, o), tQ = __shfl_up_sync(FULL, Q, o);
        const bool take = reach >= o;
        V += take ? tV : 0.0;
        Vd += take ? tVd : 0.0;
        Vdd += take ? tVdd : 0.0;
        Q += take ? tQ : 0.0;
      }
      int n = __popc(lrun);
      int len = reach + 1;
      if (open_left) { V += cV; Vd += cVd; Vdd += cVdd; Q += cQ; n += cn; len += clen; }
      // what the next row inherits (lane 31's run when it stays open)
      {
        const bool open31 = __shfl_sync(FULL, (int)(in && !tail), 31) != 0;
        const unsigned lr31 = __shfl_sync(FULL, lrun, 31);
        const bool left31 = __shfl_sync(FULL, (int)open_left, 31) != 0;
        const double kk = __shfl_sync(FULL, K, lr31 ? 31 - __clz(lr31) : 31);
        const double nV = __shfl_sync(FULL, V, 31), nVd = __shfl_sync(FULL, Vd, 31);
        const double nVdd = __shfl_sync(FULL, Vdd, 31), nQ = __shfl_sync(FULL, Q, 31);
        const int nn = __shfl_sync(FULL, n, 31), nlen = __shfl_sync(FULL, len, 31);
        if (open31) {
          if (lr31 && !(left31 && cHasK)) { cK = kk; cHasK = true; }
          else if (!left31) cHasK = false;
          cV = nV; cVd = nVd; cVdd = nVdd; cQ = nQ; cn = nn; clen = nlen;
        } else {
          cV = 0.0; cVd = 0.0; cVdd = 0.0; cQ = 0.0; cn = 0; clen = 0; cHasK = false;
        }
      }
      // the pixels that end in this row
      bool pass = tail && n >= 2 && V > 0.0 && V * V >= p.neff_min * Q;
      double sd = 0.0, h = 0.0;
      if (pass) {
        const double rV = rcp_fast(V);
        const double mo = Vd * rV;
        const double var = fma(-Vd, mo, Vdd) * rV;
        pass = var > 0.0;
        sd = pass ? sqrt(var) : 0.0;
        h = 1.06 * sd * exp_fast<false>(-0.2 * log_fast((double)n, logtab), exptab);   // Eq. D1: n^(-1/5) = e^(-ln n / 5)
      }
      unsigned pm = __ballot_sync(FULL, pass);
      while (pm) {
        const int tl = __ffs(pm) - 1;
        pm &= pm - 1;
        const int n_p = __shfl_sync(FULL, n, tl), len_p = __shfl_sync(FULL, len, tl);
        const int32_t prow = __shfl_sync(FULL, r, tl);
        double h_p = __shfl_sync(FULL, h, tl);
        const int64_t r1 = c0 + tl + 1, r0 = r1 - len_p;
        if (p.bw_rule == 1) {                            // Eq. D2
          const double sd_p = __shfl_sync(FULL, sd, tl);
          const double iqr = live_quantile(scr, r0, r1, n_p, 0.75, KeyZ(), lane) -
                             live_quantile(scr, r0, r1, n_p, 0.25, KeyZ(), lane);
          const double spread = iqr / 1.34 < sd_p ? iqr / 1.34 : sd_p;
          h_p = 0.9 * spread * pow((double)n_p, -0.2);
          if (!(h_p > 0.0)) continue;
        } else if (p.bw_rule >= 2) {                     // Eq. D3-D4: as printed (2) or inside Scott's rule (3)
          const double zeta2 = live_biweight(scr, r0, r1, n_p, lane);
          h_p = p.bw_rule == 2 ? zeta2 : 1.06 * sqrt(zeta2) * pow((double)n_p, -0.2);
          if (!(h_p > 0.0) || !isfinite(h_p)) continue;
        }
        const double part = kde_pixel<LosT>(scr, r0, r1, h_p, prow, p, dzg, s_w, s_b, exptab, lane);
        if (__any_sync(FULL, part > 0.0)) {
          esum += part;
          ++np;
          nu += n_p;
        }
      }
    }
    esum = wsum(esum);
    if (lane == 0) {
      p.part_e[o] = esum;
      p.part_np[o] = np;
      p.part_nu[o] = nu;
    }
    __syncwarp();   // the scratch slice is rewritten by the next unit
  }
}

// log L_i = shift + ln(sum over the event's chunks, in order) - ln S_i; npass, nused summed the same way
__global__ void kde_combine_kernel(const KdeParams p) {
  const int64_t o = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (o >= p.n_theta * p.n_events) return;
  const int64_t t = o / p.n_events, ev = o - t * p.n_events;
  const int64_t S = p.ev_off[ev + 1] - p.ev_off[ev];
  if (!(p.tvalid[t] == 1.0)) {   // theta outside the domain or changed since the build: NaN (sticky flag set)
    p.logL[o] = CUDART_NAN;
    if (p.npass) p.npass[o] = 0;
    if (p.nused) p.nused[o] = 0;
    return;
  }
  double e = 0.0;
  int64_t np = 0, nu = 0;
  for (int64_t c = p.chunk_off[ev]; c < p.chunk_off[ev + 1]; ++c) {
    const size_t q = (size_t)t * (size_t)p.n_chunks + (size_t)c;
    e += p.part_e[q];
    np += p.part_np[q];
    nu += p.part_nu[q];
  }
  p.logL[o] = (S > 0 && e > 0.0) ? p.seg_shift[ev] + log(e) - log((double)S) : -CUDART_INF;
  if (p.npass) p.npass[o] = np;
  if (p.nused) p.nused[o] = nu;
}

}  // namespace

// upper bound of the number of chunks of a catalogue (what the chunk arrays are sized for)
int64_t kde_chunk_bound(int64_t n_samples, int64_t n_events) { return n_samples / KDE_CHUNK + n_events + 1; }

// chunk table of a catalogue: d_cnt [n_events] scratch, d_chunk_off [n_events + 1] (its last entry = number of
// chunks), start / end / event [kde_chunk_bound], d_max_len[0] = longest chunk, d_max_len[1] = 1 when an event's
// offsets do not ascend inside [0, n_samples] (both must hold 0 before the call)
int launch_kde_chunks(const int64_t* ev_off, int64_t n_events, const int32_t* row, int64_t* d_cnt,
                      int64_t* d_chunk_off, int64_t* d_start, int64_t* d_end, int32_t* d_event, int64_t* d_max_len,
                      int64_t n_samples, cudaStream_t s) {
  if (n_events <= 0) return 0;
  kde_chunk_count_kernel<<<(unsigned)((n_events + 255) / 256), 256, 0, s>>>(ev_off, n_events, n_samples, d_cnt,
                                                                            d_max_len + 1);
  kde_chunk_scan_kernel<<<1, 256, 0, s>>>(d_cnt, n_events, d_chunk_off);
  kde_chunk_bounds_kernel<<<(unsigned)n_events, 64, 0, s>>>(ev_off, n_events, d_chunk_off, row, d_start, d_end, d_event,
                                                            d_max_len, kde_chunk_bound(n_samples, n_events));
  return cudaGetLastError() == cudaSuccess ? 3 : -1;
}

size_t kde_theta_bytes(int64_t n_theta) { return (size_t)n_theta * sizeof(ThetaK); }
size_t kde_weight_bytes(int64_t n_theta) { return (size_t)n_theta * 32 * KDE_NPL * sizeof(NodeW); }

int launch_kde(int model, const Node64* d_ftab, const double* d_theta, const void* d_tab, const double* d_tconst, const double* d_tvalid, int64_t n_theta, int M, int Mp,
               gwc_prec tab_prec, double tab_zq, int64_t n_events, const int64_t* ev_off, const double* dL,
               const double* m1z, const double* m2z, const double* lprior, const int32_t* row, const double* seg_shift,
               const void* los, gwc_prec los_prec, int64_t n_rows, int n_z, double los_zmax, int n_grid, double neff_min,
               int bw_rule, double* logL, int64_t* npass, int64_t* nused, void* scratch, int64_t scr_stride, int n_blocks,
               int64_t n_chunks, const int64_t* d_chunk_off, const int64_t* d_start, const int64_t* d_end,
               const int32_t* d_event, void* d_thk, void* d_gw, double* d_part_e, int32_t* d_part_np,
               int64_t* d_part_nu, int* d_flag, cudaStream_t s) {
  if (n_theta <= 0 || n_events <= 0) return 0;
  KdeParams p;
  p.flag = d_flag;
  p.model = model; p.ftab = d_ftab; p.theta = d_theta; p.tab = d_tab; p.tconst = d_tconst; p.tvalid = d_tvalid; p.n_theta = n_theta; p.n_events = n_events;
  p.M = M; p.Mp = Mp; p.tab_zq = tab_zq; p.ev_off = ev_off; p.dL = dL; p.m1z = m1z; p.m2z = m2z; p.lprior = lprior;
  p.row = row; p.seg_shift = seg_shift; p.los = los; p.n_rows = n_rows; p.n_z = n_z; p.los_zmax = los_zmax;
  p.n_grid = n_grid; p.neff_min = neff_min; p.bw_rule = bw_rule; p.logL = logL; p.npass = npass; p.nused = nused;
  p.scr = (double2*)scratch; p.scr_stride = scr_stride;
  p.thk = (const ThetaK*)d_thk; p.gw = (const NodeW*)d_gw; p.n_chunks = n_chunks; p.chunk_start = d_start;
  p.chunk_end = d_end; p.chunk_event = d_event; p.chunk_off = d_chunk_off; p.part_e = d_part_e; p.part_np = d_part_np;
  p.part_nu = d_part_nu;
  if (model == 1) kde_theta_prep_kernel<true><<<(unsigned)n_theta, 32, 0, s>>>(p, (ThetaK*)d_thk, (NodeW*)d_gw);
  else kde_theta_prep_kernel<false><<<(unsigned)n_theta, 32, 0, s>>>(p, (ThetaK*)d_thk, (NodeW*)d_gw);
  const size_t smem = sizeof(MathTables) + sizeof(int) * 32 * KDE_NPL;
  const int64_t blocks = n_blocks;
  if (n_chunks > 0) {
#define GWC_KDE_LAUNCH1(NodeT, LosT, MP)                                                                              \
  do {                                                                                                                \
    if (cudaFuncSetAttribute(kde_kernel<NodeT, LosT, MP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != \
        cudaSuccess)                                                                                                  \
      return -1;                                                                                                      \
    kde_kernel<NodeT, LosT, MP><<<(unsigned)blocks, KDE_THREADS, smem, s>>>(p);                                      \
  } while (0)
#define GWC_KDE_LAUNCH(NodeT, LosT)                   \
  do {                                                \
    if (model == 1) GWC_KDE_LAUNCH1(NodeT, LosT, true); \
    else GWC_KDE_LAUNCH1(NodeT, LosT, false);           \
  } while (0)
    if (tab_prec == GWC_F64) {
      if (los_prec == GWC_F64) GWC_KDE_LAUNCH(Node64, double); else GWC_KDE_LAUNCH(Node64, float);
    } else {
      if (los_prec == GWC_F64) GWC_KDE_LAUNCH(Node32, double); else GWC_KDE_LAUNCH(Node32, float);
    }
#undef GWC_KDE_LAUNCH
#undef GWC_KDE_LAUNCH1
  }
  const int64_t n_out = n_theta * n_events;
  kde_combine_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, s>>>(p);
  return cudaGetLastError() == cudaSuccess ? (n_chunks > 0 ? 3 : 2) : -1;
}

// grid of the KDE kernel (persistent, two CTAs of 8 warps per SM) and the scratch it needs: one slice of the longest
// chunk's (z, v) pairs per resident warp
int kde_grid_blocks(int64_t n_theta, int64_t n_chunks, int n_sm) {
  const int64_t units = n_theta * n_chunks;
  int64_t blocks = (units + KDE_WARPS - 1) / KDE_WARPS;
  if (blocks > (int64_t)n_sm * 2) blocks = (int64_t)n_sm * 2;
  return (int)(blocks < 1 ? 1 : blocks);
}
size_t kde_scratch_bytes(int n_blocks, int64_t max_chunk_len) {
  return (size_t)n_blocks * KDE_WARPS * (size_t)(max_chunk_len > 0 ? max_chunk_len : 1) * sizeof(double2);
}

}  // namespace gwc
