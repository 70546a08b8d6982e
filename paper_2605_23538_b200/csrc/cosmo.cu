// cosmo.cu -- A1 + A2: per-theta inverse-cosmology table and population constants.
//
// Eq. 1 of the paper: d_L(z) = (1+z) (c/H0) D(z), D(z) = int_0^z dz'/E(z'),
// E = sqrt(Om (1+z)^3 + 1 - Om).  In the dimensionless u = d_L H0/c = (1+z) D(z) the inverse z(u)
// depends on Om only.  One CTA per theta:
//   1. forward cumulative quadrature: 3-point Gauss-Legendre on each of QUAD_K uniform z intervals,
//      compensated prefix sum -> D(z_k), u(z_k) in shared memory;
//   2. monotone inversion: for every node u_m = m du, du = u(z_max)/(M-1), bracket by binary search
//      in u(z_k), then Newton on (1+z)(D(z_k) + int_{z_k}^{z} dz'/E) = u_m (the short remainder
//      integral again by 3-point Gauss-Legendre);
//   3. node slope d_m = du * dz/du = du / (u/(1+z) + (1+z)/E(z))  (cubic-Hermite data, R9);
//   4. thread 0 writes the constant block of the population laws (R2-R4).
// Not a hot kernel (n_theta * M Newton solves); libdevice sqrt/div/pow/erf are used as they are.
#include <math_constants.h>

#include "gwc_internal.h"

namespace gwc {

namespace {

constexpr double C_KMS = 299792.458;
constexpr int CB_THREADS = 256;

__device__ __forceinline__ double invE(double z, double Om, double OL) {
  double x = 1.0 + z;
  return rsqrt(fma(Om * x * x, x, OL));
}

// int_a^b dz/E by 3-point Gauss-Legendre
__device__ __forceinline__ double gl3(double a, double b, double Om, double OL) {
  const double XN = 0.77459666924148337704;  // sqrt(3/5)
  double hm = 0.5 * (b - a), c = 0.5 * (a + b);
  double s = 5.0 * (invE(c - hm * XN, Om, OL) + invE(c + hm * XN, Om, OL)) + 8.0 * invE(c, Om, OL);
  return hm * s * (1.0 / 9.0);
}

__device__ __forceinline__ void store_node(Node64* t, double z, double d, double) { t->z = z; t->d = d; }
// 32-bit storage (R22): z_m as a fixed-point fraction of z_max (absolute step z_max / (2^32 - 1), 256x
// finer than an f32 near z_max), the slope in the same units as an f32.
__device__ __forceinline__ void store_node(Node32* t, double z, double d, double inv_q) {
  t->zq = __double2uint_rn(fmin(z * inv_q, NODE32_QMAX));
  t->d = __double2float_rn(d * inv_q);
}

__device__ bool theta_valid(const double* th, int model) {
  const int npar = model == 1 ? GWC_NPAR_MULTIPEAK : GWC_NPAR;
  for (int i = 0; i < npar; ++i)
    if (!isfinite(th[i])) return false;
  if (model == 1) {   // MULTIPEAK (R35): delta_m, mu_low, sigma_low, lambda_low = th[12..15]
    if (!(th[12] >= 0.0 && th[4] + th[12] < th[5])) return false;
    if (!(th[14] > 0.0)) return false;
    if (!(th[15] >= 0.0 && th[15] <= 1.0)) return false;
  }
  if (!(th[0] > 0.0)) return false;
  if (!(th[1] > 0.0 && th[1] <= 1.0)) return false;
  if (!(th[7] > 0.0)) return false;
  if (!(th[4] > 0.0 && th[4] < th[5])) return false;
  if (!(th[8] >= 0.0 && th[8] <= 1.0)) return false;
  if (!(th[11] > -1.0)) return false;
  if (fabs(th[2] - 1.0) < 1e-6) return false;
  if (fabs(th[3] + 1.0) < 1e-6) return false;
  return true;
}

// 8-point Gauss-Legendre on [-1, 1]
__constant__ double GL8_X[8] = {-0.96028985649753623168, -0.79666647741362673959, -0.52553240991632898582,
                                -0.18343464249564980494, 0.18343464249564980494,  0.52553240991632898582,
                                0.79666647741362673959,  0.96028985649753623168};
__constant__ double GL8_W[8] = {0.10122853629037625915, 0.22238103445337447054, 0.31370664587788728734,
                                0.36268378337836198297, 0.36268378337836198297, 0.31370664587788728734,
                                0.22238103445337447054, 0.10122853629037625915};

// MULTIPEAK smoothing (R34) at m' = m - mmin inside (0, dm): S and 1 - S, each without cancellation
__device__ __forceinline__ void mp_smooth(double mp, double dm, double& S, double& oneMinusS) {
  const double e = dm / mp + dm / (mp - dm);
  S = 1.0 / (1.0 + exp(e));          // exp overflows to +inf near mmin: S = 0
  oneMinusS = 1.0 / (1.0 + exp(-e));
}

struct MpMix {   // the MULTIPEAK mixture before smoothing, components normalised on [mmin, mmax]
  double a_pl, alpha, a_gl, mul, isl, a_gh, muh, ish;
  __device__ double operator()(double m) const {
    const double yl = (m - mul) * isl, yh = (m - muh) * ish;
    return a_pl * pow(m, -alpha) + a_gl * exp(-0.5 * yl * yl) + a_gh * exp(-0.5 * yh * yh);
  }
};

template <typename NodeT>
__global__ void __launch_bounds__(CB_THREADS) cosmo_build_kernel(const double* __restrict__ theta, int model,
                                                                  double z_max, int M, int Mp, NodeT* __restrict__ tab,
                                                                  double* __restrict__ tconst,
                                                                  Node64* __restrict__ ftab,
                                                                  double* __restrict__ theta_snap,
                                                                  double* __restrict__ tvalid, int* flag) {
  __shared__ double Dg[QUAD_K + 1];
  __shared__ double ug[QUAD_K + 1];
  __shared__ double part[CB_THREADS];
  __shared__ double s_umax;
  const int t = blockIdx.x, tid = threadIdx.x;
  const int npar = model == 1 ? GWC_NPAR_MULTIPEAK : GWC_NPAR, ncst = nconst_of(model);
  const double* th = theta + (size_t)t * npar;
  NodeT* row = tab + (size_t)t * Mp;
  double* tc = tconst + (size_t)t * ncst;
  const bool valid = theta_valid(th, model);
  // the copy of theta the tables belong to (the dependent calls compare the caller's array with it)
  if (tid < npar) theta_snap[(size_t)t * npar + tid] = th[tid];
  if (tid == 0) tvalid[t] = valid ? 1.0 : CUDART_NAN;
  if (!valid) {
    for (int m = tid; m < Mp; m += CB_THREADS) store_node(row + m, 0.0, 0.0, 0.0);
    if (model == 1)
      for (int m = tid; m < MF_PITCH; m += CB_THREADS) ftab[(size_t)t * MF_PITCH + m] = Node64{0.0, 0.0};
    if (tid < ncst) tc[tid] = (tid == C_VALID) ? CUDART_NAN : 0.0;
    if (tid == 0) atomicOr(flag, FLAG_DOMAIN);
    return;
  }
  const double Om = th[1], OL = 1.0 - Om;
  const double hz = z_max / QUAD_K;
  constexpr int PER = QUAD_K / CB_THREADS;
  // 1. interval integrals, thread-local prefix, compensated scan of the thread totals
  double loc[PER];
  double run = 0.0;
#pragma unroll
  for (int j = 0; j < PER; ++j) {
    int k = tid * PER + j;
    run += gl3(k * hz, (k + 1) * hz, Om, OL);
    loc[j] = run;
  }
  part[tid] = run;
  __syncthreads();
  if (tid == 0) {
    double s = 0.0, comp = 0.0;  // Neumaier-compensated exclusive scan
    for (int i = 0; i < CB_THREADS; ++i) {
      double v = part[i];
      part[i] = s + comp;
      double tsum = s + v;
      comp += (fabs(s) >= fabs(v)) ? ((s - tsum) + v) : ((v - tsum) + s);
      s = tsum;
    }
    Dg[0] = 0.0;
    ug[0] = 0.0;
  }
  __syncthreads();
  {
    double base = part[tid];
#pragma unroll
    for (int j = 0; j < PER; ++j) {
      int k = tid * PER + j + 1;
      double D = base + loc[j];
      Dg[k] = D;
      ug[k] = (1.0 + k * hz) * D;
    }
  }
  __syncthreads();
  if (tid == 0) s_umax = ug[QUAD_K];
  __syncthreads();
  const double umax = s_umax;
  const double du = umax / (M - 1);
  // 2-3. nodes
  for (int m = tid; m < Mp; m += CB_THREADS) {
    double z, d;
    if (m >= M - 1) {
      z = z_max;
      d = (m == M - 1) ? du / (umax / (1.0 + z) + (1.0 + z) * invE(z, Om, OL)) : 0.0;
    } else {
      double u = m * du;
      int lo = 0, hi = QUAD_K;  // ug[lo] <= u < ug[hi]
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (ug[mid] <= u) lo = mid; else hi = mid;
      }
      double zk = lo * hz, Dk = Dg[lo];
      z = zk + (u - ug[lo]) / (ug[lo + 1] - ug[lo]) * hz;
#pragma unroll 1
      for (int it = 0; it < 5; ++it) {
        double Dz = Dk + gl3(zk, z, Om, OL);
        double x = 1.0 + z;
        double f = x * Dz - u;
        double fp = Dz + x * invE(z, Om, OL);
        z -= f / fp;
      }
      if (m == 0) z = 0.0;
      double x = 1.0 + z;
      d = du / (u / x + x * invE(z, Om, OL));
    }
    store_node(row + m, z, d, NODE32_QMAX / z_max);
  }
  // 4. MULTIPEAK (R33-R36): N1 = int mix S = 1 - int_window mix (1 - S), and the table of
  //    |F|(m1) = |beta+1| C(m1) / (S(m1) m1^(beta+1)), C(m1) = int_mmin^m1 m^beta S(m) dm, on MF_NODES uniform nodes of
  //    the window [mmin, mmin + delta_m] with the analytic slopes F' = (beta+1)/m - F (S'/S + (beta+1)/m),
  //    S'/S = (1 - S) delta_m (1/m'^2 + 1/(m' - delta_m)^2).  Every table interval by 4 panels of 8-point
  //    Gauss-Legendre.  (The first two intervals, where S < e^-255, are inaccurate in relative terms: the integrand
  //    is an essential singularity there; samples that low carry no weight.)
  __shared__ double cI[MF_NODES], dI[MF_NODES];
  __shared__ double s_n1, s_ctop;
  const double alpha = th[2], beta = th[3], mmin = th[4], mmax = th[5], mu = th[6], sigma = th[7], lam = th[8];
  const double n_pl = (1.0 - alpha) / (pow(mmax, 1.0 - alpha) - pow(mmin, 1.0 - alpha));
  const double rs2 = 1.0 / (sigma * 1.41421356237309504880);
  const double n_g = 1.0 / (0.5 * (erf((mmax - mu) * rs2) - erf((mmin - mu) * rs2)));
  double n_gl = 0.0;
  if (model == 1) {
    const double dm = th[12], mul = th[13], sigl = th[14], laml = th[15];
    const double rsl = 1.0 / (sigl * 1.41421356237309504880);
    n_gl = 1.0 / (0.5 * (erf((mmax - mul) * rsl) - erf((mmin - mul) * rsl)));
    MpMix mix;
    mix.a_pl = (1.0 - lam) * n_pl;
    mix.alpha = alpha;
    mix.a_gl = lam * laml * n_gl / (sigl * 2.50662827463100050242);
    mix.mul = mul;
    mix.isl = 1.0 / sigl;
    mix.a_gh = lam * (1.0 - laml) * n_g / (sigma * 2.50662827463100050242);
    mix.muh = mu;
    mix.ish = 1.0 / sigma;
    const double hF = dm / (MF_NODES - 1);
    for (int k = tid; k < MF_NODES - 1; k += CB_THREADS) {
      double sc = 0.0, sd = 0.0;
      const double w = 0.25 * hF;
      for (int sub = 0; sub < 4; ++sub) {
        const double a = (k * 4 + sub) * w;
        for (int i = 0; i < 8; ++i) {
          const double mp = a + 0.5 * w * (GL8_X[i] + 1.0);
          double S, nS;
          mp_smooth(mp, dm, S, nS);
          const double m = mmin + mp;
          sc = fma(GL8_W[i], pow(m, beta) * S, sc);
          sd = fma(GL8_W[i], mix(m) * nS, sd);
        }
      }
      cI[k] = 0.5 * w * sc;
      dI[k] = 0.5 * w * sd;
    }
    __syncthreads();
    if (tid == 0) {   // cumulative C at the nodes (ascending, compensated), total deficit
      double s = 0.0, comp = 0.0, d = 0.0;
      for (int k = 0; k < MF_NODES - 1; ++k) {
        const double v = dm > 0.0 ? cI[k] : 0.0;
        d += dm > 0.0 ? dI[k] : 0.0;
        const double tsum = s + v;
        comp += (s - tsum) + v;
        s = tsum;
        cI[k] = s + comp;   // C at node k + 1
      }
      s_ctop = s + comp;
      s_n1 = 1.0 - d;
    }
    __syncthreads();
    const double sgn = (beta + 1.0 > 0.0) ? 1.0 : -1.0;
    Node64* fr = ftab + (size_t)t * MF_PITCH;
    for (int k = tid; k < MF_PITCH; k += CB_THREADS) {
      double F = 0.0, dF = 0.0;
      if (k >= 1 && dm > 0.0) {
        const int kk = k < MF_NODES - 1 ? k : MF_NODES - 1;
        const double mp = kk * hF, m = mmin + mp, C = cI[kk - 1];
        double S = 1.0, nS = 0.0, q = 0.0;   // q = S'/S
        if (kk < MF_NODES - 1) {
          mp_smooth(mp, dm, S, nS);
          q = nS * dm * (1.0 / (mp * mp) + 1.0 / ((mp - dm) * (mp - dm)));
        }
        const double Fs = S > 0.0 ? (beta + 1.0) * C / (S * pow(m, beta + 1.0)) : 0.0;
        const double dFs = S > 0.0 ? (beta + 1.0) / m - Fs * (q + (beta + 1.0) / m) : 0.0;
        F = sgn * Fs;
        dF = (k <= MF_NODES - 1) ? sgn * dFs * hF : 0.0;
        if (!(isfinite(F) && isfinite(dF))) { F = 0.0; dF = 0.0; }
      }
      fr[k] = Node64{F, dF};
    }
  }
  // 5. constants
  if (tid == 0) {
    const double H0 = th[0], gam = th[9], kap = th[10], zp = th[11];
    const double h = H0 / C_KMS;
    const double psi0 = 1.0 + pow(1.0 + zp, -(gam + kap));
    double common = fabs(beta + 1.0) * psi0 * h;
    double lam_hi = lam;   // coefficient of the (high) Gaussian peak
    double e1c = (beta + 1.0) * log(mmin);
    if (model == 1) {
      const double dm = th[12], mul = th[13], sigl = th[14], laml = th[15], top = mmin + dm;
      common /= s_n1;
      lam_hi = lam * (1.0 - laml);
      e1c = log(pow(top, beta + 1.0) - (beta + 1.0) * s_ctop);
      const double lam_lo = lam * laml;
      tc[C_CG2] = (lam_lo > 0.0) ? log(lam_lo * n_gl / (sigl * 2.50662827463100050242) * common) : -CUDART_INF;
      tc[C_INVSIG2] = 1.0 / sigl;
      tc[C_NMUSIG2] = -mul / sigl;
      tc[C_DM] = dm;
      tc[C_FIDX] = dm > 0.0 ? (MF_NODES - 1) / dm : 0.0;
      tc[C_N1] = s_n1;
      tc[C_CTOP] = s_ctop;
      tc[C_NGL] = n_gl;
      for (int i = C_COUNT_MP; i < NCONST_MP; ++i) tc[i] = 0.0;
    } else {
      for (int i = C_COUNT; i < NCONST; ++i) tc[i] = 0.0;
    }
    tc[C_H] = h;
    tc[C_UMAX] = umax;
    tc[C_INVDU] = (M - 1) / umax;
    tc[C_MMIN] = mmin;
    tc[C_MMAX] = mmax;
    tc[C_BETA] = beta;
    tc[C_GM1] = gam - 1.0;
    tc[C_NALPHA] = -alpha;
    tc[C_CPL] = (lam < 1.0) ? log((1.0 - lam) * n_pl * common) : -CUDART_INF;
    tc[C_CG] = (lam_hi > 0.0) ? log(lam_hi * n_g / (sigma * 2.50662827463100050242) * common) : -CUDART_INF;
    tc[C_INVSIG] = 1.0 / sigma;
    tc[C_NMUSIG] = -mu / sigma;
    tc[C_NBP1] = -(beta + 1.0);
    tc[C_E1C] = e1c;
    tc[C_SGN] = (beta + 1.0 > 0.0) ? 1.0 : -1.0;
    tc[C_GK] = gam + kap;
    tc[C_E2C] = -(gam + kap) * log1p(zp);
    tc[C_OM] = Om;
    tc[C_OL] = OL;
    tc[C_VALID] = 1.0;
  }
}

__device__ __forceinline__ double node_z(const Node64& n, double) { return n.z; }
__device__ __forceinline__ double node_d(const Node64& n, double) { return n.d; }
__device__ __forceinline__ double node_z(const Node32& n, double z_max) { return (double)n.zq * (z_max / NODE32_QMAX); }
__device__ __forceinline__ double node_d(const Node32& n, double z_max) { return (double)n.d * (z_max / NODE32_QMAX); }

template <typename NodeT>
__global__ void export_cosmo_kernel(const NodeT* __restrict__ tab, const double* __restrict__ tconst, int ncst,
                                    int64_t n_theta, int M, int Mp, double z_max, double* z, double* dz, double* umax) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n_theta * M) return;
  int64_t t = i / M;
  int m = (int)(i - t * M);
  NodeT nd = tab[t * Mp + m];
  if (z) z[i] = node_z(nd, z_max);
  if (dz) dz[i] = node_d(nd, z_max);
  if (umax && m == 0) umax[t] = tconst[t * ncst + C_UMAX];
}

}  // namespace

int launch_cosmo_build(const double* d_theta, int64_t n_theta, int model, double z_max, int M, int Mp, gwc_prec prec,
                       void* d_tab, double* d_tconst, Node64* d_ftab, double* d_theta_snap, double* d_tvalid,
                       int* d_flag, cudaStream_t s) {
  if (n_theta <= 0) return 0;
  if (prec == GWC_F64)
    cosmo_build_kernel<Node64><<<(unsigned)n_theta, CB_THREADS, 0, s>>>(d_theta, model, z_max, M, Mp, (Node64*)d_tab,
                                                                         d_tconst, d_ftab, d_theta_snap, d_tvalid,
                                                                         d_flag);
  else
    cosmo_build_kernel<Node32><<<(unsigned)n_theta, CB_THREADS, 0, s>>>(d_theta, model, z_max, M, Mp, (Node32*)d_tab,
                                                                         d_tconst, d_ftab, d_theta_snap, d_tvalid,
                                                                         d_flag);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

namespace {
// one thread per theta: bitwise comparison of the caller's row with the copy the tables were built from
__global__ void verify_theta_kernel(const double* __restrict__ theta, const double* __restrict__ snap,
                                    const double* __restrict__ tconst, int64_t n_theta, int npar, int ncst,
                                    double* __restrict__ tvalid, int* flag) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= n_theta) return;
  bool same = true;
  for (int i = 0; i < npar; ++i)
    same = same && __double_as_longlong(theta[t * npar + i]) == __double_as_longlong(snap[t * npar + i]);
  tvalid[t] = same ? tconst[t * ncst + C_VALID] : CUDART_NAN;
  if (!same) atomicOr(flag, FLAG_STALE);
}
}  // namespace

namespace {
// One table can serve the batch only if every row is inside the model's domain as well: cosmo_build_kernel writes an
// all-zero table for a row outside it, and a tile stages the table of its FIRST theta for all of its points.
__global__ void omega_same_kernel(const double* __restrict__ theta, int64_t n_theta, int npar, int model,
                                  int* __restrict__ same, int* __restrict__ flag) {
  const long long ref = __double_as_longlong(theta[1]);
  bool ok = true;
  for (int64_t t = threadIdx.x; t < n_theta; t += blockDim.x)
    ok = ok && __double_as_longlong(theta[t * npar + 1]) == ref && theta_valid(theta + t * npar, model);
  const int all = __syncthreads_and(ok ? 1 : 0);
  if (threadIdx.x == 0) {
    *same = all;
    if (flag && !all) atomicOr(flag, FLAG_OMEGA);
  }
}
}  // namespace

int launch_omega_same(const double* d_theta, int64_t n_theta, int model, int* d_same, cudaStream_t s, int* d_flag) {
  if (n_theta <= 0) return 0;
  omega_same_kernel<<<1, 256, 0, s>>>(d_theta, n_theta, model == 1 ? GWC_NPAR_MULTIPEAK : GWC_NPAR, model, d_same,
                                      d_flag);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_verify_theta(const double* d_theta, const double* d_theta_snap, const double* d_tconst, int64_t n_theta,
                        int model, double* d_tvalid, int* d_flag, cudaStream_t s) {
  if (n_theta <= 0) return 0;
  verify_theta_kernel<<<(unsigned)((n_theta + 127) / 128), 128, 0, s>>>(
      d_theta, d_theta_snap, d_tconst, n_theta, model == 1 ? GWC_NPAR_MULTIPEAK : GWC_NPAR, nconst_of(model), d_tvalid,
      d_flag);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_export_cosmo(const void* d_tab, const double* d_tconst, int ncst, int64_t n_theta, int M, int Mp,
                        gwc_prec prec, double z_max, double* d_z, double* d_dz, double* d_umax, cudaStream_t s) {
  int64_t n = n_theta * M;
  if (n <= 0) return 0;
  unsigned blocks = (unsigned)((n + 255) / 256);
  if (prec == GWC_F64)
    export_cosmo_kernel<Node64><<<blocks, 256, 0, s>>>((const Node64*)d_tab, d_tconst, ncst, n_theta, M, Mp, z_max, d_z,
                                                       d_dz, d_umax);
  else
    export_cosmo_kernel<Node32><<<blocks, 256, 0, s>>>((const Node32*)d_tab, d_tconst, ncst, n_theta, M, Mp, z_max, d_z,
                                                       d_dz, d_umax);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace gwc
