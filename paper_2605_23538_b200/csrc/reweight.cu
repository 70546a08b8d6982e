// reweight.cu -- A3/A5: the fused re-weighting kernel over (theta, segment, sample), plus the small
// kernels around it (per-sample preparation, work grouping, A4 finalisation, A6 total).
//
// One sample's weight is Eq. 7 of the paper, w = p(z, m1, m2 | theta) / pi_PE, with the
// line-of-sight prior of Eq. 5 read at the sample's own redshift and pixel
// (R1), and Eq. 4 for the injections with the all-sky prior.  Written out
// (readings R2-R8):
//   u = d_L H0/c -> z by cubic Hermite on the per-theta table (A1);  x = 1+z;  m1 = m1z/x, m2 = m2z/x
//   live iff u < umax, z < z_max, mmin < m1 <= mmax, m2 >= mmin, m2z <= m1z, p_los > 0
//   w = [exp(CPL + c - alpha t1) + exp(CG + c - y^2/2)] p_los / [(u + x^2/E)(1 - e1)(1 + e2)]
// with the per-theta constants of gwc_internal.h and the per-sample values prepared once per call
// (ln m1z, ln(m2z/m1z), -ln pi - ln m1z - shift).  The sums over a segment's samples are taken in the
// linear domain relative to a per-segment shift (the log-sum-exp reference, chosen before the sum
// instead of tracked as a running maximum); log L_i = shift + ln(sum) - ln S_i  (A4).
//
// Mapping: a persistent CTA per SM takes work items (segment group, theta tile) from an atomic counter,
// group-major so that CTAs running at the same time share the group's samples and LOS rows in L2.
// The tile's inverse-cosmology tables and constants live in shared memory; samples are staged in
// chunks; lanes are samples, each thread holds SPT samples per theta for independent FP64 chains;
// per-(warp, theta) partial sums live in shared memory and are combined in a fixed order.
#include <math_constants.h>

#include <type_traits>

#include "gwc_internal.h"
#include "math64.cuh"

namespace gwc {

namespace {

constexpr int SMEM_RESERVE = 256;  // static shared memory of the kernel + slack

struct SmemLayout {
  size_t math, tconst, acc, cnt, A, m2z, C, P, row, allsky, tab, total;
};

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

// Per-chunk sample staging: A = (d_L, m1z) and m2z feed the first half of a term, C = (ln m1z, ln(m2z/m1z))
// and P the second half; pairs are read with one 128-bit shared load.
__host__ __device__ inline SmemLayout smem_layout(int T, int Mp, size_t node_bytes, bool inj, int n_z) {
  SmemLayout L;
  size_t o = 0;
  L.math = o;   o = align16(o + sizeof(MathTables));
  L.tconst = o; o = align16(o + sizeof(double) * T * NCONST);
  L.acc = o;    o = align16(o + sizeof(double) * NWARPS * T * 2);
  L.cnt = o;    o = align16(o + sizeof(int) * NWARPS * T);
  L.A = o;      o = align16(o + sizeof(double2) * CHUNK);
  L.m2z = o;    o = align16(o + sizeof(double) * CHUNK);
  L.C = o;      o = align16(o + sizeof(double2) * CHUNK);
  L.P = o;      o = align16(o + sizeof(double) * CHUNK);
  L.row = o;    o = align16(o + (inj ? 0 : sizeof(int32_t) * CHUNK));
  L.allsky = o; o = align16(o + (inj ? sizeof(double) * n_z : 0));
  L.tab = o;    o = align16(o + node_bytes * (size_t)T * Mp);
  L.total = o;
  return L;
}

__device__ __forceinline__ double widen(double v) { return v; }
__device__ __forceinline__ double widen(float v) { return (double)v; }

// Hermite data of one table interval, widened to f64
__device__ __forceinline__ void load_nodes(const Node64* t, int m, double& z0, double& d0, double& z1, double& d1) {
  const double2* q = reinterpret_cast<const double2*>(t + m);
  double2 a = q[0], b = q[1];
  z0 = a.x; d0 = a.y; z1 = b.x; d1 = b.y;
}
// (32-bit nodes: values in units of z_max / (2^32 - 1); the conversions run on the XU pipe, node_scale() follows)
__device__ __forceinline__ void load_nodes(const Node32* t, int m, double& z0, double& d0, double& z1, double& d1) {
  const uint2* q = reinterpret_cast<const uint2*>(t + m);
  const uint2 a = q[0], b = q[1];
  z0 = (double)a.x; d0 = (double)__uint_as_float(a.y); z1 = (double)b.x; d1 = (double)__uint_as_float(b.y);
}
__device__ __forceinline__ double node_scale(const Node64*, double z, double) { return z; }
__device__ __forceinline__ double node_scale(const Node32*, double z, double zq) { return z * zq; }

// What the first half of a term hands to the second half (carried across one step of the theta pipeline).
template <typename LosT>
struct Mid {
  double u, z, m1, fz;
  LosT q0, q1;
  bool ok;
};

__device__ __forceinline__ bool lt(double a, double b) { return a < b; }

// LOS node loads.  From global memory they are volatile asm: the load stays in the pipeline stage that computes
// its address (the compiler would otherwise sink it next to its use, one stage later, and expose the L2 latency).
template <bool GLOBAL>
__device__ __forceinline__ float los_load(const float* p) {
  if (!GLOBAL) return *p;
  float v;
  asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}
template <bool GLOBAL>
__device__ __forceinline__ double los_load(const double* p) {
  if (!GLOBAL) return *p;
  double v;
  asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

// First half of one (theta, sample) term: u -> z by cubic Hermite on the per-theta table, source-frame masses,
// support tests, and the loads of the two line-of-sight nodes around z.  `lrow` points at the sample's LOS row
// (global memory) or at the all-sky table (shared memory).  No branch, no warp-synchronous operation.
template <typename NodeT, typename LosT, bool GLOBAL>
__device__ __forceinline__ void term_head(const double* __restrict__ tc, const NodeT* __restrict__ tab, double2 A,
                                          double m2z, const LosT* __restrict__ lrow, double inv_dz, double los_zmax,
                                          double zq, int bmax, Mid<LosT>& o) {
  const double u0 = A.x * tc[C_H];
  bool ok = u0 < tc[C_UMAX];  // false for NaN (samples marked dead by the preparation kernel)
  const double u = ok ? u0 : 0.0;
  const double th = fma(u, tc[C_INVDU], -0.5);
  double tm = th + KM[K_MAGIC];
  const int m = __double2loint(tm);  // round(t - 1/2): floor(t) except on exact integers, where f = 1 gives the same z
  tm -= KM[K_MAGIC];
  const double f = fma(u, tc[C_INVDU], -tm);
  double z0, d0, z1, d1;
  load_nodes(tab, m, z0, d0, z1, d1);
  const double dl = z1 - z0;
  const double sd = d0 + d1;
  const double c3 = fma(-2.0, dl, sd);
  const double c2 = fma(3.0, dl, -(sd + d0));
  const double z = node_scale(tab, fma(f, fma(f, fma(f, c3, c2), d0), z0), zq);
  const double rx = rcp_fast(1.0 + z);
  const double m1 = A.y * rx, m2 = m2z * rx;
  ok = ok & lt(z, los_zmax) & (m1 > tc[C_MMIN]) & (m1 <= tc[C_MMAX]) & (m2 >= tc[C_MMIN]);
  // line-of-sight prior: the two nodes around z (index clamped for dead samples beyond the table)
  double tb = fma(z, inv_dz, -0.5) + KM[K_MAGIC];
  const int b = min(__double2loint(tb), bmax);
  tb -= KM[K_MAGIC];
  o.fz = fma(z, inv_dz, -tb);
  o.q0 = los_load<GLOBAL>(lrow + b);
  o.q1 = los_load<GLOBAL>(lrow + b + 1);
  o.u = u; o.z = z; o.m1 = m1; o.ok = ok;
}

// Second half: population, rate, Jacobian and the LOS interpolation.  C = (ln m1z, ln(m2z/m1z)),
// P = -ln pi - ln m1z - shift.  Returns the weight relative to the segment shift (0 when dead).
template <typename LosT>
__device__ __forceinline__ double term_tail(const double* __restrict__ tc, const MathTables& mt, double2 C, double P,
                                            const Mid<LosT>& h, bool& live) {
  const double x = 1.0 + h.z;
  const double lx = log_fast(x, mt.logtab);
  const double t1 = C.x - lx;  // ln m1
  const double c = fma(tc[C_GM1], lx, fma(tc[C_BETA], C.y, P));
  // lambda = 1 / lambda = 0: CPL / CG is -inf, the clamped exponential returns e^-700 (~1e-304, nothing)
  const double y = fma(h.m1, tc[C_INVSIG], tc[C_NMUSIG]);
  const double num = exp_fast<true>(fma(tc[C_NALPHA], t1, c + tc[C_CPL]), mt.exptab) +
                     exp_fast<true>(fma(-0.5 * y, y, c + tc[C_CG]), mt.exptab);
  const double e1 = exp_fast<false>(fma(tc[C_NBP1], t1, tc[C_E1C]), mt.exptab);
  const double e2 = exp_fast<false>(fma(tc[C_GK], lx, tc[C_E2C]), mt.exptab);
  const double x2 = x * x;
  const double rE = rsqrt_fast(fma(tc[C_OM] * x2, x, tc[C_OL]));
  double den = fma(x2, rE, h.u);                   // u + x^2/E
  den *= fma(-tc[C_SGN], e1, tc[C_SGN]);           // sign(beta+1) (1 - e1)
  den *= 1.0 + e2;
  const double q0 = widen(h.q0), q1 = widen(h.q1);
  const double plos = fma(h.fz, q1 - q0, q0);
  const double w = num * plos * rcp_fast(den);
  const bool ok = h.ok & (plos > 0.0) & lt(w, CUDART_INF);  // also rejects NaN from a vanishing denominator
  live = ok;
  return ok ? w : 0.0;
}

// Sums of four per-lane values over the warp in a fixed order: (a0, a1) belong to one theta, (b0, b1) to another.
// Returns the total of a0 on lane 0, a1 on lane 8, b0 on lane 16, b1 on lane 24 (6 shuffles instead of 20).
__device__ __forceinline__ double warp_sum4(double a0, double a1, double b0, double b1, int lane) {
  const unsigned FULL = 0xffffffffu;
  const bool up = (lane & 16) != 0;
  double k0 = up ? b0 : a0, k1 = up ? b1 : a1;
  k0 += __shfl_xor_sync(FULL, up ? a0 : b0, 16);
  k1 += __shfl_xor_sync(FULL, up ? a1 : b1, 16);
  const bool up8 = (lane & 8) != 0;
  double k = up8 ? k1 : k0;
  k += __shfl_xor_sync(FULL, up8 ? k0 : k1, 8);
  k += __shfl_xor_sync(FULL, k, 4);
  k += __shfl_xor_sync(FULL, k, 2);
  k += __shfl_xor_sync(FULL, k, 1);
  return k;
}

// index of the lowest set bit, which is then cleared (-1 when empty)
__device__ __forceinline__ int pop_lowest(unsigned& mask) {
  if (!mask) return -1;
  const int j = __ffs(mask) - 1;
  mask &= mask - 1;
  return j;
}

template <typename NodeT, typename LosT, bool INJ>
__global__ void __launch_bounds__(NTHREADS, 1) reweight_kernel(const ReweightParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ unsigned s_item;
  typedef typename std::conditional<INJ, double, LosT>::type RowT;  // the all-sky table is f64
  const SmemLayout L = smem_layout(p.T, p.Mp, sizeof(NodeT), INJ, p.n_z);
  MathTables& mt = *reinterpret_cast<MathTables*>(smem + L.math);
  double* s_tc = reinterpret_cast<double*>(smem + L.tconst);
  double* s_acc = reinterpret_cast<double*>(smem + L.acc);
  int* s_cnt = reinterpret_cast<int*>(smem + L.cnt);
  double2* s_A = reinterpret_cast<double2*>(smem + L.A);
  double* s_m2z = reinterpret_cast<double*>(smem + L.m2z);
  double2* s_C = reinterpret_cast<double2*>(smem + L.C);
  double* s_P = reinterpret_cast<double*>(smem + L.P);
  int32_t* s_row = reinterpret_cast<int32_t*>(smem + L.row);
  double* s_allsky = reinterpret_cast<double*>(smem + L.allsky);
  NodeT* s_tab = reinterpret_cast<NodeT*>(smem + L.tab);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int T = p.T, Mp = p.Mp;
  init_math_tables(mt, tid);
  if (INJ) {
    const double* a = reinterpret_cast<const double*>(p.los);
    for (int i = tid; i < p.n_z; i += NTHREADS) s_allsky[i] = a[i];
  }
  const unsigned n_items = (unsigned)p.n_groups * (unsigned)p.n_tiles;
  const int bmax = p.n_z - 2;
  const double inv_dz = p.inv_dz, los_zmax = p.los_zmax, zq = p.tab_zq;
  int cur_tile = -1;

  for (;;) {
    __syncthreads();
    if (tid == 0) s_item = atomicAdd(p.unit_counter, 1u);
    __syncthreads();
    const unsigned item = s_item;
    if (item >= n_items) break;
    const int group = (int)(item / (unsigned)p.n_tiles);
    const int tile = (int)(item - (unsigned)group * (unsigned)p.n_tiles);
    const int t0 = tile * T;
    const int nt = min(T, p.n_theta - t0);
    if (tile != cur_tile) {
      // stage the tile's tables and constants (16-byte copies; rows are contiguous in global memory)
      const uint4* src = reinterpret_cast<const uint4*>(reinterpret_cast<const NodeT*>(p.tab) + (size_t)t0 * Mp);
      uint4* dst = reinterpret_cast<uint4*>(s_tab);
      const int n16 = (int)(((size_t)nt * Mp * sizeof(NodeT)) / 16);
      for (int i = tid; i < n16; i += NTHREADS) dst[i] = src[i];
      for (int i = tid; i < nt * NCONST; i += NTHREADS) s_tc[i] = p.tconst[(size_t)t0 * NCONST + i];
      cur_tile = tile;
    }
    for (int i = tid; i < NWARPS * T * 2; i += NTHREADS) s_acc[i] = 0.0;
    for (int i = tid; i < NWARPS * T; i += NTHREADS) s_cnt[i] = 0;
    __syncthreads();

    const int seg_lo = p.group_off[group], seg_hi = p.group_off[group + 1];
    for (int seg = seg_lo; seg < seg_hi; ++seg) {
      const int64_t s0 = p.seg_off[seg], s1 = p.seg_off[seg + 1];
      for (int64_t c0 = s0; c0 < s1; c0 += CHUNK) {
        const int n = (int)min((int64_t)CHUNK, s1 - c0);
        // stage the chunk (coalesced); slots past the end are dead
#pragma unroll
        for (int k = 0; k < SPT; ++k) {
          const int i = tid + k * NTHREADS;
          const bool in = i < n;
          const int64_t g = c0 + i;
          s_A[i] = make_double2(in ? p.dLc[g] : CUDART_NAN, in ? p.m1z[g] : 1.0);
          s_m2z[i] = in ? p.m2z[g] : 1.0;
          s_C[i] = make_double2(in ? p.L1[g] : 0.0, in ? p.Q[g] : 0.0);
          s_P[i] = in ? p.P[g] : 0.0;
          if (!INJ) {
            const int32_t r = in ? p.row[g] : 0;
            s_row[i] = ((unsigned)r < (unsigned)p.n_rows) ? r : 0;  // out-of-range rows are dead (dLc = NaN)
          }
        }
        __syncthreads();
        // Samples stay in shared memory (read where used: registers go to the interleaved chains instead);
        // a thread keeps only the address of each of its samples' LOS rows.
        const RowT* lrow[SPT];
        double dmin = CUDART_INF;  // smallest d_L of the warp's samples: a whole-warp range test per theta
#pragma unroll
        for (int k = 0; k < SPT; ++k) {
          const int i = tid + k * NTHREADS;
          if (INJ) lrow[k] = reinterpret_cast<const RowT*>(s_allsky);
          else lrow[k] = reinterpret_cast<const RowT*>(p.los) + (size_t)s_row[i] * (size_t)p.n_z;
          dmin = fmin(dmin, s_A[i].x);  // fmin drops the NaN of dead samples
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dmin = fmin(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        // theta points of the tile for which at least one sample of this warp lies inside the table
        // (none for warps entirely past the ragged tail)
        unsigned todo = __ballot_sync(0xffffffffu, lane < nt && dmin * s_tc[min(lane, nt - 1) * NCONST + C_H] <
                                                                    s_tc[min(lane, nt - 1) * NCONST + C_UMAX]);
        // Software pipeline over the theta points: the first half of the next point (table look-up, LOS loads)
        // is issued together with the second half of the current one, so its latencies hide behind FP64 work.
        int ja = pop_lowest(todo);
        if (ja >= 0) {
          Mid<RowT> cur[SPT], nxt[SPT];
#pragma unroll
          for (int k = 0; k < SPT; ++k) {
            const int i = tid + k * NTHREADS;
            term_head<NodeT, RowT, !INJ>(s_tc + ja * NCONST, s_tab + (size_t)ja * Mp, s_A[i], s_m2z[i], lrow[k], inv_dz,
                                   los_zmax, zq, bmax, cur[k]);
          }
          for (;;) {
            const int jb = pop_lowest(todo);
            const int jh = jb >= 0 ? jb : ja;  // (a redundant look-up when the list ends on an odd count)
            double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
            int cnt = 0;
            {
              const double* tch = s_tc + jh * NCONST;
              const double* tct = s_tc + ja * NCONST;
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                const int i = tid + k * NTHREADS;
                term_head<NodeT, RowT, !INJ>(tch, s_tab + (size_t)jh * Mp, s_A[i], s_m2z[i], lrow[k], inv_dz, los_zmax, zq,
                                       bmax, nxt[k]);
              }
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                const int i = tid + k * NTHREADS;
                bool live;
                const double w = term_tail<RowT>(tct, mt, s_C[i], s_P[i], cur[k], live);
                a0 += w;
                a1 = fma(w, w, a1);
                cnt += live ? 1 : 0;
              }
            }
            const int jc = pop_lowest(todo);
            {
              // (when the list ends on an odd count this second step runs on a repeated point and is discarded:
              // a branch here would let the compiler sink the loads of the first step behind it)
              const bool second = jb >= 0;
              const int jh2 = jc >= 0 ? jc : jh;
              const double* tch = s_tc + jh2 * NCONST;
              const double* tct = s_tc + jh * NCONST;
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                const int i = tid + k * NTHREADS;
                term_head<NodeT, RowT, !INJ>(tch, s_tab + (size_t)jh2 * Mp, s_A[i], s_m2z[i], lrow[k], inv_dz,
                                             los_zmax, zq, bmax, cur[k]);
              }
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                const int i = tid + k * NTHREADS;
                bool live;
                double w = term_tail<RowT>(tct, mt, s_C[i], s_P[i], nxt[k], live);
                live = live & second;
                w = live ? w : 0.0;
                b0 += w;
                b1 = fma(w, w, b1);
                cnt += live ? 0x10000 : 0;
              }
            }
            cnt = __reduce_add_sync(0xffffffffu, cnt);
            if (cnt) {  // warp-uniform
              const double k = warp_sum4(a0, a1, b0, b1, lane);
              if ((lane & 7) == 0) {
                const int j = (lane & 16) ? jb : ja;
                if (j >= 0) {
                  s_acc[(warp * T + j) * 2 + ((lane >> 3) & 1)] += k;
                  if ((lane & 8) == 0) s_cnt[warp * T + j] += (lane & 16) ? (cnt >> 16) : (cnt & 0xffff);
                }
              }
            }
            if (jc < 0) break;
            ja = jc;
          }
        }
        __syncthreads();
      }
      // segment complete: combine the warps' partials in a fixed order and write them out
      if (tid < nt) {
        double a = 0.0, b = 0.0;
        int c = 0;
        for (int w = 0; w < NWARPS; ++w) {
          a += s_acc[(w * T + tid) * 2];
          b += s_acc[(w * T + tid) * 2 + 1];
          c += s_cnt[w * T + tid];
          s_acc[(w * T + tid) * 2] = 0.0;
          s_acc[(w * T + tid) * 2 + 1] = 0.0;
          s_cnt[w * T + tid] = 0;
        }
        const size_t o = (size_t)(t0 + tid) * (size_t)p.n_seg + (size_t)seg;
        p.out_w[2 * o] = a;
        p.out_w[2 * o + 1] = b;
        p.out_n[o] = c;
      }
      // (the barrier after the next chunk's staging orders this reset before the next accumulation)
    }
  }
}

template <typename NodeT, typename LosT, bool INJ>
int launch_one(const ReweightParams& p, int n_blocks, size_t smem, cudaStream_t s) {
  reweight_kernel<NodeT, LosT, INJ><<<n_blocks, NTHREADS, smem, s>>>(p);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

template <typename NodeT, typename LosT, bool INJ>
int configure_one(int smem_optin) {
  return cudaFuncSetAttribute(reweight_kernel<NodeT, LosT, INJ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              smem_optin) == cudaSuccess ? 0 : -1;
}

}  // namespace

size_t reweight_smem_bytes(int T, int Mp, gwc_prec tab_prec, bool inj, int n_z) {
  return smem_layout(T, Mp, tab_prec == GWC_F64 ? sizeof(Node64) : sizeof(Node32), inj, n_z).total;
}

int reweight_max_T(int Mp, gwc_prec tab_prec, bool inj, int n_z, int smem_optin) {
  int best = 0;
  for (int T = 1; T <= MAX_T; ++T)
    if (reweight_smem_bytes(T, Mp, tab_prec, inj, n_z) + SMEM_RESERVE <= (size_t)smem_optin) best = T;
  return best;
}

int reweight_configure(int smem_optin) {
  smem_optin -= SMEM_RESERVE;  // room for the kernel's static shared memory
  int rc = 0;
  rc |= configure_one<Node64, double, false>(smem_optin);
  rc |= configure_one<Node64, float, false>(smem_optin);
  rc |= configure_one<Node32, double, false>(smem_optin);
  rc |= configure_one<Node32, float, false>(smem_optin);
  rc |= configure_one<Node64, double, true>(smem_optin);
  rc |= configure_one<Node32, double, true>(smem_optin);
  return rc;
}

int launch_reweight(const ReweightParams& p, gwc_prec tab_prec, gwc_prec los_prec, bool inj, int n_blocks,
                    cudaStream_t s) {
  const size_t smem = reweight_smem_bytes(p.T, p.Mp, tab_prec, inj, p.n_z);
  if (inj) {
    return tab_prec == GWC_F64 ? launch_one<Node64, double, true>(p, n_blocks, smem, s)
                               : launch_one<Node32, double, true>(p, n_blocks, smem, s);
  }
  if (tab_prec == GWC_F64)
    return los_prec == GWC_F64 ? launch_one<Node64, double, false>(p, n_blocks, smem, s)
                               : launch_one<Node64, float, false>(p, n_blocks, smem, s);
  return los_prec == GWC_F64 ? launch_one<Node32, double, false>(p, n_blocks, smem, s)
                             : launch_one<Node32, float, false>(p, n_blocks, smem, s);
}

}  // namespace gwc
