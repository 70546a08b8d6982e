// reweight.cu -- A3/A5: the fused re-weighting kernel over (theta, segment, sample).
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
// Mapping.  A persistent CTA per SM takes work items (segment group, theta tile) from an atomic counter,
// group-major so that CTAs running at the same time share the group's samples and LOS rows in L2.  The
// tile's inverse-cosmology tables live in shared memory.  Lanes are samples: a warp takes a block of
// 32 * SPT consecutive samples of the segment straight from global memory into registers (coalesced; no
// shared-memory staging, no barrier per block) and loops over the tile's theta points, software-pipelined:
// the table look-up and the LOS loads of the next point are issued with the FP64 tail of the current one.
// The per-theta constants are warp-uniform and come from the constant bank (uniform loads feeding the FP64
// instructions directly: no shared-memory traffic, no vector registers); the bank holds KT_THETA points, so
// a batch is processed in launches of at most that many.  What bounds the kernel besides the FP64 pipe is the
// shared-memory pipe (one wavefront per clock per SM): the random look-ups of the exp / log tables are
// conflict-free by replication (math64.cuh), leaving the Hermite node gathers as the only conflicted reads.
// Per-(warp, theta) partial sums live in shared memory and are combined in a fixed order at the end of a
// segment: no floating-point atomics, results are bitwise reproducible.
#include <math_constants.h>

#include <mutex>
#include <type_traits>

#include "gwc_internal.h"
#include "math64.cuh"

namespace gwc {

namespace {

constexpr int SMEM_RESERVE = 256;  // static shared memory of the kernel + slack
constexpr int BLK = 32 * SPT;      // samples one warp holds in registers at a time

// per-theta constants of the current launch (A2), read with uniform loads
__constant__ double KT[KT_THETA * NCONST];

// The constant bank is one per device, shared by every context (and stream) of the process.  Launches that use it are
// therefore chained across streams: a launch waits (cudaStreamWaitEvent) for the event recorded behind the previous
// launch whenever that one went to another stream, so no copy into the bank can overtake a kernel still reading it.
// Kernels of this size fill the GPU, so nothing is lost by running them one after the other (gwc.h, "Streams").
constexpr int MAX_DEVICES = 64;
struct BankGuard {
  std::mutex mu;
  cudaEvent_t last = nullptr;     // recorded behind the last kernel that read the bank
  cudaStream_t last_stream = nullptr;
  bool used = false;
};
BankGuard g_bank[MAX_DEVICES];

struct SmemLayout {
  size_t math, acc, cnt, np, carry, carryn, lead, leadn, allsky, ftab, tab, total;
};

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

// tabs: z(u) tables per tile (T, or 1 when the whole batch has one Omega_m and so one table)
__host__ __device__ inline SmemLayout smem_layout(int T, int tabs, int Mp, size_t node_bytes, bool inj, int n_z, bool pix,
                                                   bool mp) {
  SmemLayout L;
  size_t o = 0;
  L.math = o;   o = align16(o + sizeof(MathTables));
  // (two sets of everything: a warp may start the next segment while the slowest finish this one)
  L.acc = o;    o = align16(o + sizeof(double) * NWARPS * T * 2 * 2);
  L.cnt = o;    o = align16(o + sizeof(int) * NWARPS * T * 2);
  // pixel-cut mode only: passing pixels; the run a block leaves open (W, Q, n); the run open at the range start
  L.np = o;     o = align16(o + (pix ? sizeof(int) * NWARPS * T * 2 : 0));
  L.carry = o;  o = align16(o + (pix ? sizeof(double) * NWARPS * T * 2 * 2 : 0));
  L.carryn = o; o = align16(o + (pix ? sizeof(int) * NWARPS * T * 2 : 0));
  L.lead = o;   o = align16(o + (pix ? sizeof(double) * NWARPS * T * 2 * 2 : 0));
  L.leadn = o;  o = align16(o + (pix ? sizeof(int) * NWARPS * T * 2 : 0));
  L.allsky = o; o = align16(o + (inj ? sizeof(double) * n_z : 0));
  L.ftab = o;   o = align16(o + (mp ? sizeof(Node64) * (size_t)T * MF_PITCH : 0));   // MULTIPEAK: F(m1) tables
  L.tab = o;    o = align16(o + node_bytes * (size_t)tabs * Mp);
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
  double m2;   // MULTIPEAK only (unused fields vanish)
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
template <typename NodeT, typename LosT, bool GLOBAL, bool MP>
__device__ __forceinline__ void term_head(const double* __restrict__ tc, const NodeT* __restrict__ tab, double2 A,
                                          double m2z, const LosT* __restrict__ lrow, double inv_dz, double los_zmax,
                                          double zq, int bmax, Mid<LosT>& o, int* chk, int Mp) {
  const double u0 = A.x * tc[C_H];
  bool ok = u0 < tc[C_UMAX];  // false for NaN (samples marked dead by the preparation kernel)
  const double u = ok ? u0 : 0.0;
  const double th = fma(u, tc[C_INVDU], -0.5);
  double tm = th + KM[K_MAGIC];
  const int m = __double2loint(tm);  // round(t - 1/2): floor(t) except on exact integers, where f = 1 gives the same z
  tm -= KM[K_MAGIC];
  const double f = fma(u, tc[C_INVDU], -tm);
  double z0, d0, z1, d1;
  GWC_DEV_CHECK(chk, m >= 0 && m <= Mp - 2, FLAG_CHK_TABLE);
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
  GWC_DEV_CHECK(chk, b >= 0 && b <= bmax, FLAG_CHK_LOS);
  o.q0 = los_load<GLOBAL>(lrow + b);
  o.q1 = los_load<GLOBAL>(lrow + b + 1);
  o.u = u; o.z = z; o.m1 = m1; o.ok = ok;
  if (MP) o.m2 = m2;
}

// Second half: population, rate, Jacobian and the LOS interpolation.  C = (ln m1z, ln(m2z/m1z)),
// P = -ln pi - ln m1z - shift.  Returns the weight relative to the segment shift (0 when dead).
// MULTIPEAK (R33-R36): a second Gaussian peak in the numerator; the normaliser of p(m2 | m1) inside the
// smoothing window from the per-theta table `ftab` of |F|(m1) = |beta+1| C(m1) / (S(m1) m1^(beta+1)) (S(m1) of p(m1)
// cancels against the one in C), above it sign(beta+1) (1 - e1) with the window's integral folded into E1C; and
// 1 / S(m2) = 1 + exp(dm (2 m' - dm) / (m' (m' - dm))), m' = m2 - mmin, in the denominator.
template <typename LosT, bool MP>
__device__ __forceinline__ double term_tail(const double* __restrict__ tc, const double2* __restrict__ logtab,
                                            const double* __restrict__ exptab, const Node64* __restrict__ ftab,
                                            double2 C, double P, const Mid<LosT>& h, bool& live, int* chk) {
  const double x = 1.0 + h.z;
  const double lx = log_fast(x, logtab);
  const double t1 = C.x - lx;  // ln m1
  const double c = fma(tc[C_GM1], lx, fma(tc[C_BETA], C.y, P));
  // lambda = 1 / lambda = 0: CPL / CG is -inf, the clamped exponential returns e^-700 (~1e-304, nothing)
  const double y = fma(h.m1, tc[C_INVSIG], tc[C_NMUSIG]);
  double num = exp_fast<true>(fma(tc[C_NALPHA], t1, c + tc[C_CPL]), exptab) +
               exp_fast<true>(fma(-0.5 * y, y, c + tc[C_CG]), exptab);
  const double e1 = exp_fast<false>(fma(tc[C_NBP1], t1, tc[C_E1C]), exptab);
  const double e2 = exp_fast<false>(fma(tc[C_GK], lx, tc[C_E2C]), exptab);
  const double x2 = x * x;
  const double rE = rsqrt_fast(fma(tc[C_OM] * x2, x, tc[C_OL]));
  double den = fma(x2, rE, h.u);                   // u + x^2/E
  double F = fma(-tc[C_SGN], e1, tc[C_SGN]);       // sign(beta+1) (1 - e1)
  bool ok = h.ok;
  if (MP) {
    const double yl = fma(h.m1, tc[C_INVSIG2], tc[C_NMUSIG2]);
    num += exp_fast<true>(fma(-0.5 * yl, yl, c + tc[C_CG2]), exptab);
    // m1 inside the smoothing window: cubic Hermite on the table (lanes outside read a clamped interval, unused)
    const double m1p = h.m1 - tc[C_MMIN];
    double tm = fma(m1p, tc[C_FIDX], -0.5) + KM[K_MAGIC];
    const int k = max(0, min(__double2loint(tm), MF_NODES - 2));
    const double f = fma(m1p, tc[C_FIDX], -(double)k);
    GWC_DEV_CHECK(chk, k >= 0 && k <= MF_NODES - 2, FLAG_CHK_FTAB);
    const double2* q = reinterpret_cast<const double2*>(ftab + k);
    const double2 a = q[0], b = q[1];
    const double dl = b.x - a.x, sd = a.y + b.y;
    const double c3 = fma(-2.0, dl, sd), c2 = fma(3.0, dl, -(sd + a.y));
    const double Fin = fma(f, fma(f, fma(f, c3, c2), a.y), a.x);
    F = m1p < tc[C_DM] ? Fin : F;
    // 1 / S(m2)
    const double m2p = h.m2 - tc[C_MMIN];
    const bool win2 = m2p < tc[C_DM];
    const double E = tc[C_DM] * fma(2.0, m2p, -tc[C_DM]) * rcp_fast(m2p * (m2p - tc[C_DM]));
    ok = ok & !(win2 & !(E <= 250.0));   // a smoothing factor below e^-250 is zero (R35); also m2 = mmin and NaN
    const double f2 = exp_fast<true>(win2 ? E : -700.0, exptab);
    den *= 1.0 + f2;
  }
  den *= F;
  den *= 1.0 + e2;
  const double q0 = widen(h.q0), q1 = widen(h.q1);
  const double plos = fma(h.fz, q1 - q0, q0);
  const double w = num * plos * rcp_fast(den);
  ok = ok & (plos > 0.0) & lt(w, CUDART_INF);  // also rejects NaN from a vanishing denominator
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

// ---- per-pixel effective-sample cut (Eq. 8; R25) -------------------------------------
// A pixel is a maximal run of consecutive samples of the segment with the same sample_row.  Pixel-cut mode works on
// the pixel-aligned copy of the samples (pack.cu: every run starts at an even position and has an even length, odd
// runs end on a dead slot) and a lane owns the SPT = 2 CONSECUTIVE positions 2 lane, 2 lane + 1 of the warp's block:
// a lane belongs to exactly one run, and the per-(theta, pixel) sums are one segmented scan over the 32 lanes.
// PixShape is the run structure of the block (the same for every theta).
struct PixShape {
  bool tail;            // the lane's run ends on this lane
  bool lead;            // ... and it began before this warp's range of the segment: the segment-end stitch decides
  bool left;            // the lane's run began before the block
  int reach;            // lanes back to the first lane of the run inside the block
  int nsteps;           // scan steps the block needs (warp-uniform)
  unsigned runm;        // lanes of the run up to this one (live counts)
  bool blk_left;        // lane 0's run is open to the left: the carry of the previous block enters (warp-uniform)
  bool last_open;       // lane 31's run continues in the next block (warp-uniform)
  bool interior;        // the whole block lies inside one run that began earlier and goes on (warp-uniform)
  bool has_head;        // a run starts in the block (warp-uniform)
};

__device__ __forceinline__ void pix_shape(PixShape& ps, bool in, bool head, bool tail, bool lead_open, int lane) {
  const unsigned FULL = 0xffffffffu;
  const unsigned hall = __ballot_sync(FULL, head), inall = __ballot_sync(FULL, in);
  const unsigned le = 0xffffffffu >> (31 - lane);   // lanes <= this one
  const unsigned hm = hall & le;
  ps.left = hm == 0;
  const int first = ps.left ? 0 : 31 - __clz(hm);
  ps.reach = lane - first;
  ps.runm = le & (0xffffffffu << first);
  ps.tail = tail;
  ps.lead = lead_open && ps.left;
  const int maxd = __reduce_max_sync(FULL, in ? ps.reach : 0);
  ps.nsteps = maxd == 0 ? 0 : 32 - __clz(maxd);
  ps.blk_left = (inall & 1u) && !(hall & 1u);
  ps.last_open = (__ballot_sync(FULL, in && !tail) >> 31) != 0;
  ps.interior = hall == 0 && inall == FULL && ps.last_open;
  ps.has_head = hall != 0;
}

// From the per-sample weights of TWO theta points (a, b: two independent chains, so that the shuffle latencies of one
// hide behind the other) to what the passing pixels add to this lane's sums.  No branch: the scan always takes its
// five steps (a lane whose run does not reach that far adds nothing).
//   in : w[k], live[k]; carry = (W, Q, n) of the run left open by the previous block (slot of this warp and theta)
//        lead: where the run that was open at the start of the warp's range is put when it ends here
//        second = false: b is a repeated point (odd theta count), its slots are left alone
//   out: cW, cQ, cn (weights, squared weights, live samples of the passing pixel that ends on this lane), cp = 0 | 1
struct PixSlot {
  double* carryWQ;
  int* carryN;
  double* leadWQ;
  int* leadN;
};
__device__ __forceinline__ void pix_reduce2(const PixShape& ps, const double* wa, const bool* la, const double* wb,
                                            const bool* lb, bool second, double neff_min, PixSlot sa, PixSlot sb,
                                            int lane, double& aW, double& aQ, int& an, int& ap, double& bW, double& bQ,
                                            int& bn, int& bp) {
  const unsigned FULL = 0xffffffffu;
  double XA = wa[0] + wa[1], QA = fma(wa[1], wa[1], wa[0] * wa[0]);
  double XB = wb[0] + wb[1], QB = fma(wb[1], wb[1], wb[0] * wb[0]);
  __syncwarp();        // the carry slots were written by other lanes (previous block of this warp)
  // the run open at the block's start continues on lane 0 (the slots hold zeros when there is none)
  const int inNA = ps.left ? *sa.carryN : 0, inNB = ps.left ? *sb.carryN : 0;
  if (lane == 0) {
    XA += sa.carryWQ[0];
    QA += sa.carryWQ[1];
    XB += sb.carryWQ[0];
    QB += sb.carryWQ[1];
  }
  // inclusive segmented scan over the lanes
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double tA = __shfl_up_sync(FULL, XA, o), uA = __shfl_up_sync(FULL, QA, o);
    const double tB = __shfl_up_sync(FULL, XB, o), uB = __shfl_up_sync(FULL, QB, o);
    if (ps.reach >= o) {
      XA += tA;
      QA += uA;
      XB += tB;
      QB += uB;
    }
  }
  const unsigned a0 = __ballot_sync(FULL, la[0]), a1 = __ballot_sync(FULL, la[1]);
  const unsigned b0 = __ballot_sync(FULL, lb[0]), b1 = __ballot_sync(FULL, lb[1]);
  const int nA = __popc(a0 & ps.runm) + __popc(a1 & ps.runm) + inNA;
  const int nB = __popc(b0 & ps.runm) + __popc(b1 & ps.runm) + inNB;
  // what the next block inherits: lane 31 holds the sums of the run that stays open
  __syncwarp();
  if (lane == 31) {
    sa.carryWQ[0] = ps.last_open ? XA : 0.0;
    sa.carryWQ[1] = ps.last_open ? QA : 0.0;
    *sa.carryN = ps.last_open ? nA : 0;
    if (second) {
      sb.carryWQ[0] = ps.last_open ? XB : 0.0;
      sb.carryWQ[1] = ps.last_open ? QB : 0.0;
      *sb.carryN = ps.last_open ? nB : 0;
    }
  }
  // began in an earlier warp's range: the segment-end stitch decides (one lane of the block at most)
  if (ps.tail && ps.lead) {
    sa.leadWQ[0] = XA; sa.leadWQ[1] = QA; *sa.leadN = nA;
    if (second) { sb.leadWQ[0] = XB; sb.leadWQ[1] = QB; *sb.leadN = nB; }
  }
  const bool own = ps.tail && !ps.lead;
  const bool pa = own && XA > 0.0 && XA * XA >= neff_min * QA;
  const bool pb = own && second && XB > 0.0 && XB * XB >= neff_min * QB;
  aW = pa ? XA : 0.0; aQ = pa ? QA : 0.0; an = pa ? nA : 0; ap = pa ? 1 : 0;
  bW = pb ? XB : 0.0; bQ = pb ? QB : 0.0; bn = pb ? nB : 0; bp = pb ? 1 : 0;
}

// One sample's theta-independent values, held in registers while the warp loops over the tile's theta points.
template <typename RowT>
struct Sample {
  double2 A;  // (d_L or NaN when dead, m1z)
  double m2z;
  double2 C;  // (ln m1z, ln(m2z/m1z))
  double P;   // -ln pi - ln m1z - shift
  const RowT* lrow;
};

// TEAMS: short segments share the CTA (chosen by the host for catalogues of short events; see launch_reweight).
// ODD: a theta list that ends on an odd count takes a tail-only path instead of a discarded pipeline step (chosen by
// the host for batches of a few theta points, the sampler's one-point-per-call pattern: 0.79 -> 0.51 ms for one
// theta on the O5 catalogue; compiled into the batch kernel the branch costs it 1.7 %).
template <typename NodeT, typename LosT, bool INJ, bool PIX, bool TEAMS, bool ODD, bool MP>
__global__ void __launch_bounds__(NTHREADS, 1) reweight_kernel(const ReweightParams p) {
  constexpr int NC = MP ? NCONST_MP : NCONST;   // row length of the constant bank
  // ASYNC: no barrier between segments.  The sums of consecutive segments go to alternating buffers; the last warp to
  // finish a segment combines it (fixed warp order) while the others are already on the next one, and the blocks are
  // dealt round-robin across segment boundaries, so the warps' loads even out over the group.
  // (Pixel-cut mode keeps contiguous ranges per warp; what evens out there is the cost of its blocks, which differs
  // between blocks inside one pixel and blocks full of pixel ends.)
  constexpr bool ASYNC = !TEAMS;
  constexpr int NBUF = 2;
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ unsigned s_item;
  typedef typename std::conditional<INJ, double, LosT>::type RowT;  // the all-sky table is f64
  const SmemLayout L = smem_layout(p.T, p.shared_tab ? 1 : p.T, p.Mp, sizeof(NodeT), INJ, p.n_z, PIX, MP);
  MathTables& mt = *reinterpret_cast<MathTables*>(smem + L.math);
  double* s_acc = reinterpret_cast<double*>(smem + L.acc);
  int* s_cnt = reinterpret_cast<int*>(smem + L.cnt);
  int* s_np = reinterpret_cast<int*>(smem + L.np);
  double* s_carry = reinterpret_cast<double*>(smem + L.carry);
  int* s_carryn = reinterpret_cast<int*>(smem + L.carryn);
  double* s_lead = reinterpret_cast<double*>(smem + L.lead);
  int* s_leadn = reinterpret_cast<int*>(smem + L.leadn);
  __shared__ int s_arrive[2], s_done;  // ASYNC: warps that finished a segment (per buffer), segments combined so far
  __shared__ int s_hashead[2][NWARPS];  // pixel-cut mode: the warp's range of the segment contains a pixel start
  double* s_allsky = reinterpret_cast<double*>(smem + L.allsky);
  NodeT* s_tab = reinterpret_cast<NodeT*>(smem + L.tab);
  Node64* s_ftab = reinterpret_cast<Node64*>(smem + L.ftab);

  const unsigned FULL = 0xffffffffu;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int T = p.T, Mp = p.Mp;
  const int tstride = p.shared_tab ? 0 : Mp;   // one Omega_m in the batch: every theta of the tile reads the same table
  init_math_tables(mt, tid, NTHREADS);
  const double2* logtab = mt.logtab + (lane & (LOG_REP - 1));  // this lane's copies: conflict-free look-ups
  const double* exptab = mt.exptab + (lane & (EXP_REP - 1));
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
    const int gslot = (int)(item / (unsigned)p.n_tiles);
    const int tile = (int)(item - (unsigned)gslot * (unsigned)p.n_tiles);
#ifdef GWC_NO_ORDER
    const int group = gslot;
#else
    const int group = p.group_order[gslot];   // heaviest group first
#endif
    const int t0 = tile * T;  // first theta of the tile, relative to this launch
    const int nt = min(T, p.n_theta - t0);
    if (tile != cur_tile) {
      // stage the tile's tables (16-byte copies; rows are contiguous in global memory)
      const uint4* src =
          reinterpret_cast<const uint4*>(reinterpret_cast<const NodeT*>(p.tab) + (size_t)(p.t_begin + t0) * Mp);
      uint4* dst = reinterpret_cast<uint4*>(s_tab);
      const int n16 = (int)(((size_t)(p.shared_tab ? 1 : nt) * Mp * sizeof(NodeT)) / 16);
      for (int i = tid; i < n16; i += NTHREADS) dst[i] = src[i];
      if (MP) {
        const uint4* fsrc = reinterpret_cast<const uint4*>(p.ftab + (size_t)(p.t_begin + t0) * MF_PITCH);
        uint4* fdst = reinterpret_cast<uint4*>(s_ftab);
        for (int i = tid; i < nt * MF_PITCH; i += NTHREADS) fdst[i] = fsrc[i];
      }
      cur_tile = tile;
    }
    for (int i = tid; i < NWARPS * T * 2 * NBUF; i += NTHREADS) s_acc[i] = 0.0;
    for (int i = tid; i < NWARPS * T * NBUF; i += NTHREADS) s_cnt[i] = 0;
    if (tid == 0) {
      s_arrive[0] = 0;
      s_arrive[1] = 0;
      s_done = 0;
    }
    int rot = 0;  // ASYNC: the warp that takes the first block of the current segment
    if (PIX) {
      for (int i = tid; i < NWARPS * T * 2 * NBUF; i += NTHREADS) {
        s_carry[i] = 0.0;
        s_lead[i] = 0.0;
      }
      for (int i = tid; i < NWARPS * T * NBUF; i += NTHREADS) {
        s_np[i] = 0;
        s_carryn[i] = 0;
        s_leadn[i] = 0;
      }
    }
    __syncthreads();

    const int seg_lo = p.group_off[group], seg_hi = p.group_off[group + 1];
    for (int seg0 = seg_lo; seg0 < seg_hi;) {
      // Short segments share the CTA: when the next 2 (4) segments each fit one block per warp of a half (quarter) of
      // the CTA, the halves (quarters) take one segment each, so that no warp idles through a segment with fewer
      // blocks than the CTA has warps.
      int sh = 0;  // log2 of the number of segments taken at once
      if (TEAMS && seg0 + 2 <= seg_hi) {
        const int64_t o0 = p.seg_off[seg0], o1 = p.seg_off[seg0 + 1], o2 = p.seg_off[seg0 + 2];
        if (o1 - o0 <= (NWARPS / 2) * BLK && o2 - o1 <= (NWARPS / 2) * BLK) {
          sh = 1;
          if (seg0 + 4 <= seg_hi) {
            const int64_t o3 = p.seg_off[seg0 + 3], o4 = p.seg_off[seg0 + 4];
            if (o1 - o0 <= (NWARPS / 4) * BLK && o2 - o1 <= (NWARPS / 4) * BLK && o3 - o2 <= (NWARPS / 4) * BLK &&
                o4 - o3 <= (NWARPS / 4) * BLK)
              sh = 2;
          }
        }
      }
      const int nteam = 1 << sh;
      const int tsz = NWARPS >> sh;            // warps per team
      const int seg = seg0 + (warp / (NWARPS / 4) >> (2 - sh));   // this warp's segment
      const int wt = warp & (tsz - 1);         // this warp inside its team
      const int64_t s0 = p.seg_off[seg], s1 = p.seg_off[seg + 1];
      const int sidx = seg0 - seg_lo;
      const int buf = ASYNC ? (sidx & 1) : 0;
      double* acc_b = s_acc + buf * (NWARPS * T * 2);
      int* cnt_b = s_cnt + buf * (NWARPS * T);
      // pixel-cut mode: this segment's set of the per-(warp, theta) pixel state
      int* np_b = s_np + buf * (NWARPS * T);
      double* carry_b = s_carry + buf * (NWARPS * T * 2);
      int* carryn_b = s_carryn + buf * (NWARPS * T);
      double* lead_b = s_lead + buf * (NWARPS * T * 2);
      int* leadn_b = s_leadn + buf * (NWARPS * T);
      if (ASYNC && sidx >= 2) {
        // this buffer last held segment sidx-2: wait until it has been combined and cleared
        while (*(volatile int*)&s_done < sidx - 1) __nanosleep(PIX ? 400 : 100);   // (no issue slots burnt while waiting)
        __threadfence_block();  // the cleared buffer is seen after the release
      }
#ifdef GWC_CHECKED
      if (ASYNC && lane < nt) {   // this warp's slots of the buffer must be clear before it adds to them
        GWC_DEV_CHECK(p.flag, *(volatile double*)&acc_b[(warp * T + lane) * 2] == 0.0 &&
                                  *(volatile double*)&acc_b[(warp * T + lane) * 2 + 1] == 0.0 &&
                                  *(volatile int*)&cnt_b[warp * T + lane] == 0,
                      FLAG_CHK_HANDOFF);
      }
#endif
      // The segment's samples in blocks of BLK, dealt to the warps round-robin; no barrier until the segment ends.
      // Pixel-cut mode: each warp takes one contiguous range of whole blocks instead, so that the run a block
      // leaves open is continued by the same warp's next block; the pixels that cross from one warp's range
      // into the next are put together when the segment ends (lead / trail sums below).
      int64_t w_lo = s0 + (int64_t)(ASYNC ? ((warp - rot) & (NWARPS - 1)) : wt) * BLK, w_hi = s1, w_step = (int64_t)tsz * BLK;
      if (ASYNC) rot = (rot + (int)((s1 - s0 + BLK - 1) / BLK)) & (NWARPS - 1);
      bool lead_open = true;  // no pixel start seen yet in this warp's range
      if (PIX) {
        // (the ranges are dealt to the warps rotated by one per segment, so that the range that is one block longer
        // than the others does not always fall on the same warp)
        const int64_t nb = (s1 - s0 + BLK - 1) / BLK;
        const int rw = (warp + sidx) & (NWARPS - 1);   // this warp's range of the segment
        w_lo = s0 + nb * rw / NWARPS * BLK;
        w_hi = min(s1, s0 + nb * (rw + 1) / NWARPS * BLK);
        w_step = BLK;
      }
      if (ODD && nt == 1) {
        // One theta point (the sampler's one-point-per-call pattern): there is no theta loop to hide the loads
        // behind, so the pipeline runs across the warp's BLOCKS instead: the samples of the next block are requested
        // before the second half of the current one is computed.  (warp-uniform branch; the tile is theta t0)
        auto load_block = [&](int64_t c0, Sample<RowT>* sm) {
#pragma unroll
          for (int k = 0; k < SPT; ++k) {
            const int64_t g = c0 + k * 32 + lane;
            const bool in = g < w_hi;
            GWC_DEV_CHECK(p.flag, !in || (g >= 0 && g < p.n_samples), FLAG_CHK_SAMPLE);
            sm[k].A = make_double2(in ? p.dLc[g] : CUDART_NAN, in ? p.m1z[g] : 1.0);
            sm[k].m2z = in ? p.m2z[g] : 1.0;
            sm[k].C = make_double2(in ? p.L1[g] : 0.0, in ? p.Q[g] : 0.0);
            sm[k].P = in ? p.P[g] : 0.0;
            if (INJ) {
              sm[k].lrow = reinterpret_cast<const RowT*>(s_allsky);
            } else {
              int32_t r = in ? p.row[g] : 0;
              r = ((unsigned)r < (unsigned)p.n_rows) ? r : 0;
              sm[k].lrow = reinterpret_cast<const RowT*>(p.los) + (size_t)r * (size_t)p.n_z;
            }
          }
        };
        const double* tc1 = KT + t0 * NC;
        if (w_lo < w_hi) {
          Sample<RowT> sa[SPT], sb[SPT];
          Mid<RowT> cur[SPT];
          load_block(w_lo, sa);
#pragma unroll
          for (int k = 0; k < SPT; ++k)
            term_head<NodeT, RowT, !INJ, MP>(tc1, s_tab, sa[k].A, sa[k].m2z, sa[k].lrow, inv_dz, los_zmax, zq, bmax, cur[k],
                                             p.flag, Mp);
          double a0 = 0.0, a1 = 0.0;   // per-lane sums over the warp's blocks of this segment: one reduction at the end
          int cnt = 0;
          for (int64_t c0 = w_lo;;) {
            const int64_t cn = c0 + w_step;
            const bool more = cn < w_hi;   // warp-uniform
            if (more) load_block(cn, sb);
#pragma unroll
            for (int k = 0; k < SPT; ++k) {
              bool live;
              const double w = term_tail<RowT, MP>(tc1, logtab, exptab, s_ftab, sa[k].C, sa[k].P, cur[k], live, p.flag);
              a0 += w;
              a1 = fma(w, w, a1);
              cnt += live ? 1 : 0;
            }
            if (!more) break;
#pragma unroll
            for (int k = 0; k < SPT; ++k) {
              term_head<NodeT, RowT, !INJ, MP>(tc1, s_tab, sb[k].A, sb[k].m2z, sb[k].lrow, inv_dz, los_zmax, zq, bmax, cur[k],
                                               p.flag, Mp);
              sa[k].C = sb[k].C;
              sa[k].P = sb[k].P;
            }
            c0 = cn;
          }
          cnt = __reduce_add_sync(FULL, cnt);
          if (cnt) {
            const double k = warp_sum4(a0, a1, 0.0, 0.0, lane);
            if ((lane & 23) == 0) acc_b[(warp * T) * 2 + ((lane >> 3) & 1)] += k;
            if (lane == 0) cnt_b[warp * T] += cnt;
          }
        }
      } else
      for (int64_t c0 = w_lo; c0 < w_hi; c0 += w_step) {
        Sample<RowT> sm[SPT];
        PixShape ps;
        double dmin = CUDART_INF;  // smallest d_L of the warp's samples: a whole-warp range test per theta
        if (PIX) {
          // run structure of the block (pixel-aligned copy: the lane's two positions lie in one run)
          static_assert(!PIX || SPT == 2, "pixel-cut mode: two consecutive samples per lane");
          const int64_t g0 = c0 + 2 * lane;
          const bool in = g0 < w_hi;
          const int32_t r0 = in ? p.row[g0] : 0;
          const bool head = in && (g0 == s0 || p.row[g0 - 1] != r0);
          // (ranges end on block boundaries or on the segment's last sample, which is a tail)
          const bool tail = in && (g0 + 2 >= s1 || p.row[g0 + 2] != r0);
          pix_shape(ps, in, head, tail, lead_open, lane);
          // (no short-circuit: a vote under a branch makes ptxas treat the whole loop as divergent, and the per-theta
          // constants then come through vector loads instead of uniform ones)
          lead_open = lead_open & !ps.has_head;
        }
#pragma unroll
        for (int k = 0; k < SPT; ++k) {
          const int64_t g = PIX ? c0 + SPT * lane + k : c0 + k * 32 + lane;
          const bool in = g < w_hi;  // slots past the end are dead
          GWC_DEV_CHECK(p.flag, !in || (g >= 0 && g < p.n_samples), FLAG_CHK_SAMPLE);
          sm[k].A = make_double2(in ? p.dLc[g] : CUDART_NAN, in ? p.m1z[g] : 1.0);
          sm[k].m2z = in ? p.m2z[g] : 1.0;
          sm[k].C = make_double2(in ? p.L1[g] : 0.0, in ? p.Q[g] : 0.0);
          sm[k].P = in ? p.P[g] : 0.0;
          if (INJ) {
            sm[k].lrow = reinterpret_cast<const RowT*>(s_allsky);
          } else {
            int32_t r = in ? p.row[g] : 0;
            r = ((unsigned)r < (unsigned)p.n_rows) ? r : 0;  // out-of-range rows are dead (dLc = NaN)
            GWC_DEV_CHECK(p.flag, r >= 0 && (int64_t)r < p.n_rows, FLAG_CHK_LOS);
            sm[k].lrow = reinterpret_cast<const RowT*>(p.los) + (size_t)r * (size_t)p.n_z;
          }
          dmin = fmin(dmin, sm[k].A.x);  // fmin drops the NaN of dead samples
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dmin = fmin(dmin, __shfl_xor_sync(FULL, dmin, o));
        // theta points of the tile for which at least one sample of this warp lies inside the table
        const double* tcl = KT + (t0 + min(lane, nt - 1)) * NC;
        unsigned todo = __ballot_sync(FULL, lane < nt && dmin * tcl[C_H] < tcl[C_UMAX]);
        // every theta sees every block: open runs are carried through (a ballot: the compiler then knows the list is
        // warp-uniform and reads the constants of its points through uniform loads)
        if (PIX) todo = __ballot_sync(FULL, lane < nt);
        // Software pipeline over the theta points: the first half of the next point (table look-up, LOS loads)
        // is issued together with the second half of the current one, so its latencies hide behind FP64 work.
        // (pixel-cut mode: a block that lies inside one pixel is summed like a block of the uncut estimator; the two
        // forms of the loop are separate instantiations, so that no branch sits inside the pipeline)
        auto theta_loop = [&](auto interior_c) {
        constexpr bool plain = !PIX || decltype(interior_c)::value;
        int ja = pop_lowest(todo);
        if (ja >= 0) {
          Mid<RowT> cur[SPT], nxt[SPT];
#pragma unroll
          for (int k = 0; k < SPT; ++k)
            term_head<NodeT, RowT, !INJ, MP>(KT + (t0 + ja) * NC, s_tab + (size_t)ja * tstride, sm[k].A, sm[k].m2z, sm[k].lrow,
                                         inv_dz, los_zmax, zq, bmax, cur[k], p.flag, Mp);
          for (;;) {
            const int jb = pop_lowest(todo);
            if (ODD && jb < 0) {
              // the list ends on an odd count: only the second half of the last point is left (warp-uniform)
              double a0 = 0.0, a1 = 0.0;
              int cnt = 0;
              const double* tct = KT + (t0 + ja) * NC;
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                bool live;
                const double w = term_tail<RowT, MP>(tct, logtab, exptab, s_ftab + ja * MF_PITCH, sm[k].C, sm[k].P, cur[k], live, p.flag);
                a0 += w;
                a1 = fma(w, w, a1);
                cnt += live ? 1 : 0;
              }
              cnt = __reduce_add_sync(FULL, cnt);
              if (cnt) {
                const double k = warp_sum4(a0, a1, 0.0, 0.0, lane);
                if ((lane & 23) == 0) acc_b[(warp * T + ja) * 2 + ((lane >> 3) & 1)] += k;
                if (lane == 0) cnt_b[warp * T + ja] += cnt;
              }
              break;
            }
            const int jh = jb >= 0 ? jb : ja;  // (a redundant look-up when the list ends on an odd count)
            double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
            int cnt = 0, cntb = 0, npa = 0, npb = 0;  // (cntb, npa, npb: pixel-cut mode)
            double wa[SPT];   // (pixel-cut mode: the first point's weights wait for the second's)
            bool la[SPT];
            {
              const double* tch = KT + (t0 + jh) * NC;
              const double* tct = KT + (t0 + ja) * NC;
#pragma unroll
              for (int k = 0; k < SPT; ++k)
                term_head<NodeT, RowT, !INJ, MP>(tch, s_tab + (size_t)jh * tstride, sm[k].A, sm[k].m2z, sm[k].lrow, inv_dz,
                                             los_zmax, zq, bmax, nxt[k], p.flag, Mp);
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                wa[k] = term_tail<RowT, MP>(tct, logtab, exptab, s_ftab + ja * MF_PITCH, sm[k].C, sm[k].P, cur[k], la[k], p.flag);
                if (plain) {
                  a0 += wa[k];
                  a1 = fma(wa[k], wa[k], a1);
                  cnt += la[k] ? 1 : 0;
                }
              }
            }
            const int jc = pop_lowest(todo);
            {
              // (when the list ends on an odd count this second step runs on a repeated point and is discarded:
              // a branch here would let the compiler sink the loads of the first step behind it)
              const bool second = jb >= 0;
              const int jh2 = jc >= 0 ? jc : jh;
              const double* tch = KT + (t0 + jh2) * NC;
              const double* tct = KT + (t0 + jh) * NC;
#pragma unroll
              for (int k = 0; k < SPT; ++k)
                term_head<NodeT, RowT, !INJ, MP>(tch, s_tab + (size_t)jh2 * tstride, sm[k].A, sm[k].m2z, sm[k].lrow, inv_dz,
                                             los_zmax, zq, bmax, cur[k], p.flag, Mp);
              double wv[SPT];
              bool lv[SPT];
#pragma unroll
              for (int k = 0; k < SPT; ++k) {
                wv[k] = term_tail<RowT, MP>(tct, logtab, exptab, s_ftab + jh * MF_PITCH, sm[k].C, sm[k].P, nxt[k], lv[k], p.flag);
                lv[k] = lv[k] & second;
                wv[k] = lv[k] ? wv[k] : 0.0;
                if (plain) {
                  b0 += wv[k];
                  b1 = fma(wv[k], wv[k], b1);
                  cnt += lv[k] ? 0x10000 : 0;
                }
              }
              if (!plain) {
                const PixSlot sa = {carry_b + (warp * T + ja) * 2, carryn_b + warp * T + ja, lead_b + (warp * T + ja) * 2,
                                    leadn_b + warp * T + ja};
                const PixSlot sb = {carry_b + (warp * T + jh) * 2, carryn_b + warp * T + jh, lead_b + (warp * T + jh) * 2,
                                    leadn_b + warp * T + jh};
                pix_reduce2(ps, wa, la, wv, lv, second, p.neff_min, sa, sb, lane, a0, a1, cnt, npa, b0, b1, cntb, npb);
              }
            }
            if (!plain) {
              // pixel-cut mode: the live counts of whole pixels do not fit the 16-bit packing; three reductions
              cnt = __reduce_add_sync(FULL, cnt);
              cntb = __reduce_add_sync(FULL, cntb);
              npa = __reduce_add_sync(FULL, npa | (npb << 16));   // (at most 32 pixels end in a block)
              npb = npa >> 16;
              npa &= 0xffff;
              const double k = warp_sum4(a0, a1, b0, b1, lane);
              if ((lane & 7) == 0) {
                const int j = (lane & 16) ? jb : ja;
                if (j >= 0) {
                  GWC_DEV_CHECK(p.flag, j < nt, FLAG_CHK_ACC);
                  acc_b[(warp * T + j) * 2 + ((lane >> 3) & 1)] += k;
                  if ((lane & 8) == 0) {
                    cnt_b[warp * T + j] += (lane & 16) ? cntb : cnt;
                    np_b[warp * T + j] += (lane & 16) ? npb : npa;
                  }
                }
              }
              if (jc < 0) break;
              ja = jc;
              continue;
            }
            cnt = __reduce_add_sync(FULL, cnt);
            if (cnt) {  // warp-uniform
              // (pixel-cut mode, a block inside one pixel: the sums go on the run that stays open)
              double* sum_b = PIX ? carry_b : acc_b;
              int* n_b = PIX ? carryn_b : cnt_b;
              const double k = warp_sum4(a0, a1, b0, b1, lane);
              if ((lane & 7) == 0) {
                const int j = (lane & 16) ? jb : ja;
                if (j >= 0) {
                  GWC_DEV_CHECK(p.flag, j < nt, FLAG_CHK_ACC);
                  sum_b[(warp * T + j) * 2 + ((lane >> 3) & 1)] += k;
                  if ((lane & 8) == 0) n_b[warp * T + j] += (lane & 16) ? (cnt >> 16) : (cnt & 0xffff);
                }
              }
            }
            if (jc < 0) break;
            ja = jc;
          }
        }
        };
        if (PIX && ps.interior) theta_loop(std::true_type{});   // warp-uniform, the same for every theta
        else theta_loop(std::false_type{});
      }
      if (PIX) {
        // What this warp's range leaves for the stitch: the run open at its start (lead), whether a pixel starts
        // inside it, and the run open at its end (trail = the carry slot).  No pixel start at all: the whole range
        // is one open run and belongs to the lead.
        __syncwarp();
        if (lead_open && lane < nt) {
          lead_b[(warp * T + lane) * 2] += carry_b[(warp * T + lane) * 2];
          lead_b[(warp * T + lane) * 2 + 1] += carry_b[(warp * T + lane) * 2 + 1];
          leadn_b[warp * T + lane] += carryn_b[warp * T + lane];
          carry_b[(warp * T + lane) * 2] = 0.0;
          carry_b[(warp * T + lane) * 2 + 1] = 0.0;
          carryn_b[warp * T + lane] = 0;
        }
        if (lane == 0) s_hashead[buf][warp] = lead_open ? 0 : 1;
      }
      if (ASYNC) {
        __syncwarp();
        int last = 0;
        if (lane == 0) {
          __threadfence_block();  // this warp's sums before its arrival
          last = atomicAdd(&s_arrive[buf], 1) == NWARPS - 1;
        }
        last = __shfl_sync(FULL, last, 0);
        if (last) {  // every warp has arrived: this one combines the segment, in warp order, and clears the buffer
          __threadfence_block();
          GWC_DEV_CHECK(p.flag, *(volatile int*)&s_arrive[buf] == NWARPS && *(volatile int*)&s_done == sidx,
                        FLAG_CHK_HANDOFF);
          if (lane < nt) {
            double a = 0.0, b = 0.0;
            int c = 0, np = 0;
            for (int w = 0; w < NWARPS; ++w) {
              a += *(volatile double*)&acc_b[(w * T + lane) * 2];
              b += *(volatile double*)&acc_b[(w * T + lane) * 2 + 1];
              c += *(volatile int*)&cnt_b[w * T + lane];
              acc_b[(w * T + lane) * 2] = 0.0;
              acc_b[(w * T + lane) * 2 + 1] = 0.0;
              cnt_b[w * T + lane] = 0;
              if (PIX) {
                np += *(volatile int*)&np_b[w * T + lane];
                np_b[w * T + lane] = 0;
              }
            }
            if (PIX) {
              // pixels that cross warp ranges: walk the ranges in order, close the open run wherever a pixel starts
              double oW = 0.0, oQ = 0.0;
              int oN = 0;
              for (int r = 0; r <= NWARPS; ++r) {
                const int w = r < NWARPS ? ((r - sidx) & (NWARPS - 1)) : NWARPS;   // the warp that had range r
                if (w < NWARPS) {
                  oW += *(volatile double*)&lead_b[(w * T + lane) * 2];
                  oQ += *(volatile double*)&lead_b[(w * T + lane) * 2 + 1];
                  oN += *(volatile int*)&leadn_b[w * T + lane];
                }
                if (w == NWARPS || *(volatile int*)&s_hashead[buf][w]) {
                  if (oW > 0.0 && oW * oW >= p.neff_min * oQ) {
                    a += oW;
                    b += oQ;
                    c += oN;
                    np += 1;
                  }
                  if (w < NWARPS) {
                    oW = *(volatile double*)&carry_b[(w * T + lane) * 2];
                    oQ = *(volatile double*)&carry_b[(w * T + lane) * 2 + 1];
                    oN = *(volatile int*)&carryn_b[w * T + lane];
                  }
                }
                if (w < NWARPS) {
                  lead_b[(w * T + lane) * 2] = 0.0;
                  lead_b[(w * T + lane) * 2 + 1] = 0.0;
                  leadn_b[w * T + lane] = 0;
                  carry_b[(w * T + lane) * 2] = 0.0;
                  carry_b[(w * T + lane) * 2 + 1] = 0.0;
                  carryn_b[w * T + lane] = 0;
                }
              }
            }
            const size_t o = (size_t)(p.t_begin + t0 + lane) * (size_t)p.n_seg + (size_t)seg;
            p.out_w[2 * o] = a;
            p.out_w[2 * o + 1] = b;
            p.out_n[o] = c;
            if (PIX) p.out_np[o] = np;
          }
          __syncwarp();
          if (lane == 0) {
            s_arrive[buf] = 0;
            __threadfence_block();  // the cleared buffer before the release
            atomicAdd(&s_done, 1);
          }
        }
        seg0 += 1;
        continue;
      }
      __syncthreads();
      // segment complete: combine the warps' partials in a fixed order and write them out
      if ((tid & 31) < nt && (tid >> 5) < nteam) {  // (acc_b = s_acc here: one buffer)
        const int team = tid >> 5, j = tid & 31;  // one thread per (segment of this round, theta)
        double a = 0.0, b = 0.0;
        int c = 0;
        for (int w = team * tsz; w < (team + 1) * tsz; ++w) {
          a += s_acc[(w * T + j) * 2];
          b += s_acc[(w * T + j) * 2 + 1];
          c += s_cnt[w * T + j];
          s_acc[(w * T + j) * 2] = 0.0;
          s_acc[(w * T + j) * 2 + 1] = 0.0;
          s_cnt[w * T + j] = 0;
        }
        const size_t o = (size_t)(p.t_begin + t0 + j) * (size_t)p.n_seg + (size_t)(seg0 + team);
        p.out_w[2 * o] = a;
        p.out_w[2 * o + 1] = b;
        p.out_n[o] = c;
      }
      __syncthreads();  // the reset above precedes the next segment's accumulation
      seg0 += nteam;
    }
  }
}

template <typename NodeT, typename LosT, bool INJ, bool PIX = false, bool TEAMS = false, bool ODD = false,
          bool MP = false>
int launch_one(const ReweightParams& p, int n_blocks, size_t smem, cudaStream_t s) {
  reweight_kernel<NodeT, LosT, INJ, PIX, TEAMS, ODD, MP><<<n_blocks, NTHREADS, smem, s>>>(p);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

template <typename NodeT, typename LosT, bool INJ, bool PIX = false, bool TEAMS = false, bool ODD = false,
          bool MP = false>
int configure_one(int smem_optin) {
  return cudaFuncSetAttribute(reweight_kernel<NodeT, LosT, INJ, PIX, TEAMS, ODD, MP>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize,
                              smem_optin) == cudaSuccess ? 0 : -1;
}

// the variants of one (NodeT, LosT) pair of event kernels; MULTIPEAK has the plain and the pixel-cut kernel
template <typename NodeT, typename LosT>
int configure_events(int smem_optin) {
  int rc = 0;
  rc |= configure_one<NodeT, LosT, false>(smem_optin);
  rc |= configure_one<NodeT, LosT, false, true>(smem_optin);
  rc |= configure_one<NodeT, LosT, false, false, true>(smem_optin);
  rc |= configure_one<NodeT, LosT, false, false, false, true>(smem_optin);
  rc |= configure_one<NodeT, LosT, false, false, false, false, true>(smem_optin);
  rc |= configure_one<NodeT, LosT, false, true, false, false, true>(smem_optin);
  return rc;
}

template <typename NodeT, typename LosT>
int launch_events(const ReweightParams& p, int n_blocks, size_t smem, cudaStream_t s) {
  if (p.model == 1)
    return p.pixcut ? launch_one<NodeT, LosT, false, true, false, false, true>(p, n_blocks, smem, s)
                    : launch_one<NodeT, LosT, false, false, false, false, true>(p, n_blocks, smem, s);
  if (p.pixcut) return launch_one<NodeT, LosT, false, true>(p, n_blocks, smem, s);
  if (p.odd) return launch_one<NodeT, LosT, false, false, false, true>(p, n_blocks, smem, s);
  if (p.teams) return launch_one<NodeT, LosT, false, false, true>(p, n_blocks, smem, s);
  return launch_one<NodeT, LosT, false>(p, n_blocks, smem, s);
}

template <typename NodeT>
int launch_inj(const ReweightParams& p, int n_blocks, size_t smem, cudaStream_t s) {
  if (p.model == 1) return launch_one<NodeT, double, true, false, false, false, true>(p, n_blocks, smem, s);
  if (p.odd) return launch_one<NodeT, double, true, false, false, true>(p, n_blocks, smem, s);
  return launch_one<NodeT, double, true>(p, n_blocks, smem, s);
}

}  // namespace

size_t reweight_smem_bytes(int T, int Mp, gwc_prec tab_prec, bool inj, int n_z, bool pix, bool mp, bool shared_tab) {
  return smem_layout(T, shared_tab ? 1 : T, Mp, tab_prec == GWC_F64 ? sizeof(Node64) : sizeof(Node32), inj, n_z, pix, mp)
      .total;
}

int reweight_max_T(int Mp, gwc_prec tab_prec, bool inj, int n_z, int smem_optin, bool pix, bool mp, bool shared_tab) {
  int best = 0;
  for (int T = 1; T <= MAX_T; ++T)
    if (reweight_smem_bytes(T, Mp, tab_prec, inj, n_z, pix, mp, shared_tab) + SMEM_RESERVE <= (size_t)smem_optin) best = T;
  return best;
}

int reweight_configure(int smem_optin) {
  smem_optin -= SMEM_RESERVE;  // room for the kernel's static shared memory
  int rc = 0;
  rc |= configure_events<Node64, double>(smem_optin);
  rc |= configure_events<Node64, float>(smem_optin);
  rc |= configure_events<Node32, double>(smem_optin);
  rc |= configure_events<Node32, float>(smem_optin);
  rc |= configure_one<Node64, double, true, false, false, true>(smem_optin);
  rc |= configure_one<Node32, double, true, false, false, true>(smem_optin);
  rc |= configure_one<Node64, double, true>(smem_optin);
  rc |= configure_one<Node32, double, true>(smem_optin);
  rc |= configure_one<Node64, double, true, false, false, false, true>(smem_optin);
  rc |= configure_one<Node32, double, true, false, false, false, true>(smem_optin);
  return rc;
}

// The theta batch goes through in launches of at most KT_THETA points (a whole number of tiles): each launch
// first copies its points' constants into the constant bank (stream-ordered) and resets the work counter.
int launch_reweight(const ReweightParams& p0, gwc_prec tab_prec, gwc_prec los_prec, bool inj, int n_sm, int device,
                    cudaStream_t s) {
  const bool mp = p0.model == 1;
  const int nc = nconst_of(p0.model);
  const size_t smem = reweight_smem_bytes(p0.T, p0.Mp, tab_prec, inj, p0.n_z, p0.pixcut != 0, mp, p0.shared_tab != 0);
  const int cap = ((mp ? KT_THETA_MP : KT_THETA) / p0.T) * p0.T;
  int launched = 0;
  if (device < 0 || device >= MAX_DEVICES) return -1;
  BankGuard& bank = g_bank[device];
  std::lock_guard<std::mutex> lock(bank.mu);   // the enqueue order below is the order of the event chain
  if (!bank.last && cudaEventCreateWithFlags(&bank.last, cudaEventDisableTiming) != cudaSuccess) return -1;
  for (int tb = 0; tb < p0.n_theta; tb += cap) {
    ReweightParams p = p0;
    p.t_begin = tb;
    p.n_theta = p0.n_theta - tb < cap ? p0.n_theta - tb : cap;
    p.n_tiles = (p.n_theta + p.T - 1) / p.T;
    const int64_t n_items = (int64_t)p.n_groups * p.n_tiles;
    const int n_blocks = (int)(n_items < n_sm ? n_items : n_sm);
    if (bank.used && bank.last_stream != s && cudaStreamWaitEvent(s, bank.last, 0) != cudaSuccess) return -1;
    if (cudaMemcpyToSymbolAsync(KT, p0.tconst + (size_t)tb * nc, sizeof(double) * nc * (size_t)p.n_theta, 0,
                                cudaMemcpyDeviceToDevice, s) != cudaSuccess)
      return -1;
    if (cudaMemsetAsync(p.unit_counter, 0, sizeof(unsigned int), s) != cudaSuccess) return -1;
    int rc;
    if (inj) {
      rc = tab_prec == GWC_F64 ? launch_inj<Node64>(p, n_blocks, smem, s) : launch_inj<Node32>(p, n_blocks, smem, s);
    } else if (tab_prec == GWC_F64) {
      rc = los_prec == GWC_F64 ? launch_events<Node64, double>(p, n_blocks, smem, s)
                               : launch_events<Node64, float>(p, n_blocks, smem, s);
    } else {
      rc = los_prec == GWC_F64 ? launch_events<Node32, double>(p, n_blocks, smem, s)
                               : launch_events<Node32, float>(p, n_blocks, smem, s);
    }
    if (rc < 0) return -1;
    launched += rc;
    if (cudaEventRecord(bank.last, s) != cudaSuccess) return -1;
    bank.used = true;
    bank.last_stream = s;
  }
  return launched;
}

}  // namespace gwc
