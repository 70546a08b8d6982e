// gwc_internal.h -- shared declarations of the CUDA library (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gwc.h"

namespace gwc {

// ---- per-theta constant block (A2), doubles, consumed by the fused re-weighting kernel ----------
// With x = 1+z, lx = ln x, t1 = ln m1z - lx (= ln m1), Q = ln(m2z/m1z), P' = -ln pi - ln m1z - shift:
//   w = [exp(CPL + c - alpha t1) + exp(CG + c - y^2/2)] * p_los / [(u + x^2/E)(1 - e1)(1 + e2)]
//   c = beta Q + P' + (gamma-1) lx,  y = m1/sigma - mu/sigma,
//   e1 = exp(E1C + NBP1 t1) = (mmin/m1)^(beta+1),  e2 = exp(GK lx + E2C) = ((1+z)/(1+zp))^(gamma+kappa)
enum : int {
  C_H = 0,     // H0 / c                          (u = d_L * h)
  C_UMAX,      // u(z_max) of this theta's table
  C_INVDU,     // (M-1) / umax
  C_MMIN,
  C_MMAX,
  C_BETA,
  C_GM1,       // gamma - 1
  C_NALPHA,    // -alpha
  C_CPL,       // ln[(1-lambda) n_pl |beta+1| psi0 h]   (-inf when lambda = 1)
  C_CG,        // ln[lambda n_g /(sigma sqrt(2 pi)) |beta+1| psi0 h]   (-inf when lambda = 0)
  C_INVSIG,    // 1/sigma
  C_NMUSIG,    // -mu/sigma
  C_NBP1,      // -(beta+1)
  C_E1C,       // (beta+1) ln mmin
  C_SGN,       // sign(beta+1)
  C_GK,        // gamma + kappa
  C_E2C,       // -(gamma+kappa) ln(1+zp)
  C_OM,
  C_OL,        // 1 - Om
  C_VALID,     // 1.0 or NaN (theta-domain violation)
  C_COUNT,
  // ---- MULTIPEAK rows only (row length NCONST_MP; R33-R36).  There CPL / CG carry 1/N1, CG / INVSIG /
  // NMUSIG belong to the HIGH peak, and E1C = ln(top^(beta+1) - (beta+1) C_top), top = mmin + delta_m, so that above
  // the smoothing window |beta+1| C(m1) / m1^(beta+1) = sign(beta+1) (1 - e1) as in the power-law+peak model.
  C_CG2 = C_COUNT,  // ln[lambda_g lambda_low n_g,low / (sigma_low sqrt(2 pi)) |beta+1| psi0 h / N1]   (-inf when absent)
  C_INVSIG2,   // 1/sigma_low
  C_NMUSIG2,   // -mu_low/sigma_low
  C_DM,        // delta_m
  C_FIDX,      // (MF_NODES - 1) / delta_m   (0 when delta_m = 0)
  C_N1,        // int mix S dm over [mmin, mmax]                       (read by the KDE kernel)
  C_CTOP,      // C(top) = int over the smoothing window of m^beta S(m) dm   (read by the KDE kernel)
  C_NGL,       // normalisation of the low Gaussian on [mmin, mmax]    (read by the KDE kernel)
  C_COUNT_MP
};
constexpr int NCONST = 24;     // padded row length (>= C_COUNT), keeps rows 64-byte aligned
constexpr int NCONST_MP = 32;  // row length under MULTIPEAK (>= C_COUNT_MP)
constexpr int MF_NODES = 513;  // nodes of the per-theta table of F(m1) = |beta+1| C(m1) / (S(m1) m1^(beta+1)) on the window
constexpr int MF_PITCH = 514;
__host__ __device__ inline int nconst_of(int model) { return model == 1 ? NCONST_MP : NCONST; }

#ifndef GWC_NTHREADS
#define GWC_NTHREADS 512
#endif
#ifndef GWC_SPT
#define GWC_SPT 2
#endif
constexpr int NTHREADS = GWC_NTHREADS;  // threads per CTA of the fused kernel (one CTA per SM)
constexpr int NWARPS = NTHREADS / 32;
constexpr int SPT = GWC_SPT;      // samples per thread per theta (independent chains in flight)
constexpr int KT_THETA = 340;     // theta points whose constants fit the constant bank (one launch)
constexpr int KT_THETA_MP = KT_THETA * NCONST / NCONST_MP;   // ... with MULTIPEAK rows (255)
#ifndef GWC_MAX_T
#define GWC_MAX_T 16
#endif
constexpr int MAX_T = GWC_MAX_T;  // theta points per tile (upper bound)
constexpr int INJ_SEG = 8192;     // injections per segment of the selection reduction
constexpr int QUAD_K = 1024;      // forward quadrature intervals of the cosmology builder
constexpr int MAX_NODES = 8193;

struct Node64 { double z, d; };   // table node: z_m and du * z'(u_m)
struct Node32 { uint32_t zq; float d; };  // 32-bit storage: z_m = zq * z_max / (2^32 - 1), d in the same units
constexpr double NODE32_QMAX = 4294967295.0;

// table row length: M nodes + 1 pad node (index M is read when u rounds onto the last node), even
__host__ __device__ inline int table_pitch(int M) { return (M + 2) & ~1; }

struct ReweightParams {
  int model;                // gwc_mass_model
  const Node64* ftab;       // MULTIPEAK: [n_theta][MF_PITCH] (F, dm/(MF_NODES-1) F') of the smoothing window
  const void* tab;          // [n_theta][Mp] Node64 | Node32
  const double* tconst;     // [n_theta][NCONST]
  int n_theta, M, Mp, T, n_tiles;   // n_theta, n_tiles: of the batch (set per launch by launch_reweight)
  int t_begin;              // first theta of this launch
  const double *dLc, *m1z, *m2z, *L1, *Q, *P;   // [n_samples] prepared per-sample values
  const int32_t* row;       // [n_samples] (events) or nullptr (injections)
  const int64_t* seg_off;   // [n_seg+1] device
  const int32_t* group_off; // [n_groups+1] device: segments of each work group
  int n_groups;
  int64_t n_seg;
  const void* los;          // [n_rows][n_z] (events) | allsky [n_z] f64 (injections)
  int64_t n_rows;
  int n_z;
  double inv_dz, los_zmax;
  double tab_zq;            // Node32 tables: z_max of the cosmology table / (2^32 - 1)
  double* out_w;            // [n_theta][n_seg][2]: sum w', sum w'^2
  int32_t* out_n;           // [n_theta][n_seg]   : n_live
  int32_t* out_np;          // [n_theta][n_seg]   : passing pixels (pixel-cut mode)
  int odd;                  // 1: kernel variant with a tail-only path for odd theta counts (batches of a few points)
  int teams;                // 1: kernel variant in which short segments share the CTA (catalogues of short events)
  int pixcut;               // 1: per-pixel effective-sample cut (Eq. 8), threshold neff_min
  double neff_min;
  unsigned int* unit_counter;
  int* flag;                // sticky device flag word (written by -DGWC_CHECKED builds only)
  int64_t n_samples;        // length of the sample arrays (checked builds)
  const int32_t* group_order; // [n_groups] device: the groups, heaviest first (the order work items are handed out in)
  int shared_tab;           // 1: the batch has a single Omega_m, the tile stages ONE z(u) table (of its first theta)
};

// kernels / launchers (each returns the number of kernels it launched, or -1 on a launch error)
// sticky device flag word (gwc_ctx::d_flag[0]); d_flag[1] belongs to the A0 packing alone
enum : int {
  FLAG_DOMAIN = 1,   // a theta point outside the model's domain (gwc_build_cosmo)
  FLAG_STALE = 4,    // d_theta differs from the copy taken by gwc_build_cosmo
  FLAG_RANGE = 8,    // every live weight of a segment lies below e^-300 of the segment's reference
  FLAG_OMEGA = 16,   // GWC_OMEGA_SINGLE was promised (gwc_set_omega_hint) and the batch has several Omega_m or an invalid row
  // -DGWC_CHECKED builds only (tests/sanitizer_cases.py): a device-side check failed
  FLAG_CHK_TABLE = 1 << 8,     // index into a z(u) table outside [0, Mp - 2]
  FLAG_CHK_LOS = 1 << 9,       // LOS node index outside [0, n_z - 2], or a row outside the table
  FLAG_CHK_SAMPLE = 1 << 10,   // sample index outside [0, n_samples)
  FLAG_CHK_ACC = 1 << 11,      // accumulator slot outside the warp's own (warp, theta) range
  FLAG_CHK_HANDOFF = 1 << 12,  // barrier-free segment hand-off: a sum buffer reused before it was combined and cleared,
                               // a wrong arrival count, or segments combined out of order
  FLAG_CHK_MATH = 1 << 13,     // exp / log table index out of range
  FLAG_CHK_FTAB = 1 << 14,     // MULTIPEAK F-table index outside [0, MF_NODES - 2]
  FLAG_CHK_KDE = 1 << 15,      // KDE kernel: scratch slot outside the warp's slice, grid node or LOS bin out of range
  FLAG_CHK_ANY = 0xff << 8
};
#ifdef GWC_CHECKED
#define GWC_DEV_CHECK(flagp, cond, bit)              \
  do {                                               \
    if (!(cond)) atomicOr((flagp), (int)(bit));      \
  } while (0)
#else
#define GWC_DEV_CHECK(flagp, cond, bit) \
  do {                                  \
  } while (0)
#endif
// smallest linear-domain segment sum (relative to the segment's reference) that is still trusted: below it the
// clamped exponentials (e^-700) and the squares of the weights lose their meaning (R23)
constexpr double RANGE_MIN_SUM = 5.148200222412013e-131;   // e^-300

// model: gwc_mass_model; theta rows have gwc_theta_len(model) doubles, tconst rows nconst_of(model); d_ftab only under
// MULTIPEAK
int launch_cosmo_build(const double* d_theta, int64_t n_theta, int model, double z_max, int M, int Mp, gwc_prec prec,
                       void* d_tab, double* d_tconst, Node64* d_ftab, double* d_theta_snap, double* d_tvalid,
                       int* d_flag, cudaStream_t s);
// compares d_theta with the copy gwc_build_cosmo took: tvalid[t] = tconst[t][C_VALID] or NaN (+ FLAG_STALE)
int launch_verify_theta(const double* d_theta, const double* d_theta_snap, const double* d_tconst, int64_t n_theta,
                        int model, double* d_tvalid, int* d_flag, cudaStream_t s);
int launch_export_cosmo(const void* d_tab, const double* d_tconst, int ncst, int64_t n_theta, int M, int Mp,
                        gwc_prec prec, double z_max, double* d_z, double* d_dz, double* d_umax, cudaStream_t s);
// per-sample, theta-independent preparation (+ per-segment shift = max(-ln pi - ln m1z))
int launch_prep_samples(int64_t n, int64_t n_seg, const int64_t* seg_off, const double* dL, const double* m1z,
                        const double* m2z, const double* lprior, const int32_t* row, int64_t n_rows, double* dLc,
                        double* L1, double* Q, double* P, double* seg_shift, cudaStream_t s);
int launch_make_groups(const int64_t* seg_off, int64_t n_seg, int64_t target, int n_groups, int32_t* group_off,
                       int32_t* group_order, bool uniform, cudaStream_t s);
int launch_uniform_segments(int64_t n, int64_t seg, int64_t n_seg, int64_t* seg_off, cudaStream_t s);
size_t reweight_smem_bytes(int T, int Mp, gwc_prec tab_prec, bool inj, int n_z, bool pix, bool mp, bool shared_tab);
int reweight_max_T(int Mp, gwc_prec tab_prec, bool inj, int n_z, int smem_optin, bool pix, bool mp, bool shared_tab);
// *d_same = 1 when every theta row has the same Omega_m bits and lies inside the model's domain (one z(u) table
// serves the batch), else 0
// d_flag != nullptr: a 0 answer also raises FLAG_OMEGA there (the caller's promise is checked, nobody waits for it)
int launch_omega_same(const double* d_theta, int64_t n_theta, int model, int* d_same, cudaStream_t s,
                      int* d_flag = nullptr);
int reweight_configure(int smem_optin);
int launch_reweight(const ReweightParams& p, gwc_prec tab_prec, gwc_prec los_prec, bool inj, int n_sm, int device,
                    cudaStream_t s);
// tvalid [n_theta]: 1.0, or NaN for a theta outside the domain / changed since the build
int launch_finalize_events(const double* part_w, const int32_t* part_n, const int64_t* seg_off, const double* seg_shift,
                           const double* tvalid, int64_t n_theta, int64_t n_events, double* logL,
                           double* neff, int64_t* nlive, int* d_flag, cudaStream_t s);
int launch_finalize_inj(const double* part_w, const int32_t* part_n, const double* seg_shift, const double* tvalid,
                        int64_t n_theta, int64_t n_seg, double n_draw, double* logxi, double* neff, int* d_flag,
                        cudaStream_t s);
int launch_widen_i32(const int32_t* in, const double* tvalid, int64_t n_theta, int64_t n, int64_t* out,
                     cudaStream_t s);
int launch_combine_total(const double* logL, const double* logxi, int64_t n_theta, int64_t n_events, double* total,
                         cudaStream_t s);
// event / injection sharding: pieces [n_parts][n_theta] of R ranks -> total, log xi, N_eff,inj [n_theta] (rank order);
// the kernel and the host loop run the same function
int launch_combine_sharded(const double* sum_parts, const double* logxi_parts, const double* neff_parts, int n_parts,
                           int64_t n_theta, int64_t n_events_total, double* total, double* logxi, double* neff,
                           cudaStream_t s);
void combine_sharded_host(const double* sum_parts, const double* logxi_parts, const double* neff_parts, int n_parts,
                          int64_t n_theta, int64_t n_events_total, double* total, double* logxi, double* neff);
int launch_allsky(const void* table, gwc_prec prec, int64_t n_rows, int n_z, double* scratch, double* allsky,
                  cudaStream_t s);
size_t allsky_scratch_doubles(int64_t n_rows, int n_z);
int launch_kde(int model, const Node64* d_ftab, const double* d_theta, const void* d_tab, const double* d_tconst, const double* d_tvalid, int64_t n_theta, int M, int Mp,
               gwc_prec tab_prec, double tab_zq, int64_t n_events, const int64_t* ev_off, const double* dL,
               const double* m1z, const double* m2z, const double* lprior, const int32_t* row, const double* seg_shift,
               const void* los, gwc_prec los_prec, int64_t n_rows, int n_z, double los_zmax, int n_grid, double neff_min,
               int bw_rule, double* logL, int64_t* npass, int64_t* nused, void* scratch, int64_t scr_stride, int n_blocks,
               int64_t n_chunks, const int64_t* d_chunk_off, const int64_t* d_start, const int64_t* d_end,
               const int32_t* d_event, void* d_thk, void* d_gw, double* d_part_e, int32_t* d_part_np,
               int64_t* d_part_nu, int* d_flag, cudaStream_t s);
// KDE work units are (chunk, theta): the chunk table of a catalogue (runs of whole pixels, about 1024 samples)
int64_t kde_chunk_bound(int64_t n_samples, int64_t n_events);
int launch_kde_chunks(const int64_t* ev_off, int64_t n_events, const int32_t* row, int64_t* d_cnt,
                      int64_t* d_chunk_off, int64_t* d_start, int64_t* d_end, int32_t* d_event, int64_t* d_max_len,
                      int64_t n_samples, cudaStream_t s);
size_t kde_theta_bytes(int64_t n_theta);
size_t kde_weight_bytes(int64_t n_theta);
int kde_grid_blocks(int64_t n_theta, int64_t n_chunks, int n_sm);
size_t kde_scratch_bytes(int n_blocks, int64_t max_chunk_len);
int launch_max_segment(const int64_t* seg_off, int64_t n_seg, int64_t* d_out, cudaStream_t s);
int launch_probe_fp64(int64_t iters, int n_blocks, double* d_sink, cudaStream_t s, double* n_instr);
int launch_math_selftest(int which, int64_t n, const double* d_in, double* d_out, cudaStream_t s);

// A0 packing (device radix sort + run detection); returns launches or -1
size_t pack_scratch_bytes(int64_t n_samples, int64_t n_events);
int launch_pack(int64_t n_samples, int64_t n_events, const int32_t* d_event_id, const int32_t* d_row, int64_t* d_perm,
                int64_t* d_ev_sample_off, int64_t* d_ev_pix_off, int32_t* d_ev_pix_rows, int64_t* d_pix_sample_off,
                int64_t* d_n_pixrefs, int* d_flag, void* scratch, size_t scratch_bytes, cudaStream_t s);

// pixel-aligned padded copy of the prepared samples (pixel-cut mode): pads per segment and the padded offsets, then
// the scatter; seg_off_pad [n_seg + 1], seg_pads [n_seg]
int launch_pixpad_count(const int64_t* d_seg_off, int64_t n_seg, const int32_t* d_row, int64_t* d_seg_pads,
                        int64_t* d_seg_off_pad, cudaStream_t s);
int launch_pixpad_scatter(const int64_t* d_seg_off, int64_t n_seg, const int64_t* d_seg_off_pad, const double* dLc,
                          const double* m1z, const double* m2z, const double* L1, const double* Q, const double* P,
                          const int32_t* row, double* o_dLc, double* o_m1z, double* o_m2z, double* o_L1, double* o_Q,
                          double* o_P, int32_t* o_row, cudaStream_t s);

// injections in order of d_L (selection term): sorted copies of the four arrays
size_t injsort_scratch_bytes(int64_t n);
int launch_injsort(int64_t n, const double* dL, const double* m1z, const double* m2z, const double* lp, double* o_dL,
                   double* o_m1z, double* o_m2z, double* o_lp, void* scratch, size_t scratch_bytes, cudaStream_t s);

size_t cap_scratch_bytes(int64_t n_samples);
int launch_cap_pixels(int64_t n, int64_t n_events, int64_t n_pix, const int64_t* d_perm_in, int64_t* d_ev_sample_off,
                      int64_t* d_pix_sample_off, int64_t cap, uint64_t seed, int64_t* d_perm_out, int64_t* d_n_kept,
                      void* scratch, size_t scratch_bytes, cudaStream_t s);

}  // namespace gwc
