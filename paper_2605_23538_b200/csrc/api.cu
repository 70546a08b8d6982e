// api.cu -- the C ABI of include/gwc.h: context, argument checks, scratch memory and the launch
// sequence of the hot path A1..A6.  No arithmetic of the method lives here.
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "gwc_internal.h"

using namespace gwc;

namespace {

struct Buf {
  void* p = nullptr;
  size_t cap = 0;
};

struct HostCopy {  // device mirrors used by gwc_total_loglik_host
  Buf theta, ev_off, ev_dL, ev_m1z, ev_m2z, ev_lp, ev_row, inj_dL, inj_m1z, inj_m2z, inj_lp, los, allsky, out;
};

}  // namespace

// Per-sample prepared values (d_L or NaN, ln m1z, ln(m2z/m1z), -l_pi - ln m1z - shift) and the per-segment shift of
// one sample set, with the identity of the arrays they were computed from.
struct PrepSet {
  Buf dLc, L1, Q, P, seg_shift;
  const void *k_dL = nullptr, *k_m1z = nullptr, *k_m2z = nullptr, *k_lp = nullptr, *k_row = nullptr, *k_off = nullptr;
  int64_t k_n = -1, k_nseg = -1, k_nrows = -1;
  bool valid = false;
};

// Pixel-aligned padded copy of a prepared sample set (pixel-cut mode; pack.cu): every pixel starts at an even position
// and has an even length.  Valid as long as the PrepSet it was made from is.
struct PadSet {
  Buf dLc, m1z, m2z, L1, Q, P, row, seg_off, seg_pads;
  int64_t n_pad = 0;
  bool valid = false;
};

// The injections in order of d_L (pack.cu): sorted copies of the caller's four arrays, with their identity.
struct InjSorted {
  Buf dL, m1z, m2z, lp;
  const void *k_dL = nullptr, *k_m1z = nullptr, *k_m2z = nullptr, *k_lp = nullptr;
  int64_t k_n = -1;
  bool valid = false;
};

struct gwc_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int n_sm = 0, smem_optin = 0;
  std::string err;
  int64_t launches = 0;
  int* d_flag = nullptr;
  unsigned int* d_counter = nullptr;
  // A1/A2 state
  int model = 0;            // gwc_mass_model: theta rows have npar doubles, constant rows nconst_of(model)
  int npar = GWC_NPAR;
  Buf ftab;                 // MULTIPEAK: [n_theta][MF_PITCH] Node64, F(m1) over the smoothing window
  Buf tab, tconst;
  Buf theta_snap, tvalid;   // the theta rows the tables were built from; per-theta validity (1.0 | NaN)
  const double* built_theta = nullptr;
  int64_t built_n = 0;
  bool fresh_build = false;   // inside gwc_total_loglik*: the build was enqueued by this very call, no verification
  int M = 0, Mp = 0;
  bool tab_shared = false;  // the batch of the last build has one Omega_m: one z(u) table serves every theta
  int omega_hint = GWC_OMEGA_DETECT;   // gwc_set_omega_hint
  gwc_prec tab_prec = GWC_F64;
  double z_max = 0.0;
  // per-call scratch
  Buf seg_off, group_off, part_w, part_n, part_np, kde_scr, kde_len, allsky_scr, pack_scr, logL, logxi, probe;
  Buf kde_cnt, kde_coff, kde_cstart, kde_cend, kde_cev, kde_thk, kde_gw, kde_pe, kde_pnp, kde_pnu;   // KDE chunks, partials
  HostCopy hc;
  // theta-independent preparation of the events [0] and the injections [1] (kept between calls when caching is on)
  PrepSet prep[2];
  PadSet pad;               // of prep[0]
  InjSorted injs;           // what prep[1] is computed from
  bool cache_prep = false;
  // timing
  bool timing = false;
  std::vector<cudaEvent_t> ev_pairs, inj_pairs;
  std::vector<cudaEvent_t> pool;
};

namespace {

std::string g_create_error;  // text of the last failed gwc_create (no context exists to hold it)

gwc_status fail(gwc_ctx* c, gwc_status st, const char* msg) {
  if (c) c->err = msg;
  return st;
}

gwc_status cuda_fail(gwc_ctx* c, cudaError_t e, const char* where) {
  if (c) c->err = std::string(where) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? GWC_ERR_NOMEM : GWC_ERR_CUDA;
}

#define GWC_CUDA(call)                                     \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
  } while (0)

#define GWC_TRY(call)                \
  do {                               \
    gwc_status s_ = (call);          \
    if (s_ != GWC_OK) return s_;     \
  } while (0)

// grow-only device buffer; growth synchronises the stream (work in flight may still read the old block)
gwc_status ensure(gwc_ctx* ctx, Buf& b, size_t bytes) {
  if (bytes <= b.cap) return GWC_OK;
  GWC_CUDA(cudaStreamSynchronize(ctx->stream));
  if (b.p) cudaFree(b.p);
  b.p = nullptr;
  b.cap = 0;
  size_t want = bytes + bytes / 8 + 256;
  cudaError_t e = cudaMalloc(&b.p, want);
  if (e != cudaSuccess) {
    want = bytes;
    e = cudaMalloc(&b.p, want);
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    return cuda_fail(ctx, e, "cudaMalloc");
  }
  b.cap = want;
#ifdef GWC_CHECKED
  cudaMemsetAsync(b.p, 0xff, want, ctx->stream);   // poison (NaN / -1): a read of scratch never written shows in the results
#endif
  return GWC_OK;
}

void release(Buf& b) {
  if (b.p) cudaFree(b.p);
  b.p = nullptr;
  b.cap = 0;
}

gwc_status count(gwc_ctx* ctx, int rc, const char* what) {
  if (rc < 0) {
    cudaError_t e = cudaGetLastError();
    ctx->err = std::string(what) + ": launch failed: " + cudaGetErrorString(e);
    return GWC_ERR_CUDA;
  }
  ctx->launches += rc;
  return GWC_OK;
}

cudaEvent_t get_event(gwc_ctx* ctx) {
  if (!ctx->pool.empty()) {
    cudaEvent_t e = ctx->pool.back();
    ctx->pool.pop_back();
    return e;
  }
  cudaEvent_t e;
  cudaEventCreate(&e);
  return e;
}

// The tables in the context belong to the theta rows gwc_build_cosmo saw.  Host side: same pointer and count.
// Device side: the caller's rows are compared bit for bit with the copy taken at build time (an in-place update, or
// another tensor that the allocator put at the same address, is caught here): a row that differs gets NaN outputs and
// raises the sticky FLAG_STALE, which gwc_check reports as GWC_ERR_NOT_BUILT.
gwc_status check_built(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, double los_zmax) {
  if (!ctx->built_theta || ctx->built_theta != d_theta || ctx->built_n != n_theta)
    return fail(ctx, GWC_ERR_NOT_BUILT, "gwc_build_cosmo was not called with this d_theta / n_theta");
  if (los_zmax > ctx->z_max * (1.0 + 1e-12))
    return fail(ctx, GWC_ERR_NOT_BUILT, "cosmology table built with a smaller z_max than the LOS table's");
  if (ctx->fresh_build) return GWC_OK;
  return count(ctx, launch_verify_theta(d_theta, (const double*)ctx->theta_snap.p, (const double*)ctx->tconst.p,
                                        n_theta, ctx->model, (double*)ctx->tvalid.p, ctx->d_flag, ctx->stream),
               "verify_theta");
}

// theta-independent preparation of a sample set; skipped when caching is on and the same arrays come again
gwc_status prepare_samples(gwc_ctx* ctx, PrepSet& ps, int64_t n, int64_t n_seg, const int64_t* d_seg_off,
                           const double* dL, const double* m1z, const double* m2z, const double* lprior,
                           const int32_t* row, int64_t n_rows) {
  if (ctx->cache_prep && ps.valid && ps.k_dL == dL && ps.k_m1z == m1z && ps.k_m2z == m2z && ps.k_lp == lprior &&
      ps.k_row == row && ps.k_off == d_seg_off && ps.k_n == n && ps.k_nseg == n_seg && ps.k_nrows == n_rows)
    return GWC_OK;
  ps.valid = false;
  if (&ps == &ctx->prep[0]) ctx->pad.valid = false;
  const size_t nd = (size_t)(n > 0 ? n : 1) * sizeof(double);
  GWC_TRY(ensure(ctx, ps.dLc, nd));
  GWC_TRY(ensure(ctx, ps.L1, nd));
  GWC_TRY(ensure(ctx, ps.Q, nd));
  GWC_TRY(ensure(ctx, ps.P, nd));
  GWC_TRY(ensure(ctx, ps.seg_shift, (size_t)(n_seg > 0 ? n_seg : 1) * sizeof(double)));
  GWC_TRY(count(ctx, launch_prep_samples(n, n_seg, d_seg_off, dL, m1z, m2z, lprior, row, n_rows, (double*)ps.dLc.p,
                                         (double*)ps.L1.p, (double*)ps.Q.p, (double*)ps.P.p, (double*)ps.seg_shift.p,
                                         ctx->stream),
                "prep_samples"));
  ps.k_dL = dL; ps.k_m1z = m1z; ps.k_m2z = m2z; ps.k_lp = lprior; ps.k_row = row; ps.k_off = d_seg_off;
  ps.k_n = n; ps.k_nseg = n_seg; ps.k_nrows = n_rows;
  ps.valid = true;
  return GWC_OK;
}

// pixel-cut mode: the pixel-aligned padded copy of the prepared events (one host synchronisation for its length)
gwc_status prepare_padded(gwc_ctx* ctx, const PrepSet& ps, int64_t n, int64_t n_seg, const int64_t* d_seg_off,
                          const double* m1z, const double* m2z, const int32_t* row) {
  PadSet& pd = ctx->pad;
  if (ctx->cache_prep && pd.valid) return GWC_OK;
  pd.valid = false;
  cudaStream_t s = ctx->stream;
  GWC_TRY(ensure(ctx, pd.seg_off, (size_t)(n_seg + 1) * sizeof(int64_t)));
  GWC_TRY(ensure(ctx, pd.seg_pads, (size_t)(n_seg > 0 ? n_seg : 1) * sizeof(int64_t)));
  GWC_TRY(count(ctx, launch_pixpad_count(d_seg_off, n_seg, row, (int64_t*)pd.seg_pads.p, (int64_t*)pd.seg_off.p, s),
                "pixpad_count"));
  int64_t n_pad = 0;
  GWC_CUDA(cudaMemcpyAsync(&n_pad, (const int64_t*)pd.seg_off.p + n_seg, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
  GWC_CUDA(cudaStreamSynchronize(s));
  if (n_pad < n || n_pad > 2 * n) return fail(ctx, GWC_ERR_SHAPE, "ev_sample_off is not ascending from 0 to n_samples");
  const size_t nd = (size_t)(n_pad > 0 ? n_pad : 1) * sizeof(double);
  GWC_TRY(ensure(ctx, pd.dLc, nd));
  GWC_TRY(ensure(ctx, pd.m1z, nd));
  GWC_TRY(ensure(ctx, pd.m2z, nd));
  GWC_TRY(ensure(ctx, pd.L1, nd));
  GWC_TRY(ensure(ctx, pd.Q, nd));
  GWC_TRY(ensure(ctx, pd.P, nd));
  GWC_TRY(ensure(ctx, pd.row, (size_t)(n_pad > 0 ? n_pad : 1) * sizeof(int32_t)));
  GWC_TRY(count(ctx, launch_pixpad_scatter(d_seg_off, n_seg, (const int64_t*)pd.seg_off.p, (const double*)ps.dLc.p, m1z,
                                           m2z, (const double*)ps.L1.p, (const double*)ps.Q.p, (const double*)ps.P.p,
                                           row, (double*)pd.dLc.p, (double*)pd.m1z.p, (double*)pd.m2z.p,
                                           (double*)pd.L1.p, (double*)pd.Q.p, (double*)pd.P.p, (int32_t*)pd.row.p, s),
                "pixpad_scatter"));
  pd.n_pad = n_pad;
  pd.valid = true;
  return GWC_OK;
}

// shared launch sequence of A3 (events) and A5 (injections): prep -> groups -> fused kernel
gwc_status run_reweight(gwc_ctx* ctx, int64_t n_theta, int64_t n, int64_t n_seg, const int64_t* d_seg_off,
                        const double* dL, const double* m1z, const double* m2z, const double* lprior,
                        const int32_t* row, const void* los_table, gwc_prec los_prec, int64_t n_rows, int n_z,
                        double los_zmax, bool inj, bool pixcut = false, double neff_min = 0.0) {
  cudaStream_t s = ctx->stream;
  PrepSet& ps = ctx->prep[inj ? 1 : 0];
  GWC_TRY(prepare_samples(ctx, ps, n, n_seg, d_seg_off, dL, m1z, m2z, lprior, row, n_rows));
  // what the fused kernel reads: the prepared arrays, or in pixel-cut mode their pixel-aligned padded copy
  const double *k_dLc = (const double*)ps.dLc.p, *k_m1z = m1z, *k_m2z = m2z, *k_L1 = (const double*)ps.L1.p,
               *k_Q = (const double*)ps.Q.p, *k_P = (const double*)ps.P.p;
  if (pixcut) {
    GWC_TRY(prepare_padded(ctx, ps, n, n_seg, d_seg_off, m1z, m2z, row));
    const PadSet& pd = ctx->pad;
    k_dLc = (const double*)pd.dLc.p; k_m1z = (const double*)pd.m1z.p; k_m2z = (const double*)pd.m2z.p;
    k_L1 = (const double*)pd.L1.p; k_Q = (const double*)pd.Q.p; k_P = (const double*)pd.P.p;
    row = (const int32_t*)pd.row.p;
    d_seg_off = (const int64_t*)pd.seg_off.p;
    n = pd.n_pad;
  }
  GWC_TRY(ensure(ctx, ctx->part_w, (size_t)n_theta * n_seg * 2 * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->part_n, (size_t)n_theta * n_seg * sizeof(int32_t)));
  if (pixcut) GWC_TRY(ensure(ctx, ctx->part_np, (size_t)n_theta * n_seg * sizeof(int32_t)));
  // theta tile: as many tables as shared memory holds, balanced over the tiles
  const bool mp = ctx->model == GWC_MASS_MULTIPEAK;
  const bool shared_tab = ctx->tab_shared;
  int T = reweight_max_T(ctx->Mp, ctx->tab_prec, inj, n_z, ctx->smem_optin, pixcut, mp, shared_tab);
  if (T < 1) return fail(ctx, GWC_ERR_SHAPE, "n_nodes / n_z too large for shared memory");
  if ((int64_t)T > n_theta) T = (int)n_theta;
  int n_tiles = (int)((n_theta + T - 1) / T);
  T = (int)((n_theta + n_tiles - 1) / n_tiles);
  // the kernel takes the theta points of a tile two at a time: an odd tile pays for one point more than it holds
  if (T > 2 && (T & 1) && n_theta > T) {
    const int Tmax = reweight_max_T(ctx->Mp, ctx->tab_prec, inj, n_z, ctx->smem_optin, pixcut, mp, shared_tab);
    T = T + 1 <= Tmax ? T + 1 : T - 1;
    n_tiles = (int)((n_theta + T - 1) / T);
  }
  // segment groups: enough work items to balance the SMs, small enough that a group's LOS rows stay in L2
  // (a launch holds the tiles of at most KT_THETA points: the items that have to balance the SMs are those of ONE launch)
  const int kt_cap = ((mp ? KT_THETA_MP : KT_THETA) / T) * T;
  const int tiles_per_launch = n_tiles < kt_cap / T ? n_tiles : kt_cap / T;
  int64_t target = (int64_t)((double)n * tiles_per_launch / ((double)ctx->n_sm * 16.0));
  if (target > 131072) target = 131072;   // (O5 event kernel: 1003 ms at 65536, 998 at 131072 / 262144, 1029 at 524288)
  if (target < 4096) target = 4096;
  while ((n / target + 2) * (int64_t)n_tiles > (int64_t)0x7fffffff) target *= 2;
  const int n_groups = (int)(n > 0 ? (n + target - 1) / target : 1);
  GWC_TRY(ensure(ctx, ctx->group_off, (size_t)(2 * n_groups + 1) * sizeof(int32_t)));   // offsets, then the order
  int32_t* d_group_order = (int32_t*)ctx->group_off.p + n_groups + 1;
  GWC_TRY(count(ctx, launch_make_groups(d_seg_off, n_seg, target, n_groups, (int32_t*)ctx->group_off.p, d_group_order, inj, s),
                "make_groups"));
  ReweightParams p;
  memset(&p, 0, sizeof(p));
  p.model = ctx->model;
  p.ftab = (const Node64*)ctx->ftab.p;
  p.tab = ctx->tab.p;
  p.tconst = (const double*)ctx->tconst.p;
  p.n_theta = (int)n_theta;
  p.M = ctx->M;
  p.Mp = ctx->Mp;
  p.T = T;
  p.n_tiles = n_tiles;
  p.dLc = k_dLc;
  p.m1z = k_m1z;
  p.m2z = k_m2z;
  p.L1 = k_L1;
  p.Q = k_Q;
  p.P = k_P;
  p.row = row;
  p.seg_off = d_seg_off;
  p.group_off = (const int32_t*)ctx->group_off.p;
  p.group_order = d_group_order;
  p.shared_tab = shared_tab ? 1 : 0;
  p.n_groups = n_groups;
  p.n_seg = n_seg;
  p.los = los_table;
  p.n_rows = n_rows;
  p.n_z = n_z;
  p.inv_dz = (double)(n_z - 1) / los_zmax;
  p.los_zmax = los_zmax;
  p.tab_zq = ctx->z_max / NODE32_QMAX;
  p.out_w = (double*)ctx->part_w.p;
  p.out_n = (int32_t*)ctx->part_n.p;
  p.out_np = pixcut ? (int32_t*)ctx->part_np.p : nullptr;
  p.pixcut = pixcut ? 1 : 0;
  // events shorter on average than 2048 samples leave warps of a 16-warp CTA without a block: let them share it
  // batches of a few theta points (the sampler's one-point-per-call pattern): no discarded pipeline step
  // (MULTIPEAK has the plain and the pixel-cut kernel only)
  p.odd = (!mp && !pixcut && n_theta <= 9 && (n_theta & 1)) ? 1 : 0;
  p.teams = (!mp && !inj && !pixcut && !p.odd && n_seg > 0 && n / n_seg < 2048) ? 1 : 0;
  p.neff_min = neff_min;
  p.unit_counter = ctx->d_counter;
  p.flag = ctx->d_flag;
  p.n_samples = n;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (ctx->timing) {
    e0 = get_event(ctx);
    e1 = get_event(ctx);
    cudaEventRecord(e0, s);
  }
  GWC_TRY(count(ctx, launch_reweight(p, ctx->tab_prec, los_prec, inj, ctx->n_sm, ctx->device, s), "reweight"));
  if (ctx->timing) {
    cudaEventRecord(e1, s);
    auto& v = inj ? ctx->inj_pairs : ctx->ev_pairs;
    v.push_back(e0);
    v.push_back(e1);
  }
  return GWC_OK;
}

// scope guard of gwc_total_loglik*: between the build and the dependent calls of one entry point
struct FreshBuild {
  gwc_ctx* c;
  explicit FreshBuild(gwc_ctx* ctx) : c(ctx) { c->fresh_build = true; }
  ~FreshBuild() { c->fresh_build = false; }
};

gwc_status check_theta_args(gwc_ctx* ctx, const double* d_theta, int64_t n_theta) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (!d_theta) return fail(ctx, GWC_ERR_INVALID_ARG, "d_theta is NULL");
  if (n_theta < 1 || n_theta > (int64_t)1 << 24) return fail(ctx, GWC_ERR_SHAPE, "n_theta out of range");
  return GWC_OK;
}

gwc_status check_los(gwc_ctx* ctx, const gwc_los* los, bool need_table, bool need_allsky) {
  if (!los) return fail(ctx, GWC_ERR_INVALID_ARG, "los is NULL");
  if (los->n_z < 2 || los->n_z > 65536) return fail(ctx, GWC_ERR_SHAPE, "los->n_z out of range");
  if (!(los->z_max > 0.0)) return fail(ctx, GWC_ERR_INVALID_ARG, "los->z_max must be positive");
  if (los->prec != GWC_F64 && los->prec != GWC_F32) return fail(ctx, GWC_ERR_INVALID_ARG, "los->prec");
  if (need_table && (!los->table || los->n_rows < 1 || los->n_rows > 0x7fffffffLL))
    return fail(ctx, GWC_ERR_INVALID_ARG, "los->table is NULL or n_rows out of range");
  if (need_allsky && !los->allsky) return fail(ctx, GWC_ERR_INVALID_ARG, "los->allsky is NULL");
  return GWC_OK;
}

}  // namespace

extern "C" {

gwc_status gwc_create(gwc_ctx** out, int device, void* cuda_stream) {
  if (!out) return GWC_ERR_INVALID_ARG;
  *out = nullptr;
  gwc_ctx* ctx = new (std::nothrow) gwc_ctx;
  if (!ctx) return GWC_ERR_NOMEM;
  ctx->device = device;
  ctx->stream = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaSetDevice(device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
  if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_flag, 4 * sizeof(int));   // [0] sticky flags, [1] A0 packing, [2] one-Omega_m answer
  if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->d_counter, sizeof(unsigned int));
  if (e == cudaSuccess) e = cudaMemset(ctx->d_flag, 0, 4 * sizeof(int));
  if (e == cudaSuccess && reweight_configure(ctx->smem_optin) != 0) e = cudaGetLastError();
  if (e != cudaSuccess) {
    g_create_error = std::string("gwc_create: ") + cudaGetErrorString(e);
    cudaGetLastError();
    delete ctx;
    return e == cudaErrorMemoryAllocation ? GWC_ERR_NOMEM : GWC_ERR_CUDA;
  }
  *out = ctx;
  return GWC_OK;
}

void gwc_destroy(gwc_ctx* ctx) {
  if (!ctx) return;
  cudaSetDevice(ctx->device);
  cudaStreamSynchronize(ctx->stream);
  Buf* bufs[] = {&ctx->ftab, &ctx->tab, &ctx->tconst, &ctx->theta_snap, &ctx->tvalid, &ctx->seg_off, &ctx->prep[0].dLc, &ctx->prep[0].L1, &ctx->prep[0].Q,
                 &ctx->prep[0].P, &ctx->prep[0].seg_shift, &ctx->prep[1].dLc, &ctx->prep[1].L1, &ctx->prep[1].Q,
                 &ctx->prep[1].P, &ctx->prep[1].seg_shift,
                 &ctx->injs.dL, &ctx->injs.m1z, &ctx->injs.m2z, &ctx->injs.lp,
                 &ctx->pad.dLc, &ctx->pad.m1z, &ctx->pad.m2z, &ctx->pad.L1, &ctx->pad.Q, &ctx->pad.P, &ctx->pad.row,
                 &ctx->pad.seg_off, &ctx->pad.seg_pads,
                 &ctx->kde_cnt, &ctx->kde_coff, &ctx->kde_cstart, &ctx->kde_cend, &ctx->kde_cev, &ctx->kde_thk, &ctx->kde_gw,
                 &ctx->kde_pe, &ctx->kde_pnp, &ctx->kde_pnu,
                 &ctx->group_off, &ctx->part_w, &ctx->part_n, &ctx->part_np, &ctx->kde_scr, &ctx->kde_len, &ctx->allsky_scr, &ctx->pack_scr, &ctx->logL,
                 &ctx->logxi, &ctx->probe, &ctx->hc.theta, &ctx->hc.ev_off, &ctx->hc.ev_dL, &ctx->hc.ev_m1z,
                 &ctx->hc.ev_m2z, &ctx->hc.ev_lp, &ctx->hc.ev_row, &ctx->hc.inj_dL, &ctx->hc.inj_m1z,
                 &ctx->hc.inj_m2z, &ctx->hc.inj_lp, &ctx->hc.los, &ctx->hc.allsky, &ctx->hc.out};
  for (Buf* b : bufs) release(*b);
  for (cudaEvent_t e : ctx->ev_pairs) cudaEventDestroy(e);
  for (cudaEvent_t e : ctx->inj_pairs) cudaEventDestroy(e);
  for (cudaEvent_t e : ctx->pool) cudaEventDestroy(e);
  if (ctx->d_flag) cudaFree(ctx->d_flag);
  if (ctx->d_counter) cudaFree(ctx->d_counter);
  delete ctx;
}

gwc_status gwc_check(gwc_ctx* ctx) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  GWC_CUDA(cudaStreamSynchronize(ctx->stream));
  int flag = 0;
  GWC_CUDA(cudaMemcpy(&flag, ctx->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
  if (flag) {
    GWC_CUDA(cudaMemset(ctx->d_flag, 0, sizeof(int)));
    if (flag & FLAG_CHK_ANY) {
      char msg[160];
      snprintf(msg, sizeof(msg), "GWC_CHECKED: a device-side bounds / hand-off check failed (flag bits 0x%x, see gwc_internal.h)",
               flag & FLAG_CHK_ANY);
      return fail(ctx, GWC_ERR_CUDA, msg);
    }
    if (flag & FLAG_STALE)
      return fail(ctx, GWC_ERR_NOT_BUILT,
                  "d_theta changed after gwc_build_cosmo: the outputs of the changed points are NaN (rebuild first)");
    if (flag & FLAG_OMEGA)
      return fail(ctx, GWC_ERR_INVALID_ARG,
                  "GWC_OMEGA_SINGLE was promised but a theta batch has several Omega_m or a point outside the domain: "
                  "discard the outputs computed from that build");
    if (flag & FLAG_DOMAIN)
      return fail(ctx, GWC_ERR_DOMAIN, "a theta point is outside the model's domain (its outputs are NaN)");
    if (flag & FLAG_RANGE)
      return fail(ctx, GWC_ERR_RANGE,
                  "the live weights of a segment all lie more than 300 nats below its reference (its outputs are NaN): "
                  "log_pe_prior / log_pdraw has too wide a spread inside one event");
  }
  return GWC_OK;
}

const char* gwc_last_error(const gwc_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int64_t gwc_launch_count(const gwc_ctx* ctx) { return ctx ? ctx->launches : 0; }

gwc_status gwc_set_mass_model(gwc_ctx* ctx, gwc_mass_model model) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (model != GWC_MASS_PLPEAK && model != GWC_MASS_MULTIPEAK) return fail(ctx, GWC_ERR_INVALID_ARG, "unknown mass model");
  ctx->model = (int)model;
  ctx->npar = gwc_theta_len(model);
  ctx->built_theta = nullptr;   // tables and constants of the other model are of no use
  ctx->built_n = 0;
  return GWC_OK;
}

gwc_status gwc_set_omega_hint(gwc_ctx* ctx, gwc_omega_hint hint) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (hint != GWC_OMEGA_DETECT && hint != GWC_OMEGA_VARIES && hint != GWC_OMEGA_SINGLE)
    return fail(ctx, GWC_ERR_INVALID_ARG, "unknown Omega_m hint");
  ctx->omega_hint = (int)hint;
  return GWC_OK;
}

int32_t gwc_theta_len(gwc_mass_model model) {
  return model == GWC_MASS_PLPEAK ? GWC_NPAR : model == GWC_MASS_MULTIPEAK ? GWC_NPAR_MULTIPEAK : 0;
}

gwc_status gwc_build_cosmo(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, double z_max, int32_t n_nodes,
                           gwc_prec table_prec) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!(z_max > 0.0) || !(z_max < 1e4)) return fail(ctx, GWC_ERR_INVALID_ARG, "z_max must be positive and finite");
  if (n_nodes < 2 || n_nodes > MAX_NODES) return fail(ctx, GWC_ERR_SHAPE, "n_nodes must lie in [2, 8193]");
  if (table_prec != GWC_F64 && table_prec != GWC_F32) return fail(ctx, GWC_ERR_INVALID_ARG, "table_prec");
  const int Mp = table_pitch(n_nodes);
  const size_t node = table_prec == GWC_F64 ? sizeof(Node64) : sizeof(Node32);
  ctx->built_theta = nullptr;
  GWC_TRY(ensure(ctx, ctx->tab, (size_t)n_theta * Mp * node));
  GWC_TRY(ensure(ctx, ctx->tconst, (size_t)n_theta * nconst_of(ctx->model) * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->theta_snap, (size_t)n_theta * ctx->npar * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->tvalid, (size_t)n_theta * sizeof(double)));
  if (ctx->model == GWC_MASS_MULTIPEAK) GWC_TRY(ensure(ctx, ctx->ftab, (size_t)n_theta * MF_PITCH * sizeof(Node64)));
  GWC_TRY(count(ctx, launch_cosmo_build(d_theta, n_theta, ctx->model, z_max, n_nodes, Mp, table_prec, ctx->tab.p,
                                        (double*)ctx->tconst.p, (Node64*)ctx->ftab.p, (double*)ctx->theta_snap.p,
                                        (double*)ctx->tvalid.p, ctx->d_flag, ctx->stream),
                "cosmo_build"));
  // One Omega_m in the whole batch (a population-only batch: configs Tiny and O4): z(u) depends on Omega_m alone, so
  // one table serves every theta and a tile holds MAX_T points instead of what fits next to T tables.  Asked of the
  // device (one small kernel and a 4-byte read: the call synchronises) only when it would change the tile.
  ctx->tab_shared = false;
  // (and only for batches of at least four tiles: the synchronisation costs a small batch more than the tile gains)
  if (ctx->omega_hint == GWC_OMEGA_SINGLE) {
    // the caller's promise: shared without waiting; checked on the device, a broken promise raises FLAG_OMEGA
    GWC_TRY(count(ctx, launch_omega_same(d_theta, n_theta, ctx->model, ctx->d_flag + 2, ctx->stream, ctx->d_flag), "omega_same"));
    ctx->tab_shared = true;
  } else if (ctx->omega_hint == GWC_OMEGA_DETECT &&
             n_theta >= 4 * reweight_max_T(Mp, table_prec, false, 2, ctx->smem_optin, false, ctx->model == GWC_MASS_MULTIPEAK, false)) {
    int same = 0;
    GWC_TRY(count(ctx, launch_omega_same(d_theta, n_theta, ctx->model, ctx->d_flag + 2, ctx->stream), "omega_same"));
    GWC_CUDA(cudaMemcpyAsync(&same, ctx->d_flag + 2, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    GWC_CUDA(cudaStreamSynchronize(ctx->stream));
    ctx->tab_shared = same != 0;
  }
  ctx->built_theta = d_theta;
  ctx->built_n = n_theta;
  ctx->M = n_nodes;
  ctx->Mp = Mp;
  ctx->tab_prec = table_prec;
  ctx->z_max = z_max;
  return GWC_OK;
}

gwc_status gwc_export_cosmo(gwc_ctx* ctx, double* d_z, double* d_dz, double* d_umax) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (!ctx->built_theta) return fail(ctx, GWC_ERR_NOT_BUILT, "no cosmology table built");
  return count(ctx, launch_export_cosmo(ctx->tab.p, (const double*)ctx->tconst.p, nconst_of(ctx->model), ctx->built_n, ctx->M, ctx->Mp,
                                        ctx->tab_prec, ctx->z_max, d_z, d_dz, d_umax, ctx->stream),
               "export_cosmo");
}

gwc_status gwc_pack_events(gwc_ctx* ctx, int64_t n_samples, int64_t n_events, const int32_t* d_event_id,
                           const int32_t* d_row, int64_t* d_perm, int64_t* d_ev_sample_off, int64_t* d_ev_pix_off,
                           int32_t* d_ev_pix_rows, int64_t* d_pix_sample_off, int64_t* h_n_pixrefs) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (n_samples < 0 || n_events < 0 || n_events > 0x7fffffffLL) return fail(ctx, GWC_ERR_SHAPE, "sizes out of range");
  if (!d_ev_sample_off || !d_ev_pix_off || !d_pix_sample_off || !h_n_pixrefs)
    return fail(ctx, GWC_ERR_INVALID_ARG, "an output pointer is NULL");
  if (n_samples > 0 && (!d_event_id || !d_row || !d_perm || !d_ev_pix_rows))
    return fail(ctx, GWC_ERR_INVALID_ARG, "an array pointer is NULL");
  const size_t bytes = pack_scratch_bytes(n_samples, n_events);
  GWC_TRY(ensure(ctx, ctx->pack_scr, bytes + 8));
  int64_t* d_np = (int64_t*)((unsigned char*)ctx->pack_scr.p + bytes);
  // the packing has a flag word of its own (d_flag[1]): a theta-domain flag left by an earlier call is neither
  // reported here nor consumed
  GWC_CUDA(cudaMemsetAsync(ctx->d_flag + 1, 0, sizeof(int), ctx->stream));
  GWC_TRY(count(ctx, launch_pack(n_samples, n_events, d_event_id, d_row, d_perm, d_ev_sample_off, d_ev_pix_off,
                                 d_ev_pix_rows, d_pix_sample_off, d_np, ctx->d_flag + 1, ctx->pack_scr.p, bytes,
                                 ctx->stream),
                "pack_events"));
  int bad = 0;
  GWC_CUDA(cudaMemcpyAsync(h_n_pixrefs, d_np, sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->stream));
  GWC_CUDA(cudaMemcpyAsync(&bad, ctx->d_flag + 1, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  GWC_CUDA(cudaStreamSynchronize(ctx->stream));
  if (bad) return fail(ctx, GWC_ERR_DOMAIN, "gwc_pack_events: an event id or row is out of range");
  return GWC_OK;
}

gwc_status gwc_cap_pixels(gwc_ctx* ctx, int64_t n_samples, int64_t n_events, int64_t n_pixrefs,
                          const int64_t* d_perm, int64_t* d_ev_sample_off, int64_t* d_pix_sample_off, int64_t cap,
                          uint64_t seed, int64_t* d_perm_out, int64_t* h_n_kept) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (n_samples < 0 || n_events < 0 || n_pixrefs < 0 || n_pixrefs > n_samples || n_pixrefs > 0x7fffffffLL)
    return fail(ctx, GWC_ERR_SHAPE, "sizes out of range");
  if (cap < 1) return fail(ctx, GWC_ERR_INVALID_ARG, "cap must be >= 1");
  if (!d_ev_sample_off || !d_pix_sample_off || !h_n_kept) return fail(ctx, GWC_ERR_INVALID_ARG, "a pointer is NULL");
  if (n_samples > 0 && (!d_perm || !d_perm_out)) return fail(ctx, GWC_ERR_INVALID_ARG, "a permutation pointer is NULL");
  const size_t bytes = cap_scratch_bytes(n_samples);
  GWC_TRY(ensure(ctx, ctx->pack_scr, bytes + 8));
  int64_t* d_nk = (int64_t*)((unsigned char*)ctx->pack_scr.p + bytes);
  GWC_TRY(count(ctx, launch_cap_pixels(n_samples, n_events, n_pixrefs, d_perm, d_ev_sample_off, d_pix_sample_off, cap,
                                       seed, d_perm_out, d_nk, ctx->pack_scr.p, bytes, ctx->stream),
                "cap_pixels"));
  GWC_CUDA(cudaMemcpyAsync(h_n_kept, d_nk, sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->stream));
  GWC_CUDA(cudaStreamSynchronize(ctx->stream));
  return GWC_OK;
}

gwc_status gwc_los_allsky(gwc_ctx* ctx, const gwc_los* los, double* d_allsky) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  GWC_TRY(check_los(ctx, los, true, false));
  if (!d_allsky) return fail(ctx, GWC_ERR_INVALID_ARG, "d_allsky is NULL");
  GWC_TRY(ensure(ctx, ctx->allsky_scr, allsky_scratch_doubles(los->n_rows, los->n_z) * sizeof(double)));
  return count(ctx, launch_allsky(los->table, los->prec, los->n_rows, los->n_z, (double*)ctx->allsky_scr.p, d_allsky,
                                  ctx->stream),
               "los_allsky");
}

gwc_status gwc_event_loglik(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                            const gwc_los* los, double* d_logL, double* d_neff, int64_t* d_nlive) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!ev || !d_logL) return fail(ctx, GWC_ERR_INVALID_ARG, "ev or d_logL is NULL");
  GWC_TRY(check_los(ctx, los, true, false));
  if (ev->n_events < 0 || ev->n_samples < 0 || ev->n_events > 0x7fffffffLL)
    return fail(ctx, GWC_ERR_SHAPE, "event / sample counts out of range");
  if (ev->n_events == 0) return GWC_OK;
  if (!ev->ev_sample_off) return fail(ctx, GWC_ERR_INVALID_ARG, "ev->ev_sample_off is NULL");
  if (ev->n_samples > 0 && (!ev->dL || !ev->m1z || !ev->m2z || !ev->sample_row))
    return fail(ctx, GWC_ERR_INVALID_ARG, "a sample array is NULL");
  GWC_TRY(check_built(ctx, d_theta, n_theta, los->z_max));
  GWC_TRY(run_reweight(ctx, n_theta, ev->n_samples, ev->n_events, ev->ev_sample_off, ev->dL, ev->m1z, ev->m2z,
                       ev->log_pe_prior, ev->sample_row, los->table, los->prec, los->n_rows, los->n_z, los->z_max,
                       false));
  return count(ctx, launch_finalize_events((const double*)ctx->part_w.p, (const int32_t*)ctx->part_n.p,
                                           ev->ev_sample_off, (const double*)ctx->prep[0].seg_shift.p,
                                           (const double*)ctx->tvalid.p, n_theta, ev->n_events, d_logL, d_neff,
                                           d_nlive, ctx->d_flag, ctx->stream),
               "finalize_events");
}

gwc_status gwc_event_loglik_pixcut(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                   const gwc_los* los, double neff_min, double* d_logL, double* d_neff,
                                   int64_t* d_nlive, int64_t* d_npass) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!ev || !d_logL) return fail(ctx, GWC_ERR_INVALID_ARG, "ev or d_logL is NULL");
  if (!(neff_min >= 0.0)) return fail(ctx, GWC_ERR_INVALID_ARG, "neff_min must be >= 0");
  GWC_TRY(check_los(ctx, los, true, false));
  if (ev->n_events < 0 || ev->n_samples < 0 || ev->n_events > 0x7fffffffLL)
    return fail(ctx, GWC_ERR_SHAPE, "event / sample counts out of range");
  if (ev->n_events == 0) return GWC_OK;
  if (!ev->ev_sample_off) return fail(ctx, GWC_ERR_INVALID_ARG, "ev->ev_sample_off is NULL");
  if (ev->n_samples > 0 && (!ev->dL || !ev->m1z || !ev->m2z || !ev->sample_row))
    return fail(ctx, GWC_ERR_INVALID_ARG, "a sample array is NULL");
  GWC_TRY(check_built(ctx, d_theta, n_theta, los->z_max));
  GWC_TRY(run_reweight(ctx, n_theta, ev->n_samples, ev->n_events, ev->ev_sample_off, ev->dL, ev->m1z, ev->m2z,
                       ev->log_pe_prior, ev->sample_row, los->table, los->prec, los->n_rows, los->n_z, los->z_max,
                       false, true, neff_min));
  GWC_TRY(count(ctx, launch_finalize_events((const double*)ctx->part_w.p, (const int32_t*)ctx->part_n.p,
                                            ev->ev_sample_off, (const double*)ctx->prep[0].seg_shift.p,
                                            (const double*)ctx->tvalid.p, n_theta, ev->n_events, d_logL, d_neff,
                                            d_nlive, ctx->d_flag, ctx->stream),
                "finalize_events"));
  if (d_npass)
    GWC_TRY(count(ctx, launch_widen_i32((const int32_t*)ctx->part_np.p, (const double*)ctx->tvalid.p, n_theta,
                                        ev->n_events, d_npass, ctx->stream),
                  "widen_npass"));
  return GWC_OK;
}

gwc_status gwc_event_loglik_kde(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                const gwc_los* los, int32_t n_grid, double neff_min, int32_t bw_rule, double* d_logL,
                                int64_t* d_npass, int64_t* d_nused) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!ev || !d_logL) return fail(ctx, GWC_ERR_INVALID_ARG, "ev or d_logL is NULL");
  if (!(neff_min >= 0.0)) return fail(ctx, GWC_ERR_INVALID_ARG, "neff_min must be >= 0");
  if (n_grid < 2 || n_grid > 256) return fail(ctx, GWC_ERR_SHAPE, "n_grid must be in [2, 256]");
  if (bw_rule < GWC_BW_SCOTT || bw_rule > GWC_BW_BIWEIGHT_SCOTT) return fail(ctx, GWC_ERR_INVALID_ARG, "unknown bw_rule");
  GWC_TRY(check_los(ctx, los, true, false));
  if (ev->n_events < 0 || ev->n_samples < 0 || ev->n_events > 0x7fffffffLL)
    return fail(ctx, GWC_ERR_SHAPE, "event / sample counts out of range");
  if (ev->n_events == 0) return GWC_OK;
  if (!ev->ev_sample_off) return fail(ctx, GWC_ERR_INVALID_ARG, "ev->ev_sample_off is NULL");
  if (ev->n_samples > 0 && (!ev->dL || !ev->m1z || !ev->m2z || !ev->sample_row))
    return fail(ctx, GWC_ERR_INVALID_ARG, "a sample array is NULL");
  GWC_TRY(check_built(ctx, d_theta, n_theta, los->z_max));
  // the per-event reference of the linear-domain sums (and nothing else) comes from the sample preparation
  cudaStream_t s = ctx->stream;
  const int64_t n = ev->n_samples, n_seg = ev->n_events;
  GWC_TRY(prepare_samples(ctx, ctx->prep[0], n, n_seg, ev->ev_sample_off, ev->dL, ev->m1z, ev->m2z, ev->log_pe_prior,
                          ev->sample_row, los->n_rows));
  // work units are (chunk, theta): the chunk table of the catalogue (runs of whole pixels of about 1024 samples), then
  // one host synchronisation for its size and the longest chunk (the scratch slice of a warp)
  const int64_t nc_max = kde_chunk_bound(n, n_seg);
  GWC_TRY(ensure(ctx, ctx->kde_len, 2 * sizeof(int64_t)));
  GWC_TRY(ensure(ctx, ctx->kde_cnt, (size_t)n_seg * sizeof(int64_t)));
  GWC_TRY(ensure(ctx, ctx->kde_coff, (size_t)(n_seg + 1) * sizeof(int64_t)));
  GWC_TRY(ensure(ctx, ctx->kde_cstart, (size_t)nc_max * sizeof(int64_t)));
  GWC_TRY(ensure(ctx, ctx->kde_cend, (size_t)nc_max * sizeof(int64_t)));
  GWC_TRY(ensure(ctx, ctx->kde_cev, (size_t)nc_max * sizeof(int32_t)));
  GWC_CUDA(cudaMemsetAsync(ctx->kde_len.p, 0, 2 * sizeof(int64_t), s));
  GWC_TRY(count(ctx, launch_kde_chunks(ev->ev_sample_off, n_seg, ev->sample_row, (int64_t*)ctx->kde_cnt.p,
                                       (int64_t*)ctx->kde_coff.p, (int64_t*)ctx->kde_cstart.p, (int64_t*)ctx->kde_cend.p,
                                       (int32_t*)ctx->kde_cev.p, (int64_t*)ctx->kde_len.p, n, s),
                "kde_chunks"));
  int64_t len_bad[2] = {0, 0}, n_chunks = 0;
  GWC_CUDA(cudaMemcpyAsync(len_bad, ctx->kde_len.p, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, s));
  GWC_CUDA(cudaMemcpyAsync(&n_chunks, (const int64_t*)ctx->kde_coff.p + n_seg, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
  GWC_CUDA(cudaStreamSynchronize(s));
  const int64_t max_len = len_bad[0];
  if (len_bad[1] != 0 || max_len < 0 || max_len > n || n_chunks < 0 || n_chunks > nc_max)
    return fail(ctx, GWC_ERR_SHAPE, "ev_sample_off is not ascending inside [0, n_samples]");
  const int n_blocks = kde_grid_blocks(n_theta, n_chunks, ctx->n_sm);
  GWC_TRY(ensure(ctx, ctx->kde_scr, kde_scratch_bytes(n_blocks, max_len)));
  GWC_TRY(ensure(ctx, ctx->kde_thk, kde_theta_bytes(n_theta)));
  GWC_TRY(ensure(ctx, ctx->kde_gw, kde_weight_bytes(n_theta)));
  const size_t n_part = (size_t)n_theta * (size_t)(n_chunks > 0 ? n_chunks : 1);
  GWC_TRY(ensure(ctx, ctx->kde_pe, n_part * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->kde_pnp, n_part * sizeof(int32_t)));
  GWC_TRY(ensure(ctx, ctx->kde_pnu, n_part * sizeof(int64_t)));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (ctx->timing) {   // (taken after the last step that can fail before the launch: nothing leaks on an error return)
    e0 = get_event(ctx);
    e1 = get_event(ctx);
    cudaEventRecord(e0, s);
  }
  // the population parameters come from the copy of theta the tables were built from, never from a changed array
  const gwc_status st_kde = count(ctx, launch_kde(ctx->model, (const Node64*)ctx->ftab.p, (const double*)ctx->theta_snap.p, ctx->tab.p, (const double*)ctx->tconst.p, (const double*)ctx->tvalid.p, n_theta, ctx->M, ctx->Mp,
                                ctx->tab_prec, ctx->z_max / NODE32_QMAX, ev->n_events, ev->ev_sample_off, ev->dL,
                                ev->m1z, ev->m2z, ev->log_pe_prior, ev->sample_row, (const double*)ctx->prep[0].seg_shift.p,
                                los->table, los->prec, los->n_rows, los->n_z, los->z_max, n_grid, neff_min, bw_rule,
                                d_logL,
                                d_npass, d_nused, ctx->kde_scr.p, max_len > 0 ? max_len : 1, n_blocks, n_chunks,
                                (const int64_t*)ctx->kde_coff.p, (const int64_t*)ctx->kde_cstart.p,
                                (const int64_t*)ctx->kde_cend.p, (const int32_t*)ctx->kde_cev.p, ctx->kde_thk.p,
                                ctx->kde_gw.p, (double*)ctx->kde_pe.p, (int32_t*)ctx->kde_pnp.p, (int64_t*)ctx->kde_pnu.p,
                                ctx->d_flag, s),
                "kde");
  if (ctx->timing) {
    cudaEventRecord(e1, s);
    ctx->ev_pairs.push_back(e0);
    ctx->ev_pairs.push_back(e1);
  }
  return st_kde;
}

gwc_status gwc_selection_logxi(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_injections* inj,
                               const gwc_los* los, double* d_logxi, double* d_neff_inj) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!inj || !d_logxi) return fail(ctx, GWC_ERR_INVALID_ARG, "inj or d_logxi is NULL");
  GWC_TRY(check_los(ctx, los, false, true));
  if (inj->n_found < 0) return fail(ctx, GWC_ERR_SHAPE, "n_found < 0");
  if (!(inj->n_draw > 0.0)) return fail(ctx, GWC_ERR_INVALID_ARG, "n_draw must be positive");
  if (inj->n_found > 0 && (!inj->dL || !inj->m1z || !inj->m2z || !inj->log_pdraw))
    return fail(ctx, GWC_ERR_INVALID_ARG, "an injection array is NULL");
  if (los->n_z > GWC_MAX_NZ_SELECTION)
    return fail(ctx, GWC_ERR_SHAPE, "los->n_z > 4096 is not supported by the selection term (all-sky table in shared memory)");
  GWC_TRY(check_built(ctx, d_theta, n_theta, los->z_max));
  const int64_t n = inj->n_found;
  const int64_t n_seg = n > 0 ? (n + INJ_SEG - 1) / INJ_SEG : 1;
  GWC_TRY(ensure(ctx, ctx->seg_off, (size_t)(n_seg + 1) * sizeof(int64_t)));
  GWC_TRY(count(ctx, launch_uniform_segments(n, INJ_SEG, n_seg, (int64_t*)ctx->seg_off.p, ctx->stream),
                "uniform_segments"));
  // the injections in order of d_L (whole warps then leave a theta's table together); kept with the catalogue cache.
  // Only when the call is large enough to pay for the sort (about 0.1 ms + 0.1 ns per injection against 8 % of the
  // selection kernel): 2e8 (theta x injection) terms and up.
  const bool sort_inj = (double)n * (double)n_theta >= 2e8;
  InjSorted& js = ctx->injs;
  if (!sort_inj) {
    GWC_TRY(run_reweight(ctx, n_theta, n, n_seg, (const int64_t*)ctx->seg_off.p, inj->dL, inj->m1z, inj->m2z,
                         inj->log_pdraw, nullptr, los->allsky, GWC_F64, 1, los->n_z, los->z_max, true));
  } else {
  if (!(ctx->cache_prep && js.valid && js.k_dL == inj->dL && js.k_m1z == inj->m1z && js.k_m2z == inj->m2z &&
        js.k_lp == inj->log_pdraw && js.k_n == n)) {
    js.valid = false;
    ctx->prep[1].valid = false;   // (the sorted buffers keep their addresses while their contents change)
    const size_t nd = (size_t)(n > 0 ? n : 1) * sizeof(double);
    GWC_TRY(ensure(ctx, js.dL, nd));
    GWC_TRY(ensure(ctx, js.m1z, nd));
    GWC_TRY(ensure(ctx, js.m2z, nd));
    GWC_TRY(ensure(ctx, js.lp, nd));
    const size_t sb = injsort_scratch_bytes(n);
    GWC_TRY(ensure(ctx, ctx->pack_scr, sb));
    GWC_TRY(count(ctx, launch_injsort(n, inj->dL, inj->m1z, inj->m2z, inj->log_pdraw, (double*)js.dL.p, (double*)js.m1z.p,
                                      (double*)js.m2z.p, (double*)js.lp.p, ctx->pack_scr.p, sb, ctx->stream),
                  "injsort"));
    js.k_dL = inj->dL; js.k_m1z = inj->m1z; js.k_m2z = inj->m2z; js.k_lp = inj->log_pdraw; js.k_n = n;
    js.valid = true;
  }
  GWC_TRY(run_reweight(ctx, n_theta, n, n_seg, (const int64_t*)ctx->seg_off.p, (const double*)js.dL.p,
                       (const double*)js.m1z.p, (const double*)js.m2z.p, (const double*)js.lp.p, nullptr, los->allsky,
                       GWC_F64, 1, los->n_z, los->z_max, true));
  }
  return count(ctx, launch_finalize_inj((const double*)ctx->part_w.p, (const int32_t*)ctx->part_n.p,
                                        (const double*)ctx->prep[1].seg_shift.p, (const double*)ctx->tvalid.p, n_theta,
                                        n_seg, inj->n_draw, d_logxi, d_neff_inj, ctx->d_flag, ctx->stream),
               "finalize_inj");
}

gwc_status gwc_combine_total(gwc_ctx* ctx, const double* d_logL, const double* d_logxi, int64_t n_theta,
                             int64_t n_events, double* d_total) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (!d_logxi || !d_total || (n_events > 0 && !d_logL)) return fail(ctx, GWC_ERR_INVALID_ARG, "NULL pointer");
  if (n_theta < 1 || n_events < 0) return fail(ctx, GWC_ERR_SHAPE, "sizes out of range");
  return count(ctx, launch_combine_total(d_logL, d_logxi, n_theta, n_events, d_total, ctx->stream), "combine_total");
}

gwc_status gwc_combine_sharded(gwc_ctx* ctx, int32_t n_parts, int64_t n_theta, int64_t n_events_total,
                               const double* d_sum_logL_parts, const double* d_logxi_parts,
                               const double* d_neff_inj_parts, double* d_total, double* d_logxi, double* d_neff_inj) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (!d_sum_logL_parts || !d_logxi_parts) return fail(ctx, GWC_ERR_INVALID_ARG, "NULL pointer");
  if (d_neff_inj && !d_neff_inj_parts) return fail(ctx, GWC_ERR_INVALID_ARG, "d_neff_inj needs d_neff_inj_parts");
  if (n_parts < 1 || n_parts > 65536 || n_theta < 1 || n_events_total < 0)
    return fail(ctx, GWC_ERR_SHAPE, "sizes out of range");
  return count(ctx, launch_combine_sharded(d_sum_logL_parts, d_logxi_parts, d_neff_inj_parts, n_parts, n_theta,
                                           n_events_total, d_total, d_logxi, d_neff_inj, ctx->stream),
               "combine_sharded");
}

gwc_status gwc_combine_sharded_host(int32_t n_parts, int64_t n_theta, int64_t n_events_total,
                                    const double* h_sum_logL_parts, const double* h_logxi_parts,
                                    const double* h_neff_inj_parts, double* h_total, double* h_logxi,
                                    double* h_neff_inj) {
  if (!h_sum_logL_parts || !h_logxi_parts || (h_neff_inj && !h_neff_inj_parts)) return GWC_ERR_INVALID_ARG;
  if (n_parts < 1 || n_parts > 65536 || n_theta < 1 || n_events_total < 0) return GWC_ERR_SHAPE;
  combine_sharded_host(h_sum_logL_parts, h_logxi_parts, h_neff_inj_parts, n_parts, n_theta, n_events_total, h_total,
                       h_logxi, h_neff_inj);
  return GWC_OK;
}

gwc_status gwc_total_loglik(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                            const gwc_injections* inj, const gwc_los* los, int32_t n_nodes, gwc_prec table_prec,
                            double* d_logL_total) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!ev || !inj || !d_logL_total) return fail(ctx, GWC_ERR_INVALID_ARG, "NULL argument");
  GWC_TRY(check_los(ctx, los, true, true));
  if (los->n_z > GWC_MAX_NZ_SELECTION)   // before any work: the selection term at the end would refuse it
    return fail(ctx, GWC_ERR_SHAPE, "los->n_z > 4096 is not supported by the selection term");
  GWC_TRY(gwc_build_cosmo(ctx, d_theta, n_theta, los->z_max, n_nodes, table_prec));
  const int64_t E = ev->n_events;
  GWC_TRY(ensure(ctx, ctx->logL, (size_t)n_theta * (size_t)(E > 0 ? E : 1) * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->logxi, (size_t)n_theta * sizeof(double)));
  FreshBuild fresh(ctx);   // the tables were enqueued by this call on this stream: no verification launches
  GWC_TRY(gwc_event_loglik(ctx, d_theta, n_theta, ev, los, (double*)ctx->logL.p, nullptr, nullptr));
  GWC_TRY(gwc_selection_logxi(ctx, d_theta, n_theta, inj, los, (double*)ctx->logxi.p, nullptr));
  return gwc_combine_total(ctx, (const double*)ctx->logL.p, (const double*)ctx->logxi.p, n_theta, E, d_logL_total);
}

gwc_status gwc_total_loglik_pixcut(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                   const gwc_injections* inj, const gwc_los* los, int32_t n_nodes,
                                   gwc_prec table_prec, double neff_min, double* d_logL_total) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!ev || !inj || !d_logL_total) return fail(ctx, GWC_ERR_INVALID_ARG, "NULL argument");
  GWC_TRY(check_los(ctx, los, true, true));
  if (los->n_z > GWC_MAX_NZ_SELECTION)
    return fail(ctx, GWC_ERR_SHAPE, "los->n_z > 4096 is not supported by the selection term");
  GWC_TRY(gwc_build_cosmo(ctx, d_theta, n_theta, los->z_max, n_nodes, table_prec));
  const int64_t E = ev->n_events;
  GWC_TRY(ensure(ctx, ctx->logL, (size_t)n_theta * (size_t)(E > 0 ? E : 1) * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->logxi, (size_t)n_theta * sizeof(double)));
  FreshBuild fresh(ctx);
  GWC_TRY(gwc_event_loglik_pixcut(ctx, d_theta, n_theta, ev, los, neff_min, (double*)ctx->logL.p, nullptr, nullptr,
                                  nullptr));
  GWC_TRY(gwc_selection_logxi(ctx, d_theta, n_theta, inj, los, (double*)ctx->logxi.p, nullptr));
  return gwc_combine_total(ctx, (const double*)ctx->logL.p, (const double*)ctx->logxi.p, n_theta, E, d_logL_total);
}

gwc_status gwc_total_loglik_kde(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                const gwc_injections* inj, const gwc_los* los, int32_t n_nodes, gwc_prec table_prec,
                                int32_t n_grid, double neff_min, int32_t bw_rule, double* d_logL_total) {
  GWC_TRY(check_theta_args(ctx, d_theta, n_theta));
  if (!ev || !inj || !d_logL_total) return fail(ctx, GWC_ERR_INVALID_ARG, "NULL argument");
  GWC_TRY(check_los(ctx, los, true, true));
  if (los->n_z > GWC_MAX_NZ_SELECTION)
    return fail(ctx, GWC_ERR_SHAPE, "los->n_z > 4096 is not supported by the selection term");
  GWC_TRY(gwc_build_cosmo(ctx, d_theta, n_theta, los->z_max, n_nodes, table_prec));
  const int64_t E = ev->n_events;
  GWC_TRY(ensure(ctx, ctx->logL, (size_t)n_theta * (size_t)(E > 0 ? E : 1) * sizeof(double)));
  GWC_TRY(ensure(ctx, ctx->logxi, (size_t)n_theta * sizeof(double)));
  FreshBuild fresh(ctx);
  GWC_TRY(gwc_event_loglik_kde(ctx, d_theta, n_theta, ev, los, n_grid, neff_min, bw_rule, (double*)ctx->logL.p,
                               nullptr, nullptr));
  GWC_TRY(gwc_selection_logxi(ctx, d_theta, n_theta, inj, los, (double*)ctx->logxi.p, nullptr));
  return gwc_combine_total(ctx, (const double*)ctx->logL.p, (const double*)ctx->logxi.p, n_theta, E, d_logL_total);
}

gwc_status gwc_total_loglik_host(gwc_ctx* ctx, const double* h_theta, int64_t n_theta, const gwc_events* h_ev,
                                 const gwc_injections* h_inj, const gwc_los* h_los, int32_t n_nodes,
                                 gwc_prec table_prec, double* h_logL_total, int64_t* h2d_bytes, int64_t* d2h_bytes) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  if (!h_theta || !h_ev || !h_inj || !h_los || !h_logL_total) return fail(ctx, GWC_ERR_INVALID_ARG, "NULL argument");
  if (n_theta < 1) return fail(ctx, GWC_ERR_SHAPE, "n_theta out of range");
  GWC_TRY(check_los(ctx, h_los, true, false));
  if (h_ev->n_events < 0 || h_ev->n_samples < 0 || h_inj->n_found < 0) return fail(ctx, GWC_ERR_SHAPE, "negative size");
  if (h_ev->n_events > 0 && !h_ev->ev_sample_off) return fail(ctx, GWC_ERR_INVALID_ARG, "ev_sample_off is NULL");
  if (h_ev->n_samples > 0 && (!h_ev->dL || !h_ev->m1z || !h_ev->m2z || !h_ev->sample_row))
    return fail(ctx, GWC_ERR_INVALID_ARG, "a sample array is NULL");
  if (h_inj->n_found > 0 && (!h_inj->dL || !h_inj->m1z || !h_inj->m2z || !h_inj->log_pdraw))
    return fail(ctx, GWC_ERR_INVALID_ARG, "an injection array is NULL");
  cudaStream_t s = ctx->stream;
  HostCopy& h = ctx->hc;
  int64_t up = 0;
  auto upload = [&](Buf& b, const void* src, size_t bytes) -> gwc_status {
    GWC_TRY(ensure(ctx, b, bytes > 0 ? bytes : 8));
    if (bytes > 0) {
      GWC_CUDA(cudaMemcpyAsync(b.p, src, bytes, cudaMemcpyHostToDevice, s));
      up += (int64_t)bytes;
    }
    return GWC_OK;
  };
  const size_t ns = (size_t)h_ev->n_samples, ni = (size_t)h_inj->n_found;
  const size_t los_el = h_los->prec == GWC_F64 ? 8 : 4;
  GWC_TRY(upload(h.theta, h_theta, (size_t)n_theta * ctx->npar * 8));
  GWC_TRY(upload(h.ev_off, h_ev->ev_sample_off, (size_t)(h_ev->n_events + 1) * 8));
  GWC_TRY(upload(h.ev_dL, h_ev->dL, ns * 8));
  GWC_TRY(upload(h.ev_m1z, h_ev->m1z, ns * 8));
  GWC_TRY(upload(h.ev_m2z, h_ev->m2z, ns * 8));
  if (h_ev->log_pe_prior) GWC_TRY(upload(h.ev_lp, h_ev->log_pe_prior, ns * 8));
  GWC_TRY(upload(h.ev_row, h_ev->sample_row, ns * 4));
  GWC_TRY(upload(h.inj_dL, h_inj->dL, ni * 8));
  GWC_TRY(upload(h.inj_m1z, h_inj->m1z, ni * 8));
  GWC_TRY(upload(h.inj_m2z, h_inj->m2z, ni * 8));
  GWC_TRY(upload(h.inj_lp, h_inj->log_pdraw, ni * 8));
  GWC_TRY(upload(h.los, h_los->table, (size_t)h_los->n_rows * h_los->n_z * los_el));
  GWC_TRY(ensure(ctx, h.allsky, (size_t)h_los->n_z * 8));
  GWC_TRY(ensure(ctx, h.out, (size_t)n_theta * 8));
  gwc_events ev = *h_ev;
  ev.ev_sample_off = (const int64_t*)h.ev_off.p;
  ev.dL = (const double*)h.ev_dL.p;
  ev.m1z = (const double*)h.ev_m1z.p;
  ev.m2z = (const double*)h.ev_m2z.p;
  ev.log_pe_prior = h_ev->log_pe_prior ? (const double*)h.ev_lp.p : nullptr;
  ev.sample_row = (const int32_t*)h.ev_row.p;
  ev.ev_pix_off = nullptr;
  ev.ev_pix_rows = nullptr;
  gwc_injections inj = *h_inj;
  inj.dL = (const double*)h.inj_dL.p;
  inj.m1z = (const double*)h.inj_m1z.p;
  inj.m2z = (const double*)h.inj_m2z.p;
  inj.log_pdraw = (const double*)h.inj_lp.p;
  gwc_los los = *h_los;
  los.table = h.los.p;
  los.allsky = (const double*)h.allsky.p;
  if (h_los->allsky) {
    GWC_CUDA(cudaMemcpyAsync(h.allsky.p, h_los->allsky, (size_t)h_los->n_z * 8, cudaMemcpyHostToDevice, s));
    up += (int64_t)h_los->n_z * 8;
  } else {
    GWC_TRY(gwc_los_allsky(ctx, &los, (double*)h.allsky.p));
  }
  // the mirrors keep their addresses from one call to the next while their contents change: the cached preparation
  // (gwc_cache_catalogue) must not match them
  ctx->prep[0].valid = false;
  ctx->prep[1].valid = false;
  ctx->pad.valid = false;
  ctx->injs.valid = false;
  const gwc_status st_run = gwc_total_loglik(ctx, (const double*)h.theta.p, n_theta, &ev, &inj, &los, n_nodes,
                                             table_prec, (double*)h.out.p);
  ctx->prep[0].valid = false;
  ctx->prep[1].valid = false;
  ctx->pad.valid = false;
  ctx->injs.valid = false;
  ctx->built_theta = nullptr;  // the mirrored theta buffer is internal: do not let later calls match it
  GWC_TRY(st_run);
  GWC_CUDA(cudaMemcpyAsync(h_logL_total, h.out.p, (size_t)n_theta * 8, cudaMemcpyDeviceToHost, s));
  GWC_CUDA(cudaStreamSynchronize(s));
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = n_theta * 8;
  return GWC_OK;
}

gwc_status gwc_cache_catalogue(gwc_ctx* ctx, int on) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  ctx->cache_prep = on != 0;
  ctx->prep[0].valid = false;
  ctx->prep[1].valid = false;
  ctx->pad.valid = false;
  ctx->injs.valid = false;
  return GWC_OK;
}

gwc_status gwc_set_timing(gwc_ctx* ctx, int on) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  ctx->timing = on != 0;
  return GWC_OK;
}

gwc_status gwc_get_timing(gwc_ctx* ctx, int64_t* n_ev_launches, double* ms_ev, int64_t* n_inj_launches,
                          double* ms_inj) {
  if (!ctx) return GWC_ERR_INVALID_ARG;
  GWC_CUDA(cudaStreamSynchronize(ctx->stream));
  auto drain = [&](std::vector<cudaEvent_t>& v, int64_t* n, double* ms) {
    double tot = 0.0;
    for (size_t i = 0; i + 1 < v.size(); i += 2) {
      float t = 0.f;
      cudaEventElapsedTime(&t, v[i], v[i + 1]);
      tot += t;
    }
    if (n) *n = (int64_t)(v.size() / 2);
    if (ms) *ms = tot;
    for (cudaEvent_t e : v) ctx->pool.push_back(e);
    v.clear();
  };
  drain(ctx->ev_pairs, n_ev_launches, ms_ev);
  drain(ctx->inj_pairs, n_inj_launches, ms_inj);
  return GWC_OK;
}

gwc_status gwc_probe_fp64(gwc_ctx* ctx, int64_t iters, double* ms, double* n_fp64_instr) {
  if (!ctx || !ms || !n_fp64_instr || iters < 1) return GWC_ERR_INVALID_ARG;
  GWC_TRY(ensure(ctx, ctx->probe, 64));
  cudaEvent_t e0 = get_event(ctx), e1 = get_event(ctx);
  double n = 0.0;
  // warm-up launch, then the timed one
  GWC_TRY(count(ctx, launch_probe_fp64(iters / 8 + 1, ctx->n_sm, (double*)ctx->probe.p, ctx->stream, &n), "probe"));
  cudaEventRecord(e0, ctx->stream);
  GWC_TRY(count(ctx, launch_probe_fp64(iters, ctx->n_sm, (double*)ctx->probe.p, ctx->stream, &n), "probe"));
  cudaEventRecord(e1, ctx->stream);
  GWC_CUDA(cudaStreamSynchronize(ctx->stream));
  float t = 0.f;
  cudaEventElapsedTime(&t, e0, e1);
  ctx->pool.push_back(e0);
  ctx->pool.push_back(e1);
  *ms = t;
  *n_fp64_instr = n;
  return GWC_OK;
}

gwc_status gwc_math_selftest(gwc_ctx* ctx, int which, int64_t n, const double* d_in, double* d_out) {
  if (!ctx || !d_in || !d_out || n < 0) return GWC_ERR_INVALID_ARG;
  return count(ctx, launch_math_selftest(which, n, d_in, d_out, ctx->stream), "math_selftest");
}

}  // extern "C"
