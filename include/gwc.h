/*
 * gwc.h -- C ABI of the B200-native dark-siren hierarchical likelihood (libgwc.so).
 *
 * The operation is the one stated in arxiv/paper_2605_23538, evaluated for a BATCH of
 * hyper-parameter points theta (the paper's Lambda):
 *
 *   log L(theta) = sum_i log L_i(theta) - N_det * log xi(theta)          Eq. 3
 *   L_i   = (1/S_i) sum_k w_ik,  w = p(z, m1, m2 | theta) p(z | pixel) / (J pi_PE)   Eq. 5, 7, :77-91
 *   xi    = (1/N_draw) sum_j w_j over found injections, all-sky p(z)      Eq. 4
 *   N_eff = (sum w)^2 / sum w^2                                           Eq. 8
 *   z from d_L through flat-LambdaCDM Eq. 1, inverted by a per-theta table.
 *
 * The line-of-sight prior is read at each sample's own redshift (direct Monte-Carlo sum, the
 * zero-bandwidth limit of the KDE of Eq. 6; reading R1).  The power-law+peak mass law,
 * the Madau-Dickinson rate, the Jacobian and the table scheme are DESIGN.md readings R2-R9.
 *
 * Conventions
 *  - Plain C ABI; no exception crosses it.  Every function returns a gwc_status; gwc_last_error()
 *    gives text for the last non-OK status of that context.
 *  - Pointers named d_* are DEVICE pointers owned by the caller (e.g. PyTorch tensors); h_* are HOST
 *    pointers.  The library never frees caller memory and keeps no reference to it after a call
 *    returns (work already enqueued on the stream still reads it: keep it alive until you sync).
 *  - All work is enqueued on the CUDA stream given to gwc_create and is asynchronous unless stated.
 *    Scratch memory lives in the context and only grows (cudaMalloc happens when a size grows).
 *  - Argument errors that the host can see are returned synchronously.  theta-domain violations
 *    (H0<=0, Om not in (0,1], sigma<=0, mmin<=0, mmin>=mmax, lambda not in [0,1], zp<=-1, any
 *    non-finite value, |alpha-1|<1e-6, |beta+1|<1e-6) make that theta's outputs NaN and raise a
 *    sticky device flag that gwc_check() reports as GWC_ERR_DOMAIN.  They are the only source of NaN.
 *    -inf is a legal output (no live sample).
 *  - Units: d_L in Mpc, masses in solar masses (detector frame), H0 in km/s/Mpc.
 *  - Results are deterministic: no floating-point atomics, every reduction has a fixed order.
 *  - Range (R23): the sums of an event (of a block of 8192 injections) are taken in the linear domain in
 *    FP64, relative to a reference fixed before theta is known: max over its valid samples of
 *    (-log_pe_prior - ln m1z).  The result is exact to the stated tolerances as long as the largest live weight
 *    of the event lies within 300 nats of that reference -- true of any physical input, whose spread inside one
 *    event is a few nats.  When a log_pe_prior / log_pdraw of enormous spread breaks this (every live weight more
 *    than 300 nats below the reference), the outputs of that (theta, event) are NaN and gwc_check() returns
 *    GWC_ERR_RANGE; nothing is clamped silently.  (Single weights more than 700 nats below the reference count as
 *    e^-700 of it, far below the rounding of the sum.  A block of injections in that state is simply left out when
 *    even an upper bound of its sum lies 60 nats under the largest block of that theta: it cannot change log xi;
 *    only a block that could matter makes log xi NaN.  gwc_event_loglik_pixcut decides per pixel: a pixel whose
 *    own weights all lie more than 300 nats below its event's reference may be counted wrongly in d_npass /
 *    d_nlive while contributing nothing to log L_i.)
 *  - theta and the tables: gwc_build_cosmo keeps, next to the tables, a copy of the theta rows it was given.  The
 *    calls that need the tables take the same d_theta pointer and count (else GWC_ERR_NOT_BUILT at once) and
 *    compare the rows on the device with that copy: a row that was changed in place since the build (or a new
 *    array that landed at the same address) gets NaN outputs and gwc_check() returns GWC_ERR_NOT_BUILT.  Any
 *    change to theta needs a new gwc_build_cosmo.  A later build (other n_nodes / table_prec / z_max) replaces
 *    the earlier one: the dependent calls always use the latest.
 *  - Streams: every context enqueues on its own stream, and several contexts may be used from several host
 *    threads.  The fused re-weighting kernels of ALL contexts on one device run one after the other (they share
 *    the device's constant bank for the per-theta constants; each launch waits for the previous one through an
 *    event, whichever stream it was on).  Each of them fills the GPU, so nothing is lost.  A single context
 *    must not be used from two threads at the same time.
 */
#ifndef GWC_H_
#define GWC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GWC_NPAR 12 /* theta row: H0, Om, alpha, beta, mmin, mmax, mu, sigma, lambda, gamma, kappa, zp */
/* MULTIPEAK theta row (gwc_set_mass_model): the 12 columns above, in which (mu, sigma) are the HIGH Gaussian peak and
 * lambda is lambda_g, the fraction in the two peaks; then delta_m, mu_g,low, sigma_g,low, lambda_g,low (the share of
 * lambda_g in the low peak).  Table III. */
#define GWC_NPAR_MULTIPEAK 16
#define GWC_NPAR_MAX 16

typedef enum {
  GWC_OK = 0,
  GWC_ERR_INVALID_ARG = 1,
  GWC_ERR_SHAPE = 2,
  GWC_ERR_DOMAIN = 3,
  GWC_ERR_NOT_BUILT = 4,
  GWC_ERR_NOMEM = 5,
  GWC_ERR_CUDA = 6,
  GWC_ERR_RANGE = 7
} gwc_status;

#define GWC_MAX_NZ_SELECTION 4096 /* largest los->n_z of the selection term (the all-sky table sits in shared memory) */

typedef enum { GWC_F64 = 0, GWC_F32 = 1 } gwc_prec;
/* bandwidth rule of the KDE numerator: Scott, Eq. D1 (the paper's default) | Silverman, Eq. D2 (:300) |
 * the biweight midvariance of Eq. D3-D4 (:303-309) taken as printed, h = D3 | the same robust scale in Scott's rule,
 * h = 1.06 sqrt(D3) n^(-1/5) (R37).  D3 and the IQR are over the pixel's live redshifts, unweighted. */
typedef enum { GWC_BW_SCOTT = 0, GWC_BW_SILVERMAN = 1, GWC_BW_BIWEIGHT = 2, GWC_BW_BIWEIGHT_SCOTT = 3 } gwc_bw_rule;

/* Mass model (App. A; Table III, :263-274).  GWC_MASS_PLPEAK: truncated power law + one Gaussian peak,
 * conditional power law in m2 (R2, R3).  GWC_MASS_MULTIPEAK: power law + two Gaussian peaks, the primary
 * and the secondary law both multiplied by the low-mass smoothing S(m | mmin, delta_m) and normalised numerically per
 * theta (R33-R36; the formula is not printed in the paper). */
typedef enum { GWC_MASS_PLPEAK = 0, GWC_MASS_MULTIPEAK = 1 } gwc_mass_model;

typedef struct gwc_ctx gwc_ctx;

/* Create a context on CUDA device `device`; `cuda_stream` is a cudaStream_t (NULL = default stream). */
gwc_status gwc_create(gwc_ctx** ctx, int device, void* cuda_stream);
void gwc_destroy(gwc_ctx* ctx);
/* Synchronise the stream and report sticky device errors, then clear them: GWC_ERR_NOT_BUILT (theta changed since
 * the build), GWC_ERR_INVALID_ARG (a broken GWC_OMEGA_SINGLE promise, gwc_set_omega_hint), GWC_ERR_DOMAIN (a theta
 * point outside the model's domain), GWC_ERR_RANGE (see "Range" above), in that order of precedence; GWC_ERR_CUDA. */
gwc_status gwc_check(gwc_ctx* ctx);
const char* gwc_last_error(const gwc_ctx* ctx);
/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
int64_t gwc_launch_count(const gwc_ctx* ctx);

/* Select the mass model of this context (default GWC_MASS_PLPEAK).  From then on every d_theta / h_theta argument has
 * rows of gwc_theta_len(model) doubles.  Tables of an earlier gwc_build_cosmo are dropped (GWC_ERR_NOT_BUILT until the
 * next build).  Additional theta-domain rules under MULTIPEAK: 0 <= delta_m, mmin + delta_m < mmax, sigma_g,low > 0,
 * 0 <= lambda_g,low <= 1.  Supported by gwc_build_cosmo, gwc_event_loglik, gwc_event_loglik_pixcut,
 * gwc_event_loglik_kde, gwc_selection_logxi, gwc_total_loglik, gwc_total_loglik_kde and gwc_total_loglik_host. */
gwc_status gwc_set_mass_model(gwc_ctx* ctx, gwc_mass_model model);
/* Doubles per theta row of a mass model: GWC_NPAR or GWC_NPAR_MULTIPEAK (0 for an unknown model). */
int32_t gwc_theta_len(gwc_mass_model model);

/*
 * A1 + A2.  For each theta: D(z) = int_0^z dz'/E(z') by cumulative Gauss-Legendre
 * quadrature on a uniform z grid (Eq. 1), u(z) = (1+z) D(z) = d_L H0/c, monotone
 * inversion by Newton onto the uniform grid u_m = m*du, du = u(z_max)/(n_nodes-1), node slopes
 * z'(u) = 1/(u/(1+z) + (1+z)/E(z)); and the per-theta population constants.  Tables are kept in the
 * context (storage precision `table_prec`; arithmetic is always FP64) and are used by the calls below.
 * table_prec = GWC_F32 selects 32-bit storage (8 bytes per node instead of 16): z_m as an unsigned 32-bit
 * fixed-point fraction of z_max (absolute step z_max/(2^32-1)), the slope as a binary32 in the same units
 * (R22).
 *   d_theta [n_theta][gwc_theta_len(model)] f64, row-major.   z_max > 0.   n_nodes in [2, 8193] (1025 typical).
 * Under GWC_MASS_MULTIPEAK the same call also builds, per theta, the normalisation N1 of p(m1) and a 513-node
 * cubic-Hermite table of the normaliser of p(m2 | m1) over the smoothing window [mmin, mmin + delta_m] (above the
 * window it is elementary), by 4 x 8-point Gauss-Legendre quadrature per table interval (R36).
 * For batches of 40 theta points or more the call also asks the device whether every row has the same Omega_m and is
 * inside the model's domain (then
 * one z(u) table serves the whole batch and a tile of the fused kernel holds 16 points instead of 10) and reads the
 * 4-byte answer: it SYNCHRONISES the stream in that case; smaller batches stay asynchronous.
 */
gwc_status gwc_build_cosmo(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, double z_max, int32_t n_nodes,
                           gwc_prec table_prec);
/*
 * What the caller knows about Omega_m in its theta batches, so that gwc_build_cosmo need not ask the device (and
 * synchronise) for batches of 40 points and more.  Applies to every later build of this context.
 *   GWC_OMEGA_DETECT (default): as described above, one synchronisation per large batch.
 *   GWC_OMEGA_VARIES: never share a table; no question, no synchronisation.  Always correct (a batch that does have a
 *     single Omega_m merely runs with 10 points per tile instead of 16).
 *   GWC_OMEGA_SINGLE: the caller promises that every batch has one Omega_m and no point outside the model's domain
 *     (a population-only analysis with a fixed cosmology): the table is shared without synchronising.  The promise is
 *     checked on the device all the same: a batch that breaks it raises a sticky flag, gwc_check() returns
 *     GWC_ERR_INVALID_ARG, and the outputs computed from that build must be discarded.
 */
typedef enum { GWC_OMEGA_DETECT = 0, GWC_OMEGA_VARIES = 1, GWC_OMEGA_SINGLE = 2 } gwc_omega_hint;
gwc_status gwc_set_omega_hint(gwc_ctx* ctx, gwc_omega_hint hint);
/* Copy the tables of the last gwc_build_cosmo out (widened to f64): d_z, d_dz [n_theta][n_nodes]
 * (dz = du * z'(u_m)), d_umax [n_theta].  Any pointer may be NULL. */
gwc_status gwc_export_cosmo(gwc_ctx* ctx, double* d_z, double* d_dz, double* d_umax);

typedef struct {                 /* caller-owned device arrays */
  int64_t n_events, n_samples;   /* n_samples = sum_i S_i */
  const int64_t* ev_sample_off;  /* [n_events+1], ascending, [0] = 0, [n_events] = n_samples */
  const double *dL, *m1z, *m2z;  /* [n_samples] */
  const double* log_pe_prior;    /* [n_samples] or NULL => 2 ln d_L  (PE prior ∝ d_L^2, flat in detector masses) */
  const int32_t* sample_row;     /* [n_samples] row of the LOS table (sky pixel) of each sample */
  const int64_t* ev_pix_off;     /* [n_events+1] or NULL (not read by the hot path) */
  const int32_t* ev_pix_rows;    /* [sum_i P_i]  or NULL (not read by the hot path) */
} gwc_events;

typedef struct {
  int64_t n_rows;
  int32_t n_z;                   /* >= 2 node values per row at z_b = b z_max/(n_z-1), both ends included */
  double z_max;
  gwc_prec prec;                 /* storage type of `table` */
  const void* table;             /* [n_rows][n_z] row-major, p(z | pixel) up to a theta-independent constant */
  const double* allsky;          /* [n_z] f64: mean over rows (gwc_los_allsky fills it); read by the selection term */
} gwc_los;

typedef struct {
  int64_t n_found;
  double n_draw;                 /* number of injections drawn, found or not */
  const double *dL, *m1z, *m2z;  /* [n_found] */
  const double* log_pdraw;       /* [n_found] log draw density in (d_L, m1z, m2z) coordinates */
} gwc_injections;

/*
 * A0 (one-time per catalogue).  Stable sort of samples by (event, row); ties keep input order, so
 * the answer is unique and is compared bit-exactly with the oracle.
 *   in : d_event_id, d_row [n_samples] i32, any order; event ids in [0, n_events), rows >= 0.
 *   out: d_perm [n_samples] (sorted position -> input index), d_ev_sample_off [n_events+1],
 *        d_ev_pix_off [n_events+1], d_ev_pix_rows [<= n_samples] (distinct rows per event, ascending),
 *        d_pix_sample_off [<= n_samples+1] (start of each (event,row) run, then n_samples),
 *        *h_n_pixrefs (host) = number of distinct (event,row) pairs.  Synchronises the stream.
 * An event id outside [0, n_events) or a negative row -> GWC_ERR_DOMAIN (reported by this call itself; the sticky
 * flags that gwc_check reports are neither read nor cleared).
 */
gwc_status gwc_pack_events(gwc_ctx* ctx, int64_t n_samples, int64_t n_events, const int32_t* d_event_id,
                           const int32_t* d_row, int64_t* d_perm, int64_t* d_ev_sample_off, int64_t* d_ev_pix_off,
                           int32_t* d_ev_pix_rows, int64_t* d_pix_sample_off, int64_t* h_n_pixrefs);

/*
 * The per-pixel sample cap, "the option to randomly downsample the GW posterior samples in a given pixel"
 * (fiducial cap 2500; R31), applied to the output of gwc_pack_events (one-time,
 * integer work, compared bit for bit with the oracle).  A pixel ((event, row) run) with more than `cap` samples keeps
 * the `cap` samples with the smallest (hash32(seed, original sample index), packed position), hash32 = upper half of
 * splitmix64's output function of seed + (index + 1) * 0x9E3779B97F4A7C15; smaller pixels keep everything; kept
 * samples keep their packed order.  The choice depends on the original indices only, not on the packing.
 *   in : d_perm [n_samples] (gwc_pack_events' permutation), n_pixrefs
 *   in/out: d_ev_sample_off [n_events+1], d_pix_sample_off [n_pixrefs+1]: rewritten for the kept samples
 *   out: d_perm_out [n_samples] (first *h_n_kept entries valid; must not alias d_perm), h_n_kept (host)
 * ev_pix_off / ev_pix_rows are unchanged (every pixel keeps at least one sample).  cap < 1 -> GWC_ERR_INVALID_ARG.
 * Synchronises the stream.
 */
gwc_status gwc_cap_pixels(gwc_ctx* ctx, int64_t n_samples, int64_t n_events, int64_t n_pixrefs,
                          const int64_t* d_perm, int64_t* d_ev_sample_off, int64_t* d_pix_sample_off, int64_t cap,
                          uint64_t seed, int64_t* d_perm_out, int64_t* h_n_kept);

/* All-sky prior of the denominator: arithmetic mean over all rows, in f64, fixed order. */
gwc_status gwc_los_allsky(gwc_ctx* ctx, const gwc_los* los, double* d_allsky /* [n_z] */);

/*
 * gwc_los_allsky for callers that must not allocate device memory.  Who they are: a program that has given all of the
 * GPU's memory to its own pool or arena (a cudaMalloc made behind its back fails, or eats memory the pool counts on);
 * a sampling or serving loop with other streams busy (cudaMalloc / cudaFree take a device-wide lock and can wait for
 * the device, stalling every stream); and, because of either, code that may not even call gwc_create (which
 * allocates).  So this call takes NO context, and neither it nor anything under it calls cudaMalloc, cudaFree or an
 * allocating library routine: the partial sums that gwc_los_allsky keeps in context scratch live in a fixed array
 * inside the library image (4 MiB of device memory, held by every GPU that loads libgwc.so until the process exits).
 *   in : los->table [n_rows][n_z] (device, f64 or f32 per los->prec), los->n_rows, los->n_z, los->z_max > 0;
 *        los->allsky is not read.   out: d_allsky [n_z] f64 (device, caller-owned).   cuda_stream: a cudaStream_t of
 *        the calling thread's CURRENT device (NULL = default stream); the table and d_allsky must be on that device.
 * Result: bit-identical to gwc_los_allsky (same kernels, same fixed summation order).  Asynchronous on cuda_stream.
 * Limit: ceil(n_rows / GWC_ALLSKY_STATIC_ROWS_PER_PART) * n_z <= GWC_ALLSKY_STATIC_MAX_DOUBLES (the O5-scale table,
 *   200000 rows x 1000 nodes, needs 391000 and fits); a larger table is refused with GWC_ERR_SHAPE before anything is
 *   enqueued, d_allsky untouched.  Other argument errors as gwc_los_allsky.  The text of the last non-OK status of
 *   the calling thread comes from gwc_los_allsky_static_error() (there is no context to hold it).
 * Set-up: the FIRST call on each device asks the runtime for the array's address on that device (one
 *   cudaGetSymbolAddress, which may also make the runtime load the library's device code).  Make that first call
 *   during start-up, before any stream capture and before the phase in which allocation is forbidden.
 * Sharing: all calls on one GPU use the same array, from every thread and stream.  Nothing in it needs to be zero at
 *   entry (each call overwrites exactly the part it then reads), so calls one after the other on one stream, or
 *   ordered by events, are safe; two calls that can RUN AT THE SAME TIME on one GPU (different streams, no ordering
 *   between them) race on it and give wrong sums.  Serialise them.
 */
#define GWC_ALLSKY_STATIC_ROWS_PER_PART 512
#define GWC_ALLSKY_STATIC_MAX_DOUBLES (1 << 19)
gwc_status gwc_los_allsky_static(const gwc_los* los, double* d_allsky /* [n_z] */, void* cuda_stream);
const char* gwc_los_allsky_static_error(void);

/*
 * A3 + A4.  log L_i(theta) = log( (1/S_i) sum_k w_ik ) for every (theta, event); optional
 * N_eff,i (Eq. 8) and the number of live samples.  Needs gwc_build_cosmo(d_theta, n_theta) first
 * (same pointer and count) else GWC_ERR_NOT_BUILT; needs los->z_max <= the z_max of that build.
 *   d_logL [n_theta][n_events] f64;  d_neff same shape or NULL;  d_nlive same shape i64 or NULL.
 */
gwc_status gwc_event_loglik(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                            const gwc_los* los, double* d_logL, double* d_neff, int64_t* d_nlive);

/*
 * A3 + A4 with the per-pixel effective-sample cut of Eq. 8 (fiducial threshold 2,
 * PAPER.md:194; R25).  A pixel of an event is a maximal run of consecutive samples with the same
 * sample_row (gwc_pack_events orders the samples so that every (event, row) is one run).  With W_j = sum_k w_k
 * and Q_j = sum_k w_k^2 over the samples of pixel j, the pixel contributes iff it has a live sample and
 * W_j^2 >= neff_min * Q_j (N_eff,j >= neff_min, decided in FP64 in this form); then
 *   log L_i = log( (1/S_i) sum over passing pixels of W_j ),   S_i = all samples of the event,
 * N_eff,i and the live count over the samples of the passing pixels, and the number of passing pixels.
 * neff_min = 0 gives gwc_event_loglik's results.  Same preconditions and errors as gwc_event_loglik;
 * neff_min < 0 or NaN -> GWC_ERR_INVALID_ARG.
 *   d_logL [n_theta][n_events] f64;  d_neff f64, d_nlive i64, d_npass i64: same shape or NULL.
 * The kernel works on a pixel-aligned copy of the samples kept in the context (every pixel on an even slot, odd
 * pixels padded by one dead slot: at most twice the samples, typically a few per cent more); building it
 * SYNCHRONISES the stream once (its length), unless gwc_cache_catalogue is on and the copy is still valid.
 */
gwc_status gwc_event_loglik_pixcut(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                   const gwc_los* los, double neff_min, double* d_logL, double* d_neff,
                                   int64_t* d_nlive, int64_t* d_npass);

/*
 * The event term with the paper's own numerator: a Gaussian kernel density estimate in redshift per sky pixel
 * (Eq. 5-7; Scott bandwidth Eq. D1; n_grid = 256 fiducial, PAPER.md:213;
 * DESIGN.md R26-R30).  Pixels as in gwc_event_loglik_pixcut.  For pixel j:
 *   v_k = p(m1, m2 | theta) / (J pi_PE)  (Eq. 7 without the redshift prior),  n_j = its live samples,
 *   h_j = 1.06 sigma_j n_j^(-1/5) with sigma_j the v-weighted standard deviation of the z_k (bw_rule = GWC_BW_SCOTT),
 *         or 0.9 min(sigma_j, IQR_j / 1.34) n_j^(-1/5) with the interquartile range of the live z_k, plain quantiles
 *         by linear interpolation (GWC_BW_SILVERMAN; R32), or from the biweight midvariance D3 of the live z_k
 *         (Eq. D3-D4): h_j = D3 as printed (GWC_BW_BIWEIGHT) or 1.06 sqrt(D3) n_j^(-1/5) (GWC_BW_BIWEIGHT_SCOTT; R37),
 *   I_j = trapezoid over the n_grid-node uniform grid on [0, los->z_max] of
 *         [sum_k v_k N(z; z_k, h_j)] p_los(z | row_j) psi(z) / (1+z),
 *   log L_i = log( (1/S_i) sum_j I_j )  over the pixels with n_j >= 2, sigma_j > 0 and N_eff,j >= neff_min.
 * All arithmetic FP64.  Needs gwc_build_cosmo(d_theta, n_theta) first.  n_grid in [2, 256] else GWC_ERR_SHAPE;
 * neff_min < 0 or NaN -> GWC_ERR_INVALID_ARG.
 *   d_logL [n_theta][n_events] f64;  d_npass, d_nused same shape i64 or NULL (pixels that contributed, and their
 *   live samples: n_grid * d_nused Gaussian evaluations were needed).
 * A Gaussian kernel value below e^-700 counts as zero (R38).  Work is split into chunks of whole pixels of about 1024
 * samples (a table built on the device per call).  Synchronises the stream once (the number of chunks and the
 * longest chunk size the scratch buffers).
 */
gwc_status gwc_event_loglik_kde(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                const gwc_los* los, int32_t n_grid, double neff_min, int32_t bw_rule, double* d_logL,
                                int64_t* d_npass, int64_t* d_nused);

/*
 * A5.  log xi(theta) = log( (1/n_draw) sum_j w_j ) over found injections with the all-sky prior
 * los->allsky and log_pdraw in place of the PE prior; optional N_eff of the injection sum.
 *   d_logxi [n_theta];  d_neff_inj [n_theta] or NULL.
 * los->n_z <= GWC_MAX_NZ_SELECTION (4096) else GWC_ERR_SHAPE (here and, before any work, in gwc_total_loglik*).
 * Calls of 2e8 (theta x injection) terms and up work on a copy of the injections in order of d_L kept in the context
 * (whole warps then leave a theta's table together; the sum does not depend on the order beyond rounding).
 */
gwc_status gwc_selection_logxi(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_injections* inj,
                               const gwc_los* los, double* d_logxi, double* d_neff_inj);

/* A6 alone: d_total[t] = sum_i d_logL[t][i] - n_events * d_logxi[t]  (fixed order; -inf stays -inf, never NaN). */
gwc_status gwc_combine_total(gwc_ctx* ctx, const double* d_logL, const double* d_logxi, int64_t n_theta,
                             int64_t n_events, double* d_total);

/*
 * A6 for a catalogue split over R ranks (SURVEY.md 8e-2; the sampler's one-theta-per-call pattern, PAPER.md:129, :166,
 * leaves nothing to split but the events and the injections).  Rank r owns a block of events and a block of the found
 * injections and computes, with the ordinary calls on its block,
 *   S_r[t]  = sum over ITS events of log L_i(theta_t)       (gwc_combine_total with a zero log xi; 0 without events),
 *   x_r[t]  = log xi_r(theta_t), N_r[t] = N_eff,r            (gwc_selection_logxi with the GLOBAL n_draw),
 * the ranks exchange these (an all-gather of 3 x n_theta doubles per rank), and every rank combines them here in
 * rank order, so that all ranks hold the same bits (Eq. 3-4):
 *   xi = sum_r xi_r,   N_eff,inj = (sum_r xi_r)^2 / sum_r (xi_r^2 / N_r),   log L = sum_r S_r - n_events_total log xi.
 *   d_sum_logL_parts, d_logxi_parts, d_neff_inj_parts: [n_parts][n_theta] f64 (the last may be NULL when d_neff_inj is);
 *   d_total, d_logxi, d_neff_inj: [n_theta] f64, each may be NULL.   n_parts in [1, 65536].
 * A NaN in any piece of a theta makes its outputs NaN; -inf stays -inf.  The _host form takes HOST pointers, needs
 * no context and no GPU (the same function compiled for the host): for ranks that gathered through host memory.
 */
gwc_status gwc_combine_sharded(gwc_ctx* ctx, int32_t n_parts, int64_t n_theta, int64_t n_events_total,
                               const double* d_sum_logL_parts, const double* d_logxi_parts,
                               const double* d_neff_inj_parts, double* d_total, double* d_logxi, double* d_neff_inj);
gwc_status gwc_combine_sharded_host(int32_t n_parts, int64_t n_theta, int64_t n_events_total,
                                    const double* h_sum_logL_parts, const double* h_logxi_parts,
                                    const double* h_neff_inj_parts, double* h_total, double* h_logxi,
                                    double* h_neff_inj);

/*
 * The whole hot path A1..A6 for one theta batch: build_cosmo(z_max = los->z_max, n_nodes, table_prec),
 * event_loglik, selection_logxi, combine.   d_logL_total [n_theta] f64.
 */
gwc_status gwc_total_loglik(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                            const gwc_injections* inj, const gwc_los* los, int32_t n_nodes, gwc_prec table_prec,
                            double* d_logL_total);

/*
 * gwc_total_loglik with the per-pixel effective-sample cut of Eq. 8 on the event term: the direct
 * Monte-Carlo sum over the samples of the pixels that pass N_eff,j >= neff_min (gwc_event_loglik_pixcut), the same
 * selection term, the same total.  neff_min = 0 gives gwc_total_loglik's result.  Same arguments and errors as
 * gwc_total_loglik; synchronises the stream once (the padded copy of gwc_event_loglik_pixcut), twice for batches of
 * 40 theta points or more (gwc_build_cosmo).
 */
gwc_status gwc_total_loglik_pixcut(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                   const gwc_injections* inj, const gwc_los* los, int32_t n_nodes,
                                   gwc_prec table_prec, double neff_min, double* d_logL_total);

/*
 * The paper's likelihood in one call: Eq. 5 with the KDE numerator (gwc_event_loglik_kde: n_grid, neff_min), the
 * per-pixel cut of Eq. 8 and the selection term of Eq. 4:  build_cosmo(z_max = los->z_max, n_nodes, table_prec),
 * the KDE event term, gwc_selection_logxi, gwc_combine_total.  Same arguments, errors and NaN / -inf rules as
 * gwc_total_loglik; synchronises the stream once (gwc_event_loglik_kde).
 */
gwc_status gwc_total_loglik_kde(gwc_ctx* ctx, const double* d_theta, int64_t n_theta, const gwc_events* ev,
                                const gwc_injections* inj, const gwc_los* los, int32_t n_nodes, gwc_prec table_prec,
                                int32_t n_grid, double neff_min, int32_t bw_rule, double* d_logL_total /* [n_theta] */);

/*
 * Same as gwc_total_loglik but every pointer (inside the structs too) is a HOST pointer: the call
 * uploads theta, the catalogue, the injections and the LOS table (computing the all-sky mean on the
 * device when los->allsky is NULL), runs A1..A6 and downloads h_logL_total, then synchronises.
 * Pinned host memory makes the copies asynchronous and faster; pageable memory works.
 * *h2d_bytes / *d2h_bytes (may be NULL) receive the bytes copied.
 */
gwc_status gwc_total_loglik_host(gwc_ctx* ctx, const double* h_theta, int64_t n_theta, const gwc_events* h_ev,
                                 const gwc_injections* h_inj, const gwc_los* h_los, int32_t n_nodes,
                                 gwc_prec table_prec, double* h_logL_total, int64_t* h2d_bytes, int64_t* d2h_bytes);

/*
 * Small-batch (latency) mode: the sampler's pattern is one theta point per call on a catalogue that never changes
 * (PAPER.md:129, :166).  With caching on, the theta-independent preparation of the events and of the injections
 * (per-sample logarithms and the per-segment reference of the sums) is kept in the context and reused by every later
 * call that presents the same device pointers and sizes.  THE CALLER PROMISES that the contents of those arrays have
 * not changed in between; turning the cache off (or on again) forgets everything.  Off by default.
 */
gwc_status gwc_cache_catalogue(gwc_ctx* ctx, int on);

/*
 * Measurement helpers (not on the hot path).
 * gwc_set_timing: when on, the fused re-weighting kernel (A3/A5) is bracketed by CUDA events on the
 * context's stream; gwc_get_timing returns, for launches since the last call, the number of such
 * launches and their summed duration in ms for events and injections (synchronises).
 * gwc_probe_fp64: runs a dependent-free DFMA kernel on all SMs and returns its duration and the
 * number of FP64 instructions (thread-level) it executed: the measured FP64 roofline denominator.
 */
gwc_status gwc_set_timing(gwc_ctx* ctx, int on);
gwc_status gwc_get_timing(gwc_ctx* ctx, int64_t* n_ev_launches, double* ms_ev, int64_t* n_inj_launches,
                          double* ms_inj);
gwc_status gwc_probe_fp64(gwc_ctx* ctx, int64_t iters, double* ms, double* n_fp64_instr);
/* Accuracy self-test of the kernel's own FP64 elementary functions: d_out[i] = f(d_in[i]) with
 * which = 0: exp (clamped below -700), 1: ln, 2: 1/x, 3: x^-1/2, 4: exp (unclamped).  n device doubles. */
gwc_status gwc_math_selftest(gwc_ctx* ctx, int which, int64_t n, const double* d_in, double* d_out);

#ifdef __cplusplus
}
#endif
#endif /* GWC_H_ */
