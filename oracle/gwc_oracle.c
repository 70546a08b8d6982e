/*
 * gwc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, scalar CPU oracle for the dark-siren hierarchical likelihood
 * (arxiv/paper_2605_23538, "Scalable dark siren cosmology with gwcosmo").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call it.  It shares no code, header, table or constant
 * generator with the CUDA path under paper_2605_23538_b200/csrc/.
 *
 * What it computes, and the passage each piece follows (PAPER.md line numbers):
 *   - d_L(z) for flat LambdaCDM                         Eq. 1
 *   - sample weights w = p(z,theta'|Lambda)/pi_PE        Eq. 7
 *   - the pixelated event likelihood, with the line-of-sight prior
 *     p(z|Omega_j) read at each sample's redshift (the h->0 limit of the
 *     KDE of Eq. 6; reading R1)                 Eq. 5-6
 *   - the selection term from found injections          Eq. 4
 *   - N_eff = (sum w)^2 / sum w^2                        Eq. 8
 *   - log L = sum_i log L_i - N_det log xi              Eq. 3
 *   - Madau-Dickinson rate, SNR>12 injections           App. A
 * The power-law+peak mass law, the Jacobian and the table scheme are not
 * written in the paper; they follow SURVEY.md section 8(c) / DESIGN.md readings.
 *
 * Pins: tests/test_oracle_*.py (closed forms, scipy quadrature, brute force,
 * invariances, the 1-event Monte-Carlo toy).  No value printed by the paper
 * exists for a likelihood, so beyond those pins parity is "unpinned" only in
 * the sense stated in DESIGN.md section 5.
 *
 * Arithmetic: IEEE binary64, libm, no FMA contraction (-ffp-contract=off),
 * sums of exponentials in long double.  OpenMP is used only as a plain
 * "parallel for" over hyper-parameter points; each point is computed serially.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* theta row, power law + peak (model 0): H0, Om, alpha, beta, mmin, mmax, mu, sigma, lambda, gamma, kappa, zp.
 * MULTIPEAK (model 1; App. A, Table III :263-274; R33-R36) appends delta_m, mu_g,low,
 * sigma_g,low, lambda_g,low; there mu, sigma are the HIGH peak and lambda is lambda_g, the Gaussian fraction. */
enum { P_H0 = 0, P_OM, P_ALPHA, P_BETA, P_MMIN, P_MMAX, P_MU, P_SIGMA, P_LAMBDA, P_GAMMA, P_KAPPA, P_ZP,
       P_DM, P_MULOW, P_SIGLOW, P_LAMLOW };
static int g_model = 0;   /* set once before a run by the test that wants MULTIPEAK; never changed during one */
void orc_set_mass_model(int model) { g_model = model == 1 ? 1 : 0; }
int orc_npar(void) { return g_model == 1 ? 16 : 12; }
#define ORC_NPAR (orc_npar())

static const double C_KMS = 299792.458; /* km/s, exact */

/* ------------------------------------------------------------------ */
/* Gauss-Legendre nodes on [-1,1], computed once by Newton on P_n.      */
/* ------------------------------------------------------------------ */
#define GL_N 32
static double gl_x[GL_N], gl_w[GL_N];
static int gl_ready = 0;

static void gl_init(void) {
  if (gl_ready) return;
  const int n = GL_N;
  for (int i = 0; i < (n + 1) / 2; ++i) {
    double x = cos(M_PI * (i + 0.75) / (n + 0.5));
    double pp = 0.0;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 0; j < n; ++j) {
        double p3 = p2;
        p2 = p1;
        p1 = ((2.0 * j + 1.0) * x * p2 - j * p3) / (j + 1.0);
      }
      pp = n * (x * p1 - p2) / (x * x - 1.0);
      double dx = p1 / pp;
      x -= dx;
      if (fabs(dx) < 1e-16) break;
    }
    gl_x[i] = -x;
    gl_x[n - 1 - i] = x;
    gl_w[i] = 2.0 / ((1.0 - x * x) * pp * pp);
    gl_w[n - 1 - i] = gl_w[i];
  }
  gl_ready = 1;
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ------------------------------------------------------------------ */
/* Cosmology: Eq. 1, flat LambdaCDM.                   */
/* ------------------------------------------------------------------ */
double orc_E(double z, double Om) {
  double x = 1.0 + z;
  return sqrt(Om * x * x * x + (1.0 - Om));
}

/* D(z) = int_0^z dz'/E(z'), 32-point Gauss-Legendre on panels of width <= 0.5 */
double orc_D(double z, double Om) {
  gl_init();
  if (z <= 0.0) return 0.0;
  int np = (int)ceil(z / 0.5);
  double h = z / np, total = 0.0;
  for (int p = 0; p < np; ++p) {
    double a = p * h, s = 0.0;
    for (int i = 0; i < GL_N; ++i) {
      double zz = a + 0.5 * h * (gl_x[i] + 1.0);
      s += gl_w[i] / orc_E(zz, Om);
    }
    total += 0.5 * h * s;
  }
  return total;
}

/* d_L in Mpc (H0 in km/s/Mpc): Eq. 1 */
double orc_dL(double z, double H0, double Om) { return (1.0 + z) * (C_KMS / H0) * orc_D(z, Om); }

/* dimensionless u(z) = d_L H0 / c = (1+z) D(z) */
double orc_u_of_z(double z, double Om) { return (1.0 + z) * orc_D(z, Om); }

/* du/dz = D + (1+z)/E  (= u/(1+z) + (1+z)/E) */
static double dudz(double z, double u, double Om) { return u / (1.0 + z) + (1.0 + z) / orc_E(z, Om); }

/* EXACT inverse: z with (1+z) D(z) = u.  Newton from z0 = u, safeguarded by a bracket. */
double orc_z_of_u(double u, double Om) {
  if (!(u > 0.0)) return 0.0;
  double lo = 0.0, hi = (u > 1.0 ? u : 1.0);
  while (orc_u_of_z(hi, Om) < u) hi *= 2.0;
  double z = (u < hi ? u : 0.5 * hi);
  for (int it = 0; it < 200; ++it) {
    double uz = orc_u_of_z(z, Om);
    double f = uz - u;
    if (f > 0.0) hi = z; else lo = z;
    double dz = f / dudz(z, uz, Om);
    double zn = z - dz;
    if (!(zn > lo && zn < hi)) zn = 0.5 * (lo + hi);
    if (fabs(zn - z) < 1e-15 * (1.0 + fabs(z))) { z = zn; break; }
    z = zn;
  }
  return z;
}

double orc_z_of_dL(double dL, double H0, double Om) { return orc_z_of_u(dL * H0 / C_KMS, Om); }

/*
 * TABLE mode (SURVEY 8c step 2 / DESIGN.md reading R9): uniform nodes u_m = m*du,
 * du = u(z_max)/(M-1); z_m exact inverse at u_m; dz_m = du * z'(u_m),
 * z' = 1/(u/(1+z) + (1+z)/E(z)).
 */
void orc_build_table(double Om, double z_max, int M, double* ztab, double* dztab, double* umax) {
  double um = orc_u_of_z(z_max, Om);
  double du = um / (M - 1);
  *umax = um;
  for (int m = 0; m < M; ++m) {
    double u = m * du;
    double z = (m == M - 1) ? z_max : orc_z_of_u(u, Om);
    ztab[m] = z;
    dztab[m] = du / dudz(z, u, Om);
  }
}

/* cubic Hermite lookup; returns 0 and sets *z, or returns 1 if u >= umax (dead) */
int orc_z_table(double u, const double* ztab, const double* dztab, int M, double umax, double* z) {
  if (!(u < umax)) return 1;
  double du = umax / (M - 1);
  double t = u / du;
  int m = (int)floor(t);
  if (m > M - 2) m = M - 2;
  if (m < 0) m = 0;
  double f = t - m;
  double g = 1.0 - f;
  *z = (1.0 + 2.0 * f) * g * g * ztab[m] + f * g * g * dztab[m] + f * f * (3.0 - 2.0 * f) * ztab[m + 1] +
       f * f * (f - 1.0) * dztab[m + 1];
  return 0;
}

/* ------------------------------------------------------------------ */
/* Population (readings R2-R4).                               */
/* ------------------------------------------------------------------ */
int orc_theta_valid(const double* th) {
  for (int i = 0; i < ORC_NPAR; ++i)
    if (!isfinite(th[i])) return 0;
  if (!(th[P_H0] > 0.0)) return 0;
  if (!(th[P_OM] > 0.0 && th[P_OM] <= 1.0)) return 0;
  if (!(th[P_SIGMA] > 0.0)) return 0;
  if (!(th[P_MMIN] > 0.0 && th[P_MMIN] < th[P_MMAX])) return 0;
  if (!(th[P_LAMBDA] >= 0.0 && th[P_LAMBDA] <= 1.0)) return 0;
  if (!(th[P_ZP] > -1.0)) return 0;
  if (g_model == 1) {
    if (!(th[P_DM] >= 0.0 && th[P_MMIN] + th[P_DM] < th[P_MMAX])) return 0;
    if (!(th[P_SIGLOW] > 0.0)) return 0;
    if (!(th[P_LAMLOW] >= 0.0 && th[P_LAMLOW] <= 1.0)) return 0;
  }
  return 1;
}

double orc_norm_pl(const double* th) {
  double a = th[P_ALPHA], lo = th[P_MMIN], hi = th[P_MMAX];
  if (a == 1.0) return 1.0 / log(hi / lo);
  return (1.0 - a) / (pow(hi, 1.0 - a) - pow(lo, 1.0 - a));
}

double orc_norm_g(const double* th) {
  double mu = th[P_MU], s = th[P_SIGMA];
  double c = 0.5 * (erf((th[P_MMAX] - mu) / (s * M_SQRT2)) - erf((th[P_MMIN] - mu) / (s * M_SQRT2)));
  return 1.0 / c;
}

/* per-theta constants of the population laws, computed once per theta */
typedef struct {
  double n_pl, n_g, psi0;
  double n_gl;   /* MULTIPEAK: normalisation of the low Gaussian on [mmin, mmax] */
  double N1;     /* MULTIPEAK: int_mmin^mmax mix(m) S(m) dm */
  double Cwin;   /* MULTIPEAK: int over the smoothing window [mmin, mmin + delta_m] of m^beta S(m) dm */
} orc_pop;

/* ---- MULTIPEAK with low-mass smoothing (readings R33-R36; the formula is not in the paper) ----------------
 *   S(m) = 0 (m <= mmin), 1 (m >= mmin + dm), else 1 / (1 + exp(dm/m' + dm/(m' - dm))), m' = m - mmin;
 *          a smoothing factor below e^-250 counts as 0 (R35)
 *   mix(m) = (1-lam) P(m) + lam lam_low G(m; mu_low, s_low) + lam (1-lam_low) G(m; mu_high, s_high),
 *            P = power law m^-alpha, G = Gaussian, each truncated to and normalised on [mmin, mmax]
 *   p(m1) = mix(m1) S(m1) / N1,   N1 = int mix S
 *   p(m2 | m1) = m2^beta S(m2) / C(m1),   C(m1) = int_mmin^m1 m^beta S(m) dm                                */
double orc_mp_smooth(double m, double mmin, double dm) {
  double mp = m - mmin;
  if (!(mp >= 0.0)) return 0.0;
  if (mp >= dm) return 1.0;
  if (mp == 0.0) return 0.0;
  double e = dm / mp + dm / (mp - dm);
  if (e > 250.0) return 0.0;
  return 1.0 / (1.0 + exp(e));
}

static double gl_panels(double (*f)(double, const void*), const void* ctx, double a, double b, int np) {
  gl_init();
  double h = (b - a) / np, total = 0.0;
  for (int p = 0; p < np; ++p) {
    double lo = a + p * h, s = 0.0;
    for (int i = 0; i < GL_N; ++i) s += gl_w[i] * f(lo + 0.5 * h * (gl_x[i] + 1.0), ctx);
    total += 0.5 * h * s;
  }
  return total;
}

typedef struct { const double* th; double n_pl, n_gl, n_gh; } mp_ctx;

static double gauss_norm(double mu, double s, double lo, double hi) {
  return 1.0 / (0.5 * (erf((hi - mu) / (s * M_SQRT2)) - erf((lo - mu) / (s * M_SQRT2))));
}

/* the mixture before smoothing */
static double mp_mix(double m, const void* vc) {
  const mp_ctx* c = (const mp_ctx*)vc;
  const double* th = c->th;
  double lam = th[P_LAMBDA], ll = th[P_LAMLOW];
  double v = (1.0 - lam) * c->n_pl * pow(m, -th[P_ALPHA]);
  if (lam > 0.0) {
    double xl = (m - th[P_MULOW]) / th[P_SIGLOW], xh = (m - th[P_MU]) / th[P_SIGMA];
    if (ll > 0.0) v += lam * ll * c->n_gl * exp(-0.5 * xl * xl) / (th[P_SIGLOW] * sqrt(2.0 * M_PI));
    if (ll < 1.0) v += lam * (1.0 - ll) * c->n_gh * exp(-0.5 * xh * xh) / (th[P_SIGMA] * sqrt(2.0 * M_PI));
  }
  return v;
}
static double mp_mix_s(double m, const void* vc) {
  const mp_ctx* c = (const mp_ctx*)vc;
  return mp_mix(m, vc) * orc_mp_smooth(m, c->th[P_MMIN], c->th[P_DM]);
}
static double mp_pow_s(double m, const void* vc) {
  const double* th = (const double*)vc;
  return pow(m, th[P_BETA]) * orc_mp_smooth(m, th[P_MMIN], th[P_DM]);
}
#define MP_WIN_PANELS 16

/* C(m1) = int_mmin^m1 m^beta S(m) dm: quadrature inside the smoothing window, elementary above it */
static double mp_C(double m1, const double* th, const orc_pop* P) {
  double lo = th[P_MMIN], top = th[P_MMIN] + th[P_DM], b = th[P_BETA];
  if (!(m1 > lo)) return 0.0;
  if (m1 < top) return gl_panels(mp_pow_s, th, lo, m1, MP_WIN_PANELS);
  double above = (b == -1.0) ? log(m1 / top) : (pow(m1, b + 1.0) - pow(top, b + 1.0)) / (b + 1.0);
  return P->Cwin + above;
}

static void pop_init(const double* th, orc_pop* P) {
  P->n_pl = orc_norm_pl(th);
  P->n_g = orc_norm_g(th);
  P->psi0 = 1.0 + pow(1.0 + th[P_ZP], -(th[P_GAMMA] + th[P_KAPPA]));
  P->n_gl = P->N1 = P->Cwin = 0.0;
  if (g_model == 1) {
    double lo = th[P_MMIN], hi = th[P_MMAX], top = lo + th[P_DM];
    P->n_gl = gauss_norm(th[P_MULOW], th[P_SIGLOW], lo, hi);
    mp_ctx c = {th, P->n_pl, P->n_gl, P->n_g};
    /* N1: the window in MP_WIN_PANELS panels, the rest in panels no wider than the narrower peak */
    double w = th[P_SIGLOW] < th[P_SIGMA] ? th[P_SIGLOW] : th[P_SIGMA];
    double np = ceil((hi - top) / w);
    if (np > 20000.0) np = 20000.0;
    if (np < 1.0) np = 1.0;
    P->N1 = (th[P_DM] > 0.0 ? gl_panels(mp_mix_s, &c, lo, top, MP_WIN_PANELS) : 0.0) +
            gl_panels(mp_mix_s, &c, top, hi, (int)np);
    P->Cwin = th[P_DM] > 0.0 ? gl_panels(mp_pow_s, th, lo, top, MP_WIN_PANELS) : 0.0;
  }
}

/* p(m1|theta): truncated power law + truncated Gaussian peak on (mmin, mmax] */
static double p1_c(double m1, const double* th, const orc_pop* P) {
  if (!(m1 > th[P_MMIN] && m1 <= th[P_MMAX])) return 0.0;
  if (g_model == 1) {
    mp_ctx c = {th, P->n_pl, P->n_gl, P->n_g};
    return mp_mix(m1, &c) * orc_mp_smooth(m1, th[P_MMIN], th[P_DM]) / P->N1;
  }
  double lam = th[P_LAMBDA], mu = th[P_MU], s = th[P_SIGMA];
  double pl = (1.0 - lam) * P->n_pl * pow(m1, -th[P_ALPHA]);
  double g = 0.0;
  if (lam > 0.0) {
    double x = (m1 - mu) / s;
    g = lam * P->n_g * exp(-0.5 * x * x) / (s * sqrt(2.0 * M_PI));
  }
  return pl + g;
}

double orc_p1(double m1, const double* th) {
  orc_pop P;
  pop_init(th, &P);
  return p1_c(m1, th, &P);
}

/* p(m2|m1,theta) = (beta+1) m2^beta / (m1^(beta+1) - mmin^(beta+1)) on [mmin, m1] */
static double p2_c(double m2, double m1, const double* th, const orc_pop* P) {
  double b = th[P_BETA], lo = th[P_MMIN];
  if (!(m2 >= lo && m2 <= m1 && m1 > lo)) return 0.0;
  if (g_model == 1) {
    double s = orc_mp_smooth(m2, lo, th[P_DM]);
    if (!(s > 0.0)) return 0.0;
    return pow(m2, b) * s / mp_C(m1, th, P);
  }
  if (b == -1.0) return 1.0 / (m2 * log(m1 / lo));
  return (b + 1.0) * pow(m2, b) / (pow(m1, b + 1.0) - pow(lo, b + 1.0));
}

double orc_p2(double m2, double m1, const double* th) {
  orc_pop P;
  pop_init(th, &P);
  return p2_c(m2, m1, th, &P);
}

/* exposed for the pins: C(m1) and N1 of the MULTIPEAK model */
double orc_mp_C(double m1, const double* th) {
  orc_pop P;
  pop_init(th, &P);
  return mp_C(m1, th, &P);
}
double orc_mp_N1(const double* th) {
  orc_pop P;
  pop_init(th, &P);
  return P.N1;
}

/* Madau-Dickinson psi(z), psi(0) = 1 (App. A; Table III :271-273) */
static double psi_c(double z, const double* th, const orc_pop* P) {
  double g = th[P_GAMMA], k = th[P_KAPPA], zp = th[P_ZP];
  return P->psi0 * pow(1.0 + z, g) / (1.0 + pow((1.0 + z) / (1.0 + zp), g + k));
}

double orc_psi(double z, const double* th) {
  orc_pop P;
  pop_init(th, &P);
  return psi_c(z, th, &P);
}

/* ------------------------------------------------------------------ */
/* Line-of-sight table access (node-valued, uniform nodes on [0,z_max]) */
/* ------------------------------------------------------------------ */
typedef struct {
  int64_t n_rows;
  int32_t n_z;
  double z_max;
  int32_t prec;       /* 0 = f64, 1 = f32 */
  const void* table;  /* [n_rows][n_z] */
} orc_los;

static double los_node(const orc_los* L, int64_t r, int32_t b) {
  if (L->prec == 0) return ((const double*)L->table)[r * (int64_t)L->n_z + b];
  return (double)((const float*)L->table)[r * (int64_t)L->n_z + b];
}

/* linear interpolation at z in row r; caller guarantees 0 <= z < z_max */
double orc_los_lerp(const orc_los* L, int64_t r, double z) {
  double dz = L->z_max / (L->n_z - 1);
  double t = z / dz;
  int32_t b = (int32_t)floor(t);
  if (b > L->n_z - 2) b = L->n_z - 2;
  if (b < 0) b = 0;
  double f = t - b;
  double t0 = los_node(L, r, b), t1 = los_node(L, r, b + 1);
  return t0 + f * (t1 - t0);
}

/* all-sky prior: arithmetic mean over rows in fixed row order, in f64 (reading R13) */
void orc_los_allsky(const orc_los* L, double* allsky) {
  for (int32_t b = 0; b < L->n_z; ++b) {
    long double s = 0.0L;
    for (int64_t r = 0; r < L->n_rows; ++r) s += (long double)los_node(L, r, b);
    allsky[b] = (double)(s / (long double)L->n_rows);
  }
}

/* ------------------------------------------------------------------ */
/* One sample's log weight: Eq. 7 with SURVEY 8c step 3.  */
/* mode 0 = TABLE cosmology, 1 = EXACT.  Returns -INFINITY when dead.   */
/* ------------------------------------------------------------------ */
typedef struct {
  int M;
  double umax;          /* of the cosmology table (z_max_cosmo) */
  const double* ztab;   /* [M] */
  const double* dztab;  /* [M] */
  double z_max_cosmo;
  orc_pop pop;          /* per-theta population constants */
} orc_cosmo_tab;

double orc_log_weight(const double* th, int mode, const orc_cosmo_tab* ct, double dL, double m1z, double m2z,
                      double lpi, const orc_los* L, int64_t row, int* live) {
  *live = 0;
  if (!(isfinite(dL) && isfinite(m1z) && isfinite(m2z) && isfinite(lpi))) return -INFINITY;
  if (!(dL > 0.0 && m1z > 0.0 && m2z > 0.0)) return -INFINITY;
  if (row < 0 || row >= L->n_rows) return -INFINITY;
  double H0 = th[P_H0], Om = th[P_OM];
  double u = dL * H0 / C_KMS;
  double z;
  if (mode == 0) {
    if (orc_z_table(u, ct->ztab, ct->dztab, ct->M, ct->umax, &z)) return -INFINITY;
  } else {
    if (!(u < ct->umax)) return -INFINITY;
    z = orc_z_of_u(u, Om);
  }
  if (!(z < L->z_max)) return -INFINITY;
  double x = 1.0 + z;
  double m1 = m1z / x, m2 = m2z / x;
  /* support: mmin < m1 <= mmax, mmin <= m2 <= m1 (m2 <= m1 <=> m2z <= m1z; reading R15) */
  if (!(m1 > th[P_MMIN] && m1 <= th[P_MMAX] && m2 >= th[P_MMIN] && m2z <= m1z)) return -INFINITY;
  double p1 = p1_c(m1, th, &ct->pop);
  double p2 = p2_c(m2 <= m1 ? m2 : m1, m1, th, &ct->pop);
  double R = psi_c(z, th, &ct->pop) / x;
  double plos = orc_los_lerp(L, row, z);
  if (!(plos > 0.0) || !(p1 > 0.0) || !(p2 > 0.0)) return -INFINITY;
  double J = x * x * (C_KMS / H0) * (u / x + x / orc_E(z, Om));
  *live = 1;
  return log(p1) + log(p2) + log(R) + log(plos) - log(J) - lpi;
}

/* two-pass log-sum-exp in long double; also LSE of 2*lw for N_eff */
static void lse2(const double* lw, int64_t n, double* lse1, double* lse_sq) {
  double mx = -INFINITY;
  for (int64_t k = 0; k < n; ++k)
    if (lw[k] > mx) mx = lw[k];
  if (mx == -INFINITY) {
    *lse1 = -INFINITY;
    *lse_sq = -INFINITY;
    return;
  }
  long double s1 = 0.0L, s2 = 0.0L;
  for (int64_t k = 0; k < n; ++k) {
    if (lw[k] == -INFINITY) continue;
    long double e = expl((long double)lw[k] - (long double)mx);
    s1 += e;
    s2 += e * e;
  }
  *lse1 = mx + (double)logl(s1);
  *lse_sq = 2.0 * mx + (double)logl(s2);
}

/* exposed for the LSE pins */
void orc_lse(const double* lw, int64_t n, double* lse1, double* neff) {
  double a, b;
  lse2(lw, n, &a, &b);
  *lse1 = a;
  *neff = (a == -INFINITY) ? 0.0 : exp(2.0 * a - b);
}

/* ------------------------------------------------------------------ */
/* Drivers.                                                            */
/* ------------------------------------------------------------------ */
typedef struct {
  int64_t n_events, n_samples;
  const int64_t* ev_sample_off; /* [n_events+1] */
  const double *dL, *m1z, *m2z;
  const double* log_pe_prior; /* or NULL => 2 ln dL */
  const int32_t* sample_row;
} orc_events;

typedef struct {
  int64_t n_found;
  double n_draw;
  const double *dL, *m1z, *m2z, *log_pdraw;
} orc_injections;

static int prep_cosmo(const double* th, int mode, double z_max, int M, orc_cosmo_tab* ct, double** buf) {
  ct->M = M;
  ct->z_max_cosmo = z_max;
  pop_init(th, &ct->pop);
  if (mode == 0) {
    *buf = (double*)malloc(sizeof(double) * 2 * (size_t)M);
    if (!*buf) return 1;
    double um;
    orc_build_table(th[P_OM], z_max, M, *buf, *buf + M, &um);
    ct->ztab = *buf;
    ct->dztab = *buf + M;
    ct->umax = um;
  } else {
    *buf = NULL;
    ct->ztab = ct->dztab = NULL;
    ct->umax = orc_u_of_z(z_max, th[P_OM]);
  }
  return 0;
}

/* optional 32-bit storage of the cosmology table (reading R22): with q = z_max / (2^32 - 1),
 * a node z_m is stored as the unsigned 32-bit integer nearest to z_m / q, its slope du z'_m as the binary32
 * nearest to (du z'_m) / q; what the look-up reads back is integer * q and (double)float * q.
 * buf = [z_0 .. z_{M-1}, d_0 .. d_{M-1}] is rewritten in place.  Pinned by tests/test_oracle_pins.py
 * (test_round_table_32_*): the quantisation bounds q/2 and 2^-24, the stored values being representable, and the
 * bound both imply on log L_i. */
void orc_round_table_32(double* buf, int M, double z_max) {
  const double qmax = 4294967295.0;
  const double q = z_max / qmax;
  for (int i = 0; i < M; ++i) {
    double k = nearbyint(buf[i] / q);
    if (k > qmax) k = qmax;
    if (k < 0.0) k = 0.0;
    buf[i] = k * q;
  }
  for (int i = M; i < 2 * M; ++i) buf[i] = (double)(float)(buf[i] / q) * q;
}

/*
 * log L_i(theta) = LSE_k log w_ik - ln S_i, N_eff,i, nlive_i  for every (theta, event).
 * Outputs [n_theta][n_events] row-major.  table_prec: 0 = f64 cosmology table, 1 = 32-bit storage (R22).
 */
int orc_event_loglik(const double* theta, int64_t n_theta, const orc_events* ev, const orc_los* L, int mode,
                     double z_max, int M, int table_prec, double* logL, double* neff, int64_t* nlive) {
  int err = 0;
  int64_t smax = 0;
  for (int64_t i = 0; i < ev->n_events; ++i) {
    int64_t s = ev->ev_sample_off[i + 1] - ev->ev_sample_off[i];
    if (s > smax) smax = s;
  }
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t t = 0; t < n_theta; ++t) {
    const double* th = theta + t * ORC_NPAR;
    double* lw = (double*)malloc(sizeof(double) * (size_t)(smax > 0 ? smax : 1));
    if (!orc_theta_valid(th) || !lw) {
      for (int64_t i = 0; i < ev->n_events; ++i) {
        logL[t * ev->n_events + i] = NAN;
        if (neff) neff[t * ev->n_events + i] = NAN;
        if (nlive) nlive[t * ev->n_events + i] = 0;
      }
      if (!lw) err = 1;
      free(lw);
      continue;
    }
    orc_cosmo_tab ct;
    double* buf = NULL;
    if (prep_cosmo(th, mode, z_max, M, &ct, &buf)) { err = 1; free(lw); continue; }
    if (mode == 0 && table_prec == 1) orc_round_table_32(buf, M, z_max);
    for (int64_t i = 0; i < ev->n_events; ++i) {
      int64_t a = ev->ev_sample_off[i], b = ev->ev_sample_off[i + 1];
      int64_t cnt = 0;
      for (int64_t k = a; k < b; ++k) {
        double lpi = ev->log_pe_prior ? ev->log_pe_prior[k] : 2.0 * log(ev->dL[k]);
        int live;
        lw[k - a] = orc_log_weight(th, mode, &ct, ev->dL[k], ev->m1z[k], ev->m2z[k], lpi, L,
                                   (int64_t)ev->sample_row[k], &live);
        cnt += live;
      }
      double l1, l2;
      lse2(lw, b - a, &l1, &l2);
      logL[t * ev->n_events + i] = (b > a) ? l1 - log((double)(b - a)) : -INFINITY;
      if (neff) neff[t * ev->n_events + i] = (l1 == -INFINITY) ? 0.0 : exp(2.0 * l1 - l2);
      if (nlive) nlive[t * ev->n_events + i] = cnt;
    }
    free(buf);
    free(lw);
  }
  return err;
}

/*
 * NEXT row 2: the per-pixel effective-sample cut of Eq. 8 (fiducial threshold 2,
 * PAPER.md:194).  A pixel of event i is a maximal run of consecutive samples with the same sample_row (the A0
 * packing makes every (event, row) one run).  With the weights of Eq. 7 taken relative to the run's largest,
 *   W_j = sum_k w_k,  Q_j = sum_k w_k^2,  N_eff,j = W_j^2 / Q_j,
 * pixel j contributes iff it has a live sample and W_j^2 >= neff_min * Q_j (decided in this linear form, so that
 * a pixel of n equal weights has N_eff = n exactly); "If a pixel does not pass this threshold ... it does not
 * contribute to the total likelihood".  Then  log L_i = LSE over the samples of the passing pixels - ln S_i
 * (S_i still counts every sample of the event: DESIGN.md R25), N_eff,i and nlive_i over the same samples, and
 * npass_i = number of passing pixels.
 */
int orc_event_loglik_pixcut(const double* theta, int64_t n_theta, const orc_events* ev, const orc_los* L, int mode,
                            double z_max, int M, int table_prec, double neff_min, double* logL, double* neff,
                            int64_t* nlive, int64_t* npass) {
  int err = 0;
  int64_t smax = 0;
  for (int64_t i = 0; i < ev->n_events; ++i) {
    int64_t s = ev->ev_sample_off[i + 1] - ev->ev_sample_off[i];
    if (s > smax) smax = s;
  }
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t t = 0; t < n_theta; ++t) {
    const double* th = theta + t * ORC_NPAR;
    double* lw = (double*)malloc(sizeof(double) * (size_t)(smax > 0 ? smax : 1));
    double* keep = (double*)malloc(sizeof(double) * (size_t)(smax > 0 ? smax : 1));
    int* lv = (int*)malloc(sizeof(int) * (size_t)(smax > 0 ? smax : 1));
    if (!orc_theta_valid(th) || !lw || !keep || !lv) {
      for (int64_t i = 0; i < ev->n_events; ++i) {
        logL[t * ev->n_events + i] = NAN;
        if (neff) neff[t * ev->n_events + i] = NAN;
        if (nlive) nlive[t * ev->n_events + i] = 0;
        if (npass) npass[t * ev->n_events + i] = 0;
      }
      if (!lw || !keep || !lv) err = 1;
      free(lw); free(keep); free(lv);
      continue;
    }
    orc_cosmo_tab ct;
    double* buf = NULL;
    if (prep_cosmo(th, mode, z_max, M, &ct, &buf)) { err = 1; free(lw); free(keep); free(lv); continue; }
    if (mode == 0 && table_prec == 1) orc_round_table_32(buf, M, z_max);
    for (int64_t i = 0; i < ev->n_events; ++i) {
      int64_t a = ev->ev_sample_off[i], b = ev->ev_sample_off[i + 1];
      for (int64_t k = a; k < b; ++k) {
        double lpi = ev->log_pe_prior ? ev->log_pe_prior[k] : 2.0 * log(ev->dL[k]);
        lw[k - a] = orc_log_weight(th, mode, &ct, ev->dL[k], ev->m1z[k], ev->m2z[k], lpi, L,
                                   (int64_t)ev->sample_row[k], &lv[k - a]);
      }
      int64_t nkeep = 0, cnt = 0, np = 0;
      int64_t r0 = a;
      while (r0 < b) {                       /* one pixel: samples r0 .. r1-1 */
        int64_t r1 = r0 + 1;
        while (r1 < b && ev->sample_row[r1] == ev->sample_row[r0]) ++r1;
        double m = -INFINITY;
        for (int64_t k = r0; k < r1; ++k) if (lw[k - a] > m) m = lw[k - a];
        if (m > -INFINITY) {
          long double W = 0.0L, Q = 0.0L;
          for (int64_t k = r0; k < r1; ++k) {
            if (lw[k - a] == -INFINITY) continue;
            double e = exp(lw[k - a] - m);
            W += e;
            Q += (long double)e * e;
          }
          double Wd = (double)W, Qd = (double)Q;
          if (Wd * Wd >= neff_min * Qd) {
            ++np;
            for (int64_t k = r0; k < r1; ++k) { keep[nkeep++] = lw[k - a]; cnt += lv[k - a]; }
          }
        }
        r0 = r1;
      }
      double l1, l2;
      lse2(keep, nkeep, &l1, &l2);
      logL[t * ev->n_events + i] = (b > a) ? l1 - log((double)(b - a)) : -INFINITY;
      if (neff) neff[t * ev->n_events + i] = (l1 == -INFINITY) ? 0.0 : exp(2.0 * l1 - l2);
      if (nlive) nlive[t * ev->n_events + i] = cnt;
      if (npass) npass[t * ev->n_events + i] = np;
    }
    free(buf);
    free(lw); free(keep); free(lv);
  }
  return err;
}

/* ------------------------------------------------------------------------------------------------ */
/* NEXT row 1: the paper's own numerator, a kernel density estimate in z per sky pixel   */
/* (Eq. 5-7; bandwidth Eq. D1; 256-node grid).             */
/* Readings R26-R30 of DESIGN.md.  For pixel j of event i (a run of equal sample_row, R25):            */
/*   v_k  = p(m1, m2 | theta) / (J pi_PE)      the weight of Eq. 7 without the redshift prior          */
/*   h_j  = 1.06 sigma_j n_j^(-1/5)            sigma_j = v-weighted standard deviation of the z_k,      */
/*                                             n_j = live samples of the pixel                          */
/*   f_j(z) = sum_k v_k N(z; z_k, h_j)          Eq. 6, Gaussian kernel                                   */
/*   I_j  = trapezoid over the G-node uniform grid on [0, z_max] of f_j(z) p_los(z | row_j) R(z; theta) */
/*   L_i  = (1/S_i) sum_j I_j over the pixels with n_j >= 2, sigma_j > 0 and N_eff,j >= neff_min.      */
/* ------------------------------------------------------------------------------------------------ */
/* log v_k and z_k of one sample; -INFINITY when dead (same support rules as orc_log_weight, minus p_los > 0) */
static double kde_sample(const double* th, int mode, const orc_cosmo_tab* ct, double dL, double m1z, double m2z,
                         double lpi, double los_z_max, int64_t row, int64_t n_rows, double* z_out) {
  *z_out = 0.0;
  if (!(isfinite(dL) && isfinite(m1z) && isfinite(m2z) && isfinite(lpi))) return -INFINITY;
  if (!(dL > 0.0 && m1z > 0.0 && m2z > 0.0)) return -INFINITY;
  if (row < 0 || row >= n_rows) return -INFINITY;
  double H0 = th[P_H0], Om = th[P_OM];
  double u = dL * H0 / C_KMS;
  double z;
  if (mode == 0) {
    if (orc_z_table(u, ct->ztab, ct->dztab, ct->M, ct->umax, &z)) return -INFINITY;
  } else {
    if (!(u < ct->umax)) return -INFINITY;
    z = orc_z_of_u(u, Om);
  }
  if (!(z < los_z_max)) return -INFINITY;
  double x = 1.0 + z;
  double m1 = m1z / x, m2 = m2z / x;
  if (!(m1 > th[P_MMIN] && m1 <= th[P_MMAX] && m2 >= th[P_MMIN] && m2z <= m1z)) return -INFINITY;
  double p1 = p1_c(m1, th, &ct->pop);
  double p2 = p2_c(m2 <= m1 ? m2 : m1, m1, th, &ct->pop);
  if (!(p1 > 0.0) || !(p2 > 0.0)) return -INFINITY;
  double J = x * x * (C_KMS / H0) * (u / x + x / orc_E(z, Om));
  *z_out = z;
  return log(p1) + log(p2) - log(J) - lpi;
}

/* per-sample (z_k, log v_k) of one theta, for the pins (numpy recomputes bandwidths and closed forms from them) */
int orc_kde_samples(const double* th, const orc_events* ev, int64_t n_rows, double los_z_max, int mode, double z_max,
                    int M, double* z_out, double* lv_out) {
  if (!orc_theta_valid(th)) return 1;
  orc_cosmo_tab ct;
  double* buf = NULL;
  if (prep_cosmo(th, mode, z_max, M, &ct, &buf)) return 1;
  for (int64_t k = 0; k < ev->n_samples; ++k) {
    double lpi = ev->log_pe_prior ? ev->log_pe_prior[k] : 2.0 * log(ev->dL[k]);
    lv_out[k] = kde_sample(th, mode, &ct, ev->dL[k], ev->m1z[k], ev->m2z[k], lpi, los_z_max,
                           (int64_t)ev->sample_row[k], n_rows, &z_out[k]);
  }
  free(buf);
  return 0;
}

/*
 * log L_i(theta) with the KDE numerator, for every (theta, event); npass = pixels that contributed.
 * n_grid = G (>= 2).  Outputs [n_theta][n_events].
 */
static int dbl_cmp(const void* a, const void* b) {
  double x = *(const double*)a, y = *(const double*)b;
  return x < y ? -1 : (x > y ? 1 : 0);
}

/* q-quantile of sorted x[0..n-1] by linear interpolation between the order statistics at q (n-1) (the "linear"
 * definition: numpy's default) */
static double quantile_sorted(const double* x, int64_t n, double q) {
  double pos = q * (double)(n - 1);
  int64_t lo = (int64_t)floor(pos);
  if (lo >= n - 1) return x[n - 1];
  double f = pos - (double)lo;
  return x[lo] + f * (x[lo + 1] - x[lo]);
}

/* Biweight midvariance, Eq. D3-D4, of x[0..n-1]; `work` holds 2n doubles.
 *   Q = median, MAD = median |x_i - Q|, u_i = (x_i - Q) / (9 MAD),
 *   D3 = n sum_{|u_i|<1} (x_i - Q)^2 (1 - u_i^2)^4 / (sum_{|u_i|<1} (1 - u_i^2)(1 - 5 u_i^2))^2.
 * Returns NaN when MAD = 0 or the denominator vanishes (no scale: the pixel has no bandwidth, reading R37). */
double orc_biweight_midvariance(const double* x, int64_t n, double* work) {
  if (n < 1) return NAN;
  for (int64_t i = 0; i < n; ++i) work[i] = x[i];
  qsort(work, (size_t)n, sizeof(double), dbl_cmp);
  double Q = quantile_sorted(work, n, 0.5);
  for (int64_t i = 0; i < n; ++i) work[n + i] = fabs(x[i] - Q);
  qsort(work + n, (size_t)n, sizeof(double), dbl_cmp);
  double mad = quantile_sorted(work + n, n, 0.5);
  if (!(mad > 0.0)) return NAN;
  long double num = 0.0L, den = 0.0L;
  for (int64_t i = 0; i < n; ++i) {
    double d = x[i] - Q, u = d / (9.0 * mad);
    if (!(fabs(u) < 1.0)) continue;
    double a = 1.0 - u * u;
    num += (long double)(d * d) * (a * a) * (a * a);
    den += (long double)a * (1.0 - 5.0 * u * u);
  }
  if (den == 0.0L) return NAN;
  return (double)((long double)n * num / (den * den));
}

/* bw_rule: 0 = Scott, Eq. D1; 1 = Silverman, Eq. D2:
 * h = 0.9 min(sigma, IQR / 1.34) n^(-1/5) with the IQR of the pixel's live z_k (plain quantiles, reading R32);
 * 2 = biweight midvariance as printed, h = D3 (reading R37); 3 = the same robust scale in Scott's
 * rule, h = 1.06 sqrt(D3) n^(-1/5) (R37).  D3 is taken over the pixel's live z_k, unweighted like the IQR. */
int orc_event_loglik_kde(const double* theta, int64_t n_theta, const orc_events* ev, const orc_los* L, int mode,
                         double z_max, int M, int table_prec, int n_grid, double neff_min, int bw_rule, double* logL,
                         int64_t* npass, int64_t* nused) {
  int err = 0;
  int64_t smax = 0;
  for (int64_t i = 0; i < ev->n_events; ++i) {
    int64_t s = ev->ev_sample_off[i + 1] - ev->ev_sample_off[i];
    if (s > smax) smax = s;
  }
  const double dzg = L->z_max / (n_grid - 1);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t t = 0; t < n_theta; ++t) {
    const double* th = theta + t * ORC_NPAR;
    size_t nb = (size_t)(smax > 0 ? smax : 1);
    double* lv = (double*)malloc(sizeof(double) * nb);
    double* zz = (double*)malloc(sizeof(double) * nb);
    double* lI = (double*)malloc(sizeof(double) * nb);   /* log I_j of the passing pixels of one event */
    double* Rg = (double*)malloc(sizeof(double) * (size_t)n_grid);
    double* wk = (double*)malloc(sizeof(double) * 3 * nb);   /* biweight: the live z_k and two sorted copies */
    if (!wk) { free(lv); lv = NULL; }
    if (!orc_theta_valid(th) || !lv || !zz || !lI || !Rg) {
      for (int64_t i = 0; i < ev->n_events; ++i) {
        logL[t * ev->n_events + i] = NAN;
        if (npass) npass[t * ev->n_events + i] = 0;
        if (nused) nused[t * ev->n_events + i] = 0;
      }
      if (!lv || !zz || !lI || !Rg) err = 1;
      free(lv); free(zz); free(lI); free(Rg); free(wk);
      continue;
    }
    orc_cosmo_tab ct;
    double* buf = NULL;
    if (prep_cosmo(th, mode, z_max, M, &ct, &buf)) { err = 1; free(lv); free(zz); free(lI); free(Rg); free(wk); continue; }
    if (mode == 0 && table_prec == 1) orc_round_table_32(buf, M, z_max);
    for (int g = 0; g < n_grid; ++g) {            /* rate term on the grid: R(z) = psi(z) / (1+z), reading R4 */
      double zg = g * dzg;
      Rg[g] = psi_c(zg, th, &ct.pop) / (1.0 + zg);
    }
    for (int64_t i = 0; i < ev->n_events; ++i) {
      int64_t a = ev->ev_sample_off[i], b = ev->ev_sample_off[i + 1];
      for (int64_t k = a; k < b; ++k) {
        double lpi = ev->log_pe_prior ? ev->log_pe_prior[k] : 2.0 * log(ev->dL[k]);
        lv[k - a] = kde_sample(th, mode, &ct, ev->dL[k], ev->m1z[k], ev->m2z[k], lpi, L->z_max,
                               (int64_t)ev->sample_row[k], L->n_rows, &zz[k - a]);
      }
      int64_t np = 0, nu = 0;
      int64_t r0 = a;
      while (r0 < b) {                            /* one pixel: samples r0 .. r1-1 */
        int64_t r1 = r0 + 1;
        while (r1 < b && ev->sample_row[r1] == ev->sample_row[r0]) ++r1;
        int64_t row = ev->sample_row[r0];
        int64_t n = 0;
        double m = -INFINITY;
        for (int64_t k = r0; k < r1; ++k)
          if (lv[k - a] > -INFINITY) { ++n; if (lv[k - a] > m) m = lv[k - a]; }
        if (n >= 2) {
          long double V = 0.0L, Vz = 0.0L, Q = 0.0L;
          for (int64_t k = r0; k < r1; ++k) {
            if (lv[k - a] == -INFINITY) continue;
            double e = exp(lv[k - a] - m);
            V += e; Vz += (long double)e * zz[k - a]; Q += (long double)e * e;
          }
          double mu = (double)(Vz / V);
          long double S2 = 0.0L;
          for (int64_t k = r0; k < r1; ++k) {
            if (lv[k - a] == -INFINITY) continue;
            double e = exp(lv[k - a] - m), d = zz[k - a] - mu;
            S2 += (long double)e * d * d;
          }
          double var = (double)(S2 / V);
          double Vd = (double)V, Qd = (double)Q;
          if (var > 0.0 && Vd * Vd >= neff_min * Qd) {
            double h = 1.06 * sqrt(var) * pow((double)n, -0.2);            /* Eq. D1 */
            if (bw_rule == 1) {                                              /* Eq. D2 */
              int64_t c = 0;
              for (int64_t k = r0; k < r1; ++k)
                if (lv[k - a] > -INFINITY) lI[np + c++] = zz[k - a];          /* (free tail of lI as a work area) */
              qsort(lI + np, (size_t)c, sizeof(double), dbl_cmp);
              double iqr = quantile_sorted(lI + np, c, 0.75) - quantile_sorted(lI + np, c, 0.25);
              double spread = sqrt(var);
              if (iqr / 1.34 < spread) spread = iqr / 1.34;
              h = 0.9 * spread * pow((double)n, -0.2);
              if (!(h > 0.0)) { r0 = r1; continue; }                          /* IQR = 0: no bandwidth, no contribution */
            } else if (bw_rule == 2 || bw_rule == 3) {                        /* Eq. D3-D4 */
              int64_t c = 0;
              for (int64_t k = r0; k < r1; ++k)
                if (lv[k - a] > -INFINITY) wk[c++] = zz[k - a];
              double zeta2 = orc_biweight_midvariance(wk, c, wk + c);
              h = bw_rule == 2 ? zeta2 : 1.06 * sqrt(zeta2) * pow((double)n, -0.2);
              if (!(h > 0.0) || !isfinite(h)) { r0 = r1; continue; }          /* no scale: no contribution */
            }
            double norm = 1.0 / (h * sqrt(2.0 * M_PI));
            long double I = 0.0L;
            for (int g = 0; g < n_grid; ++g) {
              double zg = g * dzg;
              double f = 0.0;                                                /* Eq. 6 at z_g, relative to e^m */
              for (int64_t k = r0; k < r1; ++k) {
                if (lv[k - a] == -INFINITY) continue;
                double q = (zg - zz[k - a]) / h;
                double g2 = 0.5 * q * q;
                if (g2 > 700.0) continue;      /* a kernel value below e^-700 is zero (reading R38) */
                f += exp(lv[k - a] - m) * norm * exp(-g2);
              }
              double zl = zg < L->z_max ? zg : L->z_max;                     /* last node: the table's last value */
              double prior = orc_los_lerp(L, row, zl) * Rg[g];
              double c = (g == 0 || g == n_grid - 1) ? 0.5 * dzg : dzg;      /* trapezoid */
              I += (long double)c * f * prior;
            }
            if (I > 0.0L) { lI[np++] = m + (double)logl(I); nu += n; }
          }
        }
        r0 = r1;
      }
      double l1, l2;
      lse2(lI, np, &l1, &l2);
      logL[t * ev->n_events + i] = (b > a) ? l1 - log((double)(b - a)) : -INFINITY;
      if (npass) npass[t * ev->n_events + i] = np;
      if (nused) nused[t * ev->n_events + i] = nu;
    }
    free(buf);
    free(lv); free(zz); free(lI); free(Rg); free(wk);
  }
  return err;
}

/*
 * log xi(theta) = LSE_j log w_j - ln n_draw over found injections, with the all-sky
 * prior (a 1-row f64 table) in place of the pixel row and log_pdraw in place of the PE prior.
 */
int orc_selection_logxi(const double* theta, int64_t n_theta, const orc_injections* inj, const double* allsky,
                        int32_t n_z, double los_z_max, int mode, double z_max, int M, int table_prec,
                        double* logxi, double* neff_inj) {
  int err = 0;
  orc_los A;
  A.n_rows = 1;
  A.n_z = n_z;
  A.z_max = los_z_max;
  A.prec = 0;
  A.table = allsky;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t t = 0; t < n_theta; ++t) {
    const double* th = theta + t * ORC_NPAR;
    double* lw = (double*)malloc(sizeof(double) * (size_t)(inj->n_found > 0 ? inj->n_found : 1));
    if (!orc_theta_valid(th) || !lw) {
      logxi[t] = NAN;
      if (neff_inj) neff_inj[t] = NAN;
      if (!lw) err = 1;
      free(lw);
      continue;
    }
    orc_cosmo_tab ct;
    double* buf = NULL;
    if (prep_cosmo(th, mode, z_max, M, &ct, &buf)) { err = 1; free(lw); continue; }
    if (mode == 0 && table_prec == 1) orc_round_table_32(buf, M, z_max);
    for (int64_t k = 0; k < inj->n_found; ++k) {
      int live;
      lw[k] = orc_log_weight(th, mode, &ct, inj->dL[k], inj->m1z[k], inj->m2z[k], inj->log_pdraw[k], &A, 0, &live);
    }
    double l1, l2;
    lse2(lw, inj->n_found, &l1, &l2);
    logxi[t] = l1 - log(inj->n_draw);
    if (neff_inj) neff_inj[t] = (l1 == -INFINITY) ? 0.0 : exp(2.0 * l1 - l2);
    free(buf);
    free(lw);
  }
  return err;
}

/* log L(theta) = sum_i log L_i - n_events * log xi  (Eq. 3/5; any -inf term => -inf, never NaN) */
void orc_total_from_parts(const double* logL, const double* logxi, int64_t n_theta, int64_t n_events, double* total) {
  for (int64_t t = 0; t < n_theta; ++t) {
    long double s = 0.0L;
    int neg_inf = 0, nan = 0;
    for (int64_t i = 0; i < n_events; ++i) {
      double v = logL[t * n_events + i];
      if (isnan(v)) nan = 1;
      else if (v == -INFINITY) neg_inf = 1;
      else s += v;
    }
    double x = logxi[t];
    if (isnan(x)) nan = 1;
    if (nan) total[t] = NAN;
    else if (neg_inf || x == -INFINITY) total[t] = -INFINITY;
    else total[t] = (double)(s - (long double)n_events * (long double)x);
  }
}

/* ------------------------------------------------------------------ */
/* A0 packing: stable sort of samples by (event, row); CSR pieces.      */
/* ------------------------------------------------------------------ */
typedef struct { int32_t ev, row; int64_t idx; } pack_key;

static int pack_cmp(const void* a, const void* b) {
  const pack_key* x = (const pack_key*)a;
  const pack_key* y = (const pack_key*)b;
  if (x->ev != y->ev) return x->ev < y->ev ? -1 : 1;
  if (x->row != y->row) return x->row < y->row ? -1 : 1;
  if (x->idx != y->idx) return x->idx < y->idx ? -1 : 1; /* ties keep input order */
  return 0;
}

/*
 * Inputs: per-sample event id and LOS row, arbitrary order.  Outputs: perm (sorted position ->
 * input index), ev_sample_off[n_events+1], ev_pix_off[n_events+1], ev_pix_rows[n_pixrefs],
 * pix_sample_off[n_pixrefs+1]; returns n_pixrefs (distinct (event,row) pairs), or -1 on error.
 */
int64_t orc_pack_events(int64_t n_samples, int64_t n_events, const int32_t* event_id, const int32_t* row,
                        int64_t* perm, int64_t* ev_sample_off, int64_t* ev_pix_off, int32_t* ev_pix_rows,
                        int64_t* pix_sample_off) {
  pack_key* keys = (pack_key*)malloc(sizeof(pack_key) * (size_t)(n_samples > 0 ? n_samples : 1));
  if (!keys) return -1;
  for (int64_t k = 0; k < n_samples; ++k) {
    if (event_id[k] < 0 || event_id[k] >= n_events) { free(keys); return -1; }
    keys[k].ev = event_id[k];
    keys[k].row = row[k];
    keys[k].idx = k;
  }
  qsort(keys, (size_t)n_samples, sizeof(pack_key), pack_cmp);
  for (int64_t i = 0; i <= n_events; ++i) ev_sample_off[i] = 0;
  for (int64_t k = 0; k < n_samples; ++k) {
    perm[k] = keys[k].idx;
    ev_sample_off[keys[k].ev + 1] += 1;
  }
  for (int64_t i = 0; i < n_events; ++i) ev_sample_off[i + 1] += ev_sample_off[i];
  int64_t np = 0;
  for (int64_t i = 0; i < n_events; ++i) {
    ev_pix_off[i] = np;
    for (int64_t k = ev_sample_off[i]; k < ev_sample_off[i + 1]; ++k) {
      if (k == ev_sample_off[i] || keys[k].row != keys[k - 1].row) {
        ev_pix_rows[np] = keys[k].row;
        pix_sample_off[np] = k;
        ++np;
      }
    }
  }
  ev_pix_off[n_events] = np;
  pix_sample_off[np] = n_samples;
  free(keys);
  return np;
}

/*
 * NEXT row 3b: the per-pixel sample cap, "the option to randomly downsample the GW posterior
 * samples in a given pixel" (fiducial 2500).  Reading R31: applied to a packed
 * catalogue; a pixel ((event, row) run) of n > cap samples keeps the cap samples with the smallest
 * (hash32(seed, original sample index), packed position); smaller pixels keep everything; kept samples keep their
 * packed order.  hash32 = the upper half of splitmix64's output function applied to seed + (index+1) * golden.
 * perm_in [n_samples], ev_sample_off [n_events+1] and pix_sample_off [n_pix+1] are those of orc_pack_events;
 * the two offset arrays are rewritten for the kept samples, perm_out receives the kept entries of perm_in.
 * Returns the number of kept samples.
 */
static uint32_t cap_hash32(uint64_t seed, uint64_t index) {
  uint64_t z = seed + (index + 1ULL) * 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  z = z ^ (z >> 31);
  return (uint32_t)(z >> 32);
}

typedef struct { uint32_t h; int64_t pos; } cap_key;
static int cap_cmp(const void* a, const void* b) {
  const cap_key* x = (const cap_key*)a;
  const cap_key* y = (const cap_key*)b;
  if (x->h != y->h) return x->h < y->h ? -1 : 1;
  return x->pos < y->pos ? -1 : (x->pos > y->pos ? 1 : 0);
}

int64_t orc_cap_pixels(int64_t n_samples, int64_t n_events, int64_t n_pix, const int64_t* perm_in,
                       int64_t* ev_sample_off, int64_t* pix_sample_off, int64_t cap, uint64_t seed,
                       int64_t* perm_out) {
  if (cap < 1) return -1;
  char* keep = (char*)calloc((size_t)(n_samples > 0 ? n_samples : 1), 1);
  cap_key* keys = (cap_key*)malloc(sizeof(cap_key) * (size_t)(n_samples > 0 ? n_samples : 1));
  int64_t* newpos = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n_samples + 1));
  if (!keep || !keys || !newpos) { free(keep); free(keys); free(newpos); return -1; }
  for (int64_t j = 0; j < n_pix; ++j) {
    int64_t a = pix_sample_off[j], b = pix_sample_off[j + 1];
    if (b - a <= cap) {
      for (int64_t k = a; k < b; ++k) keep[k] = 1;
      continue;
    }
    for (int64_t k = a; k < b; ++k) { keys[k - a].h = cap_hash32(seed, (uint64_t)perm_in[k]); keys[k - a].pos = k; }
    qsort(keys, (size_t)(b - a), sizeof(cap_key), cap_cmp);
    for (int64_t r = 0; r < cap; ++r) keep[keys[r].pos] = 1;
  }
  int64_t nk = 0;
  for (int64_t k = 0; k < n_samples; ++k) {
    newpos[k] = nk;
    if (keep[k]) perm_out[nk++] = perm_in[k];
  }
  newpos[n_samples] = nk;
  for (int64_t i = 0; i <= n_events; ++i) ev_sample_off[i] = newpos[ev_sample_off[i]];
  for (int64_t j = 0; j <= n_pix; ++j) pix_sample_off[j] = newpos[pix_sample_off[j]];
  free(keep); free(keys); free(newpos);
  return nk;
}

