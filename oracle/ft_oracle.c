/*
 * ft_oracle.c — CPU ORACLE for the fasttracks hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  The product (paper_2411_18370_b200/) never does, and this
 * file shares no code, header, table or helper with the CUDA path.
 *
 * What it computes is the PLAIN DEFINITION of the paper's method ("without using any
 * computational approximations"): for every template, for every SFT, evaluate the
 * frequency track (Eq. 2, extended with f1/t_ref as BASELINE.json north_star
 * writes it), round to a frequency bin ("frequency is naturally discretised in steps of
 * 1/T_SFT"), gather the spectrogram pixel and reduce (Eq. 3 for the
 * weighted normalized power, Eq. 7 for the number count).  No blocking, hoisting,
 * fusion or reordering: one loop over templates, one loop over SFTs, in the order and with the
 * operation sequence DESIGN.md "Canonical computation" lists.  All arithmetic is IEEE binary64
 * (compile with -ffp-contract=off so no FMA is formed); the spectrogram and the weights are
 * fp32 data, so (double)w*(double)p is exact.
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): noise mean/variance (Eq. 13-14),
 * binomial number count (Eq. 7, 11), a_p = 0 reduction, straight-line column sum,
 * injected-track recovery (Eq. 3, Eq. 24 m=0), one-bin resolution property (Eq. 27, A1),
 * exact-rational / 50-digit evaluation of the track, hand-built half-integer rounding cases,
 * linearity and permutation invariance, pure-Python brute force on tiny inputs; width of the
 * near-tie window (hand-built x = k + 0.5 -+ 5e-10 / 2e-9); antenna-pattern weights (Eq. 4-5): sky
 * average 2/5 of a^2 + b^2, time independence at the poles, F+^2 + Fx^2 from the detector tensor,
 * sum w = 1; standardised statistic z (Eq. 36): noise mean 0 / variance 1; xi coordinates (Eq. A11):
 * round trip, marginal densities f0^5, a_p^2, Omega^3 (Eq. A9), uniformity of the counter generator.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define FTO_OK 0
#define FTO_ERR_RANGE (-4) /* a track left [0, n_bins): DESIGN.md reading R9, an error, not a clamp */

static const double TWO_PI = 6.283185307179586; /* nearest double to 2*pi */
static const double C_LIGHT = 299792458.0;      /* m/s */

typedef struct {
  /* spectrogram and per-SFT tables (PAPER.md:60 SFT data model; rows = SFTs of all detectors) */
  const float* P;       /* [n_sft][ld] normalized power on the Exponential(1) scale (Eq. 6 / 2) */
  int64_t n_sft, n_bins, ld;
  const double* t_mid;  /* [n_sft] SFT mid-times, s */
  const double* vel;    /* [n_sft][3] detector velocity, m/s, equatorial */
  const float* w;       /* wkind 1: [n_sft]; wkind 2: [n_sft][ld] (Eq. 4-5, used as given) */
  int32_t wkind;
  double f_min, df;     /* bin k is centred at f_min + k*df */
  /* template grid axes */
  double f0_start, df0; int64_t n_f0;
  double f1_start, df1; int64_t n_f1;
  double t_ref;
  int64_t n_sky;  const double* sky;        /* [n_sky][3] unit vectors */
  int64_t n_ap;   const double* a_p;        /* light-seconds */
  int64_t n_porb; const double* P_orb;      /* seconds */
  int64_t n_tasc; const double* tasc_frac;  /* t_asc = t_ref + u*P_orb */
  double rho_th;
  /* sky-dependent weights (Eq. 4-5): per-SFT detector latitude, arm-bisector orientation gamma (counter-
   * clockwise from East) and local sidereal angle at the SFT mid-time, radians; all NULL = weights as given */
  const double* det_lat; const double* det_gamma; const double* lst;
} fto_problem;

/* canonical linear template index -> axis indices (fastest axis: f0) */
static void fto_unravel(const fto_problem* pb, uint64_t idx, int64_t ax[6]) {
  ax[5] = (int64_t)(idx % (uint64_t)pb->n_f0);   idx /= (uint64_t)pb->n_f0;
  ax[4] = (int64_t)(idx % (uint64_t)pb->n_f1);   idx /= (uint64_t)pb->n_f1;
  ax[3] = (int64_t)(idx % (uint64_t)pb->n_tasc); idx /= (uint64_t)pb->n_tasc;
  ax[2] = (int64_t)(idx % (uint64_t)pb->n_porb); idx /= (uint64_t)pb->n_porb;
  ax[1] = (int64_t)(idx % (uint64_t)pb->n_ap);   idx /= (uint64_t)pb->n_ap;
  ax[0] = (int64_t)idx;
}

/*
 * Amplitude-modulation functions a(t), b(t) of an interferometer with perpendicular arms: Eq. (12)-(13) of
 * Jaranowski, Krolak & Schutz, Phys. Rev. D 58, 063001 (1998) -- the paper's ref. [20], "a and b are the
 * detector's response functions".  lat = detector latitude lambda, gamma = angle from East to
 * the bisector of the arms (counter-clockwise), lst = phi_r + Omega_r t, the local sidereal angle of the
 * detector at time t; (ra, dec) the source.  F+ = sin(zeta) [a cos 2psi + b sin 2psi].
 */
void fto_antenna_ab(double lat, double gamma, double lst, double ra, double dec, double* a, double* b) {
  const double ph = ra - lst;
  *a = (1.0 / 16.0) * sin(2.0 * gamma) * (3.0 - cos(2.0 * lat)) * (3.0 - cos(2.0 * dec)) * cos(2.0 * ph)
     - 0.25 * cos(2.0 * gamma) * sin(lat) * (3.0 - cos(2.0 * dec)) * sin(2.0 * ph)
     + 0.25 * sin(2.0 * gamma) * sin(2.0 * lat) * sin(2.0 * dec) * cos(ph)
     - 0.5 * cos(2.0 * gamma) * cos(lat) * sin(2.0 * dec) * sin(ph)
     + 0.75 * sin(2.0 * gamma) * cos(lat) * cos(lat) * cos(dec) * cos(dec);
  *b = cos(2.0 * gamma) * sin(lat) * sin(dec) * cos(2.0 * ph)
     + 0.25 * sin(2.0 * gamma) * (3.0 - cos(2.0 * lat)) * sin(dec) * sin(2.0 * ph)
     + cos(2.0 * gamma) * cos(lat) * cos(dec) * cos(ph)
     + 0.5 * sin(2.0 * gamma) * sin(2.0 * lat) * cos(dec) * sin(ph);
}

/* One explicit template lambda = (f0, f1, n, a_p, P_orb, t_asc): "no assumption on the properties of
 * lambda"; random template banks are drawn this way. */
typedef struct { double f0, f1, nx, ny, nz, a_p, P_orb, t_asc; } fto_template;

/*
 * One template: track -> bin per SFT (Eq. 2), then the statistics (Eq. 3, Eq. 7).
 * k_out / x_out may be NULL.  Returns FTO_ERR_RANGE if any bin falls outside the spectrogram.
 */
static int fto_one_params(const fto_problem* pb, const fto_template* tp, double t_ref, double* power,
                          int32_t* count, double* wcount, uint8_t* near_tie, int64_t* k_out,
                          double* x_out, double* z_out, double* sigma_out) {
  const double inv_df = 1.0 / pb->df;
  const double f0 = tp->f0, f1 = tp->f1;
  const double nx = tp->nx, ny = tp->ny, nz = tp->nz;
  const double a_p = tp->a_p;
  const double Om = TWO_PI / tp->P_orb;          /* Omega */
  const double t_asc = tp->t_asc;                /* phi_b = t_asc * Omega */
  const float rho = (float)pb->rho_th;

  /* Eq. (4)-(5): w_a(n) = u_a r_a / sum_b u_b r_b, u = a^2 + b^2, r = the per-SFT weights given (∝ 1/S_a) */
  const int skyw = pb->det_lat != NULL;
  double ra = 0.0, dec = 0.0, wnorm = 1.0;
  if (skyw) {
    if (pb->wkind == 2) return FTO_ERR_RANGE + 100;  /* per-bin weights cannot be normalised per sky point */
    ra = atan2(ny, nx);
    dec = atan2(nz, sqrt(nx * nx + ny * ny));
    double sum = 0.0;
    for (int64_t a = 0; a < pb->n_sft; ++a) {
      double aa, bb;
      fto_antenna_ab(pb->det_lat[a], pb->det_gamma[a], pb->lst[a], ra, dec, &aa, &bb);
      sum += (aa * aa + bb * bb) * (double)pb->w[a];
    }
    wnorm = sum;
  }

  double s_power = 0.0, s_wcount = 0.0, s_mu = 0.0, s_var = 0.0;
  int32_t s_count = 0;
  uint8_t tie = 0;
  for (int64_t a = 0; a < pb->n_sft; ++a) {
    const double t = pb->t_mid[a];
    const double dt = t - t_ref;
    const double fs = f0 + f1 * dt;                               /* spun-down frequency */
    const double V = ((pb->vel[3 * a] * nx + pb->vel[3 * a + 1] * ny) + pb->vel[3 * a + 2] * nz) / C_LIGHT;
    double B = 0.0;                                               /* a_p = 0: isolated */
    if (a_p != 0.0) B = (a_p * Om) * cos(Om * (t - t_asc));
    const double D = (1.0 + V) - B;                               /* bracket of Eq. 2 */
    const double x = ((fs * D) - pb->f_min) * inv_df;             /* position in bins */
    const double kr = nearbyint(x);                               /* round-half-to-even (R5) */
    if (fabs((x - floor(x)) - 0.5) < 1e-9) tie = 1;               /* within 1e-9 bin of a tie */
    const int64_t k = (int64_t)kr;
    if (k_out) k_out[a] = k;
    if (x_out) x_out[a] = x;
    if (k < 0 || k >= pb->n_bins) return FTO_ERR_RANGE;
    const float p = pb->P[a * pb->ld + k];
    const float wf = (pb->wkind == 2) ? pb->w[a * pb->ld + k] : pb->w[a];
    double w = (double)wf;
    if (skyw) {
      double aa, bb;
      fto_antenna_ab(pb->det_lat[a], pb->det_gamma[a], pb->lst[a], ra, dec, &aa, &bb);
      w = (aa * aa + bb * bb) * (double)wf / wnorm;
    }
    s_power += w * (double)p;                                     /* Eq. 3 */
    if (p > rho) {                                                /* Eq. 7, strict > in fp32 */
      s_count += 1;
      s_wcount += w;                                              /* weighted count */
    }
    /* Eq. (13)-(14) on the P = s/2 scale: mu_G = sum w, sigma_G^2 = sum w^2.  Per-bin weights: the box-level
     * weights are the row means (reading R21), a template-independent standardisation like mu_G(b) */
    double wz = w;
    if (pb->wkind == 2 && (z_out || sigma_out)) {
      double m = 0.0;
      for (int64_t q = 0; q < pb->n_bins; ++q) m += (double)pb->w[a * pb->ld + q];
      wz = m / (double)pb->n_bins;
    }
    s_mu += wz;
    s_var += wz * wz;
  }
  if (power) *power = s_power;
  if (count) *count = s_count;
  if (wcount) *wcount = s_wcount;
  if (near_tie) *near_tie = tie;
  if (sigma_out) *sigma_out = sqrt(s_var);
  if (z_out) *z_out = (s_power - s_mu) / sqrt(s_var);             /* Eq. 36 */
  return FTO_OK;
}

/* Grid template: canonical index -> parameters (f0 = f0_start + i df0, ..., t_asc = t_ref + u P_orb). */
static int fto_one_template(const fto_problem* pb, uint64_t idx, double* power, int32_t* count,
                            double* wcount, uint8_t* near_tie, int64_t* k_out, double* x_out,
                            double* z_out, double* sigma_out) {
  int64_t ax[6];
  fto_unravel(pb, idx, ax);
  fto_template tp;
  tp.f0 = pb->f0_start + (double)ax[5] * pb->df0;
  tp.f1 = pb->f1_start + (double)ax[4] * pb->df1;
  tp.nx = pb->sky[3 * ax[0] + 0]; tp.ny = pb->sky[3 * ax[0] + 1]; tp.nz = pb->sky[3 * ax[0] + 2];
  tp.a_p = pb->a_p[ax[1]];
  tp.P_orb = pb->P_orb[ax[2]];
  tp.t_asc = pb->t_ref + pb->tasc_frac[ax[3]] * tp.P_orb;
  return fto_one_params(pb, &tp, pb->t_ref, power, count, wcount, near_tie, k_out, x_out, z_out, sigma_out);
}

/* Track of ONE template: bins k[n_sft] and positions x[n_sft]. */
int fto_track(const fto_problem* pb, uint64_t idx, int64_t* k_out, double* x_out) {
  return fto_one_template(pb, idx, NULL, NULL, NULL, NULL, k_out, x_out, NULL, NULL);
}

/* Statistics of the contiguous canonical index range [idx_begin, idx_end).  Outputs are
 * indexed by (idx - idx_begin); any may be NULL.  OpenMP over templates only. */
int fto_eval_range(const fto_problem* pb, uint64_t idx_begin, uint64_t idx_end, double* power,
                   int32_t* count, double* wcount, uint8_t* near_tie) {
  int status = FTO_OK;
  const int64_t n = (int64_t)(idx_end - idx_begin);
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    const int rc = fto_one_template(pb, idx_begin + (uint64_t)j, power ? power + j : NULL,
                                    count ? count + j : NULL, wcount ? wcount + j : NULL,
                                    near_tie ? near_tie + j : NULL, NULL, NULL, NULL, NULL);
    if (rc != FTO_OK) {
#pragma omp atomic write
      status = rc;
    }
  }
  return status;
}

/* The same with the standardised statistic z (Eq. 36) and sigma_G of every template. */
int fto_eval_range_z(const fto_problem* pb, uint64_t idx_begin, uint64_t idx_end, double* power,
                     int32_t* count, double* wcount, uint8_t* near_tie, double* z, double* sigma) {
  int status = FTO_OK;
  const int64_t n = (int64_t)(idx_end - idx_begin);
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    const int rc = fto_one_template(pb, idx_begin + (uint64_t)j, power ? power + j : NULL,
                                    count ? count + j : NULL, wcount ? wcount + j : NULL,
                                    near_tie ? near_tie + j : NULL, NULL, NULL, z ? z + j : NULL,
                                    sigma ? sigma + j : NULL);
    if (rc != FTO_OK) {
#pragma omp atomic write
      status = rc;
    }
  }
  return status;
}

/* Statistics of an explicit list of canonical indices. */
int fto_eval_list(const fto_problem* pb, const uint64_t* idx, int64_t n, double* power,
                  int32_t* count, double* wcount, uint8_t* near_tie) {
  int status = FTO_OK;
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    const int rc = fto_one_template(pb, idx[j], power ? power + j : NULL, count ? count + j : NULL,
                                    wcount ? wcount + j : NULL, near_tie ? near_tie + j : NULL,
                                    NULL, NULL, NULL, NULL);
    if (rc != FTO_OK) {
#pragma omp atomic write
      status = rc;
    }
  }
  return status;
}

/* Statistics of an explicit list of templates (an unstructured bank); t_ref is the reference
 * time of f0 and f1.  The grid axes of pb are not used. */
int fto_eval_templates(const fto_problem* pb, const fto_template* tl, int64_t n, double t_ref,
                       double* power, int32_t* count, double* wcount, uint8_t* near_tie) {
  int status = FTO_OK;
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    const int rc = fto_one_params(pb, tl + j, t_ref, power ? power + j : NULL, count ? count + j : NULL,
                                  wcount ? wcount + j : NULL, near_tie ? near_tie + j : NULL, NULL, NULL,
                                  NULL, NULL);
    if (rc != FTO_OK) {
#pragma omp atomic write
      status = rc;
    }
  }
  return status;
}

/* The same with the standardised statistic z (Eq. 36) and sigma_G of every template of the list: the quantities the
 * paper's per-box procedure ranks a random bank by. */
int fto_eval_templates_z(const fto_problem* pb, const fto_template* tl, int64_t n, double t_ref,
                         double* power, int32_t* count, double* wcount, uint8_t* near_tie, double* z, double* sigma) {
  int status = FTO_OK;
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    const int rc = fto_one_params(pb, tl + j, t_ref, power ? power + j : NULL, count ? count + j : NULL,
                                  wcount ? wcount + j : NULL, near_tie ? near_tie + j : NULL, NULL, NULL,
                                  z ? z + j : NULL, sigma ? sigma + j : NULL);
    if (rc != FTO_OK) {
#pragma omp atomic write
      status = rc;
    }
  }
  return status;
}

/* Track (bins, positions) of ONE explicit template. */
int fto_track_template(const fto_problem* pb, const fto_template* tp, double t_ref, int64_t* k_out, double* x_out) {
  return fto_one_params(pb, tp, t_ref, NULL, NULL, NULL, NULL, k_out, x_out, NULL, NULL);
}

/*
 * Random template bank, uniform in the xi coordinates of Eq. (A11):
 *   xi = (f0^6/6, alpha, sin delta, a_p^3/3, Omega^4/4, phi_b)   up to the constant k^(1/6),
 * "draw n templates uniformly in xi, map them to lambda".  The region Delta-lambda is
 * a box in lambda (Eq. A12-A13 map its corners).  f1 (north_star's extension; the paper neglects spindown) is
 * drawn uniformly: the track is linear in f1 so its resolution does not depend on lambda (reading R22).
 * The uniforms come from a counter-based generator, u(seed, i, d) = splitmix64 finaliser of
 * seed + 0x9E3779B97F4A7C15 * (8 i + d + 1), top 53 bits, so template i does not depend on n or on the order
 * of evaluation (each side of the parity test implements it on its own).
 */
typedef struct {
  double f0_lo, f0_hi;         /* Hz */
  double f1_lo, f1_hi;         /* Hz/s */
  double ra_lo, ra_hi;         /* right ascension, rad (all-sky: 0, 2 pi) */
  double sd_lo, sd_hi;         /* sin(declination) (all-sky: -1, 1) */
  double ap_lo, ap_hi;         /* light-seconds; ap_hi == 0: isolated bank (a_p = 0, orbit unused) */
  double porb_lo, porb_hi;     /* seconds (Omega = 2 pi / P_orb) */
  double t_ref;                /* t_asc = t_ref + phi_b / Omega, phi_b uniform in [0, 2 pi) */
} fto_bank_box;

double fto_uniform(uint64_t seed, uint64_t i, uint32_t d) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * (8ull * i + (uint64_t)d + 1ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z ^= z >> 31;
  return ((double)(z >> 11) + 0.5) * (1.0 / 9007199254740992.0);   /* (0, 1), 53 bits */
}

/* xi -> lambda for one coordinate with density lambda^p: lambda = (lo^(p+1) + u (hi^(p+1) - lo^(p+1)))^(1/(p+1)) */
static double fto_inv_power(double lo, double hi, double u, int p1) {
  const double a = pow(lo, (double)p1), b = pow(hi, (double)p1);
  return pow(a + u * (b - a), 1.0 / (double)p1);
}

void fto_bank_draw(const fto_bank_box* bx, uint64_t seed, uint64_t first, int64_t n, fto_template* out) {
  for (int64_t j = 0; j < n; ++j) {
    const uint64_t i = first + (uint64_t)j;
    fto_template* tp = out + j;
    tp->f0 = fto_inv_power(bx->f0_lo, bx->f0_hi, fto_uniform(seed, i, 0), 6);        /* xi[0] = f0^6 / 6 */
    const double ra = bx->ra_lo + fto_uniform(seed, i, 1) * (bx->ra_hi - bx->ra_lo);   /* xi[1] = alpha */
    const double sd = bx->sd_lo + fto_uniform(seed, i, 2) * (bx->sd_hi - bx->sd_lo);   /* xi[2] = sin delta */
    const double cd = sqrt(1.0 - sd * sd);
    tp->nx = cd * cos(ra); tp->ny = cd * sin(ra); tp->nz = sd;
    if (bx->ap_hi > 0.0) {
      tp->a_p = fto_inv_power(bx->ap_lo, bx->ap_hi, fto_uniform(seed, i, 3), 3);      /* xi[3] = a_p^3 / 3 */
      const double Om = fto_inv_power(TWO_PI / bx->porb_hi, TWO_PI / bx->porb_lo, fto_uniform(seed, i, 4), 4); /* xi[4] = Omega^4 / 4 */
      tp->P_orb = TWO_PI / Om;
      tp->t_asc = bx->t_ref + (TWO_PI * fto_uniform(seed, i, 5)) / Om;                /* xi[5] = phi_b */
    } else {
      tp->a_p = 0.0; tp->P_orb = 86400.0; tp->t_asc = bx->t_ref;
    }
    tp->f1 = bx->f1_lo + fto_uniform(seed, i, 6) * (bx->f1_hi - bx->f1_lo);
  }
}

#ifdef _OPENMP
#include <omp.h>
int fto_num_threads(void) { return omp_get_max_threads(); }
#else
int fto_num_threads(void) { return 1; }
#endif
