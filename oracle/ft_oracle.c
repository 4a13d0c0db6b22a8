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
 * linearity and permutation invariance, pure-Python brute force on tiny inputs.
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

/* One explicit template lambda = (f0, f1, n, a_p, P_orb, t_asc): "no assumption on the properties of
 * lambda"; random template banks are drawn this way. */
typedef struct { double f0, f1, nx, ny, nz, a_p, P_orb, t_asc; } fto_template;

/*
 * One template: track -> bin per SFT (Eq. 2), then the statistics (Eq. 3, Eq. 7).
 * k_out / x_out may be NULL.  Returns FTO_ERR_RANGE if any bin falls outside the spectrogram.
 */
static int fto_one_params(const fto_problem* pb, const fto_template* tp, double t_ref, double* power,
                          int32_t* count, double* wcount, uint8_t* near_tie, int64_t* k_out,
                          double* x_out) {
  const double inv_df = 1.0 / pb->df;
  const double f0 = tp->f0, f1 = tp->f1;
  const double nx = tp->nx, ny = tp->ny, nz = tp->nz;
  const double a_p = tp->a_p;
  const double Om = TWO_PI / tp->P_orb;          /* Omega */
  const double t_asc = tp->t_asc;                /* phi_b = t_asc * Omega */
  const float rho = (float)pb->rho_th;

  double s_power = 0.0, s_wcount = 0.0;
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
    const float w = (pb->wkind == 2) ? pb->w[a * pb->ld + k] : pb->w[a];
    s_power += (double)w * (double)p;                             /* Eq. 3 */
    if (p > rho) {                                                /* Eq. 7, strict > in fp32 */
      s_count += 1;
      s_wcount += (double)w;                                      /* weighted count */
    }
  }
  if (power) *power = s_power;
  if (count) *count = s_count;
  if (wcount) *wcount = s_wcount;
  if (near_tie) *near_tie = tie;
  return FTO_OK;
}

/* Grid template: canonical index -> parameters (f0 = f0_start + i df0, ..., t_asc = t_ref + u P_orb). */
static int fto_one_template(const fto_problem* pb, uint64_t idx, double* power, int32_t* count,
                            double* wcount, uint8_t* near_tie, int64_t* k_out, double* x_out) {
  int64_t ax[6];
  fto_unravel(pb, idx, ax);
  fto_template tp;
  tp.f0 = pb->f0_start + (double)ax[5] * pb->df0;
  tp.f1 = pb->f1_start + (double)ax[4] * pb->df1;
  tp.nx = pb->sky[3 * ax[0] + 0]; tp.ny = pb->sky[3 * ax[0] + 1]; tp.nz = pb->sky[3 * ax[0] + 2];
  tp.a_p = pb->a_p[ax[1]];
  tp.P_orb = pb->P_orb[ax[2]];
  tp.t_asc = pb->t_ref + pb->tasc_frac[ax[3]] * tp.P_orb;
  return fto_one_params(pb, &tp, pb->t_ref, power, count, wcount, near_tie, k_out, x_out);
}

/* Track of ONE template: bins k[n_sft] and positions x[n_sft]. */
int fto_track(const fto_problem* pb, uint64_t idx, int64_t* k_out, double* x_out) {
  return fto_one_template(pb, idx, NULL, NULL, NULL, NULL, k_out, x_out);
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
                                    near_tie ? near_tie + j : NULL, NULL, NULL);
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
                                    NULL, NULL);
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
                                  wcount ? wcount + j : NULL, near_tie ? near_tie + j : NULL, NULL, NULL);
    if (rc != FTO_OK) {
#pragma omp atomic write
      status = rc;
    }
  }
  return status;
}

#ifdef _OPENMP
#include <omp.h>
int fto_num_threads(void) { return omp_get_max_threads(); }
#else
int fto_num_threads(void) { return 1; }
#endif
