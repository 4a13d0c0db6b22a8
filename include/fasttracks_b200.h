/*
 * fasttracks_b200.h — C ABI of the B200-native hot path of arXiv:2411.18370's `fasttracks` engine:
 * brute-force evaluation of short-coherence, track-based detection statistics over a template
 * grid, and the per-frequency-sub-band loudest-candidate (top-k) reduction.
 *
 * Paper passages (line numbers of /root/reference/PAPER.md):
 *   track            f(t;lambda) = f0 [1 + v(t).n/c - a_p Omega cos(Omega t - phi_b)]   Eq. (2)  :53
 *   statistic        s(lambda) = sum_{X,alpha} w_{X alpha} s[t_{X alpha}; f(t_{X alpha};lambda)] Eq. (3) :64
 *   weights          w ∝ (a^2+b^2)/S_n, sum w = 1                                      Eq. (4)-(5) :69, :84
 *   spectrogram      s[t;f] = 4 |x~|^2 / (T_SFT S_n)                                    Eq. (6)  :88
 *   number count     nc = 1 if s > 3.2 else 0; weighted count "akin to Eq. (3)"         Eq. (7)  :95-97
 *   batching         vmap s : {lambda_i} -> {s(lambda_i)}                                Sec. III :213
 *   post-processing  loudest candidate per parameter-space region                        Sec. IV.B :330-351
 * Extensions fixed by BASELINE.json north_star: spindown f1 with reference time t_ref, SFT
 * mid-times, regions = frequency sub-bands, loudest -> top-k.  DESIGN.md lists every reading.
 *
 * Canonical arithmetic (IEEE binary64, round-to-nearest-even,
 * no fused multiply-add), per template and per SFT alpha in ascending row order:
 *     dt = t_mid[a] - t_ref;            fs = f0 + f1*dt
 *     V  = ((vx*nx + vy*ny) + vz*nz)/c; B = (a_p*Om)*cos(Om*(t_mid[a] - t_asc))   (B = 0 if a_p == 0)
 *     D  = (1 + V) - B;                 x = ((fs*D) - f_min)*(1/df);   k = rint(x)  (half-to-even)
 *     power += (double)w*(double)P[a][k];   count += (P[a][k] > (float)rho_th)
 * with f0 = f0_start + i*df0, f1 = f1_start + j*df1, Om = 2pi/P_orb, t_asc = t_ref + u*P_orb.
 *
 * Conventions.  Every call returns an ft_status (0 = OK, negative = error); nothing throws or
 * aborts across this boundary; ft_last_error() gives a handle-owned message.  "device" pointers
 * are CUDA device memory owned by the caller (PyTorch allocates them in the harness) and are
 * BORROWED until ft_destroy (inputs) or until the call's work has completed on the stream
 * (outputs).  "host" pointers are read during the call and copied.  All device work is enqueued
 * on the CUDA stream given to ft_create; calls that write host memory synchronise that stream
 * before returning.  A handle is not thread-safe.  There is no CPU fallback: without a CUDA
 * device ft_create fails with FT_ERR_CUDA.
 */
#ifndef FASTTRACKS_B200_H
#define FASTTRACKS_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ft_ctx ft_ctx; /* opaque handle */

typedef enum {
  FT_OK = 0,
  FT_ERR_ARG = -1,         /* NULL / non-finite / non-positive argument, bad enum */
  FT_ERR_ALLOC = -2,       /* host or device allocation failed */
  FT_ERR_CUDA = -3,        /* CUDA runtime error (message in ft_last_error) */
  FT_ERR_TRACK_RANGE = -4, /* some track of the grid could leave [0, n_bins): rejected, not clamped */
  FT_ERR_BAND = -5,        /* band_width is not an integer number of f0 steps */
  FT_ERR_STATE = -6,       /* no grid bound / candidate buffers overflowed by exact ties */
  FT_ERR_UNSUPPORTED = -7  /* option combination the selected kernel cannot run */
} ft_status;

typedef enum { FT_STAT_POWER = 0, FT_STAT_HOUGH = 1, FT_STAT_BOTH = 2 } ft_stat;
typedef enum { FT_W_PER_SFT = 1, FT_W_PER_SFT_BIN = 2 } ft_wkind;

/*
 * ft_create — bind the normalized spectrogram (Eq. 6, on the Exponential(1) scale P = s/2,
 * footnote 2 :141) and the per-SFT tables (SFT data model :60; detectors concatenated along alpha).
 *   out         [host]   receives the handle.
 *   P_dev       [device] fp32 [n_sft][ld_bins], row alpha = one SFT, column k = frequency bin centred
 *                        at f_min + k*df; borrowed until ft_destroy; must be 16-byte aligned and
 *                        ld_bins a multiple of 4 (TMA bulk copies) else FT_ERR_ARG.
 *   t_mid_host  [host]   fp64 [n_sft] SFT mid-times in seconds (copied).
 *   vel_host    [host]   fp64 [n_sft][3] detector velocity in m/s, equatorial Cartesian (copied).
 *   w, wkind             FT_W_PER_SFT: [host] fp32 [n_sft] (copied);
 *                        FT_W_PER_SFT_BIN: [device] fp32 [n_sft][ld_bins] (borrowed).  Weights are
 *                        used as given (Eq. 4-5 are the caller's; no renormalisation).
 *   f_min, df            frequency of bin 0 and bin width (= 1/T_SFT, :248), Hz; df > 0.
 *   cuda_stream          a cudaStream_t (NULL = default stream); all work of the handle runs on it.
 * ft_create also builds the library-owned gather array Q[a][k] = fl(fl(w P) - c_a), c_a the row mean
 * (one pass over P on the stream), and synchronises the stream.
 */
int ft_create(ft_ctx** out, const float* P_dev, int64_t n_sft, int64_t n_bins, int64_t ld_bins,
              const double* t_mid_host, const double* vel_host, const float* w, int wkind,
              double f_min, double df, void* cuda_stream);

/*
 * Template grid (a product grid; all axis arrays are host arrays, copied by ft_eval).
 * Canonical linear template index (uint64), f0 fastest:
 *   idx = (((((i_sky*n_ap + i_ap)*n_porb + i_porb)*n_tasc + i_tasc)*n_f1 + i_f1)*n_f0 + i_f0
 */
typedef struct {
  double f0_start, df0; int64_t n_f0;       /* f0_i = f0_start + (double)i*df0, Hz             */
  double f1_start, df1; int32_t n_f1;       /* f1_j = f1_start + (double)j*df1, Hz/s           */
  double t_ref;                              /* reference time of f0 and f1, s                  */
  int64_t n_sky;  const double* sky;         /* [n_sky][3] unit vectors n, equatorial Cartesian */
  int32_t n_ap;   const double* a_p;         /* projected semi-major axis, light-seconds; {0} = isolated (:56) */
  int32_t n_porb; const double* P_orb;       /* orbital period, s (Omega = 2 pi / P_orb)        */
  int32_t n_tasc; const double* tasc_frac;   /* u in [0,1): t_asc = t_ref + u*P_orb (phi_b = t_asc*Omega, :56) */
} ft_grid;

/*
 * ft_eval — bind a template grid and (optionally) evaluate the statistic of EVERY template
 * (vmap s, :213).
 *   stat        ft_stat.  rho_th: number-count threshold on the scale of P (1.6 <-> the paper's
 *               3.2, Eq. 7), compared in fp32 with strict '>'.
 *   out_power_dev [device] fp32 [n_templates] or NULL: Eq. (3) for every canonical index.
 *   out_count_dev [device] int32 [n_templates] or NULL: Eq. (7) summed along the track (integer).
 *   Both NULL: bind the grid only (for ft_topk_per_band); no statistic kernel is launched.
 * Validation before any launch: finite arguments, positive sizes, and a conservative bound on
 * every track of the grid must stay inside [0, n_bins) else FT_ERR_TRACK_RANGE (so kernels need
 * no per-evaluation bounds check).  Kernel choice: the tile kernel (TMA-staged strips, fp32 accumulation
 * of the folded, row-centred array Q = w P - c_row, bins bit-identical to the canonical arithmetic except
 * within 1e-9 bin of a rounding tie; number count on a packed byte hit map, exact) when df0 == df;
 * otherwise the generic kernel (canonical arithmetic per evaluation, fp64 accumulation).  Asynchronous
 * on the handle's stream.
 */
int ft_eval(ft_ctx* ctx, const ft_grid* grid, int stat, double rho_th, float* out_power_dev,
            int32_t* out_count_dev);

/* One candidate.  power / wcount are re-evaluated in fp64 in the canonical order (bit-identical
 * to the plain definition); count is the integer number count; idx the canonical index. */
typedef struct {
  double power;   /* Eq. (3) */
  double wcount;  /* sum_alpha w_alpha [P > rho_th]  (:97) */
  uint64_t idx;
  int32_t count;  /* Eq. (7) summed */
  int32_t band;   /* i_f0 / bins_per_band */
} ft_cand;

/*
 * ft_topk_per_band — evaluate the bound grid and keep, for every frequency sub-band
 * b = i_f0 / round(band_width_hz/df0), the k loudest templates under the total order
 * (ranking value descending, canonical index ascending).  Ranking value: power for
 * FT_STAT_POWER / FT_STAT_BOTH, integer count for FT_STAT_HOUGH.  The selection is fused into
 * the evaluation kernel (the full statistic array is never written); survivors of the fp32
 * selection (a superset) are re-evaluated in fp64 before the final ranking.
 *   out_host    [host] ft_cand [n_bands][k]; bands with fewer than k templates are padded with
 *               idx = UINT64_MAX.   n_bands_out [host] receives n_bands = ceil(n_f0/bins_per_band).
 * Errors: FT_ERR_STATE if no grid is bound; FT_ERR_BAND if band_width_hz/df0 is not an integer
 * within 1e-9 or k < 1.  Synchronises the stream.
 */
int ft_topk_per_band(ft_ctx* ctx, double band_width_hz, int32_t k, ft_cand* out_host,
                     int32_t* n_bands_out);

/*
 * ft_eval_list — canonical fp64 evaluation of an explicit list of templates of the bound grid
 * (the refinement step of the selection, exposed for spot checks of full-size runs).
 *   idx_host [host] uint64 [n]; out_host [host] ft_cand [n] (band = -1).  Synchronises.
 */
int ft_eval_list(ft_ctx* ctx, const uint64_t* idx_host, int64_t n, ft_cand* out_host);

/*
 * One explicit template lambda = (f0, f1, n, a_p, P_orb, t_asc): the unstructured-bank form of the
 * problem ("no assumption on the properties of lambda", :213; random template banks :312-316).
 */
typedef struct {
  double f0, f1;        /* Hz at t_ref, Hz/s                                   */
  double nx, ny, nz;    /* unit vector n, equatorial Cartesian                 */
  double a_p, P_orb;    /* light-seconds (0 = isolated), seconds (> 0 always)  */
  double t_asc;         /* time of ascending node, seconds (absolute, not a fraction) */
} ft_template;

/*
 * ft_eval_templates — statistic of every template of an explicit list (vmap s over an arbitrary
 * bank, :213), by the canonical fp64 arithmetic per (template, SFT): kernel K1, bound by the fp64
 * pipe.  Needs no bound grid and does not disturb one.
 *   templates_dev [device] ft_template [n], borrowed until the call returns.
 *   t_ref         reference time of f0 / f1, seconds.
 *   stat, rho_th  as ft_eval.   out_power_dev [device] fp32 [n] or NULL; out_count_dev [device] int32 [n] or NULL.
 * Synchronises the stream.  A track that leaves [0, n_bins) is an error, not a clamp: the call
 * returns FT_ERR_TRACK_RANGE, that template's outputs are NaN / -1 and the others are valid.
 */
int ft_eval_templates(ft_ctx* ctx, const ft_template* templates_dev, int64_t n, double t_ref, int stat,
                      double rho_th, float* out_power_dev, int32_t* out_count_dev);

/* Options (ft_set_option): */
typedef enum {
  FT_OPT_KERNEL = 0,        /* 0 auto (default), 1 force generic kernel, 2 force tile kernel (FT_ERR_UNSUPPORTED if ineligible) */
  FT_OPT_FUSED_TOPK = 1,    /* 1 (default) fused selection; 0 full write-out to scratch then select */
  FT_OPT_POINTS_PER_CTA = 2, /* 0 auto; else number of outer points a CTA shares one staged strip among */
  FT_OPT_PACKED_COUNT = 3,  /* 1 (default) number count on the packed byte hit map when n_sft <= 65535; 0 fp32 0/1 map */
  FT_OPT_F0_TILES = 4,      /* 0 auto; else split the f0 axis into exactly this many tiles (tuning / tests) */
  FT_OPT_SELECT_CAP = 5,    /* 0 auto; else entries per band of the fused selection's append buffers (tests of the
                               overflow recovery: a band that overflows tightens its threshold and the pass repeats) */
  FT_OPT_COUNT_FLOOR = 6,   /* 0 off (default); n > 0: with FT_STAT_BOTH bound, ft_topk_per_band keeps the loudest
                               normalized power among templates whose integer number count is >= n (the number-count
                               veto of :496-502; for uniform weights the paper's weighted-count floor times n_sft) */
  FT_OPT_ONE_PASS_BOTH = 7  /* 1 (default): narrow bands compute both statistics in one gather (hit bit in the LSB of
                               the folded pixel); 0: one pass per statistic */
} ft_option;
int ft_set_option(ft_ctx* ctx, int option, int64_t value);

typedef struct {
  uint64_t near_ties;        /* canonical track evaluations that fell within 1e-9 bin of a rounding tie, since ft_create */
  uint64_t refine_fallbacks; /* selections that had to be redone with a tighter threshold */
  uint64_t appended;         /* candidates that passed the fused fp32 filter (last top-k call) */
  uint64_t refined;          /* candidates re-evaluated in fp64 (last top-k call) */
  uint64_t kernel_launches;  /* CUDA kernels launched by this handle since ft_create */
  uint64_t stat_launches;    /* statistic-kernel launches (K0/K2) of the last ft_eval / ft_topk_per_band call */
  double last_kernel_ms;     /* summed device time of those launches (CUDA events on the handle's stream) */
} ft_counters;
int ft_get_counters(ft_ctx* ctx, ft_counters* out);

const char* ft_last_error(const ft_ctx* ctx); /* never NULL; valid until the next call on ctx */
/* Which kernel the bound grid runs and its launch geometry (diagnostics; never NULL; valid until the next ft_eval). */
const char* ft_describe(const ft_ctx* ctx);
void ft_destroy(ft_ctx* ctx);                 /* synchronises the stream, frees library-owned memory */

#ifdef __cplusplus
}
#endif
#endif /* FASTTRACKS_B200_H */
