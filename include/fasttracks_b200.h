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
 *   post-processing  loudest candidate per parameter-space region (hyperboxes)           Sec. IV.B :330-351
 *   standardisation  z(lambda; b) = (s(lambda) - mu_G(b)) / sigma_G(b)                    Eq. (36) :346
 *   noise moments    mu_G = 2 sum w, sigma_G^2 = 4 sum w^2 (chi^2_2 scale)                Eq. (13)-(14) :130-132
 *   number-count veto  loudest power subject to a minimal weighted number count           Sec. VI.B :496-502
 *   random banks     templates drawn uniformly in xi = (f0^6/6, alpha, sin delta, a_p^3/3, Omega^4/4, phi_b)
 *                                                                                        :312-316, Eq. (A11) :602-614
 *   mismatch         m = (s(lambda) - s(lambda')) / (s(lambda) - mu_G)                    Eq. (24) :190
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
 * before returning.  A handle is not thread-safe; different handles may be driven from different host threads (the
 * process-wide tables of the library are guarded).  There is no CPU fallback: without a CUDA
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

/* FT_STAT_WHOUGH: the weighted number count sum_a w_a [P > rho_th] (:97) as the statistic (fp32 array, ranking). */
typedef enum { FT_STAT_POWER = 0, FT_STAT_HOUGH = 1, FT_STAT_BOTH = 2, FT_STAT_WHOUGH = 3 } ft_stat;
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
 *   out_power_dev [device] fp32 [n_templates] or NULL: Eq. (3) for every canonical index (FT_STAT_WHOUGH: the
 *               weighted number count sum_a w_a [P > rho_th] instead).
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
 * One candidate of ft_topk_per_box: ft_cand plus the standardised statistic of Eq. (36).
 * z = (power - mu_G) / sigma_G with the noise moments of the template's own weights on the scale of P
 * (Eq. 13-14 / footnote 2: mu_G = sum_a w_a, sigma_G^2 = sum_a w_a^2; per-bin weights: the row means of w,
 * DESIGN.md reading R21; sky-dependent weights: those of the template's sky point, mu_G = 1).
 */
typedef struct {
  double power, wcount;
  uint64_t idx;
  int32_t count;
  int32_t box;     /* region: pbox[point] * n_bands + i_f0 / bins_per_band */
  double z, sigma; /* Eq. (36); sigma_G */
} ft_cand_box;

/*
 * ft_topk_per_box — the paper's post-processing (:338-347): the parameter space is divided into disjoint
 * regions and the k loudest templates of every region are kept (the paper keeps k = 1, :476).  A region is
 * (box of outer points) x (frequency sub-band):
 *     region = pbox[point] * n_bands + i_f0 / round(band_width_hz/df0),   point = canonical idx / n_f0,
 * i.e. any partition of the outer axes (sky, a_p, P_orb, t_asc, f1 -- regular hyperboxes in the xi coordinates
 * are blocks of those axes) times the sub-bands of ft_topk_per_band.
 *   pbox_host   [host] int32 [n_points], values in [0, n_pbox), or NULL (one box: regions = sub-bands).
 *   rank_by_z   0: rank inside a region by the bound statistic (as ft_topk_per_band);
 *               1: rank by z (Eq. 36) -- with sky-dependent weights (ft_set_antenna) sigma_G differs between
 *               the sky points of a box, so the order differs from the order by power.  Needs FT_STAT_POWER/BOTH.
 *   out_host    [host] ft_cand_box [n_regions][k], padded with idx = UINT64_MAX.
 *   n_regions_out [host] receives n_pbox * n_bands.
 * Errors as ft_topk_per_band; FT_ERR_ARG for a pbox value out of range.  Synchronises the stream.
 */
int ft_topk_per_box(ft_ctx* ctx, const int32_t* pbox_host, int32_t n_pbox, double band_width_hz, int32_t k,
                    int rank_by_z, ft_cand_box* out_host, int32_t* n_regions_out);

/*
 * ft_set_antenna — sky-dependent weights (Eq. 4-5, :67-84): w_a(n) = u_a(n) w_a / sum_b u_b(n) w_b with
 * u_a(n) = a^2(t_a; n) + b^2(t_a; n), a and b the amplitude-modulation functions of the paper's ref. [20]
 * (Jaranowski, Krolak & Schutz 1998, Eq. 12-13) for perpendicular arms, and w_a the per-SFT weights given to
 * ft_create (∝ 1/S_a).  Per SFT (host arrays [n_sft], radians, copied): detector latitude, orientation
 * gamma of the arm bisector counter-clockwise from East, local sidereal angle at the SFT mid-time.
 * All three NULL: back to the weights as given.  Needs FT_W_PER_SFT weights (else FT_ERR_UNSUPPORTED) and a
 * grid the tile kernel accepts (checked at ft_eval).  Unbinds the grid.  The unstructured-bank calls
 * (ft_eval_templates, ft_eval_bank) honour the setting too: every template is weighted by the antenna pattern of
 * its own sky position (the paper's random banks, :312-316), at ~12 more fp64 operations per evaluation.
 */
int ft_set_antenna(ft_ctx* ctx, const double* det_lat_host, const double* det_gamma_host, const double* lst_host);

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
 * After ft_set_antenna the power is sum_a w_a(n) P with the sky-dependent weights of Eq. (4)-(5) of the template's n.
 * Synchronises the stream.  A track that leaves [0, n_bins) is an error, not a clamp: the call
 * returns FT_ERR_TRACK_RANGE, that template's outputs are NaN / -1 and the others are valid.
 */
int ft_eval_templates(ft_ctx* ctx, const ft_template* templates_dev, int64_t n, double t_ref, int stat,
                      double rho_th, float* out_power_dev, int32_t* out_count_dev);

/*
 * ft_eval_templates_noalloc — the computation of ft_eval_templates (same kernel K1, same canonical arithmetic,
 * same results bit for bit) as ONE self-contained call that never enters the CUDA allocator: no handle, no
 * cudaMalloc / cudaFree / cudaMallocAsync, no library routine that allocates.
 *
 * Who needs it.  Every other call of this header works on a handle, and ft_create and the handle's grow-only
 * buffers allocate device memory (ft_eval_templates itself re-allocates its ordering buffer whenever a longer
 * list arrives).  Some hosts cannot live with that:
 *   - a process that has handed the whole device to one memory pool (a framework's caching allocator, an RMM arena,
 *     a serving runtime with a fixed memory plan): a cudaMalloc made behind the pool's back fails with
 *     out-of-memory although the pool holds free blocks, or eats into the head-room the plan relies on;
 *   - a follow-up loop with a latency budget: cudaMalloc and cudaFree stall every stream of the device, not just
 *     the caller's, so one call that grows a buffer delays unrelated work on the same GPU;
 *   - code that runs after start-up in a system whose rule is "no allocation after initialisation".
 * Such a caller allocates the inputs and outputs below through whatever allocator it is allowed to use and calls
 * this function; the kernel's own work space is a fixed array inside the library.
 *
 * The work space.  K1 needs global-memory scratch beyond its inputs and outputs: the f0-ordered evaluation order
 * (one uint32 per template plus a 4096-entry histogram), the out-of-range flag and the near-tie counter.  Here
 * they live in a file-scope static __device__ array of (FT_NOALLOC_MAX_TEMPLATES + 4096) * 4 + 256 bytes
 * (4 MiB + 16.25 KiB).  It is part of the library image: every GPU on which this process uses the library holds
 * that much from the moment the module is loaded there until the process exits, whether or not this function is
 * ever called.  n > FT_NOALLOC_MAX_TEMPLATES is rejected with FT_ERR_ARG (split the bank into batches; template
 * results do not depend on the batching).
 *
 * Rules that follow from the shared array:
 *   - The FIRST call on a device looks the array's device address up (cudaGetSymbolAddress, once per device,
 *     cached) and thereby makes the CUDA runtime load the library's module on that device.  Make that first call
 *     during start-up, before any stream capture begins on the device.
 *   - All calls on a device use the same array, and it keeps what the previous call left there.  The function
 *     clears what must start at zero (histogram, flag, counter) at the beginning of every call, and the ordering
 *     is rewritten in full for the n templates of the call, so nothing stale is ever read.
 *   - Two calls in flight on one GPU at the same time would race on the array.  The function therefore holds a
 *     per-device lock from its first enqueue until its stream has drained, which serialises host threads of one
 *     process (separate processes do not interact: each has its own copy of the array).
 *
 * Arguments.  The device that is CURRENT when the function is called must be the one that owns every device
 * pointer and the stream.  All device arrays are caller-owned and only read, except the two outputs.
 *   P_dev        [device] fp32 [n_sft][ld_bins]: the spectrogram as in ft_create (any alignment, ld_bins >= n_bins).
 *   t_mid_dev    [device] fp64 [n_sft];  vel_dev [device] fp64 [n_sft][3]  (host arrays in ft_create, device arrays here).
 *   w_dev, wkind [device] FT_W_PER_SFT: fp32 [n_sft];  FT_W_PER_SFT_BIN: fp32 [n_sft][ld_bins].
 *   f_min, df    as ft_create.
 *   templates_dev [device] ft_template [n];  n in [0, FT_NOALLOC_MAX_TEMPLATES];  t_ref, stat (FT_STAT_POWER / _HOUGH /
 *                _BOTH), rho_th, out_power_dev [device] fp32 [n] or NULL, out_count_dev [device] int32 [n] or NULL:
 *                as ft_eval_templates.
 *   near_ties_host [host] or NULL: receives the number of evaluations of THIS call within 1e-9 bin of a rounding tie.
 *   cuda_stream  a cudaStream_t (NULL = default stream); the work is enqueued there and the function returns after
 *                that stream has drained.
 *   err_msg_host, err_msg_cap  [host] or NULL / 0: on a non-zero return, a NUL-terminated description of the error
 *                (there is no handle to keep one).
 * Returns FT_OK; FT_ERR_ARG (NULL / non-finite / out-of-range argument, n beyond the maximum, a pointer that is not
 * device memory of the current device); FT_ERR_CUDA; FT_ERR_TRACK_RANGE (some track leaves [0, n_bins): that
 * template's outputs are NaN / -1, the others are valid).  Sky-dependent weights (ft_set_antenna) are not available here.
 */
#define FT_NOALLOC_MAX_TEMPLATES 1048576
int ft_eval_templates_noalloc(const float* P_dev, int64_t n_sft, int64_t n_bins, int64_t ld_bins,
                              const double* t_mid_dev, const double* vel_dev, const float* w_dev, int wkind,
                              double f_min, double df, const ft_template* templates_dev, int64_t n, double t_ref,
                              int stat, double rho_th, float* out_power_dev, int32_t* out_count_dev,
                              uint64_t* near_ties_host, void* cuda_stream, char* err_msg_host, int64_t err_msg_cap);

/*
 * ft_bank_draw — a random template bank drawn uniformly in the xi coordinates of Eq. (A11) (:602-614) over a
 * box of the physical parameters ("draw n templates uniformly in xi, map them to lambda", :312-316, :627):
 *   f0 ~ f0^5, (alpha, sin delta) uniform, a_p ~ a_p^2, Omega = 2 pi / P_orb ~ Omega^3, phi_b = Omega (t_asc - t_ref)
 *   uniform in [0, 2 pi); f1 uniform (reading R22).  ap_hi == 0 draws an isolated bank (a_p = 0).
 * Template i of stream `seed` is a pure function of (seed, i): u(seed, i, d) = splitmix64 finaliser of
 * seed + 0x9E3779B97F4A7C15 (8 i + d + 1), top 53 bits; so banks can be drawn in batches of any size.
 *   out_dev [device] ft_template [n]: templates first .. first + n - 1.  Asynchronous on the handle's stream.
 */
typedef struct {
  double f0_lo, f0_hi, f1_lo, f1_hi, ra_lo, ra_hi, sd_lo, sd_hi, ap_lo, ap_hi, porb_lo, porb_hi, t_ref;
} ft_bank_box;
int ft_bank_draw(ft_ctx* ctx, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, ft_template* out_dev);

/*
 * ft_eval_bank — draw (ft_bank_draw) AND evaluate templates first .. first + n - 1 of a xi-uniform bank in one
 * call (the paper's benchmark counts "generating random templates, computing the frequency indices,
 * gathering, reducing", :228): the templates are generated in registers and never stored.  Returns the
 * loudest template of the batch under (statistic desc, index asc) -- the per-box loudest of :476 -- re-evaluated
 * in fp64, and optionally every statistic.
 *   stat: FT_STAT_POWER or FT_STAT_HOUGH (ranking value).  out_power_dev / out_count_dev as ft_eval_templates, or NULL.
 *   best_host [host] ft_cand (idx = position in the stream; band = -1) and best_template_host [host] ft_template, or NULL.
 * Synchronises the stream.
 */
int ft_eval_bank(ft_ctx* ctx, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, int stat,
                 double rho_th, float* out_power_dev, int32_t* out_count_dev, ft_cand* best_host,
                 ft_template* best_template_host);

/*
 * ft_eval_bank_veto — the paper's per-box step on a random bank, end to end (:476 "retrieve the loudest template per
 * box"; :496-502 "the loudest normalized power ... subject to a minimal weighted number count"; Eq. 36 :346): draw
 * and evaluate templates first .. first + n - 1 of the xi-uniform bank as ft_eval_bank does, with BOTH statistics
 * from one gather, and return the template with the largest z (rank_by_z != 0) or normalized power among those whose
 * weighted number count sum_a w_a [P > rho_th] is >= wcount_floor (0 = no veto); ties to the lower position.
 * With sky-dependent weights (ft_set_antenna) every template carries the weights, mu_G = 1 and sigma_G of its own
 * sky position, so the order by z differs from the order by power.
 *   out_power_dev / out_count_dev  [device] fp32 / int32 [n] or NULL: every statistic, as ft_eval_bank.
 *   best_host [host] ft_cand_box or NULL: the winner re-evaluated in fp64 (power, wcount, count, z, sigma; idx =
 *             position in the stream; box = -1).  idx = UINT64_MAX if the veto leaves no template (FT_OK).
 *   best_template_host [host] ft_template or NULL (untouched when there is no winner).
 * The veto and the ranking use the kernel's fp64 sums (for fixed weights the same bits as the plain definition; with
 * sky-dependent weights within ~1e-15 of it).  Synchronises the stream.
 */
int ft_eval_bank_veto(ft_ctx* ctx, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, double rho_th,
                      double wcount_floor, int rank_by_z, float* out_power_dev, int32_t* out_count_dev,
                      ft_cand_box* best_host, ft_template* best_template_host);

/*
 * ft_track — the track of ONE explicit template: bin k_a (Eq. 2 rounded to the bin grid, :248) for every SFT.
 *   template_host [host]; k_out_host [host] int64 [n_sft].  For building injections (a "data stream containing a
 *   CW signal", :322) without leaving the library.  Synchronises.  FT_ERR_TRACK_RANGE if a bin is outside.
 */
int ft_track(ft_ctx* ctx, const ft_template* template_host, double t_ref, int64_t* k_out_host);

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
  FT_OPT_ONE_PASS_BOTH = 7, /* 1 (default): narrow bands compute both statistics in one gather (hit bit in the LSB of
                               the folded pixel); 0: one pass per statistic */
  FT_OPT_WCOUNT_FLOOR = 8,  /* ft_set_option_f64: 0 off (default); x > 0: with FT_STAT_BOTH bound, the selection keeps the
                               loudest normalized power among templates whose WEIGHTED number count sum_a w_a [P > rho_th]
                               is >= x -- the veto as the paper states it (:496-502; "three standard deviations above
                               the average number count in Gaussian noise": x = p sum w + 3 sqrt(p (1 - p) sum w^2),
                               p = exp(-rho_th)).  Costs one weighted-count pass over the bank. */
  FT_OPT_VETO_FIRST = 9,    /* 1 (default): with a floor set, the number-count pass runs first with the floor as its fused
                               filter; if its survivors fit the candidate buffers (a floor of mu + 3 sigma leaves ~1e-3 of a
                               noise bank) only they are evaluated for power and the bank-wide power pass is skipped.
                               0: always both bank-wide passes.  Same candidates either way. */
  FT_OPT_TAIL_PACKING = 10  /* 1 (default): a narrow band whose f0 count is 32 m + t with 1 <= t <= 16 runs two outer points
                               per warp, their t-wide tails sharing one load (fewer shared-memory wavefronts); 0: one
                               point per warp.  Same results bit for bit. */
} ft_option;
int ft_set_option(ft_ctx* ctx, int option, int64_t value);
int ft_set_option_f64(ft_ctx* ctx, int option, double value);

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

/*
 * ft_measure_peaks — micro-benchmarks of the units that bound the kernels of this library, on the handle's
 * device and stream (the roofline denominators MEASURED_PEAKS.json does not hold):
 *   smem_gbs       shared-memory read bandwidth, conflict-free LDS.32 from every SM (the bound of the tile kernel)
 *   fp64_gflops    DFMA throughput x 2 (the bound of the per-evaluation track arithmetic, kernel K1)
 *   fp64_cvt_gops  F2I.F64 + I2F.F64 pairs per second (conversions share the fp64 pipe at a lower rate)
 *   l2_gbs         read bandwidth of a 32 MiB buffer resident in L2
 *   sm_clock_mhz   SM clock during the shared-memory run (cycles counted on the device / event time)
 * Synchronises the stream.
 */
typedef struct { double smem_gbs, fp64_gflops, fp64_cvt_gops, l2_gbs, sm_clock_mhz; } ft_peaks;
int ft_measure_peaks(ft_ctx* ctx, ft_peaks* out);

/*
 * ft_selftest — device-side checks of arithmetic identities the kernels rely on; *n_fail_out receives the
 * number of failures among n random cases of stream `seed`.
 *   which = 0: the unstructured-bank kernel divides v.n by c with a reciprocal multiply and one fused
 *              correction; every quotient must equal the IEEE division __ddiv_rn(dot, c) bit for bit (up to the sign of a zero)
 *              (dot drawn over the range of |v.n| <= 5e4 m/s, every binade from 2^-300 to 2^300, exact multiples of c, +-0).
 *   which = 1: the integer-arithmetic fp32 -> fp64 conversion of K1 equals (double)x for every finite input.
 *   which = 2: K1's orbital cosine (magic-number range reduction by pi, Taylor series) is within 4e-16 of cos(x)
 *              for |x| up to 1e8 rad (so the track moves by < 1e-14 bin).
 */
int ft_selftest(ft_ctx* ctx, int which, int64_t n, uint64_t seed, uint64_t* n_fail_out);

const char* ft_last_error(const ft_ctx* ctx); /* never NULL; valid until the next call on ctx */
/* Which kernel the bound grid runs and its launch geometry (diagnostics; never NULL; valid until the next ft_eval). */
const char* ft_describe(const ft_ctx* ctx);
void ft_destroy(ft_ctx* ctx);                 /* synchronises the stream, frees library-owned memory */

#ifdef __cplusplus
}
#endif
#endif /* FASTTRACKS_B200_H */
