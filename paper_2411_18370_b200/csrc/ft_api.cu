// C ABI of libfasttracks_b200 (include/fasttracks_b200.h): handle, validation, binding a grid, evaluation.
// The selection calls (ft_topk_per_band, ft_topk_per_box) are in ft_topk.cu, the unstructured-bank calls in ft_list.cu.
#include <algorithm>
#include <new>

#include "ft_ctx.cuh"

int ft_fail(ft_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}

void ft_tick(ft_ctx* c) {
  if (c->ev_used + 2 > c->evs.size()) {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    c->evs.push_back(e0); c->evs.push_back(e1);
  }
  cudaEventRecord(c->evs[c->ev_used], c->stream);
}
void ft_tock(ft_ctx* c, int launches) {
  cudaEventRecord(c->evs[c->ev_used + 1], c->stream);
  c->ev_used += 2;
  c->counters.stat_launches += (uint64_t)launches;
  c->counters.kernel_launches += (uint64_t)launches;
}

int ft_enter(ft_ctx* c) {
  int dev = -1;
  if (cudaGetDevice(&dev) == cudaSuccess && dev == c->device) return FT_OK;
  FT_CUDA(c, cudaSetDevice(c->device));
  return FT_OK;
}

int ft_tile_err_status(ft_ctx* c, int32_t e) {
  if (e == 0) return FT_OK;
  cudaMemsetAsync(c->tile_err_dev, 0, sizeof e, c->stream);
  return ft_fail(c, FT_ERR_STATE, e == 1 ? "tile kernel: a track left its staged strip (internal planning error); the outputs of the previous evaluation are invalid"
                                         : "tile kernel: more than one break in a warp range (internal planning error); the outputs of the previous evaluation are invalid");
}

int ft_check_tile_err(ft_ctx* c) {
  if (!c->tile_err_dev) return FT_OK;
  int32_t e = 0;
  FT_CUDA(c, cudaMemcpyAsync(&e, c->tile_err_dev, sizeof e, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  return ft_tile_err_status(c, e);
}

namespace {

bool finite_all(const double* p, size_t n) {
  for (size_t i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return false;
  return true;
}

// One gather-reduce pass of a tile plan over array A.
int tile_pass(ft_ctx* c, const FtTilePlan& plan, const FtPass& p, const float* A, double add_back, const float* c_row,
              float* out_f, int32_t* out_i, bool filter, int zmode) {
  FtTileRun run;
  run.A = A; run.add_back = add_back; run.c_row = c_row;
  run.out_f = out_f; run.out_i = out_i; run.out_base = p.out_base;
  run.sel = filter ? &c->sel : nullptr;
  run.bpb = p.bpb; run.pbox = p.pbox; run.n_bands = p.n_bands;
  run.zmode = zmode; run.out_key = zmode ? p.out_key : 0;
  run.z_mu = c->d.mu_G; run.z_inv_sigma = c->d.sigma_G > 0.0 ? 1.0 / c->d.sigma_G : 1.0;
  run.near_ties = c->near_ties_dev;
  run.sky_norm = c->skyn_dev; run.norm_cb = (A == c->WH_dev) ? 3 : 2;
  run.skip_host = p.skip_host; run.n_skip_host = p.n_skip_host;
  int launches = 0;
  ft_tick(c);
  const cudaError_t e = ft_launch_tile(c->d, plan, run, p.pt_begin, p.pt_end, c->stream, &launches, p.glist, p.n_glist, p.gskip);
  ft_tock(c, launches);
  if (e != cudaSuccess) return ft_fail(c, FT_ERR_CUDA, std::string("tile kernel launch: ") + cudaGetErrorString(e));
  return FT_OK;
}

}  // namespace

// Statistic over points [pt_begin, pt_end) (or the sampled / remaining CTA groups): full write-out and/or fused
// filter into c->sel.  Chooses the tile or the generic kernel.  One gather-reduce pass per statistic: power over
// Q, weighted count over the folded w x hit map, number count over the hit map; both statistics from one pass
// over QB on narrow bands.
int ft_run_stat(ft_ctx* c, const FtPass& p) {
  const bool use_tile = c->tile_ok && c->opt_kernel != 1;
  const int stat = p.stat;
  if (!use_tile) {
    if (p.filter || p.glist || p.gskip) return ft_fail(c, FT_ERR_UNSUPPORTED, "fused filter needs the tile kernel");
    if (c->d.skyw) return ft_fail(c, FT_ERR_UNSUPPORTED, "sky-dependent weights need the tile kernel");
    ft_tick(c);
    FT_CUDA(c, ft_launch_generic(c->d, stat, p.pt_begin, p.pt_end, p.out_f, p.out_i, p.out_base, c->stream));
    ft_tock(c, 1);
    if (p.zmode && p.out_key && p.out_f) {
      FT_CUDA(c, ft_keys_affine(p.out_f, (int64_t)(p.pt_end - p.pt_begin) * c->d.n_f0, c->d.mu_G, 1.0 / c->d.sigma_G, c->stream));
      c->counters.kernel_launches += 1;
    }
    return FT_OK;
  }
  const bool skyw = c->d.skyw != 0;
  const FtTilePlan& fplan = skyw ? c->planw : c->plan;   // the fp32 gather of this binding
  if (stat == FT_STAT_BOTH && c->tileb_ok && !skyw && ((p.out_f && p.out_i) || p.filter))
    // narrow bands: both statistics (and the count veto of the fused filter) from one gather
    return tile_pass(c, c->planb, p, c->QB_dev, c->add_back, nullptr, p.out_f, p.out_i, p.filter, p.zmode);
  if ((stat == FT_STAT_POWER || stat == FT_STAT_BOTH) && (p.out_f || p.filter)) {
    const int rc = tile_pass(c, fplan, p, c->Q_dev, c->add_back, c->cQ_dev, p.out_f, nullptr, p.filter, p.zmode);
    if (rc != FT_OK) return rc;
  }
  if (stat == FT_STAT_WHOUGH && (p.out_f || p.filter)) {
    const int rc = tile_pass(c, fplan, p, c->WH_dev, c->add_back_wh, c->cWH_dev, p.out_f, nullptr, p.filter, 0);
    if (rc != FT_OK) return rc;
  }
  if (stat != FT_STAT_POWER && (p.out_i || (p.filter && stat == FT_STAT_HOUGH))) {
    const bool fil = p.filter && stat == FT_STAT_HOUGH;
    const int rc = tile_pass(c, c->tile8_ok ? c->plan8 : c->plan, p, c->H_dev, 0.0, nullptr,
                             stat == FT_STAT_HOUGH ? p.out_f : nullptr, p.out_i, fil, 0);
    if (rc != FT_OK) return rc;
  }
  return FT_OK;
}

extern "C" {

int ft_create(ft_ctx** out, const float* P_dev, int64_t n_sft, int64_t n_bins, int64_t ld_bins,
              const double* t_mid_host, const double* vel_host, const float* w, int wkind,
              double f_min, double df, void* cuda_stream) {
  if (!out) return FT_ERR_ARG;
  *out = nullptr;
  ft_ctx* c = new (std::nothrow) ft_ctx();
  if (!c) return FT_ERR_ALLOC;
  *out = c;  // returned even on error so ft_last_error can be read; caller still calls ft_destroy
  if (!P_dev || !t_mid_host || !vel_host || !w) return ft_fail(c, FT_ERR_ARG, "ft_create: NULL pointer argument");
  if (n_sft < 1 || n_bins < 1 || ld_bins < n_bins) return ft_fail(c, FT_ERR_ARG, "ft_create: need n_sft >= 1, 1 <= n_bins <= ld_bins");
  if (n_sft > (1 << 24)) return ft_fail(c, FT_ERR_ARG, "ft_create: n_sft > 2^24 (integer counts are selected as exact fp32 keys)");
  if ((ld_bins & 3) || (reinterpret_cast<uintptr_t>(P_dev) & 15)) return ft_fail(c, FT_ERR_ARG, "ft_create: P must be 16-byte aligned with ld_bins a multiple of 4");
  if (wkind != FT_W_PER_SFT && wkind != FT_W_PER_SFT_BIN) return ft_fail(c, FT_ERR_ARG, "ft_create: bad wkind");
  if (!(df > 0.0) || !std::isfinite(df) || !std::isfinite(f_min)) return ft_fail(c, FT_ERR_ARG, "ft_create: need finite f_min and df > 0");
  if (!finite_all(t_mid_host, (size_t)n_sft) || !finite_all(vel_host, (size_t)n_sft * 3)) return ft_fail(c, FT_ERR_ARG, "ft_create: non-finite t_mid / vel");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return ft_fail(c, FT_ERR_CUDA, "ft_create: no CUDA device (this library has no CPU fallback)");
  {
    cudaPointerAttributes attr{};
    if (cudaPointerGetAttributes(&attr, P_dev) == cudaSuccess && attr.type == cudaMemoryTypeDevice) c->device = attr.device;
    else FT_CUDA(c, cudaGetDevice(&c->device));
    cudaGetLastError();
    FT_CUDA(c, cudaSetDevice(c->device));
  }
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->t_mid.assign(t_mid_host, t_mid_host + n_sft);
  c->vel.assign(vel_host, vel_host + 3 * n_sft);
  for (int64_t a = 0; a < n_sft; ++a) {
    const double* v = vel_host + 3 * a;
    c->vmax = std::fmax(c->vmax, std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
  }
  FT_CUDA(c, cudaMalloc(&c->t_mid_dev, sizeof(double) * n_sft));
  FT_CUDA(c, cudaMalloc(&c->vel_dev, sizeof(double) * 3 * n_sft));
  FT_CUDA(c, cudaMemcpyAsync(c->t_mid_dev, t_mid_host, sizeof(double) * n_sft, cudaMemcpyHostToDevice, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(c->vel_dev, vel_host, sizeof(double) * 3 * n_sft, cudaMemcpyHostToDevice, c->stream));
  FT_CUDA(c, cudaMalloc(&c->near_ties_dev, sizeof(unsigned long long)));
  FT_CUDA(c, cudaMemsetAsync(c->near_ties_dev, 0, sizeof(unsigned long long), c->stream));
  FT_CUDA(c, cudaMalloc(&c->flag_dev, sizeof(int32_t)));
  FT_CUDA(c, cudaMalloc(&c->tile_err_dev, sizeof(int32_t)));
  FT_CUDA(c, cudaMemsetAsync(c->tile_err_dev, 0, sizeof(int32_t), c->stream));
  c->plan.err = c->plan8.err = c->planb.err = c->planw.err = c->tile_err_dev;
  FT_CUDA(c, cudaMalloc(&c->vr_dev, sizeof(double) * 2 * n_sft));
  FT_CUDA(c, cudaMalloc(&c->maxw_dev, sizeof(int32_t) * 4));
  FtDev& d = c->d;
  d.P = P_dev; d.n_sft = n_sft; d.n_bins = n_bins; d.ld = ld_bins;
  d.t_mid = c->t_mid_dev; d.vel = c->vel_dev;
  d.wkind = wkind; d.f_min = f_min; d.inv_df = 1.0 / df;
  c->df = df;
  c->per_bin = (wkind == FT_W_PER_SFT_BIN);
  // A0: Q = fl(fl(w P) - c_row) (the fp64 refinement uses w and P unfolded); add_back = sum c_row
  FT_CUDA(c, cudaMalloc(&c->Q_dev, sizeof(float) * (size_t)n_sft * ld_bins));
  FT_CUDA(c, cudaMalloc(&c->cQ_dev, sizeof(float) * n_sft));
  if (!c->per_bin) {
    FT_CUDA(c, cudaMalloc(&c->w_dev, sizeof(float) * n_sft));
    FT_CUDA(c, cudaMemcpyAsync(c->w_dev, w, sizeof(float) * n_sft, cudaMemcpyHostToDevice, c->stream));
    d.w = c->w_dev;
  } else {
    if (reinterpret_cast<uintptr_t>(w) & 15) return ft_fail(c, FT_ERR_ARG, "ft_create: per-bin weights must be 16-byte aligned");
    d.w = w;
    FT_CUDA(c, cudaMalloc(&c->w_row_dev, sizeof(double) * n_sft));
  }
  {
    cudaError_t e = ft_launch_fold_centered(P_dev, c->per_bin ? nullptr : c->w_dev, c->per_bin ? w : nullptr,
                                            c->Q_dev, c->cQ_dev, c->w_row_dev, n_sft, n_bins, ld_bins, 0, 0.f, c->stream);
    std::vector<float> c_row((size_t)n_sft);
    std::vector<double> w_row((size_t)n_sft);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c_row.data(), c->cQ_dev, sizeof(float) * n_sft, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && c->per_bin) e = cudaMemcpyAsync(w_row.data(), c->w_row_dev, sizeof(double) * n_sft, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return ft_fail(c, FT_ERR_CUDA, std::string("ft_create: fold: ") + cudaGetErrorString(e));
    c->add_back = 0.0;
    for (float v : c_row) c->add_back += (double)v;
    // Eq. (13)-(14) on the P = s/2 scale: mu_G = sum w, sigma_G^2 = sum w^2 (per-bin weights: row means, reading R21)
    double mu = 0.0, var = 0.0;
    for (int64_t a = 0; a < n_sft; ++a) {
      const double wa = c->per_bin ? w_row[(size_t)a] : (double)w[a];
      mu += wa; var += wa * wa;
    }
    d.mu_G = mu; d.sigma_G = std::sqrt(var);
  }
  c->counters.kernel_launches += 1;
  d.Q = c->Q_dev; d.H = nullptr; d.c_row = c->cQ_dev;
  return FT_OK;   // (the stream was synchronised above: host tables may be freed by the caller now)
}

int ft_set_option(ft_ctx* c, int option, int64_t value) {
  if (!c) return FT_ERR_ARG;
  switch (option) {
    case FT_OPT_KERNEL: if (value < 0 || value > 2) return ft_fail(c, FT_ERR_ARG, "FT_OPT_KERNEL: 0..2"); c->opt_kernel = value; break;
    case FT_OPT_FUSED_TOPK: c->opt_fused = value ? 1 : 0; break;
    case FT_OPT_PACKED_COUNT: c->opt_packed = value ? 1 : 0; break;
    case FT_OPT_SELECT_CAP: if (value < 0 || value > (1 << 20)) return ft_fail(c, FT_ERR_ARG, "FT_OPT_SELECT_CAP: 0 .. 2^20"); c->opt_cap = value; break;
    case FT_OPT_COUNT_FLOOR: if (value < 0 || value > (1 << 24)) return ft_fail(c, FT_ERR_ARG, "FT_OPT_COUNT_FLOOR: 0 .. 2^24"); c->opt_floor = value; break;
    case FT_OPT_ONE_PASS_BOTH: c->opt_onepass = value ? 1 : 0; break;
    case FT_OPT_VETO_FIRST: c->opt_veto_first = value ? 1 : 0; break;
    case FT_OPT_TAIL_PACKING: c->opt_tail = value ? 1 : 0; break;
    case FT_OPT_F0_TILES: if (value < 0) return ft_fail(c, FT_ERR_ARG, "FT_OPT_F0_TILES >= 0"); c->opt_tiles = value; break;
    case FT_OPT_POINTS_PER_CTA: if (value < 0) return ft_fail(c, FT_ERR_ARG, "FT_OPT_POINTS_PER_CTA >= 0"); c->opt_ppc = value; break;
    default: return ft_fail(c, FT_ERR_ARG, "unknown option");
  }
  if (c->bound) c->bound = false;  // options change the plan: re-bind with ft_eval
  return FT_OK;
}

int ft_set_option_f64(ft_ctx* c, int option, double value) {
  if (!c) return FT_ERR_ARG;
  if (option != FT_OPT_WCOUNT_FLOOR) return ft_fail(c, FT_ERR_ARG, "ft_set_option_f64: unknown option");
  if (!(value >= 0.0) || !std::isfinite(value)) return ft_fail(c, FT_ERR_ARG, "FT_OPT_WCOUNT_FLOOR >= 0");
  c->opt_wfloor = value;
  c->bound = false;
  return FT_OK;
}

int ft_set_antenna(ft_ctx* c, const double* lat, const double* gam, const double* lst) {
  if (!c) return FT_ERR_ARG;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_set_antenna: handle not created");
  if (int rc = ft_enter(c)) return rc;
  c->bound = false;
  if (!lat && !gam && !lst) { c->d.skyw = 0; c->d.ant = nullptr; return FT_OK; }
  if (!lat || !gam || !lst) return ft_fail(c, FT_ERR_ARG, "ft_set_antenna: all three arrays or none");
  if (c->per_bin) return ft_fail(c, FT_ERR_UNSUPPORTED, "ft_set_antenna: sky-dependent weights need per-SFT weights (FT_W_PER_SFT)");
  const size_t n = (size_t)c->d.n_sft;
  if (!finite_all(lat, n) || !finite_all(gam, n) || !finite_all(lst, n)) return ft_fail(c, FT_ERR_ARG, "ft_set_antenna: non-finite value");
  // a(t; n) = sum_m A_m Y_m(n), b(t; n) = sum_m B_m Z_m(n): the detector / time part of ref. [20] Eq. (12)-(13)
  std::vector<double> tab(9 * n);
  for (size_t a = 0; a < n; ++a) {
    const double s2g = std::sin(2.0 * gam[a]), c2g = std::cos(2.0 * gam[a]);
    const double sl = std::sin(lat[a]), cl = std::cos(lat[a]), s2l = std::sin(2.0 * lat[a]), c2l = std::cos(2.0 * lat[a]);
    const double a1 = (1.0 / 16.0) * s2g * (3.0 - c2l), a2 = 0.25 * c2g * sl, a3 = 0.25 * s2g * s2l, a4 = 0.5 * c2g * cl,
                 a5 = 0.75 * s2g * cl * cl;
    const double b1 = c2g * sl, b2 = 0.25 * s2g * (3.0 - c2l), b3 = c2g * cl, b4 = 0.5 * s2g * s2l;
    const double ct = std::cos(lst[a]), st = std::sin(lst[a]), c2t = std::cos(2.0 * lst[a]), s2t = std::sin(2.0 * lst[a]);
    double* r = tab.data() + 9 * a;
    r[0] = a1 * c2t + a2 * s2t; r[1] = a1 * s2t - a2 * c2t; r[2] = a3 * ct + a4 * st; r[3] = a3 * st - a4 * ct; r[4] = a5;
    r[5] = b1 * c2t - b2 * s2t; r[6] = b1 * s2t + b2 * c2t; r[7] = b3 * ct - b4 * st; r[8] = b3 * st + b4 * ct;
  }
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (!c->ant_dev) FT_CUDA(c, cudaMalloc(&c->ant_dev, sizeof(double) * 9 * n));
  FT_CUDA(c, cudaMemcpy(c->ant_dev, tab.data(), sizeof(double) * 9 * n, cudaMemcpyHostToDevice));
  c->d.ant = c->ant_dev; c->d.skyw = 1;
  return FT_OK;
}

int ft_eval(ft_ctx* c, const ft_grid* g, int stat, double rho_th, float* out_power_dev, int32_t* out_count_dev) {
  if (!c || !g) return FT_ERR_ARG;
  c->bound = false;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_eval: handle not created");
  if (stat < 0 || stat > 3) return ft_fail(c, FT_ERR_ARG, "ft_eval: bad stat");
  if (!g->sky || !g->a_p || !g->P_orb || !g->tasc_frac) return ft_fail(c, FT_ERR_ARG, "ft_eval: NULL grid axis");
  if (g->n_f0 < 1 || g->n_f1 < 1 || g->n_sky < 1 || g->n_ap < 1 || g->n_porb < 1 || g->n_tasc < 1) return ft_fail(c, FT_ERR_ARG, "ft_eval: empty grid axis");
  const double scal[] = {g->f0_start, g->df0, g->f1_start, g->df1, g->t_ref, rho_th};
  if (!finite_all(scal, 6) || !finite_all(g->sky, 3 * (size_t)g->n_sky) || !finite_all(g->a_p, g->n_ap) ||
      !finite_all(g->P_orb, g->n_porb) || !finite_all(g->tasc_frac, g->n_tasc))
    return ft_fail(c, FT_ERR_ARG, "ft_eval: non-finite grid value");
  if (g->n_f0 > 1 && !(g->df0 > 0.0)) return ft_fail(c, FT_ERR_ARG, "ft_eval: df0 must be > 0");
  for (int i = 0; i < g->n_porb; ++i) if (!(g->P_orb[i] > 0.0)) return ft_fail(c, FT_ERR_ARG, "ft_eval: P_orb must be > 0");
  if (int rc = ft_enter(c)) return rc;
  // conservative bound on every track (header: FT_ERR_TRACK_RANGE; reading R9)
  double ap_max = 0.0, porb_min = g->P_orb[0], n_max = 0.0;
  for (int i = 0; i < g->n_ap; ++i) ap_max = std::fmax(ap_max, std::fabs(g->a_p[i]));
  for (int i = 0; i < g->n_porb; ++i) porb_min = std::fmin(porb_min, g->P_orb[i]);
  for (int64_t i = 0; i < g->n_sky; ++i) {
    const double* n = g->sky + 3 * i;
    n_max = std::fmax(n_max, std::sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]));
  }
  const double eps = c->vmax * n_max / FT_C_LIGHT + ap_max * FT_TWO_PI / porb_min;
  double dt_lo = c->t_mid[0] - g->t_ref, dt_hi = dt_lo;
  for (double t : c->t_mid) { dt_lo = std::fmin(dt_lo, t - g->t_ref); dt_hi = std::fmax(dt_hi, t - g->t_ref); }
  const double f1a = g->f1_start, f1b = g->f1_start + (double)(g->n_f1 - 1) * g->df1;
  const double cands[4] = {f1a * dt_lo, f1a * dt_hi, f1b * dt_lo, f1b * dt_hi};
  double f1dt_lo = cands[0], f1dt_hi = cands[0];
  for (double v : cands) { f1dt_lo = std::fmin(f1dt_lo, v); f1dt_hi = std::fmax(f1dt_hi, v); }
  const double fs_lo = g->f0_start + f1dt_lo, fs_hi = g->f0_start + (double)(g->n_f0 - 1) * g->df0 + f1dt_hi;
  if (!(fs_lo > 0.0) || !(eps < 0.01)) return ft_fail(c, FT_ERR_ARG, "ft_eval: need positive frequencies and |Doppler| < 1e-2");
  const double x_lo = (fs_lo * (1.0 - eps) - c->d.f_min) / c->df, x_hi = (fs_hi * (1.0 + eps) - c->d.f_min) / c->df;
  if (x_lo < -0.49 || x_hi > (double)(c->d.n_bins - 1) + 0.49) {
    char buf[256];
    std::snprintf(buf, sizeof buf, "ft_eval: tracks may leave the spectrogram: bound [%.2f, %.2f] bins vs [0, %lld)", x_lo, x_hi, (long long)c->d.n_bins);
    return ft_fail(c, FT_ERR_TRACK_RANGE, buf);
  }
  if (int rc = ft_check_tile_err(c)) return rc;  // synchronises (previous work may still read the old axes / plans);
                                                 // a planning error of the previous evaluation surfaces here
  // copy axes (the staging vector lives in the handle: no second synchronisation)
  const size_t n_ax = 3 * (size_t)g->n_sky + g->n_ap + g->n_porb + g->n_tasc;
  std::vector<double>& ax = c->axes_host;
  ax.resize(n_ax);
  std::memcpy(ax.data(), g->sky, sizeof(double) * 3 * g->n_sky);
  size_t o = 3 * (size_t)g->n_sky;
  std::memcpy(ax.data() + o, g->a_p, sizeof(double) * g->n_ap); o += g->n_ap;
  std::memcpy(ax.data() + o, g->P_orb, sizeof(double) * g->n_porb); o += g->n_porb;
  std::memcpy(ax.data() + o, g->tasc_frac, sizeof(double) * g->n_tasc);
  FT_CUDA(c, ft_grow(c->axes_dev, c->axes_cap, n_ax));
  FT_CUDA(c, cudaMemcpyAsync(c->axes_dev, ax.data(), sizeof(double) * n_ax, cudaMemcpyHostToDevice, c->stream));
  FtDev& d = c->d;
  d.sky = c->axes_dev; d.a_p = d.sky + 3 * g->n_sky; d.P_orb = d.a_p + g->n_ap; d.tasc = d.P_orb + g->n_porb;
  d.n_f0 = g->n_f0; d.n_sky = g->n_sky; d.n_f1 = g->n_f1; d.n_ap = g->n_ap; d.n_porb = g->n_porb; d.n_tasc = g->n_tasc;
  d.f0_start = g->f0_start; d.df0 = g->df0; d.f1_start = g->f1_start; d.df1 = g->df1; d.t_ref = g->t_ref;
  d.rho = (float)rho_th;
  d.n_points = (uint64_t)g->n_sky * g->n_ap * g->n_porb * g->n_tasc * g->n_f1;
  c->stat = stat;
  // binary grids: cos(Om (t - t_asc)) per (P_orb, t_asc, SFT) once, shared by every a_p (<= 1 GiB)
  // (rebuilt only when t_ref, P_orb[] or tasc_frac[] change: the table does not depend on anything else)
  d.ctab = nullptr;
  const size_t ctab_elems = (size_t)g->n_porb * g->n_tasc * (size_t)d.n_sft;
  if (ap_max != 0.0 && g->n_porb * (int64_t)g->n_tasc <= 65535 && ctab_elems <= ((size_t)1 << 27)) {
    std::vector<double> key;
    key.push_back(g->t_ref); key.push_back((double)g->n_porb); key.push_back((double)g->n_tasc);
    key.insert(key.end(), g->P_orb, g->P_orb + g->n_porb);
    key.insert(key.end(), g->tasc_frac, g->tasc_frac + g->n_tasc);
    if (c->ctab_cap < ctab_elems) {
      c->ctab_key.clear();
      FT_CUDA(c, ft_grow(c->ctab_dev, c->ctab_cap, ctab_elems));
    }
    if (key != c->ctab_key) {
      FT_CUDA(c, ft_launch_ctab(d, c->ctab_dev, c->stream));
      c->counters.kernel_launches += 1;
      c->ctab_key = key;
    }
    d.ctab = c->ctab_dev;
  }
  // ---- tile-kernel eligibility and plans: tilings on the host, strip tables on the device, ONE synchronisation
  const bool skyw = d.skyw != 0;
  const bool want_wh = stat == FT_STAT_WHOUGH || (stat == FT_STAT_BOTH && c->opt_wfloor > 0.0);
  c->tile_ok = c->tile8_ok = c->tileb_ok = c->tilew_ok = false;
  if (c->opt_kernel != 1) {
    FtTileHostIn hin{c->t_mid.data(), c->vel.data(), g->sky, g->a_p, g->P_orb, c->df, eps, (int)c->opt_ppc, (int)c->opt_tiles, (int)c->opt_tail};
    std::string why8, whyb, whyw;
    bool t0 = ft_tile_choose(d, hin, 0, &c->plan, &c->why);
    bool t8 = t0 && stat != FT_STAT_POWER && c->opt_packed && ft_tile_choose(d, hin, 1, &c->plan8, &why8);
    // narrow bands (< 6 chunks of 128 f0 per warp) are bound by the per-(warp, SFT) bookkeeping, which the
    // fp32 map amortises over four times as many loads: measured faster there (config 3, 450 f0)
    t8 = t8 && c->plan8.J >= 6;
    // both statistics in one pass only where the fp32 plan itself is narrow (J <= 16): wide bands run power on
    // K2 and the count packed
    bool tb = t0 && stat == FT_STAT_BOTH && c->opt_onepass && !skyw && (c->plan.J <= 16 || c->plan.ppw == 2) &&
              ft_tile_choose(d, hin, 2, &c->planb, &whyb) && c->planb.n_tiles == c->plan.n_tiles;
    bool tw = t0 && skyw && ft_tile_choose(d, hin, 3, &c->planw, &whyw);
    if (t0) {
      FT_CUDA(c, ft_launch_vrange(d, c->vr_dev, c->stream));
      FT_CUDA(c, cudaMemsetAsync(c->maxw_dev, 0, sizeof(int32_t) * 4, c->stream));
      int launches = 1;
      FtTilePlan* pls[4] = {&c->plan, &c->plan8, &c->planb, &c->planw};
      const bool on[4] = {t0, t8, tb, tw};
      for (int m = 0; m < 4; ++m)
        if (on[m]) { FT_CUDA(c, ft_tile_strips(d, hin, pls[m], c->vr_dev, c->maxw_dev + m, c->stream)); ++launches; }
      c->counters.kernel_launches += launches;
      int32_t maxw[4] = {0, 0, 0, 0};
      FT_CUDA(c, cudaMemcpyAsync(maxw, c->maxw_dev, sizeof maxw, cudaMemcpyDeviceToHost, c->stream));
      FT_CUDA(c, cudaStreamSynchronize(c->stream));
      t0 = ft_tile_finish(d, &c->plan, maxw[0], &c->why);
      t8 = t8 && t0 && ft_tile_finish(d, &c->plan8, maxw[1], &why8);
      tb = tb && t0 && ft_tile_finish(d, &c->planb, maxw[2], &whyb);
      tw = tw && t0 && ft_tile_finish(d, &c->planw, maxw[3], &whyw);
    }
    c->tile_ok = t0; c->tile8_ok = t8; c->tileb_ok = tb; c->tilew_ok = tw;
    if (skyw && t0 && !tw) { c->tile_ok = false; c->why = "sky-dependent weights: " + whyw; }
    if (!c->tile_ok && c->opt_kernel == 2) return ft_fail(c, FT_ERR_UNSUPPORTED, "tile kernel not eligible: " + c->why);
  }
  if (skyw && !c->tile_ok)
    return ft_fail(c, FT_ERR_UNSUPPORTED, "sky-dependent weights (ft_set_antenna) need a grid the tile kernel accepts: " +
                                              (c->opt_kernel == 1 ? std::string("generic kernel forced") : c->why));
  // ---- gather arrays that depend on rho_th (rebuilt only when it changes) ---------------------------------
  if (c->tile8_ok && !(c->H8_valid && c->H8_rho == d.rho)) {
    const int64_t ld8 = (d.n_bins + 15) / 16 * 16;
    if (!c->H8_dev) FT_CUDA(c, cudaMalloc(&c->H8_dev, (size_t)4 * d.n_sft * ld8 + 16384));
    FT_CUDA(c, cudaMemsetAsync(c->H8_dev + (size_t)4 * d.n_sft * ld8, 0, 16384, c->stream));
    FT_CUDA(c, ft_launch_hitmap8(d.P, d.rho, c->H8_dev, d.n_sft, d.n_bins, d.ld, ld8, c->stream));
    c->counters.kernel_launches += 1;
    c->H8_rho = d.rho; c->H8_valid = true;
    d.ld8 = ld8;
  }
  d.H8 = c->H8_dev;
  if (c->tile_ok && !c->tile8_ok && stat != FT_STAT_POWER && !(c->H_valid && c->H_rho == d.rho)) {
    if (!c->H_dev) FT_CUDA(c, cudaMalloc(&c->H_dev, sizeof(float) * (size_t)d.n_sft * d.ld));
    FT_CUDA(c, ft_launch_hitmap(d.P, d.rho, c->H_dev, d.n_sft * d.ld, c->stream));
    c->counters.kernel_launches += 1;
    c->H_rho = d.rho; c->H_valid = true;
  }
  d.H = c->H_dev;
  if (c->tileb_ok && !(c->QB_valid && c->QB_rho == d.rho)) {
    if (!c->QB_dev) FT_CUDA(c, cudaMalloc(&c->QB_dev, sizeof(float) * (size_t)d.n_sft * d.ld));
    FT_CUDA(c, ft_launch_qb(d.Q, d.P, d.rho, c->QB_dev, d.n_sft * d.ld, c->stream));
    c->counters.kernel_launches += 1;
    c->QB_rho = d.rho; c->QB_valid = true;
  }
  if (c->tile_ok && want_wh && !(c->WH_valid && c->WH_rho == d.rho)) {
    // folded, centred w x [P > rho]: the weighted number count is the same gather-reduce as the power
    if (!c->WH_dev) FT_CUDA(c, cudaMalloc(&c->WH_dev, sizeof(float) * (size_t)d.n_sft * d.ld));
    if (!c->cWH_dev) FT_CUDA(c, cudaMalloc(&c->cWH_dev, sizeof(float) * d.n_sft));
    FT_CUDA(c, ft_launch_fold_centered(d.P, c->per_bin ? nullptr : c->w_dev, c->per_bin ? d.w : nullptr, c->WH_dev, c->cWH_dev,
                                       nullptr, d.n_sft, d.n_bins, d.ld, 1, d.rho, c->stream));
    std::vector<float> c_row((size_t)d.n_sft);
    FT_CUDA(c, cudaMemcpyAsync(c_row.data(), c->cWH_dev, sizeof(float) * d.n_sft, cudaMemcpyDeviceToHost, c->stream));
    FT_CUDA(c, cudaStreamSynchronize(c->stream));
    c->add_back_wh = 0.0;
    for (float v : c_row) c->add_back_wh += (double)v;
    c->counters.kernel_launches += 1;
    c->WH_rho = d.rho; c->WH_valid = true;
  }
  if (c->tilew_ok) {
    // sky-dependent weights: normalisation, add-back and sigma_G of every sky point of the grid (one small pass)
    FT_CUDA(c, ft_grow(c->skyn_dev, c->skyn_cap, 4 * (size_t)d.n_sky));
    FT_CUDA(c, ft_launch_skyw_norm(d, c->cQ_dev, (want_wh && c->WH_valid) ? c->cWH_dev : nullptr, c->skyn_dev, c->stream));
    c->counters.kernel_launches += 1;
  }
  {
    char buf[400];
    auto geom = [&](const FtTilePlan& pl) {
      std::snprintf(buf, sizeof buf, "J=%d wpp=%d%s R=%d n_tiles=%d tile_w=%d threads=%d pitch=%d copy=%d stages=%dx%d smem=%zu",
                    pl.J, pl.wpp, pl.ppw == 2 ? " (two points per warp)" : "", pl.R, pl.n_tiles, pl.tile_w,
                    (pl.R * pl.wpp / pl.ppw + 1) * 32, pl.pitch, pl.copy_floats, pl.n_stages, pl.rows_per_stage, pl.smem_bytes);
      return std::string(buf);
    };
    if (c->tile_ok && c->opt_kernel != 1) c->desc = "K2 tile kernel: " + geom(c->plan);
    else c->desc = std::string("K0 generic kernel (") + (c->opt_kernel == 1 ? "forced" : c->why.c_str()) + ")";
    if (c->tilew_ok) c->desc += "; sky-dependent weights: row-weighted tile kernel " + geom(c->planw);
    if (c->tileb_ok) c->desc += "; both statistics: one-pass tile kernel " + geom(c->planb);
    if (c->tile8_ok) c->desc += "; number count: packed tile kernel " + geom(c->plan8);
  }
  c->bound = true;
  if (out_power_dev || out_count_dev) {
    c->ev_used = 0; c->counters.stat_launches = 0;
    FtPass p;
    p.stat = stat; p.pt_begin = 0; p.pt_end = d.n_points; p.out_f = out_power_dev; p.out_i = out_count_dev;
    const int rc = ft_run_stat(c, p);
    if (rc != FT_OK) return rc;
  }
  return FT_OK;
}

int ft_eval_list(ft_ctx* c, const uint64_t* idx_host, int64_t n, ft_cand* out_host) {
  if (!c || !idx_host || !out_host || n < 0) return FT_ERR_ARG;
  if (!c->bound) return ft_fail(c, FT_ERR_STATE, "ft_eval_list: no grid bound");
  if (n == 0) return FT_OK;
  if (int rc = ft_enter(c)) return rc;
  const uint64_t n_templates = c->d.n_points * (uint64_t)c->d.n_f0;
  for (int64_t i = 0; i < n; ++i)
    if (idx_host[i] >= n_templates) return ft_fail(c, FT_ERR_ARG, "ft_eval_list: index out of range");
  FT_CUDA(c, cudaStreamSynchronize(c->stream));   // the grow-only scratch may still be in use
  FT_CUDA(c, ft_grow(c->io_dev, c->io_cap, (sizeof(uint64_t) + sizeof(FtCandDev)) * (size_t)n));
  uint64_t* idx_dev = reinterpret_cast<uint64_t*>(c->io_dev);
  FtCandDev* out_dev = reinterpret_cast<FtCandDev*>(c->io_dev + sizeof(uint64_t) * (size_t)n);
  std::vector<FtCandDev> tmp((size_t)n);
  FT_CUDA(c, cudaMemcpyAsync(idx_dev, idx_host, sizeof(uint64_t) * n, cudaMemcpyHostToDevice, c->stream));
  FT_CUDA(c, ft_launch_refine(c->d, idx_dev, nullptr, n, out_dev, c->near_ties_dev, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(tmp.data(), out_dev, sizeof(FtCandDev) * n, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  c->counters.kernel_launches += 1;
  for (int64_t i = 0; i < n; ++i) {
    const FtCandDev& s = tmp[(size_t)i];
    out_host[i] = ft_cand{s.power, s.wcount, s.idx, s.count, s.band};
  }
  return ft_check_tile_err(c);
}

int ft_get_counters(ft_ctx* c, ft_counters* out) {
  if (!c || !out) return FT_ERR_ARG;
  if (int rc = ft_enter(c)) return rc;
  unsigned long long nt = 0;
  int32_t terr = 0;
  FT_CUDA(c, cudaMemcpyAsync(&nt, c->near_ties_dev, sizeof nt, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(&terr, c->tile_err_dev, sizeof terr, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (int rc2 = ft_tile_err_status(c, terr)) return rc2;
  c->counters.near_ties = nt;
  double ms_sum = 0.0;
  for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->evs[i], c->evs[i + 1]) == cudaSuccess) ms_sum += ms;
  }
  c->counters.last_kernel_ms = ms_sum;
  *out = c->counters;
  return FT_OK;
}

const char* ft_last_error(const ft_ctx* c) { return c ? c->err.c_str() : "null handle"; }
const char* ft_describe(const ft_ctx* c) { return c ? c->desc.c_str() : "null handle"; }

void ft_destroy(ft_ctx* c) {
  if (!c) return;
  if (c->d.P) { cudaSetDevice(c->device); cudaStreamSynchronize(c->stream); }
  ft_dfree(c->sel.thr); ft_dfree(c->sel.cnt); ft_dfree(c->sel.key); ft_dfree(c->sel.idx);
  ft_dfree(c->final_idx); ft_dfree(c->final_region); ft_dfree(c->final_n); ft_dfree(c->cand); ft_dfree(c->out_dev);
  ft_tile_plan_free(&c->plan);
  ft_tile_plan_free(&c->plan8);
  ft_tile_plan_free(&c->planb);
  ft_tile_plan_free(&c->planw);
  ft_dfree(c->H8_dev); ft_dfree(c->QB_dev); ft_dfree(c->WH_dev); ft_dfree(c->cWH_dev); ft_dfree(c->cQ_dev);
  ft_dfree(c->t_mid_dev); ft_dfree(c->vel_dev); ft_dfree(c->w_dev); ft_dfree(c->Q_dev); ft_dfree(c->H_dev);
  ft_dfree(c->ctab_dev); ft_dfree(c->axes_dev); ft_dfree(c->w_row_dev); ft_dfree(c->ant_dev); ft_dfree(c->vr_dev);
  ft_dfree(c->skyn_dev); ft_dfree(c->maxw_dev); ft_dfree(c->scratch_f); ft_dfree(c->scratch_i); ft_dfree(c->veto_cnt); ft_dfree(c->veto_w);
  ft_dfree(c->surv_dev); ft_dfree(c->glist_dev); ft_dfree(c->pbox_dev); ft_dfree(c->io_dev); ft_dfree(c->near_ties_dev); ft_dfree(c->flag_dev);
  ft_dfree(c->tile_err_dev);
  for (cudaEvent_t e : c->evs) cudaEventDestroy(e);
  delete c;
}

}  // extern "C"
