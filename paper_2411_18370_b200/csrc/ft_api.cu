// C ABI of libfasttracks_b200 (include/fasttracks_b200.h): handle, validation, launch orchestration.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/fasttracks_b200.h"
#include "ft_common.cuh"
#include "ft_select.cuh"
#include "ft_tile.cuh"

struct ft_ctx {
  cudaStream_t stream = nullptr;
  FtDev d{};
  bool per_bin = false;
  // library-owned device memory
  double* t_mid_dev = nullptr;
  double* vel_dev = nullptr;
  float* w_dev = nullptr;       // per-SFT weights copy
  float* Q_dev = nullptr;       // folded w*P (tile kernel input)
  float* H_dev = nullptr;       // hit map (tile kernel input for the number count)
  float H_rho = 0.f; bool H_valid = false;
  double add_back = 0.0;        // sum over SFTs of the per-row constant the fold removed from Q
  double* axes_dev = nullptr;   // sky | a_p | P_orb | tasc (grow-only buffer)
  size_t axes_cap = 0;
  double* ctab_dev = nullptr;   // orbital cosine table of the bound grid (binary grids; grow-only buffer)
  size_t ctab_cap = 0;
  std::vector<double> ctab_key; // (t_ref, P_orb[], tasc_frac[]) the table was built for
  // host copies used for validation
  std::vector<double> t_mid, vel;
  double vmax = 0.0, dt_min = 0.0, dt_max = 0.0;
  // bound grid
  bool bound = false;
  int stat = 0;
  double df = 0.0;
  bool tile_ok = false;
  FtTilePlan plan{};            // fp32 gather (power; number count when the packed kernel is not eligible)
  FtTilePlan plan8{};           // packed number-count kernel (ft_tile8.cu)
  bool tile8_ok = false;
  FtTilePlan planb{};           // both statistics in one pass (ft_tileb.cu), narrow bands
  bool tileb_ok = false;
  float* QB_dev = nullptr;      // Q with the hit bit in the LSB
  float QB_rho = 0.f; bool QB_valid = false;
  uint8_t* H8_dev = nullptr;    // four byte-shifted hit maps
  float H8_rho = 0.f; bool H8_valid = false;
  // options
  int64_t opt_kernel = 0, opt_fused = 1, opt_ppc = 0, opt_packed = 1, opt_tiles = 0, opt_cap = 0, opt_floor = 0, opt_onepass = 1;
  // selection buffers
  FtSelectDev sel{};
  uint64_t* final_idx = nullptr;
  int32_t* final_band = nullptr;
  uint32_t* final_n = nullptr;   // [0] final_n, [1] overflow
  FtCandDev* cand = nullptr;
  FtCandDev* out_dev = nullptr;
  uint32_t final_cap = 0;
  size_t out_cap = 0;
  float* scratch_f = nullptr;
  int32_t* scratch_i = nullptr;
  int32_t* veto_cnt = nullptr;  // number count of every template (FT_OPT_COUNT_FLOOR), grow-only
  size_t veto_cap = 0;
  size_t scratch_elems = 0;
  unsigned long long* near_ties_dev = nullptr;
  // bookkeeping
  ft_counters counters{};
  std::vector<cudaEvent_t> evs;  // pairs around every statistic-kernel pass of the last call
  size_t ev_used = 0;
  std::string err = "";
  std::string desc = "no grid bound";
  std::string why;
};

namespace {

int fail(ft_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
#define FT_CUDA(c, expr)                                                                     \
  do {                                                                                       \
    cudaError_t e__ = (expr);                                                                \
    if (e__ != cudaSuccess)                                                                  \
      return fail((c), e__ == cudaErrorMemoryAllocation ? FT_ERR_ALLOC : FT_ERR_CUDA,        \
                  std::string(#expr) + ": " + cudaGetErrorString(e__));                      \
  } while (0)

template <typename T>
void dfree(T*& p) {
  if (p) cudaFree(p);
  p = nullptr;
}

bool finite_all(const double* p, size_t n) {
  for (size_t i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return false;
  return true;
}

void free_select(ft_ctx* c) {
  dfree(c->sel.thr); dfree(c->sel.cnt); dfree(c->sel.key); dfree(c->sel.idx);
  dfree(c->final_idx); dfree(c->final_band); dfree(c->final_n); dfree(c->cand); dfree(c->out_dev);
  c->sel = FtSelectDev{};
  c->final_cap = 0; c->out_cap = 0;
}

int ensure_select(ft_ctx* c, int32_t n_bands, int32_t k) {
  uint32_t cap = (uint32_t)((1u << 24) / (uint32_t)n_bands);
  cap = cap > 65536u ? 65536u : (cap < 4096u ? 4096u : cap);
  if (c->opt_cap > 0) cap = (uint32_t)c->opt_cap;  // FT_OPT_SELECT_CAP (tests of the overflow recovery)
  const uint32_t final_cap = (uint32_t)n_bands * 2048u;
  if (c->sel.n_bands != n_bands || c->sel.cap != cap || c->out_cap < (size_t)n_bands * k) {
    free_select(c);
    FT_CUDA(c, cudaMalloc(&c->sel.thr, sizeof(float) * n_bands));
    FT_CUDA(c, cudaMalloc(&c->sel.cnt, sizeof(uint32_t) * n_bands));
    FT_CUDA(c, cudaMalloc(&c->sel.key, sizeof(float) * (size_t)n_bands * cap));
    FT_CUDA(c, cudaMalloc(&c->sel.idx, sizeof(uint64_t) * (size_t)n_bands * cap));
    c->sel.cap = cap; c->sel.n_bands = n_bands;
    FT_CUDA(c, cudaMalloc(&c->final_idx, sizeof(uint64_t) * final_cap));
    FT_CUDA(c, cudaMalloc(&c->final_band, sizeof(int32_t) * final_cap));
    FT_CUDA(c, cudaMalloc(&c->final_n, sizeof(uint32_t) * 2));
    FT_CUDA(c, cudaMalloc(&c->cand, sizeof(FtCandDev) * final_cap));
    FT_CUDA(c, cudaMalloc(&c->out_dev, sizeof(FtCandDev) * (size_t)n_bands * k));
    c->final_cap = final_cap; c->out_cap = (size_t)n_bands * k;
  }
  return FT_OK;
}

int ensure_scratch(ft_ctx* c, size_t elems, bool need_int) {
  if (c->scratch_elems < elems) {
    dfree(c->scratch_f); dfree(c->scratch_i);
    c->scratch_elems = 0;
    FT_CUDA(c, cudaMalloc(&c->scratch_f, sizeof(float) * elems));
    c->scratch_elems = elems;
  }
  if (need_int && !c->scratch_i) FT_CUDA(c, cudaMalloc(&c->scratch_i, sizeof(int32_t) * c->scratch_elems));
  return FT_OK;
}

// CUDA events on the handle's stream around each statistic pass (ft_counters.last_kernel_ms)
void tick(ft_ctx* c) {
  if (c->ev_used + 2 > c->evs.size()) {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    c->evs.push_back(e0); c->evs.push_back(e1);
  }
  cudaEventRecord(c->evs[c->ev_used], c->stream);
}
void tock(ft_ctx* c, int launches) {
  cudaEventRecord(c->evs[c->ev_used + 1], c->stream);
  c->ev_used += 2;
  c->counters.stat_launches += (uint64_t)launches;
  c->counters.kernel_launches += (uint64_t)launches;
}

// Statistic over points [pt_begin, pt_end): full write-out (out_* indexed from out_base) and/or
// fused filter into c->sel.  Chooses the tile or the generic kernel.
int run_stat(ft_ctx* c, int stat, uint64_t pt_begin, uint64_t pt_end, float* out_power, int32_t* out_count,
             uint64_t out_base, bool filter, int32_t bpb, uint32_t stride = 1, uint64_t n_strided = 0,
             bool complement = false) {
  const bool use_tile = c->tile_ok && c->opt_kernel != 1;
  if (use_tile) {
    // one gather-reduce pass per statistic: power over Q, number count over the hit map
    const FtSelectDev* sel = filter ? &c->sel : nullptr;
    int launches = 0;
    if (stat == FT_STAT_BOTH && c->tileb_ok && ((out_power && out_count) || filter)) {
      // narrow bands: both statistics (and the count veto of the fused filter) from one gather
      tick(c);
      FT_CUDA(c, ft_launch_tile(c->d, c->planb, c->QB_dev, c->add_back, pt_begin, pt_end, out_power, out_count, out_base,
                                sel, bpb, c->near_ties_dev, c->stream, &launches, stride, n_strided, complement));
      tock(c, launches);
      return FT_OK;
    }
    if (stat != FT_STAT_HOUGH && (out_power || (filter && stat == FT_STAT_POWER))) {
      tick(c);
      FT_CUDA(c, ft_launch_tile(c->d, c->plan, c->d.Q, c->add_back, pt_begin, pt_end, out_power, nullptr, out_base,
                                stat == FT_STAT_POWER ? sel : nullptr, bpb, c->near_ties_dev, c->stream, &launches, stride, n_strided, complement));
      tock(c, launches);
    }
    if (stat != FT_STAT_POWER && (out_count || (filter && stat == FT_STAT_HOUGH))) {
      tick(c);
      FT_CUDA(c, ft_launch_tile(c->d, c->tile8_ok ? c->plan8 : c->plan, c->d.H, 0.0, pt_begin, pt_end, nullptr, out_count, out_base,
                                stat == FT_STAT_HOUGH ? sel : nullptr, bpb, c->near_ties_dev, c->stream, &launches, stride, n_strided, complement));
      tock(c, launches);
    }
  } else {
    if (filter) return fail(c, FT_ERR_UNSUPPORTED, "fused filter needs the tile kernel");
    tick(c);
    FT_CUDA(c, ft_launch_generic(c->d, stat, pt_begin, pt_end, out_power, out_count, out_base, c->stream));
    tock(c, 1);
  }
  return FT_OK;
}

// The tile kernel raises plan.err if a track left its staged strip (a planning bug, never data):
// surfaced at the next synchronising call instead of silently wrong sums.
int check_tile_err(ft_ctx* c) {
  for (const FtTilePlan* pl : {&c->plan, &c->plan8, &c->planb}) {
    if (!pl->err) continue;
    int32_t e = 0;
    FT_CUDA(c, cudaMemcpy(&e, pl->err, sizeof e, cudaMemcpyDeviceToHost));
    if (e != 0) return fail(c, FT_ERR_STATE, e == 1 ? "tile kernel: a track left its staged strip (internal planning error)"
                                                    : "tile kernel: more than one break in a warp range (internal planning error)");
  }
  return FT_OK;
}

}  // namespace

extern "C" {

int ft_create(ft_ctx** out, const float* P_dev, int64_t n_sft, int64_t n_bins, int64_t ld_bins,
              const double* t_mid_host, const double* vel_host, const float* w, int wkind,
              double f_min, double df, void* cuda_stream) {
  if (!out) return FT_ERR_ARG;
  *out = nullptr;
  ft_ctx* c = new (std::nothrow) ft_ctx();
  if (!c) return FT_ERR_ALLOC;
  *out = c;  // returned even on error so ft_last_error can be read; caller still calls ft_destroy
  if (!P_dev || !t_mid_host || !vel_host || !w) return fail(c, FT_ERR_ARG, "ft_create: NULL pointer argument");
  if (n_sft < 1 || n_bins < 1 || ld_bins < n_bins) return fail(c, FT_ERR_ARG, "ft_create: need n_sft >= 1, 1 <= n_bins <= ld_bins");
  if (n_sft > (1 << 24)) return fail(c, FT_ERR_ARG, "ft_create: n_sft > 2^24 (integer counts are selected as exact fp32 keys)");
  if ((ld_bins & 3) || (reinterpret_cast<uintptr_t>(P_dev) & 15)) return fail(c, FT_ERR_ARG, "ft_create: P must be 16-byte aligned with ld_bins a multiple of 4");
  if (wkind != FT_W_PER_SFT && wkind != FT_W_PER_SFT_BIN) return fail(c, FT_ERR_ARG, "ft_create: bad wkind");
  if (!(df > 0.0) || !std::isfinite(df) || !std::isfinite(f_min)) return fail(c, FT_ERR_ARG, "ft_create: need finite f_min and df > 0");
  if (!finite_all(t_mid_host, (size_t)n_sft) || !finite_all(vel_host, (size_t)n_sft * 3)) return fail(c, FT_ERR_ARG, "ft_create: non-finite t_mid / vel");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(c, FT_ERR_CUDA, "ft_create: no CUDA device (this library has no CPU fallback)");
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
  FtDev& d = c->d;
  d.P = P_dev; d.n_sft = n_sft; d.n_bins = n_bins; d.ld = ld_bins;
  d.t_mid = c->t_mid_dev; d.vel = c->vel_dev;
  d.wkind = wkind; d.f_min = f_min; d.inv_df = 1.0 / df;
  c->df = df;
  c->per_bin = (wkind == FT_W_PER_SFT_BIN);
  // A0: Q = fl(fl(w P) - c_row) (the fp64 refinement uses w and P unfolded); add_back = sum c_row
  FT_CUDA(c, cudaMalloc(&c->Q_dev, sizeof(float) * (size_t)n_sft * ld_bins));
  float* c_row_dev = nullptr;
  FT_CUDA(c, cudaMalloc(&c_row_dev, sizeof(float) * n_sft));
  if (!c->per_bin) {
    FT_CUDA(c, cudaMalloc(&c->w_dev, sizeof(float) * n_sft));
    FT_CUDA(c, cudaMemcpyAsync(c->w_dev, w, sizeof(float) * n_sft, cudaMemcpyHostToDevice, c->stream));
    d.w = c->w_dev;
  } else {
    if (reinterpret_cast<uintptr_t>(w) & 15) { cudaFree(c_row_dev); return fail(c, FT_ERR_ARG, "ft_create: per-bin weights must be 16-byte aligned"); }
    d.w = w;
  }
  {
    cudaError_t e = ft_launch_fold_centered(P_dev, c->per_bin ? nullptr : c->w_dev, c->per_bin ? w : nullptr,
                                            c->Q_dev, c_row_dev, n_sft, n_bins, ld_bins, c->stream);
    std::vector<float> c_row((size_t)n_sft);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c_row.data(), c_row_dev, sizeof(float) * n_sft, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(c_row_dev);
    if (e != cudaSuccess) return fail(c, FT_ERR_CUDA, std::string("ft_create: fold: ") + cudaGetErrorString(e));
    c->add_back = 0.0;
    for (float v : c_row) c->add_back += (double)v;
  }
  c->counters.kernel_launches += 1;
  d.Q = c->Q_dev; d.H = nullptr;
  FT_CUDA(c, cudaStreamSynchronize(c->stream));  // host tables may be freed by the caller now
  return FT_OK;
}

int ft_set_option(ft_ctx* c, int option, int64_t value) {
  if (!c) return FT_ERR_ARG;
  switch (option) {
    case FT_OPT_KERNEL: if (value < 0 || value > 2) return fail(c, FT_ERR_ARG, "FT_OPT_KERNEL: 0..2"); c->opt_kernel = value; break;
    case FT_OPT_FUSED_TOPK: c->opt_fused = value ? 1 : 0; break;
    case FT_OPT_PACKED_COUNT: c->opt_packed = value ? 1 : 0; break;
    case FT_OPT_SELECT_CAP: if (value < 0 || value > (1 << 20)) return fail(c, FT_ERR_ARG, "FT_OPT_SELECT_CAP: 0 .. 2^20"); c->opt_cap = value; break;
    case FT_OPT_COUNT_FLOOR: if (value < 0 || value > (1 << 24)) return fail(c, FT_ERR_ARG, "FT_OPT_COUNT_FLOOR: 0 .. 2^24"); c->opt_floor = value; break;
    case FT_OPT_ONE_PASS_BOTH: c->opt_onepass = value ? 1 : 0; break;
    case FT_OPT_F0_TILES: if (value < 0) return fail(c, FT_ERR_ARG, "FT_OPT_F0_TILES >= 0"); c->opt_tiles = value; break;
    case FT_OPT_POINTS_PER_CTA: if (value < 0) return fail(c, FT_ERR_ARG, "FT_OPT_POINTS_PER_CTA >= 0"); c->opt_ppc = value; break;
    default: return fail(c, FT_ERR_ARG, "unknown option");
  }
  if (c->bound) c->bound = false;  // options change the plan: re-bind with ft_eval
  return FT_OK;
}

int ft_eval(ft_ctx* c, const ft_grid* g, int stat, double rho_th, float* out_power_dev, int32_t* out_count_dev) {
  if (!c || !g) return FT_ERR_ARG;
  c->bound = false;
  if (stat < 0 || stat > 2) return fail(c, FT_ERR_ARG, "ft_eval: bad stat");
  if (!g->sky || !g->a_p || !g->P_orb || !g->tasc_frac) return fail(c, FT_ERR_ARG, "ft_eval: NULL grid axis");
  if (g->n_f0 < 1 || g->n_f1 < 1 || g->n_sky < 1 || g->n_ap < 1 || g->n_porb < 1 || g->n_tasc < 1) return fail(c, FT_ERR_ARG, "ft_eval: empty grid axis");
  const double scal[] = {g->f0_start, g->df0, g->f1_start, g->df1, g->t_ref, rho_th};
  if (!finite_all(scal, 6) || !finite_all(g->sky, 3 * (size_t)g->n_sky) || !finite_all(g->a_p, g->n_ap) ||
      !finite_all(g->P_orb, g->n_porb) || !finite_all(g->tasc_frac, g->n_tasc))
    return fail(c, FT_ERR_ARG, "ft_eval: non-finite grid value");
  if (g->n_f0 > 1 && !(g->df0 > 0.0)) return fail(c, FT_ERR_ARG, "ft_eval: df0 must be > 0");
  for (int i = 0; i < g->n_porb; ++i) if (!(g->P_orb[i] > 0.0)) return fail(c, FT_ERR_ARG, "ft_eval: P_orb must be > 0");
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
  if (!(fs_lo > 0.0) || !(eps < 0.01)) return fail(c, FT_ERR_ARG, "ft_eval: need positive frequencies and |Doppler| < 1e-2");
  const double x_lo = (fs_lo * (1.0 - eps) - c->d.f_min) / c->df, x_hi = (fs_hi * (1.0 + eps) - c->d.f_min) / c->df;
  if (x_lo < -0.49 || x_hi > (double)(c->d.n_bins - 1) + 0.49) {
    char buf[256];
    std::snprintf(buf, sizeof buf, "ft_eval: tracks may leave the spectrogram: bound [%.2f, %.2f] bins vs [0, %lld)", x_lo, x_hi, (long long)c->d.n_bins);
    return fail(c, FT_ERR_TRACK_RANGE, buf);
  }
  // copy axes
  const size_t n_ax = 3 * (size_t)g->n_sky + g->n_ap + g->n_porb + g->n_tasc;
  std::vector<double> ax(n_ax);
  std::memcpy(ax.data(), g->sky, sizeof(double) * 3 * g->n_sky);
  size_t o = 3 * (size_t)g->n_sky;
  std::memcpy(ax.data() + o, g->a_p, sizeof(double) * g->n_ap); o += g->n_ap;
  std::memcpy(ax.data() + o, g->P_orb, sizeof(double) * g->n_porb); o += g->n_porb;
  std::memcpy(ax.data() + o, g->tasc_frac, sizeof(double) * g->n_tasc);
  FT_CUDA(c, cudaStreamSynchronize(c->stream));  // previous work may still read the old axes
  if (c->axes_cap < n_ax) {
    dfree(c->axes_dev);
    c->axes_cap = 0;
    FT_CUDA(c, cudaMalloc(&c->axes_dev, sizeof(double) * n_ax));
    c->axes_cap = n_ax;
  }
  FT_CUDA(c, cudaMemcpyAsync(c->axes_dev, ax.data(), sizeof(double) * n_ax, cudaMemcpyHostToDevice, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
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
      dfree(c->ctab_dev);
      c->ctab_cap = 0; c->ctab_key.clear();
      FT_CUDA(c, cudaMalloc(&c->ctab_dev, sizeof(double) * ctab_elems));
      c->ctab_cap = ctab_elems;
    }
    if (key != c->ctab_key) {
      FT_CUDA(c, ft_launch_ctab(d, c->ctab_dev, c->stream));
      c->counters.kernel_launches += 1;
      c->ctab_key = key;
    }
    d.ctab = c->ctab_dev;
  }
  // tile-kernel eligibility and plan
  c->tile_ok = false;
  if (c->opt_kernel != 1) {
    std::string& why = c->why;
    int launches = 0;
    FtTileHostIn hin{c->t_mid.data(), c->vel.data(), g->sky, g->a_p, g->P_orb, c->df, eps, (int)c->opt_ppc, (int)c->opt_tiles};
    const cudaError_t e = ft_tile_plan(d, hin, c->stream, &c->plan, &why, &launches);
    c->counters.kernel_launches += launches;
    if (e != cudaSuccess) return fail(c, FT_ERR_CUDA, std::string("ft_tile_plan: ") + cudaGetErrorString(e));
    c->tile_ok = why.empty();
    if (!c->tile_ok && c->opt_kernel == 2) return fail(c, FT_ERR_UNSUPPORTED, "tile kernel not eligible: " + why);
  }
  // number count: the packed kernel when it is eligible (n_sft <= 65535), else the fp32 0/1 map
  c->tile8_ok = false;
  if (c->tile_ok && stat != FT_STAT_POWER && c->opt_packed) {
    std::string why8;
    int launches = 0;
    FtTileHostIn hin{c->t_mid.data(), c->vel.data(), g->sky, g->a_p, g->P_orb, c->df, eps, (int)c->opt_ppc, (int)c->opt_tiles};
    const cudaError_t e = ft_tile_plan(d, hin, c->stream, &c->plan8, &why8, &launches, 1);
    c->counters.kernel_launches += launches;
    if (e != cudaSuccess) return fail(c, FT_ERR_CUDA, std::string("ft_tile_plan (packed): ") + cudaGetErrorString(e));
    // narrow bands (< 6 chunks of 128 f0 per warp) are bound by the per-(warp, SFT) bookkeeping, which the
    // fp32 map amortises over four times as many loads: measured faster there (config 3, 450 f0)
    c->tile8_ok = why8.empty() && c->plan8.J >= 6;
  }
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
  // both statistics bound on a narrow band: one-pass kernel on QB (Q with the hit bit in the LSB)
  c->tileb_ok = false;
  if (c->tile_ok && stat == FT_STAT_BOTH && c->opt_onepass) {
    std::string whyb;
    int launches = 0;
    FtTileHostIn hin{c->t_mid.data(), c->vel.data(), g->sky, g->a_p, g->P_orb, c->df, eps, (int)c->opt_ppc, (int)c->opt_tiles};
    const cudaError_t e = ft_tile_plan(d, hin, c->stream, &c->planb, &whyb, &launches, 2);
    c->counters.kernel_launches += launches;
    if (e != cudaSuccess) return fail(c, FT_ERR_CUDA, std::string("ft_tile_plan (both): ") + cudaGetErrorString(e));
    // only where the fp32 plan itself is narrow (J <= 16): wide bands run power on K2 and the count packed
    c->tileb_ok = whyb.empty() && c->plan.J <= 16 && c->planb.n_tiles == c->plan.n_tiles;
    if (c->tileb_ok && !(c->QB_valid && c->QB_rho == d.rho)) {
      if (!c->QB_dev) FT_CUDA(c, cudaMalloc(&c->QB_dev, sizeof(float) * (size_t)d.n_sft * d.ld));
      FT_CUDA(c, ft_launch_qb(d.Q, d.P, d.rho, c->QB_dev, d.n_sft * d.ld, c->stream));
      c->counters.kernel_launches += 1;
      c->QB_rho = d.rho; c->QB_valid = true;
    }
  }
  {
    char buf[320];
    if (c->tile_ok && c->opt_kernel != 1)
      std::snprintf(buf, sizeof buf, "K2 tile kernel: J=%d wpp=%d R=%d n_tiles=%d tile_w=%d threads=%d pitch=%d copy=%d stages=%dx%d smem=%zu",
                    c->plan.J, c->plan.wpp, c->plan.R, c->plan.n_tiles, c->plan.tile_w, (c->plan.R * c->plan.wpp + 1) * 32,
                    c->plan.pitch, c->plan.copy_floats, c->plan.n_stages, c->plan.rows_per_stage, c->plan.smem_bytes);
    else
      std::snprintf(buf, sizeof buf, "K0 generic kernel (%s)", c->opt_kernel == 1 ? "forced" : c->why.c_str());
    c->desc = buf;
    if (c->tileb_ok) {
      std::snprintf(buf, sizeof buf, "; both statistics: one-pass tile kernel J=%d wpp=%d R=%d threads=%d",
                    c->planb.J, c->planb.wpp, c->planb.R, (c->planb.R * c->planb.wpp + 1) * 32);
      c->desc += buf;
    }
    if (c->tile8_ok) {
      std::snprintf(buf, sizeof buf, "; number count: packed tile kernel J=%d wpp=%d R=%d n_tiles=%d tile_w=%d threads=%d pitch=%d copy=%d stages=%dx%d",
                    c->plan8.J, c->plan8.wpp, c->plan8.R, c->plan8.n_tiles, c->plan8.tile_w, (c->plan8.R * c->plan8.wpp + 1) * 32,
                    c->plan8.pitch, c->plan8.copy_floats, c->plan8.n_stages, c->plan8.rows_per_stage);
      c->desc += buf;
    }
  }
  c->bound = true;
  if (out_power_dev || out_count_dev) {
    c->ev_used = 0; c->counters.stat_launches = 0;
    const int rc = run_stat(c, stat, 0, d.n_points, out_power_dev, out_count_dev, 0, false, 1);
    if (rc != FT_OK) return rc;
  }
  return FT_OK;
}

int ft_topk_per_band(ft_ctx* c, double band_width_hz, int32_t k, ft_cand* out_host, int32_t* n_bands_out) {
  if (!c || !out_host || !n_bands_out) return FT_ERR_ARG;
  if (!c->bound) return fail(c, FT_ERR_STATE, "ft_topk_per_band: no grid bound (call ft_eval first)");
  const FtDev& d = c->d;
  const double ratio = band_width_hz / d.df0;
  const long long bpb = std::llround(ratio);
  if (k < 1 || k > 1024 || !(band_width_hz > 0.0) || bpb < 1 || std::fabs(ratio - (double)bpb) > 1e-9 * std::fmax(1.0, ratio))
    return fail(c, FT_ERR_BAND, "ft_topk_per_band: band_width must be an integer number of f0 steps and 1 <= k <= 1024");
  const int64_t n_bands64 = (d.n_f0 + bpb - 1) / bpb;
  if (n_bands64 > (1 << 20)) return fail(c, FT_ERR_BAND, "ft_topk_per_band: too many bands");
  const int32_t n_bands = (int32_t)n_bands64;
  *n_bands_out = n_bands;
  int rc = ensure_select(c, n_bands, k);
  if (rc != FT_OK) return rc;
  const bool by_count = (c->stat == FT_STAT_HOUGH);
  // FT_STAT_BOTH ranks by power and the fp64 refinement supplies the count: select on power alone
  const int sel_stat = by_count ? FT_STAT_HOUGH : FT_STAT_POWER;
  const float margin = by_count ? 0.f : 4e-5f;  // fp32 accumulation error bound 1e-5
  const bool use_tile = c->tile_ok && c->opt_kernel != 1;
  const bool fused = use_tile && c->opt_fused;
  uint32_t* overflow = c->final_n + 1;
  FT_CUDA(c, ft_select_reset(c->sel, c->final_n, overflow, c->stream));
  c->counters.kernel_launches += 1;
  c->ev_used = 0; c->counters.stat_launches = 0;
  // Number-count veto (the loudest normalized power "with the extra restriction of
  // scoring at least a pre-established ... number count"): when both statistics are bound and a floor
  // is set, one pass of the number count over the whole bank first; the power selection then skips
  // every template below the floor.
  const int32_t floor = (c->stat == FT_STAT_BOTH) ? (int32_t)c->opt_floor : 0;
  c->sel.veto_cnt = nullptr; c->sel.veto_floor = 0;
  // narrow bands with the one-pass kernel: the count is in registers when the filter runs, no bank-wide pass
  const bool onepass_veto = floor > 0 && fused && c->tileb_ok;
  if (onepass_veto) c->sel.veto_floor = floor;
  if (floor > 0 && !onepass_veto) {
    const uint64_t n_templates = d.n_points * (uint64_t)d.n_f0;
    if (n_templates > ((uint64_t)1 << 34)) return fail(c, FT_ERR_ALLOC, "ft_topk_per_band: count floor needs 4 B per template (bank too large)");
    if (c->veto_cap < n_templates) {
      dfree(c->veto_cnt); c->veto_cap = 0;
      FT_CUDA(c, cudaMalloc(&c->veto_cnt, sizeof(int32_t) * n_templates));
      c->veto_cap = n_templates;
    }
    rc = run_stat(c, FT_STAT_HOUGH, 0, d.n_points, nullptr, c->veto_cnt, 0, false, (int32_t)bpb);
    if (rc != FT_OK) return rc;
    c->sel.veto_cnt = c->veto_cnt; c->sel.veto_floor = floor;
  }
  std::vector<uint32_t> cnt(n_bands);
  if (fused) {
    // Phase A: per-band thresholds from a strided sample of point groups (every stride-th CTA group
    // of the bank, so the sample sees every region of parameter space), written out in full.
    const FtTilePlan& spl = onepass_veto ? c->planb : ((by_count && c->tile8_ok) ? c->plan8 : c->plan);  // the plan the statistic pass runs
    const int pass_stat = onepass_veto ? (int)FT_STAT_BOTH : sel_stat;
    const bool want_i = by_count || onepass_veto, want_f = !by_count;
    const uint64_t R = (uint64_t)spl.R;
    const uint64_t n_groups = (d.n_points + R - 1) / R;
    // (a test override of the buffer capacity does not enlarge the sample: it is there to provoke overflow)
    uint64_t n_sg = (ft_tile_sample_points(spl, d.n_points, (uint32_t)k, c->opt_cap > 0 ? 65536u : c->sel.cap) + R - 1) / R;
    n_sg = n_sg < 1 ? 1 : (n_sg > n_groups ? n_groups : n_sg);
    const uint64_t stride = n_groups / n_sg;
    const int64_t rows = (int64_t)(n_sg * R);
    rc = ensure_scratch(c, (size_t)rows * d.n_f0, want_i);
    if (rc != FT_OK) return rc;
    // rows of a ragged last group are never written: make them lose every comparison
    if (want_i) FT_CUDA(c, cudaMemsetAsync(c->scratch_i, 0x80, sizeof(int32_t) * (size_t)rows * d.n_f0, c->stream));
    if (want_f) { FT_CUDA(c, ft_fill_f32(c->scratch_f, rows * d.n_f0, -INFINITY, c->stream)); c->counters.kernel_launches += 1; }
    if (stride > 1)
      rc = run_stat(c, pass_stat, 0, d.n_points, want_f ? c->scratch_f : nullptr, want_i ? c->scratch_i : nullptr,
                    0, false, (int32_t)bpb, (uint32_t)stride, n_sg);
    else
      rc = run_stat(c, pass_stat, 0, std::min<uint64_t>(d.n_points, (uint64_t)rows), want_f ? c->scratch_f : nullptr,
                    want_i ? c->scratch_i : nullptr, 0, false, (int32_t)bpb);
    if (rc != FT_OK) return rc;
    if (by_count) { FT_CUDA(c, ft_count_to_key(c->scratch_i, c->scratch_f, rows * d.n_f0, c->stream)); c->counters.kernel_launches += 1; }
    if (onepass_veto) {
      FT_CUDA(c, ft_select_mask_keys_local(c->scratch_f, c->scratch_i, rows * d.n_f0, floor, c->stream));
      c->counters.kernel_launches += 1;
    } else if (floor > 0) {
      FT_CUDA(c, ft_select_mask_keys(c->scratch_f, rows, d.n_f0, 0, (uint32_t)R, (uint32_t)stride, d.n_points, c->veto_cnt, floor, c->stream));
      c->counters.kernel_launches += 1;
    }
    FT_CUDA(c, ft_select_threshold(c->scratch_f, rows, d.n_f0, (int32_t)bpb, (uint32_t)k, margin, c->sel, c->stream));
    c->counters.kernel_launches += 1;
    // Phase B: the sample's own survivors from the scratch array, the rest of the bank through the
    // fused filter.  If a band's buffer overflows (a region far louder than the sample suggested),
    // tighten its threshold from the entries kept and repeat.
    for (int attempt = 0;; ++attempt) {
      FT_CUDA(c, ft_select_append_keys(c->scratch_f, rows, d.n_f0, (int32_t)bpb, 0, c->sel, c->stream, (uint32_t)R,
                                       (uint32_t)stride, d.n_points));
      c->counters.kernel_launches += 1;
      if (stride > 1) rc = run_stat(c, pass_stat, 0, d.n_points, nullptr, nullptr, 0, true, (int32_t)bpb, (uint32_t)stride, n_sg, true);
      else rc = run_stat(c, pass_stat, std::min<uint64_t>(d.n_points, (uint64_t)rows), d.n_points, nullptr, nullptr, 0, true, (int32_t)bpb);
      if (rc != FT_OK) return rc;
      FT_CUDA(c, cudaMemcpyAsync(cnt.data(), c->sel.cnt, sizeof(uint32_t) * n_bands, cudaMemcpyDeviceToHost, c->stream));
      FT_CUDA(c, cudaStreamSynchronize(c->stream));
      uint32_t worst = 0;
      for (uint32_t v : cnt) worst = std::max(worst, v);
      if (worst <= c->sel.cap) break;
      if (attempt == 3) return fail(c, FT_ERR_STATE, "ft_topk_per_band: a band's candidate buffer keeps overflowing (too many exact ties at the k-th value)");
      c->counters.refine_fallbacks += 1;
      FT_CUDA(c, ft_select_tighten(c->sel, (uint32_t)k, margin, c->stream));
      FT_CUDA(c, cudaMemsetAsync(c->sel.cnt, 0, sizeof(uint32_t) * n_bands, c->stream));
      c->counters.kernel_launches += 1;
    }
  } else {
    // full write-out in chunks of <= 512 MB; every chunk tightens the thresholds with its own k-th
    // largest (a valid lower bound of the band's), then appends what passes
    uint64_t chunk_pts = ((uint64_t)1 << 27) / (uint64_t)d.n_f0;
    chunk_pts = chunk_pts < 1 ? 1 : (chunk_pts > d.n_points ? d.n_points : chunk_pts);
    rc = ensure_scratch(c, (size_t)chunk_pts * d.n_f0, by_count);
    if (rc != FT_OK) return rc;
    for (uint64_t pt = 0; pt < d.n_points; pt += chunk_pts) {
      const uint64_t pe = (pt + chunk_pts < d.n_points) ? pt + chunk_pts : d.n_points;
      rc = run_stat(c, sel_stat, pt, pe, by_count ? nullptr : c->scratch_f, by_count ? c->scratch_i : nullptr,
                    pt * (uint64_t)d.n_f0, false, (int32_t)bpb);
      if (rc != FT_OK) return rc;
      const int64_t rows = (int64_t)(pe - pt);
      if (by_count) { FT_CUDA(c, ft_count_to_key(c->scratch_i, c->scratch_f, rows * d.n_f0, c->stream)); c->counters.kernel_launches += 1; }
      if (floor > 0) {
        FT_CUDA(c, ft_select_mask_keys(c->scratch_f, rows, d.n_f0, pt, 1, 1, d.n_points, c->veto_cnt, floor, c->stream));
        c->counters.kernel_launches += 1;
      }
      FT_CUDA(c, ft_select_threshold(c->scratch_f, rows, d.n_f0, (int32_t)bpb, (uint32_t)k, margin, c->sel, c->stream));
      FT_CUDA(c, ft_select_append_keys(c->scratch_f, rows, d.n_f0, (int32_t)bpb, pt, c->sel, c->stream));
      c->counters.kernel_launches += 2;
    }
  }
  FT_CUDA(c, ft_select_trim(c->sel, (uint32_t)k, margin, c->final_idx, c->final_band, c->final_n, c->final_cap, overflow, c->stream));
  FT_CUDA(c, ft_launch_refine(d, c->final_idx, c->final_n, c->final_cap, c->cand, c->near_ties_dev, c->stream));
  FT_CUDA(c, ft_select_rank(c->cand, c->final_band, c->final_n, c->final_cap, by_count ? 1 : 0, (uint32_t)k, n_bands, c->out_dev, overflow, c->stream));
  c->counters.kernel_launches += 3;
  uint32_t fin[2] = {0, 0};
  FT_CUDA(c, cudaMemcpyAsync(fin, c->final_n, sizeof fin, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(cnt.data(), c->sel.cnt, sizeof(uint32_t) * n_bands, cudaMemcpyDeviceToHost, c->stream));
  static_assert(sizeof(ft_cand) == sizeof(FtCandDev), "ft_cand layout");
  FT_CUDA(c, cudaMemcpyAsync(out_host, c->out_dev, sizeof(ft_cand) * (size_t)n_bands * k, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (int rc2 = check_tile_err(c)) return rc2;
  uint64_t appended = 0;
  for (uint32_t v : cnt) appended += v;
  c->counters.appended = appended;
  c->counters.refined = fin[0];
  if (fin[1] != 0 || fin[0] > c->final_cap) {
    char buf[200];
    std::snprintf(buf, sizeof buf, "ft_topk_per_band: candidate buffers overflowed (%u attempts in one band / %u refined): too many exact ties at the k-th value", fin[1], fin[0]);
    return fail(c, FT_ERR_STATE, buf);
  }
  return FT_OK;
}

int ft_eval_list(ft_ctx* c, const uint64_t* idx_host, int64_t n, ft_cand* out_host) {
  if (!c || !idx_host || !out_host || n < 0) return FT_ERR_ARG;
  if (!c->bound) return fail(c, FT_ERR_STATE, "ft_eval_list: no grid bound");
  if (n == 0) return FT_OK;
  const uint64_t n_templates = c->d.n_points * (uint64_t)c->d.n_f0;
  for (int64_t i = 0; i < n; ++i)
    if (idx_host[i] >= n_templates) return fail(c, FT_ERR_ARG, "ft_eval_list: index out of range");
  uint64_t* idx_dev = nullptr;
  FtCandDev* out_dev = nullptr;
  FT_CUDA(c, cudaMalloc(&idx_dev, sizeof(uint64_t) * n));
  cudaError_t e = cudaMalloc(&out_dev, sizeof(FtCandDev) * n);
  if (e == cudaSuccess) e = cudaMemcpyAsync(idx_dev, idx_host, sizeof(uint64_t) * n, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) e = ft_launch_refine(c->d, idx_dev, nullptr, n, out_dev, c->near_ties_dev, c->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(out_host, out_dev, sizeof(ft_cand) * n, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(idx_dev);
  cudaFree(out_dev);
  c->counters.kernel_launches += 1;
  if (e != cudaSuccess) return fail(c, FT_ERR_CUDA, std::string("ft_eval_list: ") + cudaGetErrorString(e));
  return FT_OK;
}

int ft_eval_templates(ft_ctx* c, const ft_template* templates_dev, int64_t n, double t_ref, int stat,
                      double rho_th, float* out_power_dev, int32_t* out_count_dev) {
  if (!c) return FT_ERR_ARG;
  if (n < 0 || (n > 0 && !templates_dev)) return fail(c, FT_ERR_ARG, "ft_eval_templates: NULL list");
  if (stat < 0 || stat > 2) return fail(c, FT_ERR_ARG, "ft_eval_templates: bad stat");
  if (!std::isfinite(t_ref) || !std::isfinite(rho_th)) return fail(c, FT_ERR_ARG, "ft_eval_templates: non-finite argument");
  if (!c->d.P) return fail(c, FT_ERR_STATE, "ft_eval_templates: handle not created");
  static_assert(sizeof(ft_template) == 64, "ft_template layout");
  if (n == 0) return FT_OK;
  int32_t* err_dev = nullptr;
  FT_CUDA(c, cudaMalloc(&err_dev, sizeof(int32_t)));
  FtDev d = c->d;
  d.rho = (float)rho_th;
  cudaError_t e = cudaMemsetAsync(err_dev, 0, sizeof(int32_t), c->stream);
  c->ev_used = 0; c->counters.stat_launches = 0;
  tick(c);
  if (e == cudaSuccess) e = ft_launch_list(d, stat, templates_dev, n, t_ref, out_power_dev, out_count_dev, err_dev,
                                           c->near_ties_dev, c->stream);
  tock(c, 1);
  int32_t flag = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&flag, err_dev, sizeof flag, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(err_dev);
  if (e != cudaSuccess) return fail(c, FT_ERR_CUDA, std::string("ft_eval_templates: ") + cudaGetErrorString(e));
  if (flag) return fail(c, FT_ERR_TRACK_RANGE, "ft_eval_templates: some tracks leave the spectrogram (their outputs are NaN / -1)");
  return FT_OK;
}

int ft_get_counters(ft_ctx* c, ft_counters* out) {
  if (!c || !out) return FT_ERR_ARG;
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (int rc2 = check_tile_err(c)) return rc2;
  unsigned long long nt = 0;
  FT_CUDA(c, cudaMemcpy(&nt, c->near_ties_dev, sizeof nt, cudaMemcpyDeviceToHost));
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
  cudaStreamSynchronize(c->stream);
  free_select(c);
  ft_tile_plan_free(&c->plan);
  ft_tile_plan_free(&c->plan8);
  ft_tile_plan_free(&c->planb);
  dfree(c->H8_dev); dfree(c->QB_dev);
  dfree(c->t_mid_dev); dfree(c->vel_dev); dfree(c->w_dev); dfree(c->Q_dev); dfree(c->H_dev); dfree(c->ctab_dev); dfree(c->axes_dev);
  dfree(c->scratch_f); dfree(c->scratch_i); dfree(c->veto_cnt); dfree(c->near_ties_dev);
  for (cudaEvent_t e : c->evs) cudaEventDestroy(e);
  delete c;
}

}  // extern "C"
