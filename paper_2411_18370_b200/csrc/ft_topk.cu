// ft_topk_per_band / ft_topk_per_box: orchestration of the per-region selection (PAPER.md:330-351, :476,
// :496-502).  DESIGN.md "Selection".
//
// Regions = (box of outer points) x (frequency sub-band).  Phase A evaluates a sample of CTA groups (one wave
// of the tile kernel, spread over the bank, plus enough rows of every box of points), written out in full;
// its k-th largest key per region is a lower bound of the region's k-th value, hence a valid threshold.  Phase B
// runs the rest of the bank through the tile kernel's fused filter (keys >= threshold are appended).  The
// appended keys are trimmed to those within the fp32 margin of the region's k-th largest, re-evaluated in fp64
// with the canonical arithmetic, and ranked exactly under (value desc, idx asc).
#include <algorithm>

#include "ft_ctx.cuh"

namespace {

void free_select(ft_ctx* c) {
  ft_dfree(c->sel.thr); ft_dfree(c->sel.cnt); ft_dfree(c->sel.key); ft_dfree(c->sel.idx);
  ft_dfree(c->final_idx); ft_dfree(c->final_region); ft_dfree(c->final_n); ft_dfree(c->cand); ft_dfree(c->out_dev);
  c->sel = FtSelectDev{};
  c->final_cap = 0; c->out_cap = 0;
}

int ensure_select(ft_ctx* c, int32_t n_regions, int32_t k) {
  uint32_t cap = (uint32_t)((1u << 24) / (uint32_t)n_regions);
  cap = cap > 65536u ? 65536u : (cap < 1024u ? 1024u : cap);
  if (c->opt_cap > 0) cap = (uint32_t)c->opt_cap;  // FT_OPT_SELECT_CAP (tests of the overflow recovery)
  cap = std::max(cap, 2u * (uint32_t)k);           // a buffer must at least hold the k it is asked for
  const uint32_t final_cap = (uint32_t)std::min<uint64_t>((uint64_t)n_regions * 2048u, 1u << 26);
  if (c->sel.n_regions != n_regions || c->sel.cap != cap || c->out_cap < (size_t)n_regions * k) {
    free_select(c);
    FT_CUDA(c, cudaMalloc(&c->sel.thr, sizeof(float) * n_regions));
    FT_CUDA(c, cudaMalloc(&c->sel.cnt, sizeof(uint32_t) * n_regions));
    FT_CUDA(c, cudaMalloc(&c->sel.key, sizeof(float) * (size_t)n_regions * cap));
    FT_CUDA(c, cudaMalloc(&c->sel.idx, sizeof(uint64_t) * (size_t)n_regions * cap));
    c->sel.cap = cap; c->sel.n_regions = n_regions;
    FT_CUDA(c, cudaMalloc(&c->final_idx, sizeof(uint64_t) * final_cap));
    FT_CUDA(c, cudaMalloc(&c->final_region, sizeof(int32_t) * final_cap));
    FT_CUDA(c, cudaMalloc(&c->final_n, sizeof(uint32_t) * 2));
    FT_CUDA(c, cudaMalloc(&c->cand, sizeof(FtCandDev) * final_cap));
    FT_CUDA(c, cudaMalloc(&c->out_dev, sizeof(FtCandDev) * (size_t)n_regions * k));
    c->final_cap = final_cap; c->out_cap = (size_t)n_regions * k;
  }
  return FT_OK;
}

int ensure_scratch(ft_ctx* c, size_t elems, bool need_int) {
  if (c->scratch_elems < elems) {
    ft_dfree(c->scratch_f); ft_dfree(c->scratch_i);
    c->scratch_elems = 0;
    FT_CUDA(c, cudaMalloc(&c->scratch_f, sizeof(float) * elems));
    c->scratch_elems = elems;
  }
  if (need_int && !c->scratch_i) FT_CUDA(c, cudaMalloc(&c->scratch_i, sizeof(int32_t) * c->scratch_elems));
  return FT_OK;
}

struct TopkSpec {
  const int32_t* pbox_host;
  int32_t n_pbox;
  double band_width_hz;
  int32_t k;
  int rank_by_z;
};

// CSR of the rows of a key array by box of points: row_start[n_pbox + 1], rows[n_rows]
void rows_by_pbox(const int32_t* pbox, int32_t n_pbox, const std::vector<uint64_t>& row_pt, uint64_t n_points,
                  std::vector<uint32_t>* row_start, std::vector<uint32_t>* rows) {
  row_start->assign((size_t)n_pbox + 1, 0u);
  for (uint64_t pt : row_pt)
    if (pt < n_points) (*row_start)[(size_t)pbox[pt] + 1] += 1u;
  for (int32_t b = 0; b < n_pbox; ++b) (*row_start)[(size_t)b + 1] += (*row_start)[(size_t)b];
  rows->assign(row_start->back(), 0u);
  std::vector<uint32_t> fill(row_start->begin(), row_start->end() - 1);
  for (size_t r = 0; r < row_pt.size(); ++r)
    if (row_pt[r] < n_points) (*rows)[fill[(size_t)pbox[row_pt[r]]]++] = (uint32_t)r;
}

int topk_regions(ft_ctx* c, const TopkSpec& sp, std::vector<FtCandDev>* out, int32_t* n_regions_out) {
  if (!c->bound) return ft_fail(c, FT_ERR_STATE, "top-k: no grid bound (call ft_eval first)");
  if (int rc = ft_enter(c)) return rc;
  const FtDev& d = c->d;
  const int32_t k = sp.k;
  long long bpb = 1;
  if (d.n_f0 > 1) {
    const double ratio = sp.band_width_hz / d.df0;
    bpb = std::isfinite(ratio) ? std::llround(ratio) : 0;
    if (!(sp.band_width_hz > 0.0) || bpb < 1 || std::fabs(ratio - (double)bpb) > 1e-9 * std::fmax(1.0, ratio))
      return ft_fail(c, FT_ERR_BAND, "top-k: band_width must be an integer number of f0 steps");
  } else if (!(sp.band_width_hz > 0.0)) {
    return ft_fail(c, FT_ERR_BAND, "top-k: band_width must be > 0");
  }
  if (k < 1 || k > 1024) return ft_fail(c, FT_ERR_BAND, "top-k: 1 <= k <= 1024");
  if (bpb > d.n_f0) bpb = d.n_f0;
  const int64_t n_bands64 = (d.n_f0 + bpb - 1) / bpb;
  const int32_t n_pbox = sp.pbox_host ? sp.n_pbox : 1;
  if (n_pbox < 1) return ft_fail(c, FT_ERR_ARG, "top-k: n_pbox >= 1");
  if (n_bands64 * (int64_t)n_pbox > (1 << 20)) return ft_fail(c, FT_ERR_BAND, "top-k: too many regions (> 2^20)");
  const int32_t n_bands = (int32_t)n_bands64, n_regions = n_bands * n_pbox;
  *n_regions_out = n_regions;
  if (d.n_points > 0xffffffffull && sp.pbox_host) return ft_fail(c, FT_ERR_ARG, "top-k: boxes of points need n_points < 2^32");
  const int32_t* pbox_dev = nullptr;
  if (sp.pbox_host) {
    for (uint64_t i = 0; i < d.n_points; ++i)
      if (sp.pbox_host[i] < 0 || sp.pbox_host[i] >= n_pbox) return ft_fail(c, FT_ERR_ARG, "top-k: pbox value out of [0, n_pbox)");
    FT_CUDA(c, cudaStreamSynchronize(c->stream));
    FT_CUDA(c, ft_grow(c->pbox_dev, c->pbox_cap, (size_t)d.n_points));
    FT_CUDA(c, cudaMemcpyAsync(c->pbox_dev, sp.pbox_host, sizeof(int32_t) * d.n_points, cudaMemcpyHostToDevice, c->stream));
    pbox_dev = c->pbox_dev;
  }
  int rc = ensure_select(c, n_regions, k);
  if (rc != FT_OK) return rc;
  // ---- what ranks, what vetoes ---------------------------------------------------------------------------
  const bool by_count = c->stat == FT_STAT_HOUGH, by_wcount = c->stat == FT_STAT_WHOUGH;
  const int zmode = sp.rank_by_z ? 1 : 0;
  if (zmode && (by_count || by_wcount)) return ft_fail(c, FT_ERR_ARG, "top-k: ranking by z needs the power statistic bound (FT_STAT_POWER / FT_STAT_BOTH)");
  if (zmode && !(d.sigma_G > 0.0)) return ft_fail(c, FT_ERR_ARG, "top-k: sigma_G = 0 (all weights zero)");
  // FT_STAT_BOTH ranks by power and the fp64 refinement supplies the count: select on power alone
  const int sel_stat = by_count ? FT_STAT_HOUGH : by_wcount ? FT_STAT_WHOUGH : FT_STAT_POWER;
  const int rank_by = by_count ? FT_RANK_COUNT : by_wcount ? FT_RANK_WCOUNT : zmode ? FT_RANK_Z : FT_RANK_POWER;
  // fp32 accumulation error bound 1e-5 relative to the statistic; standardised keys carry
  // it as (|z| + mu/sigma) (sky-dependent weights: sigma >= 1/sqrt(n_sft))
  FtMargin margin{by_count ? 0.f : 4e-5f, 0.f};
  if (zmode) margin.shift = (float)(d.skyw ? std::sqrt((double)d.n_sft) : d.mu_G / d.sigma_G);
  const bool use_tile = c->tile_ok && c->opt_kernel != 1;
  const bool fused = use_tile && c->opt_fused;
  uint32_t* overflow = c->final_n + 1;
  FT_CUDA(c, ft_select_reset(c->sel, c->final_n, overflow, c->stream));
  c->counters.kernel_launches += 1;
  c->ev_used = 0; c->counters.stat_launches = 0;
  // Number-count veto (the loudest normalized power "with the extra restriction of scoring at
  // least a pre-established weighted number count value"): when both statistics are bound and a floor is set,
  // one pass of the (weighted) number count over the whole bank first; the power selection then skips every
  // template below the floor.  Narrow bands with the one-pass kernel have the integer count in registers.
  const int32_t floor = (c->stat == FT_STAT_BOTH) ? (int32_t)c->opt_floor : 0;
  const double wfloor = (c->stat == FT_STAT_BOTH) ? c->opt_wfloor : 0.0;
  c->sel.veto_cnt = nullptr; c->sel.veto_floor = 0; c->sel.veto_w = nullptr; c->sel.veto_wlo = c->sel.veto_whi = 0.f;
  const bool onepass_veto = floor > 0 && fused && c->tileb_ok;
  if (onepass_veto) c->sel.veto_floor = floor;
  const uint64_t n_templates = d.n_points * (uint64_t)d.n_f0;
  const int rank_by_v = by_count ? FT_RANK_COUNT : by_wcount ? FT_RANK_WCOUNT : zmode ? FT_RANK_Z : FT_RANK_POWER;
  bool by_survivors = false;   // veto-first: the selection was made from the survivors of the number-count pass
  if ((floor > 0 && !onepass_veto) || wfloor > 0.0) {
    if (n_templates > ((uint64_t)1 << 34)) return ft_fail(c, FT_ERR_ALLOC, "top-k: a number-count floor needs 4 B per template (bank too large)");
    // Veto first (FT_OPT_VETO_FIRST, default on, fused selection): the LAST number-count pass also runs the fused filter
    // with the floor as the threshold of every region.  A floor of mu + 3 sigma leaves ~1e-3 of a noise bank: if the
    // survivors fit the append buffers, only they are evaluated for power (fp64, the refinement kernel) and the
    // bank-wide power pass is not needed.  Otherwise the pass has still written the veto array and the selection goes
    // on as before (power pass with the array looked up by the fused filter).
    const bool try_first = fused && c->opt_veto_first;
    FtPass p;
    p.pt_begin = 0; p.pt_end = d.n_points;
    p.bpb = (int32_t)bpb; p.n_bands = n_bands; p.pbox = pbox_dev;
    if (floor > 0 && !onepass_veto) {
      FT_CUDA(c, ft_grow(c->veto_cnt, c->veto_cap, (size_t)n_templates));
      p.stat = FT_STAT_HOUGH; p.out_i = c->veto_cnt; p.out_f = nullptr;
      p.filter = try_first && !(wfloor > 0.0);
      if (p.filter) { FT_CUDA(c, ft_fill_f32(c->sel.thr, n_regions, (float)floor, c->stream)); c->counters.kernel_launches += 1; }
      if ((rc = ft_run_stat(c, p)) != FT_OK) return rc;
      c->sel.veto_cnt = c->veto_cnt; c->sel.veto_floor = floor;
    }
    if (wfloor > 0.0) {
      FT_CUDA(c, ft_grow(c->veto_w, c->vetow_cap, (size_t)n_templates));
      p.stat = FT_STAT_WHOUGH; p.out_f = c->veto_w; p.out_i = nullptr;
      // the fp32 weighted count decides only outside a 4e-5 band around the floor; inside, the fp64 refinement does
      const float wlo = (float)(wfloor * (1.0 - 4e-5)), whi = (float)(wfloor * (1.0 + 4e-5));
      p.filter = try_first;
      if (p.filter) { FT_CUDA(c, ft_fill_f32(c->sel.thr, n_regions, wlo, c->stream)); c->counters.kernel_launches += 1; }
      if ((rc = ft_run_stat(c, p)) != FT_OK) return rc;   // (an integer floor set above is applied by the filter: that pass is complete)
      c->sel.veto_w = c->veto_w;
      c->sel.veto_wlo = wlo; c->sel.veto_whi = whi;
    }
    if (try_first) {
      std::vector<uint32_t> cnt0(n_regions);
      FT_CUDA(c, cudaMemcpyAsync(cnt0.data(), c->sel.cnt, sizeof(uint32_t) * n_regions, cudaMemcpyDeviceToHost, c->stream));
      FT_CUDA(c, cudaStreamSynchronize(c->stream));
      std::vector<uint32_t> off((size_t)n_regions + 1, 0u);
      uint64_t total = 0;
      bool fits = true;
      for (int32_t b = 0; b < n_regions; ++b) { fits = fits && cnt0[b] <= c->sel.cap; total += cnt0[b]; off[(size_t)b + 1] = (uint32_t)std::min<uint64_t>(total, 0xffffffffu); }
      if (fits && total < ((uint64_t)1 << 26)) {
        by_survivors = true;
        c->counters.appended = total;
        // survivors: list | refined records | region offsets (grow-only)
        const size_t need = sizeof(uint64_t) * (size_t)total + sizeof(FtCandDev) * (size_t)total + sizeof(uint32_t) * off.size() + 64;
        FT_CUDA(c, ft_grow(c->surv_dev, c->surv_cap, need));
        FtCandDev* s_cand = reinterpret_cast<FtCandDev*>(c->surv_dev);
        uint64_t* s_idx = reinterpret_cast<uint64_t*>(s_cand + total);
        uint32_t* s_off = reinterpret_cast<uint32_t*>(s_idx + total);
        FT_CUDA(c, cudaMemcpyAsync(s_off, off.data(), sizeof(uint32_t) * off.size(), cudaMemcpyHostToDevice, c->stream));
        if (total > 0) {
          FT_CUDA(c, ft_select_take_all(c->sel, s_off, s_idx, c->stream));
          FT_CUDA(c, ft_launch_refine(d, s_idx, nullptr, (int64_t)total, s_cand, c->near_ties_dev, c->stream));
        }
        FT_CUDA(c, ft_select_trim_refined(s_cand, s_off, n_regions, rank_by_v, (uint32_t)k, floor, wfloor, c->cand, c->final_region,
                                          c->final_n, c->final_cap, c->stream));
        FT_CUDA(c, ft_select_rank(c->cand, c->final_region, c->final_n, c->final_cap, rank_by_v, (uint32_t)k, n_regions, floor,
                                  wfloor, c->out_dev, overflow, c->stream));
        c->counters.kernel_launches += 4;
        FT_CUDA(c, cudaStreamSynchronize(c->stream));   // (off is a local: the upload must have completed)
      } else {
        // too many survivors for the buffers: thresholds and counters back to the start, the veto arrays stay
        FT_CUDA(c, ft_select_reset(c->sel, c->final_n, overflow, c->stream));
        c->counters.kernel_launches += 1;
      }
    }
  }
  const int pass_stat = onepass_veto ? (int)FT_STAT_BOTH : sel_stat;
  std::vector<uint32_t> cnt(n_regions);
  FtRowMap map{};
  map.pbox = pbox_dev; map.n_bands = n_bands; map.bpb = (int32_t)bpb; map.n_pbox = n_pbox; map.pt_end = d.n_points;
  if (by_survivors) {
    // (selection complete: only the copies to the host remain)
  } else if (fused) {
    // ---- Phase A: thresholds from a sample of CTA groups --------------------------------------------------
    const FtTilePlan& spl = pass_stat == FT_STAT_BOTH ? c->planb : (by_count && c->tile8_ok) ? c->plan8
                          : d.skyw ? c->planw : c->plan;   // the plan the statistic pass runs
    const bool want_i = by_count || onepass_veto, want_f = !by_count;
    const uint64_t R = (uint64_t)spl.R;
    const uint64_t n_groups = (d.n_points + R - 1) / R;
    // (a test override of the buffer capacity does not enlarge the sample: it is there to provoke overflow)
    uint64_t n_sg = (ft_tile_sample_points(spl, d.n_points, (uint32_t)k, c->opt_cap > 0 ? 65536u : c->sel.cap) + R - 1) / R;
    n_sg = n_sg < 1 ? 1 : (n_sg > n_groups ? n_groups : n_sg);
    const uint64_t stride = n_groups / n_sg;
    std::vector<uint32_t> glist;
    std::vector<bool> in_sample((size_t)n_groups, false);
    for (uint64_t i = 0; i < n_sg; ++i) { glist.push_back((uint32_t)(i * stride)); in_sample[(size_t)(i * stride)] = true; }
    if (sp.pbox_host) {
      // every box of points needs enough sampled rows for k keys per region
      const int64_t bw_min = std::min<int64_t>(bpb, d.n_f0 - (int64_t)(n_bands - 1) * bpb);
      const uint32_t need = (uint32_t)((k + bw_min - 1) / bw_min);
      std::vector<uint32_t> have((size_t)n_pbox, 0u);
      for (uint32_t g : glist)
        for (uint64_t pt = (uint64_t)g * R; pt < std::min<uint64_t>(d.n_points, ((uint64_t)g + 1) * R); ++pt) have[(size_t)sp.pbox_host[pt]] += 1u;
      bool short_any = false;
      for (uint32_t h : have) short_any |= h < need;
      if (short_any)
        for (uint64_t pt = 0; pt < d.n_points; ++pt) {
          const int32_t b = sp.pbox_host[pt];
          const uint64_t g = pt / R;
          if (have[(size_t)b] >= need || in_sample[(size_t)g]) continue;
          in_sample[(size_t)g] = true;
          glist.push_back((uint32_t)g);
          for (uint64_t q = g * R; q < std::min<uint64_t>(d.n_points, (g + 1) * R); ++q) have[(size_t)sp.pbox_host[q]] += 1u;
        }
    }
    const uint32_t n_list = (uint32_t)glist.size();
    std::vector<uint32_t> glist_sorted(glist);
    std::sort(glist_sorted.begin(), glist_sorted.end());
    const int64_t rows = (int64_t)n_list * (int64_t)R;
    // one upload: group list | skip bitmask | row_start | rows
    const size_t n_words = ((size_t)n_groups + 31) / 32;
    std::vector<uint32_t> up(glist);
    up.resize((size_t)n_list + n_words, 0u);
    for (uint32_t g : glist) up[(size_t)n_list + (g >> 5)] |= 1u << (g & 31);
    size_t off_rs = 0, off_rows = 0;
    if (sp.pbox_host) {
      std::vector<uint64_t> row_pt((size_t)rows);
      for (int64_t r = 0; r < rows; ++r) row_pt[(size_t)r] = (uint64_t)glist[(size_t)(r / (int64_t)R)] * R + (uint64_t)(r % (int64_t)R);
      std::vector<uint32_t> rs, rw;
      rows_by_pbox(sp.pbox_host, n_pbox, row_pt, d.n_points, &rs, &rw);
      off_rs = up.size(); up.insert(up.end(), rs.begin(), rs.end());
      off_rows = up.size(); up.insert(up.end(), rw.begin(), rw.end());
    }
    if (c->glist_cap < up.size()) FT_CUDA(c, cudaStreamSynchronize(c->stream));   // (about to free lists that may still be read)
    FT_CUDA(c, ft_grow(c->glist_dev, c->glist_cap, up.size()));
    FT_CUDA(c, cudaMemcpyAsync(c->glist_dev, up.data(), sizeof(uint32_t) * up.size(), cudaMemcpyHostToDevice, c->stream));
    const uint32_t* glist_dev = c->glist_dev;
    const uint32_t* gskip_dev = c->glist_dev + n_list;
    map.glist = glist_dev; map.R = (uint32_t)R; map.pt_begin = 0;
    if (sp.pbox_host) { map.row_start = c->glist_dev + off_rs; map.rows = c->glist_dev + off_rows; }
    rc = ensure_scratch(c, (size_t)rows * d.n_f0, want_i);
    if (rc != FT_OK) return rc;
    // rows of a ragged last group are never written: make them lose every comparison
    if (want_i) FT_CUDA(c, cudaMemsetAsync(c->scratch_i, 0x80, sizeof(int32_t) * (size_t)rows * d.n_f0, c->stream));
    if (want_f) { FT_CUDA(c, ft_fill_f32(c->scratch_f, rows * d.n_f0, -INFINITY, c->stream)); c->counters.kernel_launches += 1; }
    FtPass p;
    p.stat = pass_stat; p.pt_begin = 0; p.pt_end = d.n_points;
    p.out_f = want_f ? c->scratch_f : nullptr; p.out_i = want_i ? c->scratch_i : nullptr;
    p.bpb = (int32_t)bpb; p.n_bands = n_bands; p.pbox = pbox_dev; p.zmode = zmode; p.out_key = zmode;
    p.glist = glist_dev; p.n_glist = n_list;
    if ((rc = ft_run_stat(c, p)) != FT_OK) return rc;
    if (by_count) { FT_CUDA(c, ft_count_to_key(c->scratch_i, c->scratch_f, rows * d.n_f0, c->stream)); c->counters.kernel_launches += 1; }
    if (onepass_veto) {
      FT_CUDA(c, ft_select_mask_keys_local(c->scratch_f, c->scratch_i, rows * d.n_f0, floor, c->stream));
      c->counters.kernel_launches += 1;
    }
    FT_CUDA(c, ft_select_threshold(c->scratch_f, rows, d.n_f0, map, (uint32_t)k, margin, c->sel, c->stream));
    c->counters.kernel_launches += 1;
    // ---- Phase B: the sample's own survivors from the scratch array, the rest of the bank through the fused
    // filter.  If a region's buffer overflows (a region far louder than the sample suggested), tighten its
    // threshold from the entries kept and repeat.
    for (int attempt = 0;; ++attempt) {
      FT_CUDA(c, ft_select_append_keys(c->scratch_f, rows, d.n_f0, map, c->sel, c->stream));
      c->counters.kernel_launches += 1;
      if ((uint64_t)n_list < n_groups) {
        FtPass pb = p;
        pb.out_f = nullptr; pb.out_i = nullptr; pb.filter = true; pb.glist = nullptr; pb.n_glist = 0; pb.gskip = gskip_dev; pb.out_key = 0;
        pb.skip_host = glist_sorted.data(); pb.n_skip_host = (uint32_t)glist_sorted.size();
        if ((rc = ft_run_stat(c, pb)) != FT_OK) return rc;
      }
      FT_CUDA(c, cudaMemcpyAsync(cnt.data(), c->sel.cnt, sizeof(uint32_t) * n_regions, cudaMemcpyDeviceToHost, c->stream));
      FT_CUDA(c, cudaStreamSynchronize(c->stream));
      uint32_t worst = 0;
      for (uint32_t v : cnt) worst = std::max(worst, v);
      if (worst <= c->sel.cap) break;
      if (attempt == 3) return ft_fail(c, FT_ERR_STATE, "top-k: a region's candidate buffer keeps overflowing (too many exact ties at the k-th value)");
      c->counters.refine_fallbacks += 1;
      FT_CUDA(c, ft_select_tighten(c->sel, (uint32_t)k, margin, c->stream));
      FT_CUDA(c, cudaMemsetAsync(c->sel.cnt, 0, sizeof(uint32_t) * n_regions, c->stream));
      c->counters.kernel_launches += 1;
    }
  } else {
    // full write-out in chunks of <= 512 MB; every chunk tightens the thresholds with its own k-th
    // largest (a valid lower bound of the region's), then appends what passes
    uint64_t chunk_pts = ((uint64_t)1 << 27) / (uint64_t)d.n_f0;
    chunk_pts = chunk_pts < 1 ? 1 : (chunk_pts > d.n_points ? d.n_points : chunk_pts);
    rc = ensure_scratch(c, (size_t)chunk_pts * d.n_f0, by_count);
    if (rc != FT_OK) return rc;
    for (uint64_t pt = 0; pt < d.n_points; pt += chunk_pts) {
      const uint64_t pe = (pt + chunk_pts < d.n_points) ? pt + chunk_pts : d.n_points;
      const int64_t rows = (int64_t)(pe - pt);
      FtPass p;
      p.stat = sel_stat; p.pt_begin = pt; p.pt_end = pe;
      p.out_f = by_count ? nullptr : c->scratch_f; p.out_i = by_count ? c->scratch_i : nullptr;
      p.out_base = pt * (uint64_t)d.n_f0;
      p.bpb = (int32_t)bpb; p.n_bands = n_bands; p.pbox = pbox_dev; p.zmode = zmode; p.out_key = zmode;
      if ((rc = ft_run_stat(c, p)) != FT_OK) return rc;
      if (by_count) { FT_CUDA(c, ft_count_to_key(c->scratch_i, c->scratch_f, rows * d.n_f0, c->stream)); c->counters.kernel_launches += 1; }
      map.glist = nullptr; map.R = 1; map.pt_begin = pt;
      if (sp.pbox_host) {
        std::vector<uint64_t> row_pt((size_t)rows);
        for (int64_t r = 0; r < rows; ++r) row_pt[(size_t)r] = pt + (uint64_t)r;
        std::vector<uint32_t> rs, rw;
        rows_by_pbox(sp.pbox_host, n_pbox, row_pt, d.n_points, &rs, &rw);
        rs.insert(rs.end(), rw.begin(), rw.end());
        FT_CUDA(c, cudaStreamSynchronize(c->stream));
        FT_CUDA(c, ft_grow(c->glist_dev, c->glist_cap, rs.size()));
        FT_CUDA(c, cudaMemcpy(c->glist_dev, rs.data(), sizeof(uint32_t) * rs.size(), cudaMemcpyHostToDevice));
        map.row_start = c->glist_dev; map.rows = c->glist_dev + n_pbox + 1;
      }
      FT_CUDA(c, ft_select_threshold(c->scratch_f, rows, d.n_f0, map, (uint32_t)k, margin, c->sel, c->stream));
      FT_CUDA(c, ft_select_append_keys(c->scratch_f, rows, d.n_f0, map, c->sel, c->stream));
      c->counters.kernel_launches += 2;
    }
  }
  if (!by_survivors) {
    FT_CUDA(c, ft_select_trim(c->sel, (uint32_t)k, margin, c->final_idx, c->final_region, c->final_n, c->final_cap, overflow, c->stream));
    FT_CUDA(c, ft_launch_refine(d, c->final_idx, c->final_n, c->final_cap, c->cand, c->near_ties_dev, c->stream));
    FT_CUDA(c, ft_select_rank(c->cand, c->final_region, c->final_n, c->final_cap, rank_by, (uint32_t)k, n_regions, floor,
                              wfloor, c->out_dev, overflow, c->stream));
    c->counters.kernel_launches += 3;
  }
  uint32_t fin[2] = {0, 0};
  int32_t terr = 0;
  out->resize((size_t)n_regions * k);
  FT_CUDA(c, cudaMemcpyAsync(fin, c->final_n, sizeof fin, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(&terr, c->tile_err_dev, sizeof terr, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(cnt.data(), c->sel.cnt, sizeof(uint32_t) * n_regions, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(out->data(), c->out_dev, sizeof(FtCandDev) * (size_t)n_regions * k, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (int rc2 = ft_tile_err_status(c, terr)) return rc2;
  if (!by_survivors) {
    uint64_t appended = 0;
    for (uint32_t v : cnt) appended += v;
    c->counters.appended = appended;
  }
  c->counters.refined = by_survivors ? c->counters.appended : fin[0];
  if (fin[1] != 0 || fin[0] > c->final_cap) {
    char buf[200];
    std::snprintf(buf, sizeof buf, "top-k: candidate buffers overflowed (%u attempts in one region / %u refined): too many exact ties at the k-th value", fin[1], fin[0]);
    return ft_fail(c, FT_ERR_STATE, buf);
  }
  return FT_OK;
}

}  // namespace

extern "C" {

int ft_topk_per_band(ft_ctx* c, double band_width_hz, int32_t k, ft_cand* out_host, int32_t* n_bands_out) {
  if (!c || !out_host || !n_bands_out) return FT_ERR_ARG;
  std::vector<FtCandDev> tmp;
  const int rc = topk_regions(c, TopkSpec{nullptr, 1, band_width_hz, k, 0}, &tmp, n_bands_out);
  if (rc != FT_OK) return rc;
  for (size_t i = 0; i < tmp.size(); ++i) out_host[i] = ft_cand{tmp[i].power, tmp[i].wcount, tmp[i].idx, tmp[i].count, tmp[i].band};
  return FT_OK;
}

int ft_topk_per_box(ft_ctx* c, const int32_t* pbox_host, int32_t n_pbox, double band_width_hz, int32_t k, int rank_by_z,
                    ft_cand_box* out_host, int32_t* n_regions_out) {
  if (!c || !out_host || !n_regions_out) return FT_ERR_ARG;
  static_assert(sizeof(ft_cand_box) == sizeof(FtCandDev), "ft_cand_box layout");
  std::vector<FtCandDev> tmp;
  const int rc = topk_regions(c, TopkSpec{pbox_host, n_pbox, band_width_hz, k, rank_by_z}, &tmp, n_regions_out);
  if (rc != FT_OK) return rc;
  std::memcpy(out_host, tmp.data(), sizeof(FtCandDev) * tmp.size());
  return FT_OK;
}

}  // extern "C"
