// Per-region candidate buffers shared by the statistic kernels (fused filter) and ft_select.cu.
// A region is a frequency sub-band (north_star) or a box = (block of outer points) x (sub-band), the regular
// hyperboxes of PAPER.md:338-342: region = pbox[pt] * n_bands + i_f0 / bins_per_band.
#pragma once
#include "ft_common.cuh"

struct FtSelectDev {
  float* thr;      // [n_regions] current fp32 threshold (with margin); -inf = accept everything
  uint32_t* cnt;   // [n_regions] number of append attempts (may exceed cap: overflow)
  float* key;      // [n_regions][cap]
  uint64_t* idx;   // [n_regions][cap]
  uint32_t cap;
  int32_t n_regions;
  // number-count veto: templates below the floor are not candidates.  Integer count:
  // veto_cnt[idx] < veto_floor.  Weighted count (fp32 array, accumulated in fp32): below veto_wlo = certainly
  // vetoed; in [veto_wlo, veto_whi) = decided by the fp64 refinement; the fused filter admits >= veto_wlo.
  const int32_t* veto_cnt;  // [n_templates] or nullptr
  int32_t veto_floor;
  const float* veto_w;      // [n_templates] or nullptr
  float veto_wlo, veto_whi;
};

// Certainly passes the veto (only such templates may raise a threshold; the uncertain ones are admitted by
// ft_select_append and decided by the fp64 refinement).
__device__ __forceinline__ bool ft_select_sure(const FtSelectDev& sel, uint64_t idx) {
  if (sel.veto_cnt && __ldg(sel.veto_cnt + idx) < sel.veto_floor) return false;
  if (sel.veto_w && __ldg(sel.veto_w + idx) < sel.veto_whi) return false;
  return true;
}

__device__ __forceinline__ void ft_select_append(const FtSelectDev& sel, int region, float key, uint64_t idx) {
  if (sel.veto_cnt && __ldg(sel.veto_cnt + idx) < sel.veto_floor) return;
  if (sel.veto_w && __ldg(sel.veto_w + idx) < sel.veto_wlo) return;
  const uint32_t slot = atomicAdd(sel.cnt + region, 1u);
  if (slot < sel.cap) {
    sel.key[(size_t)region * sel.cap + slot] = key;
    sel.idx[(size_t)region * sel.cap + slot] = idx;
  }
}

// fp32 margin of a key: tau - rel * (|tau| + shift)   (shift = mu_G / sigma_G when the keys are standardised)
struct FtMargin { float rel, shift; };

// How the rows of a [n_rows][n_f0] key array map to outer points and regions.
struct FtRowMap {
  uint64_t pt_begin;          // glist == nullptr: row r is point pt_begin + r
  const uint32_t* glist;      // else: row r is point glist[r / R] * R + r % R   (the threshold sample's CTA groups)
  uint32_t R;
  uint64_t pt_end;            // rows mapping to points >= pt_end hold no data
  const int32_t* pbox;        // [n_points] point -> box of points, or nullptr (one box)
  int32_t n_bands, bpb;
  // rows of each point-box, for the per-region threshold (pbox != nullptr): rows[row_start[b] .. row_start[b+1])
  const uint32_t* row_start;
  const uint32_t* rows;
  int32_t n_pbox;
};

enum FtRankBy { FT_RANK_POWER = 0, FT_RANK_COUNT = 1, FT_RANK_WCOUNT = 2, FT_RANK_Z = 3 };

cudaError_t ft_select_reset(FtSelectDev sel, uint32_t* final_n, uint32_t* overflow, cudaStream_t s);
cudaError_t ft_select_threshold(const float* keys, int64_t n_rows, int64_t n_f0, const FtRowMap& map, uint32_t k,
                                FtMargin margin, FtSelectDev sel, cudaStream_t s);
cudaError_t ft_select_append_keys(const float* keys, int64_t n_rows, int64_t n_f0, const FtRowMap& map,
                                  FtSelectDev sel, cudaStream_t s);
cudaError_t ft_select_trim(FtSelectDev sel, uint32_t k, FtMargin margin, uint64_t* final_idx,
                           int32_t* final_region, uint32_t* final_n, uint32_t final_cap,
                           uint32_t* overflow, cudaStream_t s);
// exact veto applied on the refined values: count >= count_floor and wcount >= wcount_floor
cudaError_t ft_select_rank(const FtCandDev* cand, const int32_t* cand_region, const uint32_t* n_dev,
                           uint32_t cap, int rank_by, uint32_t k, int32_t n_regions, int32_t count_floor,
                           double wcount_floor, FtCandDev* out, uint32_t* overflow, cudaStream_t s);
// veto-first selection: all appended entries compacted by region (off [n_regions + 1], device); then, on the refined
// values, the candidates of each region that pass the floors and reach its k-th largest ranking value
cudaError_t ft_select_take_all(FtSelectDev sel, const uint32_t* off, uint64_t* list_idx, cudaStream_t s);
cudaError_t ft_select_trim_refined(const FtCandDev* cand, const uint32_t* off, int32_t n_regions, int rank_by, uint32_t k,
                                   int32_t count_floor, double wcount_floor, FtCandDev* out_cand, int32_t* out_region,
                                   uint32_t* out_n, uint32_t out_cap, cudaStream_t s);
cudaError_t ft_count_to_key(const int32_t* c, float* k, int64_t n, cudaStream_t s);
cudaError_t ft_select_tighten(FtSelectDev sel, uint32_t k, FtMargin margin, cudaStream_t s);
cudaError_t ft_fill_f32(float* p, int64_t n, float v, cudaStream_t s);
// keys[e] = (keys[e] - mu) * inv_sigma  (standardised keys from a statistic array, fixed weights)
cudaError_t ft_keys_affine(float* keys, int64_t n, double mu, double inv_sigma, cudaStream_t s);
// keys[e] = -inf where the element's own number count (same layout) is below the floor
cudaError_t ft_select_mask_keys_local(float* keys, const int32_t* counts, int64_t n, int32_t floor, cudaStream_t s);
