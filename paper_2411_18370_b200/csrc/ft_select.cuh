// Per-band candidate buffers shared by the statistic kernels (fused filter) and ft_select.cu.
#pragma once
#include "ft_common.cuh"

struct FtSelectDev {
  float* thr;      // [n_bands] current fp32 threshold (with margin); -inf = accept everything
  uint32_t* cnt;   // [n_bands] number of append attempts (may exceed cap: overflow)
  float* key;      // [n_bands][cap]
  uint64_t* idx;   // [n_bands][cap]
  uint32_t cap;
  int32_t n_bands;
  // number-count veto: templates with veto_cnt[idx] < veto_floor are not candidates
  const int32_t* veto_cnt;  // [n_templates] integer number count, or nullptr
  int32_t veto_floor;
};

__device__ __forceinline__ void ft_select_append(const FtSelectDev& sel, int band, float key, uint64_t idx) {
  if (sel.veto_cnt && __ldg(sel.veto_cnt + idx) < sel.veto_floor) return;
  const uint32_t slot = atomicAdd(sel.cnt + band, 1u);
  if (slot < sel.cap) {
    sel.key[(size_t)band * sel.cap + slot] = key;
    sel.idx[(size_t)band * sel.cap + slot] = idx;
  }
}

cudaError_t ft_select_reset(FtSelectDev sel, uint32_t* final_n, uint32_t* overflow, cudaStream_t s);
cudaError_t ft_select_threshold(const float* keys, int64_t n_rows, int64_t n_f0, int32_t bpb, uint32_t k,
                                float rel_margin, FtSelectDev sel, cudaStream_t s);
cudaError_t ft_select_append_keys(const float* keys, int64_t n_rows, int64_t n_f0, int32_t bpb,
                                  uint64_t pt_begin, FtSelectDev sel, cudaStream_t s, uint32_t R = 1,
                                  uint32_t stride = 1, uint64_t pt_end = ~0ull);
cudaError_t ft_select_trim(FtSelectDev sel, uint32_t k, float rel_margin, uint64_t* final_idx,
                           int32_t* final_band, uint32_t* final_n, uint32_t final_cap,
                           uint32_t* overflow, cudaStream_t s);
cudaError_t ft_select_rank(const FtCandDev* cand, const int32_t* cand_band, const uint32_t* n_dev,
                           uint32_t cap, int by_count, uint32_t k, int32_t n_bands, FtCandDev* out,
                           uint32_t* overflow, cudaStream_t s);
cudaError_t ft_count_to_key(const int32_t* c, float* k, int64_t n, cudaStream_t s);
cudaError_t ft_select_tighten(FtSelectDev sel, uint32_t k, float rel_margin, cudaStream_t s);
cudaError_t ft_fill_f32(float* p, int64_t n, float v, cudaStream_t s);
// keys[r][c] = -inf where the template's number count is below the floor (rows mapped to points as in
// ft_select_append_keys)
cudaError_t ft_select_mask_keys(float* keys, int64_t n_rows, int64_t n_f0, uint64_t pt_begin, uint32_t R,
                                uint32_t stride, uint64_t pt_end, const int32_t* veto_cnt, int32_t floor,
                                cudaStream_t s);
cudaError_t ft_select_mask_keys_local(float* keys, const int32_t* counts, int64_t n, int32_t floor, cudaStream_t s);
