// Per-region top-k selection ("retrieving the loudest candidate within each region";
// north_star: regions = frequency sub-bands, loudest -> top-k; boxes of outer points x sub-bands for the
// hyperboxes of :338-342).  DESIGN.md "Selection".
//
// fp32 keys (power, the standardised z, the weighted count, or the integer count converted exactly) are
// filtered against a per-region threshold; survivors (key, canonical idx) sit in per-region append buffers.
// A per-region radix select trims each buffer to the candidates that can still be in the top k given the
// fp32 error margin, the generic fp64 kernel refines them, and a per-region rank-by-counting writes the
// final k under the total order (value desc, idx asc).
#include <algorithm>
#include "ft_select.cuh"

namespace {

constexpr int SEL_THREADS = 1024;

// Block-wide radix select of the k-th largest key among n elements enumerated by `get(e)`.
// Returns the ordered-uint key of the k-th largest (all threads), or 0 when fewer than k keys are > -inf.
template <typename Get>
__device__ uint32_t block_kth_largest(int64_t n, uint32_t k, Get get, uint32_t* hist /*[256]*/, uint32_t* bcast /*[2]*/) {
  if (n < (int64_t)k) return 0u;
  uint32_t prefix = 0, mask = 0, remaining = k;
  for (int shift = 24; shift >= 0; shift -= 8) {
    for (int i = threadIdx.x; i < 256; i += blockDim.x) hist[i] = 0;
    __syncthreads();
    for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
      const uint32_t key = ft_key(get(e));
      if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1u);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      uint32_t cum = 0;
      int b = 255;
      for (; b > 0; --b) {
        if (cum + hist[b] >= remaining) break;
        cum += hist[b];
      }
      bcast[0] = prefix | ((uint32_t)b << shift);
      bcast[1] = remaining - cum;
    }
    __syncthreads();
    prefix = bcast[0];
    remaining = bcast[1];
    mask |= 255u << shift;
    __syncthreads();
  }
  return prefix;
}

__device__ __forceinline__ float apply_margin(float tau, FtMargin m) {
  return tau - m.rel * (fabsf(tau) + m.shift);
}

__device__ __forceinline__ void atomic_fmax(float* addr, float v) {
  int* ai = reinterpret_cast<int*>(addr);
  int old = *ai;
  while (__int_as_float(old) < v) {
    const int assumed = old;
    old = atomicCAS(ai, assumed, __float_as_int(v));
    if (old == assumed) break;
  }
}

__device__ __forceinline__ uint64_t row_point(const FtRowMap& m, uint64_t r) {
  return m.glist ? (uint64_t)m.glist[r / m.R] * m.R + r % m.R : m.pt_begin + r;
}

// k-th largest per region over a [n_rows][n_f0] key array -> thr[region] (with margin).  grid = (regions,
// row slices): the k-th largest of a slice is a valid lower bound of the region's, so thr[region] is the
// maximum over the slices (and over earlier calls: thresholds only ever tighten).  Only templates that
// certainly pass the number-count veto count (a vetoed template must not raise a threshold).
__global__ void __launch_bounds__(SEL_THREADS)
ft_region_threshold_kernel(const float* __restrict__ keys, int64_t n_rows, int64_t n_f0, FtRowMap m,
                           uint32_t k, FtMargin margin, FtSelectDev sel) {
  __shared__ uint32_t hist[256];
  __shared__ uint32_t bcast[2];
  const int region = blockIdx.x;
  const int band = region % m.n_bands, pb = region / m.n_bands;
  const uint32_t* rl = m.pbox ? m.rows + m.row_start[pb] : nullptr;
  const int64_t n_r = m.pbox ? (int64_t)(m.row_start[pb + 1] - m.row_start[pb]) : n_rows;
  const int64_t r0 = n_r * blockIdx.y / gridDim.y, r1 = n_r * (blockIdx.y + 1) / gridDim.y;
  const int64_t c0 = (int64_t)band * m.bpb;
  const int64_t bw = min((int64_t)m.bpb, n_f0 - c0);
  const int64_t n = (r1 - r0) * bw;
  const bool veto = sel.veto_cnt || sel.veto_w;
  auto get = [&](int64_t e) {
    const int64_t r = rl ? (int64_t)rl[r0 + e / bw] : r0 + e / bw;
    const int64_t c = c0 + e % bw;
    const float v = keys[r * n_f0 + c];
    if (veto) {
      const uint64_t pt = row_point(m, (uint64_t)r);
      if (pt >= m.pt_end || !ft_select_sure(sel, pt * (uint64_t)n_f0 + (uint64_t)c)) return -INFINITY;
    }
    return v;
  };
  const uint32_t kk = block_kth_largest(n, k, get, hist, bcast);
  const float t = ft_unkey(kk);
  if (threadIdx.x == 0 && n >= (int64_t)k && t > -INFINITY) atomic_fmax(sel.thr + region, apply_margin(t, margin));
}

// Append every key >= thr[region] of a [n_rows][n_f0] key array.
__global__ void ft_append_from_keys_kernel(const float* __restrict__ keys, int64_t n_rows, int64_t n_f0,
                                           FtRowMap m, FtSelectDev sel) {
  const int64_t n = n_rows * n_f0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const int64_t c = e % n_f0;
    const float v = keys[e];
    const uint64_t pt = row_point(m, (uint64_t)(e / n_f0));
    if (pt >= m.pt_end || !(v > -INFINITY)) continue;
    const int region = (m.pbox ? m.pbox[pt] * m.n_bands : 0) + (int)(c / m.bpb);
    if (v >= sel.thr[region]) ft_select_append(sel, region, v, pt * (uint64_t)n_f0 + (uint64_t)c);
  }
}

// Per region: k-th largest among the appended keys that certainly pass the veto -> tighter threshold;
// compact the survivors into the global final list (idx + region).
__global__ void __launch_bounds__(SEL_THREADS)
ft_trim_kernel(FtSelectDev sel, uint32_t k, FtMargin margin, uint64_t* __restrict__ final_idx,
               int32_t* __restrict__ final_region, uint32_t* __restrict__ final_n, uint32_t final_cap,
               uint32_t* __restrict__ overflow) {
  __shared__ uint32_t hist[256];
  __shared__ uint32_t bcast[2];
  const int b = blockIdx.x;
  const uint32_t cnt = sel.cnt[b];
  if (cnt > sel.cap) {  // the append buffer overflowed: entries were dropped
    if (threadIdx.x == 0) atomicMax(overflow, cnt);
    return;
  }
  const float* keys = sel.key + (size_t)b * sel.cap;
  const uint64_t* idxs = sel.idx + (size_t)b * sel.cap;
  const bool veto = sel.veto_w != nullptr;   // (the integer veto is exact at append time)
  auto get = [&](int64_t e) { return (veto && !ft_select_sure(sel, idxs[e])) ? -INFINITY : keys[e]; };
  const uint32_t kk = block_kth_largest((int64_t)cnt, k, get, hist, bcast);
  const float tk = ft_unkey(kk);
  const float t = (cnt < k || !(tk > -INFINITY)) ? -INFINITY : apply_margin(tk, margin);
  for (uint32_t e = threadIdx.x; e < cnt; e += blockDim.x) {
    if (keys[e] >= t) {
      const uint32_t slot = atomicAdd(final_n, 1u);
      if (slot < final_cap) {
        final_idx[slot] = idxs[e];
        final_region[slot] = b;
      }
    }
  }
}

// Overflow recovery: the k-th largest of the entries a region's buffer did keep is a valid lower bound
// of the region's true k-th value; tighten the threshold with it (the pass is then repeated).
__global__ void __launch_bounds__(SEL_THREADS)
ft_tighten_kernel(FtSelectDev sel, uint32_t k, FtMargin margin) {
  __shared__ uint32_t hist[256];
  __shared__ uint32_t bcast[2];
  const int b = blockIdx.x;
  const uint32_t n = min(sel.cnt[b], sel.cap);
  const float* keys = sel.key + (size_t)b * sel.cap;
  const uint64_t* idxs = sel.idx + (size_t)b * sel.cap;
  const bool veto = sel.veto_w != nullptr;
  auto get = [&](int64_t e) { return (veto && !ft_select_sure(sel, idxs[e])) ? -INFINITY : keys[e]; };
  const uint32_t kk = block_kth_largest((int64_t)n, k, get, hist, bcast);
  const float t = ft_unkey(kk);
  if (threadIdx.x == 0 && n >= k && t > -INFINITY) sel.thr[b] = fmaxf(sel.thr[b], apply_margin(t, margin));
}

// Per region: rank the refined candidates under (value desc, idx asc); ranks < k go to out[region][rank].
// The exact number-count veto is applied here on the refined (fp64 / integer) values.
constexpr int RANK_CAP = 2048;
__global__ void __launch_bounds__(SEL_THREADS)
ft_rank_kernel(const FtCandDev* __restrict__ cand, const int32_t* __restrict__ cand_region,
               const uint32_t* __restrict__ n_dev, uint32_t cap, int rank_by, uint32_t k, int32_t count_floor,
               double wcount_floor, FtCandDev* __restrict__ out, uint32_t* __restrict__ overflow) {
  __shared__ double sval[RANK_CAP];
  __shared__ uint64_t sidx[RANK_CAP];
  __shared__ uint32_t ssrc[RANK_CAP];
  __shared__ uint32_t m;
  const int b = blockIdx.x;
  const uint32_t n = min(*n_dev, cap);
  if (threadIdx.x == 0) m = 0;
  for (uint32_t j = threadIdx.x; j < k; j += blockDim.x) {  // pad
    FtCandDev c;
    c.power = 0.0; c.wcount = 0.0; c.idx = ~0ull; c.count = 0; c.band = b; c.z = 0.0; c.sigma = 0.0;
    out[(size_t)b * k + j] = c;
  }
  __syncthreads();
  for (uint32_t e = threadIdx.x; e < n; e += blockDim.x) {
    if (cand_region[e] == b && cand[e].count >= count_floor && cand[e].wcount >= wcount_floor) {
      const uint32_t s = atomicAdd(&m, 1u);
      if (s < RANK_CAP) {
        sval[s] = rank_by == FT_RANK_COUNT ? (double)cand[e].count : rank_by == FT_RANK_WCOUNT ? cand[e].wcount
                : rank_by == FT_RANK_Z ? cand[e].z : cand[e].power;
        sidx[s] = cand[e].idx;
        ssrc[s] = e;
      }
    }
  }
  __syncthreads();
  const uint32_t mm = m;
  if (mm > RANK_CAP) {
    if (threadIdx.x == 0) atomicMax(overflow, mm);
    return;
  }
  for (uint32_t s = threadIdx.x; s < mm; s += blockDim.x) {
    const double v = sval[s];
    const uint64_t id = sidx[s];
    uint32_t rank = 0;
    for (uint32_t q = 0; q < mm; ++q) {
      const double vq = sval[q];
      rank += (vq > v || (vq == v && sidx[q] < id)) ? 1u : 0u;
    }
    if (rank < k) {
      FtCandDev c = cand[ssrc[s]];
      c.band = b;
      out[(size_t)b * k + rank] = c;
    }
  }
}

// Veto-first selection (ft_topk.cu): every appended entry of every region, compacted region by region into one list
// (off[b] = first slot of region b; the host computed it from the append counters).
__global__ void __launch_bounds__(256)
ft_take_all_kernel(FtSelectDev sel, const uint32_t* __restrict__ off, uint64_t* __restrict__ list_idx) {
  const int b = blockIdx.x;
  const uint32_t n = min(sel.cnt[b], sel.cap), o = off[b];
  const uint64_t* idxs = sel.idx + (size_t)b * sel.cap;
  for (uint32_t e = blockIdx.y * blockDim.x + threadIdx.x; e < n; e += gridDim.y * blockDim.x) list_idx[o + e] = idxs[e];
}

// Per region: among the refined candidates cand[off[b] .. off[b+1]) that pass the exact floors, the k-th largest
// ranking value as an fp32 key (the cast is monotone, so everything >= it is a superset of the top k); those are
// copied to out_cand / out_region (the input of ft_rank_kernel).
__global__ void __launch_bounds__(SEL_THREADS)
ft_trim_refined_kernel(const FtCandDev* __restrict__ cand, const uint32_t* __restrict__ off, int rank_by, uint32_t k,
                       int32_t count_floor, double wcount_floor, FtCandDev* __restrict__ out_cand,
                       int32_t* __restrict__ out_region, uint32_t* __restrict__ out_n, uint32_t out_cap) {
  __shared__ uint32_t hist[256];
  __shared__ uint32_t bcast[2];
  const int b = blockIdx.x;
  const FtCandDev* seg = cand + off[b];
  const int64_t n = (int64_t)(off[b + 1] - off[b]);
  auto get = [&](int64_t e) {
    const FtCandDev& c = seg[e];
    if (c.count < count_floor || !(c.wcount >= wcount_floor)) return -INFINITY;
    const double v = rank_by == FT_RANK_COUNT ? (double)c.count : rank_by == FT_RANK_WCOUNT ? c.wcount
                   : rank_by == FT_RANK_Z ? c.z : c.power;
    return (float)v;
  };
  const uint32_t kk = block_kth_largest(n, k, get, hist, bcast);
  const float t = (kk == 0u) ? -INFINITY : ft_unkey(kk);   // fewer than k pass: keep every one that does
  for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
    const float v = get(e);
    if (v > -INFINITY && v >= t) {
      const uint32_t slot = atomicAdd(out_n, 1u);
      if (slot < out_cap) { out_cand[slot] = seg[e]; out_region[slot] = b; }
    }
  }
}

// keys[e] = -inf where the element's own number count (same layout) is below the floor
__global__ void ft_mask_keys_local_kernel(float* __restrict__ keys, const int32_t* __restrict__ counts, int64_t n, int32_t floor) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride)
    if (counts[e] < floor) keys[e] = -INFINITY;
}

__global__ void ft_select_reset_kernel(FtSelectDev sel, uint32_t* final_n, uint32_t* overflow) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < sel.n_regions) { sel.thr[i] = -INFINITY; sel.cnt[i] = 0u; }
  if (i == 0) { *final_n = 0u; *overflow = 0u; }
}

__global__ void ft_fill_f32_kernel(float* p, int64_t n, float v) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) p[i] = v;
}

__global__ void ft_count_to_key_kernel(const int32_t* __restrict__ c, float* __restrict__ k, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) k[i] = (float)c[i];
}

__global__ void ft_keys_affine_kernel(float* __restrict__ k, int64_t n, double mu, double inv_sigma) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    k[i] = (float)(((double)k[i] - mu) * inv_sigma);
}

}  // namespace

cudaError_t ft_select_reset(FtSelectDev sel, uint32_t* final_n, uint32_t* overflow, cudaStream_t s) {
  ft_select_reset_kernel<<<(sel.n_regions + 255) / 256, 256, 0, s>>>(sel, final_n, overflow);
  return cudaGetLastError();
}

cudaError_t ft_select_threshold(const float* keys, int64_t n_rows, int64_t n_f0, const FtRowMap& map, uint32_t k,
                                FtMargin margin, FtSelectDev sel, cudaStream_t s) {
  // slices of >= max(8 k, 32768) keys per region, at most 16 (more CTAs than regions on a 148-SM part)
  const int64_t rows_per_box = std::max<int64_t>(1, n_rows / std::max(1, map.n_pbox));
  const int64_t per_region = rows_per_box * std::min<int64_t>(map.bpb, n_f0);
  const int64_t min_slice = std::max<int64_t>(8 * (int64_t)k, 32768);
  const unsigned slices = (unsigned)std::max<int64_t>(1, std::min<int64_t>({(int64_t)16, per_region / min_slice, rows_per_box}));
  ft_region_threshold_kernel<<<dim3((unsigned)sel.n_regions, slices), SEL_THREADS, 0, s>>>(keys, n_rows, n_f0, map, k, margin, sel);
  return cudaGetLastError();
}

cudaError_t ft_select_append_keys(const float* keys, int64_t n_rows, int64_t n_f0, const FtRowMap& map,
                                  FtSelectDev sel, cudaStream_t s) {
  const int64_t n = n_rows * n_f0;
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, (int64_t)ft_sm_count() * 16);
  ft_append_from_keys_kernel<<<grid, 256, 0, s>>>(keys, n_rows, n_f0, map, sel);
  return cudaGetLastError();
}

cudaError_t ft_select_trim(FtSelectDev sel, uint32_t k, FtMargin margin, uint64_t* final_idx,
                           int32_t* final_region, uint32_t* final_n, uint32_t final_cap,
                           uint32_t* overflow, cudaStream_t s) {
  ft_trim_kernel<<<sel.n_regions, SEL_THREADS, 0, s>>>(sel, k, margin, final_idx, final_region, final_n, final_cap, overflow);
  return cudaGetLastError();
}

cudaError_t ft_select_rank(const FtCandDev* cand, const int32_t* cand_region, const uint32_t* n_dev,
                           uint32_t cap, int rank_by, uint32_t k, int32_t n_regions, int32_t count_floor,
                           double wcount_floor, FtCandDev* out, uint32_t* overflow, cudaStream_t s) {
  ft_rank_kernel<<<n_regions, SEL_THREADS, 0, s>>>(cand, cand_region, n_dev, cap, rank_by, k, count_floor, wcount_floor, out, overflow);
  return cudaGetLastError();
}

cudaError_t ft_select_take_all(FtSelectDev sel, const uint32_t* off, uint64_t* list_idx, cudaStream_t s) {
  ft_take_all_kernel<<<dim3((unsigned)sel.n_regions, 8), 256, 0, s>>>(sel, off, list_idx);
  return cudaGetLastError();
}

cudaError_t ft_select_trim_refined(const FtCandDev* cand, const uint32_t* off, int32_t n_regions, int rank_by, uint32_t k,
                                   int32_t count_floor, double wcount_floor, FtCandDev* out_cand, int32_t* out_region,
                                   uint32_t* out_n, uint32_t out_cap, cudaStream_t s) {
  ft_trim_refined_kernel<<<n_regions, SEL_THREADS, 0, s>>>(cand, off, rank_by, k, count_floor, wcount_floor, out_cand, out_region,
                                                            out_n, out_cap);
  return cudaGetLastError();
}

cudaError_t ft_count_to_key(const int32_t* c, float* k, int64_t n, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, (int64_t)ft_sm_count() * 16);
  ft_count_to_key_kernel<<<grid, 256, 0, s>>>(c, k, n);
  return cudaGetLastError();
}

cudaError_t ft_select_tighten(FtSelectDev sel, uint32_t k, FtMargin margin, cudaStream_t s) {
  ft_tighten_kernel<<<sel.n_regions, SEL_THREADS, 0, s>>>(sel, k, margin);
  return cudaGetLastError();
}

cudaError_t ft_fill_f32(float* p, int64_t n, float v, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, (int64_t)ft_sm_count() * 16);
  ft_fill_f32_kernel<<<grid, 256, 0, s>>>(p, n, v);
  return cudaGetLastError();
}

cudaError_t ft_keys_affine(float* keys, int64_t n, double mu, double inv_sigma, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, (int64_t)ft_sm_count() * 16);
  ft_keys_affine_kernel<<<grid, 256, 0, s>>>(keys, n, mu, inv_sigma);
  return cudaGetLastError();
}

cudaError_t ft_select_mask_keys_local(float* keys, const int32_t* counts, int64_t n, int32_t floor, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, (int64_t)ft_sm_count() * 16);
  ft_mask_keys_local_kernel<<<grid, 256, 0, s>>>(keys, counts, n, floor);
  return cudaGetLastError();
}
