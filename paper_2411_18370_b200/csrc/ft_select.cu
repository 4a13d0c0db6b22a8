// Per-band top-k selection ("retrieving the loudest candidate within each region";
// north_star: regions = frequency sub-bands, loudest -> top-k).  DESIGN.md "Selection".
//
// fp32 keys (power, or the integer count converted exactly) are filtered against a per-band
// threshold; survivors (key, canonical idx) sit in per-band append buffers.  A per-band radix
// select trims each buffer to the candidates that can still be in the top k given the fp32 error
// margin, the generic fp64 kernel refines them, and a per-band rank-by-counting writes the final
// k under the total order (value desc, idx asc).
#include <algorithm>
#include "ft_select.cuh"

namespace {

constexpr int SEL_THREADS = 1024;

// Block-wide radix select of the k-th largest key among n elements enumerated by `get(e)`.
// Returns the ordered-uint key of the k-th largest (all threads), or 0 when n < k.
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

__device__ __forceinline__ float apply_margin(float tau, float rel_margin) {
  return tau - rel_margin * fabsf(tau);
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

// k-th largest per band over a [n_rows][n_f0] key array -> thr[band] (with margin).  grid = (bands,
// row slices): the k-th largest of a slice is a valid lower bound of the band's, so thr[band] is the
// maximum over the slices (and over earlier calls: thresholds only ever tighten).
__global__ void __launch_bounds__(SEL_THREADS)
ft_band_threshold_kernel(const float* __restrict__ keys, int64_t n_rows, int64_t n_f0, int32_t bpb,
                         uint32_t k, float rel_margin, float* __restrict__ thr) {
  __shared__ uint32_t hist[256];
  __shared__ uint32_t bcast[2];
  const int b = blockIdx.x;
  const int64_t r0 = n_rows * blockIdx.y / gridDim.y, r1 = n_rows * (blockIdx.y + 1) / gridDim.y;
  const int64_t c0 = (int64_t)b * bpb;
  const int64_t bw = min((int64_t)bpb, n_f0 - c0);
  const int64_t n = (r1 - r0) * bw;
  auto get = [&](int64_t e) { return keys[(r0 + e / bw) * n_f0 + c0 + (e % bw)]; };
  const uint32_t kk = block_kth_largest(n, k, get, hist, bcast);
  if (threadIdx.x == 0 && n >= (int64_t)k) atomic_fmax(thr + b, apply_margin(ft_unkey(kk), rel_margin));
}

// Append every key >= thr[band] of a [n_rows][n_f0] key array (rows = points pt_begin + r).
// Row r of the key array is outer point pt_begin + (r / R) * stride * R + r % R (stride = 1: contiguous).
__global__ void ft_append_from_keys_kernel(const float* __restrict__ keys, int64_t n_rows, int64_t n_f0,
                                           int32_t bpb, uint64_t pt_begin, uint32_t R, uint32_t gstride,
                                           uint64_t pt_end, FtSelectDev sel) {
  const int64_t n = n_rows * n_f0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const int64_t c = e % n_f0;
    const int b = (int)(c / bpb);
    const float v = keys[e];
    const uint64_t r = (uint64_t)(e / n_f0);
    const uint64_t pt = pt_begin + (r / R) * (uint64_t)gstride * R + r % R;
    if (pt < pt_end && v > -INFINITY && v >= sel.thr[b]) ft_select_append(sel, b, v, pt * (uint64_t)n_f0 + (uint64_t)c);
  }
}

// Per band: k-th largest among the appended keys -> tighter threshold; compact the survivors into
// the global final list (idx + band).
__global__ void __launch_bounds__(SEL_THREADS)
ft_trim_kernel(FtSelectDev sel, uint32_t k, float rel_margin, uint64_t* __restrict__ final_idx,
               int32_t* __restrict__ final_band, uint32_t* __restrict__ final_n, uint32_t final_cap,
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
  auto get = [&](int64_t e) { return keys[e]; };
  const uint32_t kk = block_kth_largest((int64_t)cnt, k, get, hist, bcast);
  const float t = (cnt < k) ? -INFINITY : apply_margin(ft_unkey(kk), rel_margin);
  for (uint32_t e = threadIdx.x; e < cnt; e += blockDim.x) {
    if (keys[e] >= t) {
      const uint32_t slot = atomicAdd(final_n, 1u);
      if (slot < final_cap) {
        final_idx[slot] = idxs[e];
        final_band[slot] = b;
      }
    }
  }
}

// Overflow recovery: the k-th largest of the entries a band's buffer did keep is a valid lower bound
// of the band's true k-th value; tighten the threshold with it (the pass is then repeated).
__global__ void __launch_bounds__(SEL_THREADS)
ft_tighten_kernel(FtSelectDev sel, uint32_t k, float rel_margin) {
  __shared__ uint32_t hist[256];
  __shared__ uint32_t bcast[2];
  const int b = blockIdx.x;
  const uint32_t n = min(sel.cnt[b], sel.cap);
  const float* keys = sel.key + (size_t)b * sel.cap;
  auto get = [&](int64_t e) { return keys[e]; };
  const uint32_t kk = block_kth_largest((int64_t)n, k, get, hist, bcast);
  if (threadIdx.x == 0 && n >= k) sel.thr[b] = fmaxf(sel.thr[b], apply_margin(ft_unkey(kk), rel_margin));
}

// Per band: rank the refined candidates under (value desc, idx asc); ranks < k go to out[b][rank].
constexpr int RANK_CAP = 2048;
__global__ void __launch_bounds__(SEL_THREADS)
ft_rank_kernel(const FtCandDev* __restrict__ cand, const int32_t* __restrict__ cand_band,
               const uint32_t* __restrict__ n_dev, uint32_t cap, int by_count, uint32_t k,
               FtCandDev* __restrict__ out, uint32_t* __restrict__ overflow) {
  __shared__ double sval[RANK_CAP];
  __shared__ uint64_t sidx[RANK_CAP];
  __shared__ uint32_t ssrc[RANK_CAP];
  __shared__ uint32_t m;
  const int b = blockIdx.x;
  const uint32_t n = min(*n_dev, cap);
  if (threadIdx.x == 0) m = 0;
  for (uint32_t j = threadIdx.x; j < k; j += blockDim.x) {  // pad
    FtCandDev c;
    c.power = 0.0; c.wcount = 0.0; c.idx = ~0ull; c.count = 0; c.band = b;
    out[(size_t)b * k + j] = c;
  }
  __syncthreads();
  for (uint32_t e = threadIdx.x; e < n; e += blockDim.x) {
    if (cand_band[e] == b) {
      const uint32_t s = atomicAdd(&m, 1u);
      if (s < RANK_CAP) {
        sval[s] = by_count ? (double)cand[e].count : cand[e].power;
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

__global__ void ft_mask_keys_kernel(float* __restrict__ keys, int64_t n_rows, int64_t n_f0, uint64_t pt_begin,
                                    uint32_t R, uint32_t gstride, uint64_t pt_end,
                                    const int32_t* __restrict__ veto_cnt, int32_t floor) {
  const int64_t n = n_rows * n_f0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const uint64_t r = (uint64_t)(e / n_f0);
    const uint64_t pt = pt_begin + (r / R) * (uint64_t)gstride * R + r % R;
    if (pt < pt_end && veto_cnt[pt * (uint64_t)n_f0 + (uint64_t)(e % n_f0)] < floor) keys[e] = -INFINITY;
  }
}

// keys[e] = -inf where the element's own number count (same layout) is below the floor
__global__ void ft_mask_keys_local_kernel(float* __restrict__ keys, const int32_t* __restrict__ counts, int64_t n, int32_t floor) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride)
    if (counts[e] < floor) keys[e] = -INFINITY;
}

__global__ void ft_fill_f32_kernel(float* p, int64_t n, float v) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) p[i] = v;
}

__global__ void ft_count_to_key_kernel(const int32_t* __restrict__ c, float* __restrict__ k, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) k[i] = (float)c[i];
}

}  // namespace

cudaError_t ft_select_reset(FtSelectDev sel, uint32_t* final_n, uint32_t* overflow, cudaStream_t s) {
  ft_fill_f32_kernel<<<(sel.n_bands + 255) / 256, 256, 0, s>>>(sel.thr, sel.n_bands, -INFINITY);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(sel.cnt, 0, sizeof(uint32_t) * sel.n_bands, s);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(final_n, 0, sizeof(uint32_t), s);
  if (e != cudaSuccess) return e;
  return cudaMemsetAsync(overflow, 0, sizeof(uint32_t), s);
}

cudaError_t ft_select_threshold(const float* keys, int64_t n_rows, int64_t n_f0, int32_t bpb, uint32_t k,
                                float rel_margin, FtSelectDev sel, cudaStream_t s) {
  // slices of >= max(8 k, 32768) keys per band, at most 16 (more CTAs than bands on a 148-SM part)
  const int64_t per_band = n_rows * std::min<int64_t>(bpb, n_f0);
  const int64_t min_slice = std::max<int64_t>(8 * (int64_t)k, 32768);
  const unsigned slices = (unsigned)std::max<int64_t>(1, std::min<int64_t>({(int64_t)16, per_band / min_slice, n_rows}));
  ft_band_threshold_kernel<<<dim3((unsigned)sel.n_bands, slices), SEL_THREADS, 0, s>>>(keys, n_rows, n_f0, bpb, k, rel_margin, sel.thr);
  return cudaGetLastError();
}

cudaError_t ft_select_append_keys(const float* keys, int64_t n_rows, int64_t n_f0, int32_t bpb,
                                  uint64_t pt_begin, FtSelectDev sel, cudaStream_t s, uint32_t R, uint32_t stride,
                                  uint64_t pt_end) {
  const int64_t n = n_rows * n_f0;
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  ft_append_from_keys_kernel<<<grid, 256, 0, s>>>(keys, n_rows, n_f0, bpb, pt_begin, R ? R : 1, stride ? stride : 1, pt_end, sel);
  return cudaGetLastError();
}

cudaError_t ft_select_trim(FtSelectDev sel, uint32_t k, float rel_margin, uint64_t* final_idx,
                           int32_t* final_band, uint32_t* final_n, uint32_t final_cap,
                           uint32_t* overflow, cudaStream_t s) {
  ft_trim_kernel<<<sel.n_bands, SEL_THREADS, 0, s>>>(sel, k, rel_margin, final_idx, final_band, final_n, final_cap, overflow);
  return cudaGetLastError();
}

cudaError_t ft_select_rank(const FtCandDev* cand, const int32_t* cand_band, const uint32_t* n_dev,
                           uint32_t cap, int by_count, uint32_t k, int32_t n_bands, FtCandDev* out,
                           uint32_t* overflow, cudaStream_t s) {
  ft_rank_kernel<<<n_bands, SEL_THREADS, 0, s>>>(cand, cand_band, n_dev, cap, by_count, k, out, overflow);
  return cudaGetLastError();
}

cudaError_t ft_count_to_key(const int32_t* c, float* k, int64_t n, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  ft_count_to_key_kernel<<<grid, 256, 0, s>>>(c, k, n);
  return cudaGetLastError();
}

cudaError_t ft_select_tighten(FtSelectDev sel, uint32_t k, float rel_margin, cudaStream_t s) {
  ft_tighten_kernel<<<sel.n_bands, SEL_THREADS, 0, s>>>(sel, k, rel_margin);
  return cudaGetLastError();
}

cudaError_t ft_fill_f32(float* p, int64_t n, float v, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  ft_fill_f32_kernel<<<grid, 256, 0, s>>>(p, n, v);
  return cudaGetLastError();
}

cudaError_t ft_select_mask_keys(float* keys, int64_t n_rows, int64_t n_f0, uint64_t pt_begin, uint32_t R,
                                uint32_t stride, uint64_t pt_end, const int32_t* veto_cnt, int32_t floor,
                                cudaStream_t s) {
  const int64_t n = n_rows * n_f0;
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  ft_mask_keys_kernel<<<grid, 256, 0, s>>>(keys, n_rows, n_f0, pt_begin, R ? R : 1, stride ? stride : 1, pt_end, veto_cnt, floor);
  return cudaGetLastError();
}

cudaError_t ft_select_mask_keys_local(float* keys, const int32_t* counts, int64_t n, int32_t floor, cudaStream_t s) {
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  ft_mask_keys_local_kernel<<<grid, 256, 0, s>>>(keys, counts, n, floor);
  return cudaGetLastError();
}
