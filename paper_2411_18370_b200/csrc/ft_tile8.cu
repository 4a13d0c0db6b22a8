// Tile kernel for the Hough number count (Eq. 7) on a packed hit map.
//
// The count needs one BIT per evaluation, (P[a][k] > rho_th); it is exact in any integer width.
// Same CTA / warp organisation, producer ring and canonical track entries as ft_tile.cu, but
//   * the gathered array is the hit map as BYTES, in four byte-shifted copies
//       H8[m][a][b] = (P[a][b + m] > rho_th),  m = 0..3,
//     so that the 4 hits of 4 consecutive f0 starting at any bin o are ONE aligned 32-bit word of
//     copy m = o mod 4;
//   * a thread owns 4 consecutive f0 per chunk (f0 = first + 128 j + 4 lane + c), loads that word
//     and adds it to a register holding four 8-bit counters: 1 LDS.32 + 1 IADD per 4 evaluations,
//     a quarter of the shared-memory traffic of the fp32 gather;
//   * every 224 SFTs the 8-bit counters are folded into two registers of 16-bit counters
//     (n_sft <= 65535 is a plan condition), unpacked once in the epilogue.
// The staged bytes per SFT row are the same as for the fp32 strip (4 copies x 1 byte per bin).
#include "ft_tile_dev.cuh"

namespace {

constexpr int kFlushBlocks = 7;  // 7 blocks of 32 SFTs = 224 <= 255 increments per 8-bit counter

template <int J>
__global__ void __maxnreg__(ft_tile8_max_regs(J))
ft_tile8_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_cw = a.R * a.wpp;
  const int tile = (int)(blockIdx.x % (unsigned)a.n_tiles);
  const uint64_t group_l = blockIdx.x / (unsigned)a.n_tiles;
  uint64_t group = group_l * a.group_stride;
  if (a.skip_stride > 1) {
    const uint64_t m = a.skip_stride - 1, nb = a.skip_n * m;
    group = group_l < nb ? (group_l / m) * a.skip_stride + 1 + group_l % m : a.skip_n * a.skip_stride + (group_l - nb);
  }
  const int n_sft = (int)d.n_sft;
  const int NS = a.n_stages;
  const uint32_t copy_pitch = (uint32_t)a.pitch;       // bytes per byte-shifted copy of a row
  const uint32_t row_bytes = 4u * copy_pitch;           // four copies per row
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NS * kRPS * row_bytes);
  const uint32_t ring0 = smem_u32(smem_raw);
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + NS);
  if (threadIdx.x == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, n_cw);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int32_t* kst = a.kst + (size_t)tile * n_sft;

  if (warp == n_cw) {
    // ---- producer: per SFT row, the strip of each of the four copies -----------------------------
    // (the whole warp fetches the 32 strip starts of a block with one coalesced load; lane 0 issues)
    int s = 0;
    uint32_t lap = 0;
    const uint32_t nb = (uint32_t)a.copy_floats;  // bytes per copy (one byte per bin), multiple of 16
    for (int a0 = 0; a0 < n_sft; a0 += 32) {
      const int kk = (a0 + lane < n_sft) ? kst[a0 + lane] : 0;
      const int n_rows = min(32, n_sft - a0);
      for (int q = 0; q < n_rows; q += kRPS) {
        if (lap > 0) mbar_wait(empty0 + 8 * s, (lap - 1u) & 1u);
        const int rows = min(kRPS, n_rows - q);
        int kr[kRPS];
#pragma unroll
        for (int r = 0; r < kRPS; ++r) kr[r] = __shfl_sync(0xffffffffu, kk, (q + r) & 31);
        if (lane == 0) {
          mbar_expect_tx(full0 + 8 * s, 4u * nb * (uint32_t)rows);
          const uint32_t dst = ring0 + (uint32_t)(s * kRPS) * row_bytes;
#pragma unroll
          for (int r = 0; r < kRPS; ++r) {
            if (r < rows) {
#pragma unroll
              for (int m = 0; m < 4; ++m) {
                const uint8_t* src = d.H8 + ((int64_t)m * n_sft + (a0 + q + r)) * d.ld8 + kr[r];
                bulk_g2s(dst + (uint32_t)r * row_bytes + (uint32_t)m * copy_pitch, src, nb, full0 + 8 * s);
              }
            }
          }
        }
        __syncwarp();
        if (++s == NS) { s = 0; ++lap; }
      }
    }
    return;
  }
  if (warp > n_cw) return;

  // ---- consumers -------------------------------------------------------------------------------
  const int r_pt = warp / a.wpp, sub = warp % a.wpp;
  uint64_t pt = a.pt_begin + group * (uint64_t)a.R + (uint64_t)r_pt;
  const bool pt_active = pt < a.pt_end;
  if (!pt_active) pt = a.pt_end - 1;
  FtPoint* sp = reinterpret_cast<FtPoint*>(bars + 2 * NS) + warp;
  if (lane == 0) *sp = ft_decode_point(d, pt);
  __syncwarp();
  const uint32_t etab = smem_u32(reinterpret_cast<FtPoint*>(bars + 2 * NS) + n_cw) + 128u * (uint32_t)warp;
  const int tile_i0 = tile * a.tile_w;
  const int wlo = sub * J * 128;
  const int tile_n = min(a.tile_w, (int)d.n_f0 - tile_i0);
  const int warp_n = max(0, min(J * 128, tile_n - wlo));
  const int i_first = tile_i0 + wlo;
  // four 8-bit counters per register; the 16-bit levels (bytes (0, 2) and bytes (1, 3)) live in
  // shared memory, [2 j + h][consumer thread], touched once per 224 SFTs
  uint32_t c8[J];
  const uint32_t n_ct = 32u * (uint32_t)n_cw;
  const uint32_t c16 = etab - 128u * (uint32_t)warp + 128u * (uint32_t)n_cw + 4u * threadIdx.x;
#pragma unroll
  for (int j = 0; j < J; ++j) {
    c8[j] = 0u;
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(c16 + 4u * n_ct * (2 * j)), "r"(0u) : "memory");
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(c16 + 4u * n_ct * (2 * j + 1)), "r"(0u) : "memory");
  }
  const bool last_ok = warp_n > 128 * (J - 1);
  unsigned ties = 0;
  const uint32_t lane_bytes = ring0 + 4u * (uint32_t)lane;
  uint32_t stage_addr = lane_bytes;
  int s = 0;
  uint32_t ph = 0;
  int blocks_since_flush = 0;

  for (int a0 = 0; a0 < n_sft; a0 += 32) {
    uint32_t entry = 0;
    if (a0 + lane < n_sft && warp_n > 0)
      entry = ft_tile_entry(d, *sp, a0 + lane, kst[a0 + lane], i_first, warp_n, a.copy_floats, &ties, a.err);
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(etab + 4u * (uint32_t)lane), "r"(entry) : "memory");
    __syncwarp();
    const int n_rows = min(32, n_sft - a0);
    for (int q = 0; q < n_rows; q += kRPS) {
      uint32_t e4[kRPS];
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(e4[0]), "=r"(e4[1]), "=r"(e4[2]), "=r"(e4[3]) : "r"(etab + 4u * (uint32_t)q));
      mbar_wait(full0 + 8 * s, ph);
#pragma unroll
      for (int r = 0; r < kRPS; ++r) {
        if (q + r < n_rows) {
          const uint32_t e = e4[r];
          const uint32_t base = stage_addr + (uint32_t)r * row_bytes;
          const uint32_t off = e & 8191u;
          // word of copy (off mod 4) that holds bins off .. off+3 of this lane's first 4 outputs
          const uint32_t ad_lo = base + (off & 3u) * copy_pitch + (off & ~3u);
          if (e < 8192u) {
            uint32_t v[J];
#pragma unroll
            for (int j = 0; j < J; ++j)
              if (j < J - 1 || last_ok) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v[j]) : "r"(ad_lo + 128u * j));
#pragma unroll
            for (int j = 0; j < J; ++j)
              if (j < J - 1 || last_ok) c8[j] += v[j];
          } else {
            const uint32_t off_hi = (e & (1u << 24)) ? off - 1u : off + 1u;
            const uint32_t ad_hi = base + (off_hi & 3u) * copy_pitch + (off_hi & ~3u);
            const int t_lane = (int)((e >> 13) & 2047u) - 4 * lane;  // outputs of this lane's chunk 0 before the break
#pragma unroll
            for (int j = 0; j < J; ++j) {
              const int cut = t_lane - 128 * j;  // >= 4: all before the break, <= 0: all after
              uint32_t va, vb;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(va) : "r"(ad_lo + 128u * j));
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(vb) : "r"(ad_hi + 128u * j));
              const uint32_t mask = cut >= 4 ? 0xffffffffu : (cut <= 0 ? 0u : ((1u << (8 * cut)) - 1u));
              c8[j] += (va & mask) | (vb & ~mask);
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * s);
      if (++s == NS) { s = 0; ph ^= 1u; stage_addr = lane_bytes; } else { stage_addr += kRPS * row_bytes; }
    }
    if (++blocks_since_flush == kFlushBlocks) {
      blocks_since_flush = 0;
#pragma unroll
      for (int j = 0; j < J; ++j) {
        uint32_t ta, tb;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(ta) : "r"(c16 + 4u * n_ct * (2 * j)));
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tb) : "r"(c16 + 4u * n_ct * (2 * j + 1)));
        ta += c8[j] & 0x00ff00ffu;
        tb += (c8[j] >> 8) & 0x00ff00ffu;
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(c16 + 4u * n_ct * (2 * j)), "r"(ta) : "memory");
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(c16 + 4u * n_ct * (2 * j + 1)), "r"(tb) : "memory");
        c8[j] = 0u;
      }
    }
  }

  // ---- epilogue ----------------------------------------------------------------------------------
  if (a.near_ties) {
    for (int o = 16; o > 0; o >>= 1) ties += __shfl_xor_sync(0xffffffffu, ties, o);
    if (lane == 0 && pt_active && ties) atomicAdd(a.near_ties, (unsigned long long)ties);
  }
  if (!pt_active) return;
#pragma unroll
  for (int j = 0; j < J; ++j) {
    uint32_t ta, tb;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(ta) : "r"(c16 + 4u * n_ct * (2 * j)));
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tb) : "r"(c16 + 4u * n_ct * (2 * j + 1)));
    ta += c8[j] & 0x00ff00ffu;
    tb += (c8[j] >> 8) & 0x00ff00ffu;
    const int32_t cnt[4] = {(int32_t)(ta & 0xffffu), (int32_t)(tb & 0xffffu), (int32_t)(ta >> 16), (int32_t)(tb >> 16)};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const int ii = 128 * j + 4 * lane + c;
      if (ii < warp_n) {
        const int64_t i = i_first + ii;
        const uint64_t idx = pt * (uint64_t)d.n_f0 + (uint64_t)i;
        const uint64_t o = a.group_stride > 1 ? (group_l * (uint64_t)a.R + (uint64_t)r_pt) * (uint64_t)d.n_f0 + (uint64_t)i
                                              : idx - a.out_base;
        if (a.out_i) a.out_i[o] = cnt[c];
        if (a.out_f) a.out_f[o] = (float)cnt[c];
        if (a.has_sel) {
          const int band = (int)(i / a.bpb);
          const float v = (float)cnt[c];
          if (v >= __ldg(a.sel.thr + band)) ft_select_append(a.sel, band, v, idx);
        }
      }
    }
  }
}

// H8[m][a][b] = (P[a][b + m] > rho) for b + m < n_bins, else 0
__global__ void ft_hitmap8_kernel(const float* __restrict__ P, float rho, uint8_t* __restrict__ H8,
                                  int64_t n_sft, int64_t n_bins, int64_t ld, int64_t ld8) {
  const int64_t n = 4 * n_sft * ld8, stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const int64_t b = e % ld8, a = (e / ld8) % n_sft, m = e / (ld8 * n_sft);
    H8[e] = (b + m < n_bins && P[a * ld + b + m] > rho) ? 1 : 0;
  }
}

template <int J>
cudaError_t launch8_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  static bool configured = false;
  if (!configured) {
    const cudaError_t e = cudaFuncSetAttribute(ft_tile8_kernel<J>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  ft_tile8_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

cudaError_t ft_tile8_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launch8_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t ft_launch_hitmap8(const float* P, float rho, uint8_t* H8, int64_t n_sft, int64_t n_bins, int64_t ld,
                              int64_t ld8, cudaStream_t s) {
  ft_hitmap8_kernel<<<148 * 8, 256, 0, s>>>(P, rho, H8, n_sft, n_bins, ld, ld8);
  return cudaGetLastError();
}
