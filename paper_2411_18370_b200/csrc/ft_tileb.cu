// Tile kernel for BOTH statistics in one pass (narrow bands, J <= 16 chunks per warp).
//
// Identical to ft_tile_kernel (ft_tile.cu) except that the gathered array is QB: the folded, centred
// power array Q with the number-count hit bit (P > rho_th) written into the least significant mantissa
// bit of every pixel (a perturbation of at most one ulp of |Q|, 1.2e-7 relative per pixel, inside the
// accumulation budget of DESIGN.md "Accumulation").  One LDS.32 then feeds both Eq. (3) (packed fp32 add)
// and Eq. (7) (integer add of the LSB), so the binary configuration computes both statistics, and applies
// the number-count veto of PAPER.md:496-502 in the fused filter, in a single gather.
#include <algorithm>
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tileb_max_regs(J))
ft_tileb_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_cw = a.R * a.wpp;
  const int tile = (int)(blockIdx.x % (unsigned)a.n_tiles);
  const uint64_t group_l = blockIdx.x / (unsigned)a.n_tiles;  // launch-local group
  uint64_t group = group_l * a.group_stride;
  if (a.skip_stride > 1) {
    const uint64_t m = a.skip_stride - 1, nb = a.skip_n * m;
    group = group_l < nb ? (group_l / m) * a.skip_stride + 1 + group_l % m : a.skip_n * a.skip_stride + (group_l - nb);
  }
  const int n_sft = (int)d.n_sft;
  const int NS = a.n_stages;
  float* ring = reinterpret_cast<float*>(smem_raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + (size_t)NS * kRPS * a.pitch * sizeof(float));
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
  const uint32_t row_bytes = 4u * (uint32_t)a.pitch;

  if (warp == n_cw) {
    // ---- producer: streams the strips (A3).  The whole warp fetches the 32 strip starts of a block
    // with one coalesced load; lane 0 issues the bulk copies.
    const int64_t total = (int64_t)n_sft * d.ld;
    int s = 0;
    uint32_t lap = 0;  // how many times the ring has wrapped
    for (int a0 = 0; a0 < n_sft; a0 += 32) {
      const int kk = (a0 + lane < n_sft) ? kst[a0 + lane] : 0;
      const int n_rows = min(32, n_sft - a0);
      for (int q = 0; q < n_rows; q += kRPS) {
        if (lap > 0) mbar_wait(empty0 + 8 * s, (lap - 1u) & 1u);  // consumers released the previous use
        const int rows = min(kRPS, n_rows - q);
        int kr[kRPS];
#pragma unroll
        for (int r = 0; r < kRPS; ++r) kr[r] = __shfl_sync(0xffffffffu, kk, (q + r) & 31);
        if (lane == 0) {
          int64_t src[kRPS];
          uint32_t nb[kRPS], bytes = 0;
#pragma unroll
          for (int r = 0; r < kRPS; ++r) {
            if (r < rows) {
              src[r] = (int64_t)(a0 + q + r) * d.ld + kr[r];
              nb[r] = 4u * (uint32_t)min((int64_t)a.copy_floats, total - src[r]);
              bytes += nb[r];
            }
          }
          mbar_expect_tx(full0 + 8 * s, bytes);
          const uint32_t dst = smem_u32(ring) + (uint32_t)(s * kRPS) * row_bytes;
#pragma unroll
          for (int r = 0; r < kRPS; ++r)
            if (r < rows) bulk_g2s(dst + (uint32_t)r * row_bytes, a.A + src[r], nb[r], full0 + 8 * s);
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
  if (!pt_active) pt = a.pt_end - 1;  // keep the barrier protocol; results are discarded
  // the point's parameters live in shared memory (17 registers less across the main loop)
  FtPoint* sp = reinterpret_cast<FtPoint*>(bars + 2 * NS) + warp;
  if (lane == 0) *sp = ft_decode_point(d, pt);
  __syncwarp();
  // per-warp table of the 32 packed track entries of the current SFT block: one broadcast LDS.128
  // per ring stage instead of one shuffle per row
  const uint32_t etab = smem_u32(reinterpret_cast<FtPoint*>(bars + 2 * NS) + n_cw) + 128u * (uint32_t)warp;
  const int tile_i0 = tile * a.tile_w;
  const int wlo = sub * J * 32;                                        // warp's first output, tile-relative
  const int tile_n = min(a.tile_w, (int)d.n_f0 - tile_i0);             // valid f0 in this tile
  const int warp_n = max(0, min(J * 32, tile_n - wlo));                // valid outputs of this warp
  const int i_first = tile_i0 + wlo;
  const bool last_ok = warp_n > 32 * (J - 1);  // the warp's last chunk holds valid outputs (else: skipped)
  float acc[J];
  uint32_t cnt[J];
#pragma unroll
  for (int j = 0; j < J; ++j) { acc[j] = 0.f; cnt[j] = 0u; }
  unsigned ties = 0;
  const uint32_t lane_bytes = smem_u32(ring) + 4u * (uint32_t)lane;
  uint32_t stage_addr = lane_bytes;
  int s = 0;
  uint32_t ph = 0;

  for (int a0 = 0; a0 < n_sft; a0 += 32) {
    // -- A1/A2: this lane's SFT ---------------------------------------------------------------------
    uint32_t entry = 0;
    if (a0 + lane < n_sft && warp_n > 0)
      entry = ft_tile_entry(d, *sp, a0 + lane, kst[a0 + lane], i_first, warp_n, a.copy_floats, &ties, a.err);
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(etab + 4u * (uint32_t)lane), "r"(entry) : "memory");
    __syncwarp();
    // -- A4: gather + reduce over the block's SFTs -----------------------------------------------
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
          if (e < 8192u) {  // no break inside this warp's range: J conflict-free LDS.32 + FADD
            const uint32_t ad = base + 4u * e;
            float v[J];
#pragma unroll
            for (int j = 0; j < J; ++j)
              if (j < J - 1 || last_ok) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v[j]) : "r"(ad + 128u * j));
            if (!last_ok) v[J - 1] = 0.f;
#pragma unroll
            for (int j = 0; j + 1 < J; j += 2) ft_add2(acc[j], acc[j + 1], v[j], v[j + 1]);
            if (J & 1) acc[J - 1] += v[J - 1];
#pragma unroll
            for (int j = 0; j < J; ++j) cnt[j] += __float_as_uint(v[j]) & 1u;  // the hit bit rides in the LSB
          } else {
            const uint32_t ad_lo = base + 4u * (e & 8191u);
            const uint32_t ad_hi = (e & (1u << 24)) ? ad_lo - 4u : ad_lo + 4u;
            const int t_lane = (int)((e >> 13) & 2047u) - lane;
#pragma unroll
            for (int j = 0; j < J; ++j) {
              const uint32_t ad = ((32 * j >= t_lane) ? ad_hi : ad_lo) + 128u * j;
              float v;
              asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(ad));
              acc[j] += v;
              cnt[j] += __float_as_uint(v) & 1u;
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * s);
      if (++s == NS) { s = 0; ph ^= 1u; stage_addr = lane_bytes; } else { stage_addr += kRPS * row_bytes; }
    }
  }

  // ---- A5/A6: epilogue ---------------------------------------------------------------------------
  if (a.near_ties) {
    for (int o = 16; o > 0; o >>= 1) ties += __shfl_xor_sync(0xffffffffu, ties, o);
    if (lane == 0 && pt_active && ties) atomicAdd(a.near_ties, (unsigned long long)ties);
  }
  if (!pt_active) return;
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const int ii = 32 * j + lane;
    if (ii < warp_n) {
      const int64_t i = i_first + ii;
      const uint64_t idx = pt * (uint64_t)d.n_f0 + (uint64_t)i;
      const uint64_t o = a.group_stride > 1 ? (group_l * (uint64_t)a.R + (uint64_t)r_pt) * (uint64_t)d.n_f0 + (uint64_t)i
                                            : idx - a.out_base;
      const float v = (float)((double)acc[j] + a.add_back);
      if (a.out_f) a.out_f[o] = v;
      if (a.out_i) a.out_i[o] = (int32_t)cnt[j];
      if (a.has_sel && (int32_t)cnt[j] >= a.sel.veto_floor) {   // number-count veto from the count in registers
        const int band = (int)(i / a.bpb);
        if (v >= __ldg(a.sel.thr + band)) ft_select_append(a.sel, band, v, idx);
      }
    }
  }
}


// QB[a][k] = Q[a][k] with the LSB replaced by (P[a][k] > rho)
__global__ void ft_qb_kernel(const float* __restrict__ Q, const float* __restrict__ P, float rho,
                             float* __restrict__ QB, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    QB[i] = __uint_as_float((__float_as_uint(Q[i]) & ~1u) | (P[i] > rho ? 1u : 0u));
}

template <int J>
cudaError_t launchb_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  static bool configured = false;
  if (!configured) {
    const cudaError_t e = cudaFuncSetAttribute(ft_tileb_kernel<J>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  ft_tileb_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

cudaError_t ft_tileb_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launchb_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t ft_launch_qb(const float* Q, const float* P, float rho, float* QB, int64_t n, cudaStream_t s) {
  ft_qb_kernel<<<148 * 8, 256, 0, s>>>(Q, P, rho, QB, n);
  return cudaGetLastError();
}
