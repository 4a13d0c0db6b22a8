// Device-side pieces shared by the tile kernels (ft_tile.cu: fp32 gather; ft_tile8.cu: packed
// number-count gather): mbarrier / TMA bulk-copy wrappers, kernel arguments, the packed track entry
// and the canonical (shift, break) computation of one (outer point, SFT, warp range).
#pragma once
#include "ft_common.cuh"
#include "ft_select.cuh"

constexpr int kRPS = 4;  // spectrogram rows per ring stage (divides 32)

struct FtTileArgs {
  const float* A;
  const int32_t* kst;
  int32_t* err;
  int32_t tile_w, n_tiles, R, wpp, pitch, copy_floats, n_stages;
  uint64_t pt_begin, pt_end;
  double add_back;  // sum over SFTs of the per-row constant removed from A at fold time
  float* out_f;
  int32_t* out_i;
  uint64_t out_base;
  FtSelectDev sel;
  int32_t has_sel, bpb;
  unsigned long long* near_ties;
  uint32_t group_stride;  // > 1: every stride-th group only (threshold sample), outputs packed by launch-local row
  uint32_t skip_stride;   // > 1: every group EXCEPT the first skip_n multiples of skip_stride (the rest of the bank)
  uint64_t skip_n;
};

// Threads per CTA the kernel is compiled for: (consumer warps + 1 producer warp) * 32.  The
// accumulators (J) and the loads in flight (J) set the register need, hence the bound.
// (the register file is 4 x 16 384: 80 registers allow 6 warps per SM sub-partition, 72 allow 7, 64 allow 8)
__host__ __device__ constexpr int ft_tile_max_regs(int J) { return J <= 12 ? 64 : 72; }
__host__ __device__ constexpr int ft_tile_max_threads(int J) { return J <= 12 ? 1024 : 896; }
// packed number-count kernel: J registers of 8-bit counters + J loads in flight (16-bit levels in shared memory)
__host__ __device__ constexpr int ft_tile8_max_regs(int J) { return J <= 8 ? 64 : 80; }
__host__ __device__ constexpr int ft_tile8_max_threads(int J) { return J <= 8 ? 1024 : 768; }

// both statistics in one pass (ft_tileb.cu): J accumulators + J counters + J loads in flight
__host__ __device__ constexpr int ft_tileb_max_regs(int J) { return J <= 8 ? 64 : 80; }
__host__ __device__ constexpr int ft_tileb_max_threads(int J) { return J <= 8 ? 1024 : 768; }
cudaError_t ft_tileb_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s);

// packed number-count kernels (ft_tile8.cu); A = the 4 byte-shifted hit maps d.H8
cudaError_t ft_tile8_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s);

namespace {

constexpr int kMaxPitch = 8191;  // packed entry: 13 bits of strip offset

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// (a0, a1) += (v0, v1) as ONE instruction: sm_100's packed fp32 add (SASS FADD2), round-to-nearest like FADD
__device__ __forceinline__ void ft_add2(float& a0, float& a1, float v0, float v1) {
  unsigned long long a2, v2;
  asm("mov.b64 %0, {%1, %2};" : "=l"(a2) : "f"(a0), "f"(a1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(v2) : "f"(v0), "f"(v1));
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(a2) : "l"(a2), "l"(v2));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a0), "=f"(a1) : "l"(a2));
}

// Packed per-(warp, SFT) track entry: bits 0-12 strip offset of the warp's first output (floats),
// bits 13-23 break position relative to the warp's first output (0 = no break in the warp's range),
// bit 24 set when the shift decreases at the break.  No break <=> entry < 8192.
__device__ __forceinline__ uint32_t pack_entry(int off, int rel, bool neg) {
  return (uint32_t)off | ((uint32_t)rel << 13) | (neg ? (1u << 24) : 0u);
}

// A1 + A2 for one (outer point, SFT, warp range): canonical track at the first and last f0 of the
// range, and, if the two shifts differ, the canonical position of the single break.
__device__ __forceinline__ uint32_t ft_tile_entry(const FtDev& d, const FtPoint& p, int al, int kst_al,
                                               int i_first, int warp_n, int copy_floats,
                                               unsigned* ties, int32_t* err) {
  const double t = d.t_mid[al];
  const double D = ft_doppler(d, p, al, t);
  const double f1dt = __dmul_rn(p.f1, __dsub_rn(t, d.t_ref));
  auto xof = [&](int i) {
    const double f0 = __dadd_rn(d.f0_start, __dmul_rn((double)i, d.df0));
    const double x = ft_track_x(f0, f1dt, D, d.f_min, d.inv_df);
    *ties += ft_near_tie(x) ? 1u : 0u;
    return x;
  };
  const int i_last = i_first + warp_n - 1;
  const double xa = xof(i_first);
  const int ka = __double2int_rn(xa);
  const int s = ka - i_first;
  const int sb = __double2int_rn(xof(i_last)) - i_last;
  const int off = ka - kst_al;  // strip index of the warp's first output
  int rel = 0;
  const bool neg = sb < s;
  if (sb != s) {
    // smallest i in (i_first, i_last] with rint(x_i) - i != s: estimate from the slope, verify
    // with the canonical arithmetic, bisect if the estimate is off
    auto pred = [&](int i) { return (__double2int_rn(xof(i)) - i) != s; };
    int lo = i_first, hi = i_last;
    const double frac = xa - (double)ka;
    double nest = ceil((0.5 - (neg ? -frac : frac)) / fmax(fabs(D - 1.0), 1e-300));
    nest = fmin(fmax(nest, 1.0), (double)(warp_n - 1));
    const int cand = i_first + (int)nest;
    if (pred(cand)) {
      hi = cand;
      if (cand - 1 > lo) { if (!pred(cand - 1)) lo = cand - 1; else hi = cand - 1; }
    } else {
      lo = cand;
      if (cand + 1 < hi) { if (pred(cand + 1)) hi = cand + 1; else lo = cand + 1; }
    }
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (pred(mid)) hi = mid; else lo = mid;
    }
    rel = hi - i_first;
    if (sb - s > 1 || s - sb > 1) atomicExch(err, 2);
  }
  // every pixel read for a valid output must lie inside the copied strip (else: a planning bug)
  const int hi_idx = off + (warp_n - 1) + ((rel && !neg) ? 1 : 0);
  if (off < 0 || off > kMaxPitch || hi_idx >= copy_floats) {
    atomicExch(err, 1);
    return 0u;
  }
  return pack_entry(off, rel, neg);
}

}  // namespace
