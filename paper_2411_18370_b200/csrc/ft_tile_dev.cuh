// Device side of the tile kernels: ONE kernel body (prologue, TMA producer ring, canonical track entries,
// row loop, epilogue with the fused selection) templated on a gather policy:
//   GatherF32   (ft_tile.cu)   fp32 pixels, packed fp32 add             Eq. (3) on Q, Eq. (7) on the 0/1 map
//   GatherF32W  (ft_tilew.cu)  fp32 pixels x per-(point, SFT) weight    Eq. (3)-(5) with sky-dependent weights
//   GatherBoth  (ft_tileb.cu)  fp32 pixels with the hit bit in the LSB  Eq. (3) and Eq. (7) from one gather
//   GatherHit8  (ft_tile8.cu)  packed byte hit map, 8-bit SIMD counters Eq. (7)
// DESIGN.md "Kernels".  PAPER.md:53 (Eq. 2), :64 (Eq. 3), :69-84 (Eq. 4-5), :95 (Eq. 7), :330-351 (selection).
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
  const float* c_row;   // [n_sft] that per-row constant (row-weighted gather: add-back = sum_a u_a c_a)
  float* out_f;
  int32_t* out_i;
  uint64_t out_base;
  FtSelectDev sel;
  int32_t has_sel, bpb;
  // regions of the selection: box = pbox[pt] * n_bands + i_f0 / bpb (pbox == nullptr: frequency sub-bands only)
  const int32_t* pbox;
  int32_t n_bands;
  // standardised keys z = (s - mu) / sigma (Eq. 36): fixed weights use (z_mu, z_inv_sigma); the
  // row-weighted gather computes mu = 1 and sigma per point itself
  int32_t zmode;
  int32_t out_key;      // out_f receives the selection key (z in zmode) instead of the statistic
  double z_mu, z_inv_sigma;
  float* out_sigma;     // row-weighted gather: sigma_G of every outer point, [n_points] (or nullptr)
  const double* sky_norm;  // row-weighted gather: per sky point  sum_a u_a r_a,  sum_a (u_a r_a)^2,  sum_a u_a cQ_a,  sum_a u_a cWH_a
                           // [n_sky][4] (ft_skyw_norm_kernel, bind time);  norm_cb = 2 or 3: the add-back column of this pass
  int32_t norm_cb;
  unsigned long long* near_ties;
  const uint32_t* glist;  // != nullptr: the launch runs the CTA groups glist[0 .. grid / n_tiles) (the threshold
                          // sample), outputs packed by launch-local row (group_local * R + r) * n_f0 + i_f0
  const uint32_t* gskip;  // != nullptr: bit g set = group g was in the sample; its CTAs exit at once (the rest of the bank)
  // Split tail (ft_launch_tile): CTAs [0, main_ctas) each run one whole group of R points; the groups from main_groups
  // on -- the last, partial wave of the launch -- are split in tail_split parts of R / tail_split points each, run by
  // CTAs with that many fewer consumer warps (the other warps of the block exit at once), so that every SM has work
  // until the end.  tail_split = 1: no split.
  uint32_t main_ctas, main_groups, tail_split;
};

// Which (f0 tile, launch-local group, part of the group) a CTA runs, and how many of the group's points
struct FtCtaWork { int tile; uint64_t group_l; int part, R_cta; };
template <bool SPLIT>
__device__ __forceinline__ FtCtaWork ft_cta_work(const FtTileArgs& a) {
  FtCtaWork w;
  const unsigned bid = blockIdx.x;
  if (!SPLIT || a.tail_split <= 1u || bid < a.main_ctas) {
    w.tile = (int)(bid % (unsigned)a.n_tiles); w.group_l = bid / (unsigned)a.n_tiles; w.part = 0; w.R_cta = a.R;
  } else {
    const unsigned tb = bid - a.main_ctas, rest = tb / (unsigned)a.n_tiles;
    w.tile = (int)(tb % (unsigned)a.n_tiles);
    w.part = (int)(rest % a.tail_split);
    w.group_l = (uint64_t)a.main_groups + rest / a.tail_split;
    w.R_cta = a.R / (int)a.tail_split;
  }
  return w;
}

// Threads per CTA the kernels are compiled for: (consumer warps + 1 producer warp) * 32.  The accumulators
// (J) and the loads in flight (J) set the register need, hence the bound.
// (the register file is 4 x 16 384: 80 registers allow 6 warps per SM sub-partition, 72 allow 7, 64 allow 8)
// (measured: 64 registers and 14-15 points per CTA for the wide tiles is slower, 89.7-91.0 ms against 87.9 on config 2)
__host__ __device__ constexpr int ft_tile_max_regs(int J) { return J <= 12 ? 64 : 72; }
__host__ __device__ constexpr int ft_tile_max_threads(int J) { return J <= 12 ? 1024 : 896; }
// packed number-count kernel: J registers of 8-bit counters + J loads in flight (16-bit levels in shared memory)
__host__ __device__ constexpr int ft_tile8_max_regs(int J) { return J <= 8 ? 64 : 80; }
__host__ __device__ constexpr int ft_tile8_max_threads(int J) { return J <= 8 ? 1024 : 768; }
// both statistics in one pass: J accumulators + J counters + J loads in flight
__host__ __device__ constexpr int ft_tileb_max_regs(int J) { return J <= 8 ? 64 : 80; }
__host__ __device__ constexpr int ft_tileb_max_threads(int J) { return J <= 8 ? 1024 : 768; }
// row-weighted gather: as the plain gather (the sky-point tables live in shared memory, the normalisation sums come
// from a bind-time pass)
#ifndef FT_TILEW_REGS
#define FT_TILEW_REGS 72
#endif
__host__ __device__ constexpr int ft_tilew_max_regs(int J) { return J <= 12 ? 64 : FT_TILEW_REGS; }
__host__ __device__ constexpr int ft_tilew_max_threads(int J) { return J <= 12 ? 1024 : FT_TILEW_REGS <= 72 ? 896 : 768; }

cudaError_t ft_tile_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s);
cudaError_t ft_tile2_launch(int JA, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s);
cudaError_t ft_tilew_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s);
cudaError_t ft_tileb_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s);
cudaError_t ft_tile8_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s);

#ifdef __CUDACC__
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
// Wait for a phase of an mbarrier.  With the suspend-time hint the warp sleeps in hardware until the phase completes
// (SASS: one TRYWAIT, then a blocking PHASECHK) instead of spinning on TRYWAIT + BRA in the issue slots the other
// warps need.
#ifndef FT_WAIT_HINT
#define FT_WAIT_HINT 1
#endif
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
#if FT_WAIT_HINT
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n"
#else
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
#endif
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ float lds_f32(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// (a0, a1) += (v0, v1) as ONE instruction: sm_100's packed fp32 add (SASS FADD2), round-to-nearest like FADD
__device__ __forceinline__ void ft_add2(float& a0, float& a1, float v0, float v1) {
  unsigned long long a2, v2;
  asm("mov.b64 %0, {%1, %2};" : "=l"(a2) : "f"(a0), "f"(a1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(v2) : "f"(v0), "f"(v1));
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(a2) : "l"(a2), "l"(v2));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a0), "=f"(a1) : "l"(a2));
}
// (a0, a1) += w * (v0, v1): packed fp32 fused multiply-add (SASS FFMA2)
__device__ __forceinline__ void ft_fma2(float& a0, float& a1, float v0, float v1, float w) {
  unsigned long long a2, v2, w2;
  asm("mov.b64 %0, {%1, %2};" : "=l"(a2) : "f"(a0), "f"(a1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(v2) : "f"(v0), "f"(v1));
  asm("mov.b64 %0, {%1, %1};" : "=l"(w2) : "f"(w));
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(a2) : "l"(v2), "l"(w2), "l"(a2));
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

// ---- gather policies ---------------------------------------------------------------------------------
// A policy provides: CW (f0 per chunk = per warp load instruction), PER (f0 per lane per chunk), ROWW (a
// per-(point, SFT) weight multiplies the row), VETO (the fused filter applies the number-count floor from
// registers), the accumulator state, the producer's copies of one row, the two row bodies (no break / one
// break inside the warp's range), a hook after every block of 32 SFTs, and the final value of one output.

// fp32 pixels: J conflict-free LDS.32 + J/2 packed adds per row
struct GatherF32 {
  static constexpr int CW = 32, PER = 1;
  static constexpr bool ROWW = false, VETO = false, HASCNT = false, PAIRS = false;
  template <int J> struct State { float acc[J]; };
  static __device__ __forceinline__ size_t extra_smem(int, int) { return 0; }
  template <int J> static __device__ __forceinline__ void init(State<J>& st, uint32_t, uint32_t) {
#pragma unroll
    for (int j = 0; j < J; ++j) st.acc[j] = 0.f;
  }
  static __device__ __forceinline__ void produce_row(const FtDev& d, const FtTileArgs& a, uint32_t dst, int row, int k0,
                                                     uint32_t bar) {
    const int64_t src = (int64_t)row * d.ld + k0;
    const uint32_t nb = 4u * (uint32_t)min((int64_t)a.copy_floats, d.n_sft * d.ld - src);
    bulk_g2s(dst, a.A + src, nb, bar);
  }
  static __device__ __forceinline__ uint32_t row_tx_bytes(const FtDev& d, const FtTileArgs& a, int row, int k0) {
    const int64_t src = (int64_t)row * d.ld + k0;
    return 4u * (uint32_t)min((int64_t)a.copy_floats, d.n_sft * d.ld - src);
  }
  template <int J> static __device__ __forceinline__ void row_fast(State<J>& st, uint32_t e, uint32_t base, uint32_t,
                                                                   bool last_ok, float) {
    const uint32_t ad = base + 4u * e;
    float v[J];
#pragma unroll
    for (int j = 0; j < J; ++j)
      if (j < J - 1 || last_ok) v[j] = lds_f32(ad + 128u * j);
    if (!last_ok) v[J - 1] = 0.f;
#pragma unroll
    for (int j = 0; j + 1 < J; j += 2) ft_add2(st.acc[j], st.acc[j + 1], v[j], v[j + 1]);
    if (J & 1) st.acc[J - 1] += v[J - 1];
  }
  template <int J> static __device__ __forceinline__ void row_break(State<J>& st, uint32_t e, uint32_t base, uint32_t,
                                                                    int lane, float) {
    const uint32_t ad_lo = base + 4u * (e & 8191u);
    const uint32_t ad_hi = (e & (1u << 24)) ? ad_lo - 4u : ad_lo + 4u;
    const int t_lane = (int)((e >> 13) & 2047u) - lane;
#pragma unroll
    for (int j = 0; j < J; ++j) st.acc[j] += lds_f32(((32 * j >= t_lane) ? ad_hi : ad_lo) + 128u * j);
  }
  template <int J, class S> static __device__ __forceinline__ void block_end(S&, int) {}
  template <int J, class S> static __device__ __forceinline__ void finalize(S&) {}
  // value of output (chunk j, sub-position c) before the final scale, and its integer count (HASCNT policies)
  template <int J> static __device__ __forceinline__ void result(State<J>& st, int j, int, double add_back, double* v, int32_t* c) {
    *v = (double)st.acc[j] + add_back;
    *c = 0;
  }
};

// fp32 pixels times a per-(point, SFT) weight u (sky-dependent weights, Eq. 4): packed FFMA
struct GatherF32W : GatherF32 {
  static constexpr bool ROWW = true;
  template <int J> static __device__ __forceinline__ void row_fast(State<J>& st, uint32_t e, uint32_t base, uint32_t,
                                                                   bool last_ok, float u) {
    const uint32_t ad = base + 4u * e;
    float v[J];
#pragma unroll
    for (int j = 0; j < J; ++j)
      if (j < J - 1 || last_ok) v[j] = lds_f32(ad + 128u * j);
    if (!last_ok) v[J - 1] = 0.f;
#pragma unroll
    for (int j = 0; j + 1 < J; j += 2) ft_fma2(st.acc[j], st.acc[j + 1], v[j], v[j + 1], u);
    if (J & 1) st.acc[J - 1] = fmaf(u, v[J - 1], st.acc[J - 1]);
  }
  template <int J> static __device__ __forceinline__ void row_break(State<J>& st, uint32_t e, uint32_t base, uint32_t,
                                                                    int lane, float u) {
    const uint32_t ad_lo = base + 4u * (e & 8191u);
    const uint32_t ad_hi = (e & (1u << 24)) ? ad_lo - 4u : ad_lo + 4u;
    const int t_lane = (int)((e >> 13) & 2047u) - lane;
#pragma unroll
    for (int j = 0; j < J; ++j) st.acc[j] = fmaf(u, lds_f32(((32 * j >= t_lane) ? ad_hi : ad_lo) + 128u * j), st.acc[j]);
  }
};

// fp32 pixels of QB: Q with its six low mantissa bits replaced by 00000h, h = the hit bit (P > rho_th).  One LDS
// feeds the packed fp32 add (Eq. 3) AND one integer add of the raw word (Eq. 7): the low six bits of the integer
// sum count the hits of up to 63 rows (carries only travel upwards), so they are folded into 16-bit counters once
// per block of 32 SFTs.  The pixel is rounded to 18 mantissa bits (<= 3.8e-6 of |q| per pixel, random sign:
// ~3e-8 of the statistic at n_sft = 8000; the plan keeps this kernel to 64 <= n_sft <= 65535).

struct GatherBoth : GatherF32 {
  static constexpr bool VETO = true, HASCNT = true, PAIRS = true;
  static constexpr uint32_t kLowMask = 63u;
  template <int J> struct State { float acc[J]; uint32_t raw[J]; uint32_t c16[(J + 1) / 2]; };
  template <int J> static __device__ __forceinline__ void init(State<J>& st, uint32_t, uint32_t) {
#pragma unroll
    for (int j = 0; j < J; ++j) { st.acc[j] = 0.f; st.raw[j] = 0u; }
#pragma unroll
    for (int j = 0; j < (J + 1) / 2; ++j) st.c16[j] = 0u;
  }
  template <int J> static __device__ __forceinline__ void row_fast(State<J>& st, uint32_t e, uint32_t base, uint32_t,
                                                                   bool last_ok, float) {
    const uint32_t ad = base + 4u * e;
    float v[J];
#pragma unroll
    for (int j = 0; j < J; ++j)
      if (j < J - 1 || last_ok) v[j] = lds_f32(ad + 128u * j);
    if (!last_ok) v[J - 1] = 0.f;
#pragma unroll
    for (int j = 0; j + 1 < J; j += 2) ft_add2(st.acc[j], st.acc[j + 1], v[j], v[j + 1]);
    if (J & 1) st.acc[J - 1] += v[J - 1];
    // the hit bit rides in the low bits: one integer add of the raw word
#pragma unroll
    for (int j = 0; j < J; ++j) st.raw[j] += __float_as_uint(v[j]);
  }
  // Two rows at once (both without a break in the warp's range): the raw words of the two rows and the running
  // sum are ONE three-input integer add (IADD3), so a pixel costs 1 LDS + 1/2 FADD2 + 1/2 IADD3.  Loads are issued
  // in two half batches to bound the registers in flight.
  template <int J> static __device__ __forceinline__ void rows_fast_pair(State<J>& st, uint32_t e0, uint32_t e1, uint32_t base0,
                                                                         uint32_t base1, uint32_t, bool last_ok) {
    const uint32_t ad0 = base0 + 4u * e0, ad1 = base1 + 4u * e1;
    constexpr int H = (((J + 1) / 2) + 1) & ~1;   // even, so the packed adds never straddle a batch
#pragma unroll
    for (int h0 = 0; h0 < J; h0 += H) {
      float v0[H], v1[H];
#pragma unroll
      for (int i = 0; i < H; ++i) {
        const int j = h0 + i;
        if (j < J) {
          if (j < J - 1 || last_ok) { v0[i] = lds_f32(ad0 + 128u * j); v1[i] = lds_f32(ad1 + 128u * j); }
          else { v0[i] = 0.f; v1[i] = 0.f; }
        }
      }
#pragma unroll
      for (int i = 0; i < H; i += 2) {
        const int j = h0 + i;
        if (j + 1 < J) {
          ft_add2(st.acc[j], st.acc[j + 1], v0[i], v0[i + 1]);
          ft_add2(st.acc[j], st.acc[j + 1], v1[i], v1[i + 1]);
        } else if (j < J) {
          st.acc[j] += v0[i];
          st.acc[j] += v1[i];
        }
      }
#pragma unroll
      for (int i = 0; i < H; ++i) {
        const int j = h0 + i;
        if (j < J) {
          uint32_t r = st.raw[j];
          asm("{\n.reg .u32 t;\nadd.u32 t, %1, %2;\nadd.u32 %0, %0, t;\n}" : "+r"(r) : "r"(__float_as_uint(v0[i])), "r"(__float_as_uint(v1[i])));
          st.raw[j] = r;
        }
      }
    }
  }
  template <int J> static __device__ __forceinline__ void row_break(State<J>& st, uint32_t e, uint32_t base, uint32_t,
                                                                    int lane, float) {
    const uint32_t ad_lo = base + 4u * (e & 8191u);
    const uint32_t ad_hi = (e & (1u << 24)) ? ad_lo - 4u : ad_lo + 4u;
    const int t_lane = (int)((e >> 13) & 2047u) - lane;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const float v = lds_f32(((32 * j >= t_lane) ? ad_hi : ad_lo) + 128u * j);
      st.acc[j] += v;
      st.raw[j] += __float_as_uint(v);
    }
  }
  template <int J> static __device__ __forceinline__ void flush(State<J>& st) {
#pragma unroll
    for (int j = 0; j < J; ++j) {
      st.c16[j >> 1] += (st.raw[j] & kLowMask) << (16 * (j & 1));
      st.raw[j] = 0u;
    }
  }
  template <int J, class S> static __device__ __forceinline__ void block_end(S& st, int) { flush<J>(st); }   // 32 rows <= 63
  template <int J, class S> static __device__ __forceinline__ void finalize(S& st) { flush<J>(st); }
  template <int J> static __device__ __forceinline__ void result(State<J>& st, int j, int, double add_back, double* v, int32_t* c) {
    *v = (double)st.acc[j] + add_back;
    *c = (int32_t)((st.c16[j >> 1] >> (16 * (j & 1))) & 0xffffu);
  }
};

// packed byte hit map in four byte-shifted copies: H8[m][a][b] = (P[a][b + m] > rho_th), so the 4 hits of 4
// consecutive f0 starting at any bin are ONE aligned 32-bit word of copy (bin mod 4).  A lane owns 4
// consecutive f0 per 128-wide chunk: 1 LDS.32 + 1 IADD into four 8-bit counters per 4 evaluations; every 224
// SFTs the counters are folded into 16-bit levels in shared memory (n_sft <= 65535 is a plan condition).
struct GatherHit8 {
  static constexpr int CW = 128, PER = 4;
  static constexpr bool ROWW = false, VETO = false, HASCNT = true, PAIRS = true;
  static constexpr int kFlushBlocks = 7;  // 7 blocks of 32 SFTs = 224 <= 255 increments per 8-bit counter
  template <int J> struct State { uint32_t c8[J]; uint32_t c16, n_ct; };
  template <int J> static __device__ __forceinline__ void init(State<J>& st, uint32_t extra0, uint32_t n_ct) {
    st.c16 = extra0 + 4u * threadIdx.x;
    st.n_ct = n_ct;
#pragma unroll
    for (int j = 0; j < J; ++j) {
      st.c8[j] = 0u;
      sts_u32(st.c16 + 4u * n_ct * (2 * j), 0u);
      sts_u32(st.c16 + 4u * n_ct * (2 * j + 1), 0u);
    }
  }
  static __device__ __forceinline__ void produce_row(const FtDev& d, const FtTileArgs& a, uint32_t dst, int row, int k0,
                                                     uint32_t bar) {
#pragma unroll
    for (int m = 0; m < 4; ++m)
      bulk_g2s(dst + (uint32_t)m * (uint32_t)a.pitch, d.H8 + ((int64_t)m * d.n_sft + row) * d.ld8 + k0,
               (uint32_t)a.copy_floats, bar);
  }
  static __device__ __forceinline__ uint32_t row_tx_bytes(const FtDev&, const FtTileArgs& a, int, int) {
    return 4u * (uint32_t)a.copy_floats;
  }
  template <int J> static __device__ __forceinline__ void row_fast(State<J>& st, uint32_t e, uint32_t base, uint32_t copy_pitch,
                                                                   bool last_ok, float) {
    // word of copy (off mod 4) that holds bins off .. off+3 of this lane's first 4 outputs
    const uint32_t ad = base + (e & 3u) * copy_pitch + (e & ~3u);
    uint32_t v[J];
#pragma unroll
    for (int j = 0; j < J; ++j)
      if (j < J - 1 || last_ok) v[j] = lds_u32(ad + 128u * j);
#pragma unroll
    for (int j = 0; j < J; ++j)
      if (j < J - 1 || last_ok) st.c8[j] += v[j];
  }
  // two rows at once: the packed hits of both rows and the running counters are one three-input add (IADD3)
  template <int J> static __device__ __forceinline__ void rows_fast_pair(State<J>& st, uint32_t e0, uint32_t e1, uint32_t base0,
                                                                         uint32_t base1, uint32_t copy_pitch, bool last_ok) {
    const uint32_t ad0 = base0 + (e0 & 3u) * copy_pitch + (e0 & ~3u), ad1 = base1 + (e1 & 3u) * copy_pitch + (e1 & ~3u);
    // loads in two half batches (2 x 8 in flight)
    constexpr int H = (J + 1) / 2;
#pragma unroll
    for (int h0 = 0; h0 < J; h0 += H) {
      uint32_t v0[H], v1[H];
#pragma unroll
      for (int i = 0; i < H; ++i) {
        const int j = h0 + i;
        if (j < J && (j < J - 1 || last_ok)) { v0[i] = lds_u32(ad0 + 128u * j); v1[i] = lds_u32(ad1 + 128u * j); }
      }
#pragma unroll
      for (int i = 0; i < H; ++i) {
        const int j = h0 + i;
        if (j < J && (j < J - 1 || last_ok)) {
          uint32_t r = st.c8[j];
          asm("{\n.reg .u32 t;\nadd.u32 t, %1, %2;\nadd.u32 %0, %0, t;\n}" : "+r"(r) : "r"(v0[i]), "r"(v1[i]));
          st.c8[j] = r;
        }
      }
    }
  }
  template <int J> static __device__ __forceinline__ void row_break(State<J>& st, uint32_t e, uint32_t base, uint32_t copy_pitch,
                                                                    int lane, float) {
    const uint32_t off = e & 8191u;
    const uint32_t ad_lo = base + (off & 3u) * copy_pitch + (off & ~3u);
    const uint32_t off_hi = (e & (1u << 24)) ? off - 1u : off + 1u;
    const uint32_t ad_hi = base + (off_hi & 3u) * copy_pitch + (off_hi & ~3u);
    const int t_lane = (int)((e >> 13) & 2047u) - 4 * lane;  // outputs of this lane's chunk 0 before the break
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const int cut = t_lane - 128 * j;  // >= 4: all before the break, <= 0: all after
      const uint32_t va = lds_u32(ad_lo + 128u * j), vb = lds_u32(ad_hi + 128u * j);
      const uint32_t mask = cut >= 4 ? 0xffffffffu : (cut <= 0 ? 0u : ((1u << (8 * cut)) - 1u));
      st.c8[j] += (va & mask) | (vb & ~mask);
    }
  }
  template <int J> static __device__ __forceinline__ void flush(State<J>& st) {
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const uint32_t aa = st.c16 + 4u * st.n_ct * (2 * j), ab = st.c16 + 4u * st.n_ct * (2 * j + 1);
      sts_u32(aa, lds_u32(aa) + (st.c8[j] & 0x00ff00ffu));
      sts_u32(ab, lds_u32(ab) + ((st.c8[j] >> 8) & 0x00ff00ffu));
      st.c8[j] = 0u;
    }
  }
  template <int J> static __device__ __forceinline__ void block_end(State<J>& st, int blocks_done) {
    if (blocks_done % kFlushBlocks == 0) flush<J>(st);
  }
  template <int J> static __device__ __forceinline__ void finalize(State<J>& st) { flush<J>(st); }
  template <int J> static __device__ __forceinline__ void result(State<J>& st, int j, int c, double, double* v, int32_t* cnt) {
    const uint32_t ta = lds_u32(st.c16 + 4u * st.n_ct * (2 * j)), tb = lds_u32(st.c16 + 4u * st.n_ct * (2 * j + 1));
    const uint32_t r = (c == 0) ? (ta & 0xffffu) : (c == 1) ? (tb & 0xffffu) : (c == 2) ? (ta >> 16) : (tb >> 16);
    *cnt = (int32_t)r;
    *v = (double)r;
  }
};

// ---- producer warp: streams the strips (A3).  The whole warp fetches the 32 strip starts of a block of SFTs with
// one coalesced load; lane 0 issues one bulk copy per row into the ring stage, after the consumers released it.
template <class G>
__device__ __forceinline__ void ft_tile_produce(const FtDev& d, const FtTileArgs& a, const int32_t* kst, int n_sft, int NS,
                                                uint32_t ring0, uint32_t full0, uint32_t empty0, uint32_t row_bytes, int lane) {
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
        uint32_t bytes = 0;
#pragma unroll
        for (int r = 0; r < kRPS; ++r)
          if (r < rows) bytes += G::row_tx_bytes(d, a, a0 + q + r, kr[r]);
        mbar_expect_tx(full0 + 8 * s, bytes);
        const uint32_t dst = ring0 + (uint32_t)(s * kRPS) * row_bytes;
#pragma unroll
        for (int r = 0; r < kRPS; ++r)
          if (r < rows) G::produce_row(d, a, dst + (uint32_t)r * row_bytes, a0 + q + r, kr[r], full0 + 8 * s);
      }
      __syncwarp();
      if (++s == NS) { s = 0; ++lap; }
    }
  }
}

// Shared-memory layout (bytes): ring [NS][kRPS][row_bytes] | full[NS] empty[NS] mbarriers | FtPoint[n_cw] |
// entry table [n_cw][32] u32 | (ROWW: weight table [n_cw][32] f32 | FtSkyPoint[n_cw]) | policy extra.
template <class G>
__host__ __device__ inline size_t ft_tile_state_bytes(int J, int n_cw) {
  return (sizeof(FtPoint) + 128 + (G::ROWW ? 128 + sizeof(FtSkyPoint) : 0)) * (size_t)n_cw + 16 +
         (G::PER == 4 ? (size_t)8 * J * 32 * n_cw : 0);
}

template <int J, class G>
__device__ __forceinline__ void ft_tile_body(const FtDev& d, const FtTileArgs& a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // (the packed number-count kernel sits at its register limit -- a few more live values and ptxas schedules its
  // row loop two loads at a time, 34.9 -> 44 ms on config 2 -- so its launches are never split: ft_launch_tile)
  const FtCtaWork cw = ft_cta_work<G::PER == 1>(a);
  const int n_cw = cw.R_cta * a.wpp;                          // consumer warps of this CTA
  const int tile = cw.tile;
  const uint64_t group_l = cw.group_l;                        // launch-local group
  const uint64_t group = a.glist ? (uint64_t)__ldg(a.glist + group_l) : group_l;
  if (a.gskip && ((__ldg(a.gskip + (group >> 5)) >> (group & 31)) & 1u)) return;   // (whole CTA: before any barrier)
  const int n_sft = (int)d.n_sft;
  const int NS = a.n_stages;
  const uint32_t copy_pitch = (uint32_t)a.pitch;                 // elements per staged (copy of a) row
  const uint32_t row_bytes = 4u * copy_pitch;                    // fp32: pitch floats; packed: four byte copies
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
    ft_tile_produce<G>(d, a, kst, n_sft, NS, ring0, full0, empty0, row_bytes, lane);
    return;
  }
  if (warp > n_cw) return;

  // ---- consumers -------------------------------------------------------------------------------
  const int r_pt = cw.part * cw.R_cta + warp / a.wpp, sub = warp % a.wpp;   // the point's place in its group
  uint64_t pt = a.pt_begin + group * (uint64_t)a.R + (uint64_t)r_pt;
  const bool pt_active = pt < a.pt_end;
  if (!pt_active) pt = a.pt_end - 1;  // keep the barrier protocol; results are discarded
  // the point's parameters live in shared memory (17 registers less across the main loop)
  FtPoint* sp = reinterpret_cast<FtPoint*>(bars + 2 * NS) + warp;
  if (lane == 0) *sp = ft_decode_point(d, pt);
  __syncwarp();
  // per-warp table of the 32 packed track entries of the current SFT block: one broadcast LDS.128
  // per ring stage instead of one shuffle per row (and, row-weighted, a second table of the 32 weights)
  const uint32_t etab0 = smem_u32(reinterpret_cast<FtPoint*>(bars + 2 * NS) + n_cw);
  const uint32_t etab = etab0 + 128u * (uint32_t)warp;
  const uint32_t wtab = etab0 + 128u * (uint32_t)n_cw + 128u * (uint32_t)warp;
  const uint32_t extra0 = etab0 + (G::ROWW ? 256u + (uint32_t)sizeof(FtSkyPoint) : 128u) * (uint32_t)n_cw;
  const int tile_i0 = tile * a.tile_w;
  const int wlo = sub * J * G::CW;                                     // warp's first output, tile-relative
  const int tile_n = min(a.tile_w, (int)d.n_f0 - tile_i0);             // valid f0 in this tile
  const int warp_n = max(0, min(J * G::CW, tile_n - wlo));             // valid outputs of this warp
  const int i_first = tile_i0 + wlo;
  const bool last_ok = warp_n > G::CW * (J - 1);  // the warp's last chunk holds valid outputs (else: skipped)
  typename G::template State<J> st;
  G::template init<J>(st, extra0, 32u * (uint32_t)n_cw);
  unsigned ties = 0;
  // row-weighted gather: the sky-dependent part of a(t; n), b(t; n) of this warp's point, in shared memory
  FtSkyPoint* skyp = reinterpret_cast<FtSkyPoint*>(reinterpret_cast<unsigned char*>(reinterpret_cast<FtPoint*>(bars + 2 * NS) + n_cw) +
                                                   256 * (size_t)n_cw) + warp;
  if (G::ROWW) {
    if (lane == 0) *skyp = ft_sky_point(sp->nx, sp->ny, sp->nz);
    __syncwarp();
  }
  const uint32_t lane_bytes = ring0 + 4u * (uint32_t)lane;
  uint32_t stage_addr = lane_bytes;
  // barriers of the current stage: full at fb, empty at fb + 8 NS; advanced by addition, reset when the ring wraps
  uint32_t fb = full0;
  const uint32_t fb_end = full0 + 8u * (uint32_t)NS, stage_bytes = (uint32_t)kRPS * row_bytes;
  uint32_t ph = 0;

  // (staggering the block phase of the warps of a CTA, so that they do not compute their track entries at the same
  // time, was measured: +0.6 % on config 4, 0 on configs 2 and 3, -1.6 % on K2B, -10 % on K2H -- not used)
  for (int a0 = 0; a0 < n_sft; a0 += 32) {
    // -- A1/A2: this lane's SFT ---------------------------------------------------------------------
    uint32_t entry = 0;
    if (a0 + lane < n_sft && warp_n > 0)
      entry = ft_tile_entry(d, *sp, a0 + lane, kst[a0 + lane], i_first, warp_n, a.copy_floats, &ties, a.err);
    sts_u32(etab + 4u * (uint32_t)lane, entry);
    if (G::ROWW) {
      float uf = 0.f;
      if (a0 + lane < n_sft) uf = (float)ft_antenna_u(d.ant + 9 * (size_t)(a0 + lane), *skyp);   // a^2 + b^2 (Eq. 4)
      sts_u32(wtab + 4u * (uint32_t)lane, __float_as_uint(uf));
    }
    __syncwarp();
    // -- A4: gather + reduce over the block's SFTs, one ring stage (kRPS rows) at a time ------------
    const int n_rows = min(32, n_sft - a0);
    // `rows` = kRPS for the full stages of the block (the loop below walks the entry table by pointer, so a stage
    // costs no index arithmetic); the ragged last stage of the last block comes after it
    auto stage = [&](uint32_t ep, int rows) {
      uint32_t e4[kRPS], u4[kRPS];
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(e4[0]), "=r"(e4[1]), "=r"(e4[2]), "=r"(e4[3]) : "r"(ep));
      if (G::ROWW)
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(u4[0]), "=r"(u4[1]), "=r"(u4[2]), "=r"(u4[3]) : "r"(ep + 128u * (uint32_t)n_cw));
      mbar_wait(fb, ph);
      if (rows == kRPS && (e4[0] | e4[1] | e4[2] | e4[3]) < 8192u) {
        // a full stage and no break in this warp's range in any of its rows (the common case): straight-line body
        if constexpr (G::PAIRS) {
          G::template rows_fast_pair<J>(st, e4[0], e4[1], stage_addr, stage_addr + row_bytes, copy_pitch, last_ok);
          G::template rows_fast_pair<J>(st, e4[2], e4[3], stage_addr + 2u * row_bytes, stage_addr + 3u * row_bytes, copy_pitch, last_ok);
        } else {
#pragma unroll
          for (int r = 0; r < kRPS; ++r)
            G::template row_fast<J>(st, e4[r], stage_addr + (uint32_t)r * row_bytes, copy_pitch, last_ok,
                                    G::ROWW ? __uint_as_float(u4[r]) : 1.f);
        }
      } else {
#pragma unroll
        for (int r = 0; r < kRPS; ++r) {
          if (r < rows) {
            const uint32_t e = e4[r];
            const uint32_t base = stage_addr + (uint32_t)r * row_bytes;
            const float u = G::ROWW ? __uint_as_float(u4[r]) : 1.f;
            if (e < 8192u) G::template row_fast<J>(st, e, base, copy_pitch, last_ok, u);   // no break in this warp's range
            else G::template row_break<J>(st, e, base, copy_pitch, lane, u);
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(fb + 8u * (uint32_t)NS);
      fb += 8u; stage_addr += stage_bytes;
      if (fb == fb_end) { fb = full0; ph ^= 1u; stage_addr = lane_bytes; }
    };
    const uint32_t ep_end = etab + 4u * (uint32_t)(n_rows & ~(kRPS - 1));
    for (uint32_t ep = etab; ep != ep_end; ep += 4u * kRPS) stage(ep, kRPS);
    if (n_rows & (kRPS - 1)) stage(ep_end, n_rows & (kRPS - 1));
    G::template block_end<J>(st, a0 / 32 + 1);
  }

  // ---- A5/A6: epilogue ---------------------------------------------------------------------------
  if (a.near_ties) {
    for (int o = 16; o > 0; o >>= 1) ties += __shfl_xor_sync(0xffffffffu, ties, o);
    if (lane == 0 && pt_active && ties) atomicAdd(a.near_ties, (unsigned long long)ties);
  }
  double add_back = a.add_back, scale = 1.0, z_mu = a.z_mu, z_is = a.z_inv_sigma;
  if (G::ROWW) {
    // Eq. (5): the weights of this point are u_a r_a / sum_b u_b r_b; sigma_G^2 = sum w^2 (Eq. 14 on the P = s/2 scale)
    const uint64_t i_sky = pt / ((uint64_t)d.n_ap * (uint64_t)d.n_porb * (uint64_t)d.n_tasc * (uint64_t)d.n_f1);
    const double w_sum = a.sky_norm[4 * i_sky], w_sq = a.sky_norm[4 * i_sky + 1], w_cb = a.sky_norm[4 * i_sky + a.norm_cb];
    add_back = w_cb;
    scale = 1.0 / w_sum;
    const double sigma = sqrt(w_sq) * scale;
    z_mu = 1.0; z_is = 1.0 / sigma;
    if (a.out_sigma && lane == 0 && sub == 0 && tile == 0 && pt_active) a.out_sigma[pt] = (float)sigma;
  }
  if (!pt_active) return;
  G::template finalize<J>(st);
  const int64_t box0 = a.pbox ? (int64_t)__ldg(a.pbox + pt) * a.n_bands : 0;
#pragma unroll
  for (int j = 0; j < J; ++j) {
#pragma unroll
    for (int c = 0; c < G::PER; ++c) {
      const int ii = G::CW * j + G::PER * lane + c;
      if (ii < warp_n) {
        const int64_t i = i_first + ii;
        const uint64_t idx = pt * (uint64_t)d.n_f0 + (uint64_t)i;
        const uint64_t o = a.glist ? (group_l * (uint64_t)a.R + (uint64_t)r_pt) * (uint64_t)d.n_f0 + (uint64_t)i
                                              : idx - a.out_base;
        double vd; int32_t cnt;
        G::template result<J>(st, j, c, add_back, &vd, &cnt);
        if (G::ROWW) vd *= scale;
        const float v = (float)vd;
        if (!G::HASCNT) cnt = __float2int_rn(v);   // (the 0/1 hit map gathered as fp32: the sum is the integer count)
        const float key = a.zmode ? (float)((vd - z_mu) * z_is) : v;
        if (a.out_f) a.out_f[o] = a.out_key ? key : v;
        if (a.out_i) a.out_i[o] = cnt;
        if (a.has_sel && (!G::VETO || cnt >= a.sel.veto_floor)) {   // (VETO: number-count floor from the count in registers)
          const int box = (int)(box0 + i / a.bpb);
          if (key >= __ldg(a.sel.thr + box)) ft_select_append(a.sel, box, key, idx);
        }
      }
    }
  }
}

}  // namespace
#endif  // __CUDACC__
