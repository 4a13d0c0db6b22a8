// Tile kernel for NARROW bands with a ragged tail: two outer points per consumer warp.
//
// A band of n_f0 = 32 JA + t f0 values with 1 <= t <= 16 costs the plain kernel JA + 1 shared-memory loads per
// (point, SFT), the last one for t lanes only (config 3: 450 f0 = 14 x 32 + 2: 6.7 % of the wavefronts).  Here a
// warp owns TWO consecutive outer points A, B and J = 2 JA + 1 chunks: chunks [0, JA) are A's f0 [0, 32 JA), chunks
// [JA, 2 JA) are B's, and the last chunk holds both tails (lanes [0, t): A's f0 32 JA + lane, lanes [t, 2t): B's f0
// 32 JA + lane - t).  2 JA + 1 loads per TWO (point, SFT) rows, twice the points per staged strip (half the TMA
// writes per evaluation), the same accumulators per thread as the wide-band kernel (J = 29 for config 3).
// Everything else -- producer ring, canonical track entries (one per point and SFT), epilogue with the fused
// selection -- is ft_tile_dev.cuh's; gathers fp32 pixels like ft_tile_kernel (Q, the weighted hit map, the 0/1 map).
#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int JA>
__device__ __forceinline__ void ft_tile2_body(const FtDev& d, const FtTileArgs& a) {
  constexpr int J = 2 * JA + 1;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const FtCtaWork cw = ft_cta_work<true>(a);                        // (one f0 tile; the split tail of a launch: part of a group)
  const int n_cw = cw.R_cta / 2;                              // consumer warps (points per CTA are even)
  const uint64_t group_l = cw.group_l;
  const uint64_t group = a.glist ? (uint64_t)__ldg(a.glist + group_l) : group_l;
  if (a.gskip && ((__ldg(a.gskip + (group >> 5)) >> (group & 31)) & 1u)) return;
  const int n_sft = (int)d.n_sft;
  const int NS = a.n_stages;
  const uint32_t row_bytes = 4u * (uint32_t)a.pitch;
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
  const int32_t* kst = a.kst;
  if (warp == n_cw) {
    ft_tile_produce<GatherF32>(d, a, kst, n_sft, NS, ring0, full0, empty0, row_bytes, lane);
    return;
  }
  if (warp > n_cw) return;

  // ---- consumers: points A = first + 2 warp, B = A + 1 ---------------------------------------------
  const int n_f0 = (int)d.n_f0;
  const int t = n_f0 - 32 * JA;                               // f0 per point in the shared tail chunk, 1 .. 16
  const int r_pt = cw.part * cw.R_cta + 2 * warp;             // A's place in its group
  uint64_t ptA = a.pt_begin + group * (uint64_t)a.R + (uint64_t)r_pt, ptB = ptA + 1;
  const bool actA = ptA < a.pt_end, actB = ptB < a.pt_end;
  if (!actA) ptA = a.pt_end - 1;   // keep the barrier protocol; results are discarded
  if (!actB) ptB = a.pt_end - 1;
  FtPoint* sp = reinterpret_cast<FtPoint*>(bars + 2 * NS) + 2 * warp;
  if (lane == 0) { sp[0] = ft_decode_point(d, ptA); sp[1] = ft_decode_point(d, ptB); }
  __syncwarp();
  // per-warp tables of the packed track entries of the current SFT block: A's 32 | B's 32
  const uint32_t etab = smem_u32(reinterpret_cast<FtPoint*>(bars + 2 * NS) + 2 * n_cw) + 256u * (uint32_t)warp;
  const bool tailB = lane >= t && lane < 2 * t;
  float acc[J];
#pragma unroll
  for (int j = 0; j < J; ++j) acc[j] = 0.f;
  unsigned tiesA = 0, tiesB = 0;
  const uint32_t lane_bytes = ring0 + 4u * (uint32_t)lane;
  uint32_t stage_addr = lane_bytes;
  uint32_t fb = full0;
  const uint32_t fb_end = full0 + 8u * (uint32_t)NS, stage_bytes = (uint32_t)kRPS * row_bytes;
  uint32_t ph = 0;

  // one row, no break in either point's range: 2 JA + 1 conflict-free loads
  auto row2_fast = [&](uint32_t eA, uint32_t eB, uint32_t base) {
    const uint32_t adA = base + 4u * eA;
    const uint32_t adB = base + 4u * eB - 128u * (uint32_t)JA;       // + 128 j, j in [JA, 2 JA): B's chunk j - JA
    const uint32_t adT = tailB ? base + 4u * eB + 128u * (uint32_t)JA - 4u * (uint32_t)t : adA + 128u * (uint32_t)JA;
    float v[J];
#pragma unroll
    for (int j = 0; j < JA; ++j) v[j] = lds_f32(adA + 128u * j);
#pragma unroll
    for (int j = JA; j < 2 * JA; ++j) v[j] = lds_f32(adB + 128u * j);
    v[2 * JA] = lds_f32(adT);
#pragma unroll
    for (int j = 0; j + 1 < J; j += 2) ft_add2(acc[j], acc[j + 1], v[j], v[j + 1]);
    acc[J - 1] += v[J - 1];
  };
  // one row with a break in A's and / or B's range: per-lane select between the two shifts of the point
  auto row2_slow = [&](uint32_t eA, uint32_t eB, uint32_t base) {
    const uint32_t loA = base + 4u * (eA & 8191u), hiA = (eA & (1u << 24)) ? loA - 4u : loA + 4u;
    const uint32_t loB = base + 4u * (eB & 8191u), hiB = (eB & (1u << 24)) ? loB - 4u : loB + 4u;
    const int relA = (int)((eA >> 13) & 2047u), relB = (int)((eB >> 13) & 2047u);
    const int tlA = relA ? relA - lane : 0x7fffffff, tlB = relB ? relB - lane : 0x7fffffff;   // (0: no break)
#pragma unroll
    for (int j = 0; j < JA; ++j) acc[j] += lds_f32(((32 * j >= tlA) ? hiA : loA) + 128u * j);
#pragma unroll
    for (int j = 0; j < JA; ++j) acc[JA + j] += lds_f32(((32 * j >= tlB) ? hiB : loB) + 128u * j);
    const uint32_t adT = tailB ? ((32 * JA - t >= tlB) ? hiB : loB) + 128u * (uint32_t)JA - 4u * (uint32_t)t
                               : ((32 * JA >= tlA) ? hiA : loA) + 128u * (uint32_t)JA;
    acc[2 * JA] += lds_f32(adT);
  };

  for (int a0 = 0; a0 < n_sft; a0 += 32) {
    // -- A1/A2: this lane's SFT, both points -----------------------------------------------------------
    uint32_t entA = 0, entB = 0;
    if (a0 + lane < n_sft) {
      const int ks = kst[a0 + lane];
      entA = ft_tile_entry(d, sp[0], a0 + lane, ks, 0, n_f0, a.copy_floats, &tiesA, a.err);
      entB = ft_tile_entry(d, sp[1], a0 + lane, ks, 0, n_f0, a.copy_floats, &tiesB, a.err);
    }
    sts_u32(etab + 4u * (uint32_t)lane, entA);
    sts_u32(etab + 128u + 4u * (uint32_t)lane, entB);
    __syncwarp();
    // -- A4: gather + reduce, one ring stage at a time ---------------------------------------------------
    const int n_rows = min(32, n_sft - a0);
    auto stage = [&](uint32_t ep, int rows) {
      uint32_t eA[kRPS], eB[kRPS];
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(eA[0]), "=r"(eA[1]), "=r"(eA[2]), "=r"(eA[3]) : "r"(ep));
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(eB[0]), "=r"(eB[1]), "=r"(eB[2]), "=r"(eB[3]) : "r"(ep + 128u));
      mbar_wait(fb, ph);
      if (rows == kRPS && (eA[0] | eA[1] | eA[2] | eA[3] | eB[0] | eB[1] | eB[2] | eB[3]) < 8192u) {
#pragma unroll
        for (int r = 0; r < kRPS; ++r) row2_fast(eA[r], eB[r], stage_addr + (uint32_t)r * row_bytes);
      } else {
#pragma unroll
        for (int r = 0; r < kRPS; ++r) {
          if (r < rows) {
            const uint32_t base = stage_addr + (uint32_t)r * row_bytes;
            if ((eA[r] | eB[r]) < 8192u) row2_fast(eA[r], eB[r], base);
            else row2_slow(eA[r], eB[r], base);
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
  }

  // ---- A5/A6: epilogue --------------------------------------------------------------------------------
  if (a.near_ties) {
    unsigned ties = (actA ? tiesA : 0u) + (actB ? tiesB : 0u);
    for (int o = 16; o > 0; o >>= 1) ties += __shfl_xor_sync(0xffffffffu, ties, o);
    if (lane == 0 && ties) atomicAdd(a.near_ties, (unsigned long long)ties);
  }
  if (!actA) return;
  const int64_t boxA = a.pbox ? (int64_t)__ldg(a.pbox + ptA) * a.n_bands : 0;
  const int64_t boxB = a.pbox ? (int64_t)__ldg(a.pbox + ptB) * a.n_bands : 0;
#pragma unroll
  for (int j = 0; j < J; ++j) {
    bool isB, valid;
    int i;
    if (j < JA) { isB = false; i = 32 * j + lane; valid = true; }
    else if (j < 2 * JA) { isB = true; i = 32 * (j - JA) + lane; valid = actB; }
    else { isB = tailB; i = 32 * JA + (tailB ? lane - t : lane); valid = lane < t || (tailB && actB); }
    if (valid) {
      const uint64_t pt = isB ? ptB : ptA;
      const uint64_t idx = pt * (uint64_t)n_f0 + (uint64_t)i;
      const uint64_t o = a.glist ? (group_l * (uint64_t)a.R + (uint64_t)r_pt + (isB ? 1u : 0u)) * (uint64_t)n_f0 + (uint64_t)i
                                 : idx - a.out_base;
      const double vd = (double)acc[j] + a.add_back;
      const float v = (float)vd;
      const float key = a.zmode ? (float)((vd - a.z_mu) * a.z_inv_sigma) : v;
      if (a.out_f) a.out_f[o] = a.out_key ? key : v;
      if (a.out_i) a.out_i[o] = __float2int_rn(v);   // (the 0/1 hit map gathered as fp32: the sum is the integer count)
      if (a.has_sel) {
        const int box = (int)((isB ? boxB : boxA) + i / a.bpb);
        if (key >= __ldg(a.sel.thr + box)) ft_select_append(a.sel, box, key, idx);
      }
    }
  }
}

template <int JA>
__global__ void __maxnreg__(ft_tile_max_regs(2 * JA + 1))
ft_tile2_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  ft_tile2_body<JA>(d, a);
}

template <int JA>
cudaError_t launch2_JA(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  const cudaError_t e = ft_tile_allow_smem((const void*)ft_tile2_kernel<JA>);
  if (e != cudaSuccess) return e;
  ft_tile2_kernel<JA><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

// JA = n_f0 / 32 main chunks per point (1 .. 15); the kernel's chunk count is J = 2 JA + 1
cudaError_t ft_tile2_launch(int JA, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s) {
  switch (JA) {
#define FT_CASE(j) case j: return launch2_JA<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(9) FT_CASE(10)
    FT_CASE(11) FT_CASE(12) FT_CASE(13) FT_CASE(14) FT_CASE(15)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}
