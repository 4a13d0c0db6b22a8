// Tile kernel K2: the hot path of the track statistics (PAPER.md:53 Eq. 2, :64 Eq. 3, :95 Eq. 7) for
// product grids whose f0 step equals the spectrogram bin width (Eq. A1 :554, reading R14).
//
// One CTA = R outer points (everything of a template but f0) x one f0 tile.  A producer warp streams
// the spectrogram rows of the tile, one contiguous strip per SFT, into a shared-memory ring with TMA
// bulk copies (cp.async.bulk + mbarrier complete_tx); the strip bounds are point-independent and
// come from the plan.  Each consumer warp owns ONE outer point and J consecutive 32-wide f0 chunks.
// Per block of 32 SFTs every lane computes, for its own SFT, the canonical fp64 track at the first
// and last f0 of the warp's range: along f0 the bin index is k_i = i + s with at most one break
// (reading R6: x_i - i drifts by (D-1) per step and 32 J |D-1| < 1), so (s, break position) is the
// whole track of the warp for that SFT.  The break is located with the canonical arithmetic itself
// (estimate, verify, bisect), so bins are bit-identical to the plain definition except within 1e-9
// bin of a rounding tie (counted).  The main loop is then, per SFT, one shuffle (the lane's packed
// entry) and J x (LDS.32 + FADD): a gather from shared memory, fp32 accumulation over the centred
// array.  Weights are folded into the gathered array beforehand
// (Q = w P, or the 0/1 hit map for the number count), so both statistics are the same kernel.
#include <algorithm>
#include <cmath>
#include <vector>

#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tile_max_regs(J))
ft_tile_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
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
#pragma unroll
  for (int j = 0; j < J; ++j) acc[j] = 0.f;
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
      if (a.out_i) a.out_i[o] = __float2int_rn(v);
      if (a.has_sel) {
        const int band = (int)(i / a.bpb);
        if (v >= __ldg(a.sel.thr + band)) ft_select_append(a.sel, band, v, idx);
      }
    }
  }
}

// min / max over the sky axis of v_alpha . n / c, per SFT (for the point-independent strip bounds)
__global__ void __launch_bounds__(256)
ft_vrange_kernel(const double* __restrict__ vel, const double* __restrict__ sky, int64_t n_sky,
                 double* __restrict__ vrange) {
  __shared__ double smin[256], smax[256];
  const int64_t a = blockIdx.x;
  const double vx = vel[3 * a], vy = vel[3 * a + 1], vz = vel[3 * a + 2];
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t i = threadIdx.x; i < n_sky; i += blockDim.x) {
    const double v = (vx * sky[3 * i] + vy * sky[3 * i + 1] + vz * sky[3 * i + 2]) / FT_C_LIGHT;
    lo = fmin(lo, v); hi = fmax(hi, v);
  }
  smin[threadIdx.x] = lo; smax[threadIdx.x] = hi;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      smin[threadIdx.x] = fmin(smin[threadIdx.x], smin[threadIdx.x + o]);
      smax[threadIdx.x] = fmax(smax[threadIdx.x], smax[threadIdx.x + o]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { vrange[2 * a] = smin[0]; vrange[2 * a + 1] = smax[0]; }
}

__global__ void ft_hitmap_kernel(const float* __restrict__ P, float rho, float* __restrict__ H, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    H[i] = (P[i] > rho) ? 1.f : 0.f;
}

// A0: fold the weights into the gathered array and remove a per-row constant, one CTA per SFT row:
//   q = fl(w P);  c_a = fl(mean_k q);  Q[a][k] = fl(q - c_a).
// Removing c_a keeps the running sums of K2 near zero (a random walk of ~sqrt(n_sft) pixel sigmas
// instead of a ramp to n_sft means), so one level of fp32 accumulation is enough (DESIGN.md
// "Accumulation"); sum_a c_a is added back in fp64 in the epilogue.
__global__ void __launch_bounds__(256)
ft_fold_centered_kernel(const float* __restrict__ P, const float* __restrict__ w_sft,
                        const float* __restrict__ w_bin, float* __restrict__ Q,
                        float* __restrict__ c_row, int64_t n_bins, int64_t ld) {
  __shared__ double red[256];
  const int64_t a = blockIdx.x;
  const float* Pr = P + a * ld;
  const float* wr = w_bin ? w_bin + a * ld : nullptr;
  const float ws = w_sft ? w_sft[a] : 0.f;
  double sum = 0.0;
  for (int64_t k = threadIdx.x; k < n_bins; k += blockDim.x)
    sum += (double)__fmul_rn(wr ? wr[k] : ws, Pr[k]);
  red[threadIdx.x] = sum;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  const float c = (float)(red[0] / (double)n_bins);
  if (threadIdx.x == 0) c_row[a] = c;
  for (int64_t k = threadIdx.x; k < ld; k += blockDim.x)
    Q[a * ld + k] = (k < n_bins) ? __fsub_rn(__fmul_rn(wr ? wr[k] : ws, Pr[k]), c) : 0.f;
}

// J values the kernel is instantiated for (the plan rounds the per-warp chunk count up to one)
constexpr int kJList[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 15, 16, 20, 24, 28, 29, 30, 32};

template <int J>
cudaError_t launch_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  static bool configured = false;  // one attribute call per instantiation and process
  if (!configured) {
    const cudaError_t e = cudaFuncSetAttribute(ft_tile_kernel<J>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  ft_tile_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

cudaError_t launch_any(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launch_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16) FT_CASE(20) FT_CASE(24) FT_CASE(28) FT_CASE(29) FT_CASE(30) FT_CASE(32)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

void ft_tile_plan_free(FtTilePlan* p) {
  if (p->kst) cudaFree(p->kst);
  if (p->err) cudaFree(p->err);
  if (p->vr) cudaFree(p->vr);
  *p = FtTilePlan{};
}

cudaError_t ft_tile_plan(const FtDev& d, const FtTileHostIn& in, cudaStream_t s, FtTilePlan* plan,
                         std::string* why, int* launches, int mode) {
  *launches = 0;
  why->clear();
  FtTilePlan pl;  // geometry starts from defaults; the device buffers of *plan are kept and reused
  pl.kst = plan->kst; pl.kst_cap = plan->kst_cap; pl.err = plan->err; pl.vr = plan->vr; pl.vr_cap = plan->vr_cap;
  *plan = pl;     // (an ineligible return leaves a plan with buffers only)
  if (d.df0 != in.df && d.n_f0 > 1) { *why = "f0 step differs from the bin width"; return cudaSuccess; }
  if (!d.Q) { *why = "no folded array"; return cudaSuccess; }
  if (d.n_f0 > (1 << 30)) { *why = "more than 2^30 f0 values"; return cudaSuccess; }
  if (mode == 1 && d.n_sft > 65535) { *why = "packed number count holds 16-bit counters (n_sft <= 65535)"; return cudaSuccess; }
  // chunk = the f0 a warp covers with one load instruction: 32 (one fp32 pixel per lane) or 128 (4 packed hits)
  const int cw = mode == 1 ? 128 : 32;
  const int align = mode == 1 ? 16 : 4;   // strip start / length granularity in bins (16-byte TMA copies)
  const int64_t n_sft = d.n_sft;
  // --- tiling: n_tiles x wpp warps x J chunks of 32 f0, least issue slots (J+1.5 per chunk row) -----
  const int64_t chunks = (d.n_f0 + cw - 1) / cw;
  double best = 1e300;
  int bJ = 0, bW = 0; int64_t bT = 0;
  const int maxJ_eps = (int)std::floor(0.45 / ((double)cw * std::fmax(in.eps_bound, 1e-12)));
  for (int64_t nt = 1; nt <= chunks; ++nt) {
    if (in.force_tiles > 0 && nt != in.force_tiles) continue;
    const int64_t cpt = (chunks + nt - 1) / nt;
    if (nt > 1 && in.force_tiles <= 0 && (chunks + nt - 2) / (nt - 1) == cpt) continue;  // same tile size as nt-1
    for (int wpp = 1; wpp <= 4; ++wpp) {
      const int64_t Jn = (cpt + wpp - 1) / wpp;
      if (Jn > (mode == 0 ? 32 : 16)) continue;
      int J = 0;
      for (int c : kJList) if (c >= Jn) { J = c; break; }
      if (J == 0 || J > maxJ_eps) continue;
      const double cost = (double)nt * wpp * (J + 1.5) * (1.0 + 0.02 * (double)(nt - 1));
      if (cost < best) { best = cost; bJ = J; bW = wpp; bT = nt; }
    }
    if (cpt == 1) break;
  }
  if (bJ == 0) { *why = "Doppler spread too large for a single break per warp range"; return cudaSuccess; }
  pl.J = bJ; pl.wpp = bW;
  pl.mode = mode; pl.cw = cw;
  pl.tile_w = (int32_t)(((chunks + bT - 1) / bT) * cw);
  pl.n_tiles = (int32_t)((d.n_f0 + pl.tile_w - 1) / pl.tile_w);
  // default: 24-27 consumer warps per CTA (measured best on B200 at 72 registers: R = 12 at wpp = 2,
  // R = 6 at wpp = 4, R = 27 at wpp = 1); the packed kernel keeps 23 (80 registers)
  int R = in.points_per_cta > 0 ? in.points_per_cta : (mode != 0 ? 23 / pl.wpp : (pl.wpp == 1 ? 27 : 24 / pl.wpp));
  const int max_threads = mode == 1 ? ft_tile8_max_threads(pl.J) : (mode == 2 ? ft_tileb_max_threads(pl.J) : ft_tile_max_threads(pl.J));
  R = std::min<int>(R, (max_threads / 32 - 1) / pl.wpp);  // + 1 producer warp
  R = (int)std::min<uint64_t>((uint64_t)R, d.n_points);
  pl.R = std::max(R, 1);
  // --- point-independent strip bounds per (tile, SFT) -----------------------------------------------
  if (pl.vr_cap < 2 * (size_t)n_sft) {
    if (pl.vr) cudaFree(pl.vr);
    pl.vr = nullptr; pl.vr_cap = 0; plan->vr = nullptr; plan->vr_cap = 0;
    const cudaError_t ea = cudaMalloc(&pl.vr, sizeof(double) * 2 * n_sft);
    if (ea != cudaSuccess) return ea;
    pl.vr_cap = 2 * (size_t)n_sft; plan->vr = pl.vr; plan->vr_cap = pl.vr_cap;
  }
  ft_vrange_kernel<<<(unsigned)n_sft, 256, 0, s>>>(d.vel, d.sky, d.n_sky, pl.vr);
  *launches += 1;
  std::vector<double> vr(2 * (size_t)n_sft);
  cudaError_t e = cudaMemcpyAsync(vr.data(), pl.vr, sizeof(double) * 2 * n_sft, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return e;
  double bmax = 0.0;
  {
    double apm = 0.0, pmin = in.P_orb[0];
    for (int i = 0; i < d.n_ap; ++i) apm = std::fmax(apm, std::fabs(in.a_p[i]));
    for (int i = 0; i < d.n_porb; ++i) pmin = std::fmin(pmin, in.P_orb[i]);
    bmax = apm * FT_TWO_PI / pmin;
  }
  const double f1a = d.f1_start, f1b = d.f1_start + (double)(d.n_f1 - 1) * d.df1;
  std::vector<int32_t> kst((size_t)pl.n_tiles * n_sft);
  int64_t max_w = 0;
  for (int t = 0; t < pl.n_tiles; ++t) {
    const int64_t i_lo = (int64_t)t * pl.tile_w, i_hi = std::min<int64_t>(d.n_f0, i_lo + pl.tile_w) - 1;
    const double f0_lo = d.f0_start + (double)i_lo * d.df0, f0_hi = d.f0_start + (double)i_hi * d.df0;
    for (int64_t a = 0; a < n_sft; ++a) {
      const double dt = in.t_mid[a] - d.t_ref;
      const double g_lo = std::fmin(f1a * dt, f1b * dt), g_hi = std::fmax(f1a * dt, f1b * dt);
      const double D_lo = 1.0 + vr[2 * a] - bmax, D_hi = 1.0 + vr[2 * a + 1] + bmax;
      const double x_lo = ((f0_lo + g_lo) * D_lo - d.f_min) * d.inv_df;
      const double x_hi = ((f0_hi + g_hi) * D_hi - d.f_min) * d.inv_df;
      int64_t lo = (int64_t)std::floor(x_lo) - 1, hi = (int64_t)std::ceil(x_hi) + 1;
      lo = std::max<int64_t>(lo, 0);
      hi = std::min<int64_t>(hi, d.n_bins - 1);
      const int64_t k0 = lo / align * align;
      kst[(size_t)t * n_sft + a] = (int32_t)k0;
      max_w = std::max(max_w, hi - k0 + 1);
    }
  }
  pl.copy_floats = (int32_t)((max_w + align - 1) / align * align);
  int min_warp_n = cw * pl.J;
  for (int t = 0; t < pl.n_tiles; ++t) {
    const int64_t tile_n = std::min<int64_t>(pl.tile_w, d.n_f0 - (int64_t)t * pl.tile_w);
    for (int sub = 0; sub < pl.wpp; ++sub) {
      const int64_t wn = std::min<int64_t>(cw * pl.J, tile_n - (int64_t)sub * pl.J * cw);
      if (wn > 0) min_warp_n = (int)std::min<int64_t>(min_warp_n, wn);
    }
  }
  pl.pitch = (pl.copy_floats + cw * pl.J - min_warp_n + 8 + align - 1) / align * align;
  pl.pitch = std::max(pl.pitch, (cw * pl.J + 8 + align - 1) / align * align);  // warps without valid outputs read [0, cw J)
  if (pl.copy_floats > kMaxPitch + 1) { *why = "strip too wide for the packed track entry"; return cudaSuccess; }
  // --- shared-memory ring ---------------------------------------------------------------------------
  const int threads = (pl.R * pl.wpp + 1) * 32;
  const int regs_est = (mode == 2 ? 3 : 2) * pl.J + 30;
  int ctas = std::min(4, std::min(2048 / threads, 65536 / (threads * regs_est)));
  ctas = std::max(ctas, 1);
  const size_t row_bytes = (size_t)pl.pitch * 4;
  // per-warp state: point parameters, entry table; packed mode: the 16-bit counter levels
  const size_t state_bytes = (sizeof(FtPoint) + 128) * (size_t)(pl.R * pl.wpp) + 16 +
                             (mode == 1 ? (size_t)8 * pl.J * 32 * (pl.R * pl.wpp) : 0);
  int64_t rows_fit = 0;
  for (;; --ctas) {  // fewer CTAs per SM until the ring holds two stages
    const size_t budget = (size_t)(228 * 1024) / ctas - 2048;
    rows_fit = budget > state_bytes + 1024 ? (int64_t)((budget - 1024 - state_bytes) / row_bytes) : 0;
    if (rows_fit >= 2 * kRPS || ctas == 1) break;
  }
  if (rows_fit < 2 * kRPS) { *why = "strip does not fit shared memory twice"; return cudaSuccess; }
  rows_fit = std::min<int64_t>(rows_fit, 32);
  pl.rows_per_stage = kRPS;
  pl.n_stages = (int32_t)(rows_fit / kRPS);
  pl.ctas_per_sm = ctas;
  pl.smem_bytes = (size_t)pl.n_stages * pl.rows_per_stage * row_bytes + 2 * 8 * (size_t)pl.n_stages + state_bytes;
  if (pl.kst_cap < kst.size()) {
    if (pl.kst) cudaFree(pl.kst);
    pl.kst = nullptr; pl.kst_cap = 0; plan->kst = nullptr; plan->kst_cap = 0;
    e = cudaMalloc(&pl.kst, sizeof(int32_t) * kst.size());
    if (e != cudaSuccess) return e;
    pl.kst_cap = kst.size(); plan->kst = pl.kst; plan->kst_cap = pl.kst_cap;
  }
  if (!pl.err) {
    e = cudaMalloc(&pl.err, sizeof(int32_t));
    if (e != cudaSuccess) return e;
    plan->err = pl.err;
  }
  e = cudaMemcpyAsync(pl.kst, kst.data(), sizeof(int32_t) * kst.size(), cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(pl.err, 0, sizeof(int32_t), s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);  // kst (host vector) goes out of scope
  if (e != cudaSuccess) return e;
  *plan = pl;
  return cudaSuccess;
}

// Outer points of the threshold sample: one wave of CTA groups (148), more only when the bank is so large
// that the fused pass would append more than cap / 8 entries per band (appended ~ k * groups / sample groups).
uint64_t ft_tile_sample_points(const FtTilePlan& plan, uint64_t n_points, uint32_t k, uint32_t cap) {
  const uint64_t R = (uint64_t)plan.R;
  const uint64_t n_groups = (n_points + R - 1) / R;
  uint64_t n_sg = std::max<uint64_t>(148, (8ull * k * n_groups + cap - 1) / std::max<uint32_t>(cap, 1u));
  n_sg = std::min(n_sg, n_groups);
  return std::min(n_sg * R, n_points);
}

cudaError_t ft_launch_tile(const FtDev& d, const FtTilePlan& plan, const float* A, double add_back, uint64_t pt_begin,
                           uint64_t pt_end, float* out_f, int32_t* out_i, uint64_t out_base,
                           const FtSelectDev* sel, int32_t bpb, unsigned long long* near_ties,
                           cudaStream_t s, int* launches, uint32_t group_stride, uint64_t n_groups_strided, bool complement) {
  *launches = 0;
  if (pt_end <= pt_begin) return cudaSuccess;
  FtTileArgs a{};
  a.A = A; a.kst = plan.kst; a.err = plan.err;
  a.tile_w = plan.tile_w; a.n_tiles = plan.n_tiles; a.R = plan.R; a.wpp = plan.wpp;
  a.pitch = plan.pitch; a.copy_floats = plan.copy_floats;
  a.n_stages = plan.n_stages; a.add_back = add_back;
  a.out_f = out_f; a.out_i = out_i; a.out_base = out_base;
  if (sel) { a.sel = *sel; a.has_sel = 1; }
  a.bpb = bpb > 0 ? bpb : 1;
  a.near_ties = near_ties;
  a.group_stride = (group_stride > 1 && !complement) ? group_stride : 1;
  a.skip_stride = (group_stride > 1 && complement) ? group_stride : 1;
  a.skip_n = n_groups_strided;
  const unsigned block = (unsigned)((plan.R * plan.wpp + 1) * 32);
  const uint64_t max_groups = 0x7fffffffull / (uint64_t)plan.n_tiles;
  if (group_stride > 1) {  // strided sample (or its complement): one launch
    const uint64_t all_groups = (pt_end - pt_begin + plan.R - 1) / plan.R;
    const uint64_t n_launch = complement ? all_groups - n_groups_strided : n_groups_strided;
    if (n_groups_strided == 0 || n_groups_strided > all_groups || n_launch > max_groups) return cudaErrorInvalidValue;
    if (n_launch == 0) return cudaSuccess;
    a.pt_begin = pt_begin; a.pt_end = pt_end;
    const cudaError_t e = plan.mode == 1 ? ft_tile8_launch(plan.J, d, a, (unsigned)(n_launch * plan.n_tiles), block, plan.smem_bytes, s)
                        : plan.mode == 2 ? ft_tileb_launch(plan.J, d, a, (unsigned)(n_launch * plan.n_tiles), block, plan.smem_bytes, s)
                                         : launch_any(plan.J, d, a, (unsigned)(n_launch * plan.n_tiles), block, plan.smem_bytes, s);
    if (e == cudaSuccess) *launches = 1;
    return e;
  }
  uint64_t pt = pt_begin;
  while (pt < pt_end) {
    uint64_t groups = (pt_end - pt + plan.R - 1) / plan.R;
    if (groups > max_groups) groups = max_groups;
    a.pt_begin = pt;
    a.pt_end = std::min<uint64_t>(pt_end, pt + groups * plan.R);
    const cudaError_t e = plan.mode == 1 ? ft_tile8_launch(plan.J, d, a, (unsigned)(groups * plan.n_tiles), block, plan.smem_bytes, s)
                        : plan.mode == 2 ? ft_tileb_launch(plan.J, d, a, (unsigned)(groups * plan.n_tiles), block, plan.smem_bytes, s)
                                         : launch_any(plan.J, d, a, (unsigned)(groups * plan.n_tiles), block, plan.smem_bytes, s);
    if (e != cudaSuccess) return e;
    *launches += 1;
    pt = a.pt_end;
  }
  return cudaSuccess;
}

cudaError_t ft_launch_hitmap(const float* P, float rho, float* H, int64_t n, cudaStream_t s) {
  ft_hitmap_kernel<<<148 * 8, 256, 0, s>>>(P, rho, H, n);
  return cudaGetLastError();
}

cudaError_t ft_launch_fold_centered(const float* P, const float* w_sft, const float* w_bin, float* Q, float* c_row,
                                    int64_t n_sft, int64_t n_bins, int64_t ld, cudaStream_t s) {
  ft_fold_centered_kernel<<<(unsigned)n_sft, 256, 0, s>>>(P, w_sft, w_bin, Q, c_row, n_bins, ld);
  return cudaGetLastError();
}
