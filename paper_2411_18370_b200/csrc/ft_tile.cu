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
// bin of a rounding tie (counted).  The main loop is then, per SFT, one broadcast load of the packed
// entry and J x (LDS.32 + FADD): a gather from shared memory, fp32 accumulation over the centred
// array.  Weights are folded into the gathered array beforehand
// (Q = w P, the 0/1 hit map for the number count, w x hit for the weighted count), so every statistic is
// the same kernel.  The kernel body is ft_tile_body (ft_tile_dev.cuh); this file instantiates it for the
// plain fp32 gather and holds the host side: tiling choice, strip table, launch.
#include <algorithm>
#include <mutex>
#include <cmath>
#include <vector>

#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tile_max_regs(J))
ft_tile_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  ft_tile_body<J, GatherF32>(d, a);
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

// Strip table: first staged bin of (tile, SFT) and the widest strip of the plan (A3).  Bounds hold for every
// outer point of the grid: D within 1 + [vr_lo, vr_hi] -+ max a_p Omega, every f1 of the grid.
__global__ void __launch_bounds__(256)
ft_strips_kernel(const __grid_constant__ FtDev d, const double* __restrict__ vr, double bmax, int32_t tile_w,
                 int32_t align, int32_t* __restrict__ kst, int32_t* __restrict__ max_w) {
  const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int t = blockIdx.y;
  int w = 0;
  if (a < d.n_sft) {
    const int64_t i_lo = (int64_t)t * tile_w, i_hi = min(d.n_f0, i_lo + (int64_t)tile_w) - 1;
    const double f0_lo = d.f0_start + (double)i_lo * d.df0, f0_hi = d.f0_start + (double)i_hi * d.df0;
    const double f1a = d.f1_start, f1b = d.f1_start + (double)(d.n_f1 - 1) * d.df1;
    const double dt = d.t_mid[a] - d.t_ref;
    const double g_lo = fmin(f1a * dt, f1b * dt), g_hi = fmax(f1a * dt, f1b * dt);
    const double D_lo = 1.0 + vr[2 * a] - bmax, D_hi = 1.0 + vr[2 * a + 1] + bmax;
    const double x_lo = ((f0_lo + g_lo) * D_lo - d.f_min) * d.inv_df;
    const double x_hi = ((f0_hi + g_hi) * D_hi - d.f_min) * d.inv_df;
    int64_t lo = (int64_t)floor(x_lo) - 1, hi = (int64_t)ceil(x_hi) + 1;
    lo = max(lo, (int64_t)0);
    hi = min(hi, d.n_bins - 1);
    const int64_t k0 = lo / align * align;
    kst[(size_t)t * d.n_sft + a] = (int32_t)k0;
    w = (int)(hi - k0 + 1);
  }
  for (int o = 16; o > 0; o >>= 1) w = max(w, __shfl_xor_sync(0xffffffffu, w, o));
  if ((threadIdx.x & 31) == 0 && w > 0) atomicMax(max_w, w);
}

__global__ void ft_hitmap_kernel(const float* __restrict__ P, float rho, float* __restrict__ H, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    H[i] = (P[i] > rho) ? 1.f : 0.f;
}

// A0: fold the weights into the gathered array and remove a per-row constant, one CTA per SFT row:
//   q = fl(w p);  c_a = fl(mean_k q);  Q[a][k] = fl(q - c_a),   p = P (power) or [P > rho] (weighted count).
// Removing c_a keeps the running sums of K2 near zero (a random walk of ~sqrt(n_sft) pixel sigmas
// instead of a ramp to n_sft means), so one level of fp32 accumulation is enough (DESIGN.md
// "Accumulation"); sum_a c_a is added back in fp64 in the epilogue.  Also the row mean of w (per-bin weights).
__global__ void __launch_bounds__(256)
ft_fold_centered_kernel(const float* __restrict__ P, const float* __restrict__ w_sft,
                        const float* __restrict__ w_bin, float* __restrict__ Q,
                        float* __restrict__ c_row, double* __restrict__ w_row, int64_t n_bins, int64_t ld,
                        int hits, float rho) {
  __shared__ double red[256], redw[256];
  const int64_t a = blockIdx.x;
  const float* Pr = P + a * ld;
  const float* wr = w_bin ? w_bin + a * ld : nullptr;
  const float ws = w_sft ? w_sft[a] : 0.f;
  double sum = 0.0, sumw = 0.0;
  for (int64_t k = threadIdx.x; k < n_bins; k += blockDim.x) {
    const float w = wr ? wr[k] : ws;
    const float p = hits ? ((Pr[k] > rho) ? 1.f : 0.f) : Pr[k];
    sum += (double)__fmul_rn(w, p);
    sumw += (double)w;
  }
  red[threadIdx.x] = sum; redw[threadIdx.x] = sumw;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) { red[threadIdx.x] += red[threadIdx.x + o]; redw[threadIdx.x] += redw[threadIdx.x + o]; }
    __syncthreads();
  }
  const float c = (float)(red[0] / (double)n_bins);
  if (threadIdx.x == 0) {
    c_row[a] = c;
    if (w_row) w_row[a] = redw[0] / (double)n_bins;
  }
  for (int64_t k = threadIdx.x; k < ld; k += blockDim.x) {
    const float p = hits ? ((k < n_bins && Pr[k] > rho) ? 1.f : 0.f) : (k < n_bins ? Pr[k] : 0.f);
    Q[a * ld + k] = (k < n_bins) ? __fsub_rn(__fmul_rn(wr ? wr[k] : ws, p), c) : 0.f;
  }
}

// J values the kernel is instantiated for (the plan rounds the per-warp chunk count up to one)
constexpr int kJList[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 15, 16, 20, 24, 28, 29, 30, 32};

template <int J>
cudaError_t launch_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  const cudaError_t e = ft_tile_allow_smem((const void*)ft_tile_kernel<J>);
  if (e != cudaSuccess) return e;
  ft_tile_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

int ft_sm_count() {
  static std::mutex mu;
  static int count[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  std::lock_guard<std::mutex> lock(mu);
  if (count[dev] == 0) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    count[dev] = n;
  }
  return count[dev];
}

// The opt-in to > 48 KB of dynamic shared memory is per function AND per device: remember the devices a
// function has been configured on (a bit per device; a process may drive several GPUs).
cudaError_t ft_tile_allow_smem(const void* func) {
  struct Seen { const void* f; unsigned long long mask; };
  static Seen seen[128];
  static int n_seen = 0;
  static std::mutex mu;                       // handles on different host threads share this table
  std::lock_guard<std::mutex> lock(mu);
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const unsigned long long bit = 1ull << (dev & 63);
  for (int i = 0; i < n_seen; ++i)
    if (seen[i].f == func) {
      if (seen[i].mask & bit) return cudaSuccess;
      e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
      if (e == cudaSuccess) seen[i].mask |= bit;
      return e;
    }
  e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
  if (e == cudaSuccess && n_seen < 128) seen[n_seen++] = Seen{func, bit};
  return e;
}

cudaError_t ft_tile_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launch_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16) FT_CASE(20) FT_CASE(24) FT_CASE(28) FT_CASE(29) FT_CASE(30) FT_CASE(32)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

void ft_tile_plan_free(FtTilePlan* p) {
  if (p->kst) cudaFree(p->kst);   // (err belongs to the handle)
  *p = FtTilePlan{};
}

cudaError_t ft_launch_vrange(const FtDev& d, double* vr, cudaStream_t s) {
  ft_vrange_kernel<<<(unsigned)d.n_sft, 256, 0, s>>>(d.vel, d.sky, d.n_sky, vr);
  return cudaGetLastError();
}

// Tiling of the f0 axis for one gather mode: n_tiles x wpp warps x J chunks of cw f0, least issue slots
// (J + 1.5 per chunk row).  Host arithmetic only.
bool ft_tile_choose(const FtDev& d, const FtTileHostIn& in, int mode, FtTilePlan* plan, std::string* why) {
  why->clear();
  FtTilePlan pl;  // geometry starts from defaults; the device buffers of *plan are kept and reused
  pl.kst = plan->kst; pl.kst_cap = plan->kst_cap; pl.err = plan->err;
  *plan = pl;     // (an ineligible return leaves a plan with buffers only)
  if (d.df0 != in.df && d.n_f0 > 1) { *why = "f0 step differs from the bin width"; return false; }
  if (!d.Q) { *why = "no folded array"; return false; }
  if (d.n_f0 > (1 << 30)) { *why = "more than 2^30 f0 values"; return false; }
  if (mode == 1 && d.n_sft > 65535) { *why = "packed number count holds 16-bit counters (n_sft <= 65535)"; return false; }
  if (mode == 2 && (d.n_sft > 65535 || d.n_sft < 64)) { *why = "one-pass kernel: 16-bit counters, pixels rounded to 18 bits (64 <= n_sft <= 65535)"; return false; }
  // chunk = the f0 a warp covers with one load instruction: 32 (one fp32 pixel per lane) or 128 (4 packed hits)
  const int cw = mode == 1 ? 128 : 32;
  const int64_t chunks = (d.n_f0 + cw - 1) / cw;
  double best = 1e300;
  int bJ = 0, bW = 0; int64_t bT = 0;
  // a warp's range may hold one break: cw J |D - 1| < 0.45 (clamped before the cast: eps -> 0 for a_p = 0, v = 0)
  const int maxJ_eps = (int)std::min(64.0, std::floor(0.45 / ((double)cw * std::fmax(in.eps_bound, 1e-12))));
  const double spread_bins = 2.0 * in.eps_bound * (d.f0_start + (double)d.n_f0 * d.df0) / in.df + 16.0;   // Doppler spread of a strip
  for (int64_t nt = 1; nt <= chunks; ++nt) {
    if (in.force_tiles > 0 && nt != in.force_tiles) continue;
    const int64_t cpt = (chunks + nt - 1) / nt;
    if (nt > 1 && in.force_tiles <= 0 && (chunks + nt - 2) / (nt - 1) == cpt) continue;  // same tile size as nt-1
    for (int wpp = 1; wpp <= 4; ++wpp) {
      const int64_t Jn = (cpt + wpp - 1) / wpp;
      if (Jn > ((mode == 0 || mode == 3) ? 32 : 16)) continue;
      int J = 0;
      for (int c : kJList) if (c >= Jn) { J = c; break; }
      if (J == 0 || J > maxJ_eps) continue;
      // shared-memory wavefronts per (outer point, SFT): the loads of the tile's chunks, the entry reads, and the point's
      // share of the TMA writes of the strip (tile + Doppler spread, 32 floats per wavefront, R points per CTA); every
      // further tile costs ~4 % (measured on configs 2 and 4: two tiles win on 3 600 f0, lose on 1 800)
      const double R_def = wpp == 1 ? 27.0 : (double)(24 / wpp);
      const double strip_wf = ((double)cpt * cw + spread_bins) / 32.0;
      const double cost = (double)nt * ((double)std::min<int64_t>(cpt, (int64_t)wpp * J) + 0.5 * wpp + strip_wf / R_def) *
                          (1.0 + 0.04 * (double)(nt - 1));
      if (cost < best) { best = cost; bJ = J; bW = wpp; bT = nt; }
    }
    if (cpt == 1) break;
  }
  if (bJ == 0) { *why = "Doppler spread too large for a single break per warp range"; return false; }
  pl.J = bJ; pl.wpp = bW;
  pl.mode = mode; pl.cw = cw;
  pl.align = mode == 1 ? 16 : 4;   // strip start / length granularity in bins (16-byte TMA copies)
  pl.tile_w = (int32_t)(((chunks + bT - 1) / bT) * cw);
  pl.n_tiles = (int32_t)((d.n_f0 + pl.tile_w - 1) / pl.tile_w);
  // default: 24-27 consumer warps per CTA (measured best on B200 at 72 registers: R = 12 at wpp = 2,
  // R = 6 at wpp = 4, R = 27 at wpp = 1; the one-pass kernel the same, its thread limit permitting); the 80-register
  // kernels keep 23
  int R = in.points_per_cta > 0 ? in.points_per_cta : (mode == 1 ? 23 / pl.wpp : (pl.wpp == 1 ? 27 : 24 / pl.wpp));
  const int max_threads = mode == 1 ? ft_tile8_max_threads(pl.J) : mode == 2 ? ft_tileb_max_threads(pl.J)
                        : mode == 3 ? ft_tilew_max_threads(pl.J) : ft_tile_max_threads(pl.J);
  R = std::min<int>(R, (max_threads / 32 - 1) / pl.wpp);  // + 1 producer warp
  R = (int)std::min<uint64_t>((uint64_t)R, d.n_points);
  pl.R = std::max(R, 1);
  // Narrow band with a ragged tail (n_f0 = 32 JA + t, 1 <= t <= 16, one tile, one warp per point): two points per
  // warp, their tails sharing one chunk (ft_tile2.cu): 2 JA + 1 loads per two (point, SFT) rows instead of 2 JA + 2
  if (mode == 0 && in.tail_packing && pl.n_tiles == 1 && pl.wpp == 1 && d.n_points >= 2) {
    const int JA = (int)(d.n_f0 / 32), t = (int)(d.n_f0 % 32);
    if (JA >= 1 && JA <= 15 && t >= 1 && t <= 16 && JA + 1 <= maxJ_eps) {
      pl.ppw = 2;
      pl.J = 2 * JA + 1;
      const int warps_max = ft_tile_max_threads(pl.J) / 32 - 1;
      int warps = in.points_per_cta > 0 ? std::max(1, in.points_per_cta / 2) : std::min(24, warps_max);   // (R = 48: many divisors for the split tail)
      warps = std::min(warps, warps_max);
      warps = (int)std::min<uint64_t>((uint64_t)warps, (d.n_points + 1) / 2);
      pl.R = 2 * warps;
    }
  }
  *plan = pl;
  return true;
}

// Enqueue the strip table of a chosen plan; *max_w_dev (zeroed by the caller) receives the widest strip.
cudaError_t ft_tile_strips(const FtDev& d, const FtTileHostIn& in, FtTilePlan* plan, const double* vr_dev,
                           int32_t* max_w_dev, cudaStream_t s) {
  const size_t need = (size_t)plan->n_tiles * (size_t)d.n_sft;
  if (plan->kst_cap < need) {
    if (plan->kst) cudaFree(plan->kst);
    plan->kst = nullptr; plan->kst_cap = 0;
    const cudaError_t e = cudaMalloc(&plan->kst, sizeof(int32_t) * need);
    if (e != cudaSuccess) return e;
    plan->kst_cap = need;
  }
  double apm = 0.0, pmin = in.P_orb[0];
  for (int i = 0; i < d.n_ap; ++i) apm = std::fmax(apm, std::fabs(in.a_p[i]));
  for (int i = 0; i < d.n_porb; ++i) pmin = std::fmin(pmin, in.P_orb[i]);
  const double bmax = apm * FT_TWO_PI / pmin;
  const dim3 grid((unsigned)((d.n_sft + 255) / 256), (unsigned)plan->n_tiles);
  ft_strips_kernel<<<grid, 256, 0, s>>>(d, vr_dev, bmax, plan->tile_w, plan->align, plan->kst, max_w_dev);
  return cudaGetLastError();
}

// Shared-memory ring of a plan whose widest strip is known.
bool ft_tile_finish(const FtDev& d, FtTilePlan* plan, int32_t max_w, std::string* why) {
  FtTilePlan& pl = *plan;
  const int cw = pl.cw, align = pl.align, mode = pl.mode;
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
  if (pl.ppw == 2) pl.pitch = (pl.copy_floats + 32 + 8 + align - 1) / align * align;   // idle tail lanes read up to 31 bins past a strip
  if (pl.copy_floats > kMaxPitch + 1) { *why = "strip too wide for the packed track entry"; return false; }
  const int threads = (pl.R * pl.wpp / pl.ppw + 1) * 32;
  const int regs_est = (mode == 2 ? 3 : 2) * pl.J + 30;
  int ctas = std::min(4, std::min(2048 / threads, 65536 / (threads * regs_est)));
  ctas = std::max(ctas, 1);
  const size_t row_bytes = (size_t)pl.pitch * 4;
  // per-warp state: point parameters, entry table (+ weight table); packed mode: the 16-bit counter levels
  const int n_cw = pl.R * pl.wpp;   // (two points per warp: R / 2 warps with two point records and two entry tables each)
  const size_t state_bytes = mode == 1 ? ft_tile_state_bytes<GatherHit8>(pl.J, n_cw)
                           : mode == 3 ? ft_tile_state_bytes<GatherF32W>(pl.J, n_cw)
                                       : ft_tile_state_bytes<GatherF32>(pl.J, n_cw);
  int64_t rows_fit = 0;
  for (;; --ctas) {  // fewer CTAs per SM until the ring holds two stages
    const size_t budget = (size_t)(228 * 1024) / ctas - 2048;
    rows_fit = budget > state_bytes + 1024 ? (int64_t)((budget - 1024 - state_bytes) / row_bytes) : 0;
    if (rows_fit >= 2 * kRPS || ctas == 1) break;
  }
  if (rows_fit < 2 * kRPS) { *why = "strip does not fit shared memory twice"; return false; }
  rows_fit = std::min<int64_t>(rows_fit, 32);
  pl.rows_per_stage = kRPS;
  pl.n_stages = (int32_t)(rows_fit / kRPS);
  pl.ctas_per_sm = ctas;
  pl.smem_bytes = (size_t)pl.n_stages * pl.rows_per_stage * row_bytes + 2 * 8 * (size_t)pl.n_stages + state_bytes;
  return true;
}

// Outer points of the threshold sample: one wave of CTA groups (one per SM), more only when the bank is so large
// that the fused pass would append more than cap / 8 entries per band (appended ~ k * groups / sample groups).
uint64_t ft_tile_sample_points(const FtTilePlan& plan, uint64_t n_points, uint32_t k, uint32_t cap) {
  const uint64_t R = (uint64_t)plan.R;
  const uint64_t n_groups = (n_points + R - 1) / R;
  uint64_t n_sg = std::max<uint64_t>((uint64_t)ft_sm_count(), (8ull * k * n_groups + cap - 1) / std::max<uint32_t>(cap, 1u));
  n_sg = std::min(n_sg, n_groups);
  return std::min(n_sg * R, n_points);
}

// Split tail: a launch of n_groups CTA groups (n_skip of them exit at once) runs (n_groups - n_skip) / n_SM waves; the
// last, partial wave would leave SMs idle for up to a whole CTA time.  Its groups are split in S parts of R / S points
// each (S the largest divisor of R with rem * n_tiles * S <= n_SM), run by CTAs with that many fewer consumer warps.
// Plans with one CTA per SM only.  Sets a->main_groups / main_ctas / tail_split and returns the grid size.
static uint64_t ft_split_tail(const FtTilePlan& plan, uint64_t n_groups, const uint32_t* skip_sorted, uint32_t n_skip,
                              FtTileArgs* a) {
  a->tail_split = 1; a->main_groups = 0; a->main_ctas = 0;
  const uint64_t nt = (uint64_t)plan.n_tiles;
  const uint64_t grid1 = n_groups * nt;
  const uint64_t kSMs = (uint64_t)ft_sm_count();
  if (plan.mode == 1 || plan.ctas_per_sm != 1 || n_skip > n_groups) return grid1;   // (mode 1: see ft_tile_body)
  const uint64_t eff = n_groups - n_skip;                 // groups that run (n_tiles CTAs each)
  const uint64_t W = eff * nt / kSMs;                     // full waves
  if (W == 0) return grid1;
  const uint64_t main_eff = W * kSMs / nt;                // running groups of the full waves
  const uint64_t rem = eff - main_eff;
  if (rem == 0) return grid1;
  auto nonskipped = [&](uint64_t G) {   // groups of [0, G) that run
    const uint32_t* e = std::lower_bound(skip_sorted, skip_sorted + n_skip, (uint32_t)std::min<uint64_t>(G, 0xffffffffu));
    return G - (uint64_t)(e - skip_sorted);
  };
  uint64_t lo = 0, hi = n_groups;      // smallest G with nonskipped(G) == main_eff
  while (lo < hi) {
    const uint64_t mid = (lo + hi) / 2;
    if (nonskipped(mid) >= main_eff) hi = mid; else lo = mid + 1;
  }
  const uint64_t G_main = lo;
  const int unit = plan.ppw == 2 ? 2 : 1;
  int S = 1;
  for (int s = 2; s <= plan.R; ++s)
    if (plan.R % s == 0 && (plan.R / s) % unit == 0 && rem * nt * (uint64_t)s <= kSMs) S = s;
  if (S == 1 || G_main * nt > 0x7fffffffull) return grid1;
  a->main_groups = (uint32_t)G_main; a->main_ctas = (uint32_t)(G_main * nt); a->tail_split = (uint32_t)S;
  return (G_main + (n_groups - G_main) * (uint64_t)S) * nt;
}

cudaError_t ft_launch_tile(const FtDev& d, const FtTilePlan& plan, const FtTileRun& run, uint64_t pt_begin,
                           uint64_t pt_end, cudaStream_t s, int* launches, const uint32_t* glist, uint32_t n_glist,
                           const uint32_t* gskip) {
  *launches = 0;
  if (pt_end <= pt_begin) return cudaSuccess;
  FtTileArgs a{};
  a.A = run.A; a.kst = plan.kst; a.err = plan.err;
  a.tile_w = plan.tile_w; a.n_tiles = plan.n_tiles; a.R = plan.R; a.wpp = plan.wpp;
  a.pitch = plan.pitch; a.copy_floats = plan.copy_floats;
  a.n_stages = plan.n_stages; a.add_back = run.add_back; a.c_row = run.c_row;
  a.out_f = run.out_f; a.out_i = run.out_i; a.out_base = run.out_base;
  if (run.sel) { a.sel = *run.sel; a.has_sel = 1; }
  a.bpb = run.bpb > 0 ? run.bpb : 1;
  a.pbox = run.pbox; a.n_bands = run.n_bands;
  a.zmode = run.zmode; a.out_key = run.out_key; a.z_mu = run.z_mu; a.z_inv_sigma = run.z_inv_sigma;
  a.out_sigma = run.out_sigma;
  a.sky_norm = run.sky_norm; a.norm_cb = run.norm_cb;
  a.near_ties = run.near_ties;
  a.glist = glist; a.gskip = gskip;
  const unsigned block = (unsigned)((plan.R * plan.wpp / plan.ppw + 1) * 32);
  const uint64_t max_groups = 0x7fffffffull / (uint64_t)plan.n_tiles;
  auto launch = [&](unsigned grid) {
    return plan.mode == 1 ? ft_tile8_launch(plan.J, d, a, grid, block, plan.smem_bytes, s)
         : plan.mode == 2 ? ft_tileb_launch(plan.J, d, a, grid, block, plan.smem_bytes, s)
         : plan.mode == 3 ? ft_tilew_launch(plan.J, d, a, grid, block, plan.smem_bytes, s)
         : plan.ppw == 2  ? ft_tile2_launch(plan.J / 2, d, a, grid, block, plan.smem_bytes, s)
                          : ft_tile_launch(plan.J, d, a, grid, block, plan.smem_bytes, s);
  };
  if (glist || gskip) {  // the threshold sample, or the rest of the bank: one launch over [pt_begin = 0, pt_end)
    const uint64_t all_groups = (pt_end - pt_begin + plan.R - 1) / plan.R;
    const uint64_t n_launch = glist ? (uint64_t)n_glist : all_groups;
    if (pt_begin != 0 || n_launch > max_groups) return cudaErrorInvalidValue;
    if (n_launch == 0) return cudaSuccess;
    a.pt_begin = 0; a.pt_end = pt_end;
    uint64_t grid = n_launch * (uint64_t)plan.n_tiles;
    if (gskip && (run.skip_host || run.n_skip_host == 0)) grid = ft_split_tail(plan, all_groups, run.skip_host, run.n_skip_host, &a);
    if (grid > 0x7fffffffull) return cudaErrorInvalidValue;
    const cudaError_t e = launch((unsigned)grid);
    if (e == cudaSuccess) *launches = 1;
    return e;
  }
  uint64_t pt = pt_begin;
  while (pt < pt_end) {
    uint64_t groups = (pt_end - pt + plan.R - 1) / plan.R;
    if (groups > max_groups) groups = max_groups;
    a.pt_begin = pt;
    a.pt_end = std::min<uint64_t>(pt_end, pt + groups * plan.R);
    uint64_t grid = groups * (uint64_t)plan.n_tiles;
    if (pt + groups * plan.R >= pt_end) grid = ft_split_tail(plan, groups, nullptr, 0, &a);   // the last chunk of the range
    if (grid > 0x7fffffffull) { a.tail_split = 1; grid = groups * (uint64_t)plan.n_tiles; }
    const cudaError_t e = launch((unsigned)grid);
    if (e != cudaSuccess) return e;
    *launches += 1;
    pt = a.pt_end;
  }
  return cudaSuccess;
}

cudaError_t ft_launch_hitmap(const float* P, float rho, float* H, int64_t n, cudaStream_t s) {
  ft_hitmap_kernel<<<ft_sm_count() * 8, 256, 0, s>>>(P, rho, H, n);
  return cudaGetLastError();
}

cudaError_t ft_launch_fold_centered(const float* P, const float* w_sft, const float* w_bin, float* Q, float* c_row,
                                    double* w_row, int64_t n_sft, int64_t n_bins, int64_t ld, int hits, float rho,
                                    cudaStream_t s) {
  ft_fold_centered_kernel<<<(unsigned)n_sft, 256, 0, s>>>(P, w_sft, w_bin, Q, c_row, w_row, n_bins, ld, hits, rho);
  return cudaGetLastError();
}
