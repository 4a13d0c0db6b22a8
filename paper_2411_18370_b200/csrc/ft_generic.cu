// Generic kernel K0 and the fp64 refinement kernels: the canonical track arithmetic evaluated per
// (template, SFT), gather through L1/L2, fp64 accumulation in ascending SFT order (so the result
// is the plain definition, Eq. (3) PAPER.md:64 / Eq. (7) :95, to the last bit).  K0 is the path for
// grids the tile kernel does not take (df0 != df) and the reference the tile kernel is tested
// against on the device; the refinement kernels re-evaluate the survivors of the fp32 selection
// (and give Eq. (36)'s z with the candidate's own weights, Eq. 4-5 when they depend on the sky).
#include "ft_common.cuh"

namespace {

constexpr int K0_THREADS = 256;

// CTA = one outer point x 256 consecutive f0.  Per chunk of 256 SFTs the CTA computes the
// Doppler/binary factor D_alpha and f1*dt once (they do not depend on f0), then every thread walks
// the chunk for its own f0 with the canonical x -> k -> gather.
template <int STAT>
__global__ void __launch_bounds__(K0_THREADS)
ft_generic_kernel(const __grid_constant__ FtDev d, uint64_t pt_begin, uint32_t n_fblk,
                  float* __restrict__ out_power, int32_t* __restrict__ out_count, uint64_t out_base) {
  __shared__ double sD[K0_THREADS];
  __shared__ double sF1dt[K0_THREADS];
  __shared__ float sW[K0_THREADS];
  const uint64_t pt = pt_begin + blockIdx.x / n_fblk;
  const int64_t i_f0 = (int64_t)(blockIdx.x % n_fblk) * K0_THREADS + threadIdx.x;
  const FtPoint p = ft_decode_point(d, pt);
  const bool active = i_f0 < d.n_f0;
  const double f0 = ft_f0(d, active ? i_f0 : 0);
  double power = 0.0;
  int32_t count = 0;
  for (int64_t a0 = 0; a0 < d.n_sft; a0 += K0_THREADS) {
    const int64_t a = a0 + threadIdx.x;
    __syncthreads();
    if (a < d.n_sft) {
      const double t = d.t_mid[a];
      sD[threadIdx.x] = ft_doppler(d, p, a, t);
      sF1dt[threadIdx.x] = __dmul_rn(p.f1, __dsub_rn(t, d.t_ref));
      sW[threadIdx.x] = (d.wkind == 1) ? d.w[a] : 0.f;
    }
    __syncthreads();
    const int n = (int)min((int64_t)K0_THREADS, d.n_sft - a0);
    if (active) {
#pragma unroll 4
      for (int c = 0; c < n; ++c) {
        const double x = ft_track_x(f0, sF1dt[c], sD[c], d.f_min, d.inv_df);
        const int64_t k = __double2ll_rn(x);
        const int64_t off = (a0 + c) * d.ld + k;
        const float pix = __ldg(d.P + off);
        if (STAT == 0 || STAT == 2) {
          const float w = (d.wkind == 1) ? sW[c] : __ldg(d.w + off);
          power = fma((double)w, (double)pix, power);  // product exact in fp64 -> same as mul, add
        }
        if (STAT == 3 && pix > d.rho) power += (double)((d.wkind == 1) ? sW[c] : __ldg(d.w + off));  // weighted count (:97)
        if (STAT != 0) count += (pix > d.rho) ? 1 : 0;
      }
    }
  }
  if (active) {
    const uint64_t o = pt * (uint64_t)d.n_f0 + (uint64_t)i_f0 - out_base;
    if (STAT != 1 && out_power) out_power[o] = (float)power;
    if (STAT != 0 && out_count) out_count[o] = count;
  }
}

// One warp per candidate.  Lanes take 32 consecutive SFTs, then the 32 exact products are added
// in ascending SFT order (every lane redundantly), so the sum has the oracle's rounding sequence.
// With sky-dependent weights (Eq. 4-5) the weight of SFT a is u_a r_a / sum_b u_b r_b, u = a^2 + b^2 in fp64.
// Also the standardised statistic z = (power - mu_G) / sigma_G of the candidate's weights (Eq. 36).
__device__ __forceinline__ void ft_refine_one(const FtDev& d, const FtPoint& p, double f0, double t_ref, int lane,
                                              FtCandDev* c, unsigned* ties_out, int64_t* k_out, int32_t* bad_out) {
  double power = 0.0, wcount = 0.0, wsum = 0.0, wsq = 0.0;
  int32_t count = 0;
  unsigned ties = 0;
  bool bad = false;
  FtSkyPoint sk;
  if (d.skyw) sk = ft_sky_point(p.nx, p.ny, p.nz);
  for (int64_t a0 = 0; a0 < d.n_sft; a0 += 32) {
    const int64_t a = a0 + lane;
    double prod = 0.0, wc = 0.0, wa = 0.0;
    bool hit = false, tie = false;
    if (a < d.n_sft) {
      const double t = d.t_mid[a];
      const double D = ft_doppler(d, p, a, t);
      const double x = ft_track_x(f0, __dmul_rn(p.f1, __dsub_rn(t, t_ref)), D, d.f_min, d.inv_df);
      tie = ft_near_tie(x);
      const int64_t k = __double2ll_rn(x);
      if (k_out) k_out[a] = k;
      if (k < 0 || k >= d.n_bins || !(x == x)) {
        bad = true;
      } else {
        const int64_t off = a * d.ld + k;
        const float pix = __ldg(d.P + off);
        const float wf = (d.wkind == 1) ? __ldg(d.w + a) : __ldg(d.w + off);
        wa = (double)wf;
        if (d.skyw) wa = __dmul_rn(ft_antenna_u(d.ant + 9 * a, sk), wa);
        prod = __dmul_rn(wa, (double)pix);
        hit = pix > d.rho;
        wc = hit ? wa : 0.0;
      }
    }
    count += __popc(__ballot_sync(0xffffffffu, hit));
    ties += __popc(__ballot_sync(0xffffffffu, tie));
#pragma unroll
    for (int l = 0; l < 32; ++l) {
      power = __dadd_rn(power, __shfl_sync(0xffffffffu, prod, l));
      wcount = __dadd_rn(wcount, __shfl_sync(0xffffffffu, wc, l));
      if (d.skyw) {
        const double wl = __shfl_sync(0xffffffffu, wa, l);
        wsum = __dadd_rn(wsum, wl);
        wsq = __dadd_rn(wsq, __dmul_rn(wl, wl));
      }
    }
  }
  bad = __any_sync(0xffffffffu, bad);
  double mu = d.mu_G, sigma = d.sigma_G;
  if (d.skyw) {  // Eq. (5): normalise; then mu_G = 1, sigma_G = sqrt(sum w^2)
    power = power / wsum; wcount = wcount / wsum;
    mu = 1.0; sigma = sqrt(wsq) / wsum;
  }
  c->power = power; c->wcount = wcount; c->count = count; c->band = -1;
  c->sigma = sigma; c->z = (power - mu) / sigma;
  *ties_out = ties;
  *bad_out = bad ? 1 : 0;
}

__global__ void __launch_bounds__(128)
ft_refine_kernel(const __grid_constant__ FtDev d, const uint64_t* __restrict__ idx_list,
                 const uint32_t* __restrict__ n_dev, int64_t n_max, FtCandDev* __restrict__ out,
                 unsigned long long* __restrict__ near_ties) {
  const int64_t n = n_dev ? min((int64_t)*n_dev, n_max) : n_max;
  const int lane = threadIdx.x & 31;
  const int64_t cand = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (cand >= n) return;
  const uint64_t idx = idx_list[cand];
  const uint64_t pt = idx / (uint64_t)d.n_f0;
  const int64_t i_f0 = (int64_t)(idx % (uint64_t)d.n_f0);
  const FtPoint p = ft_decode_point(d, pt);
  FtCandDev c;
  unsigned ties; int32_t bad;
  ft_refine_one(d, p, ft_f0(d, i_f0), d.t_ref, lane, &c, &ties, nullptr, &bad);
  c.idx = idx;
  if (lane == 0) {
    out[cand] = c;
    if (ties && near_ties) atomicAdd(near_ties, (unsigned long long)ties);
  }
}

// Long candidate lists (the survivors of a number-count veto, ft_topk.cu): ONE THREAD per candidate walks the SFTs
// in ascending order, so the sums have the oracle's rounding sequence without the 32-fold redundancy of the
// warp-per-candidate form (which is the faster one for the few hundred candidates of a plain top-k).
#ifndef FT_RT_MINB
#define FT_RT_MINB 8     // CTAs of 128 threads per SM the register budget is held to (8 -> 64 registers)
#endif
#ifndef FT_RT_UNROLL
#define FT_RT_UNROLL 8
#endif
#define FT_STR2(x) #x
#define FT_STR(x) FT_STR2(x)
// SKY: sky-dependent weights (their nine sky factors stay out of the register budget of the fixed-weight variant).
template <bool SKY>
__global__ void __launch_bounds__(128, SKY ? 4 : FT_RT_MINB)
ft_refine_thread_kernel(const __grid_constant__ FtDev d, const uint64_t* __restrict__ idx_list, int64_t n,
                        FtCandDev* __restrict__ out, unsigned long long* __restrict__ near_ties) {
  const int64_t cand = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (cand >= n) return;
  const uint64_t idx = idx_list[cand];
  const uint64_t pt = idx / (uint64_t)d.n_f0;
  const FtPoint p = ft_decode_point(d, pt);
  const double f0 = ft_f0(d, (int64_t)(idx % (uint64_t)d.n_f0));
  double power = 0.0, wcount = 0.0, wsum = 0.0, wsq = 0.0;
  int32_t count = 0;
  unsigned ties = 0;
  FtSkyPoint sk;
  if (SKY) sk = ft_sky_point(p.nx, p.ny, p.nz);
  // branch-free body (an out-of-range bin -- impossible for a validated grid -- contributes an exact zero), unrolled
  // so that the gathers of several SFTs are in flight; the sums are still added in ascending SFT order.
  // Round 3 (ncu: profiles/r03_refine_thread_ncu.md): the kernel was latency-bound at 94 registers = 5 CTAs per SM
  // (long-scoreboard stalls 65 % of the issue slots, 2.6 waves); the sky factors moved into a template variant
  // (64 registers, 8 CTAs per SM): 6.7 -> 4.4 ms for the 246 000 survivors of config 2 (step 95.8 -> 93.5 ms).  Staging
  // the per-SFT tables per 128-SFT chunk in shared memory measured the same at 64 registers (it spills) and 1 ms
  // slower at 80; unroll 4 and 8 measure the same.
  _Pragma(FT_STR(unroll FT_RT_UNROLL))
  for (int64_t a = 0; a < d.n_sft; ++a) {
    const double t = d.t_mid[a];
    const double D = ft_doppler_rcp(d, p, a, t);
    const double x = ft_track_x(f0, __dmul_rn(p.f1, __dsub_rn(t, d.t_ref)), D, d.f_min, d.inv_df);
    ties += ft_near_tie(x) ? 1u : 0u;
    const int64_t k = __double2ll_rn(x);
    const bool ok = k >= 0 && k < d.n_bins && x == x;
    const int64_t off = a * d.ld + (ok ? k : 0);
    const float pix = ok ? __ldg(d.P + off) : 0.f;
    double wa = (double)((d.wkind == 1) ? __ldg(d.w + a) : __ldg(d.w + off));
    if (SKY) {
      wa = __dmul_rn(ft_antenna_u(d.ant + 9 * a, sk), wa);
      wsum = __dadd_rn(wsum, wa);
      wsq = __dadd_rn(wsq, __dmul_rn(wa, wa));
    }
    power = __dadd_rn(power, __dmul_rn(wa, (double)pix));
    const bool hit = pix > d.rho;
    wcount = __dadd_rn(wcount, hit ? wa : 0.0);
    count += hit ? 1 : 0;
  }
  double mu = d.mu_G, sigma = d.sigma_G;
  if (SKY) { power = power / wsum; wcount = wcount / wsum; mu = 1.0; sigma = sqrt(wsq) / wsum; }
  FtCandDev c;
  c.power = power; c.wcount = wcount; c.idx = idx; c.count = count; c.band = -1;   // (bad cannot happen: the grid was validated at bind)
  c.sigma = sigma; c.z = (power - mu) / sigma;
  out[cand] = c;
  if (ties && near_ties) atomicAdd(near_ties, (unsigned long long)ties);
}

// The same for ONE explicit template (a record of 8 doubles), optionally with its bins: ft_track, ft_eval_bank.
__global__ void __launch_bounds__(32)
ft_refine_template_kernel(const __grid_constant__ FtDev d, const double* __restrict__ tp, double t_ref,
                          FtCandDev* __restrict__ out, int64_t* __restrict__ k_out, int32_t* __restrict__ err) {
  FtPoint p;
  p.nx = tp[2]; p.ny = tp[3]; p.nz = tp[4];
  p.Om = __ddiv_rn(FT_TWO_PI, tp[6]);
  p.apOm = __dmul_rn(tp[5], p.Om);
  p.t_asc = tp[7];
  p.f1 = tp[1];
  p.crow = nullptr;
  p.binary = tp[5] != 0.0;
  FtCandDev c;
  unsigned ties; int32_t bad;
  ft_refine_one(d, p, tp[0], t_ref, threadIdx.x & 31, &c, &ties, k_out, &bad);
  c.idx = 0;
  if (threadIdx.x == 0) {
    if (out) *out = c;
    if (bad) atomicExch(err, 1);
  }
}

// A1 hoisted to bind time for binary grids: the orbital cosine depends on (P_orb, t_asc, SFT) only,
// so the 64 a_p values of config 3 share it (Eq. 2; separability noted at :600).
__global__ void ft_ctab_kernel(const __grid_constant__ FtDev d, double* __restrict__ ctab) {
  const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t row = blockIdx.y;  // i_porb * n_tasc + i_tasc
  if (a >= d.n_sft) return;
  const double P_orb = d.P_orb[row / (uint32_t)d.n_tasc];
  const double Om = __ddiv_rn(FT_TWO_PI, P_orb);
  const double t_asc = __dadd_rn(d.t_ref, __dmul_rn(d.tasc[row % (uint32_t)d.n_tasc], P_orb));
  ctab[(size_t)row * (size_t)d.n_sft + a] = cos(__dmul_rn(Om, __dsub_rn(d.t_mid[a], t_asc)));
}

}  // namespace

cudaError_t ft_launch_ctab(const FtDev& d, double* ctab, cudaStream_t s) {
  const dim3 grid((unsigned)((d.n_sft + 255) / 256), (unsigned)(d.n_porb * d.n_tasc));
  ft_ctab_kernel<<<grid, 256, 0, s>>>(d, ctab);
  return cudaGetLastError();
}

cudaError_t ft_launch_generic(const FtDev& d, int stat, uint64_t pt_begin, uint64_t pt_end,
                              float* out_power, int32_t* out_count, uint64_t out_base_idx,
                              cudaStream_t s) {
  const uint32_t n_fblk = (uint32_t)((d.n_f0 + K0_THREADS - 1) / K0_THREADS);
  uint64_t pt = pt_begin;
  while (pt < pt_end) {  // grid.x is limited to 2^31-1 blocks
    const uint64_t n_pt = (pt_end - pt < (uint64_t)(0x7fffffffu / n_fblk)) ? pt_end - pt : (uint64_t)(0x7fffffffu / n_fblk);
    const dim3 grid((unsigned)(n_pt * n_fblk));
    if (stat == 0) ft_generic_kernel<0><<<grid, K0_THREADS, 0, s>>>(d, pt, n_fblk, out_power, out_count, out_base_idx);
    else if (stat == 1) ft_generic_kernel<1><<<grid, K0_THREADS, 0, s>>>(d, pt, n_fblk, out_power, out_count, out_base_idx);
    else if (stat == 3) ft_generic_kernel<3><<<grid, K0_THREADS, 0, s>>>(d, pt, n_fblk, out_power, out_count, out_base_idx);
    else ft_generic_kernel<2><<<grid, K0_THREADS, 0, s>>>(d, pt, n_fblk, out_power, out_count, out_base_idx);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    pt += n_pt;
  }
  return cudaSuccess;
}

cudaError_t ft_launch_refine(const FtDev& d, const uint64_t* idx_dev, const uint32_t* n_dev, int64_t n_max,
                             FtCandDev* out, unsigned long long* near_ties, cudaStream_t s) {
  if (n_max <= 0) return cudaSuccess;
  if (!n_dev && n_max >= 8192) {   // a long list of known length: one thread per candidate
    if (d.skyw) ft_refine_thread_kernel<true><<<(unsigned)((n_max + 127) / 128), 128, 0, s>>>(d, idx_dev, n_max, out, near_ties);
    else ft_refine_thread_kernel<false><<<(unsigned)((n_max + 127) / 128), 128, 0, s>>>(d, idx_dev, n_max, out, near_ties);
    return cudaGetLastError();
  }
  const int64_t warps_per_block = 4;
  const unsigned grid = (unsigned)((n_max + warps_per_block - 1) / warps_per_block);
  ft_refine_kernel<<<grid, 128, 0, s>>>(d, idx_dev, n_dev, n_max, out, near_ties);
  return cudaGetLastError();
}


cudaError_t ft_launch_refine_template(const FtDev& d, const double* template_dev, double t_ref, FtCandDev* out,
                                      int64_t* k_out, int32_t* err, cudaStream_t s) {
  ft_refine_template_kernel<<<1, 32, 0, s>>>(d, template_dev, t_ref, out, k_out, err);
  return cudaGetLastError();
}
