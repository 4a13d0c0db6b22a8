// Generic kernel K0 and the fp64 refinement kernel: the canonical track arithmetic evaluated per
// (template, SFT), gather through L1/L2, fp64 accumulation in ascending SFT order (so the result
// is the plain definition, Eq. (3) PAPER.md:64 / Eq. (7) :95, to the last bit).  K0 is the path for
// grids the tile kernel does not take (df0 != df) and the reference the tile kernel is tested
// against on the device; the refinement kernel re-evaluates the survivors of the fp32 selection.
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
        if (STAT != 1) {
          const float w = (d.wkind == 1) ? sW[c] : __ldg(d.w + off);
          power = fma((double)w, (double)pix, power);  // product exact in fp64 -> same as mul, add
        }
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
  const double f0 = ft_f0(d, i_f0);
  double power = 0.0, wcount = 0.0;
  int32_t count = 0;
  unsigned ties = 0;
  for (int64_t a0 = 0; a0 < d.n_sft; a0 += 32) {
    const int64_t a = a0 + lane;
    double prod = 0.0, wc = 0.0;
    bool hit = false, tie = false;
    if (a < d.n_sft) {
      const double t = d.t_mid[a];
      const double D = ft_doppler(d, p, a, t);
      const double x = ft_track_x(f0, __dmul_rn(p.f1, __dsub_rn(t, d.t_ref)), D, d.f_min, d.inv_df);
      tie = ft_near_tie(x);
      const int64_t k = __double2ll_rn(x);
      const int64_t off = a * d.ld + k;
      const float pix = __ldg(d.P + off);
      const float w = (d.wkind == 1) ? __ldg(d.w + a) : __ldg(d.w + off);
      prod = __dmul_rn((double)w, (double)pix);
      hit = pix > d.rho;
      wc = hit ? (double)w : 0.0;
    }
    count += __popc(__ballot_sync(0xffffffffu, hit));
    ties += __popc(__ballot_sync(0xffffffffu, tie));
#pragma unroll
    for (int l = 0; l < 32; ++l) {
      power = __dadd_rn(power, __shfl_sync(0xffffffffu, prod, l));
      wcount = __dadd_rn(wcount, __shfl_sync(0xffffffffu, wc, l));
    }
  }
  if (lane == 0) {
    FtCandDev c;
    c.power = power; c.wcount = wcount; c.idx = idx; c.count = count; c.band = -1;
    out[cand] = c;
    if (ties && near_ties) atomicAdd(near_ties, (unsigned long long)ties);
  }
}

// K1: an explicit list of templates (an unstructured bank: "no assumption on the properties of
// lambda"; random banks :312-316).  One thread per template, the canonical fp64 track
// per (template, SFT), gather through L1/L2, fp64 accumulation in ascending SFT order.  Nothing can
// be hoisted or staged (every template has its own sky position and orbit), so this kernel is bound
// by the fp64 pipe; it is the paper's own formulation of the problem.  A track leaving the
// spectrogram raises *err (reading R9: an error, not a clamp) and the template's outputs are NaN / -1.
struct FtTemplateDev { double f0, f1, nx, ny, nz, a_p, P_orb, t_asc; };

template <int STAT>
__global__ void __launch_bounds__(K0_THREADS)
ft_list_kernel(const __grid_constant__ FtDev d, const FtTemplateDev* __restrict__ tl, int64_t n, double t_ref,
               float* __restrict__ out_power, int32_t* __restrict__ out_count, int32_t* __restrict__ err,
               unsigned long long* __restrict__ near_ties) {
  __shared__ double sT[K0_THREADS], sVx[K0_THREADS], sVy[K0_THREADS], sVz[K0_THREADS];
  __shared__ float sW[K0_THREADS];
  const int64_t q = (int64_t)blockIdx.x * K0_THREADS + threadIdx.x;
  const bool active = q < n;
  FtTemplateDev tp = tl[active ? q : 0];
  const double Om = __ddiv_rn(FT_TWO_PI, tp.P_orb);
  const double apOm = __dmul_rn(tp.a_p, Om);
  const bool binary = tp.a_p != 0.0;
  const double kInvC = 1.0 / FT_C_LIGHT;
  const int n_bins = (int)min(d.n_bins, (int64_t)0x7fffffff);
  double power = 0.0;
  int32_t count = 0;
  unsigned ties = 0;
  bool bad = false;
  for (int64_t a0 = 0; a0 < d.n_sft; a0 += K0_THREADS) {
    const int64_t a = a0 + threadIdx.x;
    __syncthreads();
    if (a < d.n_sft) {
      sT[threadIdx.x] = d.t_mid[a];
      sVx[threadIdx.x] = d.vel[3 * a]; sVy[threadIdx.x] = d.vel[3 * a + 1]; sVz[threadIdx.x] = d.vel[3 * a + 2];
      sW[threadIdx.x] = (d.wkind == 1) ? d.w[a] : 0.f;
    }
    __syncthreads();
    const int m = (int)min((int64_t)K0_THREADS, d.n_sft - a0);
    if (active) {
#pragma unroll 2
      for (int c = 0; c < m; ++c) {
        const double t = sT[c];
        // V = dot / c as a Newton-corrected reciprocal multiply (3 fp64 instructions instead of a
        // ~25-instruction division).  It can differ from the IEEE quotient in the last bit at most,
        // which moves x by < 1e-10 bin: inside the 1e-9 near-tie window the comparison excludes.
        const double dot = __dadd_rn(__dadd_rn(__dmul_rn(sVx[c], tp.nx), __dmul_rn(sVy[c], tp.ny)), __dmul_rn(sVz[c], tp.nz));
        const double q0 = __dmul_rn(dot, kInvC);
        const double V = __fma_rn(__fma_rn(-q0, FT_C_LIGHT, dot), kInvC, q0);
        double B = 0.0;
        if (binary) B = __dmul_rn(apOm, cos(__dmul_rn(Om, __dsub_rn(t, tp.t_asc))));
        const double D = __dsub_rn(__dadd_rn(1.0, V), B);
        const double x = ft_track_x(tp.f0, __dmul_rn(tp.f1, __dsub_rn(t, t_ref)), D, d.f_min, d.inv_df);
        const int k = __double2int_rn(x);                       // saturates out of range, 0 for NaN
        ties += (fabs(x - (double)k) > 0.5 - 1e-9) ? 1u : 0u;   // within 1e-9 bin of a rounding tie
        if ((unsigned)k >= (unsigned)n_bins || !(x == x)) { bad = true; continue; }
        const int64_t off = (a0 + c) * d.ld + k;
        const float pix = __ldg(d.P + off);
        if (STAT != 1) {
          const float w = (d.wkind == 1) ? sW[c] : __ldg(d.w + off);
          power = fma((double)w, (double)pix, power);  // exact product: same as mul then add
        }
        if (STAT != 0) count += (pix > d.rho) ? 1 : 0;
      }
    }
  }
  if (!active) return;
  if (bad) atomicExch(err, 1);
  if (STAT != 1 && out_power) out_power[q] = bad ? __int_as_float(0x7fc00000) : (float)power;
  if (STAT != 0 && out_count) out_count[q] = bad ? -1 : count;
  if (ties && near_ties) atomicAdd(near_ties, (unsigned long long)ties);
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
  const int64_t warps_per_block = 4;
  const unsigned grid = (unsigned)((n_max + warps_per_block - 1) / warps_per_block);
  ft_refine_kernel<<<grid, 128, 0, s>>>(d, idx_dev, n_dev, n_max, out, near_ties);
  return cudaGetLastError();
}


cudaError_t ft_launch_list(const FtDev& d, int stat, const void* templates_dev, int64_t n, double t_ref,
                           float* out_power, int32_t* out_count, int32_t* err, unsigned long long* near_ties,
                           cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  const FtTemplateDev* tl = static_cast<const FtTemplateDev*>(templates_dev);
  const unsigned grid = (unsigned)((n + K0_THREADS - 1) / K0_THREADS);
  if (stat == 0) ft_list_kernel<0><<<grid, K0_THREADS, 0, s>>>(d, tl, n, t_ref, out_power, out_count, err, near_ties);
  else if (stat == 1) ft_list_kernel<1><<<grid, K0_THREADS, 0, s>>>(d, tl, n, t_ref, out_power, out_count, err, near_ties);
  else ft_list_kernel<2><<<grid, K0_THREADS, 0, s>>>(d, tl, n, t_ref, out_power, out_count, err, near_ties);
  return cudaGetLastError();
}
