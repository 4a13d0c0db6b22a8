// Kernel K1 and the unstructured-bank calls of the C ABI: ft_eval_templates, ft_bank_draw, ft_eval_bank,
// ft_track, ft_selftest.
//
// K1: an explicit list of templates (an unstructured bank: "no assumption on the properties of lambda",
// PAPER.md:213; random banks :312-316), or templates drawn on the fly uniformly in the xi coordinates of
// Eq. (A11) (:602-614).  One thread per template, the canonical fp64 track per (template, SFT), gather through
// L1/L2, fp64 accumulation in ascending SFT order.  Nothing can be hoisted or staged across templates (every
// template has its own sky position and orbit), so the kernel is bound by the fp64 pipe; what CAN be saved is
// kept off that pipe: the per-SFT tables (t - t_ref, v, w as doubles) are staged in shared memory once per
// CTA, the rounding to a bin is a magic-number add (two DADD, no F2I/I2F), the fp32 -> fp64 conversions of
// pixel and weight are integer bit moves, and the division by c is a reciprocal multiply with one fused
// correction (bit-identical to the IEEE quotient: ft_selftest 0).  A track leaving the spectrogram raises
// *err (reading R9: an error, not a clamp) and the template's outputs are NaN / -1.
#include <algorithm>
#include <cstdarg>
#include <mutex>

#include "ft_ctx.cuh"

// Work space of ft_eval_templates_noalloc (end of this file): K1's scratch for callers that may not allocate.
// Layout: uint32 perm[n] | uint32 hist[4096] (n <= FT_NOALLOC_MAX_TEMPLATES, so both fit in the first
// (MAX + 4096) words) | at byte (MAX + 4096) * 4: int32 out-of-range flag, at + 8: uint64 near-tie counter.
// In host code this name is only a stand-in for the symbol, NOT a device address: the address a kernel may be
// given comes from cudaGetSymbolAddress (ft_noalloc_scratch_ptr below), looked up once per device.
static __device__ __align__(256) unsigned char ft_noalloc_scratch[((size_t)FT_NOALLOC_MAX_TEMPLATES + 4096) * 4 + 256];

namespace {

constexpr int K1_THREADS = 256;
constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: x + kMagic rounds x to the nearest integer, ties to even

struct FtTemplateDev { double f0, f1, nx, ny, nz, a_p, P_orb, t_asc; };
struct FtBankBox { double f0_lo, f0_hi, f1_lo, f1_hi, ra_lo, ra_hi, sd_lo, sd_hi, ap_lo, ap_hi, porb_lo, porb_hi, t_ref; };

// (double)x for a finite normal or zero fp32 by integer moves (sign | exponent + 896 | mantissa << 29); the
// conversion instruction shares the fp64 pipe, these do not.  Subnormals, inf and NaN take the instruction.
__device__ __forceinline__ double ft_f2d(float x) {
  const uint32_t b = __float_as_uint(x);
  const uint32_t e = (b >> 23) & 0xffu;
  if (e - 1u < 254u) return __hiloint2double((int)((b & 0x80000000u) | ((e + 896u) << 20) | ((b >> 3) & 0xfffffu)), (int)(b << 29));
  if ((b << 1) == 0u) return __hiloint2double((int)(b & 0x80000000u), 0);
  return (double)x;
}

// cos(x) for the orbital phase of K1: k = rint(x / pi) by a magic-number fused multiply-add (no F2I / I2F), r = x - k pi
// with pi split in three doubles (each product exact in the fused multiply-add), cos(r) on [-pi/2, pi/2] by its Taylor
// series to r^24 (truncation < 1e-19; twelve fused multiply-adds), sign from the parity of k.  No table, no branch:
// 18 fp64 instructions against ~25 plus two conversions and three table loads of the library routine.  Absolute
// error < 3e-16 for |x| < 1e8 (checked against 300-bit arithmetic when the constants were derived; on the device
// against cos() in tests/test_gpu_templates.py), i.e. < 1e-14 bin on the track: far inside the 1e-9 tie window.
// (the constants live in the constant bank: a DFMA takes c[bank][offset] as an operand, whereas a 64-bit literal costs two
// UMOV issue slots per use -- 26 of the ~110 instructions of a binary evaluation before this)
__constant__ double kCosC[17] = {
    0.31830988618379069,        // 1/pi
    3.1415926535897931,         // pi = 0x1.921fb54442d18p+1
    1.2246467991473532e-16,     //    + 0x1.1a62633145c07p-53
    -2.9947698097183397e-33,    //    - 0x1.f1976b7ed8fbcp-109
    1.6117375710961184e-24,     // 1/24!
    -8.8967913924505741e-22,    // -1/22!
    4.1103176233121648e-19,     // 1/20!
    -1.5619206968586225e-16,    // -1/18!
    4.7794773323873853e-14,     // 1/16!
    -1.1470745597729725e-11,    // -1/14!
    2.08767569878681e-09,       // 1/12!
    -2.7557319223985888e-07,    // -1/10!
    2.4801587301587302e-05,     // 1/8!
    -0.0013888888888888889,     // -1/6!
    0.041666666666666664,       // 1/4!
    -0.5, 1.0};
__device__ __forceinline__ double k1_cos(double x) {
  const double tm = __fma_rn(x, kCosC[0], kMagic);                       // rint(x / pi) in the low mantissa bits
  const double k = __dsub_rn(tm, kMagic);
  double r = __fma_rn(-k, kCosC[1], x);
  r = __fma_rn(-k, kCosC[2], r);
  r = __fma_rn(-k, kCosC[3], r);
  const double z = __dmul_rn(r, r);
  double t = kCosC[4];
#pragma unroll
  for (int i = 5; i < 17; ++i) t = __fma_rn(t, z, kCosC[i]);
  return __hiloint2double(__double2hiint(t) ^ (__double2loint(tm) << 31), __double2loint(t));   // (-1)^k
}

// counter-based uniform in (0, 1): splitmix64 finaliser of seed + golden * (8 i + d + 1), top 53 bits
__device__ __forceinline__ double ft_uniform(uint64_t seed, uint64_t i, uint32_t dcoord) {
  uint64_t z = seed + 0x9E3779B97F4A7C15ull * (8ull * i + (uint64_t)dcoord + 1ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  z ^= z >> 31;
  return ((double)(z >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

// xi -> lambda for a coordinate with density lambda^p (Eq. 34 PAPER.md:297 inverted): p1 = p + 1
__device__ __forceinline__ double ft_inv_power(double lo, double hi, double u, int p1) {
  const double a = pow(lo, (double)p1), b = pow(hi, (double)p1);
  return pow(a + u * (b - a), 1.0 / (double)p1);
}

// Template i of a xi-uniform bank (Eq. A11): xi = (f0^6/6, alpha, sin delta, a_p^3/3, Omega^4/4, phi_b); f1 uniform.
__device__ __forceinline__ FtTemplateDev ft_bank_template(const FtBankBox& bx, uint64_t seed, uint64_t i) {
  FtTemplateDev tp;
  tp.f0 = ft_inv_power(bx.f0_lo, bx.f0_hi, ft_uniform(seed, i, 0), 6);
  const double ra = bx.ra_lo + ft_uniform(seed, i, 1) * (bx.ra_hi - bx.ra_lo);
  const double sd = bx.sd_lo + ft_uniform(seed, i, 2) * (bx.sd_hi - bx.sd_lo);
  const double cd = sqrt(1.0 - sd * sd);
  tp.nx = cd * cos(ra); tp.ny = cd * sin(ra); tp.nz = sd;
  if (bx.ap_hi > 0.0) {
    tp.a_p = ft_inv_power(bx.ap_lo, bx.ap_hi, ft_uniform(seed, i, 3), 3);
    const double Om = ft_inv_power(FT_TWO_PI / bx.porb_hi, FT_TWO_PI / bx.porb_lo, ft_uniform(seed, i, 4), 4);
    tp.P_orb = FT_TWO_PI / Om;
    tp.t_asc = bx.t_ref + (FT_TWO_PI * ft_uniform(seed, i, 5)) / Om;
  } else {
    tp.a_p = 0.0; tp.P_orb = 86400.0; tp.t_asc = bx.t_ref;
  }
  tp.f1 = bx.f1_lo + ft_uniform(seed, i, 6) * (bx.f1_hi - bx.f1_lo);
  return tp;
}

__global__ void ft_bank_draw_kernel(FtBankBox bx, uint64_t seed, uint64_t first, int64_t n, FtTemplateDev* __restrict__ out) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n) out[j] = ft_bank_template(bx, seed, first + (uint64_t)j);
}

// ---- evaluation order: templates bucketed by f0 so that the 32 gathers of a warp fall into a few cache lines --
// (a random bank read in storage order touches 30 sectors per warp-load; ordered by f0 the spread is the Doppler
// shift, a few lines: measured 1.5x on the isolated path).  Counting sort on 4096 buckets of the template's
// position in the spectrogram band; the order inside a bucket is arbitrary (results are stored per template).
constexpr int K1_BUCKETS = 4096;

template <bool GEN>
__device__ __forceinline__ uint32_t k1_bucket(const FtDev& d, const FtTemplateDev* tl, const FtBankBox& bx, uint64_t seed,
                                              uint64_t first, int64_t j) {
  const double f0 = GEN ? ft_inv_power(bx.f0_lo, bx.f0_hi, ft_uniform(seed, first + (uint64_t)j, 0), 6) : tl[j].f0;
  const double u = (f0 - d.f_min) * d.inv_df / (double)d.n_bins;
  return (uint32_t)min(max((int)(u * K1_BUCKETS), 0), K1_BUCKETS - 1);
}
template <bool GEN>
__global__ void k1_hist_kernel(const __grid_constant__ FtDev d, const FtTemplateDev* __restrict__ tl, const __grid_constant__ FtBankBox bx,
                               uint64_t seed, uint64_t first, int64_t n, uint32_t* __restrict__ hist) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n) atomicAdd(hist + k1_bucket<GEN>(d, tl, bx, seed, first, j), 1u);
}
__global__ void __launch_bounds__(1024) k1_scan_kernel(uint32_t* __restrict__ hist) {   // exclusive scan of 4096 counters, in place
  __shared__ uint32_t part[1024];
  uint32_t v[4], s = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) { v[i] = hist[4 * threadIdx.x + i]; s += v[i]; }
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const uint32_t t = (int)threadIdx.x >= o ? part[threadIdx.x - o] : 0u;
    __syncthreads();
    part[threadIdx.x] += t;
    __syncthreads();
  }
  uint32_t run = part[threadIdx.x] - s;
#pragma unroll
  for (int i = 0; i < 4; ++i) { hist[4 * threadIdx.x + i] = run; run += v[i]; }
}
template <bool GEN>
__global__ void k1_scatter_kernel(const __grid_constant__ FtDev d, const FtTemplateDev* __restrict__ tl, const __grid_constant__ FtBankBox bx,
                                  uint64_t seed, uint64_t first, int64_t n, uint32_t* __restrict__ cursor, uint32_t* __restrict__ perm) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j < n) perm[atomicAdd(cursor + k1_bucket<GEN>(d, tl, bx, seed, first, j), 1u)] = (uint32_t)j;
}

struct K1Acc { double power; int32_t count; unsigned ties; unsigned bad; double wsum; double wcount; double wsq; };

#ifndef FT_K1_INT_CVT
#define FT_K1_INT_CVT 0   // fp32 -> fp64 by the conversion instruction (0: measured faster, one issue slot) or by integer moves (1)
#endif
__device__ __forceinline__ double k1_f2d(float x) {
#if FT_K1_INT_CVT
  return ft_f2d(x);
#else
  return (double)x;
#endif
}

// The SFT loop over one staged chunk of m SFTs.  BIN: 0 no template of the CTA is a binary (no orbital cosine in the
// loop body), 2 every template is (cosine without a branch), 1 mixed (cosine under a per-thread branch).  PERSFT: per-SFT weights (staged as
// doubles) or per-bin weights (gathered like the pixel).  The loop has no branch: an out-of-range bin is clamped
// for the load and remembered in acc.bad (the template's outputs are then discarded).
// SKY: sky-dependent weights (Eq. 4-5, ft_set_antenna): the weight of SFT a is u_a(n) w_a, u = a^2 + b^2 from the
// staged antenna coefficients sAnt[9 c ..] and the template's sky factors sk; acc.wsum carries sum_a u_a w_a and the
// caller divides by it at the end (the order of ft_refine_one).  Implies per-SFT weights.
// EXT (ft_eval_bank_veto; STAT == 2): also the weighted number count sum_a w_a [P > rho] (acc.wcount) and, with SKY,
// sum_a (u_a w_a)^2 (acc.wsq) for sigma_G of Eq. (36).
template <int STAT, int BIN, bool PERSFT, bool SKY, bool EXT = false>
__device__ __forceinline__ void k1_chunk(const FtDev& d, const FtTemplateDev& tp, double Om, double apOm, bool binary,
                                         const double2* sA, const double2* sB, const double2* sC, const double* sAnt,
                                         const FtSkyPoint& sk, int m, int64_t a0, uint32_t n_bins, K1Acc& acc) {
  const float* __restrict__ prow = d.P + a0 * d.ld;
  const float* __restrict__ wrow = d.w + a0 * d.ld;
  const int64_t ld = d.ld;
  // loop constants pinned in registers (otherwise re-materialised with two moves per use and evaluation)
  double kInvC = 1.0 / FT_C_LIGHT, kC = FT_C_LIGHT, kTie = 0.5 - 1e-9, f_min = d.f_min, inv_df = d.inv_df;
  asm volatile("" : "+d"(kInvC), "+d"(kC), "+d"(kTie), "+d"(f_min), "+d"(inv_df));
#pragma unroll 4
  for (int c = 0; c < m; ++c) {
    const double2 vxy = sA[c], vzdt = sB[c];
    const double dot = __dadd_rn(__dadd_rn(__dmul_rn(vxy.x, tp.nx), __dmul_rn(vxy.y, tp.ny)), __dmul_rn(vzdt.x, tp.nz));
    // V = dot / c: q0 = dot (1/c), V = q0 + (dot - q0 c)(1/c)  (ft_div_c with the constants above)
    const double q0 = __dmul_rn(dot, kInvC);
    const double V = __fma_rn(__fma_rn(-q0, kC, dot), kInvC, q0);
    double D = __dadd_rn(1.0, V);
    if (BIN) {   // (an isolated template of a mixed CTA subtracts B = 0: (1 + V) - 0 = 1 + V)
      double B = 0.0;
      if (BIN == 2 || binary) B = __dmul_rn(apOm, k1_cos(__dmul_rn(Om, __dsub_rn(sC[c].y, tp.t_asc))));
      D = __dsub_rn(D, B);
    }
    const double x = ft_track_x(tp.f0, __dmul_rn(tp.f1, vzdt.y), D, f_min, inv_df);
    // (a 32.32 fixed-point variant -- one fp64 add, then integer rounding and tie test, three fp64 instructions fewer --
    // measured SLOWER, 11.7 -> 12.2 ms: the loop is as much issue- as fp64-bound)
    const double tm = __dadd_rn(x, kMagic);                 // rint(x) in the low mantissa bits
    const uint32_t k = (uint32_t)__double2loint(tm);
    const double r = __dsub_rn(x, __dsub_rn(tm, kMagic));   // x - rint(x)
    acc.ties += (fabs(r) > kTie) ? 1u : 0u;                 // within 1e-9 bin of a rounding tie
    // 0 <= rint(x) < 2^32 <=> the high word of tm is that of kMagic (false for NaN, inf, negative, huge)
    acc.bad |= (__double2hiint(tm) != 0x43380000 || k >= n_bins) ? 1u : 0u;
    const uint32_t kc = min(k, n_bins - 1u);
    const float pix = __ldg(prow + kc);
    if (STAT != 1) {
      double w = PERSFT ? sC[c].x : k1_f2d(__ldg(wrow + kc));
      if (SKY) {
        w = __dmul_rn(ft_antenna_u(sAnt + 9 * c, sk), w);
        acc.wsum = __dadd_rn(acc.wsum, w);
        if (EXT) acc.wsq = __fma_rn(w, w, acc.wsq);
      }
      acc.power = fma(w, k1_f2d(pix), acc.power);  // (fixed weights: exact product, same as mul then add)
      if (EXT) acc.wcount = __dadd_rn(acc.wcount, (pix > d.rho) ? w : 0.0);
    }
    if (STAT != 0) acc.count += (pix > d.rho) ? 1 : 0;
    prow += ld;
    if (!PERSFT) wrow += ld;
  }
}

// STAT: 0 power, 1 count, 2 both.  GEN: templates drawn in registers from (seed, first + q) instead of read.
// BEST: per-CTA loudest (value desc, index asc) to best_v / best_i [gridDim.x].
template <int STAT, bool GEN, bool BEST, bool SKY, bool EXT = false>
__global__ void __launch_bounds__(K1_THREADS)
ft_list_kernel(const __grid_constant__ FtDev d, const FtTemplateDev* __restrict__ tl, const __grid_constant__ FtBankBox bx,
               uint64_t seed, uint64_t first, int64_t n, double t_ref,
               float* __restrict__ out_power, int32_t* __restrict__ out_count, int32_t* __restrict__ err,
               unsigned long long* __restrict__ near_ties, double* __restrict__ best_v, int64_t* __restrict__ best_i,
               const uint32_t* __restrict__ perm, double wfloor = 0.0, int by_z = 0) {
  // per-SFT tables of the current chunk: (vx, vy), (vz, t - t_ref), (w, t): three LDS.128 per evaluation at most
  __shared__ double2 sA[K1_THREADS], sB[K1_THREADS], sC[K1_THREADS];
  __shared__ double sAnt[SKY ? 9 * K1_THREADS : 1];   // antenna coefficients A[5], B[4] of the chunk's SFTs
  const int64_t slot = (int64_t)blockIdx.x * K1_THREADS + threadIdx.x;
  const bool active = slot < n;
  const int64_t q = active ? (perm ? (int64_t)perm[slot] : slot) : 0;   // the template this thread evaluates
  const FtTemplateDev tp = GEN ? ft_bank_template(bx, seed, first + (uint64_t)(active ? q : 0)) : tl[active ? q : 0];
  const double Om = __ddiv_rn(FT_TWO_PI, tp.P_orb);
  const double apOm = __dmul_rn(tp.a_p, Om);
  const bool binary = tp.a_p != 0.0;
  const bool any_binary = __syncthreads_or(binary && active) != 0;
  const bool all_binary = __syncthreads_and(binary || !active) != 0;
  const uint32_t n_bins = (uint32_t)min(d.n_bins, (int64_t)0x7fffffff);
  const bool per_sft = d.wkind == 1;
  K1Acc acc{0.0, 0, 0u, 0u, 0.0, 0.0, 0.0};
  FtSkyPoint sk{};
  if (SKY) sk = ft_sky_point(tp.nx, tp.ny, tp.nz);
  for (int64_t a0 = 0; a0 < d.n_sft; a0 += K1_THREADS) {
    const int64_t a = a0 + threadIdx.x;
    __syncthreads();
    if (a < d.n_sft) {
      const double t = d.t_mid[a];
      sA[threadIdx.x] = make_double2(d.vel[3 * a], d.vel[3 * a + 1]);
      sB[threadIdx.x] = make_double2(d.vel[3 * a + 2], __dsub_rn(t, t_ref));
      sC[threadIdx.x] = make_double2(per_sft ? (double)d.w[a] : 0.0, t);
      if (SKY) {
#pragma unroll
        for (int q = 0; q < 9; ++q) sAnt[9 * threadIdx.x + q] = d.ant[9 * a + q];
      }
    }
    __syncthreads();
    const int m = (int)min((int64_t)K1_THREADS, d.n_sft - a0);
    if (active) {
      if (SKY) {   // (sky-dependent weights need per-SFT weights: ft_set_antenna)
        if (all_binary) k1_chunk<STAT, 2, true, true, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
        else if (any_binary) k1_chunk<STAT, 1, true, true, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
        else k1_chunk<STAT, 0, true, true, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
      } else if (all_binary) {
        if (per_sft) k1_chunk<STAT, 2, true, false, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
        else k1_chunk<STAT, 2, false, false, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
      } else if (any_binary) {
        if (per_sft) k1_chunk<STAT, 1, true, false, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
        else k1_chunk<STAT, 1, false, false, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
      } else {
        if (per_sft) k1_chunk<STAT, 0, true, false, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
        else k1_chunk<STAT, 0, false, false, EXT>(d, tp, Om, apOm, binary, sA, sB, sC, sAnt, sk, m, a0, n_bins, acc);
      }
    }
  }
  const double power = SKY ? acc.power / acc.wsum : acc.power;   // Eq. (5): sum_a w_a(n) = 1
  const int32_t count = acc.count;
  const bool bad = acc.bad != 0u;
  if (active) {
    if (bad) atomicExch(err, 1);
    if (STAT != 1 && out_power) out_power[q] = bad ? __int_as_float(0x7fc00000) : (float)power;
    if (STAT != 0 && out_count) out_count[q] = bad ? -1 : count;
    if (acc.ties && near_ties) atomicAdd(near_ties, (unsigned long long)acc.ties);
  }
  if (BEST) {
    // CTA-wide loudest under (value desc, index asc); out-of-range templates never win
    __shared__ double bv[K1_THREADS / 32];
    __shared__ long long bi[K1_THREADS / 32];
    double v = (active && !bad) ? (STAT == 1 ? (double)count : power) : -INFINITY;
    if (EXT) {   // the per-box step of the paper on a random bank: veto on the weighted number count, rank by z (Eq. 36)
      const double wc = SKY ? acc.wcount / acc.wsum : acc.wcount;
      const double mu = SKY ? 1.0 : d.mu_G, sigma = SKY ? sqrt(acc.wsq) / acc.wsum : d.sigma_G;
      if (by_z) v = (power - mu) / sigma;
      if (!(active && !bad) || wc < wfloor) v = -INFINITY;
    }
    long long i = active ? (long long)q : 0x7fffffffffffffffll;   // (the template's index, not the slot)
    for (int o = 16; o > 0; o >>= 1) {
      const double v2 = __shfl_xor_sync(0xffffffffu, v, o);
      const long long i2 = __shfl_xor_sync(0xffffffffu, i, o);
      if (v2 > v || (v2 == v && i2 < i)) { v = v2; i = i2; }
    }
    if ((threadIdx.x & 31) == 0) { bv[threadIdx.x >> 5] = v; bi[threadIdx.x >> 5] = i; }
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int wv = 1; wv < K1_THREADS / 32; ++wv)
        if (bv[wv] > v || (bv[wv] == v && bi[wv] < i)) { v = bv[wv]; i = bi[wv]; }
      if (EXT && v == -INFINITY) i = 0x7fffffffffffffffll;   // nobody of this CTA passed the veto
      best_v[blockIdx.x] = v; best_i[blockIdx.x] = i;
    }
  }
}

// final reduction of the per-CTA loudest: best_v[0], best_i[0] receive the winner
__global__ void __launch_bounds__(1024)
ft_best_reduce_kernel(double* __restrict__ best_v, int64_t* __restrict__ best_i, int64_t n) {
  __shared__ double sv[1024];
  __shared__ long long si[1024];
  double v = -INFINITY;
  long long i = 0x7fffffffffffffffll;
  for (int64_t e = threadIdx.x; e < n; e += blockDim.x) {
    const double v2 = best_v[e];
    const long long i2 = best_i[e];
    if (v2 > v || (v2 == v && i2 < i)) { v = v2; i = i2; }
  }
  sv[threadIdx.x] = v; si[threadIdx.x] = i;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      const double v2 = sv[threadIdx.x + o];
      const long long i2 = si[threadIdx.x + o];
      if (v2 > sv[threadIdx.x] || (v2 == sv[threadIdx.x] && i2 < si[threadIdx.x])) { sv[threadIdx.x] = v2; si[threadIdx.x] = i2; }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { best_v[0] = sv[0]; best_i[0] = si[0]; }
}

// ft_selftest kernels
__global__ void ft_selftest_div_kernel(uint64_t seed, int64_t n, unsigned long long* __restrict__ n_fail) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned fails = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const double u = ft_uniform(seed, (uint64_t)i, 0), s = ft_uniform(seed, (uint64_t)i, 1);
    double dot;
    switch (i & 7) {
      case 0: dot = (2.0 * u - 1.0) * 5e4; break;                               // the range of |v . n|, m/s
      case 1: dot = (2.0 * u - 1.0) * 3.1e4 * (0.5 + 0.5 * s); break;
      case 2: dot = ldexp(1.0 + u, (int)(s * 40.0) - 20); break;                // every binade around it
      case 3: dot = -ldexp(1.0 + u, (int)(s * 600.0) - 300); break;             // far scales
      case 4: dot = FT_C_LIGHT * (double)(1 + (long long)(u * 1e6)); break;     // exact quotients
      case 5: dot = FT_C_LIGHT * (1.0 + u) * ldexp(1.0, -52 + (int)(s * 50.0)); break;
      case 6: dot = (2.0 * u - 1.0) * 500.0; break;                             // the rotational part alone
      default: dot = (i & 8) ? 0.0 : -0.0; break;
    }
    const double a = ft_div_c(dot), b = __ddiv_rn(dot, FT_C_LIGHT);
    // (a zero quotient may come back with the other sign: D = (1 + V) - B does not see it)
    if (__double_as_longlong(a) != __double_as_longlong(b) && !(a == 0.0 && b == 0.0)) ++fails;
  }
  if (fails) atomicAdd(n_fail, (unsigned long long)fails);
}

__global__ void ft_selftest_cvt_kernel(int64_t n, unsigned long long* __restrict__ n_fail) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned fails = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    // n >= 2^32 covers every fp32 bit pattern; smaller n strides through them
    const uint32_t b = n >= (1ll << 32) ? (uint32_t)i : (uint32_t)((uint64_t)i * 0x9E3779B1ull);
    const float x = __uint_as_float(b);
    if (x != x) continue;
    if (__double_as_longlong(ft_f2d(x)) != __double_as_longlong((double)x)) ++fails;
  }
  if (fails) atomicAdd(n_fail, (unsigned long long)fails);
}

// perm (or nullptr) = scratch of n + K1_BUCKETS uint32: the evaluation order is built there first
// which = 2: k1_cos against the library cos(): failures = |difference| > 4e-16
__global__ void ft_selftest_cos_kernel(uint64_t seed, int64_t n, unsigned long long* __restrict__ n_fail) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned fails = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const double u = 2.0 * ft_uniform(seed, (uint64_t)i, 0) - 1.0;
    const double scale = (i & 3) == 0 ? 4.0 : (i & 3) == 1 ? 400.0 : (i & 3) == 2 ? 1e5 : 1e8;
    const double x = u * scale;
    if (!(fabs(k1_cos(x) - cos(x)) <= 4e-16)) ++fails;
  }
  if (fails) atomicAdd(n_fail, (unsigned long long)fails);
}

template <bool GEN, bool BEST>
cudaError_t launch_list(const FtDev& d, int stat, const FtTemplateDev* tl, const FtBankBox& bx, uint64_t seed, uint64_t first,
                        int64_t n, double t_ref, float* out_power, int32_t* out_count, int32_t* err,
                        unsigned long long* near_ties, double* best_v, int64_t* best_i, uint32_t* perm, cudaStream_t s,
                        int* launches, bool ext = false, double wfloor = 0.0, int by_z = 0) {
  *launches = 0;
  if (n <= 0) return cudaSuccess;
  const unsigned grid = (unsigned)((n + K1_THREADS - 1) / K1_THREADS);
  if (perm) {
    uint32_t* hist = perm + n;
    cudaError_t e = cudaMemsetAsync(hist, 0, sizeof(uint32_t) * K1_BUCKETS, s);
    if (e != cudaSuccess) return e;
    k1_hist_kernel<GEN><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, hist);
    k1_scan_kernel<<<1, 1024, 0, s>>>(hist);
    k1_scatter_kernel<GEN><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, hist, perm);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *launches += 3;
  }
  const bool sky = d.skyw && d.ant && stat != 1;   // (the number count does not see the weights)
  if constexpr (GEN && BEST) {
    if (ext) {   // ft_eval_bank_veto: both statistics + weighted count (+ sigma_G), veto and z in the winner search
      if (sky) ft_list_kernel<2, true, true, true, true><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm, wfloor, by_z);
      else ft_list_kernel<2, true, true, false, true><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm, wfloor, by_z);
      *launches += 1;
      return cudaGetLastError();
    }
  }
  if (stat == 0 && sky) ft_list_kernel<0, GEN, BEST, true><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm);
  else if (stat == 0) ft_list_kernel<0, GEN, BEST, false><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm);
  else if (stat == 1) ft_list_kernel<1, GEN, BEST, false><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm);
  else if (sky) ft_list_kernel<2, GEN, BEST, true><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm);
  else ft_list_kernel<2, GEN, BEST, false><<<grid, K1_THREADS, 0, s>>>(d, tl, bx, seed, first, n, t_ref, out_power, out_count, err, near_ties, best_v, best_i, perm);
  *launches += 1;
  return cudaGetLastError();
}

int check_box(ft_ctx* c, const ft_bank_box* b) {
  const double v[13] = {b->f0_lo, b->f0_hi, b->f1_lo, b->f1_hi, b->ra_lo, b->ra_hi, b->sd_lo, b->sd_hi, b->ap_lo, b->ap_hi,
                        b->porb_lo, b->porb_hi, b->t_ref};
  for (double x : v) if (!std::isfinite(x)) return ft_fail(c, FT_ERR_ARG, "ft_bank_box: non-finite value");
  if (!(b->f0_lo > 0.0) || b->f0_hi < b->f0_lo || b->f1_hi < b->f1_lo || b->ra_hi < b->ra_lo || b->sd_lo < -1.0 || b->sd_hi > 1.0 ||
      b->sd_hi < b->sd_lo || b->ap_lo < 0.0 || b->ap_hi < b->ap_lo || (b->ap_hi > 0.0 && (!(b->porb_lo > 0.0) || b->porb_hi < b->porb_lo)))
    return ft_fail(c, FT_ERR_ARG, "ft_bank_box: need 0 < f0_lo <= f0_hi, lo <= hi on every axis, |sin delta| <= 1, 0 < P_orb");
  return FT_OK;
}

FtBankBox to_dev_box(const ft_bank_box* b) {
  return FtBankBox{b->f0_lo, b->f0_hi, b->f1_lo, b->f1_hi, b->ra_lo, b->ra_hi, b->sd_lo, b->sd_hi, b->ap_lo, b->ap_hi,
                   b->porb_lo, b->porb_hi, b->t_ref};
}

}  // namespace

extern "C" {

int ft_eval_templates(ft_ctx* c, const ft_template* templates_dev, int64_t n, double t_ref, int stat,
                      double rho_th, float* out_power_dev, int32_t* out_count_dev) {
  if (!c) return FT_ERR_ARG;
  if (n < 0 || (n > 0 && !templates_dev)) return ft_fail(c, FT_ERR_ARG, "ft_eval_templates: NULL list");
  if (stat < 0 || stat > 2) return ft_fail(c, FT_ERR_ARG, "ft_eval_templates: stat must be power, hough or both");
  if (!std::isfinite(t_ref) || !std::isfinite(rho_th)) return ft_fail(c, FT_ERR_ARG, "ft_eval_templates: non-finite argument");
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_eval_templates: handle not created");
  static_assert(sizeof(ft_template) == 64 && sizeof(FtTemplateDev) == 64, "ft_template layout");
  if (n == 0) return FT_OK;
  if (int rc = ft_enter(c)) return rc;
  FtDev d = c->d;
  d.rho = (float)rho_th;
  uint32_t* perm = nullptr;
  if (n >= 4096 && n < (1ll << 32)) {   // evaluation order by f0 (small lists are launch-bound anyway)
    FT_CUDA(c, cudaStreamSynchronize(c->stream));   // the grow-only scratch may still be in use
    FT_CUDA(c, ft_grow(c->io_dev, c->io_cap, sizeof(uint32_t) * ((size_t)n + K1_BUCKETS)));
    perm = reinterpret_cast<uint32_t*>(c->io_dev);
  }
  FT_CUDA(c, cudaMemsetAsync(c->flag_dev, 0, sizeof(int32_t), c->stream));
  c->ev_used = 0; c->counters.stat_launches = 0;
  int launches = 0;
  ft_tick(c);
  const cudaError_t e = launch_list<false, false>(d, stat, reinterpret_cast<const FtTemplateDev*>(templates_dev), FtBankBox{}, 0, 0, n,
                                                  t_ref, out_power_dev, out_count_dev, c->flag_dev, c->near_ties_dev, nullptr, nullptr,
                                                  perm, c->stream, &launches);
  ft_tock(c, launches);
  if (e != cudaSuccess) return ft_fail(c, FT_ERR_CUDA, std::string("ft_eval_templates: ") + cudaGetErrorString(e));
  int32_t flag = 0;
  FT_CUDA(c, cudaMemcpyAsync(&flag, c->flag_dev, sizeof flag, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (flag) return ft_fail(c, FT_ERR_TRACK_RANGE, "ft_eval_templates: some tracks leave the spectrogram (their outputs are NaN / -1)");
  return FT_OK;
}

int ft_bank_draw(ft_ctx* c, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, ft_template* out_dev) {
  if (!c || !box) return FT_ERR_ARG;
  if (n < 0 || (n > 0 && !out_dev)) return ft_fail(c, FT_ERR_ARG, "ft_bank_draw: NULL output");
  if (int rc = check_box(c, box)) return rc;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_bank_draw: handle not created");
  if (n == 0) return FT_OK;
  if (int rc = ft_enter(c)) return rc;
  ft_bank_draw_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(to_dev_box(box), seed, first, n,
                                                                          reinterpret_cast<FtTemplateDev*>(out_dev));
  FT_CUDA(c, cudaGetLastError());
  c->counters.kernel_launches += 1;
  return FT_OK;
}

// ft_eval_bank (ext = false) and ft_eval_bank_veto (ext = true: both statistics, veto floor, rank by z; best_box_host)
static int eval_bank_impl(ft_ctx* c, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, int stat, double rho_th,
                          float* out_power_dev, int32_t* out_count_dev, ft_cand* best_host, ft_template* best_template_host,
                          bool ext, double wfloor, int by_z, ft_cand_box* best_box_host) {
  if (!c || !box) return FT_ERR_ARG;
  if (n < 1) return ft_fail(c, FT_ERR_ARG, "ft_eval_bank: n >= 1");
  if (!ext && stat != FT_STAT_POWER && stat != FT_STAT_HOUGH) return ft_fail(c, FT_ERR_ARG, "ft_eval_bank: stat must be power or hough");
  if (!std::isfinite(rho_th) || !std::isfinite(wfloor)) return ft_fail(c, FT_ERR_ARG, "ft_eval_bank: non-finite argument");
  if (int rc = check_box(c, box)) return rc;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_eval_bank: handle not created");
  if (int rc = ft_enter(c)) return rc;
  FtDev d = c->d;
  d.rho = (float)rho_th;
  const FtBankBox bx = to_dev_box(box);
  const int64_t n_blocks = (n + K1_THREADS - 1) / K1_THREADS;
  FT_CUDA(c, cudaStreamSynchronize(c->stream));   // the grow-only scratch may still be in use
  if (n >= (1ll << 32)) return ft_fail(c, FT_ERR_ARG, "ft_eval_bank: n < 2^32 per call (draw the bank in batches)");
  const size_t need = 16 * (size_t)n_blocks + sizeof(FtTemplateDev) + sizeof(FtCandDev) + sizeof(uint32_t) * ((size_t)n + K1_BUCKETS);
  FT_CUDA(c, ft_grow(c->io_dev, c->io_cap, need));
  double* best_v = reinterpret_cast<double*>(c->io_dev);
  int64_t* best_i = reinterpret_cast<int64_t*>(c->io_dev + 8 * (size_t)n_blocks);
  FtTemplateDev* tp_dev = reinterpret_cast<FtTemplateDev*>(c->io_dev + 16 * (size_t)n_blocks);
  FtCandDev* cand_dev = reinterpret_cast<FtCandDev*>(tp_dev + 1);
  uint32_t* perm = n >= 4096 ? reinterpret_cast<uint32_t*>(cand_dev + 1) : nullptr;
  FT_CUDA(c, cudaMemsetAsync(c->flag_dev, 0, sizeof(int32_t), c->stream));
  c->ev_used = 0; c->counters.stat_launches = 0;
  int launches = 0;
  ft_tick(c);
  const cudaError_t e = launch_list<true, true>(d, stat, nullptr, bx, seed, first, n, box->t_ref, out_power_dev, out_count_dev,
                                                c->flag_dev, c->near_ties_dev, best_v, best_i, perm, c->stream, &launches,
                                                ext, wfloor, by_z);
  ft_tock(c, launches);
  if (e != cudaSuccess) return ft_fail(c, FT_ERR_CUDA, std::string("ft_eval_bank: ") + cudaGetErrorString(e));
  ft_best_reduce_kernel<<<1, 1024, 0, c->stream>>>(best_v, best_i, n_blocks);
  FT_CUDA(c, cudaGetLastError());
  c->counters.kernel_launches += 1;
  int64_t win = 0;
  int32_t flag = 0;
  FT_CUDA(c, cudaMemcpyAsync(&win, best_i, sizeof win, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(&flag, c->flag_dev, sizeof flag, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (ext && (win < 0 || win >= n)) {   // the veto left no template (or every track left the spectrogram: flag below)
    if (best_box_host) { *best_box_host = ft_cand_box{}; best_box_host->idx = UINT64_MAX; best_box_host->box = -1; }
    if (flag) return ft_fail(c, FT_ERR_TRACK_RANGE, "ft_eval_bank_veto: some tracks leave the spectrogram (their outputs are NaN / -1; they never win)");
    return FT_OK;
  }
  if (win < 0 || win >= n) return ft_fail(c, FT_ERR_TRACK_RANGE, "ft_eval_bank: every track leaves the spectrogram");
  if (best_host || best_template_host || best_box_host) {
    // the winner again, in the refinement arithmetic (power, weighted count, count), from its regenerated parameters
    ft_bank_draw_kernel<<<1, 32, 0, c->stream>>>(bx, seed, first + (uint64_t)win, 1, tp_dev);
    FT_CUDA(c, cudaGetLastError());
    FT_CUDA(c, ft_launch_refine_template(d, reinterpret_cast<const double*>(tp_dev), box->t_ref, cand_dev, nullptr, c->flag_dev, c->stream));
    c->counters.kernel_launches += 2;
    FtCandDev cd;
    FtTemplateDev tp;
    FT_CUDA(c, cudaMemcpyAsync(&cd, cand_dev, sizeof cd, cudaMemcpyDeviceToHost, c->stream));
    FT_CUDA(c, cudaMemcpyAsync(&tp, tp_dev, sizeof tp, cudaMemcpyDeviceToHost, c->stream));
    FT_CUDA(c, cudaStreamSynchronize(c->stream));
    if (best_host) *best_host = ft_cand{cd.power, cd.wcount, (uint64_t)win, cd.count, -1};
    if (best_box_host) *best_box_host = ft_cand_box{cd.power, cd.wcount, (uint64_t)win, cd.count, -1, cd.z, cd.sigma};
    if (best_template_host) std::memcpy(best_template_host, &tp, sizeof tp);
  }
  if (flag) return ft_fail(c, FT_ERR_TRACK_RANGE, "ft_eval_bank: some tracks leave the spectrogram (their outputs are NaN / -1; they never win)");
  return FT_OK;
}

int ft_eval_bank(ft_ctx* c, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, int stat, double rho_th,
                 float* out_power_dev, int32_t* out_count_dev, ft_cand* best_host, ft_template* best_template_host) {
  return eval_bank_impl(c, box, seed, first, n, stat, rho_th, out_power_dev, out_count_dev, best_host, best_template_host,
                        false, 0.0, 0, nullptr);
}

int ft_eval_bank_veto(ft_ctx* c, const ft_bank_box* box, uint64_t seed, uint64_t first, int64_t n, double rho_th,
                      double wcount_floor, int rank_by_z, float* out_power_dev, int32_t* out_count_dev,
                      ft_cand_box* best_host, ft_template* best_template_host) {
  return eval_bank_impl(c, box, seed, first, n, FT_STAT_BOTH, rho_th, out_power_dev, out_count_dev, nullptr, best_template_host,
                        true, wcount_floor, rank_by_z ? 1 : 0, best_host);
}

int ft_track(ft_ctx* c, const ft_template* tp_host, double t_ref, int64_t* k_out_host) {
  if (!c || !tp_host || !k_out_host) return FT_ERR_ARG;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_track: handle not created");
  if (!std::isfinite(t_ref)) return ft_fail(c, FT_ERR_ARG, "ft_track: non-finite argument");
  if (int rc = ft_enter(c)) return rc;
  const size_t n = (size_t)c->d.n_sft;
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  FT_CUDA(c, ft_grow(c->io_dev, c->io_cap, sizeof(FtTemplateDev) + 8 * n));
  double* tp_dev = reinterpret_cast<double*>(c->io_dev);
  int64_t* k_dev = reinterpret_cast<int64_t*>(c->io_dev + sizeof(FtTemplateDev));
  FT_CUDA(c, cudaMemcpyAsync(tp_dev, tp_host, sizeof(FtTemplateDev), cudaMemcpyHostToDevice, c->stream));
  FT_CUDA(c, cudaMemsetAsync(c->flag_dev, 0, sizeof(int32_t), c->stream));
  FT_CUDA(c, ft_launch_refine_template(c->d, tp_dev, t_ref, nullptr, k_dev, c->flag_dev, c->stream));
  c->counters.kernel_launches += 1;
  int32_t flag = 0;
  FT_CUDA(c, cudaMemcpyAsync(k_out_host, k_dev, 8 * n, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaMemcpyAsync(&flag, c->flag_dev, sizeof flag, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  if (flag) return ft_fail(c, FT_ERR_TRACK_RANGE, "ft_track: the track leaves the spectrogram");
  return FT_OK;
}

int ft_selftest(ft_ctx* c, int which, int64_t n, uint64_t seed, uint64_t* n_fail_out) {
  if (!c || !n_fail_out || n < 0) return FT_ERR_ARG;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_selftest: handle not created");
  if (which < 0 || which > 2) return ft_fail(c, FT_ERR_ARG, "ft_selftest: which = 0 (division by c), 1 (fp32 -> fp64 conversion) or 2 (orbital cosine)");
  if (int rc = ft_enter(c)) return rc;
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  FT_CUDA(c, ft_grow(c->io_dev, c->io_cap, 8));
  unsigned long long* nf = reinterpret_cast<unsigned long long*>(c->io_dev);
  FT_CUDA(c, cudaMemsetAsync(nf, 0, 8, c->stream));
  if (which == 0) ft_selftest_div_kernel<<<ft_sm_count() * 8, 256, 0, c->stream>>>(seed, n, nf);
  else if (which == 1) ft_selftest_cvt_kernel<<<ft_sm_count() * 8, 256, 0, c->stream>>>(n, nf);
  else ft_selftest_cos_kernel<<<ft_sm_count() * 8, 256, 0, c->stream>>>(seed, n, nf);
  FT_CUDA(c, cudaGetLastError());
  c->counters.kernel_launches += 1;
  unsigned long long h = 0;
  FT_CUDA(c, cudaMemcpyAsync(&h, nf, 8, cudaMemcpyDeviceToHost, c->stream));
  FT_CUDA(c, cudaStreamSynchronize(c->stream));
  *n_fail_out = h;
  return FT_OK;
}

}  // extern "C"

// ---- ft_eval_templates_noalloc: K1 with its scratch in the static array at the top of this file --------------
namespace {

constexpr int kNoallocMaxDevices = 64;
constexpr size_t kNoallocTail = ((size_t)FT_NOALLOC_MAX_TEMPLATES + K1_BUCKETS) * sizeof(uint32_t);   // flag | ties
std::mutex g_noalloc_setup_mu;                          // guards the address table
std::mutex g_noalloc_call_mu[kNoallocMaxDevices];       // one call at a time per device: the array is shared
unsigned char* g_noalloc_ptr[kNoallocMaxDevices] = {};  // device address of ft_noalloc_scratch, per device ordinal

int noalloc_fail(char* msg, int64_t cap, int code, const char* fmt, ...) {
  if (msg && cap > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(msg, (size_t)cap, fmt, ap);
    va_end(ap);
  }
  return code;
}

// The array's address on the current device.  cudaGetSymbolAddress answers for the device that is current, so the
// table is per device; the first lookup on a device also loads this library's module there.
cudaError_t ft_noalloc_scratch_ptr(int dev, unsigned char** out) {
  std::lock_guard<std::mutex> g(g_noalloc_setup_mu);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, ft_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_ptr[dev];
  return cudaSuccess;
}

// true if p is device (or managed) memory reachable as such from device dev
bool noalloc_on_device(const void* p, int dev) {
  cudaPointerAttributes a{};
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return (a.type == cudaMemoryTypeDevice && a.device == dev) || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" {

int ft_eval_templates_noalloc(const float* P_dev, int64_t n_sft, int64_t n_bins, int64_t ld_bins,
                              const double* t_mid_dev, const double* vel_dev, const float* w_dev, int wkind,
                              double f_min, double df, const ft_template* templates_dev, int64_t n, double t_ref,
                              int stat, double rho_th, float* out_power_dev, int32_t* out_count_dev,
                              uint64_t* near_ties_host, void* cuda_stream, char* msg, int64_t cap) {
  if (msg && cap > 0) msg[0] = 0;
  if (near_ties_host) *near_ties_host = 0;
  if (!P_dev || !t_mid_dev || !vel_dev || !w_dev)
    return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: NULL spectrogram / table pointer");
  if (n_sft < 1 || n_bins < 1 || ld_bins < n_bins)
    return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: need n_sft >= 1, n_bins >= 1, ld_bins >= n_bins");
  if (wkind != FT_W_PER_SFT && wkind != FT_W_PER_SFT_BIN) return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: bad wkind");
  if (!std::isfinite(f_min) || !std::isfinite(df) || !(df > 0.0) || !std::isfinite(t_ref) || !std::isfinite(rho_th))
    return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: non-finite argument or df <= 0");
  if (stat < 0 || stat > 2) return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: stat must be power, hough or both");
  if (n < 0 || (n > 0 && !templates_dev)) return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: NULL list");
  if (n > (int64_t)FT_NOALLOC_MAX_TEMPLATES)
    return noalloc_fail(msg, cap, FT_ERR_ARG,
                        "ft_eval_templates_noalloc: n = %lld exceeds FT_NOALLOC_MAX_TEMPLATES = %d, the size of the built-in "
                        "work space; evaluate the bank in batches", (long long)n, FT_NOALLOC_MAX_TEMPLATES);
  if (n == 0) return FT_OK;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return noalloc_fail(msg, cap, FT_ERR_CUDA, "ft_eval_templates_noalloc: no CUDA device (%s); there is no CPU fallback", cudaGetErrorString(e));
  if (dev < 0 || dev >= kNoallocMaxDevices) return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: device ordinal %d not supported", dev);
  const void* ptrs[7] = {P_dev, t_mid_dev, vel_dev, w_dev, templates_dev, out_power_dev, out_count_dev};
  for (const void* p : ptrs)
    if (p && !noalloc_on_device(p, dev))
      return noalloc_fail(msg, cap, FT_ERR_ARG, "ft_eval_templates_noalloc: a pointer is not device memory of the current device %d", dev);
  unsigned char* scratch = nullptr;
  if ((e = ft_noalloc_scratch_ptr(dev, &scratch)) != cudaSuccess)   // first call on this device: symbol look-up (set-up)
    return noalloc_fail(msg, cap, FT_ERR_CUDA, "ft_eval_templates_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  FtDev d{};
  d.P = P_dev; d.w = w_dev; d.t_mid = t_mid_dev; d.vel = vel_dev;
  d.n_sft = n_sft; d.n_bins = n_bins; d.ld = ld_bins; d.wkind = wkind;
  d.f_min = f_min; d.inv_df = 1.0 / df; d.rho = (float)rho_th;
  uint32_t* perm = n >= 4096 ? reinterpret_cast<uint32_t*>(scratch) : nullptr;   // same ordering policy as ft_eval_templates
  int32_t* flag_dev = reinterpret_cast<int32_t*>(scratch + kNoallocTail);
  unsigned long long* ties_dev = reinterpret_cast<unsigned long long*>(scratch + kNoallocTail + 8);
  struct { int32_t flag; int32_t pad; unsigned long long ties; } tail{0, 0, 0};
  static_assert(sizeof(tail) == 16, "tail layout");
  {
    std::lock_guard<std::mutex> busy(g_noalloc_call_mu[dev]);   // held until the stream has drained: calls must not overlap
    // the array keeps the last call's contents: flag and counter start at zero here, the histogram inside launch_list
    if ((e = cudaMemsetAsync(scratch + kNoallocTail, 0, 16, s)) != cudaSuccess)
      return noalloc_fail(msg, cap, FT_ERR_CUDA, "ft_eval_templates_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
    int launches = 0;
    e = launch_list<false, false>(d, stat, reinterpret_cast<const FtTemplateDev*>(templates_dev), FtBankBox{}, 0, 0, n, t_ref,
                                  out_power_dev, out_count_dev, flag_dev, ties_dev, nullptr, nullptr, perm, s, &launches);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&tail, scratch + kNoallocTail, 16, cudaMemcpyDeviceToHost, s);
    const cudaError_t e2 = cudaStreamSynchronize(s);
    if (e == cudaSuccess) e = e2;
  }
  if (e != cudaSuccess) return noalloc_fail(msg, cap, FT_ERR_CUDA, "ft_eval_templates_noalloc: %s", cudaGetErrorString(e));
  if (near_ties_host) *near_ties_host = tail.ties;
  if (tail.flag)
    return noalloc_fail(msg, cap, FT_ERR_TRACK_RANGE, "ft_eval_templates_noalloc: some tracks leave the spectrogram (their outputs are NaN / -1)");
  return FT_OK;
}

}  // extern "C"
