// Shared device-side declarations of the fasttracks B200 library (product code; shares nothing
// with oracle/).  Canonical track arithmetic: DESIGN.md "Canonical computation", Eq. (2).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define FT_C_LIGHT 299792458.0
#define FT_TWO_PI 6.283185307179586  // nearest double to 2*pi

// Everything a kernel needs about the bound spectrogram + grid.  Passed by value (__grid_constant__).
struct FtDev {
  const float* P;       // [n_sft][ld]
  const float* w;       // per-SFT [n_sft] or per-bin [n_sft][ld]
  const float* Q;       // folded w*P, one fp32 rounding per pixel, [n_sft][ld] (tile kernel input)
  const float* H;       // hit map (P > rho) ? 1 : 0 as fp32, [n_sft][ld] (tile kernel input, number count)
  const uint8_t* H8;    // packed hit maps: H8[m][a][b] = (P[a][b+m] > rho), m = 0..3, rows of ld8 bytes (ft_tile8.cu)
  int64_t ld8;
  const double* t_mid;  // [n_sft]
  const double* vel;    // [n_sft][3]
  const double* sky;    // [n_sky][3]
  const double* a_p;    // [n_ap]
  const double* P_orb;  // [n_porb]
  const double* tasc;   // [n_tasc]
  const double* ctab;   // [n_porb*n_tasc][n_sft] cos(Om (t_mid - t_asc)) or nullptr (binary grids, bind time)
  const double* ant;    // [n_sft][9] antenna-pattern coefficients A[5], B[4] of the SFT's detector and sidereal
                        // angle (ft_set_antenna), or nullptr: weights w are used as given
  const float* c_row;   // [n_sft] per-row constant the fold removed from Q (row-weighted gather add-back)
  int64_t n_sft, n_bins, ld;
  int64_t n_f0, n_sky;
  int32_t n_f1, n_ap, n_porb, n_tasc;
  int32_t wkind;
  int32_t skyw;         // 1: sky-dependent weights w_a(n) = u_a(n) w_a / sum_b u_b(n) w_b, u = a^2 + b^2 (Eq. 4-5)
  float rho;
  double f_min, inv_df, f0_start, df0, f1_start, df1, t_ref;
  uint64_t n_points;  // n_sky*n_ap*n_porb*n_tasc*n_f1 ; canonical idx = point*n_f0 + i_f0
  double mu_G, sigma_G; // sum_a w_a and sqrt(sum_a w_a^2) of the fixed weights (Eq. 13-14 on the P = s/2 scale)
};

// Parameters of one "outer point" = everything of a template but f0.
struct alignas(16) FtPoint {
  double nx, ny, nz;
  double apOm;   // a_p * Om
  double Om;     // 2 pi / P_orb
  double t_asc;  // t_ref + u * P_orb
  double f1;
  const double* crow;  // row of ctab for this (P_orb, t_asc), or nullptr
  bool binary;   // a_p != 0
};

__device__ __forceinline__ FtPoint ft_decode_point(const FtDev& d, uint64_t pt) {
  const uint32_t i_f1 = (uint32_t)(pt % (uint64_t)d.n_f1);   pt /= (uint64_t)d.n_f1;
  const uint32_t i_ta = (uint32_t)(pt % (uint64_t)d.n_tasc); pt /= (uint64_t)d.n_tasc;
  const uint32_t i_po = (uint32_t)(pt % (uint64_t)d.n_porb); pt /= (uint64_t)d.n_porb;
  const uint32_t i_ap = (uint32_t)(pt % (uint64_t)d.n_ap);   pt /= (uint64_t)d.n_ap;
  FtPoint p;
  p.nx = d.sky[3 * pt + 0]; p.ny = d.sky[3 * pt + 1]; p.nz = d.sky[3 * pt + 2];
  const double a_p = d.a_p[i_ap];
  const double P_orb = d.P_orb[i_po];
  p.Om = __ddiv_rn(FT_TWO_PI, P_orb);
  p.t_asc = __dadd_rn(d.t_ref, __dmul_rn(d.tasc[i_ta], P_orb));
  p.apOm = __dmul_rn(a_p, p.Om);
  p.binary = (a_p != 0.0);
  p.crow = d.ctab ? d.ctab + ((size_t)i_po * (size_t)d.n_tasc + i_ta) * (size_t)d.n_sft : nullptr;
  p.f1 = __dadd_rn(d.f1_start, __dmul_rn((double)i_f1, d.df1));
  return p;
}

// V = dot / c as q0 = dot * (1/c), V = q0 + (dot - q0 c) (1/c): the residual is exact in the fused multiply-add,
// and the corrected quotient is the correctly rounded one (Markstein's theorem: 1/c is correctly rounded and q0
// is within an ulp); ft_selftest(0) compares it with __ddiv_rn bit for bit.
__device__ __forceinline__ double ft_div_c(double dot) {
  const double kInvC = 1.0 / FT_C_LIGHT;
  const double q0 = __dmul_rn(dot, kInvC);
  return __fma_rn(__fma_rn(-q0, FT_C_LIGHT, dot), kInvC, q0);
}


// D_alpha = (1 + V) - B, the bracket of Eq. (2) at SFT alpha.
__device__ __forceinline__ double ft_doppler(const FtDev& d, const FtPoint& p, int64_t a, double t) {
  const double vx = d.vel[3 * a + 0], vy = d.vel[3 * a + 1], vz = d.vel[3 * a + 2];
  const double V = __ddiv_rn(__dadd_rn(__dadd_rn(__dmul_rn(vx, p.nx), __dmul_rn(vy, p.ny)), __dmul_rn(vz, p.nz)), FT_C_LIGHT);
  double B = 0.0;
  if (p.binary) B = __dmul_rn(p.apOm, p.crow ? p.crow[a] : cos(__dmul_rn(p.Om, __dsub_rn(t, p.t_asc))));
  return __dsub_rn(__dadd_rn(1.0, V), B);
}

// The same with V = dot / c by ft_div_c (the same bits, a fraction of the instructions): per-evaluation kernels.
__device__ __forceinline__ double ft_doppler_rcp(const FtDev& d, const FtPoint& p, int64_t a, double t) {
  const double vx = d.vel[3 * a + 0], vy = d.vel[3 * a + 1], vz = d.vel[3 * a + 2];
  const double V = ft_div_c(__dadd_rn(__dadd_rn(__dmul_rn(vx, p.nx), __dmul_rn(vy, p.ny)), __dmul_rn(vz, p.nz)));
  double B = 0.0;
  if (p.binary) B = __dmul_rn(p.apOm, p.crow ? p.crow[a] : cos(__dmul_rn(p.Om, __dsub_rn(t, p.t_asc))));
  return __dsub_rn(__dadd_rn(1.0, V), B);
}

// x = ((f0 + f1dt) * D - f_min) * inv_df, every operation rounded (no FMA contraction).
__device__ __forceinline__ double ft_track_x(double f0, double f1dt, double D, double f_min, double inv_df) {
  return __dmul_rn(__dsub_rn(__dmul_rn(__dadd_rn(f0, f1dt), D), f_min), inv_df);
}
__device__ __forceinline__ double ft_f0(const FtDev& d, int64_t i) {
  return __dadd_rn(d.f0_start, __dmul_rn((double)i, d.df0));
}
__device__ __forceinline__ bool ft_near_tie(double x) {
  return fabs((x - floor(x)) - 0.5) < 1e-9;
}

// Antenna-pattern weights (Eq. 4; a, b of Jaranowski, Krolak & Schutz 1998, the paper's ref. [20],
// Eq. (12)-(13) there), written as a(t; n) = sum_m A_m(t) Y_m(n), b(t; n) = sum_m B_m(t) Z_m(n): the detector
// and time dependence A[5], B[4] sits in a per-SFT table built at ft_set_antenna, the sky dependence below
// (no trigonometric call: cos/sin of the right ascension and declination come from the unit vector n).
struct FtSkyPoint { double Y[5], Z[4]; };

__device__ __forceinline__ FtSkyPoint ft_sky_point(double nx, double ny, double nz) {
  const double rho2 = nx * nx + ny * ny;
  const double rho = sqrt(rho2), r = sqrt(rho2 + nz * nz);
  const double ca = rho > 0.0 ? nx / rho : 1.0, sa = rho > 0.0 ? ny / rho : 0.0;   // at the poles a^2 + b^2 does not depend on alpha
  const double sd = nz / r, cd = rho / r;
  const double c2a = ca * ca - sa * sa, s2a = 2.0 * sa * ca;
  const double s2d = 2.0 * sd * cd, c2d = cd * cd - sd * sd;
  FtSkyPoint p;
  p.Y[0] = (3.0 - c2d) * c2a; p.Y[1] = (3.0 - c2d) * s2a; p.Y[2] = s2d * ca; p.Y[3] = s2d * sa; p.Y[4] = cd * cd;
  p.Z[0] = sd * c2a; p.Z[1] = sd * s2a; p.Z[2] = cd * ca; p.Z[3] = cd * sa;
  return p;
}
// u = a^2 + b^2 at one SFT (ant = that SFT's row of FtDev::ant)
__device__ __forceinline__ double ft_antenna_u(const double* __restrict__ ant, const FtSkyPoint& p) {
  const double a = ant[0] * p.Y[0] + ant[1] * p.Y[1] + ant[2] * p.Y[2] + ant[3] * p.Y[3] + ant[4] * p.Y[4];
  const double b = ant[5] * p.Z[0] + ant[6] * p.Z[1] + ant[7] * p.Z[2] + ant[8] * p.Z[3];
  return a * a + b * b;
}

// order-preserving float <-> uint32 key (larger float -> larger key)
__device__ __forceinline__ uint32_t ft_key(float v) {
  const uint32_t u = __float_as_uint(v);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ft_unkey(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// Candidate record as it sits in device buffers (ft_cand: the first 32 bytes; ft_cand_box: all 48).
struct FtCandDev {
  double power;
  double wcount;
  uint64_t idx;
  int32_t count;
  int32_t band;    // region of the selection (frequency sub-band, or box)
  double z;        // (power - mu_G) / sigma_G of the template's weights (Eq. 36)
  double sigma;    // sigma_G
};

// Number of SMs of the CURRENT device (cudaDevAttrMultiProcessorCount, looked up once per device; 148 on a B200):
// grids of helper launches, the threshold sample and the split tail are sized from it.  Thread-safe.  (ft_tile.cu)
int ft_sm_count();

// ---- host-visible launchers (defined in the .cu files) ---------------------------------------
struct FtSelectBuffers;  // ft_select.cu

cudaError_t ft_launch_generic(const FtDev& d, int stat, uint64_t pt_begin, uint64_t pt_end,
                              float* out_power, int32_t* out_count, uint64_t out_base_idx,
                              cudaStream_t s);
cudaError_t ft_launch_refine(const FtDev& d, const uint64_t* idx_dev, const uint32_t* n_dev, int64_t n_max,
                             FtCandDev* out, unsigned long long* near_ties, cudaStream_t s);
// ctab[(i_porb*n_tasc + i_tasc)][a] = cos(Om (t_mid[a] - t_asc)), the same expression ft_doppler evaluates
cudaError_t ft_launch_ctab(const FtDev& d, double* ctab, cudaStream_t s);
// one explicit template (record of 8 doubles: f0, f1, nx, ny, nz, a_p, P_orb, t_asc) in fp64; optional bins k_out[n_sft]
cudaError_t ft_launch_refine_template(const FtDev& d, const double* template_dev, double t_ref, FtCandDev* out,
                                      int64_t* k_out, int32_t* err, cudaStream_t s);
