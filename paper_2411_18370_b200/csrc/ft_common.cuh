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
  int64_t n_sft, n_bins, ld;
  int64_t n_f0, n_sky;
  int32_t n_f1, n_ap, n_porb, n_tasc;
  int32_t wkind;
  float rho;
  double f_min, inv_df, f0_start, df0, f1_start, df1, t_ref;
  uint64_t n_points;  // n_sky*n_ap*n_porb*n_tasc*n_f1 ; canonical idx = point*n_f0 + i_f0
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

// D_alpha = (1 + V) - B, the bracket of Eq. (2) at SFT alpha.
__device__ __forceinline__ double ft_doppler(const FtDev& d, const FtPoint& p, int64_t a, double t) {
  const double vx = d.vel[3 * a + 0], vy = d.vel[3 * a + 1], vz = d.vel[3 * a + 2];
  const double V = __ddiv_rn(__dadd_rn(__dadd_rn(__dmul_rn(vx, p.nx), __dmul_rn(vy, p.ny)), __dmul_rn(vz, p.nz)), FT_C_LIGHT);
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

// order-preserving float <-> uint32 key (larger float -> larger key)
__device__ __forceinline__ uint32_t ft_key(float v) {
  const uint32_t u = __float_as_uint(v);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ft_unkey(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// Candidate record as it sits in device buffers.
struct FtCandDev {
  double power;
  double wcount;
  uint64_t idx;
  int32_t count;
  int32_t band;
};

// ---- host-visible launchers (defined in the .cu files) ---------------------------------------
struct FtSelectBuffers;  // ft_select.cu

cudaError_t ft_launch_generic(const FtDev& d, int stat, uint64_t pt_begin, uint64_t pt_end,
                              float* out_power, int32_t* out_count, uint64_t out_base_idx,
                              cudaStream_t s);
cudaError_t ft_launch_refine(const FtDev& d, const uint64_t* idx_dev, const uint32_t* n_dev, int64_t n_max,
                             FtCandDev* out, unsigned long long* near_ties, cudaStream_t s);
// ctab[(i_porb*n_tasc + i_tasc)][a] = cos(Om (t_mid[a] - t_asc)), the same expression ft_doppler evaluates
cudaError_t ft_launch_ctab(const FtDev& d, double* ctab, cudaStream_t s);
// K1: explicit template list (records of 8 doubles: f0, f1, nx, ny, nz, a_p, P_orb, t_asc), device memory
cudaError_t ft_launch_list(const FtDev& d, int stat, const void* templates_dev, int64_t n, double t_ref,
                           float* out_power, int32_t* out_count, int32_t* err, unsigned long long* near_ties,
                           cudaStream_t s);
