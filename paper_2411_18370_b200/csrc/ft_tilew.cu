// Tile kernel with a per-(outer point, SFT) weight: sky-dependent weights w_a(n) ∝ (a^2 + b^2)(t_a; n) / S_a
// normalised to sum 1 (Eq. 4-5).  The gathered array is the folded, centred r_a P (r_a ∝ 1/S_a
// the per-SFT weights given to ft_create); the antenna factor u_a(n) = a^2 + b^2 is computed next to the
// Doppler factor, once per (warp, SFT), and multiplies the row in a packed fp32 FMA; the normalisation
// sum_a u_a r_a, the add-back sum_a u_a c_a and sigma_G (Eq. 14) depend on the sky point only and come from a
// bind-time pass (ft_skyw_norm_kernel, fp64).
// Kernel body: ft_tile_body<J, GatherF32W> (ft_tile_dev.cuh).
#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tilew_max_regs(J))
ft_tilew_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  ft_tile_body<J, GatherF32W>(d, a);
}

// One CTA per sky point: the four sums over SFTs the epilogue of the row-weighted gather needs (fp64).
__global__ void __launch_bounds__(128)
ft_skyw_norm_kernel(const __grid_constant__ FtDev d, const float* __restrict__ cQ, const float* __restrict__ cWH,
                    double* __restrict__ out) {
  __shared__ double red[4][4];
  const int64_t i = blockIdx.x;
  const FtSkyPoint sp = ft_sky_point(d.sky[3 * i], d.sky[3 * i + 1], d.sky[3 * i + 2]);
  double s[4] = {0.0, 0.0, 0.0, 0.0};
  for (int64_t a = threadIdx.x; a < d.n_sft; a += blockDim.x) {
    const float uf = (float)ft_antenna_u(d.ant + 9 * (size_t)a, sp);   // as the gather applies it: one fp32 rounding
    const double ur = __dmul_rn((double)uf, (double)d.w[a]);
    s[0] += ur;
    s[1] += __dmul_rn(ur, ur);
    s[2] += __dmul_rn((double)uf, (double)cQ[a]);
    if (cWH) s[3] += __dmul_rn((double)uf, (double)cWH[a]);
  }
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    for (int o = 16; o > 0; o >>= 1) s[m] += __shfl_xor_sync(0xffffffffu, s[m], o);
    if ((threadIdx.x & 31) == 0) red[m][threadIdx.x >> 5] = s[m];
  }
  __syncthreads();
  if (threadIdx.x < 4) out[4 * i + threadIdx.x] = (red[threadIdx.x][0] + red[threadIdx.x][1]) + (red[threadIdx.x][2] + red[threadIdx.x][3]);
}

template <int J>
cudaError_t launchw_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  const cudaError_t e = ft_tile_allow_smem((const void*)ft_tilew_kernel<J>);
  if (e != cudaSuccess) return e;
  ft_tilew_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

cudaError_t ft_tilew_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launchw_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16) FT_CASE(20) FT_CASE(24) FT_CASE(28) FT_CASE(29) FT_CASE(30) FT_CASE(32)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t ft_launch_skyw_norm(const FtDev& d, const float* cQ, const float* cWH, double* out, cudaStream_t s) {
  ft_skyw_norm_kernel<<<(unsigned)d.n_sky, 128, 0, s>>>(d, cQ, cWH, out);
  return cudaGetLastError();
}
