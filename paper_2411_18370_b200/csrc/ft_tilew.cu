// Tile kernel with a per-(outer point, SFT) weight: sky-dependent weights w_a(n) ∝ (a^2 + b^2)(t_a; n) / S_a
// normalised to sum 1 (Eq. 4-5).  The gathered array is the folded, centred r_a P (r_a ∝ 1/S_a
// the per-SFT weights given to ft_create); the antenna factor u_a(n) = a^2 + b^2 is computed next to the
// Doppler factor, once per (warp, SFT), and multiplies the row in a packed fp32 FMA; the normalisation
// sum_a u_a r_a, the add-back sum_a u_a c_a and sigma_G (Eq. 14) are accumulated in fp64 alongside.
// Kernel body: ft_tile_body<J, GatherF32W> (ft_tile_dev.cuh).
#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tilew_max_regs(J))
ft_tilew_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  ft_tile_body<J, GatherF32W>(d, a);
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
    FT_CASE(12) FT_CASE(15) FT_CASE(16)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}
