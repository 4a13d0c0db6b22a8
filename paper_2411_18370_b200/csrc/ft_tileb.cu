// Tile kernel for BOTH statistics in one pass (narrow bands, J <= 16 chunks per warp).
//
// The gathered array is QB: the folded, centred power array Q rounded to 18 mantissa bits, with the number-count
// hit bit (P > rho_th) in the least significant of the six freed bits (a perturbation of at most 3.8e-6 of |Q|
// per pixel, random in sign: ~3e-8 of the statistic, inside the accumulation budget of DESIGN.md "Accumulation").
// One LDS.32 then feeds both Eq. (3) (packed fp32 add) and Eq. (7) (ONE integer add of the raw word; the low six
// bits of the sum are the hits of the last <= 63 rows, folded into 16-bit counters per block of 32 SFTs), so the
// binary configuration computes both statistics, and applies the number-count veto of PAPER.md:496-502 in the
// fused filter, in a single gather.  Kernel body: ft_tile_body<J, GatherBoth> (ft_tile_dev.cuh).
#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tileb_max_regs(J))
ft_tileb_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  ft_tile_body<J, GatherBoth>(d, a);
}

// QB[a][k] = Q[a][k] rounded (to nearest, on the magnitude) to a multiple of 64 ulp, low bits = (P[a][k] > rho)
__global__ void ft_qb_kernel(const float* __restrict__ Q, const float* __restrict__ P, float rho,
                             float* __restrict__ QB, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint32_t b = __float_as_uint(Q[i]);
    uint32_t r = (b + 32u) & ~63u;                       // (a carry into the exponent is the correct rounding up)
    if ((r & 0x7f800000u) == 0x7f800000u) r = b & ~63u;  // never round a finite value to infinity
    QB[i] = __uint_as_float(r | (P[i] > rho ? 1u : 0u));
  }
}

template <int J>
cudaError_t launchb_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  const cudaError_t e = ft_tile_allow_smem((const void*)ft_tileb_kernel<J>);
  if (e != cudaSuccess) return e;
  ft_tileb_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

cudaError_t ft_tileb_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launchb_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t ft_launch_qb(const float* Q, const float* P, float rho, float* QB, int64_t n, cudaStream_t s) {
  ft_qb_kernel<<<ft_sm_count() * 8, 256, 0, s>>>(Q, P, rho, QB, n);
  return cudaGetLastError();
}
