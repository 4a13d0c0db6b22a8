// Tile kernel for the Hough number count (Eq. 7) on a packed hit map.
//
// The count needs one BIT per evaluation, (P[a][k] > rho_th); it is exact in any integer width.
// Same CTA / warp organisation, producer ring and canonical track entries as ft_tile.cu, but
//   * the gathered array is the hit map as BYTES, in four byte-shifted copies
//       H8[m][a][b] = (P[a][b + m] > rho_th),  m = 0..3,
//     so that the 4 hits of 4 consecutive f0 starting at any bin o are ONE aligned 32-bit word of
//     copy m = o mod 4;
//   * a thread owns 4 consecutive f0 per chunk (f0 = first + 128 j + 4 lane + c), loads that word
//     and adds it to a register holding four 8-bit counters: 1 LDS.32 + 1 IADD per 4 evaluations,
//     a quarter of the shared-memory traffic of the fp32 gather;
//   * every 224 SFTs the 8-bit counters are folded into 16-bit counters in shared memory
//     (n_sft <= 65535 is a plan condition), unpacked once in the epilogue.
// The staged bytes per SFT row are the same as for the fp32 strip (4 copies x 1 byte per bin).
// Kernel body: ft_tile_body<J, GatherHit8> (ft_tile_dev.cuh).
#include "ft_tile.cuh"
#include "ft_tile_dev.cuh"

namespace {

template <int J>
__global__ void __maxnreg__(ft_tile8_max_regs(J))
ft_tile8_kernel(const __grid_constant__ FtDev d, const __grid_constant__ FtTileArgs a) {
  ft_tile_body<J, GatherHit8>(d, a);
}

// H8[m][a][b] = (P[a][b + m] > rho) for b + m < n_bins, else 0
__global__ void ft_hitmap8_kernel(const float* __restrict__ P, float rho, uint8_t* __restrict__ H8,
                                  int64_t n_sft, int64_t n_bins, int64_t ld, int64_t ld8) {
  const int64_t n = 4 * n_sft * ld8, stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
    const int64_t b = e % ld8, a = (e / ld8) % n_sft, m = e / (ld8 * n_sft);
    H8[e] = (b + m < n_bins && P[a * ld + b + m] > rho) ? 1 : 0;
  }
}

template <int J>
cudaError_t launch8_J(const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t s) {
  const cudaError_t e = ft_tile_allow_smem((const void*)ft_tile8_kernel<J>);
  if (e != cudaSuccess) return e;
  ft_tile8_kernel<J><<<grid, block, smem, s>>>(d, a);
  return cudaGetLastError();
}

}  // namespace

cudaError_t ft_tile8_launch(int J, const FtDev& d, const FtTileArgs& a, unsigned grid, unsigned block, size_t smem,
                            cudaStream_t s) {
  switch (J) {
#define FT_CASE(j) case j: return launch8_J<j>(d, a, grid, block, smem, s);
    FT_CASE(1) FT_CASE(2) FT_CASE(3) FT_CASE(4) FT_CASE(5) FT_CASE(6) FT_CASE(7) FT_CASE(8) FT_CASE(10)
    FT_CASE(12) FT_CASE(15) FT_CASE(16)
#undef FT_CASE
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t ft_launch_hitmap8(const float* P, float rho, uint8_t* H8, int64_t n_sft, int64_t n_bins, int64_t ld,
                              int64_t ld8, cudaStream_t s) {
  ft_hitmap8_kernel<<<ft_sm_count() * 8, 256, 0, s>>>(P, rho, H8, n_sft, n_bins, ld, ld8);
  return cudaGetLastError();
}
