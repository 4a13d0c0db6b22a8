// Tile kernel K2 (ft_tile.cu): host-side plan and launchers.
#pragma once
#include <string>

#include "ft_common.cuh"
#include "ft_select.cuh"

struct FtTilePlan {
  int32_t* kst = nullptr;     // [n_tiles][n_sft] first staged bin of the strip (multiple of 4)
  double* vrange = nullptr;   // [n_sft][2] min / max of v.n/c over the sky axis
  int32_t n_tiles = 0;        // f0 tiles
  int32_t tile_w = 0;         // f0 per tile
  int32_t pitch = 0;          // floats per staged row
  int32_t points_per_cta = 0; // R
  int32_t j_per_thread = 0;   // J
  int32_t rows_per_stage = 0; // C
  int32_t n_stages = 0;
  int32_t n_consumer_warps = 0;
  int32_t n_producer_warps = 0;
  int32_t variant = -1;
  size_t smem_bytes = 0;
  int64_t n_sft_alloc = 0;
};

// Decide eligibility (why->empty() == eligible) and build the per-(tile, SFT) strip table.
cudaError_t ft_tile_plan(const FtDev& d, double df, double eps_bound, int stat, int points_per_cta,
                         cudaStream_t s, FtTilePlan* plan, std::string* why, int* launches);
uint64_t ft_tile_sample_points(const FtTilePlan& plan, uint64_t n_points);
cudaError_t ft_launch_tile(const FtDev& d, const FtTilePlan& plan, int stat, uint64_t pt_begin,
                           uint64_t pt_end, float* out_power, int32_t* out_count, uint64_t out_base,
                           const FtSelectDev* sel, int32_t bpb, unsigned long long* near_ties,
                           cudaStream_t s, int* launches);
void ft_tile_plan_free(FtTilePlan* plan);
