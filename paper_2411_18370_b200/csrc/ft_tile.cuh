// Tile kernel K2 (ft_tile.cu): host-side plan and launchers.  DESIGN.md "Kernel K2".
#pragma once
#include <string>

#include "ft_common.cuh"
#include "ft_select.cuh"

struct FtTilePlan {
  // device buffers, grow-only across ft_tile_plan calls on the same plan object (freed by ft_tile_plan_free)
  int32_t* kst = nullptr;       // [n_tiles][n_sft] first staged bin of the strip (multiple of 4 / 16)
  size_t kst_cap = 0;
  int32_t* err = nullptr;       // [1] set by the kernel if a track left its staged strip (plan bug)
  double* vr = nullptr;         // [n_sft][2] scratch of the sky-axis velocity range
  size_t vr_cap = 0;
  int32_t mode = 0;             // 0: fp32 gather (ft_tile_kernel), 1: packed number count (ft_tile8_kernel),
                                // 2: both statistics in one pass (ft_tileb_kernel, J <= 16)
  int32_t cw = 32;              // f0 per chunk (per warp load instruction): 32 or 128
  int32_t n_tiles = 0;          // f0 tiles
  int32_t tile_w = 0;           // f0 per tile (multiple of 32; the last tile may hold fewer)
  int32_t J = 0;                // cw-wide f0 chunks per consumer warp (template parameter)
  int32_t wpp = 0;              // consumer warps per outer point
  int32_t R = 0;                // outer points per CTA
  int32_t pitch = 0;            // bins per staged row in shared memory (mode 1: per byte-shifted copy)
  int32_t copy_floats = 0;      // bins copied per row (multiple of 4, mode 1: 16; <= pitch)
  int32_t rows_per_stage = 0;   // divides 32
  int32_t n_stages = 0;
  int32_t ctas_per_sm = 0;
  size_t smem_bytes = 0;
};

// Decide eligibility (why->empty() == eligible) and build the per-(tile, SFT) strip table.
// `t_mid` / `vel` are the host copies of the per-SFT tables; `sky_host` etc. the grid axes.
struct FtTileHostIn {
  const double* t_mid; const double* vel;   // [n_sft], [n_sft][3]
  const double* sky; const double* a_p; const double* P_orb;
  double df; double eps_bound;
  int points_per_cta;
  int force_tiles;  // > 0: use exactly this many f0 tiles (FT_OPT_F0_TILES)
};
cudaError_t ft_tile_plan(const FtDev& d, const FtTileHostIn& in, cudaStream_t s, FtTilePlan* plan,
                         std::string* why, int* launches, int mode = 0);
uint64_t ft_tile_sample_points(const FtTilePlan& plan, uint64_t n_points, uint32_t k, uint32_t cap);
// One pass of the gather-reduce over array A (folded w*P for the power statistic, the 0/1 hit map
// for the number count); add_back is the constant the fold removed from A, summed over SFTs.
// Writes out_f (fp32) and/or out_i (int32) indexed from out_base, and/or
// filters into sel (bands of bpb f0 bins).  group_stride > 1: evaluate only groups 0, stride, 2 stride, ...
// (n_groups_strided of them; the threshold sample) and pack the outputs by launch-local row
// (group_local * R + r) * n_f0 + i_f0.  complement = true: every group EXCEPT those (the rest of the bank).
cudaError_t ft_launch_tile(const FtDev& d, const FtTilePlan& plan, const float* A, double add_back, uint64_t pt_begin,
                           uint64_t pt_end, float* out_f, int32_t* out_i, uint64_t out_base,
                           const FtSelectDev* sel, int32_t bpb, unsigned long long* near_ties,
                           cudaStream_t s, int* launches, uint32_t group_stride = 1, uint64_t n_groups_strided = 0,
                           bool complement = false);
cudaError_t ft_launch_hitmap(const float* P, float rho, float* H, int64_t n, cudaStream_t s);
cudaError_t ft_launch_hitmap8(const float* P, float rho, uint8_t* H8, int64_t n_sft, int64_t n_bins, int64_t ld,
                              int64_t ld8, cudaStream_t s);
// Q[a][k] = fl(fl(w P) - c_a) with c_a = fl(mean_k fl(w P)) per row; w_sft (per-SFT) or w_bin (per-bin).
cudaError_t ft_launch_fold_centered(const float* P, const float* w_sft, const float* w_bin, float* Q, float* c_row,
                                    int64_t n_sft, int64_t n_bins, int64_t ld, cudaStream_t s);
// QB = Q with the least significant bit replaced by the hit (P > rho): gather array of ft_tileb_kernel
cudaError_t ft_launch_qb(const float* Q, const float* P, float rho, float* QB, int64_t n, cudaStream_t s);
void ft_tile_plan_free(FtTilePlan* plan);
