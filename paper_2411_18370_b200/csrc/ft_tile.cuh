// Tile kernels (ft_tile.cu, ft_tilew.cu, ft_tileb.cu, ft_tile8.cu): host-side plan and launchers.  DESIGN.md "Kernel K2".
#pragma once
#include <string>

#include "ft_common.cuh"
#include "ft_select.cuh"

struct FtTilePlan {
  // device buffers, grow-only across plans on the same object (freed by ft_tile_plan_free)
  int32_t* kst = nullptr;       // [n_tiles][n_sft] first staged bin of the strip (multiple of 4 / 16)
  size_t kst_cap = 0;
  int32_t* err = nullptr;       // [1] set by the kernel if a track left its staged strip (plan bug); the handle's, shared by its plans
  int32_t mode = 0;             // 0: fp32 gather (ft_tile_kernel), 1: packed number count (ft_tile8_kernel),
                                // 2: both statistics in one pass (ft_tileb_kernel, J <= 16),
                                // 3: fp32 gather times a per-(point, SFT) weight (ft_tilew_kernel)
  int32_t cw = 32;              // f0 per chunk (per warp load instruction): 32 or 128
  int32_t align = 4;            // strip start / length granularity, bins
  int32_t n_tiles = 0;          // f0 tiles
  int32_t tile_w = 0;           // f0 per tile (multiple of cw; the last tile may hold fewer)
  int32_t J = 0;                // cw-wide f0 chunks per consumer warp (template parameter)
  int32_t wpp = 0;              // consumer warps per outer point
  int32_t R = 0;                // outer points per CTA
  int32_t ppw = 1;              // outer points per consumer warp: 2 = narrow band with a ragged tail (ft_tile2.cu; then J = 2 (n_f0 / 32) + 1)
  int32_t pitch = 0;            // bins per staged row in shared memory (mode 1: per byte-shifted copy)
  int32_t copy_floats = 0;      // bins copied per row (multiple of align; <= pitch)
  int32_t rows_per_stage = 0;   // divides 32
  int32_t n_stages = 0;
  int32_t ctas_per_sm = 0;
  size_t smem_bytes = 0;
};

// `t_mid` / `vel` are the host copies of the per-SFT tables; `sky_host` etc. the grid axes.
struct FtTileHostIn {
  const double* t_mid; const double* vel;   // [n_sft], [n_sft][3]
  const double* sky; const double* a_p; const double* P_orb;
  double df; double eps_bound;
  int points_per_cta;
  int force_tiles;  // > 0: use exactly this many f0 tiles (FT_OPT_F0_TILES)
  int tail_packing; // 1: narrow bands may run two points per warp (FT_OPT_TAIL_PACKING)
};

// A plan is built in three steps so that one bind costs ONE stream synchronisation for all gather modes:
//   ft_tile_choose  (host: tiling, *why says why the grid is not tileable)
//   ft_tile_strips  (device: the per-(tile, SFT) strip table from the sky-axis velocity range vr_dev)
//   ft_tile_finish  (host, after the widest strip came back: shared-memory ring)
bool ft_tile_choose(const FtDev& d, const FtTileHostIn& in, int mode, FtTilePlan* plan, std::string* why);
cudaError_t ft_launch_vrange(const FtDev& d, double* vr_dev /*[n_sft][2]*/, cudaStream_t s);
cudaError_t ft_tile_strips(const FtDev& d, const FtTileHostIn& in, FtTilePlan* plan, const double* vr_dev,
                           int32_t* max_w_dev, cudaStream_t s);
bool ft_tile_finish(const FtDev& d, FtTilePlan* plan, int32_t max_w, std::string* why);
uint64_t ft_tile_sample_points(const FtTilePlan& plan, uint64_t n_points, uint32_t k, uint32_t cap);
cudaError_t ft_tile_allow_smem(const void* func);

// What one pass of the gather-reduce reads and writes.
struct FtTileRun {
  const float* A = nullptr;       // gathered array (Q: power; 0/1 hit map: count; folded w x hit: weighted count; QB)
  double add_back = 0.0;          // the constant the fold removed from A, summed over SFTs
  const float* c_row = nullptr;   // that constant per SFT (row-weighted gather)
  float* out_f = nullptr;         // fp32 / int32 outputs indexed from out_base, or nullptr
  int32_t* out_i = nullptr;
  uint64_t out_base = 0;
  const FtSelectDev* sel = nullptr;   // fused filter into these buffers (regions of bpb f0 bins x pbox)
  int32_t bpb = 1;
  const int32_t* pbox = nullptr; int32_t n_bands = 1;
  int32_t zmode = 0, out_key = 0;
  double z_mu = 0.0, z_inv_sigma = 1.0;
  float* out_sigma = nullptr;
  const double* sky_norm = nullptr;   // row-weighted gather: [n_sky][4] normalisation sums (ft_launch_skyw_norm)
  int32_t norm_cb = 2;                // which add-back column of sky_norm: 2 (power array Q) or 3 (weighted hits WH)
  unsigned long long* near_ties = nullptr;
  const uint32_t* skip_host = nullptr;   // with gskip: the skipped groups, sorted ascending (host copy), for the split tail
  uint32_t n_skip_host = 0;
};
// glist != nullptr: evaluate only the CTA groups glist[0 .. n_glist) (the threshold sample; a group = R consecutive
// outer points) and pack the outputs by launch-local row (group_local * R + r) * n_f0 + i_f0.  gskip != nullptr (a
// bit per group): every group EXCEPT those whose bit is set (the rest of the bank).  Both need pt_begin = 0.
cudaError_t ft_launch_tile(const FtDev& d, const FtTilePlan& plan, const FtTileRun& run, uint64_t pt_begin,
                           uint64_t pt_end, cudaStream_t s, int* launches, const uint32_t* glist = nullptr,
                           uint32_t n_glist = 0, const uint32_t* gskip = nullptr);
cudaError_t ft_launch_hitmap(const float* P, float rho, float* H, int64_t n, cudaStream_t s);
cudaError_t ft_launch_hitmap8(const float* P, float rho, uint8_t* H8, int64_t n_sft, int64_t n_bins, int64_t ld,
                              int64_t ld8, cudaStream_t s);
// Q[a][k] = fl(fl(w p) - c_a), c_a = fl(mean_k fl(w p)) per row; p = P, or [P > rho] when hits; w_sft (per-SFT) or
// w_bin (per-bin); w_row (optional) receives the row mean of w.
cudaError_t ft_launch_fold_centered(const float* P, const float* w_sft, const float* w_bin, float* Q, float* c_row,
                                    double* w_row, int64_t n_sft, int64_t n_bins, int64_t ld, int hits, float rho,
                                    cudaStream_t s);
// QB = Q with the least significant bit replaced by the hit (P > rho): gather array of ft_tileb_kernel
cudaError_t ft_launch_qb(const float* Q, const float* P, float rho, float* QB, int64_t n, cudaStream_t s);
// Sky-dependent weights: per sky point  sum_a u_a r_a,  sum_a (u_a r_a)^2,  sum_a u_a cQ_a,  sum_a u_a cWH_a  with
// u_a = fl32(a^2 + b^2) as the row-weighted gather applies it (cWH may be nullptr).  out [n_sky][4].
cudaError_t ft_launch_skyw_norm(const FtDev& d, const float* cQ, const float* cWH, double* out, cudaStream_t s);
void ft_tile_plan_free(FtTilePlan* plan);
