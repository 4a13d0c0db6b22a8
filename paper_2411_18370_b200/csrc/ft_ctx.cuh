// The handle behind the C ABI (include/fasttracks_b200.h) and the helpers shared by ft_api.cu (create, bind,
// evaluate) and ft_topk.cu (selection orchestration).
#pragma once
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/fasttracks_b200.h"
#include "ft_common.cuh"
#include "ft_select.cuh"
#include "ft_tile.cuh"

struct ft_ctx {
  cudaStream_t stream = nullptr;
  int device = 0;               // the device the handle was created on (made current by every call)
  FtDev d{};
  bool per_bin = false;
  // library-owned device memory
  double* t_mid_dev = nullptr;
  double* vel_dev = nullptr;
  float* w_dev = nullptr;       // per-SFT weights copy
  float* Q_dev = nullptr;       // folded, centred w*P (tile kernel input)
  float* cQ_dev = nullptr;      // [n_sft] the per-row constant removed from Q
  double add_back = 0.0;        // its sum over SFTs
  float* H_dev = nullptr;       // 0/1 hit map as fp32 (tile kernel input for the number count)
  float H_rho = 0.f; bool H_valid = false;
  float* WH_dev = nullptr;      // folded, centred w*[P > rho] (weighted number count)
  float* cWH_dev = nullptr;
  double add_back_wh = 0.0;
  float WH_rho = 0.f; bool WH_valid = false;
  double* w_row_dev = nullptr;  // [n_sft] row means of per-bin weights
  double* ant_dev = nullptr;    // [n_sft][9] antenna coefficients (ft_set_antenna)
  double* skyn_dev = nullptr;   // [n_sky][4] normalisation sums of the sky-dependent weights of the bound grid (grow-only)
  size_t skyn_cap = 0;
  double* axes_dev = nullptr;   // sky | a_p | P_orb | tasc (grow-only buffer)
  size_t axes_cap = 0;
  std::vector<double> axes_host;
  double* ctab_dev = nullptr;   // orbital cosine table of the bound grid (binary grids; grow-only buffer)
  size_t ctab_cap = 0;
  std::vector<double> ctab_key; // (t_ref, P_orb[], tasc_frac[]) the table was built for
  double* vr_dev = nullptr;     // [n_sft][2] sky-axis range of v.n/c of the bound grid
  int32_t* maxw_dev = nullptr;  // [4] widest strip per gather mode
  // host copies used for validation
  std::vector<double> t_mid, vel;
  double vmax = 0.0;
  // bound grid
  bool bound = false;
  int stat = 0;
  double df = 0.0;
  bool tile_ok = false;
  FtTilePlan plan{};            // fp32 gather (power; number count when the packed kernel is not eligible)
  FtTilePlan plan8{};           // packed number-count kernel (ft_tile8.cu)
  bool tile8_ok = false;
  FtTilePlan planb{};           // both statistics in one pass (ft_tileb.cu), narrow bands
  bool tileb_ok = false;
  FtTilePlan planw{};           // row-weighted gather (ft_tilew.cu): sky-dependent weights
  bool tilew_ok = false;
  float* QB_dev = nullptr;      // Q with the hit bit in the LSB
  float QB_rho = 0.f; bool QB_valid = false;
  uint8_t* H8_dev = nullptr;    // four byte-shifted hit maps
  float H8_rho = 0.f; bool H8_valid = false;
  // options
  int64_t opt_kernel = 0, opt_fused = 1, opt_ppc = 0, opt_packed = 1, opt_tiles = 0, opt_cap = 0, opt_floor = 0, opt_onepass = 1,
          opt_veto_first = 1, opt_tail = 1;
  double opt_wfloor = 0.0;
  // selection buffers
  FtSelectDev sel{};
  uint64_t* final_idx = nullptr;
  int32_t* final_region = nullptr;
  uint32_t* final_n = nullptr;   // [0] final_n, [1] overflow
  FtCandDev* cand = nullptr;
  FtCandDev* out_dev = nullptr;
  uint32_t final_cap = 0;
  size_t out_cap = 0;
  float* scratch_f = nullptr;
  int32_t* scratch_i = nullptr;
  size_t scratch_elems = 0;
  int32_t* veto_cnt = nullptr;  // number count of every template (FT_OPT_COUNT_FLOOR), grow-only
  float* veto_w = nullptr;      // weighted number count of every template (FT_OPT_WCOUNT_FLOOR), grow-only
  size_t veto_cap = 0, vetow_cap = 0;
  unsigned char* surv_dev = nullptr;  // veto-first selection: refined records | idx list | region offsets (grow-only)
  size_t surv_cap = 0;
  uint32_t* glist_dev = nullptr; // sample group list | skip bitmask | pbox row lists (grow-only)
  size_t glist_cap = 0;
  int32_t* pbox_dev = nullptr;
  size_t pbox_cap = 0;
  // small grow-only device scratch of the list / template calls
  unsigned char* io_dev = nullptr;
  size_t io_cap = 0;
  unsigned long long* near_ties_dev = nullptr;
  int32_t* flag_dev = nullptr;   // [1] error flag of the list kernels
  int32_t* tile_err_dev = nullptr;  // [1] planning-error flag of the tile kernels (all plans of the handle)
  // bookkeeping
  ft_counters counters{};
  std::vector<cudaEvent_t> evs;  // pairs around every statistic-kernel pass of the last call
  size_t ev_used = 0;
  std::string err = "";
  std::string desc = "no grid bound";
  std::string why;
};

int ft_fail(ft_ctx* c, int code, const std::string& msg);
#define FT_CUDA(c, expr)                                                                     \
  do {                                                                                       \
    cudaError_t e__ = (expr);                                                                \
    if (e__ != cudaSuccess)                                                                  \
      return ft_fail((c), e__ == cudaErrorMemoryAllocation ? FT_ERR_ALLOC : FT_ERR_CUDA,     \
                     std::string(#expr) + ": " + cudaGetErrorString(e__));                   \
  } while (0)

template <typename T>
inline void ft_dfree(T*& p) {
  if (p) cudaFree(p);
  p = nullptr;
}

// grow-only device buffer
template <typename T>
inline cudaError_t ft_grow(T*& p, size_t& cap, size_t need) {
  if (cap >= need) return cudaSuccess;
  if (p) cudaFree(p);
  p = nullptr; cap = 0;
  const cudaError_t e = cudaMalloc(&p, sizeof(T) * need);
  if (e == cudaSuccess) cap = need;
  return e;
}

// CUDA events on the handle's stream around each statistic pass (ft_counters.last_kernel_ms)
void ft_tick(ft_ctx* c);
void ft_tock(ft_ctx* c, int launches);
// The tile kernels raise plan.err if a track left its staged strip (a planning bug, never data): surfaced at
// every synchronising call instead of silently wrong sums.
int ft_check_tile_err(ft_ctx* c);
int ft_tile_err_status(ft_ctx* c, int32_t e);   // the same for a flag value already copied to the host
// make the handle's device current
int ft_enter(ft_ctx* c);

// What a statistic pass is asked for (ft_run_stat): which statistic, over which points, where to.
struct FtPass {
  int stat = FT_STAT_POWER;
  uint64_t pt_begin = 0, pt_end = 0;
  float* out_f = nullptr;          // fp32 statistic (power / weighted count / count as float)
  int32_t* out_i = nullptr;        // integer count
  uint64_t out_base = 0;
  bool filter = false;             // fused filter into c->sel
  int32_t bpb = 1, n_bands = 1;
  const int32_t* pbox = nullptr;
  int zmode = 0, out_key = 0;
  const uint32_t* glist = nullptr; uint32_t n_glist = 0;
  const uint32_t* gskip = nullptr;
  const uint32_t* skip_host = nullptr; uint32_t n_skip_host = 0;   // the groups gskip marks, sorted (host), for the split tail
};
int ft_run_stat(ft_ctx* c, const FtPass& p);
