#include "ft_tile.cuh"
// placeholder until the tile kernel lands: never eligible
cudaError_t ft_tile_plan(const FtDev&, double, double, int, int, cudaStream_t, FtTilePlan*, std::string* why, int* launches) {
  *why = "tile kernel not built yet"; *launches = 0; return cudaSuccess;
}
uint64_t ft_tile_sample_points(const FtTilePlan&, uint64_t n_points) { return n_points; }
cudaError_t ft_launch_tile(const FtDev&, const FtTilePlan&, int, uint64_t, uint64_t, float*, int32_t*, uint64_t,
                           const FtSelectDev*, int32_t, unsigned long long*, cudaStream_t, int*) { return cudaErrorNotSupported; }
void ft_tile_plan_free(FtTilePlan* p) { if (p->kst) cudaFree(p->kst); if (p->vrange) cudaFree(p->vrange); *p = FtTilePlan{}; }
