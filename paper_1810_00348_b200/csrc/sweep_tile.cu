// sweep_tile.cu - DVM_KERNEL_TILE (placeholder until the tile kernel lands: reports "unsupported")
#include "sweep_tile.cuh"

namespace dvm {
bool tile_supported(int, int, int) { return false; }
int tile_plan(int, int, int, const int[3][2], const int[3][2], long long, TilePlan *, std::vector<BlockDesc> *) { return -1; }
cudaError_t launch_sweep_tile(const SweepParams &, const TilePlan &, int, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace dvm
