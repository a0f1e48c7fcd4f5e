// sweep_tile.cuh - host interface of the tile sweep kernel (sweep_tile.cu)
#pragma once
#include <cuda_runtime.h>
#include <vector>
#include "dvm_dev.cuh"

namespace dvm {

struct TilePlan {
    size_t fbuf_doubles = 0;
    int nthreads = 0;
    size_t smem = 0;
};

bool tile_supported(int nx, int ny, int nz);
int tile_plan(int nx, int ny, int nz, const int lo[3][2], const int cnt[3][2], long long nvel, TilePlan *plan,
              std::vector<BlockDesc> *blocks);
cudaError_t launch_sweep_tile(const SweepParams &P, const TilePlan &plan, int nblocks, cudaStream_t st);

}  // namespace dvm
