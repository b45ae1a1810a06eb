// qmc_sweep_tile_f32.cu -- instantiations of the tiled FP32C sweep kernel (qmc_sweep_tile.cuh): K moves per barrier.
// V = 4 shapes need N % 4 == 0, V = 2 shapes N % 2 == 0; every shape needs N % K == 0 and N >= 2 K (planner).
#include "qmc_sweep_tile.cuh"

namespace qmc {

template <int T, int J, int V, int K>
static cudaError_t tile_launch(qmc_ctx *c, int n_sweeps, int smem)
{
    const uint2 key = make_uint2((uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    auto kern = sweep_tile_kernel<T, J, V, K>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    kern<<<c->W, T, smem, c->stream>>>(c->sv, c->trace, c->wo, key, c->t, n_sweeps);
    return cudaGetLastError();
}

template <int T, int J, int V, int K>
static int tile_occupancy(int smem)
{
    int n = 0;
    auto kern = sweep_tile_kernel<T, J, V, K>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, T, smem) != cudaSuccess) return 0;
    return n;
}

#define XT(T, J, V, K) {T, J, V, 1, K, tile_launch<T, J, V, K>, tile_occupancy<T, J, V, K>, sweep_tile_smem_bytes(T, J, K)},
static const SweepShape kShapesTile[] = {
    XT(32, 4, 4, 2) XT(32, 8, 4, 2) XT(32, 16, 4, 2) XT(32, 32, 4, 2)
    XT(64, 4, 4, 2) XT(64, 8, 4, 2) XT(64, 16, 4, 2) XT(64, 32, 4, 2)
    XT(128, 4, 4, 2) XT(128, 8, 4, 2) XT(128, 16, 4, 2)
    XT(256, 4, 4, 2) XT(256, 8, 4, 2) XT(512, 4, 4, 2) XT(512, 8, 4, 2) XT(512, 20, 4, 2) XT(1024, 8, 4, 2) XT(1024, 10, 2, 2)
    XT(32, 4, 4, 4) XT(32, 8, 4, 4) XT(32, 16, 4, 4)
    XT(64, 4, 4, 4) XT(64, 8, 4, 4) XT(64, 16, 4, 4)
    XT(128, 4, 4, 4) XT(128, 8, 4, 4) XT(128, 16, 4, 4)
    XT(256, 4, 4, 4) XT(256, 8, 4, 4) XT(512, 4, 4, 4) XT(512, 8, 4, 4) XT(512, 20, 4, 4) XT(1024, 8, 4, 4)
};
#undef XT

const SweepShape *sweep_shapes_tile(int *n) { *n = (int)(sizeof(kShapesTile) / sizeof(kShapesTile[0])); return kShapesTile; }

}  // namespace qmc
