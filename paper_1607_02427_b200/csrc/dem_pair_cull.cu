// dem_pair_cull.cu -- launcher of k_pair_cull (the packed search kernel with exact per-feature culling, 3D).
#include "dem_ctx.h"
#include "dem_fast.cuh"

namespace dem {

size_t pair_cull_smem_header() { return cull_smem_header(); }

cudaError_t launch_pair_cull(bool same_shape, int grid, int threads, size_t smem, cudaStream_t st,
                             const PairArgs<float>& a) {
    // measured on cfg4: 167 registers without spills beat 128 / 96 / 80 with
    void (*kern)(const PairArgs<float>) = same_shape ? k_pair_cull<3, true> : k_pair_cull<3, false>;
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}

}  // namespace dem
