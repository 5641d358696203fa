// dem_pair_fast.cu -- launchers of k_pose (a3) and k_pair_fast (a4-a7, packed FP32 contact search).  Kernels: dem_fast.cuh.
#include "dem_ctx.h"
#include "dem_fast.cuh"

namespace dem {

int pose_threads() { return DEM_POSE_THREADS; }
size_t pair_fast_smem_header() { return fast_smem_header(); }

void launch_pose(int dim, bool pos_is_double, int grid, cudaStream_t st, const PoseArgs& pa) {
    if (dim == 3) {
        if (pos_is_double) k_pose<double, 3><<<grid, DEM_POSE_THREADS, 0, st>>>(pa);
        else k_pose<float, 3><<<grid, DEM_POSE_THREADS, 0, st>>>(pa);
    } else {
        if (pos_is_double) k_pose<double, 2><<<grid, DEM_POSE_THREADS, 0, st>>>(pa);
        else k_pose<float, 2><<<grid, DEM_POSE_THREADS, 0, st>>>(pa);
    }
}

// a3 with the cull tests of the 3D search kernel (the library default path); smem = the staged shape tables
void launch_pose_cull(bool pos_is_double, int grid, size_t smem, cudaStream_t st, const PoseArgs& pa) {
    if (pos_is_double) {
        if (smem > 48 * 1024) cudaFuncSetAttribute(k_pose_cull<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        k_pose_cull<double><<<grid, DEM_POSE_THREADS, smem, st>>>(pa);
    } else {
        if (smem > 48 * 1024) cudaFuncSetAttribute(k_pose_cull<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        k_pose_cull<float><<<grid, DEM_POSE_THREADS, smem, st>>>(pa);
    }
}
int pose_cull_max_words() { return DEM_CM_WORDS; }

// tv3: 3 packed outer vertex pairs per sweep (tiles of 6 vertices) instead of 2 (tiles of 4)
cudaError_t launch_pair_fast(int dim, bool tv3, int grid, int threads, size_t smem, cudaStream_t st,
                             const PairArgs<float>& a) {
    void (*kern)(const PairArgs<float>);
    if (dim == 3) kern = tv3 ? k_pair_fast<3, 2, 3, 4> : k_pair_fast<3, 2, 2, 4>;
    else kern = tv3 ? k_pair_fast<2, 2, 3, 4> : k_pair_fast<2, 2, 2, 4>;
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}

}  // namespace dem
