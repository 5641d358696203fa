// dem_pair_generic.cu -- launchers of the generic fused pair kernel k_pair (a3-a7 in one kernel: FP64 contexts, and
// FP32 contexts in 2D or after dem_set_pair_kernel(DEM_KERNEL_GENERIC)).  Kernel: dem_kernels.cuh.
#include "dem_ctx.h"
#include "dem_kernels.cuh"

namespace dem {

template <typename real>
static cudaError_t launch(void (*kern)(const PairArgs<real>), int grid, int threads, size_t smem, cudaStream_t st,
                          const PairArgs<real>& a) {
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}

cudaError_t launch_pair_generic_f32(int dim, bool pos_is_double, int grid, int threads, size_t smem, cudaStream_t st,
                                    const PairArgs<float>& a) {
    void (*kern)(const PairArgs<float>);
    if (pos_is_double) kern = dim == 3 ? k_pair<float, double, 3> : k_pair<float, double, 2>;
    else kern = dim == 3 ? k_pair<float, float, 3> : k_pair<float, float, 2>;
    return launch<float>(kern, grid, threads, smem, st, a);
}

cudaError_t launch_pair_generic_f64(int dim, int grid, int threads, size_t smem, cudaStream_t st,
                                    const PairArgs<double>& a) {
    return launch<double>(dim == 3 ? k_pair<double, double, 3> : k_pair<double, double, 2>, grid, threads, smem, st, a);
}

}  // namespace dem
