// dem_pair_cull.cu -- launcher of k_pair_cull (the packed search kernel with exact per-feature culling, 3D).
#include <algorithm>
#include "dem_ctx.h"
#include "dem_fast.cuh"

namespace dem {

size_t pair_cull_smem_header() { return cull_smem_header(); }

cudaError_t launch_pair_cull(bool same_shape, int grid, int threads, size_t smem, cudaStream_t st,
                             const PairArgs<float>& a) {
    // Blocks per SM, measured with the cull tests in k_pose_cull: small shapes (octahedra, cfg4) run best at 4 (128
    // registers, some spills: 58.6 us from the lattice, 128.8 us thermalised) against 3 (168 registers, none: 63.1 / 148.0)
    // and 5 (96: 67.9 / 155.6); large tables (truncated icosahedra, cfg5) at 3 (51.0 against 55.0 us per class launch)
    // ... and large tables also take the variant with one sweep site per phase (6 k instead of 28 k instructions: config 5
    // 0.203 -> 0.178 ms per culled step; config 4 would lose 7 % to it)
    const bool small = a.sa.len + a.sb.len <= 512;
    const bool pre = a.cmask != nullptr;  // survivor masks from k_pose_cull (never for sliced pairs)
    // small shapes whose items always fit the list (octahedra, cubes, tetrahedra; their masks always fit k_pose_cull too):
    // no sweep behind the emit sites
    const bool fits = pre && a.slices == 1 && 64 * std::max(a.sb.ne, a.sa.nv + a.sb.nv) <= 1024;
    void (*kern)(const PairArgs<float>);
    if (!small) kern = same_shape ? k_pair_cull<3, true, true, false, false> : k_pair_cull<3, false, true, false, false>;
    else if (fits) kern = same_shape ? k_pair_cull<4, true, false, true, true> : k_pair_cull<4, false, false, true, true>;
    else if (pre) kern = same_shape ? k_pair_cull<4, true, false, false, true> : k_pair_cull<4, false, false, false, true>;
    else kern = same_shape ? k_pair_cull<4, true, false, false, false> : k_pair_cull<4, false, false, false, false>;
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}

}  // namespace dem
