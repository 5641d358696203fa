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
    void (*kern)(const PairArgs<float>) =
        small ? (same_shape ? k_pair_cull<4, true, false, false> : k_pair_cull<4, false, false, false>)
              : (same_shape ? k_pair_cull<3, true, true, false> : k_pair_cull<3, false, true, false>);
    const bool fits = a.slices == 1 && 64 * std::max(a.sb.ne, a.sa.nv + a.sb.nv) <= 1024;
    // small shapes whose items always fit the list (octahedra, cubes, tetrahedra): no sweep behind the emit sites,
    // 12 k instead of 28 k instructions (cfg4: 51.0 -> 50.4 us from the lattice, 127.0 -> 125.9 thermalised)
    if (small && fits) kern = same_shape ? k_pair_cull<4, true, false, true> : k_pair_cull<4, false, false, true>;
    if (smem > 48 * 1024) {
        const cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, threads, smem, st>>>(a);
    return cudaSuccess;
}

}  // namespace dem
