// dem_noalloc.cu -- dem_energy_static: the energies of a state (U, K_trans, K_rot; include/dem.h) computed without a
// single device allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
// harnesses that forbid it).  dem_energy keeps its per-block partial sums in a buffer the context allocates and grows;
// here they go to a file-scope device array of fixed size, which every GPU that loads the library holds until exit.
//
// The array's name is a host-side stand-in in host code, not a device address: its address is taken once per device
// with cudaGetSymbolAddress (that device current) and handed to the kernels as an ordinary pointer.
//
// All calls share the array.  Nothing in it has to start at zero: a call reads only the entries its own first kernel
// has just written (3 doubles per block of that call), so contents left by earlier calls are never looked at.  Calls
// that overlap on the GPU (different streams, or graphs replayed concurrently) race on it; calls on one stream do not.
#include <mutex>

#include "dem_ctx.h"
#include "dem_kernels.cuh"

namespace dem {
namespace {

constexpr int ES_THREADS = 256;
constexpr int ES_MAX_BLOCKS = (DEM_ENERGY_STATIC_MAX_N + ES_THREADS - 1) / ES_THREADS;  // 4096 blocks: 96 KiB of scratch
constexpr int ES_MAX_DEVICES = 64;

static __device__ __align__(256) double g_energy_partial[3 * ES_MAX_BLOCKS];

// the arithmetic of k_energy (dem_integrate.cuh): per-block partial sums of U, K_trans, K_rot in double, fixed order
template <typename real, typename PosT>
__global__ void __launch_bounds__(ES_THREADS) k_energy_static(int N, int dim, const int* __restrict__ sid, MassTable mt,
                                                              const PosT* __restrict__ quat, const PosT* __restrict__ vel,
                                                              const PosT* __restrict__ ang,
                                                              const typename vec4<real>::type* __restrict__ force,
                                                              double* __restrict__ partial) {
    __shared__ double sh[3][ES_THREADS];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double U = 0, Kt = 0, Kr = 0;
    if (i < N) {
        const int s = sid[i];
        const d4 v = load4d(vel, i), L = load4d(ang, i), q = load4d(quat, i);
        U = (double)force[i].w;
        Kt = 0.5 * mt.mass[s] * (v.x * v.x + v.y * v.y + v.z * v.z);
        double M[9];
        quat_to_mat<double>(q.x, q.y, q.z, q.w, M);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (dim == 2 && a < 2) continue;
            const double Lb = M[a] * L.x + M[3 + a] * L.y + M[6 + a] * L.z;
            const double I = mt.inertia[s][a];
            if (I > 0.0) Kr += 0.5 * Lb * Lb / I;
        }
    }
    sh[0][threadIdx.x] = U; sh[1][threadIdx.x] = Kt; sh[2][threadIdx.x] = Kr;
    __syncthreads();
    for (int o = ES_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o)
            for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0)
        for (int a = 0; a < 3; ++a) partial[3 * blockIdx.x + a] = sh[a][0];
}

// one block adds the nb partial sums of this call (fixed order: strided per thread, then a tree) into out[3]
__global__ void __launch_bounds__(ES_THREADS) k_energy_static_sum(int nb, const double* __restrict__ partial,
                                                                  double* __restrict__ out) {
    __shared__ double sh[3][ES_THREADS];
    double s[3] = {0, 0, 0};
    for (int b = threadIdx.x; b < nb; b += ES_THREADS)
        for (int a = 0; a < 3; ++a) s[a] += partial[3 * b + a];
    for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] = s[a];
    __syncthreads();
    for (int o = ES_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o)
            for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 3) out[threadIdx.x] = sh[threadIdx.x][0];
}

// device address of the scratch array on the current device, looked up once per device
int scratch_address(dem_ctx* ctx, double** out) {
    static std::mutex mu;
    static double* ptr[ES_MAX_DEVICES] = {};
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= ES_MAX_DEVICES) return fail(ctx, DEM_EINVAL, "device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        CU(cudaGetSymbolAddress((void**)&p, g_energy_partial));
        if (!p) return fail(ctx, DEM_ECUDA, "cudaGetSymbolAddress returned a null address");
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return DEM_OK;
}

template <typename real>
int energy_static_t(dem_ctx* ctx, const void* quat, const void* vel, const void* ang, const int32_t* sid,
                    const void* force, int N, double* out_dev) {
    typedef typename vec4<real>::type real4;
    MassTable mt;  // from the registered shapes (host data): the context's device tables are not touched
    memset(&mt, 0, sizeof mt);
    for (size_t s = 0; s < ctx->shapes.size(); ++s) {
        mt.mass[s] = ctx->shapes[s].mass;
        for (int a = 0; a < 3; ++a) mt.inertia[s][a] = ctx->shapes[s].inertia[a];
    }
    double* partial = nullptr;
    CHECK(scratch_address(ctx, &partial));
    const int nb = nblk(N, ES_THREADS);
    k_energy_static<real, real><<<nb, ES_THREADS, 0, ctx->stream>>>(
        N, ctx->dim, sid, mt, static_cast<const real*>(quat), static_cast<const real*>(vel), static_cast<const real*>(ang),
        static_cast<const real4*>(force), partial);
    LAUNCHED(ctx);
    k_energy_static_sum<<<1, ES_THREADS, 0, ctx->stream>>>(nb, partial, out_dev);
    LAUNCHED(ctx);
    CU(cudaGetLastError());
    return DEM_OK;
}

}  // namespace
}  // namespace dem

extern "C" int dem_energy_static(dem_ctx* ctx, const void* quat, const void* vel, const void* angmom,
                                 const int32_t* shape_id, const void* force_energy, int N, double* out_dev) {
    if (!ctx) return DEM_EINVAL;
    if (!quat || !vel || !angmom || !shape_id || !force_energy || !out_dev) return dem::fail(ctx, DEM_EINVAL, "null array");
    if (N < 1) return dem::fail(ctx, DEM_EINVAL, "N must be >= 1");
    if (N > DEM_ENERGY_STATIC_MAX_N)
        return dem::fail(ctx, DEM_EINVAL, "dem_energy_static: N = %d exceeds DEM_ENERGY_STATIC_MAX_N = %d (the static scratch "
                         "holds 3 doubles per 256 particles); use dem_energy", N, DEM_ENERGY_STATIC_MAX_N);
    if (ctx->shapes.empty()) return dem::fail(ctx, DEM_EINVAL, "no shapes registered");
    return ctx->prec == DEM_F64
               ? dem::energy_static_t<double>(ctx, quat, vel, angmom, shape_id, force_energy, N, out_dev)
               : dem::energy_static_t<float>(ctx, quat, vel, angmom, shape_id, force_energy, N, out_dev);
}
