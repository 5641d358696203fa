// dem_step2d.cu -- launcher of k_particle2d (dem_step2d.cuh): the 2D hot path of a DEM_F32 context in one kernel.
#include "dem_ctx.h"
#include "dem_step2d.cuh"

namespace dem {

bool particle2d_applies(const dem_ctx* ctx) {
    return ctx->dim == 2 && ctx->prec == DEM_F32 && ctx->particle2d && ctx->max_count <= DEM_P2D_MAXNB;
}

int launch_particle2d(dem_ctx* ctx, const void* pos, const void* quat, bool pos_is_double, const int32_t* sid, int N,
                      void* force, void* torque, void* virial, const FinArgs* fin) {
    if (!ctx->have_list) return fail(ctx, DEM_ESTALE, "no neighbour list: call dem_build_neighbors first");
    if (N != ctx->N) return fail(ctx, DEM_ESTALE, "N = %d differs from the last build (%d)", N, ctx->N);
    if (!pos || !quat || !sid) return fail(ctx, DEM_EINVAL, "null particle array");
    cudaStream_t st = ctx->stream;
    Particle2DArgs a;
    memset(&a, 0, sizeof a);
    a.N = N;
    a.stride = ctx->stride;
    a.counts = ctx->counts.as<int>();
    a.list = ctx->list.as<int>();
    a.sid = sid;
    a.table = ctx->table.as<f4>();
    a.nshape = (int)ctx->shapes.size();
    for (int s = 0; s < a.nshape; ++s) {
        a.shape[s] = ctx->shape_dev[s];
        a.rounding[s] = ctx->shapes[s].rounding;
        a.circum[s] = ctx->shapes[s].circumradius;
        a.table_len = std::max(a.table_len, ctx->shape_dev[s].off + ctx->shape_dev[s].len);
    }
    a.eps = (float)ctx->eps;
    a.eps_par = (float)ctx->eps_par;
    a.cull = ctx->cull ? 1 : 0;
    a.box = box_dev(2, ctx->box);
    a.pos = pos;
    a.quat = quat;
    a.force = static_cast<f4*>(force);
    a.torque = static_cast<f4*>(torque);
    a.virial = static_cast<float*>(virial);
    if (fin) a.fin = *fin;
    if (a.fin.mode != 2 && (!force || !torque)) return fail(ctx, DEM_EINVAL, "null output array");
    if (a.fin.mode == 2 && (a.fin.pos == pos || a.fin.quat == quat))
        return fail(ctx, DEM_EINVAL, "k_particle2d: the drifted state needs buffers of its own");
    // counters are read by dem_get_counters after dem_compute; inside dem_step only bench's swept totals are kept
    if (!fin) {
        CU(cudaMemsetAsync(ctx->counters.p, 0, sizeof(unsigned long long) * 8, st));
        a.counters = ctx->counters.as<unsigned long long>();
    }
    a.swept = (ctx->timing && ctx->cum.p) ? ctx->cum.as<unsigned long long>() : nullptr;
    const size_t smem = particle2d_smem(a.table_len);
    void (*kern)(const Particle2DArgs) = pos_is_double ? k_particle2d<double> : k_particle2d<float>;
    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaEvent_t e0 = ev_mark(ctx);
    kern<<<nblk(N, DEM_P2D_THREADS), DEM_P2D_THREADS, smem, st>>>(a);
    LAUNCHED(ctx);
    ev_span(ctx, KT_PAIR, e0, ev_mark(ctx));
    CU(cudaGetLastError());
    return DEM_OK;
}

}  // namespace dem
