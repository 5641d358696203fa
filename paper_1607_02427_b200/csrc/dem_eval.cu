// dem_eval.cu -- one force evaluation over the current neighbour list (steps a3-a8 of DESIGN.md): per pair class the
// pose kernel and the pair-feature kernel, then the per-particle reduction.  Kernels: dem_fast.cuh / dem_kernels.cuh,
// launched through the per-family launchers declared in dem_ctx.h.
#include <type_traits>

#include "dem_ctx.h"
#include "dem_kernels.cuh"

namespace dem {

namespace {

template <typename real>
int evaluate_t(dem_ctx* ctx, const void* pos, const void* quat, bool pos_is_double, const int32_t* sid, int N,
               void* force, void* torque, void* virial, const FinArgs* fin) {
    typedef typename vec4<real>::type real4;
    if (!ctx->have_list) return fail(ctx, DEM_ESTALE, "no neighbour list: call dem_build_neighbors first");
    if (N != ctx->N) return fail(ctx, DEM_ESTALE, "N = %d differs from the last build (%d)", N, ctx->N);
    if (!pos || !quat || !sid || !force || !torque) return fail(ctx, DEM_EINVAL, "null particle array");
    const int* skip = fin ? fin->bail : nullptr;
    // counters[0..7] (unsigned long long) followed by the per-class lengths of the k_pose work lists and the per-class
    // tile counters of the search kernel (int): one memset
    CU(cudaMemsetAsync(ctx->counters.p, 0, sizeof(unsigned long long) * 8 + sizeof(int) * 2 * DEM_MAX_CLASSES, ctx->stream));
    int* ccount = reinterpret_cast<int*>(ctx->counters.as<unsigned long long>() + 8);
    // capacity of a class's work list: its pairs plus the padding of every k_pose block to a whole warp tile
    const int pose_block = pose_threads();
    auto list_cap = [&](int c) { return (size_t)ctx->class_np[c] + 64u * (size_t)nblk(ctx->class_np[c], pose_block); };
    size_t list_base[DEM_MAX_CLASSES + 1];
    list_base[0] = 0;
    for (int c = 0; c < ctx->nclass; ++c) list_base[c + 1] = list_base[c] + list_cap(c);
    const bool search = std::is_same<real, float>::value && !ctx->generic_kernel;
    const bool cull = search && ctx->dim == 3 && ctx->cull;
    if (search) {
        CU(ctx->pose.reserve(sizeof(f4) * 3 * std::max<size_t>(list_base[ctx->nclass], 1)));
        CU(ctx->pidx.reserve(sizeof(int4) * std::max<size_t>(list_base[ctx->nclass], 1)));
        if (cull) CU(ctx->cmask.reserve(sizeof(unsigned) * pose_cull_max_words() * std::max<size_t>(list_base[ctx->nclass], 1)));
    }
    const BoxDev bx = box_dev(ctx->dim, ctx->box);
    // classes beyond the first populated one go to side streams (their kernels write disjoint records)
    int populated = 0, side_used = 0;
    for (int c = 0; c < ctx->nclass; ++c) populated += ctx->class_np[c] > 0;
    if (populated > 1) {
        if (!ctx->ev_fork) {
            CU(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
            for (int k = 0; k < 3; ++k) {
                CU(cudaStreamCreateWithFlags(&ctx->class_stream[k], cudaStreamNonBlocking));
                CU(cudaEventCreateWithFlags(&ctx->ev_join[k], cudaEventDisableTiming));
            }
        }
        CU(cudaEventRecord(ctx->ev_fork, ctx->stream));
    }
    // with several classes in flight at once the kernels' own durations overlap: one span from fork to join is timed
    // instead (pose + pair kernels of all classes; include/dem_bench.h)
    cudaEvent_t span0 = populated > 1 ? ev_mark(ctx) : nullptr;
    int seen = 0;
    for (int c = 0; c < ctx->nclass; ++c) {
        const int np = ctx->class_np[c];
        if (np == 0) continue;
        cudaStream_t st = ctx->stream;
        const int side = seen == 0 ? -1 : (seen - 1) % 3;
        if (side >= 0) {
            st = ctx->class_stream[side];
            if (side_used < 3 && seen - 1 < 3) CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));
            side_used = std::max(side_used, side + 1);
        }
        ++seen;
        const HostShape &HA = ctx->shapes[ctx->class_sa[c]], &HB = ctx->shapes[ctx->class_sb[c]];
        PairArgs<real> a;
        memset(&a, 0, sizeof a);
        a.table = ctx->table.as<real4>();
        a.sa = ctx->shape_dev[ctx->class_sa[c]];
        a.sb = ctx->shape_dev[ctx->class_sb[c]];
        a.pairs = ctx->pairs.as<int2>() + ctx->ct.pair_base[c];
        a.npairs = np;
        a.slices = ctx->ct.slices[c];
        a.n_outer = class_outer(ctx, c);
        a.rec = ctx->rec.as<real4>() + DEM_REC * (size_t)ctx->ct.rec_base[c];
        a.rflag = ctx->rflag.as<unsigned char>() + (size_t)ctx->ct.rec_base[c];
        a.pos = pos;
        a.quat = quat;
        a.box = bx;
        a.pos_double = pos_is_double ? 1 : 0;
        const double reach = reach_of(HA, HB), sigma = HA.rounding + HB.rounding;
        a.reach2 = reach * reach;
        a.pc.rc2 = (real)(std::cbrt(2.0) * sigma * sigma);
        a.pc.sig2 = (real)(sigma * sigma);
        a.pc.eps = (real)ctx->eps;
        a.pc.eps_par = (real)ctx->eps_par;
        a.pc.degen2 = (real)((1e-6 * sigma) * (1e-6 * sigma));
        a.counters = fin ? nullptr : ctx->counters.as<unsigned long long>();  // kept for dem_compute only
        a.cum = (ctx->timing && ctx->cum.p) ? ctx->cum.as<unsigned long long>() : nullptr;
        // candidate cutoff of the FP32 search kernel: FP32 rounding of the packed formulation (1e-3 relative) plus
        // its error on near-parallel edges, at most sin(angle) x edge length with the angle below ~1e-3 where the
        // line-line solve loses its digits; 4e-3 x longest edge leaves a factor 4
        const double rc = std::pow(2.0, 1.0 / 6.0) * sigma;
        const double rcs = rc * (1.0 + 1e-3) + (ctx->dim == 3 ? 4e-3 * std::max(HA.max_edge, HB.max_edge) : 0.0);
        a.rc2_search = (real)(rcs * rcs);
        const bool same = a.sa.off == a.sb.off;
        size_t smem = sizeof(real4) * (size_t)(a.sa.len + (same ? 0 : a.sb.len));
        const long long items = (long long)((np + 31) & ~31) * a.slices;
        const int threads = 128;
        int grid = (int)std::min<long long>(nblk(items, threads), (long long)ctx->sm_count * 64);
        cudaEvent_t e0 = populated > 1 ? nullptr : ev_mark(ctx, 1, st, true), em = e0;
        if constexpr (std::is_same<real, float>::value) {
            if (search) {
                // a3 (relative poses, reach test, compaction) runs as its own kernel in front of the search kernel
                a.pose = ctx->pose.as<f4>() + 3 * list_base[c];
                a.pidx = ctx->pidx.as<int4>() + list_base[c];
                a.plane = list_cap(c);
                a.count = ccount + c;
                PoseArgs pa;
                pa.pairs = a.pairs; pa.npairs = np; pa.slices = a.slices; pa.pos = pos; pa.quat = quat; pa.box = bx;
                pa.reach2 = a.reach2;
                pa.pose = ctx->pose.as<f4>() + 3 * list_base[c];
                pa.pidx = ctx->pidx.as<int4>() + list_base[c];
                pa.count = ccount + c;
                pa.plane = list_cap(c);
                pa.pad = cull ? 64 : 32;  // a warp of k_pair_cull takes 64 entries, of k_pair_fast 32
                pa.counters = a.counters;
                pa.rflag = a.rflag;
                pa.skip = skip;
                // culling: the cull tests run in the pose kernel (k_pose_cull), which hands per-pair survivor masks to the
                // search kernel and lists only pairs with a surviving feature -- unless the masks would not fit its
                // registers or the pairs are sliced (then k_pair_cull tests for itself)
                const int mw_e = (HB.ne + 31) / 32, mw_vj = (HB.nv + 31) / 32, mw_vi = (HA.nv + 31) / 32;
                const double ra = HA.circumradius + rcs, rb = HB.circumradius + rcs;
                const bool premask = cull && a.slices == 1 && mw_e + mw_vj + mw_vi <= pose_cull_max_words();
                if (premask) {
                    pa.table = a.table; pa.sa = a.sa; pa.sb = a.sb;
                    pa.cull_a2 = (float)(ra * ra);
                    pa.cull_b2 = (float)(rb * rb);
                    pa.cmask = ctx->cmask.as<unsigned>() + (size_t)pose_cull_max_words() * list_base[c];
                    pa.mw_e = mw_e; pa.mw_vj = mw_vj; pa.mw_vi = mw_vi;
                    a.cmask = pa.cmask; a.mw_e = mw_e; a.mw_vj = mw_vj; a.mw_vi = mw_vi;
                    launch_pose_cull(pos_is_double, nblk(np, pose_block), smem, st, pa);
                } else {
                    launch_pose(ctx->dim, pos_is_double, nblk(np, pose_block), st, pa);
                }
                LAUNCHED(ctx);
                if (populated == 1) em = ev_mark(ctx, 1, st, true);
                // the padded work list bounds the tiles; grid cap in blocks per SM measured on cfg4 for k_pair_cull (one
                // tile per warp beats one persistent wave of statically dealt tiles)
                const long long list_items = (long long)list_cap(c) * a.slices / (cull ? 2 : 1);
                grid = (int)std::min<long long>(nblk(list_items, threads), (long long)ctx->sm_count * 64);
                if (!cull) {  // k_pair_fast deals its tiles out through a counter (267.7 against 270.4 us on cfg4)
                    a.tile = ccount + DEM_MAX_CLASSES + c;
                    grid = (int)std::min<long long>(grid, (long long)ctx->sm_count * 4);  // one resident wave
                }
                if (cull) {
                    smem += pair_cull_smem_header();
                    a.cull_a2 = (real)(ra * ra);
                    a.cull_b2 = (real)(rb * rb);
                    CU(launch_pair_cull(same, grid, threads, smem, st, a));
                } else {
                    smem += pair_fast_smem_header();
                    // packed outer pairs per sweep: 3 when the vertex counts fill tiles of 6 at least as well as tiles of 4
                    auto waste = [](int n, int tile) { return ((n + tile - 1) / tile) * tile - n; };
                    const bool tv3 = waste(HA.nv, 6) + waste(HB.nv, 6) <= waste(HA.nv, 4) + waste(HB.nv, 4);
                    CU(launch_pair_fast(ctx->dim, tv3, grid, threads, smem, st, a));
                }
            } else {
                CU(launch_pair_generic_f32(ctx->dim, pos_is_double, grid, threads, smem, st, a));
            }
        } else {
            CU(launch_pair_generic_f64(ctx->dim, grid, threads, smem, st, a));
        }
        LAUNCHED(ctx);
        cudaEvent_t e1 = populated > 1 ? nullptr : ev_mark(ctx, 1, st, true);
        if (em != e0) ev_span(ctx, KT_POSE, e0, em);
        ev_span(ctx, KT_PAIR, em, e1);
    }
    for (int k = 0; k < side_used; ++k) {  // join the side streams
        CU(cudaEventRecord(ctx->ev_join[k], ctx->class_stream[k]));
        CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_join[k], 0));
    }
    if (populated > 1) ev_span(ctx, KT_PAIR, span0, ev_mark(ctx));
    cudaStream_t st = ctx->stream;
    cudaEvent_t r0 = ev_mark(ctx, 2);
    {
        FinArgs fa;
        if (fin) fa = *fin;
        else memset(&fa, 0, sizeof fa);
        // lanes per particle: one for large systems, several where there are too few particles to hide the latency of a
        // serial walk over a particle's slots (N = 256: 32 lanes)
        int lanes = 1;
        while (lanes < 32 && (long long)N * lanes < 65536) lanes <<= 1;
        fa.lanes = lanes;
        const int grid = nblk((long long)N * lanes, 256);
        const int* slot = ctx->slot.as<int>();
        const real4* rec = ctx->rec.as<real4>();
        const unsigned char* rf = ctx->rflag.as<unsigned char>();
        real4 *F = static_cast<real4*>(force), *T = static_cast<real4*>(torque);
        real* W = static_cast<real*>(virial);
        if (fa.mode == 2)
            k_finish<real, 2><<<grid, 256, 0, st>>>(N, ctx->stride, slot, sid, ctx->ct, ctx->nclass, rec, rf, F, T, W, fa);
        else if (fa.mode == 1)
            k_finish<real, 1><<<grid, 256, 0, st>>>(N, ctx->stride, slot, sid, ctx->ct, ctx->nclass, rec, rf, F, T, W, fa);
        else
            k_finish<real, 0><<<grid, 256, 0, st>>>(N, ctx->stride, slot, sid, ctx->ct, ctx->nclass, rec, rf, F, T, W, fa);
    }
    LAUNCHED(ctx);
    ev_span(ctx, KT_REDUCE, r0, ev_mark(ctx, 2));
    CU(cudaGetLastError());
    return DEM_OK;
}

}  // namespace

int evaluate(dem_ctx* ctx, const void* pos, const void* quat, bool pos_is_double, const int32_t* sid, int N, void* force,
             void* torque, void* virial, const FinArgs* fin) {
    if (particle2d_applies(ctx)) return launch_particle2d(ctx, pos, quat, pos_is_double, sid, N, force, torque, virial, fin);
    if (ctx->prec == DEM_F64) return evaluate_t<double>(ctx, pos, quat, true, sid, N, force, torque, virial, fin);
    return evaluate_t<float>(ctx, pos, quat, pos_is_double, sid, N, force, torque, virial, fin);
}

}  // namespace dem
