// dem_lib.cu -- C ABI (include/dem.h) and host orchestration of libdem_b200.  Kernels: dem_kernels.cuh.
// There is no CPU path: every computing entry point launches CUDA kernels and fails with DEM_ECUDA without a device.
#include <type_traits>

#include "dem_ctx.h"
#include "dem_integrate.cuh"
#include "dem_list.cuh"

using namespace dem;

namespace {

// in-place exclusive scan of data[0..n); data must have room for n entries; uses ctx->scratch_scan
int scan_exclusive(dem_ctx* ctx, int* data, int n, int* scratch, size_t scratch_ints) {
    const int nb = nblk(n, 1024);
    if (nb == 1) {
        k_scan_block<<<1, 1024, 0, ctx->stream>>>(data, n, nullptr);
        LAUNCHED(ctx);
        return DEM_OK;
    }
    if ((size_t)nb > scratch_ints) return fail(ctx, DEM_EINVAL, "scan scratch too small");
    k_scan_block<<<nb, 1024, 0, ctx->stream>>>(data, n, scratch);
    LAUNCHED(ctx);
    CHECK(scan_exclusive(ctx, scratch, nb, scratch + ((nb + 3) & ~3), scratch_ints - ((nb + 3) & ~3)));
    k_scan_add<<<nb, 1024, 0, ctx->stream>>>(data, n, scratch);
    LAUNCHED(ctx);
    return DEM_OK;
}

template <typename real> int upload_table(dem_ctx* ctx) {
    typedef typename vec4<real>::type real4;
    std::vector<real4> host;
    ctx->shape_dev.clear();
    for (auto& S : ctx->shapes) {
        ShapeDev d;
        d.nv = S.nv; d.ne = S.ne; d.nf = S.nf; d.nfe = S.nfe;
        d.off = (int)host.size();
        d.len = S.table_len4();
        for (int g = 0; g < DEM_MAX_FACE_GROUPS; ++g) d.grp_m[g] = d.grp_n[g] = 0;
        if ((int)S.face_groups.size() <= DEM_MAX_FACE_GROUPS)
            for (size_t g = 0; g < S.face_groups.size(); ++g) {
                d.grp_m[g] = S.face_groups[g].first;
                d.grp_n[g] = S.face_groups[g].second;
            }
        for (int k = 0; k < d.len; ++k) {
            real4 v;
            v.x = (real)S.table[4 * k]; v.y = (real)S.table[4 * k + 1];
            v.z = (real)S.table[4 * k + 2]; v.w = (real)S.table[4 * k + 3];
            host.push_back(v);
        }
        ctx->shape_dev.push_back(d);
    }
    CU(ctx->table.reserve(host.size() * sizeof(real4)));
    CU(cudaMemcpyAsync(ctx->table.p, host.data(), host.size() * sizeof(real4), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));  // `host` goes out of scope
    return DEM_OK;
}

int sync_tables(dem_ctx* ctx) {
    if (!ctx->table_dirty) return DEM_OK;
    if (ctx->shapes.empty()) return fail(ctx, DEM_EINVAL, "no shapes registered");
    CHECK(ctx->prec == DEM_F64 ? upload_table<double>(ctx) : upload_table<float>(ctx));
    const int ns = (int)ctx->shapes.size();
    int c = 0;
    memset(&ctx->ct, 0, sizeof ctx->ct);
    for (int a = 0; a < ns; ++a)
        for (int b = a; b < ns; ++b) {
            ctx->ct.lut[a][b] = ctx->ct.lut[b][a] = (signed char)c;
            ctx->class_sa[c] = a;
            ctx->class_sb[c] = b;
            ++c;
        }
    ctx->nclass = c;
    for (int s = 0; s < ns; ++s) {
        ctx->mt.mass[s] = ctx->shapes[s].mass;
        for (int a = 0; a < 3; ++a) ctx->mt.inertia[s][a] = ctx->shapes[s].inertia[a];
    }
    cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, 0);
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, dev);
    ctx->table_dirty = false;
    return DEM_OK;
}

// ---- neighbour build ----------------------------------------------------------------------------------------------
template <typename PosT>
int build_neighbors_t(dem_ctx* ctx, const PosT* pos, const int32_t* sid, int N, const double box[3], double r_cut,
                      bool check_rcut) {
    if (N < 1) return fail(ctx, DEM_EINVAL, "N must be >= 1");
    if (!pos || !sid) return fail(ctx, DEM_EINVAL, "null particle array");
    if (!(r_cut > 0)) return fail(ctx, DEM_EINVAL, "r_cut must be positive");
    CHECK(sync_tables(ctx));
    for (int a = 0; a < ctx->dim; ++a)
        if (!(box[a] >= 2.0 * r_cut))
            return fail(ctx, DEM_EBOX, "box edge %d = %g < 2 r_cut = %g: minimum image invalid", a, box[a], 2 * r_cut);
    if (check_rcut && r_cut < max_reach(ctx) * (1.0 - 1e-12))
        return fail(ctx, DEM_ERCUT, "r_cut = %.17g < interaction reach %.17g", r_cut, max_reach(ctx));
    cudaStream_t st = ctx->stream;
    cudaEvent_t b0 = ev_mark(ctx, 2);
    ctx->have_list = false;
    ctx->N = N;
    for (int a = 0; a < 3; ++a) ctx->box[a] = box[a];
    ctx->r_cut = r_cut;
    const BoxDev bx = box_dev(ctx->dim, box);
    // cells at least r_cut wide (with a relative margin far above double rounding), at most ~2 N + 64 cells in all
    GridDev g;
    g.nc[0] = g.nc[1] = g.nc[2] = 1;
    for (int a = 0; a < ctx->dim; ++a) g.nc[a] = std::max(1, (int)std::floor(box[a] / (r_cut * (1.0 + 1e-9))));
    while ((double)g.nc[0] * g.nc[1] * g.nc[2] > 2.0 * N + 64.0) {
        int amax = 0;
        for (int a = 1; a < ctx->dim; ++a)
            if (g.nc[a] > g.nc[amax]) amax = a;
        if (g.nc[amax] <= 3) break;
        g.nc[amax] = std::max(3, (int)(g.nc[amax] * 0.8));
    }
    g.ncell = g.nc[0] * g.nc[1] * g.nc[2];
    ctx->grid = g;
    const size_t scan_ints = 4096 + (size_t)std::max<long long>(g.ncell, (long long)ctx->nclass * N) / 512;
    CU(ctx->cell_of.reserve(sizeof(int) * (size_t)N));
    CU(ctx->rank.reserve(sizeof(int) * (size_t)N));
    CU(ctx->order.reserve(sizeof(int) * (size_t)N));
    CU(ctx->cell_start.reserve(sizeof(int) * ((size_t)g.ncell + 1)));
    CU(ctx->xs.reserve(sizeof(d4) * (size_t)N));
    CU(ctx->counts.reserve(sizeof(int) * (size_t)N));
    CU(ctx->scratch_scan.reserve(sizeof(int) * scan_ints));
    CU(ctx->flags.reserve(sizeof(int) * 16));
    CU(ctx->counters.reserve(sizeof(unsigned long long) * 8 + sizeof(int) * 2 * DEM_MAX_CLASSES));
    CU(ctx->pos_build.reserve(sizeof(d4) * (size_t)N));
    int* cell_start = ctx->cell_start.as<int>();
    CU(cudaMemsetAsync(cell_start, 0, sizeof(int) * ((size_t)g.ncell + 1), st));
    const int B = 256;
    k_bin<PosT><<<nblk(N, B), B, 0, st>>>(pos, N, bx, g, ctx->cell_of.as<int>(), cell_start, ctx->rank.as<int>());
    LAUNCHED(ctx);
    CHECK(scan_exclusive(ctx, cell_start, g.ncell + 1, ctx->scratch_scan.as<int>(), scan_ints));
    k_place<<<nblk(N, B), B, 0, st>>>(N, ctx->cell_of.as<int>(), ctx->rank.as<int>(), cell_start, ctx->order.as<int>());
    LAUNCHED(ctx);
    k_sort_cells<<<nblk(g.ncell, B), B, 0, st>>>(g.ncell, cell_start, ctx->order.as<int>());
    LAUNCHED(ctx);
    k_gather_sorted<PosT><<<nblk(N, B), B, 0, st>>>(pos, N, ctx->order.as<int>(), ctx->xs.as<d4>());
    LAUNCHED(ctx);
    // positions of this build, in original order, for dem_step's displacement test
    if (sizeof(PosT) == sizeof(double)) {
        CU(cudaMemcpyAsync(ctx->pos_build.p, pos, sizeof(d4) * (size_t)N, cudaMemcpyDeviceToDevice, st));
    } else {
        k_f4_to_d4<<<nblk(N, B), B, 0, st>>>(N, reinterpret_cast<const f4*>(pos), ctx->pos_build.as<d4>());
        LAUNCHED(ctx);
    }
    int* flags = ctx->flags.as<int>();
    for (int attempt = 0; attempt < 8; ++attempt) {
        CU(ctx->list.reserve(sizeof(int) * (size_t)N * ctx->stride));
        CU(ctx->slot.reserve(sizeof(int) * (size_t)N * ctx->stride));
        CU(cudaMemsetAsync(flags, 0, sizeof(int) * 16, st));
        cudaEvent_t n0 = ev_mark(ctx, 2);
        k_neigh<<<nblk(N, 128), 128, 0, st>>>(N, bx, g, r_cut * r_cut, ctx->order.as<int>(), ctx->cell_of.as<int>(),
                                              cell_start, ctx->xs.as<d4>(), ctx->stride, ctx->counts.as<int>(),
                                              ctx->list.as<int>(), flags);
        LAUNCHED(ctx);
        ev_span(ctx, KT_NEIGH, n0, ev_mark(ctx, 2));
        int mc = 0;
        CU(cudaMemcpyAsync(&mc, flags, sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        ctx->max_count = mc;
        if (mc <= ctx->stride) break;
        if (attempt == 7) return fail(ctx, DEM_EOVERFLOW, "neighbour capacity could not be regrown (max count %d)", mc);
        ctx->stride = (mc + 7) & ~7;
    }
    // unique-pair work list, class-major
    const int nc = ctx->nclass;
    CU(ctx->pcnt.reserve(sizeof(int) * ((size_t)nc * N + 1)));
    int* pcnt = ctx->pcnt.as<int>();
    CU(cudaMemsetAsync(pcnt + (size_t)nc * N, 0, sizeof(int), st));
    k_pair_count<<<nblk(N, B), B, 0, st>>>(N, ctx->counts.as<int>(), ctx->list.as<int>(), ctx->stride, sid, ctx->ct, nc,
                                           (int)ctx->shapes.size(), pcnt, flags + 1);
    LAUNCHED(ctx);
    CHECK(scan_exclusive(ctx, pcnt, nc * N + 1, ctx->scratch_scan.as<int>(), scan_ints));
    int bases[DEM_MAX_CLASSES + 1];
    for (int c = 0; c <= nc; ++c)
        CU(cudaMemcpyAsync(&bases[c], pcnt + (size_t)c * N, sizeof(int), cudaMemcpyDeviceToHost, st));
    int bad_shape = 0;
    CU(cudaMemcpyAsync(&bad_shape, flags + 1, sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (bad_shape) return fail(ctx, DEM_EINVAL, "shape_id holds an id outside the %d registered shapes", (int)ctx->shapes.size());
    ctx->npairs_total = bases[nc];
    long long nrec = 0, terms = 0;
    for (int c = 0; c < nc; ++c) {
        ctx->class_np[c] = bases[c + 1] - bases[c];
        ctx->ct.pair_base[c] = bases[c];
        // slices: split a pair's outer feature loop over several lanes when there are too few pairs to fill the GPU
        int S = 1;
        const int outer = class_outer(ctx, c);
        if (ctx->force_slices > 0) {
            S = std::min(ctx->force_slices, std::max(outer, 1));
        } else if (ctx->class_np[c] > 0) {
            const long long want_lanes = (long long)ctx->sm_count * 2048;  // one full wave of resident threads
            const long long per_slice_min_terms = 64;                      // keep the per-lane setup amortised
            long long s = want_lanes / std::max(1, ctx->class_np[c]);
            s = std::min<long long>(s, class_terms(ctx, c) / per_slice_min_terms);
            s = std::min<long long>(s, outer);
            S = (int)std::max<long long>(1, s);
        }
        ctx->ct.slices[c] = S;
        ctx->ct.rec_base[c] = (int)nrec;
        nrec += (long long)ctx->class_np[c] * S;
        terms += (long long)ctx->class_np[c] * class_terms(ctx, c);
    }
    ctx->ct.pair_base[nc] = bases[nc];
    ctx->ct.rec_base[nc] = (int)nrec;
    ctx->nrec_total = nrec;
    ctx->last_terms = terms;
    if (nrec * DEM_REC > 0x7fffffffLL) return fail(ctx, DEM_EOVERFLOW, "too many pair records");
    CU(ctx->pairs.reserve(sizeof(int2) * (size_t)std::max<long long>(ctx->npairs_total, 1)));
    CU(ctx->rec.reserve((ctx->prec == DEM_F64 ? sizeof(d4) : sizeof(f4)) * DEM_REC * (size_t)std::max<long long>(nrec, 1)));
    CU(ctx->rflag.reserve((size_t)std::max<long long>(nrec, 1)));
    k_pair_fill<<<nblk(N, B), B, 0, st>>>(N, ctx->counts.as<int>(), ctx->list.as<int>(), ctx->stride, sid, ctx->ct, nc,
                                          pcnt, ctx->pairs.as<int2>(), ctx->slot.as<int>());
    LAUNCHED(ctx);
    k_slot_back<<<nblk(N, B), B, 0, st>>>(N, ctx->counts.as<int>(), ctx->list.as<int>(), ctx->stride, sid, ctx->ct, pcnt,
                                          ctx->slot.as<int>());
    LAUNCHED(ctx);
    CU(cudaGetLastError());
    ev_span(ctx, KT_BUILD, b0, ev_mark(ctx, 2));
    ctx->have_list = true;
    return DEM_OK;
}

struct NvtArgs {  // dem_step_nvt: target temperature, thermostat period, (xi, eta) in and out (host)
    double kT, tau;
    double* thermo;
};

template <typename real> int step_t(dem_ctx* ctx, void* pos, void* quat, void* vel, void* ang, const int32_t* sid,
                                    int N, const double box[3], double dt, int nsteps, double skin, void* force_out,
                                    void* torque_out, const NvtArgs* nvt = nullptr) {
    typedef typename vec4<real>::type real4;
    if (N < 1 || !pos || !quat || !vel || !ang || !sid) return fail(ctx, DEM_EINVAL, "bad particle arrays");
    if (nsteps < 0 || !(skin >= 0)) return fail(ctx, DEM_EINVAL, "bad nsteps / skin");
    CHECK(sync_tables(ctx));
    cudaStream_t st = ctx->stream;
    const int B = 256;
    const bool conv = ctx->prec == DEM_F32;
    d4 *x, *q, *v, *L;
    bool resumed = false;
    if (conv) {  // R15b: a DEM_F32 context integrates its state in double
        // Handed back the very arrays the last call returned (same pointers, same contents)?  Then the internal double
        // state, the neighbour list and the forces are still those of that state: go on from them.
        dem_ctx::Resume& rs = ctx->resume;
        if (rs.valid && rs.pos == pos && rs.quat == quat && rs.vel == vel && rs.ang == ang &&
            rs.sid == sid && rs.N == N && rs.skin == skin && rs.box[0] == box[0] && rs.box[1] == box[1] &&
            rs.box[2] == box[2] && ctx->have_list && ctx->N == N) {
            if (ctx->ev_copy_pending) {  // dem_step_host: the comparison reads all four arrays, so wait for the side copy
                CU(cudaStreamWaitEvent(st, ctx->ev_copy, 0));
                ctx->ev_copy_pending = false;
            }
            int* differ = ctx->flags.as<int>() + 12;
            CU(cudaMemsetAsync(differ, 0, sizeof(int), st));
            k_same_state<<<nblk(N, B), B, 0, st>>>(N, static_cast<const f4*>(pos), static_cast<const f4*>(quat),
                                                   static_cast<const f4*>(vel), static_cast<const f4*>(ang), sid,
                                                   (rs.cur ? ctx->st_pos2 : ctx->st_pos).as<d4>(),
                                                   (rs.cur ? ctx->st_quat2 : ctx->st_quat).as<d4>(), ctx->st_vel.as<d4>(),
                                                   ctx->st_ang.as<d4>(), ctx->sid_copy.as<int>(), differ);
            LAUNCHED(ctx);
            int h = 1;
            CU(cudaMemcpyAsync(&h, differ, sizeof(int), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            resumed = h == 0;
        }
        rs.valid = false;  // until this call returns
        CU(ctx->st_pos.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_quat.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_vel.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_ang.reserve(sizeof(d4) * (size_t)N));
        x = ctx->st_pos.as<d4>(); q = ctx->st_quat.as<d4>(); v = ctx->st_vel.as<d4>(); L = ctx->st_ang.as<d4>();
        const void* in[4] = {pos, quat, vel, ang};
        d4* out[4] = {x, q, v, L};
        for (int k = 0; k < 2 && !resumed; ++k) {  // velocities and angular momenta follow the first evaluation (see below)
            k_f4_to_d4<<<nblk(N, B), B, 0, st>>>(N, static_cast<const f4*>(in[k]), out[k]);
            LAUNCHED(ctx);
        }
    } else {
        x = static_cast<d4*>(pos); q = static_cast<d4*>(quat); v = static_cast<d4*>(vel); L = static_cast<d4*>(ang);
    }
    // the 2D per-particle kernel drifts into a second pair of position / orientation buffers (other warps still read
    // the old state): xs[cur] / qs[cur] hold the current state
    d4 *xs[2] = {x, x}, *qs[2] = {q, q};
    int cur = 0;
    if (conv && ctx->dim == 2 && ctx->particle2d) {
        CU(ctx->st_pos2.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_quat2.reserve(sizeof(d4) * (size_t)N));
        xs[1] = ctx->st_pos2.as<d4>();
        qs[1] = ctx->st_quat2.as<d4>();
        if (resumed) cur = ctx->resume.cur;
    }
    CU(ctx->st_force.reserve(sizeof(real4) * (size_t)N));
    CU(ctx->st_torque.reserve(sizeof(real4) * (size_t)N));
    real4* F = ctx->st_force.as<real4>();
    real4* T = ctx->st_torque.as<real4>();
    const double r_list = max_reach(ctx) + skin;
    const BoxDev bx = box_dev(ctx->dim, box);
    bool list_kept = false;
    if (!resumed) {
        // A list that an earlier dem_step built with the same cutoff, box and shape ids is still good if no particle is
        // farther than skin/2 from where it was at that build (the step loop's own criterion): callers that change
        // velocities, or hand in new host buffers every call (dem_step_host), then skip the build (0.3 ms on config 4).
        if (ctx->have_list && ctx->list_from_step && ctx->N == N && ctx->r_cut == r_list && ctx->box[0] == box[0] &&
            ctx->box[1] == box[1] && ctx->box[2] == box[2] && ctx->sid_copy.p) {
            int* stale = ctx->flags.as<int>() + 13;
            CU(cudaMemsetAsync(stale, 0, sizeof(int), st));
            k_list_valid<<<nblk(N, B), B, 0, st>>>(N, bx, x, ctx->pos_build.as<d4>(), sid, ctx->sid_copy.as<int>(),
                                                   0.25 * skin * skin, stale);
            LAUNCHED(ctx);
            int h = 1;
            CU(cudaMemcpyAsync(&h, stale, sizeof(int), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            list_kept = h == 0;
        }
        if (!list_kept) {
            CHECK(build_neighbors_t<double>(ctx, reinterpret_cast<const double*>(x), sid, N, box, r_list, false));
            ctx->list_from_step = true;
            CU(ctx->sid_copy.reserve(sizeof(int) * (size_t)N));
            CU(cudaMemcpyAsync(ctx->sid_copy.p, sid, sizeof(int) * (size_t)N, cudaMemcpyDeviceToDevice, st));
        }
        CHECK(evaluate(ctx, x, q, true, sid, N, F, T, nullptr, nullptr));
    }
    // The list build and the first evaluation need positions and orientations only: dem_step_host copies velocities
    // and angular momenta on a second stream meanwhile, and they are waited for (and converted) here.
    if (ctx->ev_copy_pending) {
        CU(cudaStreamWaitEvent(st, ctx->ev_copy, 0));
        ctx->ev_copy_pending = false;
    }
    if (conv && !resumed) {
        k_f4_to_d4<<<nblk(N, B), B, 0, st>>>(N, static_cast<const f4*>(vel), v);
        LAUNCHED(ctx);
        k_f4_to_d4<<<nblk(N, B), B, 0, st>>>(N, static_cast<const f4*>(ang), L);
        LAUNCHED(ctx);
    }
    // NVT (R19): k_kinetic + k_thermostat after every completed step advance (xi, eta) by the half step that
    // ends it and the half step that begins the next one; the scaling of v and L is applied by the next k_kick_drift.
    ThermoDev* th = nullptr;
    const int nbk = nblk(N, 256);
    auto thermostat = [&](int halves, const int* bail) -> int {
        k_kinetic<<<nbk, 256, 0, st>>>(N, ctx->dim, sid, ctx->mt, qs[cur], v, L, ctx->epart.as<double>());
        LAUNCHED(ctx);
        k_thermostat<<<1, 256, 0, st>>>(nbk, ctx->epart.as<double>(), ctx->dim, N, dt, nvt->kT, nvt->tau, halves, bail, th);
        LAUNCHED(ctx);
        return DEM_OK;
    };
    if (nvt && nsteps > 0) {
        CU(ctx->thermo.reserve(sizeof(ThermoDev)));
        CU(ctx->epart.reserve(sizeof(double) * 3 * (size_t)nbk));
        th = ctx->thermo.as<ThermoDev>();
        const ThermoDev h0 = {nvt->thermo[0], nvt->thermo[1], 1.0, 0.0};
        CU(cudaMemcpyAsync(th, &h0, sizeof h0, cudaMemcpyHostToDevice, st));
        CU(cudaStreamSynchronize(st));  // h0 is on the stack
        CHECK(thermostat(1, nullptr));
    }
    // Steps are queued in chunks without the host in between.  The kernel that ends an evaluation (k_finish) also
    // integrates: second half kick, which completes the step, and -- unless the step is the last of the call or a
    // thermostat has to act in between -- the first half kick, drift and rotation of the NEXT step.  Whoever drifts
    // raises a device flag when a particle leaves its skin (the list is stale); flags[0] and flags[1] are used
    // alternately: evaluation e of a chunk and everything behind it do nothing when flags[e & 1] is set (raised
    // BEFORE they started), and the drift behind evaluation e raises flags[(e + 1) & 1].  flags[2] counts the steps
    // completed.  The host reads the three once per chunk; a chunk that went stale stopped after a drift, with the
    // forces of the drifted state not yet evaluated, which is exactly the state every chunk starts from: the host
    // rebuilds the list and goes on.  The chunk length follows the last observed interval between rebuilds, so that
    // few launches are wasted behind a stale flag.
    int* flags = ctx->flags.as<int>() + 8;
    const double half_skin2 = 0.25 * skin * skin;
    if (ctx->l2_flush_bytes) CU(ctx->l2_scratch.reserve(ctx->l2_flush_bytes));
    if (!ctx->h_moved) CU(cudaHostAlloc(&ctx->h_moved, 4 * sizeof(int), cudaHostAllocDefault));
    FinArgs fa;
    memset(&fa, 0, sizeof fa);
    fa.dim = ctx->dim;
    fa.dt = dt;
    fa.vel = v; fa.ang = L;
    fa.pos_build = ctx->pos_build.as<d4>();
    fa.half_skin2 = half_skin2;
    fa.box = bx;
    fa.mt = ctx->mt;
    fa.done = flags + 2;
    auto kick_drift = [&](const int* bail, int* raise) {
        cudaEvent_t k0 = ev_mark(ctx, 2);
        k_kick_drift<real><<<2 * nblk(N, B), B, 0, st>>>(N, bx, dt, sid, ctx->mt, xs[cur], qs[cur], v, L, F, T,
                                                     ctx->pos_build.as<d4>(), half_skin2, bail, raise, th);
        LAUNCHED(ctx);
        ev_span(ctx, KT_KICK_DRIFT, k0, ev_mark(ctx, 2));
    };
    int remaining = nsteps, since = (resumed || list_kept) ? ctx->steps_since_build : 0;
    bool drifted = false;  // the state is past the drift of the next step (forces of the drifted state not yet evaluated)
    while (remaining > 0) {
        // up to the predicted number of steps until the next rebuild (at least 8); past the prediction, 16 at a time: a step
        // queued behind a stale flag costs three empty launches, a chunk boundary a host round trip
        const int predicted = std::max(ctx->rebuild_interval, 1) - since;
        const int chunk = std::min(remaining, predicted > 0 ? std::min(64, std::max(predicted, 8)) : 16);
        CU(cudaMemsetAsync(flags, 0, 3 * sizeof(int), st));
        if (!drifted) {  // the first half of the call's first step
            kick_drift(nullptr, flags);
            drifted = true;
        }
        const bool pingpong = xs[1] != xs[0] && particle2d_applies(ctx);
        int c = cur, swaps = 0;  // buffer the queued evaluations read, and how many of them drift into the other one
        for (int e = 0; e < chunk; ++e) {
            if (ctx->l2_flush_bytes) {
                cudaEvent_t f0 = ev_mark(ctx, 2);
                CU(cudaMemsetAsync(ctx->l2_scratch.p, e & 0xff, ctx->l2_flush_bytes, st));
                ev_span(ctx, KT_FLUSH, f0, ev_mark(ctx, 2));
            }
            const bool last = e == remaining - 1;  // the last step of the call ends with its second half kick
            fa.mode = (last || th) ? 1 : 2;
            fa.bail = flags + (e & 1);
            fa.raise = flags + ((e + 1) & 1);
            const int out = pingpong && fa.mode == 2 ? c ^ 1 : c;
            fa.pos = xs[out];
            fa.quat = qs[out];
            if (last && !th && ctx->early_host[0] && ctx->copy_stream) {
                // the state this evaluation reads is the final one: send x and q on their way now
                if (!ctx->ev_early) CU(cudaEventCreateWithFlags(&ctx->ev_early, cudaEventDisableTiming));
                const size_t r4b = conv ? sizeof(f4) : sizeof(d4);
                if (conv) {
                    k_d4_to_f4<<<nblk(N, B), B, 0, st>>>(N, xs[c], static_cast<f4*>(pos));
                    LAUNCHED(ctx);
                    k_d4_to_f4<<<nblk(N, B), B, 0, st>>>(N, qs[c], static_cast<f4*>(quat));
                    LAUNCHED(ctx);
                }
                CU(cudaEventRecord(ctx->ev_early, st));
                CU(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_early, 0));
                CU(cudaMemcpyAsync(ctx->early_host[0], conv ? pos : (void*)xs[c], r4b * N, cudaMemcpyDeviceToHost, ctx->copy_stream));
                CU(cudaMemcpyAsync(ctx->early_host[1], conv ? quat : (void*)qs[c], r4b * N, cudaMemcpyDeviceToHost, ctx->copy_stream));
                ctx->early_done = true;
            }
            CHECK(evaluate(ctx, xs[c], qs[c], true, sid, N, F, T, nullptr, &fa));
            if (out != c) ++swaps;
            c = out;
            if (th) {
                CHECK(thermostat(last ? 1 : 2, fa.bail));
                if (!last) kick_drift(fa.bail, fa.raise);
            }
        }
        CU(cudaMemcpyAsync(ctx->h_moved, flags, 3 * sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        const int done = ctx->h_moved[2];
        const bool stale = ctx->h_moved[0] || ctx->h_moved[1];
        if (done < 0 || done > chunk || (done < chunk && !stale))
            return fail(ctx, DEM_ECUDA, "dem_step: inconsistent step flags (done %d of %d, stale %d)", done, chunk, (int)stale);
        remaining -= done;
        cur ^= std::min(done, swaps) & 1;  // evaluations behind a stale flag did not run: the state stayed where it was
        if (stale && remaining > 0) {
            CHECK(build_neighbors_t<double>(ctx, reinterpret_cast<const double*>(xs[cur]), sid, N, box, r_list, false));
            ctx->rebuild_interval = since + done + 1;
            since = 0;
        } else {
            since += done;
        }
    }
    if (th) {
        k_scale_momenta<<<nblk(N, B), B, 0, st>>>(N, v, L, th);
        LAUNCHED(ctx);
    }
    if (conv) {
        void* out[4] = {pos, quat, vel, ang};
        d4* in[4] = {xs[cur], qs[cur], v, L};
        for (int k = ctx->early_done ? 2 : 0; k < 4; ++k) {  // (x and q may be converted and on their way already)
            k_d4_to_f4<<<nblk(N, B), B, 0, st>>>(N, in[k], static_cast<f4*>(out[k]));
            LAUNCHED(ctx);
        }
    }
    if (force_out) CU(cudaMemcpyAsync(force_out, F, sizeof(real4) * (size_t)N, cudaMemcpyDeviceToDevice, st));
    if (torque_out) CU(cudaMemcpyAsync(torque_out, T, sizeof(real4) * (size_t)N, cudaMemcpyDeviceToDevice, st));
    ThermoDev h1;
    if (th) CU(cudaMemcpyAsync(&h1, th, sizeof h1, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (th) {
        nvt->thermo[0] = h1.xi;
        nvt->thermo[1] = h1.eta;
        ctx->nvt_dof = h1.dof;
    }
    ctx->steps_since_build = since;
    if (conv) {  // what a next call must find unchanged to go on from here (sid_copy: the ids of the last build)
        dem_ctx::Resume& rs = ctx->resume;
        rs.pos = pos; rs.quat = quat; rs.vel = vel; rs.ang = ang; rs.sid = sid;
        rs.N = N; rs.cur = cur; rs.skin = skin;
        for (int a = 0; a < 3; ++a) rs.box[a] = box[a];
        rs.valid = true;
    }
    // the internal list was built from internal (double) positions; a later dem_compute on caller arrays is still valid
    return DEM_OK;
}

// ---- NPT (R22) ------------------------------------------------------------------------------------------------
// Host-driven, one step at a time: the box is a launch argument of the kernels, and the scalar equations of the
// thermostat and the barostat need the sums K_trans, K_rot, tr W of the step before.  Order of a step (h = dt/2):
// T(h) B(h) K(h) D(dt) forces K(h) B(h) T(h)  (include/dem.h: dem_step_npt).
struct NptArgs {
    double kT, tau, pressure, tau_p;
    double* state;  // xi, eta, nu (host, in and out)
    double* box;    // host, in and out
};

template <typename real> int step_npt_t(dem_ctx* ctx, void* pos, void* quat, void* vel, void* ang, const int32_t* sid,
                                        int N, double dt, int nsteps, double skin, void* force_out, void* torque_out,
                                        const NptArgs& npt) {
    typedef typename vec4<real>::type real4;
    if (N < 2 || !pos || !quat || !vel || !ang || !sid) return fail(ctx, DEM_EINVAL, "bad particle arrays");
    if (nsteps < 0 || !(skin >= 0)) return fail(ctx, DEM_EINVAL, "bad nsteps / skin");
    ctx->resume.valid = false;  // this path shares dem_step's internal state and moves the box
    ctx->list_from_step = false;  // (its lists are valid up to an affine map of the build positions only)
    CHECK(sync_tables(ctx));
    cudaStream_t st = ctx->stream;
    const int B = 256, dim = ctx->dim;
    const bool conv = ctx->prec == DEM_F32;
    d4 *x, *q, *v, *L;
    if (conv) {  // R15b: a DEM_F32 context integrates its state in double
        CU(ctx->st_pos.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_quat.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_vel.reserve(sizeof(d4) * (size_t)N));
        CU(ctx->st_ang.reserve(sizeof(d4) * (size_t)N));
        x = ctx->st_pos.as<d4>(); q = ctx->st_quat.as<d4>(); v = ctx->st_vel.as<d4>(); L = ctx->st_ang.as<d4>();
        const void* in[4] = {pos, quat, vel, ang};
        d4* out[4] = {x, q, v, L};
        for (int k = 0; k < 4; ++k) {
            k_f4_to_d4<<<nblk(N, B), B, 0, st>>>(N, static_cast<const f4*>(in[k]), out[k]);
            LAUNCHED(ctx);
        }
    } else {
        x = static_cast<d4*>(pos); q = static_cast<d4*>(quat); v = static_cast<d4*>(vel); L = static_cast<d4*>(ang);
    }
    CU(ctx->st_force.reserve(sizeof(real4) * (size_t)N));
    CU(ctx->st_torque.reserve(sizeof(real4) * (size_t)N));
    CU(ctx->st_virial.reserve(sizeof(real) * 6 * (size_t)N));
    real4* F = ctx->st_force.as<real4>();
    real4* T = ctx->st_torque.as<real4>();
    real* W = ctx->st_virial.as<real>();
    const int nbk = nblk(N, 256);
    CU(ctx->epart.reserve(sizeof(double) * 4 * (size_t)nbk));
    std::vector<double> part(4 * (size_t)nbk);
    double box[3] = {npt.box[0], npt.box[1], npt.box[2]};
    const double reach = max_reach(ctx), r_list = reach + skin;
    double box_build = box[0];  // the list's box edge along x: lambda = box[0] / box_build (the scaling is isotropic)
    double Kt = 0, Kr = 0, dofr = 0, trW = 0;
    // forces, virial and the sums of the current state
    auto forces = [&]() -> int {
        for (int a = 0; a < 3; ++a) ctx->box[a] = box[a];  // the list stays; the minimum image uses the current box
        return evaluate(ctx, x, q, true, sid, N, F, T, W, nullptr);
    };
    auto sums = [&]() -> int {
        k_npt_sums<real><<<nbk, 256, 0, st>>>(N, dim, sid, ctx->mt, q, v, L, W, ctx->epart.as<double>());
        LAUNCHED(ctx);
        CU(cudaMemcpyAsync(part.data(), ctx->epart.p, sizeof(double) * part.size(), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        Kt = Kr = dofr = trW = 0;
        for (int b = 0; b < nbk; ++b) {
            Kt += part[4 * (size_t)b];
            Kr += part[4 * (size_t)b + 1];
            dofr += part[4 * (size_t)b + 2];
            trW += part[4 * (size_t)b + 3];
        }
        return DEM_OK;
    };
    auto rebuild = [&]() -> int {
        CHECK(build_neighbors_t<double>(ctx, reinterpret_cast<const double*>(x), sid, N, box, r_list, false));
        box_build = box[0];
        return DEM_OK;
    };
    CHECK(rebuild());
    CHECK(forces());
    CHECK(sums());
    const double g = (double)dim * (N - 1) + dofr, Q = g * npt.kT * npt.tau * npt.tau;
    const double Nf = (double)dim * (N - 1), alpha = 1.0 + dim / Nf, Wb = (double)dim * N * npt.kT * npt.tau_p * npt.tau_p;
    double xi = npt.state[0], eta = npt.state[1], nu = npt.state[2], pend = 1.0;
    auto volume = [&]() { return dim == 3 ? box[0] * box[1] * box[2] : box[0] * box[1]; };
    auto thermo_half = [&]() {  // R19; the scaling of v and L stays pending in `pend`, K_trans and K_rot follow it
        xi += 0.25 * dt * (2.0 * (Kt + Kr) - g * npt.kT) / Q;
        const double s = std::exp(-xi * 0.5 * dt);
        pend *= s;
        Kt *= s * s;
        Kr *= s * s;
        eta += 0.5 * dt * xi;
        xi += 0.25 * dt * (2.0 * (Kt + Kr) - g * npt.kT) / Q;
    };
    auto baro_half = [&]() { nu += 0.5 * dt * (alpha * 2.0 * Kt + trW - dim * volume() * npt.pressure) / Wb; };
    int* flags = ctx->flags.as<int>() + 8;
    if (!ctx->h_moved) CU(cudaHostAlloc(&ctx->h_moved, 4 * sizeof(int), cudaHostAllocDefault));
    for (int step = 0; step < nsteps; ++step) {
        thermo_half();
        baro_half();
        const double s = std::exp(-alpha * nu * 0.25 * dt);
        const double z = 0.5 * nu * dt, ea = std::exp(nu * dt), eh = std::exp(z), sc = z == 0.0 ? 1.0 : std::sinh(z) / z;
        for (int a = 0; a < dim; ++a) box[a] *= ea;
        for (int a = 0; a < dim; ++a)
            if (!(box[a] >= 2.0 * reach))
                return fail(ctx, DEM_EBOX, "dem_step_npt: box edge %d shrank to %g < 2 x interaction reach %g", a, box[a], reach);
        const double lambda = box[0] / box_build;
        const double slack = 0.5 * (lambda * r_list - reach);
        const BoxDev bx = box_dev(dim, box);
        CU(cudaMemsetAsync(flags, 0, sizeof(int), st));
        k_npt_kick_drift<real><<<nblk(N, B), B, 0, st>>>(N, bx, dt, sid, ctx->mt, x, q, v, L, F, T, ctx->pos_build.as<d4>(),
                                                        lambda, slack > 0 ? slack * slack : -1.0, flags, pend, s, ea,
                                                        dt * eh * sc);
        LAUNCHED(ctx);
        pend = 1.0;
        CU(cudaMemcpyAsync(ctx->h_moved, flags, sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        // the list also has to follow the box: its cells must stay at least r_list wide for the next build only, but a
        // box that no longer holds two cutoffs is refused by the build itself
        if (ctx->h_moved[0]) CHECK(rebuild());
        CHECK(forces());
        k_npt_kick<real><<<nblk(N, B), B, 0, st>>>(N, dim, dt, sid, ctx->mt, v, L, F, T, s);
        LAUNCHED(ctx);
        CHECK(sums());
        baro_half();
        thermo_half();
    }
    if (pend != 1.0) {
        k_scale_momenta_by<<<nblk(N, B), B, 0, st>>>(N, v, L, pend);
        LAUNCHED(ctx);
    }
    if (conv) {
        void* out[4] = {pos, quat, vel, ang};
        d4* in[4] = {x, q, v, L};
        for (int k = ctx->early_done ? 2 : 0; k < 4; ++k) {  // (x and q may be converted and on their way already)
            k_d4_to_f4<<<nblk(N, B), B, 0, st>>>(N, in[k], static_cast<f4*>(out[k]));
            LAUNCHED(ctx);
        }
    }
    if (force_out) CU(cudaMemcpyAsync(force_out, F, sizeof(real4) * (size_t)N, cudaMemcpyDeviceToDevice, st));
    if (torque_out) CU(cudaMemcpyAsync(torque_out, T, sizeof(real4) * (size_t)N, cudaMemcpyDeviceToDevice, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    npt.state[0] = xi; npt.state[1] = eta; npt.state[2] = nu;
    for (int a = 0; a < 3; ++a) npt.box[a] = box[a];
    ctx->nvt_dof = g;
    return DEM_OK;
}

template <typename real, typename PosT>
int energy_t(dem_ctx* ctx, const PosT* quat, const PosT* vel, const PosT* ang, const int32_t* sid, const void* force,
             int N, double out[3]) {
    typedef typename vec4<real>::type real4;
    CHECK(sync_tables(ctx));
    const int nb = nblk(N, 256);
    CU(ctx->epart.reserve(sizeof(double) * 3 * (size_t)nb));
    k_energy<real, PosT><<<nb, 256, 0, ctx->stream>>>(N, ctx->dim, sid, ctx->mt, quat, vel, ang,
                                                     static_cast<const real4*>(force), ctx->epart.as<double>());
    LAUNCHED(ctx);
    std::vector<double> h(3 * (size_t)nb);
    CU(cudaMemcpyAsync(h.data(), ctx->epart.p, sizeof(double) * h.size(), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    out[0] = out[1] = out[2] = 0;
    for (int b = 0; b < nb; ++b)
        for (int a = 0; a < 3; ++a) out[a] += h[3 * (size_t)b + a];
    return DEM_OK;
}

}  // namespace

// =====================================================================================================================
extern "C" {

#ifndef DEM_SOURCE_HASH
#define DEM_SOURCE_HASH "unknown"
#endif
// the hash is that of the sources the library was built from (build.py); binding.lib() refuses a library that lags them
const char* dem_version(void) { return "dem_b200 0.2 (sm_100a) src " DEM_SOURCE_HASH; }

int dem_create(dem_ctx** out, int dim, double epsilon, int precision, void* cuda_stream) {
    if (!out) return DEM_EINVAL;
    *out = nullptr;
    if ((dim != 2 && dim != 3) || !(epsilon > 0) || (precision != DEM_F32 && precision != DEM_F64)) return DEM_EINVAL;
    dem_ctx* c = new (std::nothrow) dem_ctx;
    if (!c) return DEM_ENOMEM;
    c->dim = dim;
    c->eps = epsilon;
    c->prec = precision;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->particle2d = dim == 2;  // DEM_KERNEL_AUTO
    memset(&c->ct, 0, sizeof c->ct);
    memset(&c->mt, 0, sizeof c->mt);
    *out = c;
    return DEM_OK;
}

int dem_destroy(dem_ctx* c) {
    if (!c) return DEM_EINVAL;
    DevBuf* bufs[] = {&c->table, &c->cell_of, &c->rank, &c->cell_start, &c->order, &c->xs, &c->counts, &c->list, &c->slot,
                      &c->scratch_scan, &c->pcnt, &c->pairs, &c->rec, &c->rflag, &c->flags, &c->counters, &c->thermo, &c->pose, &c->pidx, &c->cmask, &c->cum, &c->st_pos, &c->st_quat,
                      &c->st_vel, &c->st_ang, &c->st_force, &c->st_torque, &c->st_virial, &c->st_pos2, &c->st_quat2, &c->sid_copy, &c->pos_build, &c->epart, &c->h_pos,
                      &c->h_quat, &c->h_vel, &c->h_ang, &c->h_sid, &c->h_force, &c->h_torque, &c->h_virial, &c->l2_scratch};
    for (DevBuf* b : bufs) b->release();
    if (c->h_moved) cudaFreeHost(c->h_moved);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->ev_copy) cudaEventDestroy(c->ev_copy);
    if (c->ev_early) cudaEventDestroy(c->ev_early);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    for (int k = 0; k < 3; ++k) {
        if (c->class_stream[k]) cudaStreamDestroy(c->class_stream[k]);
        if (c->ev_join[k]) cudaEventDestroy(c->ev_join[k]);
    }
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    delete c;
    return DEM_OK;
}

const char* dem_last_error(const dem_ctx* c) { return c ? c->err.c_str() : "null context"; }

int dem_set_eps_par(dem_ctx* ctx, double eps_par) {
    if (!ctx || !(eps_par >= 0)) return fail(ctx, DEM_EINVAL, "eps_par must be >= 0");
    ctx->eps_par = eps_par;
    ctx->resume.valid = false;  // the stored forces were evaluated with the old threshold
    return DEM_OK;
}

// Tuning / test hook: lanes per pair (0 = heuristic).  Takes effect at the next neighbour build.
int dem_set_slices(dem_ctx* ctx, int slices) {
    if (!ctx || slices < 0) return fail(ctx, DEM_EINVAL, "slices must be >= 0");
    ctx->force_slices = slices;
    ctx->have_list = false;
    ctx->resume.valid = false;
    return DEM_OK;
}

int dem_set_pair_kernel(dem_ctx* ctx, int which) {
    if (!ctx || (which != DEM_KERNEL_SEARCH && which != DEM_KERNEL_GENERIC && which != DEM_KERNEL_AUTO))
        return fail(ctx, DEM_EINVAL, "unknown pair kernel");
    ctx->generic_kernel = which == DEM_KERNEL_GENERIC;
    ctx->particle2d = which == DEM_KERNEL_AUTO && ctx->dim == 2;
    return DEM_OK;
}

int dem_set_culling(dem_ctx* ctx, int enabled) {
    if (!ctx) return DEM_EINVAL;
    ctx->cull = enabled != 0;
    return DEM_OK;
}

int dem_create_shape(dem_ctx* ctx, const double* verts, int nv, const int* face_offsets, const int* face_verts, int nf,
                     const int* edges, int ne, double rounding_radius, double mass, const double inertia[3],
                     int* shape_id) {
    if (!ctx) return DEM_EINVAL;
    if (!verts || !shape_id) return fail(ctx, DEM_EINVAL, "null argument");
    if ((int)ctx->shapes.size() >= DEM_MAX_SHAPES) return fail(ctx, DEM_EINVAL, "more than %d shapes", DEM_MAX_SHAPES);
    if (!(mass > 0)) return fail(ctx, DEM_EINVAL, "mass must be positive");
    HostShape S;
    const std::string e = build_host_shape(S, ctx->dim, verts, nv, face_offsets, face_verts, nf, edges, ne,
                                           rounding_radius, mass, inertia);
    if (!e.empty()) return fail(ctx, DEM_EINVAL, "%s", e.c_str());
    if (S.table_len4() * 32 > 100 * 1024) return fail(ctx, DEM_EINVAL, "shape too large for the shared-memory table");
    ctx->shapes.push_back(std::move(S));
    ctx->table_dirty = true;
    ctx->have_list = false;
    *shape_id = (int)ctx->shapes.size() - 1;
    return DEM_OK;
}

int dem_build_neighbors(dem_ctx* ctx, const void* pos, const int32_t* shape_id, int N, const double box[3], double r_cut) {
    if (!ctx) return DEM_EINVAL;
    if (!box) return fail(ctx, DEM_EINVAL, "null box");
    ctx->resume.valid = false;  // the caller's list replaces dem_step's
    ctx->list_from_step = false;
    if (ctx->prec == DEM_F64) return build_neighbors_t<double>(ctx, static_cast<const double*>(pos), shape_id, N, box, r_cut, true);
    return build_neighbors_t<float>(ctx, static_cast<const float*>(pos), shape_id, N, box, r_cut, true);
}

int dem_get_neighbors(dem_ctx* ctx, const int32_t** counts, const int32_t** list, int* stride, int* max_count) {
    if (!ctx) return DEM_EINVAL;
    if (!ctx->have_list) return fail(ctx, DEM_ESTALE, "no neighbour list");
    if (counts) *counts = ctx->counts.as<int32_t>();
    if (list) *list = ctx->list.as<int32_t>();
    if (stride) *stride = ctx->stride;
    if (max_count) *max_count = ctx->max_count;
    return DEM_OK;
}

int dem_copy_neighbors(dem_ctx* ctx, int32_t* counts_out, int32_t* list_out, int out_stride) {
    if (!ctx) return DEM_EINVAL;
    if (!ctx->have_list) return fail(ctx, DEM_ESTALE, "no neighbour list");
    if (!counts_out || !list_out || out_stride < ctx->max_count) return fail(ctx, DEM_EINVAL, "bad output arrays");
    CU(cudaMemcpyAsync(counts_out, ctx->counts.p, sizeof(int) * (size_t)ctx->N, cudaMemcpyDeviceToDevice, ctx->stream));
    k_copy_rows<<<nblk((long long)ctx->N * out_stride, 256), 256, 0, ctx->stream>>>(
        ctx->N, ctx->counts.as<int>(), ctx->list.as<int>(), ctx->stride, list_out, out_stride);
    LAUNCHED(ctx);
    CU(cudaGetLastError());
    return DEM_OK;
}

int dem_compute(dem_ctx* ctx, const void* pos, const void* quat, const int32_t* shape_id, int N, void* force_energy,
                void* torque, void* virial6) {
    if (!ctx) return DEM_EINVAL;
    return evaluate(ctx, pos, quat, ctx->prec == DEM_F64, shape_id, N, force_energy, torque, virial6, nullptr);
}

int dem_get_counters(dem_ctx* ctx, int64_t out[9]) {
    if (!ctx || !out) return DEM_EINVAL;
    if (!ctx->counters.p) return fail(ctx, DEM_ESTALE, "no evaluation yet");
    unsigned long long h[8];
    CU(cudaMemcpyAsync(h, ctx->counters.p, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    // terms evaluated = nominal terms of the evaluated pairs; with a single class this is exact, with several classes
    // pairs rejected by the reach test are attributed proportionally (the list is normally built at r_cut = reach)
    out[0] = (int64_t)h[0];
    out[1] = ctx->npairs_total > 0 ? (int64_t)((double)ctx->last_terms * ((double)h[0] / (double)ctx->npairs_total) + 0.5) : 0;
    out[2] = (int64_t)h[1];
    out[3] = (int64_t)h[2];
    out[4] = (int64_t)h[3];
    out[5] = ctx->npairs_total;
    // terms whose nearest-point search was executed (the search kernels count what they sweep; the generic kernel
    // sweeps every term of the pairs it evaluates)
    if (ctx->prec == DEM_F32 && (!ctx->generic_kernel || particle2d_applies(ctx))) {
        out[6] = (int64_t)(h[4] + h[5]);
        out[7] = (int64_t)h[4];
        out[8] = (int64_t)h[6];
    } else {
        const double f = ctx->npairs_total > 0 ? (double)h[0] / (double)ctx->npairs_total : 0.0;
        double ee = 0, vfe = 0;
        for (int c = 0; c < ctx->nclass; ++c) {
            const HostShape &A = ctx->shapes[ctx->class_sa[c]], &B = ctx->shapes[ctx->class_sb[c]];
            const double np = ctx->class_np[c];
            if (ctx->dim == 3) {
                ee += np * A.ne * B.ne;
                vfe += np * ((double)B.nv * A.nfe + (double)A.nv * B.nfe);
            } else {
                ee += np * ((double)B.nv * A.ne + (double)A.nv * B.ne);
            }
        }
        out[6] = out[1];
        out[7] = (int64_t)(ee * f + 0.5);
        out[8] = (int64_t)(vfe * f + 0.5);
    }
    return DEM_OK;
}

int dem_step(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N,
             const double box[3], double dt, int nsteps, double skin, void* force_energy, void* torque) {
    if (!ctx) return DEM_EINVAL;
    if (!box) return fail(ctx, DEM_EINVAL, "null box");
    if (ctx->prec == DEM_F64)
        return step_t<double>(ctx, pos, quat, vel, angmom, shape_id, N, box, dt, nsteps, skin, force_energy, torque);
    return step_t<float>(ctx, pos, quat, vel, angmom, shape_id, N, box, dt, nsteps, skin, force_energy, torque);
}

int dem_step_nvt(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N,
                 const double box[3], double dt, int nsteps, double skin, double kT, double tau, double thermostat[2],
                 double* dof, void* force_energy, void* torque) {
    if (!ctx) return DEM_EINVAL;
    if (!box || !thermostat) return fail(ctx, DEM_EINVAL, "null box / thermostat");
    if (!(kT > 0) || !(tau > 0)) return fail(ctx, DEM_EINVAL, "kT and tau must be > 0");
    if (N < 2) return fail(ctx, DEM_EINVAL, "the thermostat needs N >= 2");
    const NvtArgs nvt = {kT, tau, thermostat};
    int rc;
    if (ctx->prec == DEM_F64)
        rc = step_t<double>(ctx, pos, quat, vel, angmom, shape_id, N, box, dt, nsteps, skin, force_energy, torque, &nvt);
    else
        rc = step_t<float>(ctx, pos, quat, vel, angmom, shape_id, N, box, dt, nsteps, skin, force_energy, torque, &nvt);
    if (rc == DEM_OK && dof) *dof = ctx->nvt_dof;
    return rc;
}

int dem_step_npt(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N, double box[3],
                 double dt, int nsteps, double skin, double kT, double tau, double pressure, double tau_p, double state[3],
                 double* dof, void* force_energy, void* torque) {
    if (!ctx) return DEM_EINVAL;
    if (!box || !state) return fail(ctx, DEM_EINVAL, "null box / state");
    if (!(kT > 0) || !(tau > 0) || !(tau_p > 0)) return fail(ctx, DEM_EINVAL, "kT, tau and tau_p must be > 0");
    if (N < 2) return fail(ctx, DEM_EINVAL, "the thermostat needs N >= 2");
    const NptArgs npt = {kT, tau, pressure, tau_p, state, box};
    int rc;
    if (ctx->prec == DEM_F64)
        rc = step_npt_t<double>(ctx, pos, quat, vel, angmom, shape_id, N, dt, nsteps, skin, force_energy, torque, npt);
    else
        rc = step_npt_t<float>(ctx, pos, quat, vel, angmom, shape_id, N, dt, nsteps, skin, force_energy, torque, npt);
    if (rc == DEM_OK && dof) *dof = ctx->nvt_dof;
    return rc;
}

int dem_energy(dem_ctx* ctx, const void* quat, const void* vel, const void* angmom, const int32_t* shape_id,
               const void* force_energy, int N, double out[3]) {
    if (!ctx || !out) return DEM_EINVAL;
    if (!quat || !vel || !angmom || !shape_id || !force_energy || N < 1) return fail(ctx, DEM_EINVAL, "bad arguments");
    if (ctx->prec == DEM_F64)
        return energy_t<double, double>(ctx, static_cast<const double*>(quat), static_cast<const double*>(vel),
                                        static_cast<const double*>(angmom), shape_id, force_energy, N, out);
    return energy_t<float, float>(ctx, static_cast<const float*>(quat), static_cast<const float*>(vel),
                                  static_cast<const float*>(angmom), shape_id, force_energy, N, out);
}

int dem_compute_host(dem_ctx* ctx, const void* pos, const void* quat, const int32_t* shape_id, int N, const double box[3],
                     double r_cut, void* force_energy, void* torque, void* virial6) {
    if (!ctx) return DEM_EINVAL;
    if (!pos || !quat || !shape_id || !force_energy || !torque || !box || N < 1) return fail(ctx, DEM_EINVAL, "bad arguments");
    const size_t r4 = (ctx->prec == DEM_F64 ? sizeof(d4) : sizeof(f4)), rs = r4 / 4;
    cudaStream_t st = ctx->stream;
    CU(ctx->h_pos.reserve(r4 * N));
    CU(ctx->h_quat.reserve(r4 * N));
    CU(ctx->h_sid.reserve(sizeof(int32_t) * (size_t)N));
    CU(ctx->h_force.reserve(r4 * N));
    CU(ctx->h_torque.reserve(r4 * N));
    if (virial6) CU(ctx->h_virial.reserve(rs * 6 * N));
    CU(cudaMemcpyAsync(ctx->h_pos.p, pos, r4 * N, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(ctx->h_quat.p, quat, r4 * N, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(ctx->h_sid.p, shape_id, sizeof(int32_t) * (size_t)N, cudaMemcpyHostToDevice, st));
    CHECK(dem_build_neighbors(ctx, ctx->h_pos.p, ctx->h_sid.as<int32_t>(), N, box, r_cut));
    CHECK(dem_compute(ctx, ctx->h_pos.p, ctx->h_quat.p, ctx->h_sid.as<int32_t>(), N, ctx->h_force.p, ctx->h_torque.p,
                      virial6 ? ctx->h_virial.p : nullptr));
    CU(cudaMemcpyAsync(force_energy, ctx->h_force.p, r4 * N, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(torque, ctx->h_torque.p, r4 * N, cudaMemcpyDeviceToHost, st));
    if (virial6) CU(cudaMemcpyAsync(virial6, ctx->h_virial.p, rs * 6 * N, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return DEM_OK;
}

int dem_step_host(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N,
                  const double box[3], double dt, int nsteps, double skin, void* force_energy, void* torque) {
    if (!ctx) return DEM_EINVAL;
    if (!pos || !quat || !vel || !angmom || !shape_id || !box || N < 1) return fail(ctx, DEM_EINVAL, "bad arguments");
    const size_t r4 = (ctx->prec == DEM_F64 ? sizeof(d4) : sizeof(f4));
    cudaStream_t st = ctx->stream;
    DevBuf* bufs[4] = {&ctx->h_pos, &ctx->h_quat, &ctx->h_vel, &ctx->h_ang};
    void* host[4] = {pos, quat, vel, angmom};
    if (!ctx->copy_stream) {
        CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&ctx->ev_copy, cudaEventDisableTiming));
    }
    for (int k = 0; k < 4; ++k) CU(bufs[k]->reserve(r4 * N));
    CU(ctx->h_sid.reserve(sizeof(int32_t) * (size_t)N));
    CU(cudaStreamSynchronize(st));  // the device scratch may still be in use by earlier work of the caller's stream
    // positions, orientations and shape ids first, on the caller's stream: the list build and the first evaluation
    // start as soon as they have arrived; velocities and angular momenta travel on a second stream beside them
    for (int k = 0; k < 2; ++k) CU(cudaMemcpyAsync(bufs[k]->p, host[k], r4 * N, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(ctx->h_sid.p, shape_id, sizeof(int32_t) * (size_t)N, cudaMemcpyHostToDevice, st));
    for (int k = 2; k < 4; ++k)
        CU(cudaMemcpyAsync(bufs[k]->p, host[k], r4 * N, cudaMemcpyHostToDevice, ctx->copy_stream));
    CU(cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
    ctx->ev_copy_pending = true;
    CU(ctx->h_force.reserve(r4 * N));
    CU(ctx->h_torque.reserve(r4 * N));
    ctx->early_host[0] = pos;
    ctx->early_host[1] = quat;
    ctx->early_done = false;
    const int rc = dem_step(ctx, ctx->h_pos.p, ctx->h_quat.p, ctx->h_vel.p, ctx->h_ang.p, ctx->h_sid.as<int32_t>(), N,
                            box, dt, nsteps, skin, ctx->h_force.p, ctx->h_torque.p);
    const bool early = ctx->early_done;
    ctx->early_host[0] = ctx->early_host[1] = nullptr;
    ctx->early_done = false;
    if (rc != DEM_OK) {  // the caller's host arrays must not be in use by a copy when an error is returned
        cudaStreamSynchronize(ctx->copy_stream);
        ctx->ev_copy_pending = false;
        return rc;
    }
    // (positions and orientations were final before the last evaluation: dem_step has sent them on copy_stream already)
    for (int k = early ? 2 : 0; k < 4; ++k) CU(cudaMemcpyAsync(host[k], bufs[k]->p, r4 * N, cudaMemcpyDeviceToHost, st));
    if (force_energy) CU(cudaMemcpyAsync(force_energy, ctx->h_force.p, r4 * N, cudaMemcpyDeviceToHost, st));
    if (torque) CU(cudaMemcpyAsync(torque, ctx->h_torque.p, r4 * N, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (early) CU(cudaStreamSynchronize(ctx->copy_stream));
    return DEM_OK;
}

}  // extern "C"
