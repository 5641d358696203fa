// dem_ctx.h -- the library context and the declarations shared by the translation units of libdem_b200 (host side).
//   dem_lib.cu            C ABI (include/dem.h), neighbour build, step loops, energies
//   dem_eval.cu           one force evaluation: per-class pose + pair kernels, per-particle reduction
//   dem_pair_fast.cu      launchers of k_pose / k_pair_fast      (packed FP32 contact search)
//   dem_pair_cull.cu      launchers of k_pair_cull               (the same with exact per-feature culling)
//   dem_pair_generic.cu   launchers of k_pair                    (generic fused kernel: FP64 contexts, 2D)
//   dem_bench.cu          measurement hooks of include/dem_bench.h
// The pair kernels are template-heavy; one translation unit each lets nvcc compile them in parallel.
#pragma once
#include <cuda_runtime.h>
#include <cstdlib>

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/dem.h"
#include "dem_shape.h"
#include "dem_types.h"

namespace dem {

struct DevBuf {  // grow-only device buffer
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes) {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
        // half as much again: a lattice that melts lists 45 % more pairs (config 4: 786 k -> 1.14 M), and regrowing the
        // pair-sized buffers in the middle of a run costs tens of milliseconds of cudaFree / cudaMalloc (measured: 31 ms)
        size_t want = bytes + bytes / 2 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e == cudaSuccess) cap = want;
        return e;
    }
    void release() {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
    template <typename T> T* as() const { return static_cast<T*>(p); }
};

}  // namespace dem

using namespace dem;  // internal header: only the library's own translation units include it

struct dem_ctx {
    int dim = 3, prec = DEM_F32;
    double eps = 1.0, eps_par = 1e-6;
    cudaStream_t stream = nullptr;
    std::string err;
    std::vector<HostShape> shapes;
    bool table_dirty = true;
    std::vector<ShapeDev> shape_dev;
    DevBuf table;
    MassTable mt;
    // neighbour list state
    bool have_list = false;
    bool list_from_step = false;  // the list was built by dem_step (cutoff = reach + skin, pos_build and sid_copy valid)
    int N = 0, stride = 16, max_count = 0;
    double box[3] = {0, 0, 0}, r_cut = 0;
    GridDev grid;
    DevBuf cell_of, rank, cell_start, order, xs, counts, list, slot, scratch_scan, pcnt, pairs, rec, rflag, flags, counters, thermo;
    DevBuf cum;         // running totals of the swept-term counters while timing is on
    DevBuf pose, pidx;  // FP32 search kernel: compacted pose records per class (k_pose)
    DevBuf cmask;       // culling kernel: survivor masks per compacted pair (k_pose_cull)
    ClassTable ct;
    int nclass = 0;
    int class_sa[DEM_MAX_CLASSES], class_sb[DEM_MAX_CLASSES], class_np[DEM_MAX_CLASSES];
    long long npairs_total = 0, nrec_total = 0;
    int force_slices = 0;  // 0 = heuristic
    bool cull = true;             // packed search kernel in 3D: exact per-feature culling (dem_set_culling)
    bool generic_kernel = false;  // DEM_F32 contexts: use the generic k_pair instead of the packed search kernel
    bool particle2d = false;      // DEM_F32 contexts in 2D (DEM_KERNEL_AUTO): the per-particle kernel k_particle2d
    size_t l2_flush_bytes = 0;  // bench hygiene: overwrite this many bytes of scratch before every time step
    DevBuf l2_scratch;
    // dem_step state (double) for DEM_F32 contexts, plus forces and the positions of the last build
    DevBuf st_pos, st_quat, st_vel, st_ang, st_force, st_torque, st_virial, pos_build, epart;
    DevBuf st_pos2, st_quat2;  // second position / orientation buffers of the 2D per-particle step (ping-pong)
    // A DEM_F32 context that is handed back, unchanged, the arrays its last dem_step returned continues from its internal
    // double state, neighbour list and forces instead of converting, rebuilding and re-evaluating (dem_lib.cu: step_t)
    struct Resume {
        bool valid = false;
        const void *pos = nullptr, *quat = nullptr, *vel = nullptr, *ang = nullptr;
        const int32_t* sid = nullptr;
        int N = 0, cur = 0;
        double box[3] = {0, 0, 0}, skin = 0;
    } resume;
    DevBuf sid_copy;
    // host-buffer entry points
    DevBuf h_pos, h_quat, h_vel, h_ang, h_sid, h_force, h_torque, h_virial;
    // accounting
    int64_t launches = 0;
    // kernel-time accounting (include/dem_bench.h): CUDA events on the stream, spans labelled by kernel kind
    int timing = 0;                    // 0 off, 1 pose + pair kernels, 2 every kernel of a step
    std::vector<cudaEvent_t> ev_pool;  // events handed out by ev_mark
    size_t ev_used = 0;
    struct EvSpan { int kind; cudaEvent_t a, b; };
    std::vector<EvSpan> ev_spans;
    int64_t last_terms = 0;
    int sm_count = 148;
    int* h_moved = nullptr;        // pinned host copy of dem_step's flags (moved, halt, steps completed)
    // dem_step_host: positions and orientations are final before the last force evaluation of a call, so they travel back
    // to the host (on copy_stream) while that evaluation runs
    void* early_host[2] = {nullptr, nullptr};  // host destinations of pos and quat, or null (device-array calls)
    bool early_done = false;
    cudaEvent_t ev_early = nullptr;
    cudaStream_t copy_stream = nullptr;  // dem_step_host: second H2D stream (velocities, angular momenta)
    cudaEvent_t ev_copy = nullptr;
    bool ev_copy_pending = false;
    // pair classes beyond the first run their pose + pair kernels on side streams, so that the tails of the per-class
    // launches overlap (mixed-shape systems: config 5 has three classes); forked from and joined to `stream` with events
    cudaStream_t class_stream[3] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[3] = {nullptr, nullptr, nullptr};
    double nvt_dof = 0;            // degrees of freedom counted by the last dem_step_nvt
    int steps_since_build = 0;     // age of the list when the last dem_step returned (carried into a resumed call)
    int rebuild_interval = 8;      // steps between the last two neighbour rebuilds of dem_step (sizes its chunks)
};

namespace dem {

inline int fail(dem_ctx* c, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf;
    return code;
}

#define CU(call)                                                                                        \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess)                                                                          \
            return dem::fail(ctx, e_ == cudaErrorMemoryAllocation ? DEM_ENOMEM : DEM_ECUDA, "%s: %s", #call, \
                             cudaGetErrorString(e_));                                                   \
    } while (0)
#define CHECK(call)             \
    do {                        \
        int rc_ = (call);       \
        if (rc_ != DEM_OK) return rc_; \
    } while (0)
#define LAUNCHED(ctx) ((ctx)->launches++)

inline int nblk(long long n, int b) { return (int)((n + b - 1) / b); }

// kernel kinds of the time accounting (dem_kernel_times of include/dem_bench.h)
enum { KT_POSE = 0, KT_PAIR = 1, KT_REDUCE = 2, KT_KICK_DRIFT = 3, KT_NEIGH = 4, KT_BUILD = 5, KT_FLUSH = 6, KT_OTHER = 7, KT_COUNT = 8 };
// record an event on the context's stream (null when timing is below `level` or an event cannot be created)
inline cudaEvent_t ev_mark(dem_ctx* c, int level = 1, cudaStream_t on = nullptr, bool on_given = false) {
    if (c->timing < level) return nullptr;
    if (c->ev_used == c->ev_pool.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        c->ev_pool.push_back(e);
    }
    cudaEvent_t e = c->ev_pool[c->ev_used++];
    cudaEventRecord(e, on_given ? on : c->stream);
    return e;
}
inline void ev_span(dem_ctx* c, int kind, cudaEvent_t a, cudaEvent_t b) {
    if (a && b) c->ev_spans.push_back({kind, a, b});
}

inline double reach_of(const HostShape& a, const HostShape& b) {
    return a.circumradius + b.circumradius + std::pow(2.0, 1.0 / 6.0) * (a.rounding + b.rounding);
}
inline double max_reach(const dem_ctx* ctx) {
    double r = 0;
    for (auto& a : ctx->shapes)
        for (auto& b : ctx->shapes) r = std::max(r, reach_of(a, b));
    return r;
}
// nominal Eq. 1 / Eq. 2 terms of one pair of the class, and the outer-loop length the pair kernel slices
inline long long class_terms(const dem_ctx* ctx, int c) {
    const HostShape &A = ctx->shapes[ctx->class_sa[c]], &B = ctx->shapes[ctx->class_sb[c]];
    if (ctx->dim == 3) return (long long)A.ne * B.ne + (long long)A.nv * B.nf + (long long)B.nv * A.nf;
    return (long long)A.nv * B.ne + (long long)B.nv * A.ne;
}
inline int class_outer(const dem_ctx* ctx, int c) {
    const HostShape &A = ctx->shapes[ctx->class_sa[c]], &B = ctx->shapes[ctx->class_sb[c]];
    return ctx->dim == 3 ? B.ne + B.nv + A.nv : B.nv + A.nv;
}
inline BoxDev box_dev(int dim, const double box[3]) {
    BoxDev bx;
    bx.dim = dim;
    for (int a = 0; a < 3; ++a) bx.L[a] = box[a];
    if (dim == 2) bx.L[2] = 1.0;
    for (int a = 0; a < 3; ++a) bx.invL[a] = 1.0 / bx.L[a];
    return bx;
}

// ---- dem_eval.cu: one force evaluation over the current list (steps a3-a8) ---------------------------------------------
// pos / quat are float[N][4] or double[N][4] (pos_is_double); force / torque / virial are `real` of the context.
// fin (null outside dem_step): what the reduction kernel does behind the reduction (FinArgs: integrator, device flags).
int evaluate(dem_ctx* ctx, const void* pos, const void* quat, bool pos_is_double, const int32_t* sid, int N, void* force,
             void* torque, void* virial, const FinArgs* fin);

// ---- kernel launchers (one translation unit per kernel family) ------------------------------------------------------------
void launch_pose(int dim, bool pos_is_double, int grid, cudaStream_t st, const PoseArgs& pa);
void launch_pose_cull(bool pos_is_double, int grid, size_t smem, cudaStream_t st, const PoseArgs& pa);
int pose_cull_max_words();
cudaError_t launch_pair_fast(int dim, bool tv3, int grid, int threads, size_t smem, cudaStream_t st, const PairArgs<float>& a);
cudaError_t launch_pair_cull(bool same_shape, int grid, int threads, size_t smem, cudaStream_t st, const PairArgs<float>& a);
cudaError_t launch_pair_generic_f32(int dim, bool pos_is_double, int grid, int threads, size_t smem, cudaStream_t st,
                                    const PairArgs<float>& a);
cudaError_t launch_pair_generic_f64(int dim, int grid, int threads, size_t smem, cudaStream_t st, const PairArgs<double>& a);
// k_particle2d (dem_step2d.cu): the whole 2D evaluation (+ integrator, FinArgs) of a DEM_F32 context in one kernel.
// pos / quat are what the forces are evaluated at; in mode 2 the drifted state is written to fin->pos / fin->quat,
// which must be other buffers.  Returns false when the kernel does not apply (rows longer than its bit mask).
bool particle2d_applies(const dem_ctx* ctx);
int launch_particle2d(dem_ctx* ctx, const void* pos, const void* quat, bool pos_is_double, const int32_t* sid, int N,
                      void* force, void* torque, void* virial, const FinArgs* fin);
size_t pair_fast_smem_header();
size_t pair_cull_smem_header();
int pose_threads();

}  // namespace dem
