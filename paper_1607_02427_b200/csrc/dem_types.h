// dem_types.h -- plain structs shared by the host code and the kernels of libdem_b200 (no device code here).
#pragma once
#include <stddef.h>
#include <stdint.h>
#include <vector_types.h>  // int2

// Checked build (python -m paper_1607_02427_b200.build --checked, loaded with DEM_CHECKED=1): every index into the
// hand-rolled warp-synchronous shared-memory structures (candidate queue, item list, staged poses) and into the pair /
// record / work-list arrays is bounds-checked on the device; a violation prints its location and traps, which the host
// sees as a CUDA error.  The release build compiles the checks away.  (compute-sanitizer is not available on the GPU
// pool this library is developed on; profiles/r02_sanitizers.md.)
#ifdef DEM_CHECKED
#include <cstdio>
#define DEM_ASSERT(cond)                                                                    \
    do {                                                                                    \
        if (!(cond)) {                                                                      \
            printf("DEM_ASSERT failed: %s  (%s:%d)\n", #cond, __FILE__, __LINE__);          \
            __trap();                                                                       \
        }                                                                                   \
    } while (0)
#else
#define DEM_ASSERT(cond) ((void)0)
#endif

namespace dem {

struct alignas(16) f4 { float x, y, z, w; };
struct alignas(16) d4 { double x, y, z, w; };
template <typename real> struct vec4;
template <> struct vec4<float> { typedef f4 type; };
template <> struct vec4<double> { typedef d4 type; };

#define DEM_MAX_SHAPES_K 8
#define DEM_REC 3  // real4 per pair result record
#define DEM_MAX_CLASSES (DEM_MAX_SHAPES_K * (DEM_MAX_SHAPES_K + 1) / 2)
#define DEM_MAX_FACE_GROUPS 4
#define DEM_POSE_THREADS 512

struct ShapeDev {
    int nv, ne, nf, nfe;
    int off, len;  // block [off, off+len) of the device table, in real4 units: V | E | F | FE | OE
    // runs of faces with equal boundary-edge counts (faces are stored sorted by that count): grp_n[g] faces with
    // grp_m[g] edges each; grp_n = 0 ends the list; grp_m[0] = 0 means "more runs than fit: read each face's header"
    int grp_m[DEM_MAX_FACE_GROUPS], grp_n[DEM_MAX_FACE_GROUPS];
};

struct ClassTable {  // indexed by pair class c = lut[s_a][s_b]
    signed char lut[DEM_MAX_SHAPES_K][DEM_MAX_SHAPES_K];
    int pair_base[DEM_MAX_CLASSES + 1];  // first global pair index of the class (class-major pair list)
    int rec_base[DEM_MAX_CLASSES + 1];   // first result record of the class
    int slices[DEM_MAX_CLASSES];         // result records per pair
};

struct BoxDev {
    double L[3];
    double invL[3];  // 1 / L (the bit-exact neighbour predicate R13 divides by L; everything else multiplies)
    int dim;
};

struct GridDev {
    int nc[3];
    int ncell;
};

struct MassTable {
    double mass[DEM_MAX_SHAPES_K];
    double inertia[DEM_MAX_SHAPES_K][3];
};

template <typename real> struct PairConst {
    real rc2;      // (2^(1/6) sigma_ij)^2 = 2^(1/3) sigma^2     (Eq. 4, compared squared: R7)
    real sig2;     // sigma_ij^2, sigma_ij = rho_i + rho_j       (R6)
    real eps;      // epsilon
    real eps_par;  // near-parallel threshold                    (R5)
    real degen2;   // (1e-6 sigma)^2                             (R11)
};

template <typename real> struct PairArgs {
    typedef typename vec4<real>::type real4;
    const real4* table;   // device shape table
    ShapeDev sa, sb;      // shapes of the pair's first / second particle
    const int2* pairs;    // this class's segment of the pair list
    int npairs;
    int slices;           // lanes per pair (each takes a slice of the outer feature loop)
    int n_outer;          // outer-loop length of the class
    real4* rec;           // this class's result records: DEM_REC real4 per (pair, slice)
    unsigned char* rflag; // one byte per result record: 1 = the record was written and carries a contribution, 0 = the
                          //   (pair, slice) contributes nothing and its record was NOT written (the reduction skips it)
    const void* pos;
    const void* quat;
    int pos_double;       // pos / quat are double[N][4] (else float[N][4])
    BoxDev box;
    double reach2;        // (R_a + R_b + 2^(1/6) sigma)^2 : beyond it no term can be inside the cutoff (exact, R10)
    PairConst<real> pc;
    real rc2_search;      // FP32 search kernel: squared candidate cutoff (WCA cutoff + slack, dem_fast.cuh)
    real cull_a2, cull_b2;  // culling kernel: (R_first + rc_search)^2, (R_second + rc_search)^2 (circumradii)
    const f4* pose;       // FP32 search kernel: this class's compacted pose records, pair indices and their number
    const int4* pidx;     //   (written by k_pose: pair index, its two particles, 0)
    const int* count;
    int* tile;            //   next tile to take (zero at launch), or null: tiles are dealt out by block and warp index
    size_t plane;         //   stride of the pose planes
    const unsigned* cmask;  // culling kernel: per-pair survivor masks written by k_pose_cull, [words][plane] (null: the
    int mw_e, mw_vj, mw_vi; //   kernel runs the cull tests itself); words for edges of j, vertices of j, vertices of i
    unsigned long long* counters;  // [0] pairs evaluated, [1] active, [2] degenerate, [3] parallel, [4..6] swept terms
    unsigned long long* cum;       // running totals of [4..6] while bench's timing is on (else null)
};

// k_pose (a3): relative pose of every pair of a class, compacted (dem_fast.cuh)
struct PoseArgs {
    const int2* pairs;
    int npairs, slices;
    const void* pos;
    const void* quat;
    BoxDev box;
    double reach2;
    f4* pose;
    int4* pidx;  // (pair index or -1 for padding, first particle, second particle, 0)
    int* count;  // entries of this class's work list, padding included (zeroed before the launch)
    size_t plane;  // stride of the pose planes = capacity of the work list (pairs + 64 per k_pose block)
    int pad;       // entries per warp tile of the kernel that follows: 32 (k_pair_fast) or 64 (k_pair_cull)
    unsigned long long* counters;  // [0] += pairs inside the reach
    unsigned char* rflag;  // result-record flags of the class: pairs beyond the reach get 0 here (no record is written)
    // k_pose_cull only: the class's shapes and cull radii; survivor masks out ([mw_e + mw_vj + mw_vi][plane])
    const f4* table;
    ShapeDev sa, sb;
    float cull_a2, cull_b2;
    unsigned* cmask;
    int mw_e, mw_vj, mw_vi;
    const int* skip;  // dem_step: non-null and *skip != 0 => the list is stale, the kernel does nothing (see step_t)
};

// What k_finish does behind the per-particle reduction (dem_kernels.cuh).
//   mode 0  nothing more (dem_compute)
//   mode 1  the second half kick of velocity Verlet, which completes a time step
//   mode 2  that, and the first half of the NEXT step: half kick, drift (wrapped), free rotation, skin test
// dem_step queues many steps before the host looks at anything; two device flags, used alternately, keep that safe:
// a kernel does nothing when *bail is set (raised by a kernel BEFORE it: some particle left its skin, the list is
// stale) -- it then raises *raise, so that the word reaches the evaluation after it, which looks at the other flag --
// and raises *raise when its own drift takes a particle out of its skin.
struct FinArgs {
    int mode, dim;
    int lanes;  // lanes per particle in k_finish's reduction (power of two <= 32; small systems use several: latency)
    double dt;
    d4 *pos, *quat, *vel, *ang;
    const d4* pos_build;  // positions at the last neighbour build (skin test)
    double half_skin2;
    BoxDev box;
    MassTable mt;
    const int* bail;
    int* raise;
    int* done;  // += 1 when the kernel completed a step (modes 1, 2)
};

// Nose-Hoover thermostat (dem_step_nvt; R19): friction xi, its time integral eta, the scaling
// of v and L that the next k_kick_drift (or k_scale_momenta) still has to apply, and the degrees of freedom g.
struct ThermoDev {
    double xi, eta, scale, dof;
};

}  // namespace dem
