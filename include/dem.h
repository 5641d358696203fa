/*
 * dem.h -- C ABI of libdem_b200: the DEM conservative force / torque / energy / virial evaluation between rounded
 * polytopes of arXiv:1607.02427, hand-written CUDA for sm_100a (one GPU).
 *
 * What the library computes (citations are PAPER.md lines):
 *   Eq. 1  3D:  U_ij = sum_{E_i,E_j} U(r*_EE) + sum_{V_i,F_j} U(r*_VF) + sum_{V_j,F_i} U(r*_VF)
 *   Eq. 2  2D:  U_ij = sum_{V_i,E_j} U(r*_VE) + sum_{V_j,E_i} U(r*_VE)
 *   r* = distance between the nearest points of two features; U = WCA (Eq. 3-4)
 *   with sigma_ij = rho_i + rho_j (rounding radius = sigma/2) and r_cut^WCA = 2^(1/6) sigma_ij;
 *   force along the line between the nearest points, torque from the interaction point on each particle
 *   (PAPER.md:45); near-parallel edges interact at the midpoint of their overlap;
 *   per-particle totals = sum over neighbours; virial tensor for "the barostat ... just as in MD"
 *   (PAPER.md:115); second-order NVE integrator.
 * Readings of passages on which the paper is silent or ambiguous are DESIGN.md "Readings" R1..R13.
 *
 * Conventions
 *   - Every function returns DEM_OK (0) or a negative dem_status.  No exception crosses the ABI.
 *     dem_last_error(ctx) returns a NUL-terminated description of the last failure on that context (owned by ctx).
 *   - `real` is float for a context created with DEM_F32 and double for DEM_F64 (one precision per context).
 *     Particle arrays are passed as `void*`/`const void*` and are interpreted as real[N][4] (16-byte aligned for
 *     float, 32-byte aligned for double), row-major, unless a parameter comment says otherwise.
 *   - Parameters documented "DEVICE" are device pointers owned by the caller (e.g. torch tensors); the library
 *     never frees or retains them beyond the call.  Parameters documented "HOST" are host pointers, read or written
 *     during the call only.  The library owns only what hangs off the opaque context.
 *   - All device work is enqueued on the cudaStream_t given to dem_create (NULL = legacy default stream).  Calls that
 *     return host scalars or need a capacity check synchronise that stream (each function says so).
 *   - Positions: x,y,z,(unused).  Box: orthorhombic, edge lengths box[3], centred on the origin, periodic in the
 *     first `dim` axes (2D ignores box[2] and z).  Positions outside the box are legal: every separation goes through
 *     the minimum image  d_a -= L_a * rint(d_a / L_a).
 *   - Quaternions: w,x,y,z, unit, scalar first, body -> lab (v_lab = q v q*); 2D: (cos t/2, 0, 0, sin t/2).
 *   - Angular momentum: LAB frame, Lx,Ly,Lz,(unused); 2D uses only Lz.
 *   - There is no CPU fallback: every entry point that computes needs a CUDA device and fails with DEM_ECUDA without.
 */
#ifndef DEM_B200_H
#define DEM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dem_ctx dem_ctx; /* opaque */

typedef enum dem_status {
    DEM_OK = 0,
    DEM_EINVAL = -1,    /* bad argument / malformed shape                                                        */
    DEM_ENOMEM = -2,    /* host or device allocation failed                                                      */
    DEM_ECUDA = -3,     /* CUDA runtime error (text in dem_last_error)                                           */
    DEM_EBOX = -4,      /* a periodic box edge < 2 r_cut: the minimum image would be invalid                      */
    DEM_ERCUT = -5,     /* r_cut < max_ij (R_i + R_j + 2^(1/6) sigma_ij): interactions would be dropped silently  */
    DEM_EOVERFLOW = -6, /* neighbour capacity exceeded and could not be regrown                                  */
    DEM_ESTALE = -7     /* dem_compute without a list, or with N different from the last dem_build_neighbors     */
} dem_status;

enum { DEM_F32 = 0, DEM_F64 = 1 };

/* Create a context.  dim = 2 or 3; epsilon = the single WCA energy scale (Eq. 3); precision = DEM_F32 | DEM_F64;
 * cuda_stream = a cudaStream_t (as void*), NULL for the default stream.  Does not touch the GPU beyond
 * cudaGetDevice.  *out is owned by the caller and released with dem_destroy (which frees everything the library
 * allocated on host and device). */
int dem_create(dem_ctx** out, int dim, double epsilon, int precision, void* cuda_stream);
int dem_destroy(dem_ctx* ctx);
const char* dem_last_error(const dem_ctx* ctx);

/* Near-parallel edge threshold of PAPER.md:59 (reading R5): edges are "sufficiently close to parallel" iff
 * |d1 x d2|^2 < eps_par |d1|^2 |d2|^2.  Default 1e-6. */
int dem_set_eps_par(dem_ctx* ctx, double eps_par);

/*
 * Register a shape (inner polygon/polyhedron given by vertices V, edges E, faces F, rounded by a
 * disk/sphere of radius `rounding_radius` = sigma/2).  All pointers HOST; copied.
 *   verts          [nv][3] doubles, body frame, centre of mass at the origin, principal axes (z = 0 in 2D); nv >= 1
 *   face_offsets   [nf+1] CSR offsets into face_verts; face_verts = vertex indices of each planar convex polygon face
 *                  in boundary order (either orientation: faces are two-sided).  2D: NULL, NULL, 0.
 *   edges          [ne][2] vertex index pairs, or NULL (then ne is ignored) to derive them: 2D = the closed CCW
 *                  polygon, edge k = (k, (k+1) mod nv), a single edge for nv = 2, the degenerate edge
 *                  (0,0) for nv = 1; 3D = the unique undirected boundary edges of the faces.
 *                  Explicit edges allow the degenerate shapes used as pins: sphere = 1 vertex + edge (0,0), no face
 *                  (Eq. 1 then reduces to one central WCA); rod = 2 vertices + edge (0,1).
 *   mass, inertia  mass and the three principal moments (2D uses inertia[2]); only dem_step / dem_energy use them.
 *   *shape_id      receives the id (0, 1, ...) to be used in the shape_id arrays.
 * Errors: DEM_EINVAL for indices out of range, faces with < 3 vertices, non-planar or non-convex faces, nv < 1,
 * rounding_radius <= 0, more than DEM_MAX_SHAPES shapes.  Invalidates the current neighbour list.
 */
#define DEM_MAX_SHAPES 8
int dem_create_shape(dem_ctx* ctx, const double* verts, int nv, const int* face_offsets, const int* face_verts,
                     int nf, const int* edges, int ne, double rounding_radius, double mass,
                     const double inertia[3], int* shape_id);

/*
 * Build the cell list and the full (two-sided) neighbour list ("it and its neighbors"; reading R13):
 * j is a neighbour of i  <=>  j != i and the minimum-image |x_j - x_i|^2 < r_cut^2 (strict), evaluated in double on
 * the stored coordinate values with exactly the operation order of DESIGN.md R13, so that the list is bit-identical
 * to the all-pairs definition.  Also builds the library's internal unique-pair work list for dem_compute.
 *   pos       DEVICE real[N][4]      shape_id  DEVICE int32[N]      box  HOST double[3]
 * Does not modify caller data.  Synchronises the stream (capacity check; the list is regrown and rebuilt
 * transparently on overflow).  Errors: DEM_EBOX, DEM_ERCUT, DEM_EINVAL (N < 1, no shapes), DEM_ECUDA, DEM_ENOMEM.
 */
int dem_build_neighbors(dem_ctx* ctx, const void* pos, const int32_t* shape_id, int N, const double box[3],
                        double r_cut);

/* Device pointers (owned by ctx, valid until the next build or dem_destroy) to the list of the last build:
 * counts[i] = number of neighbours of i, row i = list[i*stride .. i*stride + counts[i]), rows in no particular
 * order.  *max_count (may be NULL) receives the largest count. */
int dem_get_neighbors(dem_ctx* ctx, const int32_t** counts, const int32_t** list, int* stride, int* max_count);

/* Copy the list of the last build into caller-owned DEVICE arrays: counts_out int32[N], list_out int32[N][out_stride]
 * (out_stride >= max_count; unused entries are set to -1).  Asynchronous on the context's stream. */
int dem_copy_neighbors(dem_ctx* ctx, int32_t* counts_out, int32_t* list_out, int out_stride);

/*
 * Evaluate Eq. 1 / Eq. 2 over the current neighbour list (steps a3-a8 of DESIGN.md).  All pointers DEVICE.
 *   pos, quat     real[N][4]        shape_id  int32[N]
 *   force_energy  real[N][4]  = Fx, Fy, Fz, U_i      with U_i = 1/2 sum_j U_ij
 *   torque        real[N][4]  = lab-frame torque, 0  (2D: only .z is non-zero)
 *   virial6       real[N][6]  = 1/2 sum_j W_ij, W^{ab} = r_ij^a F_ij^b, r_ij = x_i - x_j (xx,xy,xz,yy,yz,zz); may be NULL
 * Outputs are fully overwritten.  Asynchronous (no synchronisation).  The positions may have moved since the build
 * as long as no pair that can interact is missing from the list (dem_step takes care of that with a skin).
 * Features closer than 1e-6 sigma are outside the model (WCA diverges): the term is skipped and counted (R11).
 * Errors: DEM_ESTALE, DEM_EINVAL, DEM_ECUDA.
 */
int dem_compute(dem_ctx* ctx, const void* pos, const void* quat, const int32_t* shape_id, int N, void* force_energy,
                void* torque, void* virial6);

/* Counters of the last dem_compute (not of dem_step, whose kernels keep none) (synchronises): out[0] unique particle pairs evaluated, out[1] Eq. 1/2 terms
 * of those pairs (polygon faces, each unique pair once), out[2] terms inside the WCA cutoff, out[3] degenerate terms
 * skipped, out[4] terms that took the parallel-edge branch, out[5] unique pairs in the work list, out[6] terms whose
 * nearest-point search was actually executed (= out[1] unless exact culling proved features out of reach: see
 * dem_set_culling), out[7] of which edge-edge terms (3D; in 2D all terms are vertex-edge and are counted here),
 * out[8] face boundary-edge tests inside the executed vertex-face terms (out[7] and out[8] feed the flop count of
 * bench.py). HOST int64[9]. */
int dem_get_counters(dem_ctx* ctx, int64_t out[9]);

/*
 * nsteps of velocity-Verlet NVE with quaternion rotation (reading R15): half-kick v and L; drift x
 * (wrapped back into the centred box); free rotation of q (exact for spherical tops and in 2D, symmetric splitting
 * otherwise); force evaluation; half-kick.  pos, quat, vel, angmom: DEVICE real[N][4], updated in place;
 * shape_id DEVICE int32[N]; box HOST double[3].  The neighbour list is (re)built with r_cut = reach + skin, reach =
 * max_ij (R_i + R_j + 2^(1/6) sigma_ij), and rebuilt whenever some particle has moved more than skin/2 since the last
 * build.  A DEM_F32 context integrates its state in double internally (R15b) and rounds it to float on return.
 * force_energy / torque (DEVICE real[N][4], may be NULL) receive the forces of the final state.
 * Synchronises before returning.
 */
int dem_step(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N,
             const double box[3], double dt, int nsteps, double skin, void* force_energy, void* torque);

/*
 * NVT: dem_step with a Nose-Hoover thermostat "applied to both translational and rotational degrees of freedom"
 * (R19).  One friction variable xi for all degrees of freedom:
 *     dv/dt = F/m - xi v,   dL/dt = tau - xi L,   dxi/dt = (2K - g kT)/Q,   deta/dt = xi,   Q = g kT tau^2,
 * K = K_trans + K_rot, g = dim (N - 1) + number of (particle, rotation axis) with inertia > 0 (2D: the z axis).
 * One step = thermostat half step, the NVE step of dem_step, thermostat half step; a half step is
 *     xi += (dt/4)(2K - g kT)/Q;  s = exp(-xi dt/2);  v *= s;  L *= s;  K *= s^2;  eta += (dt/2) xi;
 *     xi += (dt/4)(2K - g kT)/Q.
 * U + K + Q xi^2 / 2 + g kT eta is conserved.  With the barostat of PAPER.md:115: dem_step_npt.
 *   kT, tau        target temperature and thermostat period (> 0)
 *   thermostat[2]  HOST, in and out: (xi, eta); start a run from (0, 0) and pass the values back in to continue it
 *   *dof           HOST, may be NULL: receives g
 * Everything else as dem_step.  Errors: those of dem_step; DEM_EINVAL for kT <= 0, tau <= 0, N < 2.
 */
int dem_step_nvt(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N,
                 const double box[3], double dt, int nsteps, double skin, double kT, double tau, double thermostat[2],
                 double* dof, void* force_energy, void* torque);

/*
 * NPT: dem_step_nvt plus a barostat that "computes the pressure from the virial tensor, just as in MD" (
 * SURVEY.md 8(f) NEXT-3).  The paper gives no equations; R22: the isotropic Martyna-Tobias-Klein barostat on
 * the strain rate nu = d ln L / dt of the box, coupled to the centres of mass only (the centre-of-mass virial
 * tr W = sum_pairs r_ij . F_ij that dem_compute produces; orientations and angular momenta do not feel the box):
 *     dx/dt = v + nu x,  dL_box/dt = nu L_box,  dv/dt = F/m - (alpha nu + xi) v,  dL/dt = tau - xi L,
 *     dnu/dt = [alpha 2 K_trans + tr W - d V P] / W_b,   alpha = 1 + d / N_f,  N_f = d (N - 1),  W_b = d N kT tau_p^2,
 *     dxi/dt = (2K - g kT)/Q, deta/dt = xi  (as in dem_step_nvt),
 * d = 2 or 3, V = the box volume (area in 2D), i.e. d V (P_int - P) + (d/N_f) 2 K_trans with the instantaneous pressure
 * P_int = (2 K_trans + tr W) / (d V).  U + K + P V + W_b nu^2/2 + Q xi^2/2 + g kT eta is conserved.
 * One step (time-reversible, second order; h = dt/2): thermostat half step, nu += h dnu/dt, v = (v s + h F/m) s with
 * s = exp(-alpha nu h / 2) and L += h tau, drift x = x e^{nu dt} + v dt e^{nu dt/2} sinh(nu dt/2)/(nu dt/2) with the box
 * scaled by e^{nu dt} and free rotation, forces, and the same three half steps in reverse order.
 *   box[3]     HOST, in and out: the box edges (all periodic edges scale by the same factor)
 *   pressure   the external pressure P;  tau_p the barostat period (> 0; infinity = constant volume)
 *   state[3]   HOST, in and out: (xi, eta, nu); start a run from (0, 0, 0) and pass the values back in to continue it
 * The neighbour list follows the box: it is rebuilt when a particle has moved more than allowed by the skin away from
 * the affine image of its position at the last build.  Everything else as dem_step_nvt (tau = infinity: no thermostat).
 * Errors: those of dem_step; DEM_EINVAL for kT, tau, tau_p <= 0 or N < 2; DEM_EBOX when the box shrinks below twice the
 * interaction reach.  Synchronises once per step (the scalar equations are advanced on the host between kernels).
 */
int dem_step_npt(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N, double box[3],
                 double dt, int nsteps, double skin, double kT, double tau, double pressure, double tau_p, double state[3],
                 double* dof, void* force_energy, void* torque);

/* U = sum_i U_i (from force_energy[.][3]), K_trans, K_rot of a state; DEVICE inputs, HOST out[3]; synchronises. */
int dem_energy(dem_ctx* ctx, const void* quat, const void* vel, const void* angmom, const int32_t* shape_id,
               const void* force_energy, int N, double out[3]);

/*
 * The same three sums without any device allocation, for callers that cannot call cudaMalloc (CUDA graph capture, tight
 * serving loops): the per-block partial sums go to a fixed device array inside the library (96 KiB, held by every GPU
 * that loads the library until exit) instead of a buffer the context allocates.
 *   quat, vel, angmom, force_energy  DEVICE real[N][4]   shape_id  DEVICE int32[N]   (as dem_energy)
 *   out_dev    DEVICE double[3]: U, K_trans, K_rot; written by the context's stream, NOT synchronised
 * N <= DEM_ENERGY_STATIC_MAX_N, else DEM_EINVAL (use dem_energy).  Calls no cudaMalloc / cudaFree, copies nothing to
 * the host and does not touch the context's own buffers.  All calls (of every context on a GPU) share the one array:
 * calls issued to one stream are safe, calls that overlap on the GPU race.  The array needs no clearing: a call reads
 * only what it has just written.  The first call on a device looks the array's address up (cudaGetSymbolAddress): make
 * it outside a graph capture.  Sums are in double in a fixed order; they differ from dem_energy's by summation order only.
 */
#define DEM_ENERGY_STATIC_MAX_N (1 << 20)
int dem_energy_static(dem_ctx* ctx, const void* quat, const void* vel, const void* angmom, const int32_t* shape_id,
                      const void* force_energy, int N, double* out_dev);

/*
 * Host-buffer forms (the end-to-end path): same semantics, every particle array is a HOST pointer (pinned memory
 * gives the best copy rate); the library copies inputs to device scratch it owns, runs dem_build_neighbors +
 * dem_compute (or dem_step), copies the results back and synchronises.
 */
int dem_compute_host(dem_ctx* ctx, const void* pos, const void* quat, const int32_t* shape_id, int N,
                     const double box[3], double r_cut, void* force_energy, void* torque, void* virial6);
int dem_step_host(dem_ctx* ctx, void* pos, void* quat, void* vel, void* angmom, const int32_t* shape_id, int N,
                  const double box[3], double dt, int nsteps, double skin, void* force_energy, void* torque);

/* Tuning / test hook: number of lanes that share one particle pair in the pair-feature kernel (each takes a slice of
 * the pair's outer feature loop; their partial results are summed by the reduction).  0 = heuristic (default: enough
 * lanes to fill the GPU when there are few pairs).  Takes effect at the next neighbour build. */
int dem_set_slices(dem_ctx* ctx, int slices);

/* Which pair-feature kernel a DEM_F32 context runs.  DEM_KERNEL_SEARCH: the packed-FP32 contact search with
 * cooperative evaluation of the candidate terms.  DEM_KERNEL_GENERIC: the fused scalar kernel
 * that DEM_F64 contexts always use (every Eq. 1 / Eq. 2 term evaluated in place).  DEM_KERNEL_AUTO (default): SEARCH in
 * 3D, GENERIC in 2D, where a pair has so few terms (2 V E) that the pose records and the candidate queue cost more than
 * they save (measured on config 3: 64 us against 91 us per evaluation).  Both produce the same contributing terms;
 * sums may differ in rounding order.  Takes effect at the next dem_compute / dem_step. */
#define DEM_KERNEL_SEARCH 0
#define DEM_KERNEL_GENERIC 1
#define DEM_KERNEL_AUTO 2
int dem_set_pair_kernel(dem_ctx* ctx, int which);

/* Exact per-feature culling in the packed search kernel (3D, DEM_F32; default ON).  Every feature of a particle lies
 * within its circumradius R of its centre, so a feature of the other particle whose distance from that centre is at
 * least R + (search cutoff) cannot be within the WCA cutoff of ANY of its features: the search skips it, with
 * identical results (same contributing terms, same arithmetic; PAPER.md:129 names such shape-local culling as the next
 * step).  0 = sweep every Eq. 1 term (the paper's method as stated).  Takes effect at the next
 * dem_compute / dem_step. */
int dem_set_culling(dem_ctx* ctx, int enabled);

/* Measurement hooks (L2 flush, kernel-time accounting, launch count, FMA microbenchmark) live in dem_bench.h. */

const char* dem_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DEM_B200_H */
