// dem_integrate.cuh -- a9: the integrator kernels (velocity Verlet with quaternion rotation, Nose-Hoover thermostat,
// energies) and the precision conversion of the state.  Included by dem_lib.cu only.
#pragma once
#include "dem_kernels.cuh"

namespace dem {

// ---- a9: NVE integrator (reading R15) --------------------------------------------------------------------
// first half of velocity Verlet: v += dt/2 F/m; x += dt v (wrapped); L += dt/2 tau; free rotation of q.
// Raises *raise when a particle is farther than skin/2 from where it was at the last neighbour build.
// Does nothing when *bail is set (the list went stale in an earlier step of the same chunk; see FinArgs).
template <typename real>
__global__ void k_kick_drift(int N, BoxDev box, double dt, const int* __restrict__ sid, MassTable mt,
                             d4* __restrict__ pos, d4* __restrict__ quat, d4* __restrict__ vel, d4* __restrict__ ang,
                             const typename vec4<real>::type* __restrict__ force,
                             const typename vec4<real>::type* __restrict__ torque, const d4* __restrict__ pos_build,
                             double half_skin2, const int* __restrict__ bail, int* __restrict__ raise,
                             const ThermoDev* __restrict__ thermo) {
    // The translational and the rotational half of a particle's update are independent: the first half of the grid
    // does x, v (and the skin test), the second q, L -- twice the memory-level parallelism, half the dependent chain.
    if (bail && *bail) {
        if (blockIdx.x == 0 && threadIdx.x == 0) *raise = 1;  // pass the word on: the next evaluation looks at *raise
        return;
    }
    const int half = gridDim.x >> 1;
    const bool rot = (int)blockIdx.x >= half;
    const int i = (blockIdx.x - (rot ? half : 0)) * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int s = sid[i];
    const double sc = thermo ? thermo->scale : 1.0;  // NVT: pending thermostat scaling of v and L (k_thermostat)
    if (!rot) {
        const double hm = 0.5 * dt / mt.mass[s];
        d4 x = pos[i], v = vel[i];
        const typename vec4<real>::type F = force[i];
        const d4 xb = pos_build[i];
        double xs[3] = {x.x, x.y, x.z}, vs[3] = {v.x * sc, v.y * sc, v.z * sc};
        const double Fs[3] = {(double)F.x, (double)F.y, (double)F.z};
#pragma unroll
        for (int a = 0; a < 3; ++a)  // (static indices: the state stays in registers)
            if (a < box.dim) {
                vs[a] += hm * Fs[a];
                xs[a] += dt * vs[a];
                xs[a] -= box.L[a] * rint(xs[a] * box.invL[a]);
            }
        x.x = xs[0]; x.y = xs[1]; x.z = xs[2];
        v.x = vs[0]; v.y = vs[1]; v.z = vs[2];
        pos[i] = x;
        vel[i] = v;
        double dx = xs[0] - xb.x, dy = xs[1] - xb.y, dz = box.dim == 3 ? xs[2] - xb.z : 0.0;
        dx -= box.L[0] * rint(dx * box.invL[0]);
        dy -= box.L[1] * rint(dy * box.invL[1]);
        dz -= box.L[2] * rint(dz * box.invL[2]);
        if (dx * dx + dy * dy + dz * dz > half_skin2) *raise = 1;
    } else {
        d4 L = ang[i], q = quat[i];
        const typename vec4<real>::type T = torque[i];
        double Ls[3] = {L.x * sc, L.y * sc, L.z * sc};
        const double Ts[3] = {(double)T.x, (double)T.y, (double)T.z};
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (box.dim == 3 || a == 2) Ls[a] += 0.5 * dt * Ts[a];
        double qs[4] = {q.x, q.y, q.z, q.w};
        free_rotate(box.dim, mt.inertia[s], Ls, dt, qs);
        L.x = Ls[0]; L.y = Ls[1]; L.z = Ls[2];
        q.x = qs[0]; q.y = qs[1]; q.z = qs[2]; q.w = qs[3];
        ang[i] = L;
        quat[i] = q;
    }
}

// NVT: per-block partial sums of K_trans + K_rot and of the rotational degrees of freedom (axes with I > 0), in double,
// fixed order.  partial[2 b] = K, partial[2 b + 1] = degrees of freedom.
__global__ void k_kinetic(int N, int dim, const int* __restrict__ sid, MassTable mt, const d4* __restrict__ quat,
                          const d4* __restrict__ vel, const d4* __restrict__ ang, double* __restrict__ partial) {
    __shared__ double sh[2][256];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double K = 0, dof = 0;
    if (i < N) {
        const int s = sid[i];
        const d4 v = vel[i], L = ang[i], q = quat[i];
        K = 0.5 * mt.mass[s] * (v.x * v.x + v.y * v.y + v.z * v.z);
        double M[9];
        quat_to_mat<double>(q.x, q.y, q.z, q.w, M);
        for (int a = (dim == 2 ? 2 : 0); a < 3; ++a) {
            const double Lb = M[a] * L.x + M[3 + a] * L.y + M[6 + a] * L.z;
            const double I = mt.inertia[s][a];
            if (I > 0.0) {
                K += 0.5 * Lb * Lb / I;
                dof += 1.0;
            }
        }
    }
    sh[0][threadIdx.x] = K; sh[1][threadIdx.x] = dof;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            sh[0][threadIdx.x] += sh[0][threadIdx.x + o];
            sh[1][threadIdx.x] += sh[1][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partial[2 * blockIdx.x] = sh[0][0];
        partial[2 * blockIdx.x + 1] = sh[1][0];
    }
}

// NVT: one block sums the partials of k_kinetic and advances (xi, eta) by `halves` thermostat half steps (1: the end
// of the run, or its start; 2: the end of one step and the start of the next, which are adjacent).  The scaling of v
// and L is left in th->scale for the next k_kick_drift / k_scale_momenta.  Does nothing when the step it follows was
// not completed (*bail set, see FinArgs).
__global__ void k_thermostat(int nb, const double* __restrict__ partial, int dim, int N, double dt, double kT,
                             double tau, int halves, const int* __restrict__ bail, ThermoDev* __restrict__ th) {
    __shared__ double sh[2][256];
    if (bail && *bail) return;
    double K = 0, dof = 0;
    for (int b = threadIdx.x; b < nb; b += 256) {
        K += partial[2 * b];
        dof += partial[2 * b + 1];
    }
    sh[0][threadIdx.x] = K; sh[1][threadIdx.x] = dof;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            sh[0][threadIdx.x] += sh[0][threadIdx.x + o];
            sh[1][threadIdx.x] += sh[1][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    K = sh[0][0];
    const double g = (double)dim * (N - 1) + sh[1][0], Q = g * kT * tau * tau;
    double xi = th->xi, eta = th->eta, scale = 1.0;
    for (int h = 0; h < halves; ++h) {
        xi += 0.25 * dt * (2.0 * K - g * kT) / Q;
        const double s = exp(-xi * 0.5 * dt);
        K *= s * s;
        scale *= s;
        eta += 0.5 * dt * xi;
        xi += 0.25 * dt * (2.0 * K - g * kT) / Q;
    }
    th->xi = xi; th->eta = eta; th->scale = scale; th->dof = g;
}

// NVT: the scaling left by the last thermostat half step of a run.
__global__ void k_scale_momenta(int N, d4* __restrict__ vel, d4* __restrict__ ang, const ThermoDev* __restrict__ th) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double s = th->scale;
    d4 v = vel[i], L = ang[i];
    v.x *= s; v.y *= s; v.z *= s;
    L.x *= s; L.y *= s; L.z *= s;
    vel[i] = v;
    ang[i] = L;
}

// ---- NPT (dem_step_npt; R22) ----------------------------------------------------------------------
// The scalar variables of the thermostat and of the barostat (xi, eta, nu, the box) are advanced on the host between
// the kernels of a step: the box is a launch argument of every kernel that takes a minimum image.  What touches the
// particles runs here.
//
// First half of an NPT step: pending thermostat scaling `pend` of v and L, half kick with the barostat drag
// v = (v s + dt/2 F/m) s  (s = exp(-alpha nu dt/4)), L += dt/2 tau, drift x = x ea + v vb  (ea = e^{nu dt},
// vb = dt e^{nu dt/2} sinh(nu dt/2)/(nu dt/2)) wrapped into the NEW box, free rotation.  Raises moved[0] when the
// particle is farther than sqrt(thr2) from the affine image lambda x_build of where it was at the last list build
// (a pair outside the list then still is outside the interaction reach: |d| >= lambda r_list - 2 u_max).
template <typename real>
__global__ void k_npt_kick_drift(int N, BoxDev box, double dt, const int* __restrict__ sid, MassTable mt,
                                 d4* __restrict__ pos, d4* __restrict__ quat, d4* __restrict__ vel, d4* __restrict__ ang,
                                 const typename vec4<real>::type* __restrict__ force,
                                 const typename vec4<real>::type* __restrict__ torque, const d4* __restrict__ pos_build,
                                 double lambda, double thr2, int* __restrict__ moved, double pend, double s, double ea,
                                 double vb) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int sh = sid[i];
    const double m = mt.mass[sh];
    d4 x = pos[i], v = vel[i], L = ang[i], q = quat[i];
    const typename vec4<real>::type F = force[i], T = torque[i];
    const d4 xb = pos_build[i];
    double xs[3] = {x.x, x.y, x.z}, vs[3] = {v.x * pend, v.y * pend, v.z * pend};
    const double Fs[3] = {(double)F.x, (double)F.y, (double)F.z};
    for (int a = 0; a < box.dim; ++a) {
        vs[a] = (vs[a] * s + 0.5 * dt * Fs[a] / m) * s;
        xs[a] = xs[a] * ea + vs[a] * vb;
        xs[a] -= box.L[a] * rint(xs[a] * box.invL[a]);
    }
    x.x = xs[0]; x.y = xs[1]; x.z = xs[2];
    v.x = vs[0]; v.y = vs[1]; v.z = vs[2];
    pos[i] = x;
    vel[i] = v;
    double dx = xs[0] - lambda * xb.x, dy = xs[1] - lambda * xb.y, dz = box.dim == 3 ? xs[2] - lambda * xb.z : 0.0;
    dx -= box.L[0] * rint(dx * box.invL[0]);
    dy -= box.L[1] * rint(dy * box.invL[1]);
    dz -= box.L[2] * rint(dz * box.invL[2]);
    if (!(dx * dx + dy * dy + dz * dz <= thr2)) moved[0] = 1;
    double Ls[3] = {L.x * pend, L.y * pend, L.z * pend};
    const double Ts[3] = {(double)T.x, (double)T.y, (double)T.z};
    for (int a = (box.dim == 2 ? 2 : 0); a < 3; ++a) Ls[a] += 0.5 * dt * Ts[a];
    double qs[4] = {q.x, q.y, q.z, q.w};
    free_rotate(box.dim, mt.inertia[sh], Ls, dt, qs);
    L.x = Ls[0]; L.y = Ls[1]; L.z = Ls[2];
    q.x = qs[0]; q.y = qs[1]; q.z = qs[2]; q.w = qs[3];
    ang[i] = L;
    quat[i] = q;
}

// Second half kick of an NPT step: v = (v s + dt/2 F/m) s, L += dt/2 tau.
template <typename real>
__global__ void k_npt_kick(int N, int dim, double dt, const int* __restrict__ sid, MassTable mt, d4* __restrict__ vel,
                           d4* __restrict__ ang, const typename vec4<real>::type* __restrict__ force,
                           const typename vec4<real>::type* __restrict__ torque, double s) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double m = mt.mass[sid[i]];
    d4 v = vel[i], L = ang[i];
    const typename vec4<real>::type F = force[i], T = torque[i];
    v.x = (v.x * s + 0.5 * dt * (double)F.x / m) * s;
    v.y = (v.y * s + 0.5 * dt * (double)F.y / m) * s;
    if (dim == 3) {
        v.z = (v.z * s + 0.5 * dt * (double)F.z / m) * s;
        L.x += 0.5 * dt * (double)T.x;
        L.y += 0.5 * dt * (double)T.y;
    }
    L.z += 0.5 * dt * (double)T.z;
    vel[i] = v;
    ang[i] = L;
}

// Per-block partial sums (double, fixed order) of K_trans, K_rot, the rotational degrees of freedom and the trace of the
// virial: partial[4 b + 0..3].  The host adds the blocks' partials in order.
template <typename real>
__global__ void k_npt_sums(int N, int dim, const int* __restrict__ sid, MassTable mt, const d4* __restrict__ quat,
                           const d4* __restrict__ vel, const d4* __restrict__ ang, const real* __restrict__ virial,
                           double* __restrict__ partial) {
    __shared__ double sh[4][256];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double Kt = 0, Kr = 0, dof = 0, trw = 0;
    if (i < N) {
        const int s = sid[i];
        const d4 v = vel[i], L = ang[i], q = quat[i];
        Kt = 0.5 * mt.mass[s] * (v.x * v.x + v.y * v.y + v.z * v.z);
        double M[9];
        quat_to_mat<double>(q.x, q.y, q.z, q.w, M);
        for (int a = (dim == 2 ? 2 : 0); a < 3; ++a) {
            const double Lb = M[a] * L.x + M[3 + a] * L.y + M[6 + a] * L.z;
            const double I = mt.inertia[s][a];
            if (I > 0.0) {
                Kr += 0.5 * Lb * Lb / I;
                dof += 1.0;
            }
        }
        const real* w = virial + 6 * (size_t)i;
        trw = (double)w[0] + (double)w[3] + (dim == 3 ? (double)w[5] : 0.0);
    }
    sh[0][threadIdx.x] = Kt; sh[1][threadIdx.x] = Kr; sh[2][threadIdx.x] = dof; sh[3][threadIdx.x] = trw;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o)
            for (int a = 0; a < 4; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0)
        for (int a = 0; a < 4; ++a) partial[4 * blockIdx.x + a] = sh[a][0];
}

// v *= s, L *= s (the thermostat scaling still pending when a run ends)
static __global__ void k_scale_momenta_by(int N, d4* __restrict__ vel, d4* __restrict__ ang, double s) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    d4 v = vel[i], L = ang[i];
    v.x *= s; v.y *= s; v.z *= s;
    L.x *= s; L.y *= s; L.z *= s;
    vel[i] = v;
    ang[i] = L;
}

// U, K_trans, K_rot: per-block partial sums in double (fixed order), summed on the host.
template <typename real, typename PosT>
__global__ void k_energy(int N, int dim, const int* __restrict__ sid, MassTable mt, const PosT* __restrict__ quat,
                         const PosT* __restrict__ vel, const PosT* __restrict__ ang,
                         const typename vec4<real>::type* __restrict__ force, double* __restrict__ partial) {
    __shared__ double sh[3][256];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double U = 0, Kt = 0, Kr = 0;
    if (i < N) {
        const int s = sid[i];
        const d4 v = load4d(vel, i), L = load4d(ang, i), q = load4d(quat, i);
        U = (double)force[i].w;
        Kt = 0.5 * mt.mass[s] * (v.x * v.x + v.y * v.y + v.z * v.z);
        double M[9];
        quat_to_mat<double>(q.x, q.y, q.z, q.w, M);
        for (int a = (dim == 2 ? 2 : 0); a < 3; ++a) {
            const double Lb = M[a] * L.x + M[3 + a] * L.y + M[6 + a] * L.z;
            const double I = mt.inertia[s][a];
            if (I > 0.0) Kr += 0.5 * Lb * Lb / I;
        }
    }
    sh[0][threadIdx.x] = U; sh[1][threadIdx.x] = Kt; sh[2][threadIdx.x] = Kr;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o)
            for (int a = 0; a < 3; ++a) sh[a][threadIdx.x] += sh[a][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0)
        for (int a = 0; a < 3; ++a) partial[3 * blockIdx.x + a] = sh[a][0];
}

// Are the caller's float arrays still what the last dem_step returned, i.e. the internal double state rounded to float
// (and the shape ids the ones the list was built with)?  Raises *differ otherwise.
static __global__ void k_same_state(int n, const f4* __restrict__ pos, const f4* __restrict__ quat, const f4* __restrict__ vel,
                                    const f4* __restrict__ ang, const int* __restrict__ sid, const d4* __restrict__ x,
                                    const d4* __restrict__ q, const d4* __restrict__ v, const d4* __restrict__ L,
                                    const int* __restrict__ sid_copy, int* __restrict__ differ) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const f4* f[4] = {pos, quat, vel, ang};
    const d4* d[4] = {x, q, v, L};
    bool same = sid[i] == sid_copy[i];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const f4 a = f[k][i];
        const d4 b = d[k][i];
        same = same && a.x == (float)b.x && a.y == (float)b.y && a.z == (float)b.z && a.w == (float)b.w;
    }
    if (!same) *differ = 1;
}

// Is the neighbour list of an earlier dem_step call still good for these positions and shape ids?  Raises *stale when a
// particle is farther than skin/2 from where it was at the build (the criterion of the step loop) or a shape id changed.
static __global__ void k_list_valid(int n, BoxDev box, const d4* __restrict__ pos, const d4* __restrict__ pos_build,
                                    const int* __restrict__ sid, const int* __restrict__ sid_build, double half_skin2,
                                    int* __restrict__ stale) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const d4 x = pos[i], xb = pos_build[i];
    double dx = x.x - xb.x, dy = x.y - xb.y, dz = box.dim == 3 ? x.z - xb.z : 0.0;
    dx -= box.L[0] * rint(dx * box.invL[0]);
    dy -= box.L[1] * rint(dy * box.invL[1]);
    dz -= box.L[2] * rint(dz * box.invL[2]);
    if (!(dx * dx + dy * dy + dz * dz <= half_skin2) || sid[i] != sid_build[i]) *stale = 1;
}

// ---- precision conversion of state arrays (DEM_F32 contexts integrate in double, R15b) --------------------------------
__global__ void k_f4_to_d4(int n, const f4* __restrict__ in, d4* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const f4 v = in[i];
    d4 r;
    r.x = v.x; r.y = v.y; r.z = v.z; r.w = v.w;
    out[i] = r;
}
__global__ void k_d4_to_f4(int n, const d4* __restrict__ in, f4* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const d4 v = in[i];
    f4 r;
    r.x = (float)v.x; r.y = (float)v.y; r.z = (float)v.z; r.w = (float)v.w;
    out[i] = r;
}

}  // namespace dem
