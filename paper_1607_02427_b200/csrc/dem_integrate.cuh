// dem_integrate.cuh -- a9: the integrator kernels (velocity Verlet with quaternion rotation, Nose-Hoover thermostat,
// energies) and the precision conversion of the state.  Included by dem_lib.cu only.
#pragma once
#include "dem_kernels.cuh"

namespace dem {

// ---- a9: NVE integrator (reading R15) --------------------------------------------------------------------
__device__ __forceinline__ void quat_mul_d(const double* a, const double* b, double* o) {
    o[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    o[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    o[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    o[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}

// Torque-free rotation over dt with the lab-frame angular momentum L held fixed.  Spherical tops (and 2D): exact,
// q <- exp(dt/2 L/I0) q.  Otherwise the symmetric splitting of the free-rotor Hamiltonian into rotations about the
// body axes x(dt/2) y(dt/2) z(dt) y(dt/2) x(dt/2) (the family of PAPER.md ref. 23).
__device__ inline void free_rotate(int dim, const double* I, const double* L, double dt, double* q) {
    const bool spherical = dim == 2 || (I[0] == I[1] && I[1] == I[2]);
    if (spherical) {
        const double I0 = I[2];
        if (!(I0 > 0.0)) return;
        // rotation by phi = |a| about a/|a| with a = (dt / 2 I0) L: rq = (cos phi, (sin phi / phi) a)
        const double h = 0.5 * dt / I0;
        const double a[3] = {h * L[0], h * L[1], h * L[2]};
        const double p2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2];
        double ch, sc;  // cos phi, sin phi / phi
        if (p2 < 0.0625) {  // Taylor series: next terms phi^12 / 12! and phi^12 / 13! are below 1.2e-16 here
            ch = 1.0 + p2 * (-1.0 / 2 + p2 * (1.0 / 24 + p2 * (-1.0 / 720 + p2 * (1.0 / 40320 + p2 * (-1.0 / 3628800)))));
            sc = 1.0 + p2 * (-1.0 / 6 + p2 * (1.0 / 120 + p2 * (-1.0 / 5040 + p2 * (1.0 / 362880 + p2 * (-1.0 / 39916800)))));
        } else {
            const double ph = sqrt(p2);
            double sh;
            sincos(ph, &sh, &ch);
            sc = sh / ph;
        }
        const double rq[4] = {ch, sc * a[0], sc * a[1], sc * a[2]};
        double o[4];
        quat_mul_d(rq, q, o);
        // |o| = |q| (1 + O(1e-16)): two Newton steps of 1/sqrt from 1 renormalise a q that is unit to float precision
        const double n2 = o[0] * o[0] + o[1] * o[1] + o[2] * o[2] + o[3] * o[3];
        double inv = 1.5 - 0.5 * n2;
        inv = inv * (1.5 - 0.5 * n2 * inv * inv);
        inv = inv * (1.5 - 0.5 * n2 * inv * inv);
        for (int k = 0; k < 4; ++k) q[k] = o[k] * inv;
        return;
    }
    double M[9], Lb[3];
    quat_to_mat<double>(q[0], q[1], q[2], q[3], M);
    for (int a = 0; a < 3; ++a) Lb[a] = M[a] * L[0] + M[3 + a] * L[1] + M[6 + a] * L[2];  // R^T L
    const int axis_seq[5] = {0, 1, 2, 1, 0};
    const double frac[5] = {0.5, 0.5, 1.0, 0.5, 0.5};
    for (int s = 0; s < 5; ++s) {
        const int a = axis_seq[s];
        if (!(I[a] > 0.0)) continue;
        const double phi = frac[s] * dt * Lb[a] / I[a];
        double sn, cs;
        sincos(phi, &sn, &cs);
        const int b = (a + 1) % 3, c = (a + 2) % 3;
        const double lb = cs * Lb[b] + sn * Lb[c], lc = -sn * Lb[b] + cs * Lb[c];
        Lb[b] = lb;
        Lb[c] = lc;
        double sh, ch;
        sincos(0.5 * phi, &sh, &ch);
        double rq[4] = {ch, 0, 0, 0}, o[4];
        rq[1 + a] = sh;
        quat_mul_d(q, rq, o);  // body-axis rotation composes on the right
        for (int k = 0; k < 4; ++k) q[k] = o[k];
    }
    const double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int k = 0; k < 4; ++k) q[k] /= n;
}

// first half of velocity Verlet: v += dt/2 F/m; x += dt v (wrapped); L += dt/2 tau; free rotation of q.
// Also raises moved[0] when a particle is farther than skin/2 from where it was at the last neighbour build.
// Does nothing once moved[1] (halt, raised by k_reduce of an earlier step of the same chunk) is set.
template <typename real>
__global__ void k_kick_drift(int N, BoxDev box, double dt, const int* __restrict__ sid, MassTable mt,
                             d4* __restrict__ pos, d4* __restrict__ quat, d4* __restrict__ vel, d4* __restrict__ ang,
                             const typename vec4<real>::type* __restrict__ force,
                             const typename vec4<real>::type* __restrict__ torque, const d4* __restrict__ pos_build,
                             double half_skin2, int* __restrict__ moved, const ThermoDev* __restrict__ thermo) {
    // The translational and the rotational half of a particle's update are independent: the first half of the grid
    // does x, v (and the skin test), the second q, L -- twice the memory-level parallelism, half the dependent chain.
    if (moved[1]) return;
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
        for (int a = 0; a < box.dim; ++a) {
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
        if (dx * dx + dy * dy + dz * dz > half_skin2) moved[0] = 1;
    } else {
        d4 L = ang[i], q = quat[i];
        const typename vec4<real>::type T = torque[i];
        double Ls[3] = {L.x * sc, L.y * sc, L.z * sc};
        const double Ts[3] = {(double)T.x, (double)T.y, (double)T.z};
        for (int a = (box.dim == 2 ? 2 : 0); a < 3; ++a) Ls[a] += 0.5 * dt * Ts[a];
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
// not completed (flags[1] = halt, see k_reduce).
__global__ void k_thermostat(int nb, const double* __restrict__ partial, int dim, int N, double dt, double kT,
                             double tau, int halves, const int* __restrict__ flags, ThermoDev* __restrict__ th) {
    __shared__ double sh[2][256];
    if (flags && flags[1]) return;
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
