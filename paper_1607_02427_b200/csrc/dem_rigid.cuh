// dem_rigid.cuh -- torque-free rotation of a rigid body over one time step (reading R15), used by the
// integrator kernels (dem_integrate.cuh) and by the fused reduction + integration kernel (dem_kernels.cuh: k_finish).
#pragma once
#include "dem_math.cuh"

namespace dem {

__device__ __forceinline__ void quat_mul_d(const double* a, const double* b, double* o) {
    o[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    o[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    o[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    o[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}

// Torque-free rotation over dt with the lab-frame angular momentum L held fixed.  Spherical tops (and 2D): exact,
// q <- exp(dt/2 L/I0) q.  Otherwise the symmetric splitting of the free-rotor Hamiltonian into rotations about the
// body axes x(dt/2) y(dt/2) z(dt) y(dt/2) x(dt/2) (the family of PAPER.md ref. 23).
__device__ __forceinline__ void free_rotate(int dim, const double* I, const double* L, double dt, double* q) {
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
#pragma unroll
        for (int k = 0; k < 4; ++k) q[k] = o[k] * inv;
        return;
    }
    double M[9], Lb[3];
    quat_to_mat<double>(q[0], q[1], q[2], q[3], M);
#pragma unroll
    for (int a = 0; a < 3; ++a) Lb[a] = M[a] * L[0] + M[3 + a] * L[1] + M[6 + a] * L[2];  // R^T L
    // (unrolled with compile-time axes: every array index is static, so that L_b and q stay in registers)
#pragma unroll
    for (int s = 0; s < 5; ++s) {
        const int a = s < 3 ? s : 4 - s;  // x y z y x
        const double fr = s == 2 ? 1.0 : 0.5;
        if (!(I[a] > 0.0)) continue;
        const double phi = fr * dt * Lb[a] / I[a];
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
#pragma unroll
        for (int k = 0; k < 4; ++k) q[k] = o[k];
    }
    const double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
#pragma unroll
    for (int k = 0; k < 4; ++k) q[k] /= n;
}

}  // namespace dem
