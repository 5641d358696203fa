// dem_math.cuh -- per-pair feature arithmetic of the DEM force field (arXiv:1607.02427), templated on `real`.
//
// Everything here is the arithmetic of ONE unique particle pair (i, j): every Eq. 1 (3D) or Eq. 2
// (2D) term, its nearest-point distance r* (PAPER.md:35, 45), WCA (Eq. 3-4) for the
// rare terms inside the cutoff, force along the line between the nearest points and torque from the interaction
// point, the near-parallel edge rule (R5).
//
// Frames.  All of it runs in particle i's BODY frame: j is brought in with R = R_i^T R_j and t = R_i^T d_ij, so i's
// features are the constant shape table (warp-uniform shared-memory broadcasts) and j's features are rotated on the
// fly into registers.  The third sum of Eq. 1 (vertices of i against faces of j) runs in j's body frame for the same
// reason and its rare active terms are rotated back.  The result (F, T, u) is in i's frame; the kernel rotates it to
// the lab frame once per pair.
//
// Device code only: the library calls these from its kernels and nothing else does (there is no CPU path in the
// product, and the oracle shares no code with this file).
#pragma once
#include <math.h>
#include <stdint.h>

#include "dem_types.h"

#if !defined(__CUDACC__)
#error "dem_math.cuh is device code: compile it with nvcc"
#endif
#define DEM_HD __device__ __forceinline__
#define DEM_HD_NOINLINE __device__ __noinline__

namespace dem {

// ---- scalar helpers ---------------------------------------------------------------------------------------------
DEM_HD float rmin(float a, float b) { return fminf(a, b); }
DEM_HD double rmin(double a, double b) { return fmin(a, b); }
DEM_HD float rmax(float a, float b) { return fmaxf(a, b); }
DEM_HD double rmax(double a, double b) { return fmax(a, b); }
DEM_HD float sat01(float x) {
#ifdef __CUDA_ARCH__
    return __saturatef(x);
#else
    return fminf(fmaxf(x, 0.f), 1.f);
#endif
}
DEM_HD double sat01(double x) { return fmin(fmax(x, 0.0), 1.0); }
// reciprocal: MUFU.RCP (1 ulp) in FP32 on the device -- the closest-point parameters are clamped and second-order
// in their error; IEEE division in FP64.
DEM_HD float rcp(float x) {
#ifdef __CUDA_ARCH__
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
#else
    return 1.f / x;
#endif
}
DEM_HD double rcp(double x) { return 1.0 / x; }

// ---- shape table view --------------------------------------------------------------------------------------------
// One shape = one block of real4 records; the pair kernel stages the blocks of the
// two shapes of its class into shared memory and builds these views over them.
//   V [nv]      (x, y, z, 0)                                   body-frame vertex
//   E [2 ne]    3D: [2k] = (a.xyz, |e|^2)  [2k+1] = (e.xyz, 1/|e|^2 or 0 if |e| = 0)      edge k = a + s e, s in [0,1]
//               2D: [2k] = (a.x, a.y, u.x, u.y)  [2k+1] = (|e|, cs, cm, |e|/2)              u = e/|e| ((1,0) if |e| = 0)
//                   cs = -(u x a), cm = -(u . a) - |e|/2: for a point q, side = u x q + cs and u . q + cm is the
//                   along-edge coordinate measured from the edge's midpoint
//   F [4 nf]    [4f] = (uhat, -uhat.o) [4f+1] = (vhat, -vhat.o) [4f+2] = (nhat, -nhat.o) [4f+3] = (first FE, count, 0, 0)
//   FE[2 nfe]   face boundary edges in the face's (uhat, vhat) coordinates, CCW about nhat: same layout as 2D edges
//   OE[2 ne]    3D only: [2k] = (a.xyz, |e|)  [2k+1] = (e/|e|, 0): the edges as the search kernel's outer features
//   EB[ne]      3D only: (midpoint, half length) of every edge;   FB[nf]  3D only: (centre, radius) of a sphere around every face
template <typename real> struct ShapeView {
    typedef typename vec4<real>::type real4;
    int nv, ne, nf;
    const real4* V;
    const real4* E;
    const real4* F;
    const real4* FE;
    const real4* OE;
    const real4* EB;  // 3D: bounding spheres of the edges (midpoint, half length) ...
    const real4* FB;  // ... and of the faces (centre, radius): OE + 2 ne, EB + ne
};

template <typename real> struct PairAcc {
    real F[3], T[3], u;  // force on i, torque on i about x_i (i's body frame), pair energy U_ij
    unsigned nactive, ndegen, npar;
};

// WCA for one term inside the cutoff; ci = interaction point on i (i frame, relative to x_i), del = c_i - c_j.
// u = 4 eps (s^12 - s^6) + eps, F = (24 eps (2 s^12 - s^6) / r^2) del: no square root is needed anywhere.
template <typename real>
DEM_HD void wca_accumulate(const PairConst<real>& pc, PairAcc<real>& acc, real cix, real ciy, real ciz, real dx,
                           real dy, real dz, real r2, bool parallel) {
    if (r2 < pc.degen2) {
        acc.ndegen++;
        return;
    }
    acc.nactive++;
    if (parallel) acc.npar++;
    const real ir2 = real(1) / r2;
    const real s2 = pc.sig2 * ir2;
    const real s6 = s2 * s2 * s2;
    acc.u += real(4) * pc.eps * (s6 * s6 - s6) + pc.eps;
    const real fr = real(24) * pc.eps * (real(2) * s6 * s6 - s6) * ir2;
    const real fx = fr * dx, fy = fr * dy, fz = fr * dz;
    acc.F[0] += fx;
    acc.F[1] += fy;
    acc.F[2] += fz;
    acc.T[0] += ciy * fz - ciz * fy;
    acc.T[1] += ciz * fx - cix * fz;
    acc.T[2] += cix * fy - ciy * fx;
}

// ---- 2D: point against one edge record (also the in-plane part of point-face) ---------------------------------------
// q = point, (ax, ay) edge start, (ux, uy) unit direction, len.  Returns squared distance; (ddx, ddy) = q - c.
template <typename real>
DEM_HD real point_edge2(real qx, real qy, real ax, real ay, real ux, real uy, real len, real& ddx, real& ddy) {
    const real wx = qx - ax, wy = qy - ay;
    const real tt = rmin(rmax(wx * ux + wy * uy, real(0)), len);
    ddx = wx - tt * ux;
    ddy = wy - tt * uy;
    return ddx * ddx + ddy * ddy;
}

// ---- 3D: point against a closed planar convex polygon face (R1/R2: interior and boundary) ----------------------------
// Hot form: squared distance only.  (x, y, h) = coordinates of the point in the face's (uhat, vhat, nhat) frame.
template <typename real>
DEM_HD real point_face_r2(const ShapeView<real>& S, int f, real px, real py, real pz) {
    typedef typename vec4<real>::type real4;
    const real4 f0 = S.F[4 * f], f1 = S.F[4 * f + 1], f2 = S.F[4 * f + 2], f3 = S.F[4 * f + 3];
    const real x = f0.x * px + f0.y * py + f0.z * pz + f0.w;
    const real y = f1.x * px + f1.y * py + f1.z * pz + f1.w;
    const real h = f2.x * px + f2.y * py + f2.z * pz + f2.w;
    const int m0 = (int)f3.x, m1 = m0 + (int)f3.y;
    real smin = real(1e30), dmin = real(1e30);
    for (int m = m0; m < m1; ++m) {
        const real4 e0 = S.FE[2 * m];
        const real len = S.FE[2 * m + 1].x;
        const real wx = x - e0.x, wy = y - e0.y;
        smin = rmin(smin, e0.z * wy - e0.w * wx);  // >= 0 on the inner side of this boundary edge
        const real tt = rmin(rmax(wx * e0.z + wy * e0.w, real(0)), len);
        const real ddx = wx - tt * e0.z, ddy = wy - tt * e0.w;
        dmin = rmin(dmin, ddx * ddx + ddy * ddy);
    }
    return h * h + (smin >= real(0) ? real(0) : dmin);
}

// Rare form: the vector del = p - c (face-owner frame) from the point's nearest point c on the face.
template <typename real>
DEM_HD_NOINLINE void point_face_del(const ShapeView<real>& S, int f, real px, real py, real pz, real& dx, real& dy,
                                    real& dz) {
    typedef typename vec4<real>::type real4;
    const real4 f0 = S.F[4 * f], f1 = S.F[4 * f + 1], f2 = S.F[4 * f + 2], f3 = S.F[4 * f + 3];
    const real x = f0.x * px + f0.y * py + f0.z * pz + f0.w;
    const real y = f1.x * px + f1.y * py + f1.z * pz + f1.w;
    const real h = f2.x * px + f2.y * py + f2.z * pz + f2.w;
    const int m0 = (int)f3.x, m1 = m0 + (int)f3.y;
    real smin = real(1e30), dmin = real(1e30), bx = 0, by = 0;
    for (int m = m0; m < m1; ++m) {
        const real4 e0 = S.FE[2 * m];
        const real len = S.FE[2 * m + 1].x;
        smin = rmin(smin, e0.z * (y - e0.y) - e0.w * (x - e0.x));
        real ddx, ddy;
        const real d2 = point_edge2(x, y, e0.x, e0.y, e0.z, e0.w, len, ddx, ddy);
        if (d2 < dmin) {
            dmin = d2;
            bx = ddx;
            by = ddy;
        }
    }
    if (smin >= real(0)) bx = by = real(0);
    dx = h * f2.x + bx * f0.x + by * f1.x;
    dy = h * f2.y + bx * f0.y + by * f1.y;
    dz = h * f2.z + bx * f0.z + by * f1.z;
}

// ---- 3D: segment-segment, everything that is not the generic skew case (rare) ------------------------------------------
// Near-parallel rule (PAPER.md:59 as read in R5), zero-length edges (degenerate shapes), exactly parallel edges.
// r = p1 - p2.  Returns true if the parallel-midpoint branch was taken.
template <typename real>
DEM_HD_NOINLINE bool segseg_special(real rx, real ry, real rz, real d1x, real d1y, real d1z, real a, real d2x, real d2y,
                                    real d2z, real e, real nn, real eps_par, real& s, real& t) {
    const real c = d1x * rx + d1y * ry + d1z * rz;  // d1 . r
    const real f = d2x * rx + d2y * ry + d2z * rz;  // d2 . r
    if (a <= real(0) && e <= real(0)) {
        s = t = real(0);
        return false;
    }
    if (a <= real(0)) {
        s = real(0);
        t = sat01(f / e);
        return false;
    }
    if (e <= real(0)) {
        t = real(0);
        s = sat01(-c / a);
        return false;
    }
    const real b = d1x * d2x + d1y * d2y + d1z * d2z;
    if (nn < eps_par * a * e) {
        // parameters of segment 2's end points along line 1 and of segment 1's end points along line 2
        const real s_a = -c / a, s_b = (b - c) / a;
        const real t_a = f / e, t_b = (b + f) / e;
        const real slo = rmax(real(0), rmin(s_a, s_b)), shi = rmin(real(1), rmax(s_a, s_b));
        const real tlo = rmax(real(0), rmin(t_a, t_b)), thi = rmin(real(1), rmax(t_a, t_b));
        if (shi > slo && thi > tlo) {
            s = real(0.5) * (slo + shi);
            t = real(0.5) * (tlo + thi);
            return true;
        }
    }
    if (nn > real(0)) {
        const real nx = d1y * d2z - d1z * d2y, ny = d1z * d2x - d1x * d2z, nz = d1x * d2y - d1y * d2x;
        const real qx = ry * d2z - rz * d2y, qy = rz * d2x - rx * d2z, qz = rx * d2y - ry * d2x;
        s = sat01(-(nx * qx + ny * qy + nz * qz) / nn);
    } else {
        s = real(0);
    }
    t = (b * s + f) / e;
    if (t < real(0)) {
        t = real(0);
        s = sat01(-c / a);
    } else if (t > real(1)) {
        t = real(1);
        s = sat01((b - c) / a);
    }
    return false;
}

// ---- single Eq. 1 / Eq. 2 terms -------------------------------------------------------------------------------------
// One term each, with the outer feature already brought into the frame of the inner feature's owner.  The pair loops
// below call them for every term; the FP32 search kernel (dem_fast.cuh) calls them only for the terms its packed
// search flags as candidates, so both paths share the arithmetic of every contributing term.

// edge (p2, d2, e = |d2|^2, inv_e) of j in i's frame against edge k of i (first sum of Eq. 1)
// (geometry of the term: true when it is inside the cutoff; ci = the interaction point on i, del = c_i - c_j, r2 and the
// parallel flag then hold what wca_accumulate wants.  term_ee = this + wca_accumulate; the search kernels call the two
// halves separately so that all term kinds share one copy of the WCA code)
template <typename real>
DEM_HD bool term_ee_geom(const ShapeView<real>& A, int k, real p2x, real p2y, real p2z, real d2x, real d2y, real d2z, real e,
                         real inv_e, const PairConst<real>& pc, real* ci, real* del, real& r2_out, bool& par_out) {
    typedef typename vec4<real>::type real4;
    const real4 a0 = A.E[2 * k], a1 = A.E[2 * k + 1];
    const real rx = a0.x - p2x, ry = a0.y - p2y, rz = a0.z - p2z;  // r = p1 - p2
    const real nx = a1.y * d2z - a1.z * d2y, ny = a1.z * d2x - a1.x * d2z, nz = a1.x * d2y - a1.y * d2x;
    const real nn = nx * nx + ny * ny + nz * nz;
    real s, tt;
    bool par = false;
    if (nn <= pc.eps_par * e * a0.w) {
        par = segseg_special<real>(rx, ry, rz, a1.x, a1.y, a1.z, a0.w, d2x, d2y, d2z, e, nn, pc.eps_par, s, tt);
    } else {
        // skew lines: s = -(d1 x d2).(r x d2) / |d1 x d2|^2 (no cancellation near parallel), then the textbook
        // clamp cascade written branch-free
        const real qx = ry * d2z - rz * d2y, qy = rz * d2x - rx * d2z, qz = rx * d2y - ry * d2x;
        s = sat01(-(nx * qx + ny * qy + nz * qz) * rcp(nn));
        const real b = a1.x * d2x + a1.y * d2y + a1.z * d2z;
        const real f = d2x * rx + d2y * ry + d2z * rz;
        const real c = a1.x * rx + a1.y * ry + a1.z * rz;
        const real tu = (b * s + f) * inv_e;
        tt = sat01(tu);
        const real s2 = sat01((b * tt - c) * a1.w);
        s = (tu != tt) ? s2 : s;
    }
    const real dx = rx + s * a1.x - tt * d2x, dy = ry + s * a1.y - tt * d2y, dz = rz + s * a1.z - tt * d2z;
    const real r2 = dx * dx + dy * dy + dz * dz;
    if (!(r2 < pc.rc2)) return false;
    ci[0] = a0.x + s * a1.x; ci[1] = a0.y + s * a1.y; ci[2] = a0.z + s * a1.z;
    del[0] = dx; del[1] = dy; del[2] = dz;
    r2_out = r2;
    par_out = par;
    return true;
}
template <typename real>
DEM_HD void term_ee(const ShapeView<real>& A, int k, real p2x, real p2y, real p2z, real d2x, real d2y, real d2z, real e,
                    real inv_e, const PairConst<real>& pc, PairAcc<real>& acc) {
    real ci[3], del[3], r2;
    bool par;
    if (term_ee_geom<real>(A, k, p2x, p2y, p2z, d2x, d2y, d2z, e, inv_e, pc, ci, del, r2, par))
        wca_accumulate<real>(pc, acc, ci[0], ci[1], ci[2], del[0], del[1], del[2], r2, par);
}

// vertex p of j (in i's frame) against face f of i (third sum of Eq. 1)
template <typename real>
DEM_HD void term_vf_own(const ShapeView<real>& A, int f, real px, real py, real pz, const PairConst<real>& pc,
                        PairAcc<real>& acc) {
    const real r2 = point_face_r2<real>(A, f, px, py, pz);
    if (r2 < pc.rc2) {
        real dx, dy, dz;  // p - c with c on i's face: c_i = c, c_j = p, del = c_i - c_j = -(p - c)
        point_face_del<real>(A, f, px, py, pz, dx, dy, dz);
        wca_accumulate<real>(pc, acc, px - dx, py - dy, pz - dz, -dx, -dy, -dz, r2, false);
    }
}

// vertex v of i (body frame; p = R^T (v - t) is the same vertex in j's frame) against face f of j (second sum of Eq. 1)
template <typename real>
DEM_HD void term_vf_other(const ShapeView<real>& B, int f, real vx, real vy, real vz, real px, real py, real pz,
                          const real* R, const PairConst<real>& pc, PairAcc<real>& acc) {
    const real r2 = point_face_r2<real>(B, f, px, py, pz);
    if (r2 < pc.rc2) {
        real dx, dy, dz;  // p' - c' in j's frame; c_i = the vertex, del = c_i - c_j = R (p' - c')
        point_face_del<real>(B, f, px, py, pz, dx, dy, dz);
        wca_accumulate<real>(pc, acc, vx, vy, vz, R[0] * dx + R[1] * dy + R[2] * dz, R[3] * dx + R[4] * dy + R[5] * dz,
                             R[6] * dx + R[7] * dy + R[8] * dz, r2, false);
    }
}

// 2D: vertex p of j (i's frame) against edge k of i
template <typename real>
DEM_HD void term_ve_own(const ShapeView<real>& A, int k, real px, real py, const PairConst<real>& pc,
                        PairAcc<real>& acc) {
    typedef typename vec4<real>::type real4;
    const real4 e0 = A.E[2 * k];
    const real len = A.E[2 * k + 1].x;
    real ddx, ddy;
    const real r2 = point_edge2<real>(px, py, e0.x, e0.y, e0.z, e0.w, len, ddx, ddy);
    if (r2 < pc.rc2)  // c_i = p - dd on i's edge, c_j = p, del = -dd
        wca_accumulate<real>(pc, acc, px - ddx, py - ddy, real(0), -ddx, -ddy, real(0), r2, false);
}

// 2D: vertex v of i (p = the same vertex in j's frame) against edge l of j
template <typename real>
DEM_HD void term_ve_other(const ShapeView<real>& B, int l, real vx, real vy, real px, real py, const real* R,
                          const PairConst<real>& pc, PairAcc<real>& acc) {
    typedef typename vec4<real>::type real4;
    const real4 e0 = B.E[2 * l];
    const real len = B.E[2 * l + 1].x;
    real ddx, ddy;
    const real r2 = point_edge2<real>(px, py, e0.x, e0.y, e0.z, e0.w, len, ddx, ddy);
    if (r2 < pc.rc2)  // c_i = the vertex, del = c_i - c_j = R dd
        wca_accumulate<real>(pc, acc, vx, vy, real(0), R[0] * ddx + R[1] * ddy, R[3] * ddx + R[4] * ddy, real(0), r2,
                             false);
}

// outer features of a pair brought into the frame of the inner feature's owner
template <typename real>
DEM_HD void edge_to_i(const ShapeView<real>& B, int l, const real* R, const real* t, real* p2, real* d2, real& e,
                      real& inv_e) {
    typedef typename vec4<real>::type real4;
    const real4 b0 = B.E[2 * l], b1 = B.E[2 * l + 1];
    p2[0] = R[0] * b0.x + R[1] * b0.y + R[2] * b0.z + t[0];
    p2[1] = R[3] * b0.x + R[4] * b0.y + R[5] * b0.z + t[1];
    p2[2] = R[6] * b0.x + R[7] * b0.y + R[8] * b0.z + t[2];
    d2[0] = R[0] * b1.x + R[1] * b1.y + R[2] * b1.z;
    d2[1] = R[3] * b1.x + R[4] * b1.y + R[5] * b1.z;
    d2[2] = R[6] * b1.x + R[7] * b1.y + R[8] * b1.z;
    e = b0.w;
    inv_e = b1.w;
}
template <typename real> DEM_HD void vertex_to_i(real vx, real vy, real vz, const real* R, const real* t, real* p) {
    p[0] = R[0] * vx + R[1] * vy + R[2] * vz + t[0];
    p[1] = R[3] * vx + R[4] * vy + R[5] * vz + t[1];
    p[2] = R[6] * vx + R[7] * vy + R[8] * vz + t[2];
}
template <typename real> DEM_HD void vertex_to_j(real vx, real vy, real vz, const real* R, const real* t, real* p) {
    const real wx = vx - t[0], wy = vy - t[1], wz = vz - t[2];  // p' = R^T (v - t)
    p[0] = R[0] * wx + R[3] * wy + R[6] * wz;
    p[1] = R[1] * wx + R[4] * wy + R[7] * wz;
    p[2] = R[2] * wx + R[5] * wy + R[8] * wz;
}

// ---- the pair: 3D --------------------------------------------------------------------------------------------------
// A = shape of i (its body frame is the working frame), B = shape of j.  R (row-major 3x3) and t bring j's body
// coordinates into i's frame: p_i = R v_j + t.  [o_begin, o_end) selects a slice of the flattened outer loop
// (E_j edges, then V_j vertices, then V_i vertices) so that several lanes can share one heavy pair.
template <typename real>
DEM_HD void pair_eval_3d(const ShapeView<real>& A, const ShapeView<real>& B, const real* R, const real* t,
                         const PairConst<real>& pc, int o_begin, int o_end, PairAcc<real>& acc) {
    typedef typename vec4<real>::type real4;
    const int oE = B.ne, oV = B.ne + B.nv;
    // (1) first sum of Eq. 1: every edge of i against every edge of j
    for (int l = o_begin; l < o_end && l < oE; ++l) {
        real p2[3], d2[3], e, inv_e;
        edge_to_i<real>(B, l, R, t, p2, d2, e, inv_e);
        for (int k = 0; k < A.ne; ++k) term_ee<real>(A, k, p2[0], p2[1], p2[2], d2[0], d2[1], d2[2], e, inv_e, pc, acc);
    }
    // (2) third sum of Eq. 1: every vertex of j against every face of i (i's frame)
    for (int o = (o_begin > oE ? o_begin : oE); o < o_end && o < oV; ++o) {
        const real4 v = B.V[o - oE];
        real p[3];
        vertex_to_i<real>(v.x, v.y, v.z, R, t, p);
        for (int f = 0; f < A.nf; ++f) term_vf_own<real>(A, f, p[0], p[1], p[2], pc, acc);
    }
    // (3) second sum of Eq. 1: every vertex of i against every face of j, in j's frame
    for (int o = (o_begin > oV ? o_begin : oV); o < o_end && o < oV + A.nv; ++o) {
        const real4 v = A.V[o - oV];
        real p[3];
        vertex_to_j<real>(v.x, v.y, v.z, R, t, p);
        for (int f = 0; f < B.nf; ++f) term_vf_other<real>(B, f, v.x, v.y, v.z, p[0], p[1], p[2], R, pc, acc);
    }
}

// ---- the pair: 2D --------------------------------------------------------------------------------------------------
// Flattened outer loop: V_j vertices (against edges of i, i's frame), then V_i vertices (against edges of j, j's frame).
template <typename real>
DEM_HD void pair_eval_2d(const ShapeView<real>& A, const ShapeView<real>& B, const real* R, const real* t,
                         const PairConst<real>& pc, int o_begin, int o_end, PairAcc<real>& acc) {
    typedef typename vec4<real>::type real4;
    const int oV = B.nv;
    for (int l = o_begin; l < o_end && l < oV; ++l) {
        const real4 v = B.V[l];
        real p[3];
        vertex_to_i<real>(v.x, v.y, real(0), R, t, p);
        for (int k = 0; k < A.ne; ++k) term_ve_own<real>(A, k, p[0], p[1], pc, acc);
    }
    for (int o = (o_begin > oV ? o_begin : oV); o < o_end && o < oV + A.nv; ++o) {
        const real4 v = A.V[o - oV];
        real p[3];
        vertex_to_j<real>(v.x, v.y, real(0), R, t, p);
        for (int l = 0; l < B.ne; ++l) term_ve_other<real>(B, l, v.x, v.y, p[0], p[1], R, pc, acc);
    }
}

// rotation matrix (row-major) of a unit quaternion (w, x, y, z): v_lab = M v_body
template <typename real> DEM_HD void quat_to_mat(real w, real x, real y, real z, real* M) {
    M[0] = real(1) - real(2) * (y * y + z * z);
    M[1] = real(2) * (x * y - w * z);
    M[2] = real(2) * (x * z + w * y);
    M[3] = real(2) * (x * y + w * z);
    M[4] = real(1) - real(2) * (x * x + z * z);
    M[5] = real(2) * (y * z - w * x);
    M[6] = real(2) * (x * z - w * y);
    M[7] = real(2) * (y * z + w * x);
    M[8] = real(1) - real(2) * (x * x + y * y);
}

// One unique pair, lab frame in and out: q_i, q_j unit quaternions, d = minimum-image x_j - x_i (lab), all given in
// double: the relative pose R = R_i^T R_j, t = R_i^T d is formed in FP64 and rounded ONCE to `real`, so that an FP32
// run starts its 10^2..10^4 feature terms from correctly rounded coordinates (~100 FP64
// operations per pair against >= 600 FP32 instructions of feature work).
// out[0..2] = force on i, out[3..5] = torque on i, out[6..8] = torque on j (all lab frame), out[9] = U_ij.
// The force on j is -out[0..2].  tau_j = -sum c_j x F + d x sum F, and c_j x F = c_i x F because F is along c_i - c_j.
// relative pose of a pair: Mi = R_i, R = R_i^T R_j, t = R_i^T d, formed in FP64 and rounded ONCE to `real`
template <typename real>
DEM_HD void pair_pose(const double* qi, const double* qj, const double* d, real* Mi, real* R, real* t) {
    double Di[9], Dj[9];
    quat_to_mat<double>(qi[0], qi[1], qi[2], qi[3], Di);
    quat_to_mat<double>(qj[0], qj[1], qj[2], qj[3], Dj);
#pragma unroll
    for (int r = 0; r < 3; ++r) {
#pragma unroll
        for (int c = 0; c < 3; ++c)
            R[3 * r + c] = (real)(Di[r] * Dj[c] + Di[3 + r] * Dj[3 + c] + Di[6 + r] * Dj[6 + c]);
        t[r] = (real)(Di[r] * d[0] + Di[3 + r] * d[1] + Di[6 + r] * d[2]);
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) Mi[k] = (real)Di[k];
}

// (F, T, u) of a pair in i's frame -> out[0..2] = force on i, out[3..5] = torque on i, out[6..8] = torque on j (all lab
// frame), out[9] = U_ij.  The force on j is -out[0..2].  tau_j = -sum c_j x F + d x sum F, and c_j x F = c_i x F
// because F is along c_i - c_j.
template <typename real>
DEM_HD void pair_finish(const real* Mi, const real* t, const real* F, const real* T, real u, real* out) {
    const real tjx = -T[0] + (t[1] * F[2] - t[2] * F[1]);
    const real tjy = -T[1] + (t[2] * F[0] - t[0] * F[2]);
    const real tjz = -T[2] + (t[0] * F[1] - t[1] * F[0]);
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        out[r] = Mi[3 * r] * F[0] + Mi[3 * r + 1] * F[1] + Mi[3 * r + 2] * F[2];
        out[3 + r] = Mi[3 * r] * T[0] + Mi[3 * r + 1] * T[1] + Mi[3 * r + 2] * T[2];
        out[6 + r] = Mi[3 * r] * tjx + Mi[3 * r + 1] * tjy + Mi[3 * r + 2] * tjz;
    }
    out[9] = u;
}

template <typename real, int DIM>
DEM_HD void pair_lab(const ShapeView<real>& A, const ShapeView<real>& B, const double* qi, const double* qj,
                     const double* d, const PairConst<real>& pc, int o_begin, int o_end, real* out, unsigned* cnt) {
    real Mi[9], R[9], t[3];
    pair_pose<real>(qi, qj, d, Mi, R, t);
    PairAcc<real> acc;
    acc.F[0] = acc.F[1] = acc.F[2] = acc.T[0] = acc.T[1] = acc.T[2] = acc.u = real(0);
    acc.nactive = acc.ndegen = acc.npar = 0u;
    if (DIM == 3)
        pair_eval_3d<real>(A, B, R, t, pc, o_begin, o_end, acc);
    else
        pair_eval_2d<real>(A, B, R, t, pc, o_begin, o_end, acc);
    pair_finish<real>(Mi, t, acc.F, acc.T, acc.u, out);
    cnt[0] = acc.nactive;
    cnt[1] = acc.ndegen;
    cnt[2] = acc.npar;
}

}  // namespace dem
