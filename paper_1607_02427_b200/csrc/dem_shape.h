// dem_shape.h -- host-side shape validation and construction of the shape-feature table (step a1 of DESIGN.md).
//
// A shape is the paper's inner polygon / polyhedron: vertices V, edges E, planar faces F, rounded by a disk / sphere of
// radius rho = sigma/2.  From the caller's description this file derives what the pair kernel
// wants to find in shared memory (layout documented at dem::ShapeView in dem_math.cuh): per-edge start / direction /
// squared length / reciprocal, and per face an orthonormal in-plane frame plus the boundary edges expressed in that
// frame, so that point-face is one 3x3 projection and a few 2D point-segment tests.
#pragma once
#include <algorithm>
#include <cmath>
#include <set>
#include <string>
#include <utility>
#include <vector>

namespace dem {

struct HostShape {
    int dim = 3;
    int nv = 0, ne = 0, nf = 0, nfe = 0;
    std::vector<double> verts;   // nv x 3
    std::vector<int> edges;      // ne x 2
    std::vector<int> face_off;   // nf + 1
    std::vector<int> face_verts;
    double rounding = 0, mass = 1, inertia[3] = {1, 1, 1}, circumradius = 0;
    // flattened table in double, in units of 4 doubles: V (nv) | E (2 ne) | F (4 nf) | FE (2 nfe) | OE (2 ne) | EB (ne) | FB (nf)
    // (OE, EB, FB in 3D only)
    std::vector<double> table;
    std::vector<std::pair<int, int>> face_groups;  // runs of faces with the same number of boundary edges
    double max_edge = 0;  // longest edge (bounds the search kernel's near-parallel slack)
    int table_len4() const { return nv + 2 * ne + 4 * nf + 2 * nfe + (dim == 3 ? 2 * ne + ne + nf : 0); }
};

inline void push4(std::vector<double>& t, double a, double b, double c, double d) {
    t.push_back(a);
    t.push_back(b);
    t.push_back(c);
    t.push_back(d);
}

// Returns "" on success, else a description of what is wrong with the shape.
inline std::string build_host_shape(HostShape& S, int dim, const double* verts, int nv, const int* face_offsets,
                                    const int* face_verts, int nf, const int* edges, int ne, double rounding,
                                    double mass, const double inertia[3]) {
    if (nv < 1) return "shape needs at least one vertex";
    if (!(rounding > 0.0)) return "rounding radius must be positive";
    if (dim == 2 && nf != 0) return "2D shapes have no faces";
    if (nf < 0 || (nf > 0 && (!face_offsets || !face_verts))) return "bad face arrays";
    S.dim = dim;
    S.nv = nv;
    S.verts.assign(verts, verts + 3 * (size_t)nv);
    if (dim == 2)
        for (int k = 0; k < nv; ++k) S.verts[3 * k + 2] = 0.0;
    S.rounding = rounding;
    S.mass = mass;
    for (int a = 0; a < 3; ++a) S.inertia[a] = inertia ? inertia[a] : 1.0;
    double r2 = 0;
    for (int k = 0; k < nv; ++k) {
        const double* v = &S.verts[3 * k];
        r2 = std::max(r2, v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    }
    S.circumradius = std::sqrt(r2);
    // faces
    S.nf = nf;
    S.face_off.assign(1, 0);
    S.face_verts.clear();
    for (int f = 0; f < nf; ++f) {
        const int b = face_offsets[f], e = face_offsets[f + 1];
        if (e - b < 3) return "a face needs at least 3 vertices";
        for (int m = b; m < e; ++m) {
            if (face_verts[m] < 0 || face_verts[m] >= nv) return "face vertex index out of range";
            S.face_verts.push_back(face_verts[m]);
        }
        S.face_off.push_back((int)S.face_verts.size());
    }
    // faces are kept sorted by vertex count (stable), so that the search kernel sweeps runs of equal-sized faces with
    // unrolled code; the order of faces has no meaning in the method (Eq. 1 sums over all of them)
    {
        std::vector<int> idx(nf);
        for (int f = 0; f < nf; ++f) idx[f] = f;
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) {
            return S.face_off[a + 1] - S.face_off[a] < S.face_off[b + 1] - S.face_off[b];
        });
        std::vector<int> off(1, 0), fv;
        for (int f : idx) {
            for (int m = S.face_off[f]; m < S.face_off[f + 1]; ++m) fv.push_back(S.face_verts[m]);
            off.push_back((int)fv.size());
        }
        S.face_off.swap(off);
        S.face_verts.swap(fv);
        S.face_groups.clear();  // (vertex count, number of faces) runs
        for (int f = 0; f < nf; ++f) {
            const int n = S.face_off[f + 1] - S.face_off[f];
            if (S.face_groups.empty() || S.face_groups.back().first != n) S.face_groups.push_back({n, 0});
            S.face_groups.back().second++;
        }
    }
    // edges: explicit, or derived (2D: closed CCW polygon; 3D: unique boundary edges of the faces)
    S.edges.clear();
    if (edges) {
        if (ne < 0) return "bad edge count";
        for (int k = 0; k < 2 * ne; ++k) {
            if (edges[k] < 0 || edges[k] >= nv) return "edge vertex index out of range";
            S.edges.push_back(edges[k]);
        }
    } else if (dim == 2) {
        if (nv == 1) {
            S.edges = {0, 0};
        } else if (nv == 2) {
            S.edges = {0, 1};
        } else {
            for (int k = 0; k < nv; ++k) {
                S.edges.push_back(k);
                S.edges.push_back((k + 1) % nv);
            }
        }
    } else {
        std::set<std::pair<int, int>> es;
        for (int f = 0; f < nf; ++f) {
            const int b = S.face_off[f], n = S.face_off[f + 1] - b;
            for (int m = 0; m < n; ++m) {
                const int u = S.face_verts[b + m], w = S.face_verts[b + (m + 1) % n];
                es.insert({std::min(u, w), std::max(u, w)});
            }
        }
        for (auto& p : es) {
            S.edges.push_back(p.first);
            S.edges.push_back(p.second);
        }
    }
    S.ne = (int)S.edges.size() / 2;

    // ---- table -----------------------------------------------------------------------------------------------
    std::vector<double>& T = S.table;
    T.clear();
    for (int k = 0; k < nv; ++k) push4(T, S.verts[3 * k], S.verts[3 * k + 1], S.verts[3 * k + 2], 0.0);
    for (int k = 0; k < S.ne; ++k) {
        const double* a = &S.verts[3 * S.edges[2 * k]];
        const double* b = &S.verts[3 * S.edges[2 * k + 1]];
        const double e[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]};
        const double ee = e[0] * e[0] + e[1] * e[1] + e[2] * e[2];
        if (dim == 3) {
            push4(T, a[0], a[1], a[2], ee);
            push4(T, e[0], e[1], e[2], ee > 0 ? 1.0 / ee : 0.0);
        } else {
            const double len = std::sqrt(ee);
            // a zero-length edge (disk, R14) gets an arbitrary unit direction: with len = 0 the nearest point is a
            // whatever u is, and the search kernel's side^2 + excess^2 form needs |u| = 1
            const double ux = len > 0 ? e[0] / len : 1.0, uy = len > 0 ? e[1] / len : 0.0;
            push4(T, a[0], a[1], ux, uy);
            // for a point (x, y): side = ux y - uy x + cs, centred along-edge coordinate = ux x + uy y + cm (0 at the
            // edge's midpoint); used by the search kernel
            push4(T, len, -(ux * a[1] - uy * a[0]), -(ux * a[0] + uy * a[1]) - 0.5 * len, 0.5 * len);
        }
    }
    std::vector<double> FE;
    int nfe = 0;
    const double scale = std::max(S.circumradius, 1e-300);
    for (int f = 0; f < nf; ++f) {
        const int b = S.face_off[f], n = S.face_off[f + 1] - b;
        auto P = [&](int m) { return &S.verts[3 * S.face_verts[b + ((m % n) + n) % n]]; };
        double nrm[3] = {0, 0, 0};  // Newell normal: the given boundary order is CCW about it
        for (int m = 0; m < n; ++m) {
            const double *p = P(m), *q = P(m + 1);
            nrm[0] += (p[1] - q[1]) * (p[2] + q[2]);
            nrm[1] += (p[2] - q[2]) * (p[0] + q[0]);
            nrm[2] += (p[0] - q[0]) * (p[1] + q[1]);
        }
        const double nl = std::sqrt(nrm[0] * nrm[0] + nrm[1] * nrm[1] + nrm[2] * nrm[2]);
        if (!(nl > 1e-14 * scale * scale)) return "degenerate face (zero area)";
        for (double& c : nrm) c /= nl;
        const double* o = P(0);
        // in-plane axis u along the longest boundary edge from vertex 0's side, v = n x u
        double u[3] = {P(1)[0] - o[0], P(1)[1] - o[1], P(1)[2] - o[2]};
        double ul = std::sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        if (!(ul > 0)) return "face has a repeated vertex";
        for (double& c : u) c /= ul;
        // make u exactly orthogonal to n (non-planar input is rejected below)
        const double un = u[0] * nrm[0] + u[1] * nrm[1] + u[2] * nrm[2];
        for (int a = 0; a < 3; ++a) u[a] -= un * nrm[a];
        ul = std::sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        for (double& c : u) c /= ul;
        const double v[3] = {nrm[1] * u[2] - nrm[2] * u[1], nrm[2] * u[0] - nrm[0] * u[2], nrm[0] * u[1] - nrm[1] * u[0]};
        std::vector<double> xy(2 * (size_t)n);
        for (int m = 0; m < n; ++m) {
            const double* p = P(m);
            const double w[3] = {p[0] - o[0], p[1] - o[1], p[2] - o[2]};
            const double h = w[0] * nrm[0] + w[1] * nrm[1] + w[2] * nrm[2];
            if (std::fabs(h) > 1e-9 * scale) return "face is not planar";
            xy[2 * m] = w[0] * u[0] + w[1] * u[1] + w[2] * u[2];
            xy[2 * m + 1] = w[0] * v[0] + w[1] * v[1] + w[2] * v[2];
        }
        for (int m = 0; m < n; ++m) {  // convexity: every turn is to the left (CCW about the Newell normal)
            const double* p0 = &xy[2 * m];
            const double* p1 = &xy[2 * ((m + 1) % n)];
            const double* p2 = &xy[2 * ((m + 2) % n)];
            const double cr = (p1[0] - p0[0]) * (p2[1] - p1[1]) - (p1[1] - p0[1]) * (p2[0] - p1[0]);
            if (cr < -1e-9 * scale * scale) return "face is not convex";
        }
        push4(T, u[0], u[1], u[2], -(u[0] * o[0] + u[1] * o[1] + u[2] * o[2]));
        push4(T, v[0], v[1], v[2], -(v[0] * o[0] + v[1] * o[1] + v[2] * o[2]));
        push4(T, nrm[0], nrm[1], nrm[2], -(nrm[0] * o[0] + nrm[1] * o[1] + nrm[2] * o[2]));
        push4(T, (double)nfe, (double)n, 0, 0);
        for (int m = 0; m < n; ++m) {
            const double* p0 = &xy[2 * m];
            const double* p1 = &xy[2 * ((m + 1) % n)];
            const double ex = p1[0] - p0[0], ey = p1[1] - p0[1];
            const double len = std::sqrt(ex * ex + ey * ey);
            if (!(len > 0)) return "face has a repeated vertex";
            // with (x, y) the point in the face frame: side = ux y - uy x + cs (>= 0 inside), centred along-edge
            // coordinate = ux x + uy y + cm (0 at the edge's midpoint)
            const double ux = ex / len, uy = ey / len;
            push4(FE, p0[0], p0[1], ux, uy);
            push4(FE, len, -(ux * p0[1] - uy * p0[0]), -(ux * p0[0] + uy * p0[1]) - 0.5 * len, 0.5 * len);
            nfe++;
        }
    }
    S.nfe = nfe;
    T.insert(T.end(), FE.begin(), FE.end());
    // OE: the edges again in the form the search kernel wants for its OUTER edge (unit direction, length)
    S.max_edge = 0;
    for (int k = 0; k < S.ne; ++k) {
        const double* a = &S.verts[3 * S.edges[2 * k]];
        const double* b = &S.verts[3 * S.edges[2 * k + 1]];
        const double e[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]};
        const double len = std::sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
        S.max_edge = std::max(S.max_edge, len);
        if (dim == 3) {
            push4(T, a[0], a[1], a[2], len);
            push4(T, len > 0 ? e[0] / len : 0.0, len > 0 ? e[1] / len : 0.0, len > 0 ? e[2] / len : 0.0, 0.0);
        }
    }
    if (dim == 3) {
        // EB, FB: bounding spheres of the edges (midpoint, half length) and of the faces (centroid of the vertices, largest
        // vertex distance), for the two-level sweeps of the culling kernel; radii rounded up so that float stays outside
        const double up = 1.0 + 1e-6;
        for (int k = 0; k < S.ne; ++k) {
            const double* a = &S.verts[3 * S.edges[2 * k]];
            const double* b = &S.verts[3 * S.edges[2 * k + 1]];
            const double e[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]};
            push4(T, a[0] + 0.5 * e[0], a[1] + 0.5 * e[1], a[2] + 0.5 * e[2],
                  0.5 * std::sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]) * up);
        }
        for (int f = 0; f < nf; ++f) {
            const int b = S.face_off[f], n = S.face_off[f + 1] - b;
            double c[3] = {0, 0, 0}, r = 0;
            for (int m = 0; m < n; ++m)
                for (int a = 0; a < 3; ++a) c[a] += S.verts[3 * S.face_verts[b + m] + a] / n;
            for (int m = 0; m < n; ++m) {
                const double* p = &S.verts[3 * S.face_verts[b + m]];
                r = std::max(r, std::sqrt((p[0] - c[0]) * (p[0] - c[0]) + (p[1] - c[1]) * (p[1] - c[1]) +
                                          (p[2] - c[2]) * (p[2] - c[2])));
            }
            push4(T, c[0], c[1], c[2], r * up);
        }
    }
    return "";
}

}  // namespace dem
