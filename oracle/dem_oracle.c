/*
 * dem_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, FP64 CPU oracle for the DEM conservative force / torque / energy / virial evaluation between
 * rounded polytopes of arXiv:1607.02427, written from the paper alone.  It shares no code with the
 * CUDA path in paper_1607_02427_b200/ and neither imports the other.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it computes is the DEFINITION: all particle pairs (O(N^2), minimum image), all feature
 * pairs of Eq. 1 (3D) / Eq. 2 (2D), nearest-point distance r*, WCA (Eq. 3-4), force along the line between the
 * nearest points, torque from the interaction point on each particle.  No neighbour list, no
 * blocking, no fusion.  Readings of silent/ambiguous passages are DESIGN.md "Readings" R1..R12.
 *
 * Pin status (tests/test_oracle_*.py):
 *   point-segment, segment-segment, point-polygon ......... pinned (brute-force dense sampling, exhaustive cases)
 *   Eq. 1 / Eq. 2 term counting ............................ pinned (PAPER.md:61 cube example: 3 faces per vertex,
 *                                                            5 edges per edge; closed-form lattices)
 *   WCA ..................................................... pinned (closed forms of Eq. 3-4, PAPER.md:61 value)
 *   force / torque / virial ................................ pinned (finite differences of U, balances, invariance)
 *   neighbour predicate .................................... pinned (brute force without minimum-image shortcut)
 *   virial tensor, all components and their index order .... pinned (finite-difference shear of an isolated cluster,
 *                                                            antisymmetric part against the torque balance)
 *   integrator ............................................. pinned (free-rotor invariants, dt^2 order, reversal;
 *                                                            asymmetric top against RK4 on Euler's equations)
 *   parallel-edge rule ....................... PARITY UNPINNED beyond the exactly-parallel case (the
 *                                                            paper gives no formula); for 0 < angle < 1e-3 only the
 *                                                            bound r - r_min <= sin(angle) max(L1, L2) is pinned
 *   per-particle split of U and virial (convention) ........ PARITY UNPINNED (system totals are pinned)
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC dem_oracle.c -o libdem_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------------------------ */
/* small vector helpers                                                                                         */
/* ------------------------------------------------------------------------------------------------------------ */
static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static void sub3(const double a[3], const double b[3], double o[3]) { o[0] = a[0] - b[0]; o[1] = a[1] - b[1]; o[2] = a[2] - b[2]; }
static void cross3(const double a[3], const double b[3], double o[3]) {
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}
static double clamp01(double t) { return t < 0.0 ? 0.0 : (t > 1.0 ? 1.0 : t); }

/* v_lab = q v q*, q = (w,x,y,z) unit, scalar first, body -> lab (reading R9). */
static void quat_rot(const double q[4], const double v[3], double o[3]) {
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    const double r00 = 1 - 2 * (y * y + z * z), r01 = 2 * (x * y - w * z), r02 = 2 * (x * z + w * y);
    const double r10 = 2 * (x * y + w * z), r11 = 1 - 2 * (x * x + z * z), r12 = 2 * (y * z - w * x);
    const double r20 = 2 * (x * z - w * y), r21 = 2 * (y * z + w * x), r22 = 1 - 2 * (x * x + y * y);
    o[0] = r00 * v[0] + r01 * v[1] + r02 * v[2];
    o[1] = r10 * v[0] + r11 * v[1] + r12 * v[2];
    o[2] = r20 * v[0] + r21 * v[1] + r22 * v[2];
}
static void quat_rot_inv(const double q[4], const double v[3], double o[3]) {
    const double qc[4] = {q[0], -q[1], -q[2], -q[3]};
    quat_rot(qc, v, o);
}

/* ------------------------------------------------------------------------------------------------------------ */
/* nearest-point primitives ("standard point-line, line-line, and point-plane formulae")            */
/* ------------------------------------------------------------------------------------------------------------ */

/* Nearest point c on segment [a,b] to p.  Zero-length edge => t = 0 (c = a).  Returns t. */
double orc_point_segment(const double p[3], const double a[3], const double b[3], double c[3]) {
    double e[3], w[3];
    sub3(b, a, e);
    sub3(p, a, w);
    const double ee = dot3(e, e);
    double t = 0.0;
    if (ee > 0.0) t = clamp01(dot3(w, e) / ee);
    c[0] = a[0] + t * e[0];
    c[1] = a[1] + t * e[1];
    c[2] = a[2] + t * e[2];
    return t;
}

/*
 * Nearest points c1 on [p1,q1] and c2 on [p2,q2] ("line-line"), with the near-parallel rule of
 * PAPER.md:59 as read in R5 (symmetric in the two edges, so that F_ij = -F_ji whichever particle is called i):
 * parallel <=> |d1 x d2|^2 < eps_par |d1|^2 |d2|^2.  If parallel, project segment 2 on the line of segment 1 and
 * segment 1 on the line of segment 2; if both projections overlap the other segment with positive length, the
 * interaction points are c1 = segment 1 at the midpoint of its overlap interval and c2 = segment 2 at the midpoint
 * of its overlap interval ("the midpoint of overlap between the two edges").  For exactly parallel edges c1 - c2 is
 * the common perpendicular, so r equals the true minimum distance.  Otherwise the textbook clamped routine.
 * Returns a branch code: 0 general, 1 parallel-midpoint, 2 a zero-length segment was involved.
 */
int orc_segment_segment(const double p1[3], const double q1[3], const double p2[3], const double q2[3],
                        double eps_par, double c1[3], double c2[3]) {
    double d1[3], d2[3], r[3], n[3];
    sub3(q1, p1, d1);
    sub3(q2, p2, d2);
    sub3(p1, p2, r);
    const double a = dot3(d1, d1), e = dot3(d2, d2);
    if (a <= 0.0 && e <= 0.0) { /* point - point */
        memcpy(c1, p1, 3 * sizeof(double));
        memcpy(c2, p2, 3 * sizeof(double));
        return 2;
    }
    if (a <= 0.0) { /* point p1 vs segment 2 */
        memcpy(c1, p1, 3 * sizeof(double));
        orc_point_segment(p1, p2, q2, c2);
        return 2;
    }
    if (e <= 0.0) {
        memcpy(c2, p2, 3 * sizeof(double));
        orc_point_segment(p2, p1, q1, c1);
        return 2;
    }
    cross3(d1, d2, n);
    const double nn = dot3(n, n);
    if (nn < eps_par * a * e) {
        /* parameters of segment 2's end points along line 1, and of segment 1's end points along line 2 */
        double w[3];
        sub3(p2, p1, w);
        const double s_a = dot3(w, d1) / a;
        sub3(q2, p1, w);
        const double s_b = dot3(w, d1) / a;
        sub3(p1, p2, w);
        const double t_a = dot3(w, d2) / e;
        sub3(q1, p2, w);
        const double t_b = dot3(w, d2) / e;
        const double slo = fmax(0.0, fmin(s_a, s_b)), shi = fmin(1.0, fmax(s_a, s_b));
        const double tlo = fmax(0.0, fmin(t_a, t_b)), thi = fmin(1.0, fmax(t_a, t_b));
        if (shi > slo && thi > tlo) {
            const double sm = 0.5 * (slo + shi), tm = 0.5 * (tlo + thi);
            for (int k = 0; k < 3; ++k) {
                c1[k] = p1[k] + sm * d1[k];
                c2[k] = p2[k] + tm * d2[k];
            }
            return 1;
        }
        /* no overlap: fall through to the general clamped routine */
    }
    /* General case (closest points of two segments with clamping to [0,1]^2). */
    const double f = dot3(d2, r), c = dot3(d1, r), b = dot3(d1, d2);
    double s, t;
    if (nn > 0.0) {
        /* s = -(d1 x d2).(r x d2) / |d1 x d2|^2 : the cross-product form of (b f - c e)/(a e - b^2) */
        double rxd2[3];
        cross3(r, d2, rxd2);
        s = clamp01(-dot3(n, rxd2) / nn);
    } else {
        s = 0.0;
    }
    t = (b * s + f) / e;
    if (t < 0.0) {
        t = 0.0;
        s = clamp01(-c / a);
    } else if (t > 1.0) {
        t = 1.0;
        s = clamp01((b - c) / a);
    }
    for (int k = 0; k < 3; ++k) {
        c1[k] = p1[k] + s * d1[k];
        c2[k] = p2[k] + t * d2[k];
    }
    return 0;
}

/*
 * Nearest point c on the CLOSED planar convex polygon v[0..n-1] (interior and boundary, reading R1/R2) to p.
 * Project p on the face plane; if the projection is inside all edge half-planes => c = projection, else c = the
 * nearest point over the boundary edges.  Faces are two-sided (unsigned distance).  n = 1, 2 degrade to point /
 * segment.  Returns 1 if the interior branch was taken, else 0.
 */
int orc_point_polygon(const double p[3], const double* v, int n, double c[3]) {
    if (n >= 3) {
        /* Newell normal */
        double nrm[3] = {0, 0, 0};
        for (int k = 0; k < n; ++k) {
            const double* a = v + 3 * k;
            const double* b = v + 3 * ((k + 1) % n);
            nrm[0] += (a[1] - b[1]) * (a[2] + b[2]);
            nrm[1] += (a[2] - b[2]) * (a[0] + b[0]);
            nrm[2] += (a[0] - b[0]) * (a[1] + b[1]);
        }
        const double nn = dot3(nrm, nrm);
        if (nn > 0.0) {
            double w[3], proj[3];
            sub3(p, v, w);
            const double h = dot3(w, nrm) / nn;
            for (int k = 0; k < 3; ++k) proj[k] = p[k] - h * nrm[k];
            int inside = 1;
            for (int k = 0; k < n && inside; ++k) {
                const double* a = v + 3 * k;
                const double* b = v + 3 * ((k + 1) % n);
                double e[3], u[3], x[3];
                sub3(b, a, e);
                sub3(proj, a, u);
                cross3(e, u, x);
                if (dot3(x, nrm) < 0.0) inside = 0;
            }
            if (inside) {
                memcpy(c, proj, 3 * sizeof(double));
                return 1;
            }
        }
    }
    double best = INFINITY;
    const int ne = (n == 1) ? 1 : (n == 2 ? 1 : n);
    for (int k = 0; k < ne; ++k) {
        const double* a = v + 3 * k;
        const double* b = v + 3 * ((k + 1) % n);
        double cc[3], w[3];
        orc_point_segment(p, a, b, cc);
        sub3(p, cc, w);
        const double r2 = dot3(w, w);
        if (r2 < best) {
            best = r2;
            memcpy(c, cc, 3 * sizeof(double));
        }
    }
    return 0;
}

/* WCA (Eq. 3-4): u = 4 eps [(s/r)^12 - (s/r)^6] + eps for r < 2^(1/6) s, else 0; fmag = -du/dr. */
void orc_wca(double r, double sigma, double eps, double* u, double* fmag) {
    const double rc2 = cbrt(2.0) * sigma * sigma;
    if (r * r < rc2) {
        const double s2 = (sigma / r) * (sigma / r);
        const double s6 = s2 * s2 * s2;
        *u = 4.0 * eps * (s6 * s6 - s6) + eps;
        *fmag = 24.0 * eps * (2.0 * s6 * s6 - s6) / r;
    } else {
        *u = 0.0;
        *fmag = 0.0;
    }
}

/* ------------------------------------------------------------------------------------------------------------ */
/* shapes                                                                                                        */
/* ------------------------------------------------------------------------------------------------------------ */
typedef struct {
    int nshapes;
    const int* vert_off;    /* [nshapes+1]  into verts                                   */
    const double* verts;    /* [sum nv][3]  body frame (z = 0 in 2D)                     */
    const int* edge_off;    /* [nshapes+1]  into edges                                   */
    const int* edges;       /* [sum ne][2]  local vertex indices                         */
    const int* face_off;    /* [nshapes+1]  into face_ptr (face f of shape s = face_off[s]+f) */
    const int* face_ptr;    /* [sum nf + 1] CSR into face_verts                          */
    const int* face_verts;  /* local vertex indices, CCW                                 */
    const double* rounding; /* [nshapes]    rounding radius rho                          */
} orc_shapes;

#define ORC_MAX_FACE_VERTS 64

static double shape_circumradius(const orc_shapes* S, int s) {
    double r2 = 0.0;
    for (int k = S->vert_off[s]; k < S->vert_off[s + 1]; ++k) {
        const double* v = S->verts + 3 * k;
        const double x = dot3(v, v);
        if (x > r2) r2 = x;
    }
    return sqrt(r2);
}

/* One record per Eq. 1 / Eq. 2 term, for the pins (optional). type: 0 EE, 1 V_i F_j, 2 V_j F_i, 3 V_i E_j, 4 V_j E_i */
typedef struct {
    int type, k, l, branch;
    double r;
    double ci[3], cj[3]; /* nearest points, relative to x_i */
} orc_term;

typedef struct {
    double Fi[3], Ti[3], Tj[3], u, W[6];
    int64_t nterms, nactive, ndegenerate, nparallel;
    double rmin;
} orc_pair_out;

/* O5: WCA + force/torque at the interaction points for one term with nearest points ci (on i), cj (on j). */
static void accumulate_term(const double ci[3], const double cj[3], const double d[3], double sigma, double eps,
                            int branch, orc_pair_out* o) {
    double del[3];
    sub3(ci, cj, del);
    const double r2 = dot3(del, del);
    const double r = sqrt(r2);
    o->nterms++;
    if (r < o->rmin) o->rmin = r;
    const double rc2 = cbrt(2.0) * sigma * sigma; /* r_cut^WCA = 2^(1/6) sigma, compared squared (R7) */
    if (!(r2 < rc2)) return;
    if (r2 < (1e-6 * sigma) * (1e-6 * sigma)) { /* R11: touching/crossing features are outside the model */
        o->ndegenerate++;
        return;
    }
    o->nactive++;
    if (branch == 1) o->nparallel++;
    double u, fm;
    orc_wca(r, sigma, eps, &u, &fm);
    double F[3] = {fm * del[0] / r, fm * del[1] / r, fm * del[2] / r}; /* force on i, along c_i - c_j */
    double lever_j[3], t[3], mF[3] = {-F[0], -F[1], -F[2]};
    sub3(cj, d, lever_j); /* c_j relative to x_j */
    for (int k = 0; k < 3; ++k) o->Fi[k] += F[k];
    cross3(ci, F, t);
    for (int k = 0; k < 3; ++k) o->Ti[k] += t[k];
    cross3(lever_j, mF, t);
    for (int k = 0; k < 3; ++k) o->Tj[k] += t[k];
    o->u += u;
    /* O6 / R12: W^{ab} += r_ij^a F_ij^b with r_ij = x_i - x_j = -d (centre-of-mass virial), upper triangle */
    o->W[0] += -d[0] * F[0];
    o->W[1] += -d[0] * F[1];
    o->W[2] += -d[0] * F[2];
    o->W[3] += -d[1] * F[1];
    o->W[4] += -d[1] * F[2];
    o->W[5] += -d[2] * F[2];
}

/*
 * O3 + O4 + O5 for ONE ordered pair (i, j): all feature pairs of Eq. 1 (dim 3) or Eq. 2 (dim 2).
 * d = minimum-image x_j - x_i.  Everything is expressed relative to x_i in the lab frame:
 * a_k = R(q_i) v_k^(i),  b_l = d + R(q_j) v_l^(j).
 */
static void pair_eval(const orc_shapes* S, int dim, int si, int sj, const double qi[4], const double qj[4],
                      const double d[3], double eps, double eps_par, orc_pair_out* o, orc_term* terms, int max_terms) {
    const int nvi = S->vert_off[si + 1] - S->vert_off[si], nvj = S->vert_off[sj + 1] - S->vert_off[sj];
    const int nei = S->edge_off[si + 1] - S->edge_off[si], nej = S->edge_off[sj + 1] - S->edge_off[sj];
    const int nfi = S->face_off[si + 1] - S->face_off[si], nfj = S->face_off[sj + 1] - S->face_off[sj];
    const double sigma = S->rounding[si] + S->rounding[sj]; /* R6: sigma_ij = rho_i + rho_j */
    double* a = (double*)malloc(sizeof(double) * 3 * (size_t)(nvi + nvj));
    double* b = a + 3 * nvi;
    for (int k = 0; k < nvi; ++k) quat_rot(qi, S->verts + 3 * (S->vert_off[si] + k), a + 3 * k);
    for (int l = 0; l < nvj; ++l) {
        quat_rot(qj, S->verts + 3 * (S->vert_off[sj] + l), b + 3 * l);
        for (int c = 0; c < 3; ++c) b[3 * l + c] += d[c];
    }
    memset(o, 0, sizeof(*o));
    o->rmin = INFINITY;
    int nt = 0;
#define RECORD(ty, kk, ll, br)                                                                                 \
    do {                                                                                                       \
        if (terms && nt < max_terms) {                                                                         \
            double w_[3];                                                                                      \
            sub3(ci, cj, w_);                                                                                  \
            terms[nt].type = ty; terms[nt].k = kk; terms[nt].l = ll; terms[nt].branch = br;                    \
            terms[nt].r = sqrt(dot3(w_, w_));                                                                  \
            memcpy(terms[nt].ci, ci, sizeof(ci)); memcpy(terms[nt].cj, cj, sizeof(cj));                        \
        }                                                                                                      \
        nt++;                                                                                                  \
    } while (0)
    double ci[3], cj[3];
    if (dim == 3) {
        /* first sum of Eq. 1: all edge-edge pairs */
        for (int k = 0; k < nei; ++k) {
            const int* ek = S->edges + 2 * (S->edge_off[si] + k);
            for (int l = 0; l < nej; ++l) {
                const int* el = S->edges + 2 * (S->edge_off[sj] + l);
                const int br = orc_segment_segment(a + 3 * ek[0], a + 3 * ek[1], b + 3 * el[0], b + 3 * el[1],
                                                   eps_par, ci, cj);
                RECORD(0, k, l, br);
                accumulate_term(ci, cj, d, sigma, eps, br, o);
            }
        }
        /* second sum: vertices of i against faces of j; third sum: vertices of j against faces of i */
        double poly[3 * ORC_MAX_FACE_VERTS];
        for (int l = 0; l < nfj; ++l) {
            const int f0 = S->face_ptr[S->face_off[sj] + l], f1 = S->face_ptr[S->face_off[sj] + l + 1];
            for (int m = f0; m < f1; ++m) memcpy(poly + 3 * (m - f0), b + 3 * S->face_verts[m], 3 * sizeof(double));
            for (int k = 0; k < nvi; ++k) {
                memcpy(ci, a + 3 * k, sizeof(ci));
                orc_point_polygon(ci, poly, f1 - f0, cj);
                RECORD(1, k, l, 0);
                accumulate_term(ci, cj, d, sigma, eps, 0, o);
            }
        }
        for (int k = 0; k < nfi; ++k) {
            const int f0 = S->face_ptr[S->face_off[si] + k], f1 = S->face_ptr[S->face_off[si] + k + 1];
            for (int m = f0; m < f1; ++m) memcpy(poly + 3 * (m - f0), a + 3 * S->face_verts[m], 3 * sizeof(double));
            for (int l = 0; l < nvj; ++l) {
                memcpy(cj, b + 3 * l, sizeof(cj));
                orc_point_polygon(cj, poly, f1 - f0, ci);
                RECORD(2, k, l, 0);
                accumulate_term(ci, cj, d, sigma, eps, 0, o);
            }
        }
    } else {
        /* Eq. 2: vertices of i against edges of j, vertices of j against edges of i */
        for (int k = 0; k < nvi; ++k) {
            for (int l = 0; l < nej; ++l) {
                const int* el = S->edges + 2 * (S->edge_off[sj] + l);
                memcpy(ci, a + 3 * k, sizeof(ci));
                orc_point_segment(ci, b + 3 * el[0], b + 3 * el[1], cj);
                RECORD(3, k, l, 0);
                accumulate_term(ci, cj, d, sigma, eps, 0, o);
            }
        }
        for (int l = 0; l < nvj; ++l) {
            for (int k = 0; k < nei; ++k) {
                const int* ek = S->edges + 2 * (S->edge_off[si] + k);
                memcpy(cj, b + 3 * l, sizeof(cj));
                orc_point_segment(cj, a + 3 * ek[0], a + 3 * ek[1], ci);
                RECORD(4, k, l, 0);
                accumulate_term(ci, cj, d, sigma, eps, 0, o);
            }
        }
    }
#undef RECORD
    free(a);
}

/* O1: minimum-image separation with the exact operation order both sides of the bit-exact test use (R13). */
static void min_image(int dim, const double box[3], const double* xi, const double* xj, double d[3]) {
    d[2] = 0.0;
    for (int a = 0; a < dim; ++a) {
        double da = xj[a] - xi[a];
        const double k = rint(da / box[a]);
        const double shift = box[a] * k;
        da = da - shift;
        d[a] = da;
    }
}
static double norm2_fma(const double d[3]) { return fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0])); }

/* Term list + sums for ONE ordered pair (pins: counting of Eq. 1/2, closed forms).  Returns the number of terms. */
int orc_pair_terms(const orc_shapes* S, int dim, int si, int sj, const double qi[4], const double qj[4],
                   const double d[3], double eps, double eps_par, orc_term* terms, int max_terms, double* out17) {
    orc_pair_out o;
    pair_eval(S, dim, si, sj, qi, qj, d, eps, eps_par, &o, terms, max_terms);
    if (out17) {
        memcpy(out17, o.Fi, 3 * sizeof(double));
        memcpy(out17 + 3, o.Ti, 3 * sizeof(double));
        memcpy(out17 + 6, o.Tj, 3 * sizeof(double));
        out17[9] = o.u;
        memcpy(out17 + 10, o.W, 6 * sizeof(double));
        out17[16] = o.rmin;
    }
    return (int)o.nterms;
}

/*
 * Neighbour rows by the definition O1: j != i with minimum-image r^2 < r_cut^2 (strict), all pairs, no cells.
 * rows: nsub = number of rows (subset[k] = particle index, or NULL => rows 0..N-1).  Row k is written sorted by j
 * into list[k*stride ...]; counts[k] = TRUE count (may exceed stride; then only the first `stride` are stored).
 * Returns the maximum count.
 */
int orc_neighbors(int dim, int N, const double box[3], const double* pos4, double r_cut, const int* subset, int nsub,
                  int* counts, int* list, int stride) {
    const double rc2 = r_cut * r_cut;
    const int rows = subset ? nsub : N;
    int maxc = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(max : maxc)
    for (int k = 0; k < rows; ++k) {
        const int i = subset ? subset[k] : k;
        int c = 0;
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            double d[3];
            min_image(dim, box, pos4 + 4 * (size_t)i, pos4 + 4 * (size_t)j, d);
            if (norm2_fma(d) < rc2) {
                if (c < stride) list[(size_t)k * stride + c] = j;
                c++;
            }
        }
        counts[k] = c;
        if (c > maxc) maxc = c;
    }
    return maxc;
}

/*
 * O2..O6: per-particle force/energy, torque, virial by the definition ("the sum of the force, torque,
 * and potential energy contributions between it and its neighbors"): for each particle i (all, or the given subset)
 * loop over ALL j != i with minimum image and evaluate every feature pair.  use_reject != 0 enables the exact early
 * reject |d| >= R_i + R_j + 2^(1/6) sigma_ij (no term can be inside the WCA cutoff; R10).
 *   force4  [rows][4] = Fx,Fy,Fz,U_i  (U_i = 1/2 sum_j U_ij)     torque4 [rows][4] = lab-frame torque, 0
 *   virial6 [rows][6] = 1/2 sum_j W_ij (xx,xy,xz,yy,yz,zz), may be NULL
 *   counters[5] (may be NULL): directed pairs evaluated, terms, active terms, degenerate terms, parallel-branch terms
 * Rows are indexed by position in `subset` (or by particle when subset == NULL).
 */
int orc_compute(const orc_shapes* S, int dim, int N, const double box[3], const double* pos4, const double* quat4,
                const int* sid, double eps, double eps_par, int use_reject, const int* subset, int nsub,
                double* force4, double* torque4, double* virial6, int64_t* counters) {
    const int rows = subset ? nsub : N;
    double* R = (double*)malloc(sizeof(double) * (size_t)S->nshapes);
    for (int s = 0; s < S->nshapes; ++s) R[s] = shape_circumradius(S, s);
    const double rcw = pow(2.0, 1.0 / 6.0);
    int64_t c0 = 0, c1 = 0, c2 = 0, c3 = 0, c4 = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : c0, c1, c2, c3, c4)
    for (int k = 0; k < rows; ++k) {
        const int i = subset ? subset[k] : k;
        double F[3] = {0, 0, 0}, T[3] = {0, 0, 0}, U = 0.0, W[6] = {0, 0, 0, 0, 0, 0};
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            double d[3];
            min_image(dim, box, pos4 + 4 * (size_t)i, pos4 + 4 * (size_t)j, d);
            if (use_reject) {
                const double reach = R[sid[i]] + R[sid[j]] + rcw * (S->rounding[sid[i]] + S->rounding[sid[j]]);
                if (dot3(d, d) >= reach * reach) continue;
            }
            orc_pair_out o;
            pair_eval(S, dim, sid[i], sid[j], quat4 + 4 * (size_t)i, quat4 + 4 * (size_t)j, d, eps, eps_par, &o, NULL, 0);
            for (int a = 0; a < 3; ++a) {
                F[a] += o.Fi[a];
                T[a] += o.Ti[a];
            }
            U += 0.5 * o.u;
            for (int a = 0; a < 6; ++a) W[a] += 0.5 * o.W[a];
            c0 += 1;
            c1 += o.nterms;
            c2 += o.nactive;
            c3 += o.ndegenerate;
            c4 += o.nparallel;
        }
        force4[4 * (size_t)k + 0] = F[0];
        force4[4 * (size_t)k + 1] = F[1];
        force4[4 * (size_t)k + 2] = F[2];
        force4[4 * (size_t)k + 3] = U;
        torque4[4 * (size_t)k + 0] = T[0];
        torque4[4 * (size_t)k + 1] = T[1];
        torque4[4 * (size_t)k + 2] = T[2];
        torque4[4 * (size_t)k + 3] = 0.0;
        if (virial6)
            for (int a = 0; a < 6; ++a) virial6[6 * (size_t)k + a] = W[a];
    }
    if (counters) {
        counters[0] = c0; counters[1] = c1; counters[2] = c2; counters[3] = c3; counters[4] = c4;
    }
    free(R);
    return 0;
}

/*
 * The same per-particle sums as orc_compute(use_reject = 1), visiting only the particles of the 3^dim adjacent cells of a
 * plain cell grid (cell width >= the interaction reach R10, so every pair the reject test keeps is found).  The
 * candidates of a row are sorted by index before they are evaluated, so every sum runs over the same pairs in the same
 * order as the all-pairs loop and the results are identical bit for bit (tests/test_oracle_system.py).  It exists so
 * that the full-size configurations (N = 262,144) can be checked row by row in seconds and so that bench.py can time
 * the oracle's feature work without the O(N) scan per particle; the all-pairs routine above stays the definition.
 */
static int cmp_int(const void* a, const void* b) {
    const int x = *(const int*)a, y = *(const int*)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

int orc_compute_cells(const orc_shapes* S, int dim, int N, const double box[3], const double* pos4, const double* quat4,
                      const int* sid, double eps, double eps_par, const int* subset, int nsub, double* force4,
                      double* torque4, double* virial6, int64_t* counters) {
    const int rows = subset ? nsub : N;
    double* R = (double*)malloc(sizeof(double) * (size_t)S->nshapes);
    for (int s = 0; s < S->nshapes; ++s) R[s] = shape_circumradius(S, s);
    const double rcw = pow(2.0, 1.0 / 6.0);
    double reach_max = 0.0;
    for (int a = 0; a < S->nshapes; ++a)
        for (int b = 0; b < S->nshapes; ++b) {
            const double r = R[a] + R[b] + rcw * (S->rounding[a] + S->rounding[b]);
            if (r > reach_max) reach_max = r;
        }
    int nc[3] = {1, 1, 1};
    for (int a = 0; a < dim; ++a) {
        nc[a] = (int)floor(box[a] / (reach_max * (1.0 + 1e-9)));
        if (nc[a] < 1) nc[a] = 1;
        if (nc[a] > 1024) nc[a] = 1024;
    }
    const int ncell = nc[0] * nc[1] * nc[2];
    int* cell_of = (int*)malloc(sizeof(int) * (size_t)N);
    int* start = (int*)calloc((size_t)ncell + 1, sizeof(int));
    int* members = (int*)malloc(sizeof(int) * (size_t)N);
    for (int i = 0; i < N; ++i) {
        int c[3] = {0, 0, 0};
        for (int a = 0; a < dim; ++a) {
            double f = pos4[4 * (size_t)i + a] / box[a] + 0.5;
            f -= floor(f);
            int ca = (int)(f * nc[a]);
            c[a] = ca < 0 ? 0 : (ca >= nc[a] ? nc[a] - 1 : ca);
        }
        cell_of[i] = (c[2] * nc[1] + c[1]) * nc[0] + c[0];
        start[cell_of[i] + 1]++;
    }
    for (int c = 0; c < ncell; ++c) start[c + 1] += start[c];
    {
        int* fill = (int*)malloc(sizeof(int) * (size_t)ncell);
        memcpy(fill, start, sizeof(int) * (size_t)ncell);
        for (int i = 0; i < N; ++i) members[fill[cell_of[i]]++] = i;
        free(fill);
    }
    int64_t c0 = 0, c1 = 0, c2 = 0, c3 = 0, c4 = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : c0, c1, c2, c3, c4)
    for (int k = 0; k < rows; ++k) {
        const int i = subset ? subset[k] : k;
        int cap = 64, ncand = 0;
        int* cand = (int*)malloc(sizeof(int) * (size_t)cap);
        int ci = cell_of[i];
        const int cx = ci % nc[0];
        ci /= nc[0];
        const int cy = ci % nc[1], cz = ci / nc[1];
        const int nx = nc[0] < 3 ? nc[0] : 3, ny = nc[1] < 3 ? nc[1] : 3, nz = nc[2] < 3 ? nc[2] : 3;
        for (int iz = 0; iz < nz; ++iz) {
            const int z = nc[2] < 3 ? iz : (cz + iz - 1 + nc[2]) % nc[2];
            for (int iy = 0; iy < ny; ++iy) {
                const int y = nc[1] < 3 ? iy : (cy + iy - 1 + nc[1]) % nc[1];
                for (int ix = 0; ix < nx; ++ix) {
                    const int x = nc[0] < 3 ? ix : (cx + ix - 1 + nc[0]) % nc[0];
                    const int c = (z * nc[1] + y) * nc[0] + x;
                    for (int m = start[c]; m < start[c + 1]; ++m) {
                        if (members[m] == i) continue;
                        if (ncand == cap) {
                            cap *= 2;
                            cand = (int*)realloc(cand, sizeof(int) * (size_t)cap);
                        }
                        cand[ncand++] = members[m];
                    }
                }
            }
        }
        qsort(cand, (size_t)ncand, sizeof(int), cmp_int);
        double F[3] = {0, 0, 0}, T[3] = {0, 0, 0}, U = 0.0, W[6] = {0, 0, 0, 0, 0, 0};
        for (int m = 0; m < ncand; ++m) {
            const int j = cand[m];
            double d[3];
            min_image(dim, box, pos4 + 4 * (size_t)i, pos4 + 4 * (size_t)j, d);
            const double reach = R[sid[i]] + R[sid[j]] + rcw * (S->rounding[sid[i]] + S->rounding[sid[j]]);
            if (dot3(d, d) >= reach * reach) continue;
            orc_pair_out o;
            pair_eval(S, dim, sid[i], sid[j], quat4 + 4 * (size_t)i, quat4 + 4 * (size_t)j, d, eps, eps_par, &o, NULL, 0);
            for (int a = 0; a < 3; ++a) {
                F[a] += o.Fi[a];
                T[a] += o.Ti[a];
            }
            U += 0.5 * o.u;
            for (int a = 0; a < 6; ++a) W[a] += 0.5 * o.W[a];
            c0 += 1;
            c1 += o.nterms;
            c2 += o.nactive;
            c3 += o.ndegenerate;
            c4 += o.nparallel;
        }
        free(cand);
        force4[4 * (size_t)k + 0] = F[0];
        force4[4 * (size_t)k + 1] = F[1];
        force4[4 * (size_t)k + 2] = F[2];
        force4[4 * (size_t)k + 3] = U;
        torque4[4 * (size_t)k + 0] = T[0];
        torque4[4 * (size_t)k + 1] = T[1];
        torque4[4 * (size_t)k + 2] = T[2];
        torque4[4 * (size_t)k + 3] = 0.0;
        if (virial6)
            for (int a = 0; a < 6; ++a) virial6[6 * (size_t)k + a] = W[a];
    }
    if (counters) {
        counters[0] = c0; counters[1] = c1; counters[2] = c2; counters[3] = c3; counters[4] = c4;
    }
    free(R);
    free(cell_of);
    free(start);
    free(members);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* NVE integrator ("second-order integrator", ref. 23; reading R15)                                  */
/* ------------------------------------------------------------------------------------------------------------ */
static void quat_mul(const double a[4], const double b[4], double o[4]) {
    o[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    o[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    o[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    o[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}
static void quat_normalize(double q[4]) {
    const double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int k = 0; k < 4; ++k) q[k] /= n;
}

/*
 * Free rotation of one rigid body over dt with lab-frame angular momentum L held fixed (torque-free flow).
 *  - spherical top (I1 = I2 = I3 = I0; in 2D I0 = I3): exact, q <- exp(dt/2 * L/I0) (x) q.
 *  - otherwise: symmetric splitting of the free-rotor Hamiltonian into rotations about the body axes
 *    x(dt/2) y(dt/2) z(dt) y(dt/2) x(dt/2)  (the splitting used by the integrators of ref. 23's family).
 */
static void free_rotate(int dim, const double I[3], const double L[3], double dt, double q[4]) {
    const int spherical = (dim == 2) || (I[0] == I[1] && I[1] == I[2]);
    if (spherical) {
        const double I0 = I[2];
        if (!(I0 > 0.0)) return;
        const double w[3] = {L[0] / I0, L[1] / I0, L[2] / I0};
        const double wn = sqrt(dot3(w, w));
        if (wn == 0.0) return;
        const double half = 0.5 * wn * dt, sn = sin(half) / wn;
        const double rq[4] = {cos(half), sn * w[0], sn * w[1], sn * w[2]};
        double o[4];
        quat_mul(rq, q, o);
        memcpy(q, o, sizeof(o));
        quat_normalize(q);
        return;
    }
    double Lb[3];
    quat_rot_inv(q, L, Lb);
    static const int axis_seq[5] = {0, 1, 2, 1, 0};
    static const double frac[5] = {0.5, 0.5, 1.0, 0.5, 0.5};
    for (int s = 0; s < 5; ++s) {
        const int a = axis_seq[s];
        if (!(I[a] > 0.0)) continue;
        const double phi = frac[s] * dt * Lb[a] / I[a];
        const double cs = cos(phi), sn = sin(phi);
        /* body-frame angular momentum rotates by -phi about axis a */
        const int b = (a + 1) % 3, c = (a + 2) % 3;
        const double lb = cs * Lb[b] + sn * Lb[c], lc = -sn * Lb[b] + cs * Lb[c];
        Lb[b] = lb;
        Lb[c] = lc;
        double rq[4] = {cos(0.5 * phi), 0, 0, 0}, o[4];
        rq[1 + a] = sin(0.5 * phi);
        quat_mul(q, rq, o); /* body-axis rotation composes on the right */
        memcpy(q, o, sizeof(o));
    }
    quat_normalize(q);
}

/* U, K_trans, K_rot of a state (force4[.][3] holds U_i). */
void orc_energy(int dim, int N, const double* mass, const double* inertia3, const int* sid, const double* quat4,
                const double* vel4, const double* ang4, const double* force4, double out3[3]) {
    double U = 0, Kt = 0, Kr = 0;
    for (int i = 0; i < N; ++i) {
        const double* v = vel4 + 4 * (size_t)i;
        U += force4[4 * (size_t)i + 3];
        Kt += 0.5 * mass[sid[i]] * dot3(v, v);
        double Lb[3];
        quat_rot_inv(quat4 + 4 * (size_t)i, ang4 + 4 * (size_t)i, Lb);
        const double* I = inertia3 + 3 * sid[i];
        for (int a = (dim == 2 ? 2 : 0); a < 3; ++a)
            if (I[a] > 0.0) Kr += 0.5 * Lb[a] * Lb[a] / I[a];
    }
    out3[0] = U; out3[1] = Kt; out3[2] = Kr;
}

/*
 * nsteps of velocity-Verlet NVE (R15): half-kick v, L; drift x (wrapped back into the centred box); free rotation;
 * force evaluation (orc_compute, all pairs, exact reject); half-kick.  Arrays are updated in place; force4/torque4
 * hold the forces of the final state.  energies (may be NULL): [(nsteps+1)][3] = U, K_trans, K_rot after each step
 * (row 0 = initial state).
 */
int orc_step(const orc_shapes* S, const double* mass, const double* inertia3, int dim, int N, const double box[3],
             double* pos4, double* quat4, double* vel4, double* ang4, const int* sid, double eps, double eps_par,
             double dt, int nsteps, double* force4, double* torque4, double* energies) {
    orc_compute(S, dim, N, box, pos4, quat4, sid, eps, eps_par, 1, NULL, 0, force4, torque4, NULL, NULL);
    if (energies) orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, energies);
    for (int step = 1; step <= nsteps; ++step) {
        for (int i = 0; i < N; ++i) {
            const double m = mass[sid[i]];
            double *x = pos4 + 4 * (size_t)i, *v = vel4 + 4 * (size_t)i, *L = ang4 + 4 * (size_t)i;
            const double *F = force4 + 4 * (size_t)i, *T = torque4 + 4 * (size_t)i;
            for (int a = 0; a < dim; ++a) {
                v[a] += 0.5 * dt * F[a] / m;
                x[a] += dt * v[a];
                x[a] -= box[a] * rint(x[a] / box[a]);
            }
            for (int a = (dim == 2 ? 2 : 0); a < 3; ++a) L[a] += 0.5 * dt * T[a];
            free_rotate(dim, inertia3 + 3 * sid[i], L, dt, quat4 + 4 * (size_t)i);
        }
        orc_compute(S, dim, N, box, pos4, quat4, sid, eps, eps_par, 1, NULL, 0, force4, torque4, NULL, NULL);
        for (int i = 0; i < N; ++i) {
            const double m = mass[sid[i]];
            double *v = vel4 + 4 * (size_t)i, *L = ang4 + 4 * (size_t)i;
            const double *F = force4 + 4 * (size_t)i, *T = torque4 + 4 * (size_t)i;
            for (int a = 0; a < dim; ++a) v[a] += 0.5 * dt * F[a] / m;
            for (int a = (dim == 2 ? 2 : 0); a < 3; ++a) L[a] += 0.5 * dt * T[a];
        }
        if (energies) orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, energies + 3 * (size_t)step);
    }
    return 0;
}

/*
 * NVT ("a standard Nose-Hoover thermostat applied to both translational and
 * rotational degrees of freedom", ref. 23).  Reading (R19): ONE friction variable xi for all degrees of
 * freedom, dv/dt = F/m - xi v, dL/dt = tau - xi L, dxi/dt = (2K - g kT)/Q, deta/dt = xi, Q = g kT tau_T^2,
 * K = K_trans + K_rot, g = dim (N - 1) + number of (particle, rotation axis) with I > 0 (2D: the z axis only).
 * One step = thermostat half step, the NVE step above, thermostat half step, where a thermostat half step is
 *     xi += (dt/4)(2K - g kT)/Q;  s = exp(-xi dt/2);  v *= s;  L *= s;  K *= s^2;  eta += (dt/2) xi;
 *     xi += (dt/4)(2K - g kT)/Q
 * (symmetric, time-reversible).  Conserved: U + K + Q xi^2/2 + g kT eta.
 * thermo[2] = (xi, eta), in and out.  energies (may be NULL): [(nsteps+1)][5] = U, K_trans, K_rot, xi, eta.
 * Returns g.
 */
static double nvt_dof(int dim, int N, const double* inertia3, const int* sid) {
    double g = (double)dim * (N - 1);
    for (int i = 0; i < N; ++i)
        for (int a = (dim == 2 ? 2 : 0); a < 3; ++a)
            if (inertia3[3 * sid[i] + a] > 0.0) g += 1.0;
    return g;
}

static void nvt_half(int dim, int N, const double* mass, const double* inertia3, const int* sid, const double* quat4,
                     double* vel4, double* ang4, const double* force4, double dt, double g, double kT, double Q,
                     double thermo[2]) {
    double e[3];
    orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, e);
    double K = e[1] + e[2];
    thermo[0] += 0.25 * dt * (2.0 * K - g * kT) / Q;
    const double s = exp(-thermo[0] * 0.5 * dt);
    for (int i = 0; i < N; ++i)
        for (int a = 0; a < 3; ++a) {
            vel4[4 * (size_t)i + a] *= s;
            ang4[4 * (size_t)i + a] *= s;
        }
    K *= s * s;
    thermo[1] += 0.5 * dt * thermo[0];
    thermo[0] += 0.25 * dt * (2.0 * K - g * kT) / Q;
}

double orc_step_nvt(const orc_shapes* S, const double* mass, const double* inertia3, int dim, int N,
                    const double box[3], double* pos4, double* quat4, double* vel4, double* ang4, const int* sid,
                    double eps, double eps_par, double dt, int nsteps, double kT, double tau_T, double thermo[2],
                    double* force4, double* torque4, double* energies) {
    const double g = nvt_dof(dim, N, inertia3, sid), Q = g * kT * tau_T * tau_T;
    orc_compute(S, dim, N, box, pos4, quat4, sid, eps, eps_par, 1, NULL, 0, force4, torque4, NULL, NULL);
    if (energies) {
        orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, energies);
        energies[3] = thermo[0];
        energies[4] = thermo[1];
    }
    for (int step = 1; step <= nsteps; ++step) {
        nvt_half(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, dt, g, kT, Q, thermo);
        orc_step(S, mass, inertia3, dim, N, box, pos4, quat4, vel4, ang4, sid, eps, eps_par, dt, 1, force4, torque4,
                 NULL);
        nvt_half(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, dt, g, kT, Q, thermo);
        if (energies) {
            double* e = energies + 5 * (size_t)step;
            orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, e);
            e[3] = thermo[0];
            e[4] = thermo[1];
        }
    }
    return g;
}

/*
 * NPT ("We simulate ... in the NPT ensemble ... a standard Nose-Hoover thermostat
 * applied to both translational and rotational degrees of freedom, and the barostat computes the pressure from the
 * virial tensor, just as in MD" (ref. 25)).  The paper gives no equations; reading DESIGN.md R22: the isotropic
 * Martyna-Tobias-Klein barostat on the box strain rate nu = d ln L / dt, coupled to the CENTRE-OF-MASS motion of the
 * rigid bodies only (orientations and angular momenta do not feel the box), with the one-variable thermostat of R19:
 *     dx/dt  = v + nu x                      dL_box/dt = nu L_box     (V = prod_a L_a, dV/dt = d nu V)
 *     dv/dt  = F/m - (alpha nu + xi) v       alpha = 1 + d / N_f,  N_f = d (N - 1)
 *     dL/dt  = tau - xi L                    (free rotation as in the NVE step)
 *     dnu/dt = [alpha 2 K_trans + tr W - d V P_ext] / W_b,   W_b = d N kT tau_P^2,   tr W = sum_i tr W_i = sum_pairs r_ij . F_ij
 *              (= d V (P_int - P_ext) + (d / N_f) 2 K_trans with P_int = (2 K_trans + tr W) / (d V): "pressure from the virial")
 *     dxi/dt = (2 K - g kT) / Q,  deta/dt = xi      (R19)
 * Conserved: U + K + P_ext V + W_b nu^2 / 2 + Q xi^2 / 2 + g kT eta.
 * One step (palindromic, hence time-reversible and second order), h = dt / 2:
 *     T(h)  thermostat half step (nvt_half above)
 *     B(h)  nu += h [alpha 2 K_trans + tr W - d V P_ext] / W_b
 *     K(h)  s = exp(-alpha nu h / 2);  v = (v s + h F / m) s;  L += h tau
 *     D(dt) x = x e^{nu dt} + v dt e^{nu dt / 2} sinh(nu dt / 2) / (nu dt / 2);  L_box *= e^{nu dt};  wrap;  free rotation
 *     force evaluation (with the virial)
 *     K(h)  B(h)  T(h)
 * state[3] = (xi, eta, nu), in and out; box[3] in and out.  energies (may be NULL): [(nsteps+1)][8] = U, K_trans,
 * K_rot, xi, eta, nu, V, tr W.  Returns g.  tau_T = inf gives NPH, tau_P = inf with nu = 0 gives orc_step_nvt.
 */
static double sum_trace_virial(int dim, int N, const double* virial6) {
    double t = 0.0;
    for (int i = 0; i < N; ++i) {
        const double* w = virial6 + 6 * (size_t)i;
        t += w[0] + w[3] + (dim == 3 ? w[5] : 0.0);
    }
    return t;
}

static double box_volume(int dim, const double box[3]) { return dim == 3 ? box[0] * box[1] * box[2] : box[0] * box[1]; }

static void npt_baro_half(int dim, int N, const double* mass, const double* inertia3, const int* sid, const double* quat4,
                          const double* vel4, const double* ang4, const double* force4, double trW, double V, double h,
                          double alpha, double P_ext, double Wb, double state[3]) {
    double e[3];
    orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, e);
    state[2] += h * (alpha * 2.0 * e[1] + trW - dim * V * P_ext) / Wb;
}

static void npt_kick_half(int dim, int N, const double* mass, const int* sid, double* vel4, double* ang4,
                          const double* force4, const double* torque4, double dt, double alpha, double nu) {
    const double s = exp(-alpha * nu * 0.25 * dt);
    for (int i = 0; i < N; ++i) {
        const double m = mass[sid[i]];
        double *v = vel4 + 4 * (size_t)i, *L = ang4 + 4 * (size_t)i;
        const double *F = force4 + 4 * (size_t)i, *T = torque4 + 4 * (size_t)i;
        for (int a = 0; a < dim; ++a) v[a] = (v[a] * s + 0.5 * dt * F[a] / m) * s;
        for (int a = (dim == 2 ? 2 : 0); a < 3; ++a) L[a] += 0.5 * dt * T[a];
    }
}

double orc_step_npt(const orc_shapes* S, const double* mass, const double* inertia3, int dim, int N, double box[3],
                    double* pos4, double* quat4, double* vel4, double* ang4, const int* sid, double eps, double eps_par,
                    double dt, int nsteps, double kT, double tau_T, double P_ext, double tau_P, double state[3],
                    double* force4, double* torque4, double* energies) {
    const double g = nvt_dof(dim, N, inertia3, sid), Q = g * kT * tau_T * tau_T;
    const double Nf = (double)dim * (N - 1), alpha = 1.0 + dim / Nf, Wb = (double)dim * N * kT * tau_P * tau_P;
    double* virial6 = (double*)malloc(sizeof(double) * 6 * (size_t)N);
    orc_compute(S, dim, N, box, pos4, quat4, sid, eps, eps_par, 1, NULL, 0, force4, torque4, virial6, NULL);
    double trW = sum_trace_virial(dim, N, virial6);
#define NPT_RECORD(row)                                                                         \
    do {                                                                                        \
        if (energies) {                                                                         \
            double* e_ = energies + 8 * (size_t)(row);                                          \
            orc_energy(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, e_);             \
            e_[3] = state[0]; e_[4] = state[1]; e_[5] = state[2];                               \
            e_[6] = box_volume(dim, box); e_[7] = trW;                                          \
        }                                                                                       \
    } while (0)
    NPT_RECORD(0);
    for (int step = 1; step <= nsteps; ++step) {
        nvt_half(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, dt, g, kT, Q, state);
        npt_baro_half(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, trW, box_volume(dim, box), 0.5 * dt,
                      alpha, P_ext, Wb, state);
        const double nu = state[2];
        npt_kick_half(dim, N, mass, sid, vel4, ang4, force4, torque4, dt, alpha, nu);
        /* drift: exact flow of dx/dt = v + nu x at constant v and nu */
        const double z = 0.5 * nu * dt, ea = exp(nu * dt), eh = exp(z), sc = (z == 0.0) ? 1.0 : sinh(z) / z;
        for (int a = 0; a < dim; ++a) box[a] *= ea;
        for (int i = 0; i < N; ++i) {
            double *x = pos4 + 4 * (size_t)i, *v = vel4 + 4 * (size_t)i;
            for (int a = 0; a < dim; ++a) {
                x[a] = x[a] * ea + v[a] * (dt * eh * sc);
                x[a] -= box[a] * rint(x[a] / box[a]);
            }
            free_rotate(dim, inertia3 + 3 * sid[i], ang4 + 4 * (size_t)i, dt, quat4 + 4 * (size_t)i);
        }
        orc_compute(S, dim, N, box, pos4, quat4, sid, eps, eps_par, 1, NULL, 0, force4, torque4, virial6, NULL);
        trW = sum_trace_virial(dim, N, virial6);
        npt_kick_half(dim, N, mass, sid, vel4, ang4, force4, torque4, dt, alpha, nu);
        npt_baro_half(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, trW, box_volume(dim, box), 0.5 * dt,
                      alpha, P_ext, Wb, state);
        nvt_half(dim, N, mass, inertia3, sid, quat4, vel4, ang4, force4, dt, g, kT, Q, state);
        NPT_RECORD(step);
    }
#undef NPT_RECORD
    free(virial6);
    return g;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
