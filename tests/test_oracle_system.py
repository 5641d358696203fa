"""Pins for the oracle's pair / system evaluation (CPU only).  Nothing here compares the oracle with itself:

* Eq. 1 / Eq. 2 term counting against the worked example PAPER.md:61 (3 faces per facing vertex, 5 edges per facing
  edge; golden file) and against brute-force dense sampling of every feature pair;
* closed forms: aligned cube / square lattices, one-vertex shapes (central WCA), rods;
* conservativeness: F = -dU/dx and tau = -dU/dphi by central finite differences of U;
* the virial against -dU/dlambda under uniform scaling;
* momentum and angular-momentum balance, translation / rotation invariance;
* the neighbour predicate against a search over explicit periodic images;
* the integrator: free-rotor invariants, dt^2 order, time reversal.
"""
import math

import numpy as np
import pytest

import dem_inputs as di
from _util import golden, quat_from_axis_angle, quat_mul, rotmat

ID = np.array([1.0, 0, 0, 0])


def _wca(r, sigma, eps=1.0):
    """Eq. 3-4 written out independently of the oracle."""
    if r >= 2 ** (1 / 6) * sigma:
        return 0.0, 0.0
    x = (sigma / r) ** 6
    return 4 * eps * (x * x - x) + eps, 24 * eps * (2 * x * x - x) / r


# ---------------------------------------------------------------------------------------------------------------
# counting of Eq. 1 / Eq. 2
# ---------------------------------------------------------------------------------------------------------------
def test_cube_face_to_face_counts_match_paper(oracle):
    g = golden()
    gap = 0.3
    sh = [di.cube(1.0, 0.15)]
    terms, sums = oracle.pair_terms(sh, 0, 0, ID, ID, [1.0 + gap, 0, 0])
    assert len(terms) == 12 * 12 + 8 * 6 + 8 * 6  # Eq. 1: E_i E_j + V_i F_j + V_j F_i
    at_gap = [t for t in terms if abs(t["r"] - gap) < 1e-12]
    # each facing vertex interacts with 3 faces
    vf = [t for t in at_gap if t["type"] in (1, 2)]
    per_vertex = {}
    for t in vf:
        key = (t["type"], t["k"] if t["type"] == 1 else t["l"])
        per_vertex[key] = per_vertex.get(key, 0) + 1
    assert len(per_vertex) == g["cube_facing_vertices"]
    assert set(per_vertex.values()) == {int(g["cube_faces_per_facing_vertex"])}
    # each facing edge interacts with 5 edges
    ee = [t for t in at_gap if t["type"] == 0]
    verts = sh[0]["verts"]
    facing_i = [k for k, e in enumerate(sh[0]["edges"]) if np.all(verts[e, 0] > 0)]
    facing_j = [k for k, e in enumerate(sh[0]["edges"]) if np.all(verts[e, 0] < 0)]
    assert len(facing_i) + len(facing_j) == g["cube_facing_edges"]
    for k in facing_i:
        assert sum(1 for t in ee if t["k"] == k) == g["cube_edges_per_facing_edge"]
    for l in facing_j:
        assert sum(1 for t in ee if t["l"] == l) == g["cube_edges_per_facing_edge"]
    # total by Eq. 1 (reading R3: the quoted 64 = 8*3 + 8*5 double-counts facing x facing edge pairs)
    assert len(at_gap) == g["cube_total_eq1"] and len(vf) == 24 and len(ee) == 32
    assert min(t["r"] for t in terms) == pytest.approx(gap, abs=1e-14)
    u1, f1 = _wca(gap, 0.3)
    assert sums["u"] == pytest.approx(56 * u1, rel=1e-12)
    assert sums["Fi"] == pytest.approx([-56 * f1, 0, 0], rel=1e-12, abs=1e-9)


def test_square_and_octahedron_counts(oracle):
    sq = [di.square(1.0, 0.15)]
    terms, sums = oracle.pair_terms(sq, 0, 0, ID, ID, [1.3, 0, 0])
    assert len(terms) == 2 * 4 * 4  # Eq. 2
    assert sum(abs(t["r"] - 0.3) < 1e-12 for t in terms) == 8  # 2 per facing vertex
    octa = [di.octahedron(0.5, 0.075)]
    terms, _ = oracle.pair_terms(octa, 0, 0, ID, ID, [1.15, 0, 0])  # vertex to vertex on an axis
    assert len(terms) == 144 + 48 + 48
    assert sum(abs(t["r"] - 0.15) < 1e-12 for t in terms) == 24


def _sample_feature(verts):
    """Dense samples of a vertex / segment / convex polygon given by its vertex array."""
    verts = np.asarray(verts)
    if len(verts) == 1:
        return verts
    if len(verts) == 2:
        t = np.linspace(0, 1, 301)[:, None]
        return verts[0] + t * (verts[1] - verts[0])
    u = np.linspace(0, 1, 61)
    uu, vv = np.meshgrid(u, u)
    keep = uu + vv <= 1 + 1e-12
    uu, vv = uu[keep][:, None], vv[keep][:, None]
    return np.concatenate([verts[0] + uu * (verts[k] - verts[0]) + vv * (verts[k + 1] - verts[0])
                           for k in range(1, len(verts) - 1)])


@pytest.mark.parametrize("maker", [lambda: di.cube(1.0, 0.15), lambda: di.tetrahedron(0.5, 0.05),
                                   lambda: di.regular_polygon(5, 0.5, 0.05)])
def test_every_term_distance_vs_brute_force(oracle, maker):
    """r* of every Eq. 1 / Eq. 2 term of random poses against dense sampling of both features."""
    sh = [maker()]
    dim = sh[0]["dim"]
    rng = np.random.default_rng(5)
    for trial in range(3):
        st = di.two_particle_state(sh[0], sh[0], seed=100 + trial)
        qi, qj = st["quat"]
        d = st["pos"][1, :3] - st["pos"][0, :3]
        terms, _ = oracle.pair_terms(sh, 0, 0, qi, qj, d, dim=dim)
        a = sh[0]["verts"] @ rotmat(qi).T
        b = sh[0]["verts"] @ rotmat(qj).T + d
        ed, fc = sh[0]["edges"], sh[0]["faces"]
        for t in terms:
            if t["type"] == 0:
                fa, fb = a[ed[t["k"]]], b[ed[t["l"]]]
            elif t["type"] == 1:
                fa, fb = a[[t["k"]]], b[fc[t["l"]]]
            elif t["type"] == 2:
                fa, fb = a[fc[t["k"]]], b[[t["l"]]]
            elif t["type"] == 3:
                fa, fb = a[[t["k"]]], b[ed[t["l"]]]
            else:
                fa, fb = a[ed[t["k"]]], b[[t["l"]]]
            pa, pb = _sample_feature(fa), _sample_feature(fb)
            brute = np.sqrt(((pa[:, None, :] - pb[None, :, :]) ** 2).sum(-1).min())
            assert t["r"] <= brute + 1e-12, (t, brute)
            assert brute - t["r"] < 0.03, (t, brute)  # sampling resolution
            # the reported nearest points lie on the features they belong to
            assert np.linalg.norm(t["ci"] - pa, axis=1).min() < 0.02
            assert np.linalg.norm(t["cj"] - pb, axis=1).min() < 0.02


# ---------------------------------------------------------------------------------------------------------------
# closed forms
# ---------------------------------------------------------------------------------------------------------------
def test_aligned_cube_lattice_closed_form(oracle):
    """Aligned unit cubes on a SC lattice of spacing 1 + sigma: every face pair has 56 terms at r = sigma."""
    sigma = 0.3
    st = di.lattice_state(3, [di.cube(1.0, sigma / 2)], (4, 4, 4), 1.0 + sigma, orient="aligned")
    f, t, w, cnt = oracle.compute(st)
    assert np.allclose(f[:, 3], 0.5 * 6 * 56 * 1.0, rtol=1e-11)  # U_i = 168 eps
    assert np.abs(f[:, :3]).max() < 1e-8 and np.abs(t[:, :3]).max() < 1e-8
    trw = (w[:, 0] + w[:, 3] + w[:, 5]).sum()
    assert trw == pytest.approx(64 * 3 * 56 * 24 * (1 + sigma) / sigma, rel=1e-11)
    assert cnt[2] == 64 * 6 * 56  # active terms over directed pairs


def test_aligned_square_lattice_closed_form(oracle):
    sigma = 0.3
    st = di.lattice_state(2, [di.square(1.0, sigma / 2)], (4, 4), 1.0 + sigma, orient="aligned")
    f, t, w, cnt = oracle.compute(st)
    assert np.allclose(f[:, 3], 0.5 * 4 * 8, rtol=1e-11)
    assert np.abs(f[:, :3]).max() < 1e-9 and np.abs(t).max() < 1e-9


def test_one_vertex_shapes_reduce_to_central_wca(oracle):
    """spheres = central WCA.  3D: one (degenerate) edge-edge term; 2D disk: two vertex-edge terms."""
    rng = np.random.default_rng(3)
    rho = 0.5
    for dim, mult, shape in ((3, 1, di.sphere(rho)), (2, 2, di.disk(rho))):
        n = 24
        pos = np.zeros((n, 4))
        pos[:, :dim] = rng.uniform(-2.0, 2.0, (n, dim))
        box = np.array([4.0, 4.0, 4.0])
        st = dict(dim=dim, shapes=[shape], box=box, pos=pos, quat=di.random_quaternions(rng, n) if dim == 3
                  else di.planar_quaternions(rng.uniform(0, 6, n)), shape_id=np.zeros(n, np.int32), epsilon=0.7, N=n)
        f, t, w, _ = oracle.compute(st, use_reject=False)
        F = np.zeros((n, 3))
        U = np.zeros(n)
        W = np.zeros((n, 6))
        for i in range(n):
            for j in range(n):
                if i == j:
                    continue
                d = pos[j, :3] - pos[i, :3]
                d -= box * np.round(d / box)
                if dim == 2:
                    d[2] = 0
                r = np.linalg.norm(d)
                u, fm = _wca(r, 2 * rho, 0.7)
                fij = -mult * fm * d / r
                F[i] += fij
                U[i] += 0.5 * mult * u
                rij = -d
                W[i] += 0.5 * np.array([rij[0] * fij[0], rij[0] * fij[1], rij[0] * fij[2], rij[1] * fij[1],
                                        rij[1] * fij[2], rij[2] * fij[2]])
        assert U.max() > 1.0  # the state really interacts
        assert np.allclose(f[:, :3], F, rtol=1e-11, atol=1e-10) and np.allclose(f[:, 3], U, rtol=1e-11)
        assert np.abs(t).max() < 1e-12  # central force on a point body: no torque
        assert np.allclose(w, W, rtol=1e-11, atol=1e-10)


def test_rod_pair_is_spherocylinder_axis_distance(oracle):
    """3D rod (2 vertices, 1 edge, no face): exactly one Eq. 1 term, WCA of the axis-axis distance."""
    rod = di.rod(1.0, 0.2)
    qa = quat_from_axis_angle([0, 1, 0], math.pi / 2)  # axis along x
    qb = quat_from_axis_angle([1, 0, 0], math.pi / 2)  # axis along -y / y
    terms, sums = oracle.pair_terms([rod], 0, 0, qa, qb, [0.1, 0.05, 0.41])
    assert len(terms) == 1 and terms[0]["r"] == pytest.approx(0.41, abs=1e-14)  # crossed rods: gap along z
    u, fm = _wca(0.41, 0.4)
    assert sums["u"] == pytest.approx(u, rel=1e-12) and sums["Fi"] == pytest.approx([0, 0, -fm], abs=1e-9)
    # rod i lies on the x axis, rod j on the line (0.1, y, 0.41): the force acts on i at (0.1, 0, 0) and on j at
    # (0.1, 0, 0.41) = x_j + (0, -0.05, 0)  (torque from the interaction point on each particle)
    assert sums["Ti"] == pytest.approx(np.cross([0.1, 0.0, 0.0], [0, 0, -fm]), abs=1e-9)
    assert sums["Tj"] == pytest.approx(np.cross([0.0, -0.05, 0.0], [0, 0, fm]), abs=1e-9)


# ---------------------------------------------------------------------------------------------------------------
# conservativeness, virial, balances, invariances
# ---------------------------------------------------------------------------------------------------------------
def _dense(kind):
    if kind == "cubes":
        # rotations well above the parallel-edge threshold (1e-3 rad) so that F is the exact gradient (R5)
        st = di.lattice_state(3, [di.cube(1.0, 0.15)], (4, 4, 4), 1.32, seed=4, jitter=0.03, orient="random")
        rng = np.random.default_rng(8)
        ang = rng.uniform(0.05, 0.25, st["N"])
        ax = rng.standard_normal((st["N"], 3))
        ax /= np.linalg.norm(ax, axis=1, keepdims=True)
        st["quat"] = np.concatenate([np.cos(ang / 2)[:, None], np.sin(ang / 2)[:, None] * ax], 1)
        return st
    if kind == "mixed":
        return di.lattice_state(3, [di.octahedron(0.5, 0.075), di.tetrahedron(0.5, 0.05)], (3, 3, 3), 0.93, seed=6,
                                jitter=0.03, shape_fractions=(0.5, 0.5))
    if kind == "pentagons":
        return di.lattice_state(2, [di.regular_polygon(5, 0.5, 0.05)], (4, 4), 0.95, seed=7, jitter=0.02)
    raise ValueError(kind)


def _total_u(oracle, st, pos=None, quat=None):
    f, _, _, cnt = oracle.compute(st, pos=pos, quat=quat)
    return f[:, 3].sum(), cnt


@pytest.mark.parametrize("kind", ["cubes", "mixed", "pentagons"])
def test_force_and_torque_are_minus_gradient_of_u(oracle, kind):
    st = _dense(kind)
    f, t, w, cnt = oracle.compute(st)
    assert cnt[2] > 20 and cnt[3] == 0, cnt  # interacting, nothing degenerate
    assert cnt[4] == 0  # parallel-edge branch not taken: F is the exact gradient here
    fmax = np.abs(f[:, :3]).max()
    dim = st["dim"]
    h = 1e-6 * 0.1
    rng = np.random.default_rng(0)
    active = np.nonzero(np.abs(f[:, :3]).sum(1) > 0)[0]
    for i in rng.choice(active, 4, replace=False):
        for a in range(dim):
            p = st["pos"].copy()
            p[i, a] += h
            up, _ = _total_u(oracle, st, pos=p)
            p[i, a] -= 2 * h
            um, _ = _total_u(oracle, st, pos=p)
            assert abs(f[i, a] + (up - um) / (2 * h)) < 2e-6 * fmax, (i, a)
        for a in ([2] if dim == 2 else [0, 1, 2]):
            axis = np.eye(3)[a]
            hq = 1e-7
            us = []
            for s in (+1, -1):
                q = st["quat"].copy()
                q[i] = quat_mul(quat_from_axis_angle(axis, s * hq), q[i])  # lab-frame rotation about x_i
                us.append(_total_u(oracle, st, quat=q)[0])
            assert abs(t[i, a] + (us[0] - us[1]) / (2 * hq)) < 2e-6 * max(np.abs(t[:, :3]).max(), 1.0), (i, a)


@pytest.mark.parametrize("kind", ["cubes", "pentagons"])
def test_virial_is_minus_du_dlambda(oracle, kind):
    st = _dense(kind)
    _, _, w, _ = oracle.compute(st)
    trw = (w[:, 0] + w[:, 3] + w[:, 5]).sum()
    h = 1e-7
    us = []
    for lam in (1 + h, 1 - h):
        s2 = dict(st)
        s2["pos"] = st["pos"] * lam
        s2["box"] = st["box"] * lam
        us.append(oracle.compute(s2)[0][:, 3].sum())
    assert trw == pytest.approx(-(us[0] - us[1]) / (2 * h), rel=2e-6)


@pytest.mark.parametrize("kind", ["cubes", "mixed", "pentagons"])
def test_virial_off_diagonals_are_minus_du_dshear(oracle, kind):
    """Pins every component of the virial tensor, off-diagonals and their index order included: for an isolated
    cluster (huge box: no image involved) sheared as x^a += gamma x^b with orientations fixed,
    dU/dgamma = sum_i dU/dx_i^a x_i^b = -sum_i F_i^a x_i^b = -sum_pairs r_ij^b F_ij^a = -W^{ba}
    with W^{ab} = r_ij^a F_ij^b (R12).  Transposing a component (r^b F^a stored as W^{ab}) fails here
    because F is not central: W is not symmetric.  The lower triangle, which is not stored, is checked against the
    angular-momentum balance: W^{ab} - W^{ba} = -(sum_i tau_i) . e_c for (a, b, c) cyclic."""
    st = _dense(kind)
    st["box"] = st["box"] * 20
    f, t, w, cnt = oracle.compute(st, use_reject=False)
    assert cnt[2] > 20 and cnt[4] == 0
    wsum = w.sum(0)                                        # xx, xy, xz, yy, yz, zz
    dim = st["dim"]
    comp = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (1, 1): 3, (1, 2): 4, (2, 2): 5}
    h = 1e-7
    scale = np.abs(wsum).max()

    def du_dshear(a, b):                                   # x^a += gamma x^b
        us = []
        for g in (+h, -h):
            p = st["pos"].copy()
            p[:, a] += g * st["pos"][:, b]
            us.append(oracle.compute(st, pos=p, use_reject=False)[0][:, 3].sum())
        return (us[0] - us[1]) / (2 * h)

    asym = 0.0
    for (a, b), k in comp.items():
        if a >= dim or b >= dim:
            continue
        # stored component W^{ab} (a <= b) is minus the derivative under x^b += gamma x^a
        assert wsum[k] == pytest.approx(-du_dshear(b, a), abs=3e-6 * scale), (a, b)
        if a != b:
            lower = -du_dshear(a, b)                       # W^{ba}
            c = 3 - a - b
            sign = 1.0 if (a, b, c) in ((0, 1, 2), (1, 2, 0), (2, 0, 1)) else -1.0
            # sum_i tau_i = -sum_pairs r_ij x F_ij, and (r x F)_c = sign (r^a F^b - r^b F^a)
            assert wsum[k] - lower == pytest.approx(-sign * t[:, c].sum(), abs=3e-6 * scale), (a, b)
            asym = max(asym, abs(wsum[k] - lower))
    assert asym > 1e-3 * scale                             # the tensor really is asymmetric: a transposition would show


@pytest.mark.parametrize("kind", ["cubes", "mixed", "pentagons"])
def test_momentum_and_angular_momentum_balance(oracle, kind):
    st = _dense(kind)
    # non-periodic cluster: put the same particles in a huge box so that x_i x F_i is meaningful
    st["box"] = st["box"] * 20
    f, t, _, cnt = oracle.compute(st, use_reject=False)
    assert cnt[2] > 20
    fmax = np.abs(f[:, :3]).max()
    assert np.abs(f[:, :3].sum(0)).max() < 1e-11 * fmax
    ang = (np.cross(st["pos"][:, :3], f[:, :3]) + t[:, :3]).sum(0)
    assert np.abs(ang).max() < 1e-10 * fmax


def test_balance_holds_in_parallel_edge_branch(oracle):
    st = di.dense_state("cubes", 4, seed=2, max_angle=5e-4, jitter=0.02)  # all rotations below the 1e-3 threshold
    st["box"] = st["box"] * 20
    f, t, _, cnt = oracle.compute(st, use_reject=False)
    assert cnt[4] > 10  # the branch is taken
    fmax = np.abs(f[:, :3]).max()
    assert np.abs(f[:, :3].sum(0)).max() < 1e-11 * fmax
    assert np.abs((np.cross(st["pos"][:, :3], f[:, :3]) + t[:, :3]).sum(0)).max() < 1e-10 * fmax


def test_reject_shortcut_changes_nothing(oracle):
    st = _dense("mixed")
    a = oracle.compute(st, use_reject=True)
    b = oracle.compute(st, use_reject=False)
    for x, y in zip(a[:3], b[:3]):
        assert np.array_equal(x, y)
    assert a[3][2] == b[3][2]


def test_cell_grid_variant_is_the_all_pairs_sum_bit_for_bit(oracle):
    """orc_compute_cells against the definition (the all-pairs loop with the exact reject): identical bits for force,
    torque, energy, virial and counters, on dense lattices, a mixed-shape state, boxes with fewer than three cells
    along an axis, a shuffled random fluid with particles outside the box, and a row subset."""
    rng = np.random.default_rng(3)
    states = [_dense("cubes"), _dense("mixed"), _dense("pentagons"), di.dense_state("cubes", 6), di.make_config(2, scale=2)]
    gas = di.lattice_state(3, [di.octahedron(0.5, 0.075), di.tetrahedron(0.5, 0.05)], (7, 5, 3), 1.25, seed=9,
                           jitter=0.12, shape_fractions=(0.4, 0.6))
    perm = rng.permutation(gas["N"])
    for k in ("pos", "quat", "shape_id"):
        gas[k] = gas[k][perm]
    gas["pos"][::3, :3] += gas["box"] * rng.integers(-2, 3, (len(gas["pos"][::3]), 3))   # images outside the box
    states.append(gas)
    for st in states:
        a = oracle.compute(st)
        b = oracle.compute(st, cells=True)
        assert a[3][0] > 0
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        sub = rng.choice(st["N"], 9, replace=False).astype(np.int32)
        c = oracle.compute(st, subset=sub, cells=True)
        assert np.array_equal(c[0], a[0][sub]) and np.array_equal(c[1], a[1][sub]) and np.array_equal(c[2], a[2][sub])


@pytest.mark.parametrize("kind", ["cubes", "pentagons"])
def test_translation_and_rotation_invariance(oracle, kind):
    st = _dense(kind)
    f0, t0, w0, _ = oracle.compute(st)
    # translation across the periodic boundary
    s2 = dict(st)
    shift = np.array([0.37, -0.81, 0.55 if st["dim"] == 3 else 0.0, 0])
    p = st["pos"] + shift
    for a in range(st["dim"]):
        p[:, a] -= st["box"][a] * np.round(p[:, a] / st["box"][a])
    s2["pos"] = p
    f1, t1, w1, _ = oracle.compute(s2)
    scale = np.abs(f0[:, :3]).max()
    assert np.allclose(f1, f0, atol=1e-9 * scale) and np.allclose(t1, t0, atol=1e-9 * scale)
    assert np.allclose(w1, w0, atol=1e-9 * scale)
    # rotation by 90 degrees about z maps the (square / cubic) box onto itself: F, tau co-rotate, U invariant
    qz = quat_from_axis_angle([0, 0, 1], math.pi / 2)
    R = rotmat(qz)
    s3 = dict(st)
    s3["pos"] = np.concatenate([st["pos"][:, :3] @ R.T, np.zeros((st["N"], 1))], 1)
    s3["quat"] = np.array([quat_mul(qz, q) for q in st["quat"]])
    f2, t2, _, _ = oracle.compute(s3)
    assert np.allclose(f2[:, :3], f0[:, :3] @ R.T, atol=1e-9 * scale)
    assert np.allclose(t2[:, :3], t0[:, :3] @ R.T, atol=1e-9 * scale)
    assert np.allclose(f2[:, 3], f0[:, 3], atol=1e-10 * max(1, f0[:, 3].max()))


def test_isolated_pair_arbitrary_rotation(oracle):
    sh = [di.truncated_icosahedron(0.5, 0.05), di.tetrahedron(0.5, 0.05)]
    rng = np.random.default_rng(21)
    found = 0
    for seed in range(200):
        st = di.two_particle_state(sh[0], sh[1], seed=seed)
        f0, t0, _, cnt = oracle.compute(st)
        if cnt[2] == 0 or cnt[3] > 0:
            continue
        found += 1
        q = di.random_quaternions(rng, 1)[0]
        R = rotmat(q)
        s2 = dict(st)
        s2["pos"] = np.concatenate([st["pos"][:, :3] @ R.T, np.zeros((2, 1))], 1)
        s2["quat"] = np.array([quat_mul(q, x) for x in st["quat"]])
        f1, t1, _, _ = oracle.compute(s2)
        sc = np.abs(f0[:, :3]).max()
        assert np.allclose(f1[:, :3], f0[:, :3] @ R.T, atol=1e-9 * sc)
        assert np.allclose(t1[:, :3], t0[:, :3] @ R.T, atol=1e-9 * sc)
        assert f1[:, 3] == pytest.approx(f0[:, 3], rel=1e-10)
        if found >= 5:
            break
    assert found >= 5
