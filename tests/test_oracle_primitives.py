"""Pins for the oracle's nearest-point primitives and WCA (CPU only).

Each pin checks the oracle against something other than itself: brute-force dense sampling of the features
(north_star: "brute-force dense sampling of feature points for r* on tiny inputs"), hand-derived special cases, the
closed forms of Eq. 3-4 and the value PAPER.md:61 prints.
"""
import numpy as np
import pytest

from _util import golden

NS = 2001  # samples per segment: sampling error of the brute-force minimum <= L / (NS - 1)


def _seg_points(a, b, n=NS):
    t = np.linspace(0.0, 1.0, n)[:, None]
    return a + t * (b - a)


def test_point_segment_vs_dense_sampling(oracle):
    rng = np.random.default_rng(11)
    regions = set()
    for _ in range(300):
        a, b, p = rng.uniform(-1, 1, (3, 3))
        if rng.random() < 0.3:
            p = a + (b - a) * rng.uniform(-1.5, 2.5) + 0.05 * rng.standard_normal(3)
        c, t = oracle.point_segment(p, a, b)
        brute = np.linalg.norm(_seg_points(a, b) - p, axis=1).min()
        r = np.linalg.norm(p - c)
        h = np.linalg.norm(b - a) / (NS - 1)
        assert r <= brute + 1e-12 and brute - r <= h
        assert np.allclose(c, a + t * (b - a), atol=1e-14)
        regions.add(0 if t == 0 else (2 if t == 1 else 1))
    assert regions == {0, 1, 2}
    # degenerate edge: zero length => nearest point is the end point itself
    c, t = oracle.point_segment([1, 2, 3], [0, 0, 0], [0, 0, 0])
    assert t == 0 and np.all(c == 0)
    # textbook special case: foot of the perpendicular
    c, t = oracle.point_segment([0.25, 3.0, 0], [0, 0, 0], [1, 0, 0])
    assert np.allclose(c, [0.25, 0, 0]) and t == pytest.approx(0.25)


def test_segment_segment_vs_dense_sampling(oracle):
    rng = np.random.default_rng(12)
    cases = set()
    n = 401
    for trial in range(400):
        p1, q1, p2, q2 = rng.uniform(-1, 1, (4, 3))
        if trial % 4 == 1:  # skew but short: favours end-point/end-point cases
            q1 = p1 + 0.3 * rng.standard_normal(3)
            q2 = p2 + 0.3 * rng.standard_normal(3)
        if trial % 4 == 2:  # crossing-ish: favours interior/interior
            m = rng.uniform(-0.2, 0.2, 3)
            u, v = rng.standard_normal((2, 3))
            p1, q1 = m - u, m + u
            off = 0.1 * np.cross(u, v) / np.linalg.norm(np.cross(u, v))
            p2, q2 = m - v + off, m + v + off
        c1, c2, br = oracle.segment_segment(p1, q1, p2, q2)
        assert br == 0
        a, b = _seg_points(p1, q1, n), _seg_points(p2, q2, n)
        brute = np.sqrt(((a[:, None, :] - b[None, :, :]) ** 2).sum(-1).min())
        r = np.linalg.norm(c1 - c2)
        h = 0.5 * (np.linalg.norm(q1 - p1) + np.linalg.norm(q2 - p2)) / (n - 1)
        assert r <= brute + 1e-12 and brute - r <= h, (trial, r, brute)
        # the returned points lie on their segments
        s = np.dot(c1 - p1, q1 - p1) / np.dot(q1 - p1, q1 - p1)
        t = np.dot(c2 - p2, q2 - p2) / np.dot(q2 - p2, q2 - p2)
        assert -1e-12 <= s <= 1 + 1e-12 and -1e-12 <= t <= 1 + 1e-12
        assert np.allclose(c1, p1 + s * (q1 - p1), atol=1e-12) and np.allclose(c2, p2 + t * (q2 - p2), atol=1e-12)
        cls = lambda x: 0 if x < 1e-12 else (2 if x > 1 - 1e-12 else 1)
        cases.add((cls(s), cls(t)))
    # every clamp case of the (s,t) box was exercised: interior, 4 edges, 4 corners
    assert cases == {(i, j) for i in range(3) for j in range(3)}


def test_segment_segment_special_cases(oracle):
    # crossing perpendicular segments at height 0.5: unique answer, hand-derived
    c1, c2, br = oracle.segment_segment([-1, 0, 0], [1, 0, 0], [0.25, -1, 0.5], [0.25, 1, 0.5])
    assert br == 0 and np.allclose(c1, [0.25, 0, 0]) and np.allclose(c2, [0.25, 0, 0.5])
    # zero-length segments reduce to point-segment / point-point
    c1, c2, br = oracle.segment_segment([0, 0, 0], [0, 0, 0], [-1, 1, 0], [3, 1, 0])
    assert br == 2 and np.allclose(c1, 0) and np.allclose(c2, [0, 1, 0])
    c1, c2, br = oracle.segment_segment([-1, 1, 0], [3, 1, 0], [0.5, 0, 0], [0.5, 0, 0])
    assert br == 2 and np.allclose(c1, [0.5, 1, 0]) and np.allclose(c2, [0.5, 0, 0])
    c1, c2, br = oracle.segment_segment([1, 2, 3], [1, 2, 3], [4, 6, 3], [4, 6, 3])
    assert br == 2 and np.linalg.norm(c1 - c2) == pytest.approx(5.0)


def test_parallel_edge_rule(oracle):
    """for (near-)parallel edges the interaction point is the midpoint of the overlap (reading R5)."""
    # exactly parallel, partial overlap [0.5, 1] of segment 1; distance = common perpendicular = 0.2
    c1, c2, br = oracle.segment_segment([0, 0, 0], [1, 0, 0], [0.5, 0.2, 0], [2.0, 0.2, 0])
    assert br == 1
    assert np.allclose(c1, [0.75, 0, 0]) and np.allclose(c2, [0.75, 0.2, 0])
    # r equals the true minimum distance for exactly parallel edges (dense sampling)
    a, b = _seg_points(np.array([0., 0, 0]), np.array([1., 0, 0]), 401), _seg_points(np.array([0.5, 0.2, 0]), np.array([2.0, 0.2, 0]), 401)
    assert np.linalg.norm(c1 - c2) == pytest.approx(np.sqrt(((a[:, None] - b[None]) ** 2).sum(-1).min()), abs=1e-12)
    # antiparallel works the same
    c1, c2, br = oracle.segment_segment([0, 0, 0], [1, 0, 0], [2.0, 0.2, 0], [0.5, 0.2, 0])
    assert br == 1 and np.allclose(c1, [0.75, 0, 0]) and np.allclose(c2, [0.75, 0.2, 0])
    # symmetric in the two edges (so F_ij = -F_ji whichever particle is called i)
    c2b, c1b, br = oracle.segment_segment([2.0, 0.2, 0], [0.5, 0.2, 0], [0, 0, 0], [1, 0, 0])
    assert br == 1 and np.allclose(c1b, c1) and np.allclose(c2b, c2)
    # parallel but no overlap (collinear end-to-end): falls through to the general routine => end points
    c1, c2, br = oracle.segment_segment([0, 0, 0], [1, 0, 0], [1.5, 0, 0], [2.5, 0, 0])
    assert br == 0 and np.allclose(c1, [1, 0, 0]) and np.allclose(c2, [1.5, 0, 0])
    # just inside / just outside the threshold sin^2(theta) < eps_par = 1e-6
    for ang, expect in ((0.9e-3, 1), (1.1e-3, 0)):
        d = np.array([np.cos(ang), np.sin(ang), 0.0])
        p2 = np.array([0.1, 0.0, 0.3])
        _, _, br = oracle.segment_segment([0, 0, 0], [1, 0, 0], p2, p2 + d)
        assert br == expect
    # eps_par = 0 disables the rule
    _, _, br = oracle.segment_segment([0, 0, 0], [1, 0, 0], [0.5, 0.2, 0], [2.0, 0.2, 0], eps_par=0.0)
    assert br == 0


def test_near_parallel_branch_stays_within_its_error_bound(oracle):
    """PAPER.md:59 gives no formula for 'sufficiently close to parallel' edges; reading R5 takes the midpoints of the
    overlap intervals.  What mathematics still fixes for 0 < theta < 1e-3: both points lie on their segments, the
    distance between them is never below the true minimum, and it exceeds it by at most sin(theta) max(L1, L2)
    (the two lines diverge by at most that much over the overlap)."""
    rng = np.random.default_rng(21)
    n = 1601
    taken = 0
    for trial in range(200):
        theta = 10.0 ** rng.uniform(-6, np.log10(0.99e-3))
        p1 = rng.uniform(-1, 1, 3)
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        w = np.cross(u, rng.standard_normal(3))
        w /= np.linalg.norm(w)
        l1, l2 = rng.uniform(0.3, 2.0, 2)
        q1 = p1 + l1 * u
        d2 = (np.cos(theta) * u + np.sin(theta) * w) * (1 if trial % 2 else -1)
        n3 = np.cross(u, w)
        start = p1 + rng.uniform(-0.5, 0.9) * l1 * u + rng.uniform(0.05, 0.4) * (n3 if trial % 3 else w)
        p2, q2 = start, start + l2 * d2
        c1, c2, br = oracle.segment_segment(p1, q1, p2, q2)
        if br != 1:
            continue                                       # no overlap: the general routine (pinned above)
        taken += 1
        s = np.dot(c1 - p1, q1 - p1) / l1 ** 2
        t = np.dot(c2 - p2, q2 - p2) / l2 ** 2
        assert 0 <= s <= 1 and 0 <= t <= 1
        assert np.allclose(c1, p1 + s * (q1 - p1), atol=1e-13) and np.allclose(c2, p2 + t * (q2 - p2), atol=1e-13)
        a, b = _seg_points(p1, q1, n), _seg_points(p2, q2, n)
        brute = np.sqrt(((a[:, None, :] - b[None, :, :]) ** 2).sum(-1).min())
        r = np.linalg.norm(c1 - c2)
        h = 0.5 * (l1 + l2) / (n - 1)                      # sampling error of the brute-force minimum
        assert r >= brute - h - 1e-12
        assert r - brute <= np.sin(theta) * max(l1, l2) + 1e-12, (trial, theta, r, brute)
    assert taken > 100


def _polygon_samples(poly, n=160):
    """Dense samples of a convex planar polygon: fan triangles sampled on a barycentric grid (incl. boundary)."""
    u = np.linspace(0, 1, n)
    uu, vv = np.meshgrid(u, u)
    keep = uu + vv <= 1 + 1e-12
    uu, vv = uu[keep], vv[keep]
    pts = []
    for k in range(1, len(poly) - 1):
        a, b, c = poly[0], poly[k], poly[k + 1]
        pts.append(a + uu[:, None] * (b - a) + vv[:, None] * (c - a))
    return np.concatenate(pts)


def test_point_polygon_vs_dense_sampling(oracle):
    rng = np.random.default_rng(13)
    kinds = set()
    for trial in range(120):
        nv = int(rng.integers(3, 7))
        ang = np.sort(rng.uniform(0, 2 * np.pi, nv))
        if np.diff(np.concatenate([ang, [ang[0] + 2 * np.pi]])).max() > np.pi * 0.95:
            continue  # keep the polygon convex and non-degenerate
        rad = 0.7
        flat = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros(nv)], 1)
        # random rigid placement
        q = rng.standard_normal(4)
        q /= np.linalg.norm(q)
        from _util import rotmat
        poly = flat @ rotmat(q).T + rng.uniform(-0.3, 0.3, 3)
        p = rng.uniform(-1.2, 1.2, 3)
        c, inside = oracle.point_polygon(p, poly)
        samples = _polygon_samples(poly)
        brute = np.linalg.norm(samples - p, axis=1).min()
        r = np.linalg.norm(p - c)
        h = 2 * rad * 1.5 / 159
        assert r <= brute + 1e-12 and brute - r <= h, (trial, r, brute)
        # c lies in the face plane
        nrm = np.cross(poly[1] - poly[0], poly[2] - poly[0])
        assert abs(np.dot(c - poly[0], nrm)) < 1e-12
        if inside:
            kinds.add("interior")
            assert np.allclose(np.cross(p - c, nrm), 0, atol=1e-12)  # c is the perpendicular foot
        else:
            d = np.linalg.norm(poly - c, axis=1).min()
            kinds.add("vertex" if d < 1e-12 else "edge")
    assert kinds == {"interior", "edge", "vertex"}


def test_point_polygon_special_cases(oracle):
    sq = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 0]], dtype=float)
    c, inside = oracle.point_polygon([0.3, 0.6, 2.0], sq)  # above the interior: perpendicular foot
    assert inside == 1 and np.allclose(c, [0.3, 0.6, 0])
    c, inside = oracle.point_polygon([0.3, 0.6, -2.0], sq)  # faces are two-sided
    assert inside == 1 and np.allclose(c, [0.3, 0.6, 0])
    c, inside = oracle.point_polygon([1.5, 0.5, 0.2], sq)  # beyond an edge: nearest point on the boundary edge
    assert inside == 0 and np.allclose(c, [1.0, 0.5, 0])
    c, inside = oracle.point_polygon([2.0, 3.0, 1.0], sq)  # beyond a corner: the corner (closed polygon, R2)
    assert inside == 0 and np.allclose(c, [1, 1, 0])
    c, inside = oracle.point_polygon([0.5, 0.5, 0.0], sq[::-1].copy())  # orientation of the vertex list is irrelevant
    assert inside == 1 and np.allclose(c, [0.5, 0.5, 0])
    # the diagonal of a quad is NOT a feature: a point above the diagonal sees one nearest point (face = polygon, R1)
    c, inside = oracle.point_polygon([0.5, 0.5, 0.1], sq)
    assert inside == 1 and np.allclose(c, [0.5, 0.5, 0])


def test_wca_closed_forms(oracle):
    g = golden()
    for sigma, eps in ((0.3, 1.0), (0.1, 2.5), (1.0, 0.7)):
        u, f = oracle.wca(sigma, sigma, eps)
        assert u == pytest.approx(g["wca_u_at_sigma_over_eps"] * eps, rel=1e-14)
        assert f * sigma / eps == pytest.approx(g["wca_f_at_sigma_times_sigma_over_eps"], rel=1e-14)
        rc = g["wca_rcut_over_sigma"] * sigma
        assert oracle.wca(rc * (1 + 1e-12), sigma, eps) == (0.0, 0.0)
        u, f = oracle.wca(rc * (1 - 1e-9), sigma, eps)  # continuous: U, F -> 0 at the cutoff
        assert 0 <= u < 1e-14 * eps + 1e-15 and 0 <= f * sigma / eps < 1e-6
        # LJ written out independently (Eq. 3) and shifted by its value at the cutoff (Eq. 4)
        for r in np.linspace(0.8, 1.12, 9) * sigma:
            lj = lambda x: 4 * eps * ((sigma / x) ** 12 - (sigma / x) ** 6)
            u, f = oracle.wca(r, sigma, eps)
            assert u == pytest.approx(lj(r) - lj(2 ** (1 / 6) * sigma), rel=1e-12, abs=1e-13)
            h = 1e-6 * sigma
            assert f == pytest.approx(-(lj(r + h) - lj(r - h)) / (2 * h), rel=1e-6)
    # a 64-fold interaction reaches 1 kT where a single one reaches 1/64: r = 1.1006 sigma ("10 %")
    u, _ = oracle.wca(g["overcount_isosurface_r_over_sigma"], 1.0, 1.0)
    assert g["cube_total_quoted"] * u == pytest.approx(1.0, abs=5e-3)
