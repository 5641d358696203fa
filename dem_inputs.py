"""Seeded synthetic inputs for the DEM hot path (shapes, particle states, the five BASELINE.json configs).

This module serves BOTH the oracle (`oracle/`) and the CUDA path (`paper_1607_02427_b200/`) and therefore holds
NONE of the method's arithmetic: no nearest-point search, no WCA, no neighbour predicate, no integrator.  It only
builds input data: shape geometry (vertices / edges / planar faces of standard polytopes, mass properties of the
uniform inner shape) and particle states (lattices, random orientations, Maxwell-Boltzmann velocities).

Conventions:
  * positions  : (N,4) float64  x,y,z,0        box centred on the origin, orthorhombic edge lengths `box[3]`
  * quaternions: (N,4) float64  w,x,y,z        unit, scalar first, body -> lab; 2D: (cos t/2, 0, 0, sin t/2)
  * velocities : (N,4) float64  vx,vy,vz,0
  * angmom     : (N,4) float64  Lx,Ly,Lz,0     LAB-frame angular momentum
  * shape ids  : (N,)  int32
  * a shape is a dict: dim, verts (nv,3) [z = 0 in 2D], edges (ne,2) int32, faces (list of CCW-from-outside vertex
    index lists; empty in 2D), rounding, mass, inertia (3,) principal body-frame moments, circumradius.

RNG recipe: numpy default_rng(seed); draws in the order position jitter, orientations, shape ids,
velocities, angular velocities.
"""
from __future__ import annotations

import math
import numpy as np

# --------------------------------------------------------------------------------------------------------------
# shape geometry
# --------------------------------------------------------------------------------------------------------------


def _polygon_shape(verts2, rounding, mass=1.0):
    """2D shape from a CCW vertex list; edge k = (k, (k+1) mod n) (PAPER.md:71 'travelling counterclockwise')."""
    v = np.asarray(verts2, dtype=np.float64).reshape(-1, 2)
    n = len(v)
    if n == 1:
        edges = np.array([[0, 0]], dtype=np.int32)
    elif n == 2:
        edges = np.array([[0, 1]], dtype=np.int32)
    else:
        edges = np.array([[k, (k + 1) % n] for k in range(n)], dtype=np.int32)
    # uniform-lamina polar moment about the centroid (shoelace integrals); vertices are expected to be centred
    izz = 0.0
    if n >= 3:
        x, y = v[:, 0], v[:, 1]
        xn, yn = np.roll(x, -1), np.roll(y, -1)
        cr = x * yn - xn * y
        area = 0.5 * cr.sum()
        cx = ((x + xn) * cr).sum() / (6 * area)
        cy = ((y + yn) * cr).sum() / (6 * area)
        assert abs(cx) < 1e-12 and abs(cy) < 1e-12, "polygon must be centred on its centroid"
        j = (cr * (x * x + x * xn + xn * xn + y * y + y * yn + yn * yn)).sum() / 12.0
        izz = mass * j / area
    v3 = np.zeros((n, 3))
    v3[:, :2] = v
    return dict(dim=2, verts=v3, edges=edges, faces=[], rounding=float(rounding), mass=float(mass),
                inertia=np.array([0.0, 0.0, izz]), circumradius=float(np.linalg.norm(v3, axis=1).max()))


def regular_polygon(n, circumradius, rounding, mass=1.0, phase=0.0):
    ang = phase + 2 * math.pi * np.arange(n) / n
    return _polygon_shape(np.stack([circumradius * np.cos(ang), circumradius * np.sin(ang)], 1), rounding, mass)


def square(edge=1.0, rounding=0.15, mass=1.0):
    h = edge / 2
    return _polygon_shape([[-h, -h], [h, -h], [h, h], [-h, h]], rounding, mass)


def disk(rounding, mass=1.0, inertia=1.0):
    s = _polygon_shape([[0.0, 0.0]], rounding, mass)
    s["inertia"] = np.array([0.0, 0.0, inertia])
    return s


def _hull_faces(verts):
    """Planar polygon faces (CCW seen from outside) of the convex hull of `verts` (coplanar hull triangles merged)."""
    from scipy.spatial import ConvexHull

    v = np.asarray(verts, dtype=np.float64)
    hull = ConvexHull(v)
    scale = np.abs(v).max()
    groups = []  # (unit normal, offset, set of vertex ids)
    for simplex, eq in zip(hull.simplices, hull.equations):
        nrm, off = eq[:3], eq[3]
        for g in groups:
            if np.dot(g[0], nrm) > 1 - 1e-9 and abs(g[1] - off) < 1e-9 * scale:
                g[2].update(int(s) for s in simplex)
                break
        else:
            groups.append([nrm.copy(), float(off), set(int(s) for s in simplex)])
    faces = []
    for nrm, _, ids in groups:
        ids = sorted(ids)
        c = v[ids].mean(0)
        u = v[ids[0]] - c
        u /= np.linalg.norm(u)
        w = np.cross(nrm, u)
        ang = [math.atan2(np.dot(v[i] - c, w), np.dot(v[i] - c, u)) for i in ids]
        order = [ids[k] for k in np.argsort(ang)]
        k0 = order.index(min(order))  # canonical start: smallest vertex id
        faces.append(order[k0:] + order[:k0])
    faces.sort()
    return faces


def _edges_from_faces(faces):
    es = set()
    for f in faces:
        for k in range(len(f)):
            a, b = f[k], f[(k + 1) % len(f)]
            es.add((min(a, b), max(a, b)))
    return np.array(sorted(es), dtype=np.int32).reshape(-1, 2)


def _polyhedron_mass_properties(v, faces):
    """Volume, centroid and inertia tensor (unit density) of a closed polyhedron by signed tetrahedra from the origin."""
    vol = 0.0
    cen = np.zeros(3)
    cov = np.zeros((3, 3))  # integral of x x^T
    canon = (np.ones((3, 3)) + np.eye(3)) / 120.0
    for f in faces:
        for k in range(1, len(f) - 1):
            a = np.stack([v[f[0]], v[f[k]], v[f[k + 1]]], 1)  # columns
            det = np.linalg.det(a)
            vol += det / 6.0
            cen += det / 24.0 * a.sum(1)
            cov += det * a @ canon @ a.T
    cen /= vol
    inertia = np.trace(cov) * np.eye(3) - cov
    return vol, cen, inertia


def convex_polyhedron(verts, rounding, mass=1.0):
    v = np.asarray(verts, dtype=np.float64).reshape(-1, 3)
    faces = _hull_faces(v)
    vol, cen, inert = _polyhedron_mass_properties(v, faces)
    assert vol > 0 and np.abs(cen).max() < 1e-12 * max(1.0, np.abs(v).max()), "polyhedron must be centred"
    inert = inert * (mass / vol)
    off = inert - np.diag(np.diag(inert))
    assert np.abs(off).max() < 1e-10 * np.abs(inert).max(), "vertices must be given in the principal frame"
    return dict(dim=3, verts=v.copy(), edges=_edges_from_faces(faces), faces=faces, rounding=float(rounding),
                mass=float(mass), inertia=np.diag(inert).copy(), circumradius=float(np.linalg.norm(v, axis=1).max()))


def cube(edge=1.0, rounding=0.15, mass=1.0):
    h = edge / 2
    return convex_polyhedron([[x, y, z] for x in (-h, h) for y in (-h, h) for z in (-h, h)], rounding, mass)


def box_shape(lx, ly, lz, rounding, mass=1.0):
    """Rectangular cuboid: an asymmetric top (used by integrator tests)."""
    return convex_polyhedron([[x, y, z] for x in (-lx / 2, lx / 2) for y in (-ly / 2, ly / 2)
                              for z in (-lz / 2, lz / 2)], rounding, mass)


def prism(n, circumradius=0.5, height=0.6, rounding=0.05, mass=1.0):
    """Right prism over a regular n-gon (two n-gon faces, n rectangles): faces with many boundary edges."""
    ang = 2 * math.pi * np.arange(n) / n
    ring = np.stack([circumradius * np.cos(ang), circumradius * np.sin(ang)], 1)
    v = np.concatenate([np.c_[ring, np.full(n, -height / 2)], np.c_[ring, np.full(n, height / 2)]])
    return convex_polyhedron(v, rounding, mass)


def octahedron(circumradius=0.5, rounding=0.075, mass=1.0):
    r = circumradius
    return convex_polyhedron([[r, 0, 0], [-r, 0, 0], [0, r, 0], [0, -r, 0], [0, 0, r], [0, 0, -r]], rounding, mass)


def tetrahedron(circumradius=0.5, rounding=0.05, mass=1.0):
    s = circumradius / math.sqrt(3.0)
    return convex_polyhedron([[s, s, s], [s, -s, -s], [-s, s, -s], [-s, -s, s]], rounding, mass)


def icosahedron(circumradius=0.5, rounding=0.05, mass=1.0):
    p = (1 + math.sqrt(5)) / 2
    v = []
    for a in (-1, 1):
        for b in (-p, p):
            v += [[0, a, b], [a, b, 0], [b, 0, a]]
    v = np.array(v, dtype=np.float64)
    return convex_polyhedron(v * (circumradius / np.linalg.norm(v[0])), rounding, mass)


def truncated_icosahedron(circumradius=0.5, rounding=0.05, mass=1.0):
    """60 vertices / 90 edges / 12 pentagons + 20 hexagons (BASELINE.json config 5)."""
    p = (1 + math.sqrt(5)) / 2
    base = [(0, 1, 3 * p), (1, 2 + p, 2 * p), (p, 2, 2 * p + 1)]
    v = set()
    for b in base:
        for sx in (-1, 1):
            for sy in (-1, 1):
                for sz in (-1, 1):
                    c = (b[0] * sx, b[1] * sy, b[2] * sz)
                    for r in range(3):  # even (cyclic) permutations
                        v.add(tuple(round(c[(k + r) % 3], 12) for k in range(3)))
    v = np.array(sorted(v), dtype=np.float64)
    assert len(v) == 60
    return convex_polyhedron(v * (circumradius / np.linalg.norm(v[0])), rounding, mass)


def triangular_plate(circumradius=0.5, rounding=0.05, mass=1.0):
    """One planar triangular face (PAPER.md:95 'triangular plates'); inertia of the uniform lamina."""
    ang = 2 * math.pi * np.arange(3) / 3
    v = np.stack([circumradius * np.cos(ang), circumradius * np.sin(ang), np.zeros(3)], 1)
    i_in = mass * circumradius ** 2 / 4.0  # equilateral lamina, any in-plane axis through the centroid
    return dict(dim=3, verts=v, edges=np.array([[0, 1], [1, 2], [0, 2]], dtype=np.int32), faces=[[0, 1, 2]],
                rounding=float(rounding), mass=float(mass), inertia=np.array([i_in, i_in, 2 * i_in]),
                circumradius=float(circumradius))


def sphere(rounding, mass=1.0, inertia=None):
    """One vertex + degenerate edge (0,0) + no face: Eq. 1 reduces to one central WCA."""
    i0 = 0.4 * mass * rounding ** 2 if inertia is None else inertia
    return dict(dim=3, verts=np.zeros((1, 3)), edges=np.array([[0, 0]], dtype=np.int32), faces=[],
                rounding=float(rounding), mass=float(mass), inertia=np.array([i0, i0, i0]), circumradius=0.0)


def rod(length, rounding, mass=1.0):
    """Two vertices + one edge: a spherocylinder."""
    h = length / 2
    i_perp = mass * length ** 2 / 12.0
    return dict(dim=3, verts=np.array([[0, 0, -h], [0, 0, h]], dtype=np.float64),
                edges=np.array([[0, 1]], dtype=np.int32), faces=[], rounding=float(rounding), mass=float(mass),
                inertia=np.array([i_perp, i_perp, 0.1 * i_perp]), circumradius=h)


# --------------------------------------------------------------------------------------------------------------
# particle states
# --------------------------------------------------------------------------------------------------------------

WCA_RCUT_FACTOR = 2.0 ** (1.0 / 6.0)  # r_cut^WCA / sigma -- an input constant, used only to size r_cut


def _quat_mul(a, b):
    w1, x1, y1, z1 = a[..., 0], a[..., 1], a[..., 2], a[..., 3]
    w2, x2, y2, z2 = b[..., 0], b[..., 1], b[..., 2], b[..., 3]
    return np.stack([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                     w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2], -1)


def quat_rotate(q, v):
    """Rotate vectors v (…,3) by unit quaternions q (…,4): v_lab = q v q* (used to place inputs, e.g. L_lab)."""
    qv = np.concatenate([np.zeros(v.shape[:-1] + (1,)), v], -1)
    qc = q * np.array([1.0, -1.0, -1.0, -1.0])
    return _quat_mul(_quat_mul(q, qv), qc)[..., 1:]


def random_quaternions(rng, n):
    q = rng.standard_normal((n, 4))
    return q / np.linalg.norm(q, axis=1, keepdims=True)


def planar_quaternions(theta):
    q = np.zeros((len(theta), 4))
    q[:, 0] = np.cos(theta / 2)
    q[:, 3] = np.sin(theta / 2)
    return q


def small_rotation_quaternions(rng, n, max_angle, dim=3):
    """Random rotations by an angle U(0, max_angle) about a random axis (z in 2D)."""
    ang = rng.uniform(0.0, max_angle, n)
    if dim == 2:
        return planar_quaternions(ang * rng.choice([-1.0, 1.0], n))
    ax = rng.standard_normal((n, 3))
    ax /= np.linalg.norm(ax, axis=1, keepdims=True)
    return np.concatenate([np.cos(ang / 2)[:, None], np.sin(ang / 2)[:, None] * ax], 1)


def thermal_velocities(rng, shapes, shape_id, quat, kT, dim):
    """v_a ~ N(0,kT/m), body omega_a ~ N(0,kT/I_a); mean velocity removed. Returns vel, L_lab."""
    n = len(shape_id)
    mass = np.array([s["mass"] for s in shapes])[shape_id]
    inertia = np.stack([s["inertia"] for s in shapes])[shape_id]
    vel = np.zeros((n, 4))
    vel[:, :dim] = rng.standard_normal((n, dim)) * np.sqrt(kT / mass)[:, None]
    vel[:, :dim] -= (vel[:, :dim] * mass[:, None]).sum(0) / mass.sum()
    w = rng.standard_normal((n, 3))
    safe = np.where(inertia > 0, inertia, 1.0)
    w = np.where(inertia > 0, w * np.sqrt(kT / safe), 0.0)
    if dim == 2:
        w[:, :2] = 0.0
    lbody = w * inertia
    ang = np.zeros((n, 4))
    ang[:, :3] = quat_rotate(quat, lbody)
    return vel, ang


def default_rcut(shapes):
    """Exact particle-level cutoff max(R_i + R_j + 2^(1/6) sigma_ij), sigma_ij = rho_i + rho_j."""
    return max(a["circumradius"] + b["circumradius"] + WCA_RCUT_FACTOR * (a["rounding"] + b["rounding"])
               for a in shapes for b in shapes)


def _state(dim, shapes, box, pos, quat, shape_id, rng, kT, **extra):
    n = len(pos)
    p4 = np.zeros((n, 4))
    p4[:, :pos.shape[1]] = pos
    box = np.asarray(box, dtype=np.float64)
    for a in range(dim):  # wrap into the centred box (input placement only)
        p4[:, a] -= box[a] * np.floor(p4[:, a] / box[a] + 0.5)
    shape_id = np.asarray(shape_id, dtype=np.int32)
    vel, ang = thermal_velocities(rng, shapes, shape_id, quat, kT, dim)
    st = dict(dim=dim, shapes=shapes, box=box, pos=p4, quat=quat, shape_id=shape_id, vel=vel, angmom=ang,
              epsilon=1.0, r_cut=default_rcut(shapes), N=n)
    st.update(extra)
    return st


def lattice_state(dim, shapes, cells, spacing, *, seed=0, jitter=0.0, orient="random", max_angle=0.0,
                  shape_fractions=None, triangular=False, kT=1.0, **extra):
    """Particles on a cells[0] x cells[1] (x cells[2]) lattice; see the RNG recipe in the module docstring."""
    rng = np.random.default_rng(seed)
    cells = list(cells) + [1] * (3 - len(cells))
    n = cells[0] * cells[1] * (cells[2] if dim == 3 else 1)
    idx = np.arange(n)
    if dim == 2:
        ix, iy = idx % cells[0], idx // cells[0]
        if triangular:  # row j: y = j a sqrt(3)/2, x = (i + (j mod 2)/2) a   (BASELINE.json config 3)
            pos = np.stack([(ix + 0.5 * (iy % 2)) * spacing, iy * spacing * math.sqrt(3) / 2], 1)
            box = [cells[0] * spacing, cells[1] * spacing * math.sqrt(3) / 2, 1.0]
        else:
            pos = np.stack([ix * spacing, iy * spacing], 1).astype(np.float64)
            box = [cells[0] * spacing, cells[1] * spacing, 1.0]
    else:
        ix, iy, iz = idx % cells[0], (idx // cells[0]) % cells[1], idx // (cells[0] * cells[1])
        pos = np.stack([ix, iy, iz], 1) * float(spacing)
        box = [c * spacing for c in cells]
    pos = pos - np.array(box[:pos.shape[1]]) / 2 + spacing / 2
    pos = pos + rng.uniform(-jitter, jitter, pos.shape)  # draw 1: jitter (drawn even when 0 to fix the stream)
    if orient == "random":  # draw 2: orientations
        quat = planar_quaternions(rng.uniform(0, 2 * math.pi, n)) if dim == 2 else random_quaternions(rng, n)
    elif orient == "small":
        quat = small_rotation_quaternions(rng, n, max_angle, dim)
    else:
        quat = np.tile([1.0, 0, 0, 0], (n, 1))
    if shape_fractions is None:  # draw 3: shape ids
        shape_id = np.zeros(n, dtype=np.int32)
    else:
        counts = [int(round(f * n)) for f in shape_fractions]
        counts[-1] = n - sum(counts[:-1])
        shape_id = rng.permutation(np.repeat(np.arange(len(counts)), counts)).astype(np.int32)
    return _state(dim, shapes, box, pos, quat, shape_id, rng, kT, **extra)  # draws 4, 5: velocities


# --------------------------------------------------------------------------------------------------------------
# BASELINE.json configs 1..5 and supplementary dense parity states (P2)
# --------------------------------------------------------------------------------------------------------------

CONFIG_NAMES = {1: "cfg1_squares_N64", 2: "cfg2_cubes_N512", 3: "cfg3_pentagons_N262144",
                4: "cfg4_octahedra_N262144", 5: "cfg5_trunc_icosa_tetra_N65536"}


def make_config(k, seed=0, scale=1):
    """BASELINE.json config k (1-based). `scale` < 1 is NOT supported; scale > 1 shrinks the lattice edge by that
    integer factor (used only to derive small parity cases with the same recipe)."""
    s = int(scale)
    if k == 1:
        return lattice_state(2, [square(1.0, 0.15)], (8 // s, 8 // s), 1.8, seed=seed, jitter=0.05,
                             dt=1e-4, nsteps=1000, dtype="f64", name=CONFIG_NAMES[1])
    if k == 2:
        return lattice_state(3, [cube(1.0, 0.15)], (8 // s,) * 3, math.sqrt(3) + 0.3, seed=seed,
                             dt=1e-3, nsteps=0, dtype="f32", name=CONFIG_NAMES[2])
    if k == 3:
        return lattice_state(2, [regular_polygon(5, 0.5, 0.05)], (512 // s, 512 // s), 1.1, seed=seed,
                             triangular=True, dt=5e-4, nsteps=1000, dtype="f32", name=CONFIG_NAMES[3])
    if k == 4:
        return lattice_state(3, [octahedron(0.5, 0.075)], (64 // s,) * 3, 1.15, seed=seed,
                             dt=2e-4, nsteps=1000, dtype="f32", name=CONFIG_NAMES[4])
    if k == 5:
        return lattice_state(3, [truncated_icosahedron(0.5, 0.05), tetrahedron(0.5, 0.05)],
                             (64 // s, 32 // s, 32 // s), 1.1, seed=seed, shape_fractions=(0.5, 0.5),
                             dt=2e-4, nsteps=0, dtype="f32", name=CONFIG_NAMES[5])
    raise ValueError(k)


TABLE1_CELLS = {256: (8, 8, 4), 4096: (16, 16, 16), 65536: (64, 32, 32)}
TABLE1_SHAPES = ("sphere", "plate", "cube", "icosahedron")


def table1_state(shape, n, seed=0):
    """Stand-ins for the paper's Table I / Figure 4 workloads ("dense fluids" of spheres, triangular
    plates, cubes and icosahedra at N = 256, 4096, 65536; densities, rounding radii and initial states are not given).
    Start states here: a simple-cubic lattice at a spacing that leaves no overlap, thermal velocities at kT = 1; the
    caller equilibrates with NVE steps before timing.  Spheres: one vertex, rho = 0.5 (sigma = 1), number density 0.8.
    Cubes (edge 1, rho = 0.15): near-aligned at spacing 1.62 (volume fraction of the rounded cube ~0.5).  Icosahedra
    (R = 0.5, rho = 0.05): near-aligned at spacing 1.0 (~0.45).  Plates (R = 0.5, rho = 0.05): random orientations at
    spacing 2R + sigma = 1.1.  Returns a state dict with dt set for the shape's sigma."""
    cells = TABLE1_CELLS[n]
    kw = dict(seed=seed, nsteps=0, dtype="f32", name="table1_%s_N%d" % (shape, n))
    if shape == "sphere":
        return lattice_state(3, [sphere(0.5, inertia=0.1)], cells, 0.8 ** (-1.0 / 3.0), jitter=0.02, orient="none",
                             dt=1e-3, **kw)
    if shape == "cube":
        return lattice_state(3, [cube(1.0, 0.15)], cells, 1.62, jitter=0.02, orient="small", max_angle=0.2,
                             dt=2e-4, **kw)
    if shape == "icosahedron":
        return lattice_state(3, [icosahedron(0.5, 0.05)], cells, 1.0, jitter=0.01, orient="small", max_angle=0.1,
                             dt=1e-4, **kw)
    if shape == "plate":
        return lattice_state(3, [triangular_plate(0.5, 0.05)], cells, 1.1, dt=2e-4, **kw)
    raise ValueError(shape)


def fig3_state(kind, seed=0):
    """Stand-ins for the systems of the paper's short-term energy-conservation test (Fig. 3): "a fluid
    of squares (with edge length 4.24 sigma) in 2D and tetrahedra (with edge length 8.49 sigma) in 3D ... thermalized at
    T* = 1"; N, density and state are not given.  Units sigma = epsilon = m = 1, so the rounding radius is 0.5.  Here:
    32 x 32 squares (circumradius 3) / 8^3 tetrahedra (circumradius 8.49 sqrt(6)/4) on a lattice of spacing
    2R + 1.2 sigma with random orientations, kT = 1; the caller thermalises with NVE steps."""
    if kind == "squares":
        r = 4.24 / math.sqrt(2.0)
        return lattice_state(2, [regular_polygon(4, r, 0.5)], (32, 32), 2 * r + 1.2, seed=seed, nsteps=0, dt=5e-3,
                             dtype="f64", name="fig3_squares_N1024")
    if kind == "tetrahedra":
        r = 8.49 * math.sqrt(6.0) / 4.0
        return lattice_state(3, [tetrahedron(r, 0.5)], (8, 8, 8), 2 * r + 1.2, seed=seed, nsteps=0, dt=5e-3,
                             dtype="f64", name="fig3_tetrahedra_N512")
    raise ValueError(kind)


def dense_state(kind, cells, seed=1, max_angle=0.05, jitter=0.02, spacing=None):
    """P2: dense near-aligned lattices in which many pairs interact through many terms.  Default
    spacings were chosen (with the oracle, offline) so that U/N is a few epsilon: in contact, nothing overlapping.
    `cells` must be large enough that every box edge is >= 2 r_cut (4 for the 3D kinds, 4 for the 2D kinds)."""
    if kind == "squares":
        return lattice_state(2, [square(1.0, 0.15)], (cells, cells), spacing or 1.34, seed=seed, jitter=jitter,
                             orient="small", max_angle=max_angle, name="dense_squares")
    if kind == "pentagons":
        return lattice_state(2, [regular_polygon(5, 0.5, 0.05)], (cells, cells), spacing or 1.055, seed=seed,
                             jitter=jitter / 2, orient="small", max_angle=max_angle, triangular=False,
                             name="dense_pentagons")
    if kind == "cubes":
        return lattice_state(3, [cube(1.0, 0.15)], (cells,) * 3, spacing or 1.34, seed=seed, jitter=jitter,
                             orient="small", max_angle=max_angle, name="dense_cubes")
    if kind == "octahedra":
        # aligned octahedra (R = 0.5) touch vertex to vertex along the axes at spacing 1.0 + r*
        return lattice_state(3, [octahedron(0.5, 0.075)], (cells,) * 3, spacing or 1.18, seed=seed, jitter=jitter,
                             orient="small", max_angle=max_angle, name="dense_octahedra")
    if kind == "mixed":
        return lattice_state(3, [truncated_icosahedron(0.5, 0.05), tetrahedron(0.5, 0.05)], (cells,) * 3,
                             spacing or 1.08, seed=seed, jitter=jitter / 2, orient="random",
                             shape_fractions=(0.5, 0.5), name="dense_mixed")
    raise ValueError(kind)


def two_particle_state(shape_a, shape_b, seed, box=20.0, spread=None):
    """P3: one isolated random pair pose (tests rejection-sample these with the oracle)."""
    rng = np.random.default_rng(seed)
    dim = shape_a["dim"]
    shapes = [shape_a, shape_b]
    reach = default_rcut(shapes) if spread is None else spread
    d = rng.standard_normal(3)
    if dim == 2:
        d[2] = 0.0
    d *= rng.uniform(0.3, 1.0) * reach / np.linalg.norm(d)
    pos = np.stack([-d / 2, d / 2])[:, :3]
    quat = planar_quaternions(rng.uniform(0, 2 * math.pi, 2)) if dim == 2 else random_quaternions(rng, 2)
    return _state(dim, shapes, [box] * 3, pos, quat, [0, 1], rng, 1.0, name="pair")
