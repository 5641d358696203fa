"""GPU parity tests: the CUDA path (through the C ABI) against the FP64 CPU oracle, element by element, on the same
seeded inputs.  Run on the B200 box with `-m gpu`.

Tolerances (north_star): neighbour list bit-exact; per-particle force and torque within 1e-4 (FP32) / 1e-10 (FP64)
of the system's max |F| (floored by eps/sigma, R19); the same bar is applied to energies and the virial.
"""
import math

import numpy as np
import pytest

import dem_inputs as di
from _gpu_util import TOL, assert_neighbors_exact, assert_parity, gpu_compute, round_state, scales

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device: the product has no CPU path")
    import paper_1607_02427_b200 as p

    p.lib()
    return p


# ---------------------------------------------------------------------------------------------------------------
# neighbour list: bit-exact against the all-pairs definition
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dense_squares", "dense_cubes", "dense_mixed"])
def test_neighbors_bit_exact(pkg, oracle, name, precision):
    st = {"cfg1": lambda: di.make_config(1), "cfg2": lambda: di.make_config(2),
          "dense_squares": lambda: di.dense_state("squares", 12), "dense_cubes": lambda: di.dense_state("cubes", 6),
          "dense_mixed": lambda: di.dense_state("mixed", 6)}[name]()
    counts = assert_neighbors_exact(st, precision, oracle)
    assert counts.sum() % 2 == 0


@pytest.mark.parametrize("dim", [2, 3])
def test_neighbors_random_gas_odd_boxes(pkg, oracle, dim):
    """Random points (several per cell, ragged cell occupancy, positions outside the box), boxes with only 2 cells
    along an axis, cutoffs that put many pairs near r_cut."""
    rng = np.random.default_rng(5)
    for box, rc, n in (([7.3, 5.1, 4.4], 1.3, 700), ([4.1, 9.0, 4.05], 2.0, 500), ([30.0, 3.0, 2.9], 1.45, 900)):
        pos = np.zeros((n, 4))
        pos[:, :dim] = rng.uniform(-0.75, 0.75, (n, dim)) * np.array(box[:dim])  # some outside the box
        sh = [di.disk(0.1)] if dim == 2 else [di.sphere(0.1)]
        st = dict(dim=dim, shapes=sh, box=np.array(box), pos=pos, quat=np.tile([1.0, 0, 0, 0], (n, 1)),
                  vel=np.zeros((n, 4)), angmom=np.zeros((n, 4)), shape_id=np.zeros(n, dtype=np.int32), N=n,
                  r_cut=rc, epsilon=1.0)
        for precision in ("f32", "f64"):
            counts = assert_neighbors_exact(st, precision, oracle)
            assert counts.max() > 16  # exercises the capacity regrow


def test_neighbors_full_size_sampled(pkg, oracle):
    """Config 4 at full size (N = 262,144): rows of 4,096 sampled particles against the all-pairs definition."""
    st = di.make_config(4)
    sub = np.random.default_rng(1).choice(st["N"], 4096, replace=False).astype(np.int32)
    assert_neighbors_exact(st, "f32", oracle, subset=sub)


# ---------------------------------------------------------------------------------------------------------------
# force / torque / energy / virial
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_config1_squares(pkg, oracle, precision):
    assert_parity(di.make_config(1), precision, oracle)


@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_config2_cubes(pkg, oracle, precision):
    r = assert_parity(di.make_config(2), precision, oracle)
    assert r["counters"]["pairs_listed"] == 1536 and r["counters"]["terms"] == 1536 * 240


DENSE = [("squares", 12), ("pentagons", 12), ("cubes", 6), ("octahedra", 6), ("mixed", 5)]


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("kind,cells", DENSE)
def test_dense_states(pkg, oracle, kind, cells, precision):
    """P2: dense near-aligned lattices in which many pairs interact through many terms."""
    r = assert_parity(di.dense_state(kind, cells), precision, oracle)
    assert r["counters"]["active"] > 50  # the state really exercises WCA / torque code


@pytest.mark.parametrize("kind,cells,slices", [("cubes", 5, 3), ("cubes", 5, 28), ("squares", 10, 2), ("mixed", 4, 7),
                                               ("octahedra", 5, 1000)])
def test_sliced_pairs_match(pkg, oracle, kind, cells, slices):
    """Several lanes per pair (slices of the outer feature loop) give the same sums."""
    assert_parity(di.dense_state(kind, cells), "f64", oracle, slices=slices)
    assert_parity(di.dense_state(kind, cells), "f32", oracle, slices=slices)


@pytest.mark.parametrize("kind,cells", [("squares", 12), ("pentagons", 12), ("cubes", 6), ("mixed", 5)])
def test_generic_kernel_fp32(pkg, oracle, kind, cells):
    """A DEM_F32 context runs the packed search kernel (default in 3D) or the generic fused kernel (default in 2D,
    always in DEM_F64 contexts); both must find the same contributing terms and the same sums up to rounding."""
    st = di.dense_state(kind, cells)
    a = assert_parity(st, "f32", oracle, kernel=1)
    b = assert_parity(st, "f32", oracle, kernel=0)
    for key in ("active", "degenerate", "parallel", "pairs_evaluated", "terms"):
        assert a["counters"][key] == b["counters"][key], key


@pytest.mark.parametrize("kind,cells,extra", [("cubes", 6, 0.45), ("pentagons", 12, 0.5), ("mixed", 5, 0.5)])
def test_list_with_skin_compacts_out_of_reach_pairs(pkg, oracle, kind, cells, extra):
    """A neighbour list built with a skin holds pairs beyond the interaction reach: the pose kernel drops them from
    the search kernel's work list and writes their zero records; sums and counters must not change."""
    st = di.dense_state(kind, cells)
    r0 = assert_parity(st, "f32", oracle, kernel=0)
    r1 = assert_parity(st, "f32", oracle, r_cut=st["r_cut"] + extra, kernel=0)
    assert r1["counters"]["pairs_listed"] > r0["counters"]["pairs_listed"]
    assert r1["counters"]["pairs_evaluated"] == r0["counters"]["pairs_evaluated"] and r1["counters"]["active"] == r0["counters"]["active"]
    assert_parity(st, "f64", oracle, r_cut=st["r_cut"] + extra)


@pytest.mark.parametrize("kind,cells,slices", [("cubes", 6, 0), ("octahedra", 6, 0), ("mixed", 5, 0), ("mixed", 4, 5)])
def test_search_kernel_with_and_without_culling(pkg, oracle, kind, cells, slices):
    """Exact per-feature culling (default) must not change which terms contribute: same counters as the kernel that
    sweeps every Eq. 1 term, same sums up to rounding; it must sweep fewer terms, and without it all of them."""
    st = di.dense_state(kind, cells)
    a = assert_parity(st, "f32", oracle, cull=False, slices=slices)
    b = assert_parity(st, "f32", oracle, cull=True, slices=slices)
    for key in ("active", "degenerate", "parallel", "pairs_evaluated", "terms"):
        assert a["counters"][key] == b["counters"][key], key
    assert a["counters"]["terms_swept"] == a["counters"]["terms"]
    assert 0 < b["counters"]["terms_swept"] < a["counters"]["terms_swept"]
    assert b["counters"]["terms_swept"] >= b["counters"]["active"]


@pytest.mark.parametrize("n", [7, 9, 24])
def test_faces_with_many_edges(pkg, oracle, n):
    """Prisms over a heptagon / nonagon: faces whose boundary-edge count has no unrolled sweep (run-time edge loop),
    mixed with quadrilaterals in one shape, against cubes.  The 24-gon prism's table (48 vertices, 72 edges, two
    24-edge faces) is a large one: the culling kernel takes its one-sweep-site variant with the two-level face sweep."""
    shapes = [di.prism(n, 0.5, 0.9, 0.06), di.cube(0.8, 0.06)]
    st = di.lattice_state(3, shapes, (5, 5, 5), 1.145, seed=4, jitter=0.01, orient="small", max_angle=0.1,
                          shape_fractions=(0.6, 0.4))
    for precision in ("f32", "f64"):
        r = assert_parity(st, precision, oracle)
        assert r["counters"]["active"] > 30


def test_exactly_aligned_cube_lattice_closed_form(pkg):
    """Aligned unit cubes at spacing 1 + sigma: every face-neighbour pair has 56 terms at r = sigma (PAPER.md:61 as
    corrected by Eq. 1), so U_i = 1/2 * 6 * 56 eps = 168 eps, F_i = tau_i = 0.  Of the 32 edge-edge terms of a pair, the
    4 facing-edge/facing-edge ones overlap and go through the parallel-midpoint rule; the 4 collinear
    side-edge pairs are parallel without overlap and fall through to the general routine (R5)."""
    sig = 0.3
    st = di.lattice_state(3, [di.cube(1.0, sig / 2)], (4, 4, 4), 1.0 + sig, orient="aligned")
    for precision in ("f32", "f64"):
        f, tq, w, cnt = gpu_compute(round_state(st, precision), precision)
        tol = 1e-4 if precision == "f32" else 1e-9
        assert np.allclose(f[:, 3], 168.0, rtol=tol)
        assert np.abs(f[:, :3]).max() < tol * 56 * 24 / sig and np.abs(tq[:, :3]).max() < tol * 56 * 24 / sig
        assert cnt["active"] == 64 * 3 * 56 and cnt["parallel"] == 64 * 3 * 4
        # sum_i tr W_i = N * 3 pairs * 56 * (24 eps / sigma) * (1 + sigma)
        assert math.isclose(w[:, [0, 3, 5]].sum(), 64 * 3 * 56 * 24 / sig * (1 + sig), rel_tol=tol)


def test_parallel_rule_just_inside_and_outside(pkg, oracle):
    """Two rods, slightly non-parallel: the angle is set just inside / outside eps_par (R5)."""
    rod = di.rod(1.0, 0.15)
    for ang in (0.5e-3, 0.9e-3, 1.1e-3, 2e-3):  # threshold: sin^2 < 1e-6  <=>  angle < 1e-3
        st = di.two_particle_state(rod, rod, seed=0)
        st["pos"][:, :3] = [[0, 0, 0], [0.31, 0.02, 0.1]]
        st["quat"][0] = [1, 0, 0, 0]
        st["quat"][1] = [math.cos(ang / 2), 0, math.sin(ang / 2), 0]
        r = assert_parity(st, "f64", oracle)
        assert r["counters"]["active"] == 1 and r["counters"]["parallel"] == (1 if ang < 1e-3 else 0)
        assert_parity(st, "f32", oracle)


PAIRS = [("square", "square"), ("pentagon", "square"), ("disk", "square"), ("cube", "cube"), ("octa", "octa"),
         ("tet", "ti"), ("ti", "ti"), ("ico", "cube"), ("sphere", "sphere"), ("sphere", "cube"), ("rod", "rod"),
         ("rod", "cube"), ("plate", "plate"), ("plate", "tet")]
SHAPES = dict(square=lambda: di.square(), pentagon=lambda: di.regular_polygon(5, 0.5, 0.05), disk=lambda: di.disk(0.2),
              cube=lambda: di.cube(), octa=lambda: di.octahedron(), tet=lambda: di.tetrahedron(),
              ti=lambda: di.truncated_icosahedron(), ico=lambda: di.icosahedron(), sphere=lambda: di.sphere(0.3),
              rod=lambda: di.rod(1.0, 0.2), plate=lambda: di.triangular_plate())


@pytest.mark.parametrize("na,nb", PAIRS)
def test_isolated_pair_poses(pkg, oracle, na, nb):
    """P3: many isolated two-particle poses, rejection-sampled (with the oracle) to be in contact, batched into ONE
    state on a sparse lattice of pairs so that every species pair -- including the degenerate shapes (sphere, rod,
    plate, disk) and both orderings of unlike shapes -- goes through the kernel."""
    sa, sb = SHAPES[na](), SHAPES[nb]()
    dim = sa["dim"]
    shapes = [sa, sb]
    sig = sa["rounding"] + sb["rounding"]
    reach = di.default_rcut(shapes)
    rng = np.random.default_rng(11)
    poses = []
    tries = 0
    want = 24 if "ti" in (na, nb) else 64
    while len(poses) < want and tries < 20000:
        tries += 1
        d = rng.standard_normal(3)
        if dim == 2:
            d[2] = 0
        d *= rng.uniform(0.3, 1.0) * reach / np.linalg.norm(d)
        if dim == 2:
            qi, qj = di.planar_quaternions(rng.uniform(0, 2 * math.pi, 2))
        else:
            qi, qj = di.random_quaternions(rng, 2)
        _, sums = oracle.pair_terms(shapes, 0, 1, qi, qj, d)
        if 0.8 * sig < sums["rmin"] < 2 ** (1 / 6) * sig:
            poses.append((d, qi, qj))
    assert len(poses) >= want // 2
    m = len(poses)
    side = int(math.ceil(m ** (1.0 / dim)))
    spacing = 3.0 * reach
    n = 2 * m
    pos, quat, sid = np.zeros((n, 4)), np.zeros((n, 4)), np.zeros(n, dtype=np.int32)
    for k, (d, qi, qj) in enumerate(poses):
        cell = np.array([k % side, (k // side) % side, k // (side * side) if dim == 3 else 0], dtype=np.float64)
        c = (cell - side / 2 + 0.5) * spacing
        a, b = (2 * k, 2 * k + 1) if k % 2 == 0 else (2 * k + 1, 2 * k)  # both index orders
        pos[a, :3], pos[b, :3] = c - d / 2, c + d / 2
        quat[a], quat[b] = qi, qj
        sid[a], sid[b] = 0, 1
    box = np.array([side * spacing] * 3)
    st = dict(dim=dim, shapes=shapes, box=box, pos=pos, quat=quat, vel=np.zeros((n, 4)), angmom=np.zeros((n, 4)),
              shape_id=sid, N=n, r_cut=reach, epsilon=1.0)
    for precision in ("f64", "f32"):
        r = assert_parity(st, precision, oracle)
        assert r["counters"]["active"] >= m


# ---------------------------------------------------------------------------------------------------------------
# full-size configs (the launch configuration bench.py times): sampled rows against the oracle + global invariants
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [3, 4, 5])
def test_full_size_configs_every_row(pkg, oracle, k):
    """Configs 3, 4, 5 at full size, as specified (t = 0): EVERY row of force / torque / energy / virial against the
    oracle, and the system-wide term counters.  The oracle rows come from its cell-grid variant, which is the
    all-pairs sum bit for bit (pinned on small states; re-checked here at full size on 4,096 random rows plus up to
    1,024 interacting ones, which go through the O(N) all-pairs definition).  Tolerance denominators are the oracle's."""
    st = round_state(di.make_config(k), "f32")
    f, tq, w, cnt = gpu_compute(st, "f32")
    of, ot, ow, ocnt = oracle.compute(st, cells=True)
    live = np.nonzero(np.abs(of[:, :3]).sum(1) > 0)[0]
    assert len(live) >= 500, len(live)                     # the compared rows really carry forces
    rng = np.random.default_rng(k)
    sub = np.union1d(rng.choice(st["N"], 4096, replace=False), rng.choice(live, min(len(live), 1024), replace=False))
    sub = sub.astype(np.int32)
    df, dt_, dw, _ = oracle.compute(st, subset=sub)        # the definition: all-pairs scan
    assert np.array_equal(df, of[sub]) and np.array_equal(dt_, ot[sub]) and np.array_equal(dw, ow[sub])
    fs, ts, us = scales(st, of, ot)
    assert np.abs(f[:, :3] - of[:, :3]).max() / fs < TOL["f32"]
    assert np.abs(tq[:, :3] - ot[:, :3]).max() / ts < TOL["f32"]
    assert np.abs(f[:, 3] - of[:, 3]).max() / us < TOL["f32"]
    assert np.abs(w - ow).max() / max(np.abs(ow).max(), 1.0) < TOL["f32"]
    assert 2 * cnt["active"] == ocnt[2] and 2 * cnt["degenerate"] == ocnt[3] and 2 * cnt["parallel"] == ocnt[4]
    assert 2 * cnt["pairs_evaluated"] == ocnt[0] and 2 * cnt["terms"] == ocnt[1]
    # properties that hold at any size: Newton's third law over the whole system, pair/term counts of the lattice
    assert np.abs(f[:, :3].sum(0)).max() < 1e-3 * fs * math.sqrt(st["N"])
    assert cnt["pairs_listed"] == 3 * st["N"]  # 6 neighbours per particle on these lattices
    per_pair = {3: 50, 4: 240}.get(k)
    if per_pair:
        assert cnt["terms"] == cnt["pairs_listed"] * per_pair


def test_neighbors_full_size_rows(pkg, oracle):
    """Configs 3 and 5 at full size: 4,096 sampled rows of the neighbour list against the all-pairs definition."""
    for k in (3, 5):
        st = di.make_config(k)
        sub = np.random.default_rng(10 + k).choice(st["N"], 4096, replace=False).astype(np.int32)
        assert_neighbors_exact(st, "f32", oracle, subset=sub)


# ---------------------------------------------------------------------------------------------------------------
# edge cases and error behaviour
# ---------------------------------------------------------------------------------------------------------------
def test_single_particle_and_isolated_particles(pkg):
    st = di.lattice_state(3, [di.cube()], (1, 1, 1), 10.0)
    f, tq, w, cnt = gpu_compute(st, "f32")
    assert np.all(f == 0) and np.all(tq == 0) and np.all(w == 0) and cnt["pairs_listed"] == 0
    st = di.lattice_state(2, [di.square()], (3, 3), 5.0)
    f, tq, w, cnt = gpu_compute(st, "f64")
    assert np.all(f == 0) and cnt["pairs_listed"] == 0


def test_error_codes(pkg):
    import torch

    st = di.make_config(2, scale=2)
    dem, t = pkg.from_state(st, "f32")
    with pytest.raises(pkg.DemError) as e:
        dem.compute(t["pos"], t["quat"], t["shape_id"])
    assert e.value.code == -7  # DEM_ESTALE: no list yet
    with pytest.raises(pkg.DemError) as e:
        dem.build_neighbors(t["pos"], t["shape_id"], st["box"], 0.5 * st["r_cut"])
    assert e.value.code == -5  # DEM_ERCUT
    with pytest.raises(pkg.DemError) as e:
        dem.build_neighbors(t["pos"], t["shape_id"], [3.0, 3.0, 3.0], st["r_cut"])
    assert e.value.code == -4  # DEM_EBOX
    dem.build_neighbors(t["pos"], t["shape_id"], st["box"], st["r_cut"])
    with pytest.raises(pkg.DemError) as e:
        dem.compute(t["pos"][:10].contiguous(), t["quat"][:10].contiguous(), t["shape_id"][:10].contiguous())
    assert e.value.code == -7
    with pytest.raises(TypeError):
        dem.compute(t["pos"].cpu(), t["quat"], t["shape_id"])  # no CPU path
    # a shape id outside the registered shapes is caught on the device during the build, not used as an index
    bad = t["shape_id"].clone()
    bad[7] = 5
    with pytest.raises(pkg.DemError) as e:
        dem.build_neighbors(t["pos"], bad, st["box"], st["r_cut"])
    assert e.value.code == -1  # DEM_EINVAL
    bad[7] = -1
    with pytest.raises(pkg.DemError) as e:
        dem.build_neighbors(t["pos"], bad, st["box"], st["r_cut"])
    assert e.value.code == -1
    dem.build_neighbors(t["pos"], t["shape_id"], st["box"], st["r_cut"])
    # a list built with a larger cutoff (skin) gives identical forces: the extra pairs contribute exactly zero
    f0, t0, _ = dem.compute(t["pos"], t["quat"], t["shape_id"])
    dem.build_neighbors(t["pos"], t["shape_id"], st["box"], 1.4 * st["r_cut"])
    f1, t1, _ = dem.compute(t["pos"], t["quat"], t["shape_id"])
    assert torch.equal(f0, f1) and torch.equal(t0, t1)
    dem.close()


@pytest.mark.parametrize("kind,cells,kw", [("mixed", 5, dict(cull=True)), ("mixed", 5, dict(cull=False)),
                                           ("cubes", 6, dict(cull=True, slices=3)), ("pentagons", 12, dict(kernel=0)),
                                           ("octahedra", 6, dict(cull=True))])
def test_run_to_run_bit_reproducible(pkg, kind, cells, kw):
    """No atomics on the accumulation path, a sorted cell list, ballot-ranked queues: repeated runs give identical bits
    for force, torque, virial and counters.  The warp-synchronous shared-memory structures of the search kernels
    (candidate queue, item list, double-buffered pose stages) are the likeliest place for a data race, and a race there
    would show up as run-to-run differences; six runs on states with hundreds of queued candidates per warp."""
    st = di.dense_state(kind, cells)
    runs = [gpu_compute(st, "f32", **kw) for _ in range(6)]
    assert runs[0][3]["active"] > 50
    for r in runs[1:]:
        assert np.array_equal(runs[0][0], r[0]) and np.array_equal(runs[0][1], r[1]) and np.array_equal(runs[0][2], r[2])
        assert runs[0][3] == r[3]


def test_host_buffer_entry_point_matches_device_path(pkg):
    import torch

    st = round_state(di.dense_state("cubes", 5), "f32")
    f, tq, w, _ = gpu_compute(st, "f32")
    dem, _ = pkg.from_state(st, "f32")
    n = st["N"]
    pos = torch.tensor(st["pos"], dtype=torch.float32).pin_memory()
    quat = torch.tensor(st["quat"], dtype=torch.float32).pin_memory()
    sid = torch.tensor(st["shape_id"], dtype=torch.int32).pin_memory()
    fo, to, wo = (torch.empty((n, 4)).pin_memory(), torch.empty((n, 4)).pin_memory(), torch.empty((n, 6)).pin_memory())
    dem.compute_host(pos, quat, sid, st["box"], st["r_cut"], fo, to, wo)
    assert np.array_equal(fo.numpy().astype(np.float64), f) and np.array_equal(to.numpy().astype(np.float64), tq)
    assert np.array_equal(wo.numpy().astype(np.float64), w)
    dem.close()


@pytest.mark.parametrize("length", [5.0, 20.0, 100.0])
def test_long_thin_near_parallel_edges(pkg, oracle, length):
    """The packed FP32 search only has to FLAG every term the exact routine would accept; its line-line solve loses its
    digits on near-parallel edges and the candidate cutoff carries a slack for that (4e-3 x longest edge, DESIGN.md
    section 5).  Rods 50, 200 and 1000 sigma long (one edge each), in pairs at angles 1e-5 ... 1e-2 and gaps around
    sigma, overlapping fully, partly and end to end: the search kernel (culling on and off) must find exactly the active,
    degenerate and parallel-branch terms of the generic FP32 kernel, and both must match the oracle."""
    sig = 0.1
    shapes = [di.rod(length, sig / 2)]
    reach = di.default_rcut(shapes)
    rng = np.random.default_rng(int(length))
    angles = [0.0, 1e-5, 1e-4, 5e-4, 9e-4, 1.1e-3, 3e-3, 1e-2]
    m = 4 * len(angles)
    spacing = 3.0 * reach
    side = int(math.ceil(m ** (1.0 / 3.0)))
    n = 2 * m
    pos, quat = np.zeros((n, 4)), np.zeros((n, 4))
    for k in range(m):
        ang = angles[k % len(angles)]
        cell = np.array([k % side, (k // side) % side, k // (side * side)], dtype=np.float64)
        c = (cell - side / 2 + 0.5) * spacing
        gap = sig * rng.uniform(0.85, 1.1)
        shift = (0.0, 0.3, 0.9, 0.999)[k // len(angles)] * length      # overlap: full, most, a tenth, end to end
        g = rng.standard_normal(3)
        g[2] = 0.0
        g /= np.linalg.norm(g)                                          # gap direction, perpendicular to the rods (z)
        pos[2 * k, :3] = c
        pos[2 * k + 1, :3] = c + gap * g + [0, 0, shift]
        quat[2 * k] = [1, 0, 0, 0]
        quat[2 * k + 1] = [math.cos(ang / 2), *(math.sin(ang / 2) * g)]  # tilt ABOUT the gap direction: the lines stay `gap` apart
    st = dict(dim=3, shapes=shapes, box=np.array([side * spacing] * 3), pos=pos, quat=quat, vel=np.zeros((n, 4)),
              angmom=np.zeros((n, 4)), shape_id=np.zeros(n, dtype=np.int32), N=n, r_cut=reach, epsilon=1.0)
    # FP32 holds the end points of an edge of length L to ulp(L): r* is then good to ~2^-23 L / sigma relative and the
    # force to 13 times that (F ~ r^-13), whichever kernel runs: the north_star tolerance is meant for the paper's
    # shapes (edge / sigma <= 8.5); here it is widened to that bound.  The point of this test is the candidate SET.
    tol = max(TOL["f32"], 4 * 13 * 2.0 ** -23 * length / sig)
    ref = assert_parity(st, "f32", oracle, kernel=1, tol=tol, wlever=0.5 * length)
    assert ref["counters"]["active"] >= m // 2 and ref["counters"]["parallel"] > 0
    for cull in (False, True):
        r = assert_parity(st, "f32", oracle, kernel=0, cull=cull, tol=tol, wlever=0.5 * length)
        for key in ("active", "degenerate", "parallel", "pairs_evaluated"):
            assert r["counters"][key] == ref["counters"][key], (key, cull)
    assert_parity(st, "f64", oracle)
