"""Pins for the oracle's neighbour predicate and NVE integrator (CPU only)."""
import math

import numpy as np
import pytest

import dem_inputs as di
from _util import rotmat


def test_neighbor_rows_vs_explicit_periodic_images(oracle):
    """O1 against a search over the 3^dim explicit periodic images (no rint shortcut)."""
    rng = np.random.default_rng(9)
    for dim in (2, 3):
        n = 150
        box = np.array([5.0, 4.0, 3.5])
        pos = np.zeros((n, 4))
        pos[:, :dim] = rng.uniform(-0.5, 0.5, (n, dim)) * box[:dim]
        st = dict(dim=dim, box=box, pos=pos, r_cut=1.2)
        counts, lst = oracle.neighbors(st)
        shifts = [np.array(s) for s in np.ndindex(*(3,) * dim)]
        for i in range(n):
            want = set()
            for j in range(n):
                if j == i:
                    continue
                best = min(np.sum((pos[j, :dim] - pos[i, :dim] + (s - 1) * box[:dim]) ** 2) for s in shifts)
                assert abs(best - 1.2 ** 2) > 1e-9  # no pair sits on the cutoff: the comparison is unambiguous
                if best < 1.2 ** 2:
                    want.add(j)
            got = list(lst[i, :counts[i]])
            assert got == sorted(got) and set(got) == want


def test_neighbor_subset_and_symmetry(oracle):
    st = di.make_config(2, scale=2)
    counts, lst = oracle.neighbors(st)
    assert counts.min() == 6 and counts.max() == 6  # SC lattice, spacing 2.03 < r_cut 2.07 < sqrt(2) * 2.03
    pairs = {(i, int(j)) for i in range(st["N"]) for j in lst[i, :counts[i]]}
    assert all((j, i) in pairs for i, j in pairs)
    sub = np.array([5, 17, 40], dtype=np.int32)
    c2, l2 = oracle.neighbors(st, subset=sub)
    assert np.array_equal(c2, counts[sub]) and np.array_equal(l2[:, :6], lst[sub, :6])


def _free_state(shape, n=6, seed=3):
    st = di.lattice_state(shape["dim"], [shape], (n, 1, 1)[: shape["dim"]] if shape["dim"] == 3 else (n, 1), 50.0,
                          seed=seed, kT=1.0)
    return st


def test_free_spherical_top_is_exact(oracle):
    """Torque-free spherical top: L and |q| conserved, orientation = exp(t L / I0) exactly (any dt)."""
    st = _free_state(di.cube(1.0, 0.15))
    out = oracle.step(st, dt=0.05, nsteps=40)
    assert np.array_equal(out["angmom"], st["angmom"]) and np.array_equal(out["vel"], st["vel"])
    assert np.allclose(np.linalg.norm(out["quat"], axis=1), 1.0, atol=1e-14)
    i0 = st["shapes"][0]["inertia"][0]
    for i in range(st["N"]):
        w = st["angmom"][i, :3] / i0
        ang = np.linalg.norm(w) * 2.0
        ax = w / np.linalg.norm(w)
        # Rodrigues rotation matrix written out independently
        K = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
        R = np.eye(3) + math.sin(ang) * K + (1 - math.cos(ang)) * K @ K
        assert np.allclose(rotmat(out["quat"][i]), R @ rotmat(st["quat"][i]), atol=1e-12)
    assert np.allclose(out["pos"][:, :3], st["pos"][:, :3] + 2.0 * st["vel"][:, :3], atol=1e-12)
    e = out["energies"]
    assert np.allclose(e[:, 1:], e[0, 1:], rtol=1e-13)


def test_free_asymmetric_top_conserves_energy_to_second_order(oracle):
    st = _free_state(di.box_shape(1.0, 0.7, 0.4, 0.05))
    errs = []
    for dt in (0.02, 0.01):
        out = oracle.step(st, dt=dt, nsteps=int(round(1.0 / dt)))
        e = out["energies"][:, 2]
        errs.append(np.abs(e - e[0]).max())
        assert np.array_equal(out["angmom"], st["angmom"])  # lab-frame L is exactly conserved by the free flow
        assert np.allclose(np.linalg.norm(out["quat"], axis=1), 1.0, atol=1e-14)
    assert errs[0] > 0 and 3.0 < errs[0] / errs[1] < 5.0  # second order


def test_2d_free_rotation(oracle):
    st = _free_state(di.square(1.0, 0.15))
    out = oracle.step(st, dt=0.01, nsteps=100)
    izz = st["shapes"][0]["inertia"][2]
    th0 = 2 * np.arctan2(st["quat"][:, 3], st["quat"][:, 0])
    th1 = 2 * np.arctan2(out["quat"][:, 3], out["quat"][:, 0])
    d = th1 - th0 - st["angmom"][:, 2] / izz * 1.0
    assert np.allclose(np.cos(d), 1.0, atol=1e-12) and np.allclose(np.sin(d), 0.0, atol=1e-10)
    assert np.all(out["quat"][:, 1:3] == 0)


def _hot_dense(kind):
    if kind == "squares":
        return di.dense_state("squares", 4, seed=5)
    return di.dense_state("cubes", 4, seed=5)


@pytest.mark.parametrize("kind", ["squares", "cubes"])
def test_energy_fluctuation_scales_as_dt_squared(oracle, kind):
    """second-order integrator, error ~ dt^2."""
    st = _hot_dense(kind)
    span = 0.02
    fl = []
    for dt in (4e-4, 2e-4):
        out = oracle.step(st, dt=dt, nsteps=int(round(span / dt)))
        e = out["energies"].sum(1)
        assert out["energies"][:, 0].max() > 1.0  # really interacting
        fl.append(np.abs(e - e[0]).max())
    assert 2.8 < fl[0] / fl[1] < 5.5, fl


def test_time_reversal(oracle):
    st = _hot_dense("squares")
    fwd = oracle.step(st, dt=2e-4, nsteps=60)
    back = dict(st)
    back.update(pos=fwd["pos"], quat=fwd["quat"], vel=-fwd["vel"], angmom=-fwd["angmom"])
    rev = oracle.step(back, dt=2e-4, nsteps=60)
    assert np.allclose(rev["pos"], st["pos"], atol=1e-10)
    assert np.allclose(np.abs(np.sum(rev["quat"] * st["quat"], axis=1)), 1.0, atol=1e-10)
    assert np.allclose(-rev["vel"], st["vel"], atol=1e-9)
