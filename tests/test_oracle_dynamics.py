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


def _euler_rk4(q, lb, inertia, t_end, h=1e-4):
    """Independent reference for torque-free rigid-body rotation: RK4 on Euler's equations in the body frame,
    dL_b/dt = L_b x omega_b (omega_b = L_b / I componentwise), dq/dt = 1/2 q (x) (0, omega_b)."""
    def rhs(y):
        q, lb = y[:4], y[4:]
        w = lb / inertia
        dq = 0.5 * np.array([-q[1] * w[0] - q[2] * w[1] - q[3] * w[2],
                             q[0] * w[0] + q[2] * w[2] - q[3] * w[1],
                             q[0] * w[1] - q[1] * w[2] + q[3] * w[0],
                             q[0] * w[2] + q[1] * w[1] - q[2] * w[0]])
        return np.concatenate([dq, np.cross(lb, w)])

    y = np.concatenate([q, lb])
    for _ in range(int(round(t_end / h))):
        k1 = rhs(y); k2 = rhs(y + 0.5 * h * k1); k3 = rhs(y + 0.5 * h * k2); k4 = rhs(y + h * k3)
        y = y + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
    return y[:4] / np.linalg.norm(y[:4]), y[4:]


def test_free_asymmetric_top_follows_eulers_equations(oracle):
    """Pins the non-spherical branch of free_rotate (direction of every sub-rotation included): the orientation after
    t = 1 agrees with an RK4 integration of Euler's equations to O(dt^2) (error ratio ~4 on halving dt).  A rotor
    running backwards, a transposed composition or a wrong axis order gives an O(1) error."""
    shape = di.box_shape(1.0, 0.7, 0.4, 0.05)
    st = _free_state(shape)
    inertia = shape["inertia"]
    assert len(set(np.round(inertia, 12))) == 3            # three different moments: the splitting branch is used
    refs = []
    for i in range(st["N"]):
        lb0 = rotmat(st["quat"][i]).T @ st["angmom"][i, :3]
        refs.append(_euler_rk4(st["quat"][i], lb0, inertia, 1.0))
    errs = []
    for dt in (0.02, 0.01):
        out = oracle.step(st, dt=dt, nsteps=int(round(1.0 / dt)))
        e = 0.0
        for i in range(st["N"]):
            rref = rotmat(refs[i][0])
            e = max(e, np.abs(rotmat(out["quat"][i]) - rref).max())
            # the body-frame angular momentum follows too (lab L is fixed: L_b = R^T L)
            assert np.allclose(rotmat(out["quat"][i]).T @ st["angmom"][i, :3], refs[i][1], atol=50 * dt * dt)
        errs.append(e)
    assert errs[1] < 2e-3 and 3.0 < errs[0] / errs[1] < 5.0, errs
    # the bodies really turned (several radians), so a sign error could not hide
    turn = [np.arccos(np.clip(0.5 * (np.trace(rotmat(refs[i][0]).T @ rotmat(st["quat"][i])) - 1.0), -1, 1)) for i in range(st["N"])]
    assert min(turn) > 0.3


def test_nearly_spherical_top_matches_the_exact_spherical_rotation(oracle):
    """I -> (I0, I0, I0 (1 + 1e-9)) sends the splitting branch to the spherical-top limit, whose exact solution is the
    Rodrigues rotation about L by |L| t / I0 (written out independently below)."""
    shape = di.cube(1.0, 0.15)
    i0 = shape["inertia"][0]
    shape["inertia"] = np.array([i0, i0, i0 * (1.0 + 1e-9)])
    st = _free_state(shape)
    errs = []
    for dt in (0.02, 0.01):
        out = oracle.step(st, dt=dt, nsteps=int(round(1.0 / dt)))
        e = 0.0
        for i in range(st["N"]):
            w = st["angmom"][i, :3] / i0
            ang = np.linalg.norm(w)
            ax = w / ang
            K = np.array([[0, -ax[2], ax[1]], [ax[2], 0, -ax[0]], [-ax[1], ax[0], 0]])
            R = np.eye(3) + math.sin(ang) * K + (1 - math.cos(ang)) * K @ K
            e = max(e, np.abs(rotmat(out["quat"][i]) - R @ rotmat(st["quat"][i])).max())
        errs.append(e)
    assert errs[1] < 2e-3 and 3.0 < errs[0] / errs[1] < 5.0, errs
