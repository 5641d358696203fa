"""Pins for the oracle's NPT step (orc_step_npt: Nose-Hoover thermostat + isotropic Martyna-Tobias-Klein barostat driven
by the virial, R22).  CPU only."""
import math

import numpy as np

import dem_inputs as di


def _dense(kind="cubes"):
    if kind == "cubes":
        return di.dense_state("cubes", 4, spacing=1.38)        # the state of the NVT pins
    return di.dense_state("squares", 6, seed=5, spacing=1.36)


def _conserved(r, st, kT, tau, p, tau_p):
    e = r["energies"]
    g, n, d = r["dof"], st["N"], st["dim"]
    return (e[:, 0] + e[:, 1] + e[:, 2] + p * e[:, 6] + 0.5 * d * n * kT * tau_p ** 2 * e[:, 5] ** 2
            + 0.5 * g * kT * tau ** 2 * e[:, 3] ** 2 + g * kT * e[:, 4])


def test_infinite_barostat_mass_is_nvt_bit_for_bit(oracle):
    st = _dense()
    a = oracle.step_nvt(st, 5e-4, 40, 0.8, 0.2)
    b = oracle.step_npt(st, 5e-4, 40, 0.8, 0.2, 3.0, math.inf)
    for k in ("pos", "quat", "vel", "angmom", "force", "torque"):
        assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(a["thermo"], b["baro"][:2]) and b["baro"][2] == 0.0
    assert np.array_equal(b["box"], st["box"])
    assert np.array_equal(a["energies"][:, :5], b["energies"][:, :5])


def test_conserved_quantity_second_order(oracle):
    """U + K + P V + W_b nu^2/2 + Q xi^2/2 + g kT eta is conserved by the equations of motion (it ties the sign and size
    of the virial term, of P V and of the alpha-coupling together): the integrator's fluctuation of it is O(dt^2)."""
    for kind in ("cubes", "squares"):
        st = _dense(kind)
        kT, tau, p, tau_p = 1.0, 0.1, 6.0, 0.25
        fl = []
        for dt in (4e-4, 2e-4):
            r = oracle.step_npt(st, dt, int(round(0.04 / dt)), kT, tau, p, tau_p)
            h = _conserved(r, st, kT, tau, p, tau_p)
            fl.append(np.abs(h - h[0]).max())
            e = r["energies"]
            assert abs(e[-1, 6] / e[0, 6] - 1.0) > 2e-3          # the box really moved
            assert np.abs(e[:, 0] + e[:, 1] + e[:, 2] - e[0, :3].sum()).max() > 30 * fl[-1]   # E alone is not conserved
            assert e[:, 7].max() > 1.0                           # interacting: the virial is at work
        assert 2.8 < fl[0] / fl[1] < 5.5, (kind, fl)


def test_time_reversal(oracle):
    st = _dense()
    kT, tau, p, tau_p, dt, n = 0.9, 0.15, 4.0, 0.3, 2e-4, 80
    a = oracle.step_npt(st, dt, n, kT, tau, p, tau_p)
    back = dict(st)
    back.update(pos=a["pos"], quat=a["quat"], vel=-a["vel"], angmom=-a["angmom"], box=a["box"])
    b = oracle.step_npt(back, dt, n, kT, tau, p, tau_p, baro=(-a["baro"][0], a["baro"][1], -a["baro"][2]))
    assert np.abs(b["box"] - st["box"]).max() < 1e-11
    assert np.abs(b["pos"] - st["pos"]).max() < 1e-10
    assert np.abs(b["vel"] + st["vel"]).max() < 1e-9 and np.abs(b["angmom"] + st["angmom"]).max() < 1e-9
    assert abs(b["baro"][0]) < 1e-10 and abs(b["baro"][1]) < 1e-10 and abs(b["baro"][2]) < 1e-10
    assert abs(a["baro"][2]) > 1e-3 and abs(a["box"][0] / st["box"][0] - 1) > 1e-4


def test_ideal_gas_follows_the_npt_equations(oracle):
    """Without interactions the equations close on (K_trans, K_rot, V, nu, xi, eta):
    dK_t/dt = -2 (alpha nu + xi) K_t, dK_r/dt = -2 xi K_r, dV/dt = d nu V, dnu/dt = (alpha 2 K_t - d V P) / W_b,
    dxi/dt = (2K - g kT)/Q, deta/dt = xi.  RK4 on these against the oracle's step; the stationary point is the ideal-gas
    law P V = (N - 1) kT alpha ... -> P V = N kT (alpha (N-1) = N)."""
    st = di.lattice_state(3, [di.cube(1.0, 0.15)], (4, 4, 4), 6.0, seed=5)    # far out of reach of one another
    n_p, d = st["N"], 3
    kT, tau, tau_p, dt, n = 0.7, 0.4, 0.5, 2e-3, 500
    v0 = np.prod(st["box"])
    p = 1.3 * n_p * kT / v0                                       # the gas is too dilute for this pressure: it shrinks
    r = oracle.step_npt(st, dt, n, kT, tau, p, tau_p)
    assert np.all(r["energies"][:, 0] == 0.0) and np.all(r["energies"][:, 7] == 0.0)
    g = r["dof"]
    q, wb = g * kT * tau * tau, d * n_p * kT * tau_p ** 2
    alpha = 1.0 + d / (d * (n_p - 1.0))

    def rhs(y):
        kt, kr, v, nu, xi, _ = y
        return np.array([-2.0 * (alpha * nu + xi) * kt, -2.0 * xi * kr, d * nu * v, (alpha * 2.0 * kt - d * v * p) / wb,
                         (2.0 * (kt + kr) - g * kT) / q, xi])

    y = np.array([r["energies"][0, 1], r["energies"][0, 2], v0, 0.0, 0.0, 0.0])
    sub, h = 20, dt / 20
    ref = [y.copy()]
    for _ in range(n):
        for _ in range(sub):
            k1 = rhs(y); k2 = rhs(y + 0.5 * h * k1); k3 = rhs(y + 0.5 * h * k2); k4 = rhs(y + h * k3)
            y = y + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
        ref.append(y.copy())
    ref = np.array(ref)
    e = r["energies"]
    for col, k in ((1, 0), (2, 1), (6, 2), (5, 3), (3, 4), (4, 5)):
        assert np.abs(e[:, col] - ref[:, k]).max() / np.abs(ref[:, k]).max() < 2e-4, (col, k)
    assert ref[:, 2].min() < 0.9 * v0                            # the volume really responded
    assert np.allclose(np.prod(r["box"]), e[-1, 6], rtol=1e-12)
    assert np.allclose(r["box"] / st["box"], (e[-1, 6] / v0) ** (1.0 / 3.0), rtol=1e-12)   # isotropic


def test_positions_scale_with_the_box(oracle):
    """Particles at rest with no thermostat and no forces: dx/dt = nu x means positions follow the box exactly,
    x(t)/L(t) constant, whatever nu does."""
    st = di.lattice_state(2, [di.square(1.0, 0.15)], (4, 4), 6.0, seed=2, jitter=0.3)
    st["vel"][:] = 0.0
    st["angmom"][:] = 0.0
    r = oracle.step_npt(st, 1e-3, 200, 1.0, math.inf, 0.05, 0.5, baro=(0.0, 0.0, -0.3))
    assert r["box"][0] < 0.97 * st["box"][0]
    assert np.allclose(r["pos"][:, :2] / r["box"][:2], st["pos"][:, :2] / st["box"][:2], atol=1e-13)
    assert np.all(r["vel"] == 0.0)
