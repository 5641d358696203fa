"""Pins of the oracle's Nose-Hoover NVT integrator (oracle/dem_oracle.c: orc_step_nvt; R19).
None of them re-types the splitting: they use the NVE oracle (itself pinned), the thermostat's differential equations
integrated by an independent RK4, the conserved quantity, and time reversal."""
import numpy as np

import dem_inputs as di


def _dense():
    return di.dense_state("cubes", 4, spacing=1.38)


def test_infinite_thermostat_mass_is_nve(oracle):
    st = _dense()
    a = oracle.step(st, 1e-3, 20)
    b = oracle.step_nvt(st, 1e-3, 20, kT=2.0, tau=1e30)
    for k in ("pos", "quat", "vel", "angmom", "force", "torque"):
        assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(a["energies"], b["energies"][:, :3])


def test_degrees_of_freedom(oracle):
    n = 64
    assert oracle.step_nvt(_dense(), 1e-3, 0, 1.0, 1.0)["dof"] == 3 * (n - 1) + 3 * n
    assert oracle.step_nvt(di.dense_state("squares", 8), 1e-3, 0, 1.0, 1.0)["dof"] == 2 * (n - 1) + n
    rods = di.lattice_state(3, [di.rod(1.0, 0.1)], (4, 4, 4), 3.0, seed=3)
    rods["shapes"][0]["inertia"][2] = 0.0     # no rotation about the rod axis
    assert oracle.step_nvt(rods, 1e-3, 0, 1.0, 1.0)["dof"] == 3 * (n - 1) + 2 * n


def _conserved(r, kT, tau):
    g = r["dof"]
    q = g * kT * tau * tau
    e = r["energies"]
    return e[:, 0] + e[:, 1] + e[:, 2] + 0.5 * q * e[:, 3] ** 2 + g * kT * e[:, 4]


def test_conserved_quantity_second_order(oracle):
    """U + K + Q xi^2/2 + g kT eta is conserved by the equations of motion; the symmetric splitting keeps it to O(dt^2).
    The target temperature differs from the initial one, so heat really flows through the thermostat."""
    st = _dense()
    kT, tau, t_end = 0.6, 0.1, 0.2
    err = []
    for dt in (5e-4, 2.5e-4):
        r = oracle.step_nvt(st, dt, int(round(t_end / dt)), kT, tau)
        h = _conserved(r, kT, tau)
        err.append(np.abs(h - h[0]).max() / st["N"])
        k = r["energies"][:, 1] + r["energies"][:, 2]
        assert abs(k[-1] - k[0]) / k[0] > 0.2          # the thermostat did work on the system
        assert np.abs((r["energies"][:, :3].sum(1)) - r["energies"][0, :3].sum()).max() / st["N"] > 100 * err[-1]
    assert err[0] < 1e-2 and 3.0 < err[0] / err[1] < 5.0, err


def test_time_reversal(oracle):
    st = _dense()
    kT, tau, dt, n = 0.6, 0.1, 5e-4, 100
    a = oracle.step_nvt(st, dt, n, kT, tau)
    back = dict(st)
    back.update(pos=a["pos"], quat=a["quat"], vel=-a["vel"], angmom=-a["angmom"])
    b = oracle.step_nvt(back, dt, n, kT, tau, thermo=(-a["thermo"][0], a["thermo"][1]))
    assert np.abs(b["pos"] - st["pos"]).max() < 1e-10
    assert np.abs(b["vel"] + st["vel"]).max() < 1e-9
    assert np.abs(b["angmom"] + st["angmom"]).max() < 1e-9
    assert abs(b["thermo"][0]) < 1e-10 and abs(b["thermo"][1]) < 1e-10
    assert abs(a["thermo"][0]) > 1e-2


def test_ideal_gas_follows_the_thermostat_equations(oracle):
    """Without interactions K obeys dK/dt = -2 xi K, dxi/dt = (2K - g kT)/Q exactly (both K_trans and K_rot scale with
    s^2, torque-free rotation conserves K_rot): compare K(t), xi(t), eta(t) with an RK4 integration of these equations."""
    st = di.lattice_state(3, [di.cube(1.0, 0.15)], (4, 4, 4), 4.0, seed=5)    # out of reach of one another
    kT, tau, dt, n = 0.5, 0.3, 2e-3, 400
    r = oracle.step_nvt(st, dt, n, kT, tau)
    assert np.all(r["energies"][:, 0] == 0.0)
    g = r["dof"]
    q = g * kT * tau * tau

    def rhs(y):
        return np.array([-2.0 * y[1] * y[0], (2.0 * y[0] - g * kT) / q, y[1]])

    y = np.array([r["energies"][0, 1] + r["energies"][0, 2], 0.0, 0.0])
    sub, h = 20, dt / 20
    ref = [y.copy()]
    for _ in range(n):
        for _ in range(sub):
            k1 = rhs(y); k2 = rhs(y + 0.5 * h * k1); k3 = rhs(y + 0.5 * h * k2); k4 = rhs(y + h * k3)
            y = y + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
        ref.append(y.copy())
    ref = np.array(ref)
    k = r["energies"][:, 1] + r["energies"][:, 2]
    assert np.abs(k - ref[:, 0]).max() / ref[:, 0].max() < 1e-4
    assert np.abs(r["energies"][:, 3] - ref[:, 1]).max() / np.abs(ref[:, 1]).max() < 1e-4
    assert np.abs(r["energies"][:, 4] - ref[:, 2]).max() / np.abs(ref[:, 2]).max() < 1e-4
    assert ref[:, 0].min() < 0.75 * ref[0, 0]              # K really relaxed towards g kT / 2
