"""Pins for O-14, NVT with a Nose-Hoover chain: the extended-system energy is conserved,
tau -> inf is NVE, the chain drives the kinetic energy towards 3/2 N kT, a frozen-force closed form."""
import numpy as np

import workloads as wl


def _system():
    w = wl.ionic_liquid_box(n_pairs=4, hidden=(16, 16))  # 96 atoms at 300 K
    w.model.scale[:] = 0.004
    return w


def _run(orc, w, n, T, tau, dt=0.5, **kw):
    return orc.nvt_nose_hoover(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc,
                               dt, n, T, tau, **kw)


def test_extended_energy_is_conserved_and_second_order(orc):
    w = _system()
    drift = {}
    for dt, n in ((0.5, 40), (0.25, 80)):
        x, v, ep, ek, cons = _run(orc, w, n, 300.0, 25.0, dt=dt)
        drift[dt] = np.abs(cons - cons[0]).max()
        assert np.abs((ep + ek) - (ep + ek)[0]).max() > 20 * drift[dt]  # the thermostat does exchange energy
    assert drift[0.5] < 5e-3 * 96 * wl.KB_EV * 300
    assert 3.4 < drift[0.5] / drift[0.25] < 4.6  # second order in dt (measured 3.93)


def test_weak_coupling_limit_is_nve(orc):
    w = _system()
    x, v, ep, ek, cons = _run(orc, w, 15, 300.0, 1e9)
    ref = orc.nve(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.0, 0.5, 15)
    assert np.abs(x - ref.positions).max() < 1e-9 and np.abs(ep - ref.epot).max() < 1e-9 * np.abs(ref.epot).max()


def test_thermostat_heats_towards_the_target(orc):
    w = _system()
    target = 1.5 * 96 * wl.KB_EV * 900.0
    x, v, ep, ek, cons = _run(orc, w, 60, 900.0, 10.0)
    x0, v0, ep0, ek0, _ = _run(orc, w, 60, 300.0, 1e9)
    assert ek[0] < 0.45 * target
    assert ek[-20:].mean() > ek0[-20:].mean() + 0.25 * target  # well above the NVE run, on the way to 900 K


def test_single_thermostat_half_step_closed_form(orc):
    """chain_length 1, one sub-step: p += d4 G; s = exp(-d2 p/Q); p += d4 G' with G' from the scaled KE."""
    dof, kT, dt = 30.0, 0.02, 0.5
    Q = np.array([dof * kT * 25.0 ** 2])
    xi, pxi = np.zeros(1), np.array([0.3])
    ke2 = 1.7
    s = orc.nhc_half_step(ke2, xi, pxi, Q, dof, kT, dt, 1, 1)
    p1 = 0.3 + dt / 4 * (ke2 - dof * kT)
    s_ref = np.exp(-dt / 2 * p1 / Q[0])
    p2 = p1 + dt / 4 * (ke2 * s_ref ** 2 - dof * kT)
    assert abs(s - s_ref) < 1e-15 and abs(pxi[0] - p2) < 1e-15 and abs(xi[0] - dt / 2 * p1 / Q[0]) < 1e-18
    # time reversal of the chain operator: flipping p and stepping again restores the state (symmetric splitting)
    xi2, pxi2 = xi.copy(), -pxi.copy()
    s2 = orc.nhc_half_step(ke2 * s * s, xi2, pxi2, Q, dof, kT, dt, 1, 1)
    assert abs(s * s2 - 1.0) < 1e-14 and abs(-pxi2[0] - 0.3) < 1e-14
