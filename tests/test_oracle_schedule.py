"""Pins for O-19, temperature schedules of the thermostats ("temperature profiles oscillating between
300 K and 600 K"; reading R32)."""
import numpy as np

import workloads as wl


def _system():
    w = wl.ionic_liquid_box(n_pairs=4, hidden=(16, 16))  # 96 atoms at 300 K
    w.model.scale[:] = 0.004
    return w


def test_profile_is_piecewise_linear_and_clamped(orc):
    sch = ([10, 30, 50], [300.0, 600.0, 300.0])  # one period of the paper's oscillation
    assert orc.schedule_temperature(sch, 0, 1.0) == 300.0 and orc.schedule_temperature(sch, 10, 1.0) == 300.0
    assert orc.schedule_temperature(sch, 20, 1.0) == 450.0 and orc.schedule_temperature(sch, 30, 1.0) == 600.0
    assert orc.schedule_temperature(sch, 45, 1.0) == 375.0
    assert orc.schedule_temperature(sch, 50, 1.0) == 300.0 and orc.schedule_temperature(sch, 9999, 1.0) == 300.0
    assert orc.schedule_temperature(None, 7, 123.0) == 123.0


def test_constant_schedule_is_no_schedule(orc):
    w = _system()
    m = orc.Model(w.model)
    args = (m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 12)
    a = orc.nvt_langevin(*args, 450.0, 0.02, 3)
    b = orc.nvt_langevin(*args, 300.0, 0.02, 3, schedule=([0, 100], [450.0, 450.0]))
    assert all(np.array_equal(p, q) for p, q in zip(a, b))
    a = orc.nvt_nose_hoover(*args, 450.0, 25.0)
    b = orc.nvt_nose_hoover(*args, 450.0, 25.0, schedule=([5], [450.0]))
    assert all(np.array_equal(p, q) for p, q in zip(a, b))


def test_strong_friction_kinetic_energy_follows_the_profile(orc):
    """gamma dt >> 1: the O step of MD step n draws velocities at T(n), so E_kin[n + 1] / (3/2 N k T(n)) = 1 within
    sampling error at every step of a 300 -> 900 K ramp (288 degrees of freedom: 8 % per step; the mean over the
    ramp to 3 %), and the late steps are three times hotter than the early ones."""
    w = _system()
    m = orc.Model(w.model)
    sch = ([0, 40], [300.0, 900.0])
    x, v, ep, ek = orc.nvt_langevin(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 40, 300.0,
                                    100.0, 17, schedule=sch)
    target = np.array([1.5 * 96 * wl.KB_EV * orc.schedule_temperature(sch, n, 0.0) for n in range(40)])
    ratio = ek[1:] / target
    assert abs(ratio.mean() - 1.0) < 0.03 and np.abs(ratio - 1.0).max() < 0.35
    assert 2.2 < ek[-8:].mean() / ek[1:9].mean() < 3.4


def test_nose_hoover_follows_a_ramp(orc):
    """The chain drives the kinetic temperature after the profile: with a fast thermostat (tau = 10 fs) a box that
    starts at 300 K is hotter at the end of a ramp to 1500 K than under the constant 300 K thermostat."""
    w = _system()
    m = orc.Model(w.model)
    args = (m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 80)
    flat = orc.nvt_nose_hoover(*args, 300.0, 10.0)
    ramp = orc.nvt_nose_hoover(*args, 300.0, 10.0, schedule=([0, 40], [300.0, 1500.0]))
    assert ramp[3][-20:].mean() > 2.0 * flat[3][-20:].mean()
    assert np.array_equal(ramp[3][:1], flat[3][:1])
