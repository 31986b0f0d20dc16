"""Pins for O-15, Langevin dynamics in the BAOAB splitting with a counter-based generator."""
import numpy as np

import workloads as wl


def _system():
    w = wl.ionic_liquid_box(n_pairs=4, hidden=(16, 16))  # 96 atoms at 300 K
    w.model.scale[:] = 0.004
    return w


def test_generator_known_value_and_normal_statistics(orc):
    # the published first output of splitmix64 seeded with 0
    assert int(orc._splitmix64(0, np.array([0], np.uint64))[0]) == 0xE220A8397B1DCDAF
    xi = np.concatenate([orc.langevin_normals(12345, t, 4096) for t in range(30)])  # 368 640 normals
    assert abs(xi.mean()) < 6e-3 and abs(xi.var() - 1.0) < 8e-3
    assert abs((xi ** 4).mean() - 3.0) < 0.05  # kurtosis of a normal
    c = np.corrcoef(xi.T)
    assert np.abs(c - np.eye(3)).max() < 8e-3  # components independent
    assert abs(np.corrcoef(xi[:-1, 0], xi[1:, 0])[0, 1]) < 8e-3  # neighbouring atoms independent
    a, b = orc.langevin_normals(7, 3, 10), orc.langevin_normals(7, 4, 10)
    assert np.array_equal(a, orc.langevin_normals(7, 3, 10)) and not np.array_equal(a, b)


def test_zero_friction_is_nve(orc):
    w = _system()
    m = orc.Model(w.model)
    x, v, ep, ek = orc.nvt_langevin(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 15,
                                    300.0, 0.0, 1)
    ref = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.0, 0.5, 15)
    assert np.abs(x - ref.positions).max() < 1e-9 and np.abs(ek - ref.ekin).max() < 1e-9 * ref.ekin.max()


def test_strong_friction_draws_maxwell_boltzmann_velocities(orc):
    """gamma dt >> 1: every O step replaces v by sqrt(kT/m) xi, so E_kin = 3/2 N kT within sampling error
    (288 degrees of freedom: 8 % standard deviation per step; averaged over 20 steps) -- pins units and c2."""
    w = _system()
    m = orc.Model(w.model)
    for T in (300.0, 1200.0):
        x, v, ep, ek = orc.nvt_langevin(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 20,
                                        T, 100.0, 99)
        target = 1.5 * 96 * wl.KB_EV * T
        assert abs(ek[1:].mean() / target - 1.0) < 0.08, (T, ek[1:].mean() / target)


def test_moderate_friction_relaxes_towards_the_target(orc):
    w = _system()
    m = orc.Model(w.model)
    x, v, ep, ek = orc.nvt_langevin(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 60,
                                    900.0, 0.05, 5)
    t300, t900 = 1.5 * 96 * wl.KB_EV * 300, 1.5 * 96 * wl.KB_EV * 900
    assert ek[0] < 1.3 * t300 and ek[-10:].mean() > 0.5 * (t300 + t900)
