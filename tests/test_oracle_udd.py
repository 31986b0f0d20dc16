"""Pins for O-13, the UDD bias (Eq. 9): the force is the finite difference of the biased
energy, the limits of Eq. 9, and energy conservation of the biased dynamics."""
import numpy as np

import workloads as wl


def _system(n_heads=4):
    w = wl.ionic_liquid_box(n_pairs=4, hidden=(16, 16), n_heads=n_heads)  # 96 atoms
    w.model.scale[:] = 0.004
    return w


def test_biased_forces_are_finite_differences_of_the_biased_energy(orc):
    w = _system(4)
    m = orc.Model(w.model)
    pos = w.positions.astype(np.float64)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.0)
    base = orc.udd_energy_forces(m, pos, w.species, w.cell, pairs, 0.0, 1.0)
    # pick B so that the exponent is O(1): the bias gradient then matters
    B = np.sqrt(base.var_e / (4 * 96))
    A = 2.0
    r = orc.udd_energy_forces(m, pos, w.species, w.cell, pairs, A, B)
    assert abs(r.e_bias - A * (np.exp(-1.0) - 1.0)) < 1e-9
    assert np.abs(r.forces - base.forces).max() > 1e-3 * np.abs(base.forces).max()  # the bias does push
    scale = np.sqrt((r.forces ** 2).mean())
    h = 1e-5
    for (i, a) in [(0, 0), (17, 1), (40, 2), (95, 0), (63, 1)]:
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h
        pm[i, a] -= h
        fd = -(orc.udd_energy_forces(m, pp, w.species, w.cell, pairs, A, B).energy
               - orc.udd_energy_forces(m, pm, w.species, w.cell, pairs, A, B).energy) / (2 * h)
        assert abs(fd - r.forces[i, a]) < 1e-6 * scale, (i, a, fd, r.forces[i, a])
    assert np.abs(r.forces.sum(0)).max() < 1e-10 * scale * 96  # translation invariance survives the bias


def test_limits_of_eq9(orc):
    w = _system(4)
    m = orc.Model(w.model)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.0)
    args = (m, w.positions, w.species, w.cell, pairs)
    plain = orc.energy_forces(m, w.positions, w.species, w.cell, pairs)  # gradient of the mean energy
    off = orc.udd_energy_forces(*args, 0.0, 1.0)
    assert off.e_bias == 0.0 and abs(off.energy - plain.energy) < 1e-10 * abs(plain.energy)
    assert np.abs(off.forces - plain.forces).max() < 1e-10 * np.abs(plain.forces).max()
    wide = orc.udd_energy_forces(*args, 3.0, 1e9)  # B -> inf: no bias
    assert abs(wide.e_bias) < 1e-9 and np.abs(wide.forces - plain.forces).max() < 1e-9
    narrow = orc.udd_energy_forces(*args, 3.0, 1e-6)  # B -> 0: the bias saturates at -A and is flat
    assert abs(narrow.e_bias + 3.0) < 1e-12 and np.abs(narrow.forces - plain.forces).max() < 1e-12
    mid = orc.udd_energy_forces(*args, 3.0, np.sqrt(off.var_e / (4 * 96)))
    assert -3.0 < mid.e_bias < 0.0
    # identical heads: sigma = 0, so no bias whatever A and B
    w.model.W[-1][:] = w.model.W[-1][:, :1]
    w.model.b[-1][:] = w.model.b[-1][:1]
    same = orc.udd_energy_forces(orc.Model(w.model), w.positions, w.species, w.cell, pairs, 3.0, 1e-3)
    assert abs(same.e_bias) < 1e-12 and same.var_e < 1e-20


def test_biased_nve_conserves_the_biased_energy_and_differs_from_the_plain_run(orc):
    w = _system(4)
    m = orc.Model(w.model)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.0)
    var0 = orc.udd_energy_forces(m, w.positions, w.species, w.cell, pairs, 0.0, 1.0).var_e
    B = np.sqrt(var0 / (4 * 96))
    x, v, ep, ek, eb = orc.nve_udd(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 20, 0.5, B)
    etot = ep + ek
    assert np.abs(etot - etot[0]).max() < 5e-3 * 96 * wl.KB_EV * 300
    assert np.ptp(eb) > 1e-6
    # A = 0 is O-12 / O-11 on the mean energy
    x0, v0, ep0, ek0, eb0 = orc.nve_udd(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 20, 0.0, B)
    ref = orc.md_switching(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, 0.5, 20, 1000)
    assert np.abs(x0 - ref.positions).max() < 1e-9 and np.abs(ep0 - ref.epot).max() < 1e-9 * np.abs(ref.epot).max()
    assert np.abs(x - x0).max() > 1e-6
