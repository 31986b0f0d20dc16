"""Pins for O-16: general (triclinic) lattices and the virial W = -sum_pairs d (x) g = -dE/d strain
("the gradient of the energy with respect to positions and the strain tensor
allow the prediction of forces and virials").  The pins are facts the oracle's loops do not supply themselves: the
numpy fp64 statement of the neighbour set, two descriptions of one lattice giving one energy, finite differences
of the energy under strain, the dimer's W = -d (x) F_1."""
import numpy as np

import workloads as wl


def _all_pairs_numpy(pos32, h32, r_list, kmax=3):
    """fp64 statement of O-1 on the fp32 inputs: every (i, j, n) with |x_j - x_i + n h| < r_list."""
    x = pos32.astype(np.float64)
    h = h32.astype(np.float64)
    out = []
    rng = range(-kmax, kmax + 1)
    for n1 in rng:
        for n2 in rng:
            for n3 in rng:
                shift = n1 * h[0] + n2 * h[1] + n3 * h[2]
                d = x[None, :, :] - x[:, None, :] + shift
                r2 = (d * d).sum(-1)
                i, j = np.nonzero(r2 < r_list * r_list)
                keep = ~((i == j) & (n1 == 0) & (n2 == 0) & (n3 == 0))
                out += [(a, b, n1, n2, n3) for a, b in zip(i[keep], j[keep])]
    return np.array(sorted(out), dtype=np.int32)


def test_triclinic_neighbours_are_the_definition_and_cells_equal_brute(orc):
    tiny = wl.triclinic_box(8, hidden=(16, 16))  # faces closer than r_list: second images are needed
    got = orc.neighbors(tiny.positions, tiny.lattice, tiny.pbc, 6.0, "brute").as_set_array()
    assert np.array_equal(got, _all_pairs_numpy(tiny.positions, tiny.lattice, 6.0, kmax=4))
    assert np.abs(got[:, 2:]).max() >= 2
    w = wl.triclinic_box(216, hidden=(16, 16))
    got = orc.neighbors(w.positions, w.lattice, w.pbc, 6.0, "brute").as_set_array()
    ref = _all_pairs_numpy(w.positions, w.lattice, 6.0)
    # (no pair of these boxes lies within fp32 rounding of r_list, where the fp32 predicate could differ from fp64)
    assert np.array_equal(got, ref)
    rev = got[:, [1, 0, 2, 3, 4]].copy()
    rev[:, 2:] *= -1
    assert np.array_equal(rev[np.lexsort(rev.T[::-1])], got)  # (i, j, n) <-> (j, i, -n)
    big = wl.triclinic_box(4096, hidden=(16, 16))  # >= 3 slabs of r_list per axis: the cell list applies
    a = orc.neighbors(big.positions, big.lattice, big.pbc, 6.0, "cells").as_set_array()
    b = orc.neighbors(big.positions, big.lattice, big.pbc, 6.0, "brute").as_set_array()
    assert np.array_equal(a, b)
    vol = abs(np.linalg.det(big.lattice.astype(np.float64)))
    expect = 4096 / vol * 4.0 / 3.0 * np.pi * 6.0 ** 3
    assert abs(len(a) / 4096 - expect) < 0.05 * expect


def test_two_descriptions_of_one_lattice_give_one_answer(orc):
    """A cubic box and the same lattice described by the rows a, a + b, c + a - b: same atoms (each folded into
    its description's cell), same E_i, same F, same virial."""
    w = wl.li3po4_box(216, hidden=(32, 32))
    m = orc.Model(w.model)
    L = float(w.cell[0])
    cubic = orc.energy_forces(m, w.positions, w.species, w.cell, orc.neighbors(w.positions, w.cell, w.pbc, 6.0))
    h = np.array([[L, 0, 0], [L, L, 0], [L, -L, L]], dtype=np.float32)
    x = orc.wrap_positions(w.positions.astype(np.float64), h, w.pbc)
    x32 = orc.to_fp32_inside(x, h)
    pairs = orc.neighbors(x32, h, w.pbc, 6.0)
    skew = orc.energy_forces(m, x32, w.species, h, pairs)
    assert len(pairs) == len(orc.neighbors(w.positions, w.cell, w.pbc, 6.0))
    # the folded fp32 positions differ from the cubic ones by lattice vectors up to fp32 rounding of the fold
    assert np.abs(skew.e_atom - cubic.e_atom).max() < 2e-5 * np.abs(cubic.e_atom).max()
    assert np.abs(skew.forces - cubic.forces).max() < 2e-4 * np.abs(cubic.forces).max()
    assert np.abs(skew.virial - cubic.virial).max() < 2e-4 * np.abs(cubic.virial).max()


def _strained_energy(orc, m, w, h, x, eps):
    F = np.eye(3) + eps
    h2 = h @ F.T
    x2 = x @ F.T
    pairs = orc.neighbors(x2, h2, w.pbc, 6.0)
    # fp64 positions and cell in the energy; the fp32 list is exact enough: E is C1 across the cutoff
    return orc.energy_forces(m, x2, w.species, h2, pairs, forces=False).energy


def test_virial_is_minus_the_strain_derivative_of_the_energy(orc):
    for w in (wl.triclinic_box(216, hidden=(32, 32)), wl.li3po4_box(216, hidden=(32, 32))):
        m = orc.Model(w.model)
        h = orc.cell9(w.box).reshape(3, 3)
        x = w.positions.astype(np.float64)
        res = orc.energy_forces(m, x, w.species, h, orc.neighbors(w.positions, w.box, w.pbc, 6.0))
        W = res.virial
        assert np.abs(W - W.T).max() < 1e-9 * np.abs(W).max()  # symmetric: E is rotation invariant
        step = 1e-6
        for a in range(3):
            for b in range(3):
                eps = np.zeros((3, 3))
                eps[a, b] = step
                fd = (_strained_energy(orc, m, w, h, x, eps) - _strained_energy(orc, m, w, h, x, -eps)) / (2 * step)
                # d'_a = d_a + eps_ab d_b  =>  dE/d eps_ab = sum g_a d_b = -W[b][a]
                assert abs(fd + W[b, a]) < 1e-6 * np.abs(W).max(), (a, b, fd, W[b, a])


def test_dimer_virial_is_minus_d_times_force(orc):
    w = wl.cluster(2, 2, hidden=(16, 16))
    pos = np.array([[20.0, 20.0, 20.0], [21.3, 22.1, 19.2]], dtype=np.float32)
    m = orc.Model(w.model)
    res = orc.energy_forces(m, pos, np.array([0, 1], np.int32), w.cell, orc.neighbors(pos, w.cell, (0, 0, 0), 5.0))
    d = (pos[1] - pos[0]).astype(np.float64)
    assert np.abs(res.forces[0]).max() > 1e-3
    assert np.allclose(res.virial, -np.outer(d, res.forces[0]), rtol=0, atol=1e-12 * np.abs(res.virial).max())


def test_virial_is_translation_invariant_and_nve_conserves_energy_in_a_triclinic_cell(orc):
    w = wl.triclinic_box(216, hidden=(32, 32))
    m = orc.Model(w.model)
    a = orc.energy_forces(m, w.positions, w.species, w.lattice, orc.neighbors(w.positions, w.lattice, w.pbc, 6.0))
    x = orc.wrap_positions(w.positions.astype(np.float64) + np.array([3.3, -1.7, 9.1]), w.lattice, w.pbc)
    x32 = orc.to_fp32_inside(x, w.lattice)
    b = orc.energy_forces(m, x32, w.species, w.lattice, orc.neighbors(x32, w.lattice, w.pbc, 6.0))
    assert abs(a.energy - b.energy) < 1e-5 * np.abs(a.e_atom).sum()
    assert np.abs(a.virial - b.virial).max() < 1e-4 * np.abs(a.virial).max()
    errs = []
    for dt in (0.5, 0.25):
        r = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.lattice, w.pbc, 0.4, dt, int(8 / dt))
        e = r.epot + r.ekin
        errs.append(np.abs(e - e[0]).max())
        assert np.isfinite(e).all()
    assert errs[1] < 0.4 * errs[0]  # second order in dt
