"""Pins for O-6..O-11: forces = central finite differences of the energy (the one test that pins
the gradient, SURVEY.md header lesson), sum F = 0, invariances, skin independence, ensemble
identities (Eq. 5, 6), NVE conservation / time reversal / dt^2 scaling."""
import numpy as np
import pytest

import workloads as wl


def _fd_check(orc, m, pos, species, cell, pairs, picks, h=1e-5, rtol=2e-7):
    res = orc.energy_forces(m, pos, species, cell, pairs)
    scale = np.sqrt((res.forces ** 2).mean())
    worst = 0.0
    for (i, a) in picks:
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h
        pm[i, a] -= h
        ep = orc.energy_forces(m, pp, species, cell, pairs, forces=False).energy
        em = orc.energy_forces(m, pm, species, cell, pairs, forces=False).energy
        fd = -(ep - em) / (2 * h)
        worst = max(worst, abs(fd - res.forces[i, a]) / scale)
    assert worst < rtol, worst
    return res


def test_forces_equal_finite_differences_config1_full_size(orc):
    """Config 1 as specified (MLP [512, 512]); box < 2 r_cut so duplicate-by-image pairs are
    exercised; 24 random (atom, axis)."""
    w = wl.tiny_box()
    m = orc.Model(w.model)
    pos = w.positions.astype(np.float64)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 5.0)
    rng = np.random.default_rng(0)
    picks = [(int(rng.integers(64)), int(rng.integers(3))) for _ in range(24)]
    res = _fd_check(orc, m, pos, w.species, w.cell, pairs, picks)
    assert np.abs(res.forces.sum(0)).max() < 1e-12 * 64 * np.abs(res.forces).max()


def test_forces_equal_finite_differences_five_species(orc):
    """Config-2-shaped (5 species, r_cut 6) at 8 ion pairs = 192 atoms; 20 random (atom, axis)."""
    w = wl.ionic_liquid_box(n_pairs=8, hidden=(64, 64))
    m = orc.Model(w.model)
    pos = w.positions.astype(np.float64)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.5)  # skin shell included in the list
    rng = np.random.default_rng(1)
    picks = [(int(rng.integers(192)), int(rng.integers(3))) for _ in range(20)]
    res = _fd_check(orc, m, pos, w.species, w.cell, pairs, picks)
    assert np.abs(res.forces.sum(0)).max() < 1e-12 * 192 * np.abs(res.forces).max()


def test_skin_does_not_change_energy_or_forces(orc):
    w = wl.li3po4_box(1024, hidden=(32, 32))
    m = orc.Model(w.model)
    a = orc.energy_forces(m, w.positions, w.species, w.cell, orc.neighbors(w.positions, w.cell, w.pbc, 6.0))
    b = orc.energy_forces(m, w.positions, w.species, w.cell, orc.neighbors(w.positions, w.cell, w.pbc, 7.0))
    assert abs(a.energy - b.energy) < 1e-10 * np.abs(a.e_atom).sum()
    assert np.allclose(a.forces, b.forces, rtol=0, atol=1e-11 * np.abs(a.forces).max())


def test_energy_is_c1_across_the_cutoff(orc):
    """Drag one atom of a trimer across r_cut: E and F continuous (f_c(r_cut) = f_c'(r_cut) = 0)."""
    spec = wl.make_model(21, 1, r_cut=5.0, hidden=(16, 16))
    m = orc.Model(spec)
    E, F = [], []
    for r in (5.0 - 1e-6, 5.0 + 1e-6):
        pos = np.array([[10.0, 10, 10], [8.0, 10.5, 10], [10.0 + r, 10, 10]])  # atoms 2-3 are > r_cut apart
        p = orc.neighbors(pos, [40, 40, 40], (0, 0, 0), 6.0)
        res = orc.energy_forces(m, pos, [0, 0, 0], [40, 40, 40], p)
        E.append(res.energy)
        F.append(res.forces)
    assert abs(E[0] - E[1]) < 1e-9
    assert np.abs(F[0] - F[1]).max() < 1e-4 * max(1.0, np.abs(F[0]).max())


def test_translation_wrap_permutation_and_cubic_symmetry(orc):
    w = wl.tiny_box(hidden=(32, 32))
    m = orc.Model(w.model)
    L = w.cell.astype(np.float64)
    pos = w.positions.astype(np.float64)

    def ef(x, sp):
        return orc.energy_forces(m, x, sp, w.cell, orc.neighbors(x, w.cell, w.pbc, 5.0))

    base = ef(pos, w.species)
    tol_e = 1e-6 * np.abs(base.e_atom).sum()  # positions are re-rounded to fp32 by neighbors() only
    # translation + wrap (fp64 positions; fp32 rounding enters the predicate only)
    t = np.array([1.234, -7.7, 3.21])
    x = pos + t
    x -= np.floor(x / L) * L
    tr = ef(x, w.species)
    assert abs(tr.energy - base.energy) < 1e-9 * np.abs(base.e_atom).sum()
    assert np.allclose(tr.forces, base.forces, atol=1e-9 * np.abs(base.forces).max())
    # permutation of the atom labels: E_i, F_i permute
    perm = np.random.default_rng(3).permutation(64)
    pr = ef(pos[perm], w.species[perm])
    assert np.allclose(pr.e_atom, base.e_atom[perm], rtol=1e-12)
    assert np.allclose(pr.forces, base.forces[perm], atol=1e-11 * np.abs(base.forces).max())
    # cubic point-group operation mapping the box to itself: (x, y, z) -> (L - y, x, z)  (proper rotation)
    x = np.stack([L[1] - pos[:, 1], pos[:, 0], pos[:, 2]], 1)
    x -= np.floor(x / L) * L
    rot = ef(x, w.species)
    assert abs(rot.energy - base.energy) < tol_e
    Frot = np.stack([-base.forces[:, 1], base.forces[:, 0], base.forces[:, 2]], 1)
    assert np.allclose(rot.forces, Frot, atol=1e-9 * np.abs(base.forces).max())
    # mirror (improper): invariants have even total rank, E unchanged (reading R6)
    x = pos.copy()
    x[:, 2] = L[2] - x[:, 2]
    x -= np.floor(x / L) * L
    mir = ef(x, w.species)
    assert abs(mir.energy - base.energy) < tol_e


def test_rotation_of_cluster_energy_and_force_covariance(orc):
    w = wl.cluster(20, 2, hidden=(32, 32))
    m = orc.Model(w.model)
    pos = w.positions.astype(np.float64)
    base = orc.energy_forces(m, pos, w.species, w.cell, orc.neighbors(pos, w.cell, w.pbc, 5.0))
    A = np.random.default_rng(8).normal(size=(3, 3))
    Qm, _ = np.linalg.qr(A)
    if np.linalg.det(Qm) < 0:
        Qm[:, 0] *= -1
    c = pos.mean(0)
    x = (pos - c) @ Qm.T + c
    rot = orc.energy_forces(m, x, w.species, w.cell, orc.neighbors(x, w.cell, w.pbc, 5.0))
    assert abs(rot.energy - base.energy) < 1e-10 * np.abs(base.e_atom).sum()
    assert np.allclose(rot.forces, base.forces @ Qm.T, atol=1e-9 * np.abs(base.forces).max())
    assert np.abs(base.forces).max() > 1e-3


# ---------------------------------------------------------------- ensemble (O-10)
def test_ensemble_identities(orc):
    w = wl.tiny_box(hidden=(32, 32), n_heads=8)
    m = orc.Model(w.model)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 5.0)
    ens = orc.ensemble(m, w.positions, w.species, w.cell, pairs, keep_heads=True)
    assert np.all(ens.e_var >= 0) and np.all(ens.f_var >= 0) and ens.f_var.max() > 0
    # numpy's population statistics (ddof = 0: Eq. 5 divides by N_ens, reading R13)
    assert np.allclose(ens.e_mean, ens.e_heads.mean(1), rtol=1e-13)
    assert np.allclose(ens.e_var, ens.e_heads.var(1), rtol=1e-10, atol=1e-14)
    assert np.allclose(ens.f_mean, ens.f_heads.mean(0), rtol=1e-12, atol=1e-14)
    assert np.allclose(ens.f_var, ens.f_heads.var(0), rtol=1e-9, atol=1e-14)
    # Eq. 6: mean of per-head forces == force of the mean energy == single head with averaged last layer
    mean_grad = orc.energy_forces(m, w.positions, w.species, w.cell, pairs)  # head_w = 1/M
    assert np.allclose(mean_grad.forces, ens.f_mean, atol=1e-11 * np.abs(ens.f_mean).max())
    spec1 = wl.tiny_box(hidden=(32, 32), n_heads=1).model
    spec1.W[:-1] = w.model.W[:-1]
    spec1.b[:-1] = w.model.b[:-1]
    spec1.W[-1] = w.model.W[-1].astype(np.float64).mean(1, keepdims=True)
    spec1.b[-1] = w.model.b[-1].astype(np.float64).mean(keepdims=True)
    spec1.beta, spec1.scale, spec1.shift = w.model.beta, w.model.scale, w.model.shift
    single = orc.energy_forces(orc.Model(spec1), w.positions, w.species, w.cell, pairs)
    assert np.allclose(single.forces, ens.f_mean, atol=1e-10 * np.abs(ens.f_mean).max())
    assert np.allclose(single.e_atom, ens.e_mean, rtol=1e-10)
    # per-head forces are FD-consistent: head 3
    hw = np.zeros(8)
    hw[3] = 1.0
    h3 = orc.energy_forces(m, w.positions, w.species, w.cell, pairs, head_w=hw)
    assert np.allclose(h3.forces, ens.f_heads[3], atol=1e-12 * np.abs(h3.forces).max())
    pos = w.positions.astype(np.float64)
    h = 1e-5
    for (i, a) in [(3, 0), (40, 2)]:
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h
        pm[i, a] -= h
        fd = -(orc.energy_forces(m, pp, w.species, w.cell, pairs, head_w=hw, forces=False).energy
               - orc.energy_forces(m, pm, w.species, w.cell, pairs, head_w=hw, forces=False).energy) / (2 * h)
        assert abs(fd - h3.forces[i, a]) < 1e-6 * np.abs(h3.forces).max()


def test_ensemble_equal_heads_has_zero_variance(orc):
    w = wl.tiny_box(hidden=(16, 16), n_heads=4)
    w.model.W[-1][:] = w.model.W[-1][:, :1]
    w.model.b[-1][:] = w.model.b[-1][:1]
    m = orc.Model(w.model)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 5.0)
    ens = orc.ensemble(m, w.positions, w.species, w.cell, pairs)
    assert np.abs(ens.e_var).max() < 1e-20 and np.abs(ens.f_var).max() < 1e-20


# ---------------------------------------------------------------- NVE (O-11)
def _small_md_system(hidden=(16, 16)):
    w = wl.ionic_liquid_box(n_pairs=4, hidden=hidden)  # 96 atoms, L = 10.0 Ang, 5 species
    w.model.scale[:] = 0.004  # random weights give a rough landscape: keep forces ~0.2 eV/Ang so dt = 0.5 fs is asymptotic
    return w


def test_nve_conserves_energy_and_momentum_and_scales_as_dt2(orc):
    w = _small_md_system()
    m = orc.Model(w.model)
    out = {}
    for dt, n in ((0.5, 40), (0.25, 80)):
        r = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.5, dt, n)
        etot = r.epot + r.ekin
        out[dt] = np.abs(etot - etot[0]).max()
        ms = w.masses.astype(np.float64)[:, None]
        p1 = (r.velocities * ms).sum(0)
        p0 = (w.velocities.astype(np.float64) * ms).sum(0)  # ~1e-8: COM removed before rounding to fp32
        assert np.abs(p1 - p0).max() < 1e-12
        assert np.ptp(r.ekin) > 1e-6  # something actually moves
    assert out[0.5] < 5e-3 * 96 * wl.KB_EV * 300
    ratio = out[0.5] / out[0.25]
    assert 3.5 < ratio < 4.6, ratio  # second-order integrator: 4 (measured 4.06)


def test_nve_time_reversal(orc):
    w = _small_md_system()
    m = orc.Model(w.model)
    big_skin = 2.0  # no rebuild inside the run, so summation order is fixed
    fwd = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, big_skin, 0.5, 25)
    assert fwd.n_rebuilds == 0
    back = orc.nve(m, fwd.positions, -fwd.velocities, w.masses, w.species, w.cell, w.pbc, big_skin, 0.5, 25)
    L = w.cell.astype(np.float64)
    d = back.positions - w.positions.astype(np.float64)
    d -= np.round(d / L) * L
    assert np.abs(d).max() < 1e-9
    assert np.allclose(-back.velocities, w.velocities.astype(np.float64), atol=1e-11)


def test_nve_skin_and_rebuilds_do_not_change_the_trajectory(orc):
    w = _small_md_system()
    m = orc.Model(w.model)
    a = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.0, 0.5, 30)
    b = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, 0.05, 0.5, 30)
    assert a.n_rebuilds == 30 and 0 < b.n_rebuilds < 30
    assert np.allclose(a.epot, b.epot, rtol=0, atol=1e-9 * np.abs(a.epot).max())
    assert np.abs(a.positions - b.positions).max() < 1e-9


def test_nve_first_step_by_hand(orc):
    """One velocity-Verlet step recomputed from the oracle's own E/F calls with numpy."""
    w = _small_md_system()
    m = orc.Model(w.model)
    x = w.positions.astype(np.float64)
    v = w.velocities.astype(np.float64)
    ms = w.masses.astype(np.float64)[:, None]
    L = w.cell.astype(np.float64)
    dt = 0.5
    f0 = orc.energy_forces(m, x, w.species, w.cell, orc.neighbors(x, w.cell, w.pbc, 6.0)).forces
    vh = v + 0.5 * dt * f0 / ms * wl.ACC_CONV
    x1 = x + dt * vh
    x1 -= np.floor(x1 / L) * L
    r1 = orc.energy_forces(m, x1, w.species, w.cell, orc.neighbors(x1, w.cell, w.pbc, 6.0))
    v1 = vh + 0.5 * dt * r1.forces / ms * wl.ACC_CONV
    r = orc.nve(m, x, v, w.masses, w.species, w.cell, w.pbc, 0.0, dt, 1)
    assert np.abs(r.positions - x1).max() < 1e-12
    assert np.abs(r.velocities - v1).max() < 1e-13
    assert abs(r.epot[1] - r1.energy) < 1e-10 * abs(r1.energy)
    ek = 0.5 * (ms * v1 ** 2).sum() / wl.ACC_CONV
    assert abs(r.ekin[1] - ek) < 1e-12 * ek
    # 3/2 N kT at 300 K within sampling noise (COM removed)
    assert abs(r.ekin[0] / (1.5 * 96 * wl.KB_EV * 300) - 1) < 0.25
