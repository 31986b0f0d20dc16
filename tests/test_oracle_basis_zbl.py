"""Pins for O-17 (Bessel-like radial basis of Kocer et al.) and O-18 (ZBL repulsion):
properties the published definitions fix -- unit norm and orthogonality structure under r^2 dr, zero at the
cutoff, the r -> 0 limits, derivative = finite difference, forces = finite differences of the energy, the bare
Coulomb limit of the screened potential, the screening function's weights summing to one, no double counting."""
import dataclasses

import numpy as np

import workloads as wl


def _bessel_model(orc, n_basis=7, r_cut=6.0):
    spec = wl.make_model(5, 2, r_cut=r_cut, n_basis=n_basis, hidden=(8, 8))
    return orc.Model(dataclasses.replace(spec, basis_kind=1))


def test_bessel_basis_norm_zeros_limits(orc):
    m = _bessel_model(orc)
    rc = 6.0
    r = np.linspace(1e-4, rc, 24001)
    vals = np.array([orc.basis(m, float(x))[0] for x in r])  # [r][n]
    # unit norm under r^2 dr (fixes the prefactor), computed by Simpson's rule
    w = np.ones_like(r)
    w[1:-1:2], w[2:-1:2] = 4.0, 2.0
    w *= (r[1] - r[0]) / 3.0
    gram = (vals * (w * r * r)[:, None]).T @ vals
    assert np.allclose(np.diag(gram), 1.0, atol=2e-6)
    # "non-orthogonal": neighbours n, n+1 share one sinc and overlap; n, n+2 share none and are orthogonal
    for n in range(6):
        assert abs(gram[n, n + 1]) > 0.2
    for n in range(5):
        assert abs(gram[n, n + 2]) < 1e-5
    # zero at the cutoff, alternating sign and finite value at the origin: f_n(0) = 2 c_n
    assert np.abs(orc.basis(m, rc)[0]).max() < 1e-12
    f0 = orc.basis(m, 1e-7)[0]
    assert np.all(np.sign(f0) == np.array([1, -1, 1, -1, 1, -1, 1]))
    c0 = np.sqrt(2.0) * np.pi / rc ** 1.5 * 2.0 / np.sqrt(5.0)
    assert abs(f0[0] - 2.0 * c0) < 1e-9
    # derivative of the basis = central difference
    for x in (0.7, 2.3, 5.1):
        phi, dphi = orc.basis(m, x)
        fd = (orc.basis(m, x + 1e-6)[0] - orc.basis(m, x - 1e-6)[0]) / 2e-6
        assert np.allclose(dphi, fd, rtol=0, atol=1e-8)


def test_bessel_radial_derivative_and_forces(orc):
    w = wl.li3po4_box(216, hidden=(32, 32))
    spec = dataclasses.replace(w.model, basis_kind=1)
    m = orc.Model(spec)
    for x in (1.1, 3.3, 5.9):
        R, dR = orc.radial(m, 0, 2, x)
        Rp, _ = orc.radial(m, 0, 2, x + 1e-6)
        Rm, _ = orc.radial(m, 0, 2, x - 1e-6)
        assert np.allclose(dR, (Rp - Rm) / 2e-6, rtol=0, atol=1e-7 * max(1.0, np.abs(dR).max()))
    assert np.abs(orc.radial(m, 0, 2, 6.0)[0]).max() == 0.0
    gauss = orc.radial(orc.Model(w.model), 0, 2, 3.3)[0]
    assert not np.allclose(gauss, orc.radial(m, 0, 2, 3.3)[0], rtol=1e-2)
    pos = w.positions.astype(np.float64)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.0)
    res = orc.energy_forces(m, pos, w.species, w.cell, pairs)
    scale = np.sqrt((res.forces ** 2).mean())
    rng = np.random.default_rng(11)
    for _ in range(10):
        i, a = int(rng.integers(216)), int(rng.integers(3))
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += 1e-5
        pm[i, a] -= 1e-5
        fd = -(orc.energy_forces(m, pp, w.species, w.cell, pairs, forces=False).energy
               - orc.energy_forces(m, pm, w.species, w.cell, pairs, forces=False).energy) / 2e-5
        assert abs(fd - res.forces[i, a]) < 2e-7 * scale


def _zbl_spec(spec, r_max=2.5, scale=1.0, zn=(3.0, 15.0, 8.0)):
    return dataclasses.replace(spec, zbl=True, zbl_r_max=r_max, zbl_scale=scale,
                               atomic_numbers=np.asarray(zn[:spec.n_species], np.float32))


def test_zbl_limits_and_derivative(orc):
    spec = _zbl_spec(wl.li3po4_box(64, hidden=(8, 8)).model, r_max=2.0)
    m = orc.Model(spec)
    # bare Coulomb limit: 2 (V/2) r -> k_e Z1 Z2 as r -> 0 (screening function and cutoff -> 1: its weights sum to 1)
    e, _ = orc.zbl_half(m, 3.0, 8.0, 1e-7)
    assert abs(2.0 * e * 1e-7 / (14.399645 * 24.0) - 1.0) < 2e-4  # the published weights sum to 1.00007
    # symmetric in the two charges, zero at and beyond r_max, continuous derivative there
    assert orc.zbl_half(m, 3.0, 8.0, 0.9) == orc.zbl_half(m, 8.0, 3.0, 0.9)
    assert orc.zbl_half(m, 3.0, 8.0, 2.0) == (0.0, 0.0)
    assert abs(orc.zbl_half(m, 3.0, 8.0, 2.0 - 1e-7)[1]) < 1e-5
    # screened below Coulomb everywhere, monotonically decreasing
    r = np.linspace(0.3, 1.9, 40)
    v = np.array([orc.zbl_half(m, 15.0, 8.0, float(x))[0] for x in r])
    assert np.all(np.diff(v) < 0) and np.all(2 * v < 14.399645 * 120.0 / r)
    for x in (0.5, 1.2, 1.8):
        e, de = orc.zbl_half(m, 15.0, 8.0, x)
        fd = (orc.zbl_half(m, 15.0, 8.0, x + 1e-6)[0] - orc.zbl_half(m, 15.0, 8.0, x - 1e-6)[0]) / 2e-6
        assert abs(de - fd) < 1e-7 * max(1.0, abs(de))
    # the scale multiplies it
    m2 = orc.Model(dataclasses.replace(spec, zbl_scale=0.25))
    assert abs(orc.zbl_half(m2, 3.0, 8.0, 0.9)[0] - 0.25 * orc.zbl_half(m, 3.0, 8.0, 0.9)[0]) < 1e-15


def test_zbl_in_the_energy_no_double_counting_and_forces(orc):
    """Dimer: E(with ZBL) - E(without) = V(r) once (two directed pairs carry V/2 each); beyond r_max nothing
    changes; forces = finite differences with the term on; a compressed box where it matters."""
    c = wl.cluster(2, 2, hidden=(16, 16))
    pos = np.array([[20.0, 20.0, 20.0], [20.6, 20.9, 19.5]], dtype=np.float32)
    sp = np.array([0, 1], np.int32)
    pairs = orc.neighbors(pos, c.cell, (0, 0, 0), 5.0)
    plain = orc.energy_forces(orc.Model(c.model), pos, sp, c.cell, pairs)
    spec = _zbl_spec(c.model, r_max=2.5, zn=(6.0, 8.0))
    withz = orc.energy_forces(orc.Model(spec), pos, sp, c.cell, pairs)
    r = float(np.linalg.norm((pos[1] - pos[0]).astype(np.float64)))
    v_half, dv_half = orc.zbl_half(orc.Model(spec), 6.0, 8.0, r)
    assert v_half > 1.0
    assert abs((withz.energy - plain.energy) - 2.0 * v_half) < 1e-12 * abs(withz.energy)
    assert np.allclose(withz.e_atom - plain.e_atom, v_half, rtol=0, atol=1e-12)
    u = (pos[1] - pos[0]).astype(np.float64) / r
    assert np.allclose(withz.forces[0] - plain.forces[0], 2.0 * dv_half * u, rtol=0, atol=1e-10)  # F_0 = +dV/dr u: pushed apart
    far = np.array([[20.0, 20.0, 20.0], [22.0, 22.0, 21.0]], dtype=np.float32)  # r = 3 > r_max
    pf = orc.neighbors(far, c.cell, (0, 0, 0), 5.0)
    assert orc.energy_forces(orc.Model(spec), far, sp, c.cell, pf).energy == orc.energy_forces(orc.Model(c.model), far, sp, c.cell, pf).energy

    w = wl.li3po4_box(216, hidden=(32, 32))
    spec = _zbl_spec(w.model, r_max=3.0)
    m = orc.Model(spec)
    pos = w.positions.astype(np.float64)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.0)
    res = orc.energy_forces(m, pos, w.species, w.cell, pairs)
    base = orc.energy_forces(orc.Model(w.model), pos, w.species, w.cell, pairs)
    assert np.abs(res.forces - base.forces).max() > 1e-2  # the term is active in this box
    scale = np.sqrt((res.forces ** 2).mean())
    rng = np.random.default_rng(12)
    for _ in range(10):
        i, a = int(rng.integers(216)), int(rng.integers(3))
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += 1e-5
        pm[i, a] -= 1e-5
        fd = -(orc.energy_forces(m, pp, w.species, w.cell, pairs, forces=False).energy
               - orc.energy_forces(m, pm, w.species, w.cell, pairs, forces=False).energy) / 2e-5
        assert abs(fd - res.forces[i, a]) < 2e-7 * scale
    assert np.abs(res.forces.sum(0)).max() < 1e-11 * 216 * np.abs(res.forces).max()
    assert np.abs(res.virial - res.virial.T).max() < 1e-9 * np.abs(res.virial).max()
    # ensemble: every head carries the term once, so it drops out of the variances
    wh = wl.li3po4_box(64, hidden=(16, 16), n_heads=4)
    ph = orc.neighbors(wh.positions, wh.cell, wh.pbc, 6.0)
    e0 = orc.ensemble(orc.Model(wh.model), wh.positions, wh.species, wh.cell, ph)
    e1 = orc.ensemble(orc.Model(_zbl_spec(wh.model, r_max=3.0)), wh.positions, wh.species, wh.cell, ph)
    assert np.allclose(e0.e_var, e1.e_var, rtol=1e-9, atol=1e-14) and np.allclose(e0.f_var, e1.f_var, rtol=1e-9, atol=1e-14)
    assert np.abs(e1.f_mean - e0.f_mean).max() > 1e-3
