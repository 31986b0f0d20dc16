"""Pins for O-12, switching-mode shallow-ensemble MD (PAPER.md:175 Eq. 6, :71 stopping criterion, Eq. 5):
things the method fixes independently of the oracle's own loop."""
import numpy as np

import workloads as wl


def _system(n_heads=4, hidden=(16, 16)):
    w = wl.ionic_liquid_box(n_pairs=4, hidden=hidden, n_heads=n_heads)  # 96 atoms, 5 species
    w.model.scale[:] = 0.004  # as the NVE pins: forces ~0.2 eV/Ang under random weights
    return w


def _run(orc, w, n_steps, rate, stop=0.0, skin=0.5):
    return orc.md_switching(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc,
                            skin, 0.5, n_steps, rate, stop)


def test_identical_heads_reduce_to_single_head_nve_with_zero_uncertainty(orc):
    """All heads equal: the mean energy IS the head's energy, so the trajectory is O-11's and sigma = 0."""
    w = _system(4)
    w.model.W[-1][:] = w.model.W[-1][:, :1]
    w.model.b[-1][:] = w.model.b[-1][:1]
    r = _run(orc, w, 12, 4)
    w1 = _system(1)
    w1.model.W[-1][:] = w.model.W[-1][:, :1]
    w1.model.b[-1][:] = w.model.b[-1][:1]
    for a, b in zip(w.model.W[:-1] + w.model.b[:-1], w1.model.W[:-1] + w1.model.b[:-1]):
        assert np.array_equal(a, b)  # same seed stream for the shared layers
    ref = orc.nve(orc.Model(w1.model), w1.positions, w1.velocities, w1.masses, w1.species, w1.cell, w1.pbc,
                  0.5, 0.5, 12)
    assert np.abs(r.positions - ref.positions).max() < 1e-11
    assert np.abs(r.epot - ref.epot).max() < 1e-11 * np.abs(ref.epot).max()
    assert np.abs(r.ekin - ref.ekin).max() < 1e-11 * np.abs(ref.ekin).max()
    assert len(r.sigma_e) == 3 and np.abs(r.sigma_e).max() < 1e-9 and np.abs(r.sigma_f_max).max() < 1e-9


def test_sampling_does_not_perturb_the_trajectory_and_samples_land_on_schedule(orc):
    """Eq. 6: both modes differentiate the same energy, so the trajectory cannot depend on sampling_rate,
    and the sample taken after step k * rate must equal Eq. 5 evaluated at that run's coordinates."""
    w = _system(4)
    a = _run(orc, w, 12, 3)
    b = _run(orc, w, 12, 6)
    c = _run(orc, w, 12, 100)  # never samples
    assert len(a.sigma_e) == 4 and len(b.sigma_e) == 2 and len(c.sigma_e) == 0
    assert np.array_equal(a.positions, b.positions) and np.array_equal(a.positions, c.positions)
    assert np.array_equal(a.epot, c.epot)
    assert np.array_equal(a.sigma_e[1::2], b.sigma_e) and np.array_equal(a.sigma_f_max[1::2], b.sigma_f_max)
    # the sample after step 6 from numpy, on a fresh brute-force list of a run stopped there
    m = orc.Model(w.model)
    six = _run(orc, w, 6, 100)
    pairs = orc.neighbors(six.positions, w.cell, w.pbc, 6.0)
    ens = orc.ensemble(m, six.positions, w.species, w.cell, pairs, keep_heads=True)
    tot = ens.e_heads.sum(0)
    assert abs(np.std(tot) - b.sigma_e[0]) < 1e-9 * max(np.std(tot), 1e-12)  # np.std: population divisor (R13)
    sf = np.sqrt(np.var(ens.f_heads, axis=0).sum(1)).max()
    assert abs(sf - b.sigma_f_max[0]) < 1e-9 * sf
    assert b.sigma_e[0] > 1e-6 and sf > 1e-6  # distinct heads: a real uncertainty


def test_mean_energy_md_conserves_the_mean_energy(orc):
    w = _system(8)
    r = _run(orc, w, 40, 10)
    etot = r.epot + r.ekin
    assert np.abs(etot - etot[0]).max() < 5e-3 * 96 * wl.KB_EV * 300
    assert np.ptp(r.ekin) > 1e-6


def test_stopping_criterion(orc):
    """the run ends at the first sample whose force uncertainty exceeds the threshold."""
    w = _system(4)
    full = _run(orc, w, 12, 3)
    assert full.n_steps_done == 12 and len(full.sigma_f_max) == 4
    k = int(np.argmax(full.sigma_f_max > full.sigma_f_max.min()))  # first sample above the smallest one
    thr = 0.5 * (full.sigma_f_max.min() + full.sigma_f_max[k]) if k > 0 else 0.5 * full.sigma_f_max[0]
    first_over = int(np.argmax(full.sigma_f_max > thr))
    r = _run(orc, w, 12, 3, stop=thr)
    assert r.n_steps_done == 3 * (first_over + 1) and len(r.sigma_f_max) == first_over + 1
    assert np.array_equal(r.sigma_f_max, full.sigma_f_max[:first_over + 1])
    assert np.array_equal(r.epot, full.epot[:r.n_steps_done + 1])
    huge = _run(orc, w, 12, 3, stop=1e9)
    assert huge.n_steps_done == 12 and np.array_equal(huge.sigma_e, full.sigma_e)
