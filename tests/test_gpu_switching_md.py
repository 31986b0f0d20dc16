"""GPU parity for switching-mode shallow-ensemble MD (Eq. 5, 6)
against oracle O-12, through the C ABI (gmnn_md_ensemble_steps)."""
import numpy as np
import pytest

import workloads as wl
from parity_utils import F_TOL, force_error

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (they must not pass on a fallback)")
    import paper_2505_22168_b200 as pkg

    return pkg


def _system(gm, w, **kw):
    import torch

    sysm = gm.System(gm.Model(w.model, **kw), w.species)
    pos = torch.from_numpy(w.positions).cuda()
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    return sysm, pos, torch.from_numpy(w.velocities).cuda(), torch.from_numpy(w.masses).cuda()


def _workload(name):
    if name == "ionic384_m8":  # config-2-shaped, image path (2 cells per axis), 8 heads
        w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64), n_heads=8)
    else:  # config-4-shaped: Li3PO4 box, 32 heads, cell path
        w = wl.li3po4_box(1024, hidden=(64, 64), n_heads=32, skin=0.5)
    return w


@pytest.mark.parametrize("mlp_precision", [0, 3])
@pytest.mark.parametrize("name", ["ionic384_m8", "li1024_m32"])
def test_switching_md_matches_oracle(gm, orc, name, mlp_precision):
    """Trajectory on the mean energy, the samples' sigma_E and worst-atom sigma_F, and the last f_var."""
    w = _workload(name)
    sysm, pos, vel, mass = _system(gm, w, mlp_precision=mlp_precision)
    n_steps, rate = 12, 4
    out = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, n_steps, rate, want_f_var=True)
    ref = orc.md_switching(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc,
                           w.skin, w.dt_fs, n_steps, rate)
    assert out["n_steps_done"] == ref.n_steps_done == n_steps
    assert len(out["sigma_e"]) == len(ref.sigma_e) == 3
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - ref.positions
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - ref.velocities).max() <= 1e-5
    ep, ek = out["epot"].cpu().numpy(), out["ekin"].cpu().numpy()
    assert np.abs(ep - ref.epot).max() <= 1e-5 * np.abs(ref.epot).max() + 1e-4
    assert np.abs(ek - ref.ekin).max() <= 1e-4 * np.abs(ref.ekin).max()
    # sigma_E: spread of head totals, each a sum of atomic energies within 1e-5 relative (north_star tolerance)
    err_e = np.abs(out["sigma_e"] - ref.sigma_e).max()
    assert err_e <= 2e-4 * ref.sigma_e.max(), (err_e, ref.sigma_e)
    assert np.abs(out["sigma_f_max"] - ref.sigma_f_max).max() <= 2e-3 * ref.sigma_f_max.max()
    fv = out["f_var"].cpu().numpy().astype(np.float64)
    assert np.abs(fv - ref.f_var_last).max() <= 2e-3 * ref.f_var_last.max()
    assert ref.sigma_f_max.min() > 0 and ref.sigma_e.min() > 0


def test_samples_do_not_change_the_trajectory_bitwise(gm):
    """Eq. 6: both modes differentiate the same energy; the kept forces are restored after each sample."""
    w = _workload("ionic384_m8")
    runs = []
    for rate in (4, 6, 1000):
        sysm, pos, vel, mass = _system(gm, w)
        out = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, 12, rate)
        runs.append((pos.cpu().numpy(), vel.cpu().numpy(), out["epot"].cpu().numpy(), out["ekin"].cpu().numpy(), out))
    for r in runs[1:]:
        for a, b in zip(runs[0][:4], r[:4]):
            assert np.array_equal(a, b)
    assert len(runs[0][4]["sigma_e"]) == 3 and len(runs[1][4]["sigma_e"]) == 2 and len(runs[2][4]["sigma_e"]) == 0
    assert runs[0][4]["sigma_f_max"][2] == runs[1][4]["sigma_f_max"][1]  # both after step 12
    # and it is the plain mean-energy MD of gmnn_md_verlet_steps on the same model
    sysm, pos, vel, mass = _system(gm, w)
    epot, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 12)
    assert np.array_equal(pos.cpu().numpy(), runs[0][0]) and np.array_equal(epot.cpu().numpy(), runs[0][2])


def test_stopping_criterion_and_single_head(gm, orc):
    w = _workload("ionic384_m8")
    sysm, pos, vel, mass = _system(gm, w)
    full = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, 12, 3)
    assert full["n_steps_done"] == 12 and len(full["sigma_f_max"]) == 4
    thr = 0.5 * float(full["sigma_f_max"][0])  # the first sample is over it
    sysm, pos, vel, mass = _system(gm, w)
    out = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, 12, 3, f_sigma_stop=thr)
    assert out["n_steps_done"] == 3 and len(out["sigma_f_max"]) == 1 and len(out["epot"]) == 4
    assert out["sigma_f_max"][0] == full["sigma_f_max"][0]
    assert np.array_equal(out["epot"].cpu().numpy(), full["epot"].cpu().numpy()[:4])
    ref = orc.md_switching(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc,
                           w.skin, w.dt_fs, 12, 3, thr)
    assert ref.n_steps_done == 3
    sysm, pos, vel, mass = _system(gm, w)
    never = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, 12, 3, f_sigma_stop=1e9)
    assert never["n_steps_done"] == 12
    # one head: no spread
    w1 = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64))
    sysm, pos, vel, mass = _system(gm, w1)
    one = sysm.md_ensemble_steps(pos, vel, mass, w1.dt_fs, 8, 4, f_sigma_stop=1e-30)
    assert one["n_steps_done"] == 8 and np.all(one["sigma_e"] == 0) and np.all(one["sigma_f_max"] == 0)


def test_bad_arguments(gm):
    w = _workload("ionic384_m8")
    sysm, pos, vel, mass = _system(gm, w)
    with pytest.raises(gm.GmnnError) as e:
        sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, 4, 0)
    assert e.value.code == gm.GMNN_INVALID_ARG


# ------------------------------------------------------------------ UDD bias (Eq. 9) against oracle O-13
def _udd_setup(gm, orc, name, mlp_precision=0):
    w = _workload(name)
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, w.model.r_cut)
    var0 = orc.udd_energy_forces(m, w.positions, w.species, w.cell, pairs, 0.0, 1.0).var_e
    B = float(np.sqrt(var0 / (w.model.n_heads * len(w.species))))  # exponent -1 at the initial state
    return w, m, pairs, B


@pytest.mark.parametrize("mlp_precision", [0, 3])
@pytest.mark.parametrize("name", ["ionic384_m8", "li1024_m32"])
def test_udd_biased_energy_and_forces(gm, orc, name, mlp_precision):
    import torch

    w, m, pairs, B = _udd_setup(gm, orc, name)
    A = 5.0
    ref = orc.udd_energy_forces(m, w.positions, w.species, w.cell, pairs, A, B)
    plain = orc.udd_energy_forces(m, w.positions, w.species, w.cell, pairs, 0.0, B)
    assert force_error(ref.forces, plain.forces) > 50 * F_TOL  # the bias force is far above the tolerance
    sysm, pos, _, _ = _system(gm, w, mlp_precision=mlp_precision)
    sysm.set_udd_bias(A, B)
    e, e_atom, f = sysm.energy_forces(pos)
    eb, var = sysm.get_udd_bias()
    assert abs(var - ref.var_e) <= 2e-4 * ref.var_e
    assert abs(eb - ref.e_bias) <= 5e-4 * abs(ref.e_bias)
    assert abs(float(e) - ref.energy) <= 1e-5 * abs(ref.e_mean) + 5e-4 * abs(ref.e_bias) + 1e-4
    assert force_error(f.cpu().numpy().astype(np.float64), ref.forces) <= F_TOL
    # switching the bias off gives the mean-energy forces again
    sysm.set_udd_bias(0.0)
    e0, _, f0 = sysm.energy_forces(pos)
    assert force_error(f0.cpu().numpy().astype(np.float64), plain.forces) <= F_TOL
    assert sysm.get_udd_bias() == (0.0, 0.0)


def test_udd_biased_md_matches_oracle_and_samples_stay_unbiased(gm, orc):
    w, m, pairs, B = _udd_setup(gm, orc, "ionic384_m8")
    A = 2.0
    n = 10
    x, v, ep, ek, eb = orc.nve_udd(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, w.dt_fs, n, A, B)
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_udd_bias(A, B)
    out = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, n, 5)
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - x
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - v).max() <= 1e-5
    assert np.abs(out["epot"].cpu().numpy() - ep).max() <= 1e-5 * np.abs(ep).max() + 1e-3
    assert abs(sysm.get_udd_bias()[0] - eb[-1]) <= 1e-3 * np.abs(eb).max()
    # and the biased run is not the plain one
    sysm2, pos2, vel2, mass2 = _system(gm, w)
    out2 = sysm2.md_ensemble_steps(pos2, vel2, mass2, w.dt_fs, n, 5)
    assert np.abs(pos2.cpu().numpy() - pos.cpu().numpy()).max() > 1e-5
    # the uncertainty sample is Eq. 5 on the unbiased heads at the biased run's positions
    xg = pos.cpu().numpy()
    xw = (xg.astype(np.float64) - np.floor(xg.astype(np.float64) / L) * L).astype(np.float32)
    xw = np.where(xw >= w.cell[None, :], 0.0, xw).astype(np.float32)
    ens = orc.ensemble(m, xw, w.species, w.cell, orc.auto_neighbors(xw, w.cell, w.pbc, w.model.r_cut))
    assert abs(out["sigma_e"][-1] - np.std(ens.e_heads.sum(0))) <= 2e-4 * np.std(ens.e_heads.sum(0))


def test_udd_bad_arguments_and_single_head(gm):
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64))
    sysm, pos, _, _ = _system(gm, w)
    with pytest.raises(gm.GmnnError):
        sysm.set_udd_bias(1.0, 0.0)
    e0, _, f0 = sysm.energy_forces(pos)
    sysm.set_udd_bias(3.0, 0.5)  # one head: sigma = 0, nothing changes
    e1, _, f1 = sysm.energy_forces(pos)
    assert float(e0) == float(e1) and bool((f0 == f1).all())
