"""GPU parity for per-species weight sets (`n_weight_sets = n_species`; north_star "the per-species atomic MLP",
SURVEY.md 8(b)/8(c-1) O-5): the CUDA path groups the rows of the MLP stage by species (every GEMM tile uses one
weight set) and must give the oracle's E_i and F within north_star's bounds on configs 1-3, in every MLP mode
and both force forms, across in-loop rebuilds, and at config 5's size."""
import dataclasses

import numpy as np
import pytest

import workloads as wl
from parity_utils import (E_ATOM_RTOL, E_TOTAL_RTOL, F_TOL, energy_atom_error, force_error, r_list32, unique_from_full)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (they must not pass on a fallback)")
    import paper_2505_22168_b200 as pkg

    return pkg


def _gpu(gm, w, **kw):
    import torch

    sysm = gm.System(gm.Model(w.model, **kw), w.species)
    pos = torch.from_numpy(w.positions).cuda()
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    return sysm, pos


def _ref(orc, w, **kw):
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    return orc.energy_forces(orc.Model(w.model), w.positions, w.species, w.cell, pairs, **kw)


def _workload(name):
    if name == "config1":
        return wl.tiny_box(n_weight_sets=2)
    if name == "config2":
        return wl.ionic_liquid_box(n_weight_sets=5)
    return wl.li3po4_box(int(name.split("_")[1]), n_weight_sets=3)


@pytest.mark.parametrize("mlp_precision,force_mode", [(0, 0), (1, 1), (3, 1), (3, 0)])
@pytest.mark.parametrize("name", ["config1", "config2", "config3_1024", "config3_8192", "config3_1000"])
def test_energy_forces_against_the_oracle(gm, orc, name, mlp_precision, force_mode):
    w = _workload(name)
    assert w.model.n_weight_sets == w.model.n_species
    ref = _ref(orc, w)
    sysm, pos = _gpu(gm, w, mlp_precision=mlp_precision, force_mode=force_mode)
    e, ea, f = sysm.energy_forces(pos)
    sysm.check()
    ea, f, e = ea.cpu().numpy().astype(np.float64), f.cpu().numpy().astype(np.float64), float(e.cpu()[0])
    assert energy_atom_error(ea, ref.e_atom) <= 1.0
    assert force_error(f, ref.forces) <= F_TOL
    assert abs(e - ref.energy) <= E_TOTAL_RTOL * np.abs(ref.e_atom).sum()
    # the sets do differ: with every atom on set 0 (the shared model of the same seed) the energies are others
    shared = _ref(orc, dataclasses.replace(w, model=dataclasses.replace(
        w.model, n_weight_sets=1, W=[x[0] for x in w.model.W], b=[x[0] for x in w.model.b])))
    assert energy_atom_error(shared.e_atom, ref.e_atom) > 100.0


def test_stage_intermediates_in_row_order(gm, orc):
    """psi, G, dG, A of the species-grouped rows, handed back in atom order, against the oracle."""
    w = wl.li3po4_box(1000, n_weight_sets=3)
    ref = _ref(orc, w, intermediates=True)
    sysm, pos = _gpu(gm, w)
    sysm.energy_forces(pos)
    perm = sysm.debug_read("perm")
    psi_ref = unique_from_full(ref.P, summed=False)[perm]
    assert np.abs(sysm.debug_read("psi") - psi_ref).max() <= 2e-6 * np.abs(psi_ref).max()
    assert np.abs(sysm.debug_read("G") - ref.G[perm]).max() <= 5e-6 * np.abs(ref.G).max()
    sig = w.model.scale[w.species][perm][:, None]
    dG_ref = ref.dG[perm] / sig
    assert np.abs(sysm.debug_read("dG") - dG_ref).max() <= 1e-4 * np.abs(dG_ref).max()
    A_ref = unique_from_full(ref.Q, summed=True)[perm]
    assert np.abs(sysm.debug_read("A") - A_ref).max() <= 1e-4 * np.abs(A_ref).max()


@pytest.mark.parametrize("mlp_precision", [0, 3])
def test_identical_sets_are_bitwise_the_shared_model(gm, mlp_precision):
    """S copies of one network: every row sees the same arithmetic as in the shared-NN layout, wherever it sits,
    so E_i and F are bit-identical (row grouping, padding rows and per-set launches change no result)."""
    w = wl.li3po4_box(1000, hidden=(64, 64))
    rep = dataclasses.replace(w, model=dataclasses.replace(
        w.model, n_weight_sets=3, W=[np.repeat(x[None], 3, 0) for x in w.model.W], b=[np.repeat(x[None], 3, 0) for x in w.model.b]))
    out = []
    for ww in (w, rep):
        sysm, pos = _gpu(gm, ww, mlp_precision=mlp_precision, force_mode=1)
        e, ea, f = sysm.energy_forces(pos)
        out.append((ea.cpu().numpy(), f.cpu().numpy(), float(e.cpu()[0])))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1]) and out[0][2] == out[1][2]


def test_md_with_rebuilds_and_heads(gm, orc):
    """Rows are re-assigned at every in-loop rebuild: 10-step trajectory against the oracle's NVE, then the
    shallow-ensemble statistics of a per-species multi-head model (Eq. 5, 6)."""
    import torch

    w = wl.li3po4_box(1024, hidden=(64, 64), skin=0.3, n_weight_sets=3)
    sysm, pos = _gpu(gm, w, mlp_precision=3, force_mode=1)
    vel = torch.from_numpy(w.velocities * 4.0).cuda()
    mass = torch.from_numpy(w.masses).cuda()
    epot, ekin, nreb = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)
    assert nreb >= 1
    ref = orc.nve(orc.Model(w.model), w.positions, w.velocities * 4.0, w.masses, w.species, w.cell, w.pbc, w.skin, w.dt_fs, 10)
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - ref.positions
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(epot.cpu().numpy() - ref.epot).max() <= 1e-5 * np.abs(ref.epot).max() + 1e-4

    wh = wl.li3po4_box(1024, hidden=(64, 64), n_heads=8, n_weight_sets=3)
    pairs = orc.auto_neighbors(wh.positions, wh.cell, wh.pbc, r_list32(wh.model.r_cut, wh.skin))
    ens = orc.ensemble(orc.Model(wh.model), wh.positions, wh.species, wh.cell, pairs)
    for prec in (0, 3):
        sysm, pos = _gpu(gm, wh, mlp_precision=prec, force_mode=1)
        e_mean, e_var, f_mean, f_var = (t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos))
        assert energy_atom_error(e_mean, ens.e_mean) <= 1.0
        assert force_error(f_mean, ens.f_mean) <= F_TOL
        assert np.abs(e_var - ens.e_var).max() <= 2e-4 * ens.e_var.max()
        assert np.abs(f_var - ens.f_var).max() <= 2e-4 * ens.f_var.max()
        _, ea, f = sysm.energy_forces(pos)  # the folded mean head per set
        assert energy_atom_error(ea.cpu().numpy().astype(np.float64), ens.e_mean) <= 1.0
        assert force_error(f.cpu().numpy().astype(np.float64), ens.f_mean) <= F_TOL


def test_config5_size_sampled_atoms(gm, orc):
    """1 048 576 atoms, per-species sets, bench.py's launch configuration: sampled atoms one by one against the
    oracle on their 2 r_cut surroundings."""
    import torch

    from test_gpu_full_size import _cluster_reference
    from workloads.inputs import splitmix64

    w = wl.make_workload("config5", n_weight_sets=3)
    sysm, pos = _gpu(gm, w, mlp_precision=gm.GMNN_MLP_3XF16, force_mode=gm.GMNN_FORCE_PAIRBUF)
    e, ea, f = sysm.energy_forces(pos)
    sysm.check()
    ea, f = ea.cpu().numpy().astype(np.float64), f.cpu().numpy().astype(np.float64)
    N = w.n_atoms
    assert abs(float(e.cpu()[0]) - ea.sum()) <= 1e-6 * np.abs(ea).sum()
    rms = np.sqrt((f ** 2).mean())
    assert np.abs(f.sum(0)).max() <= 1e-4 * rms * np.sqrt(N)
    omodel = orc.Model(w.model)
    idx = (splitmix64(777 + N, 24) % np.uint64(N)).astype(np.int64)
    e_scale = np.abs(ea).mean()
    for i in idx:
        e_ref, f_ref, _ = _cluster_reference(orc, omodel, w, int(i))
        assert abs(ea[i] - e_ref) <= E_ATOM_RTOL * max(abs(e_ref), e_scale)
        assert np.abs(f[i] - f_ref).max() <= F_TOL * rms
