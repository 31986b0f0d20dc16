"""GPU parity for general (triclinic) lattices and the virial (oracle O-16):
neighbour sets bit-exact in sheared cells (image loop with second images, cell list in fractional coordinates,
mixed periodicity), E_i / F within north_star's bounds, W = -sum_pairs d (x) g against the oracle, MD with
device-side rebuilds (k_wrap in fractional coordinates) against the oracle's trajectory."""
import numpy as np
import pytest

import workloads as wl
from parity_utils import E_TOTAL_RTOL, F_TOL, energy_atom_error, force_error, r_list32

pytestmark = pytest.mark.gpu

W_TOL = 2e-5  # max |dW_ab| / max |W|: fp32 terms d_a g_b (forces carry ~1e-5), fp64 sum; measured 3e-7 .. 2e-6


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


@pytest.mark.parametrize("name", ["tri8", "tri216", "tri4096", "tri4096_skin", "tri4096_mixed", "tri1000_flat"])
def test_neighbor_sets_bit_exact(gm, orc, name):
    if name == "tri8":
        w = wl.triclinic_box(8, hidden=(16, 16))  # faces 4 Ang apart: second images
    elif name == "tri216":
        w = wl.triclinic_box(216, hidden=(16, 16))  # < 3 slabs: image loop
    elif name == "tri4096":
        w = wl.triclinic_box(4096, hidden=(16, 16))  # cell list in fractional coordinates
    elif name == "tri4096_skin":
        w = wl.triclinic_box(4096, hidden=(16, 16), skin=1.0)
    elif name == "tri4096_mixed":
        w = wl.triclinic_box(4096, hidden=(16, 16))
        w.pbc = (1, 0, 1)
    else:
        w = wl.triclinic_box(1000, hidden=(16, 16), shear=(0.6, -0.45, 0.5), stretch=(1.3, 0.8, 1.0))  # strongly sheared
    sysm, _ = _gpu(gm, w)
    ref = orc.auto_neighbors(w.positions, w.lattice, w.pbc, r_list32(w.model.r_cut, w.skin)).as_set_array()
    got = sysm.get_neighbors()
    assert got.shape == ref.shape and np.array_equal(got, ref)
    if name == "tri8":
        assert np.abs(got[:, 2:]).max() >= 2
    if name.startswith("tri4096"):
        assert sysm.get_int("small_box") == 0 and sysm.get_int("n_cells") >= 27


@pytest.mark.parametrize("mlp_precision,force_mode", [(0, 0), (0, 1), (3, 1), (3, 0)])
@pytest.mark.parametrize("name", ["tri1000", "tri216", "config1", "config2", "config3_1024"])
def test_energy_forces_virial(gm, orc, name, mlp_precision, force_mode):
    w = wl.triclinic_box(int(name[3:])) if name.startswith("tri") else wl.make_workload(name)
    pairs = orc.auto_neighbors(w.positions, w.box, w.pbc, r_list32(w.model.r_cut, w.skin))
    ref = orc.energy_forces(orc.Model(w.model), w.positions, w.species, w.box, pairs)
    sysm, pos = _gpu(gm, w, mlp_precision=mlp_precision, force_mode=force_mode)
    e, ea, f, W = sysm.energy_forces_virial(pos)
    sysm.check()
    ea, f, e, W = ea.cpu().numpy().astype(np.float64), f.cpu().numpy().astype(np.float64), float(e.cpu()[0]), W.cpu().numpy()
    assert energy_atom_error(ea, ref.e_atom) <= 1.0
    assert force_error(f, ref.forces) <= F_TOL
    assert abs(e - ref.energy) <= E_TOTAL_RTOL * np.abs(ref.e_atom).sum()
    werr = np.abs(W - ref.virial).max()
    print("%s mlp %d forces %d: max |dW| = %.3e, max |W| = %.3e" % (name, mlp_precision, force_mode, werr, np.abs(ref.virial).max()))
    assert werr <= W_TOL * np.abs(ref.virial).max()
    assert np.abs(W - W.T).max() <= 2 * W_TOL * np.abs(ref.virial).max()
    # the plain entry gives the same energies and forces bit for bit, and the virial is reproducible
    e2, ea2, f2 = sysm.energy_forces(pos)
    assert np.array_equal(f2.cpu().numpy(), f.astype(np.float32)) and np.array_equal(ea2.cpu().numpy(), ea.astype(np.float32))
    W2 = sysm.energy_forces_virial(pos)[3].cpu().numpy()
    assert np.array_equal(W, W2)


@pytest.mark.parametrize("force_mode", [0, 1])
def test_md_in_a_sheared_cell(gm, orc, force_mode):
    """NVE in a triclinic cell with device-side rebuilds: the first 10 steps against the oracle's trajectory, the
    list of the last in-loop rebuild against the oracle's at the rebuild's positions, energy conservation."""
    import torch

    w = wl.triclinic_box(4096, hidden=(64, 64), skin=0.3)
    sysm, pos = _gpu(gm, w, mlp_precision=3, force_mode=force_mode)
    vel = torch.from_numpy(w.velocities * 4.0).cuda()
    mass = torch.from_numpy(w.masses).cuda()
    epot, ekin, nreb = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)
    ref = orc.nve(orc.Model(w.model), w.positions, w.velocities * 4.0, w.masses, w.species, w.lattice, w.pbc, w.skin, w.dt_fs, 10)
    d = pos.cpu().numpy().astype(np.float64) - ref.positions
    d -= np.round(d @ np.linalg.inv(w.lattice.astype(np.float64))) @ w.lattice.astype(np.float64)
    assert np.abs(d).max() <= 1e-4
    assert np.abs(epot.cpu().numpy() - ref.epot).max() <= 1e-5 * np.abs(ref.epot).max() + 1e-4
    ep2, ek2, nreb2 = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 30)
    assert nreb + nreb2 >= 2
    xref = sysm.debug_read("xref")
    frac = xref.astype(np.float64) @ np.linalg.inv(w.lattice.astype(np.float64))
    assert frac.min() >= -1e-5 and frac.max() < 1.0 + 1e-5  # folded into the cell by the in-loop wrap
    ref_pairs = orc.auto_neighbors(xref, w.lattice, w.pbc, r_list32(w.model.r_cut, w.skin))
    assert np.array_equal(sysm.get_neighbors(), ref_pairs.as_set_array())
    etot = np.concatenate([(epot + ekin).cpu().numpy(), (ep2 + ek2).cpu().numpy()[1:]])
    assert np.abs(etot - etot[0]).max() <= 2e-3 * np.abs(ekin.cpu().numpy()).max()
