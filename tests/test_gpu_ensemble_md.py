"""GPU parity for the shallow ensemble (Eq. 5, 6) and the NVE loop (configs 2, 4, 5 shaped)."""
import numpy as np
import pytest

import workloads as wl
from parity_utils import F_TOL, energy_atom_error, force_error, r_list32

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (they must not pass on a fallback)")
    import paper_2505_22168_b200 as pkg

    return pkg


def _build(gm, w, **kw):
    import torch

    model = gm.Model(w.model, **kw)
    sysm = gm.System(model, w.species)
    pos = torch.from_numpy(w.positions).cuda()
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    return model, sysm, pos


@pytest.mark.parametrize("name", ["tiny8", "config4_1024"])
def test_ensemble_statistics(gm, orc, name):
    w = wl.tiny_box(n_heads=8) if name == "tiny8" else wl.li3po4_box(1024, n_heads=32)
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    ref = orc.ensemble(m, w.positions, w.species, w.cell, pairs)
    _, sysm, pos = _build(gm, w)
    e_mean, e_var, f_mean, f_var = (t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos))
    assert energy_atom_error(e_mean, ref.e_mean) <= 1.0
    assert force_error(f_mean, ref.f_mean) <= F_TOL
    # variances: second moments of quantities that each carry ~1e-5 relative error
    assert np.abs(e_var - ref.e_var).max() <= 2e-4 * max(ref.e_var.max(), 1e-30)
    assert np.abs(f_var - ref.f_var).max() <= 2e-4 * ref.f_var.max()
    assert np.all(e_var >= 0) and np.all(f_var >= 0)
    # Eq. 6 on the GPU itself: the cheap mode (gradient of the mean energy) equals the mean of the heads
    _, ea, f = sysm.energy_forces(pos)
    assert force_error(f.cpu().numpy().astype(np.float64), f_mean) <= 2e-5
    assert energy_atom_error(ea.cpu().numpy().astype(np.float64), e_mean) <= 1.0


@pytest.mark.parametrize("batch", [1, 5, 12])
@pytest.mark.parametrize("mlp_precision", [2, 3])
def test_ensemble_batches_of_heads(gm, orc, batch, mlp_precision):
    """The batched pass (all heads through one backward GEMM chain, one pair-backward kernel for 8 heads at a time) in
    uneven batches -- 5 + 5 + 5 + 5 + 5 + 5 + 2, 12 + 12 + 8, and head by head -- against the oracle, at the bounds of the
    unbatched test; batches differ from one another only by the power-of-two operand scales of the split GEMMs."""
    w = wl.li3po4_box(1024, n_heads=32)
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    ref = orc.ensemble(m, w.positions, w.species, w.cell, pairs)
    mode = gm.GMNN_MLP_3XF16 if mlp_precision == 3 else gm.GMNN_MLP_3XTF32
    _, sysm, pos = _build(gm, w, mlp_precision=mode, force_mode=gm.GMNN_FORCE_PAIRBUF)
    full = [t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos)]
    sysm.set_int("ensemble_batch", batch)
    part = [t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos)]
    sysm.set_int("ensemble_batch", 0)
    for e_mean, e_var, f_mean, f_var in (full, part):
        assert energy_atom_error(e_mean, ref.e_mean) <= 1.0
        assert force_error(f_mean, ref.f_mean) <= F_TOL
        assert np.abs(e_var - ref.e_var).max() <= 2e-4 * ref.e_var.max()
        assert np.abs(f_var - ref.f_var).max() <= 2e-4 * ref.f_var.max()
    assert force_error(part[2], full[2]) <= 2e-5 and np.abs(part[3] - full[3]).max() <= 1e-4 * full[3].max()
    assert np.array_equal(part[0], full[0]) and np.array_equal(part[1], full[1])  # the forward does not depend on the batching


@pytest.mark.parametrize("lanes", [1, 2, 4, 32])
def test_ensemble_heads_kernel_lane_groupings_sheared_cell(gm, orc, lanes):
    """The batched pair backward stages the adjoints of as many heads per chunk as 96 KB of shared memory hold beside the
    128 / lanes centres of a block (1 head at one lane per atom, 3 at two, 7 at four, 8 from eight lanes on): every
    chunking against the oracle, on a sheared cell (lattice shifts inside the kernel), 12 heads."""
    w = wl.triclinic_box(1000, hidden=(64, 64), n_heads=12)
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.box, w.pbc, r_list32(w.model.r_cut, w.skin))
    ref = orc.ensemble(m, w.positions, w.species, w.box, pairs)
    _, sysm, pos = _build(gm, w, mlp_precision=gm.GMNN_MLP_3XF16, force_mode=gm.GMNN_FORCE_PAIRBUF)
    sysm.set_int("lanes_per_atom", lanes)
    e_mean, e_var, f_mean, f_var = (t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos))
    sysm.check()
    assert energy_atom_error(e_mean, ref.e_mean) <= 1.0
    assert force_error(f_mean, ref.f_mean) <= F_TOL
    assert np.abs(e_var - ref.e_var).max() <= 2e-4 * ref.e_var.max()
    assert np.abs(f_var - ref.f_var).max() <= 2e-4 * ref.f_var.max()


def test_config4_full_size(gm, orc):
    """Config 4 at its stated size (8 192 atoms, 32 heads): e_mean, e_var, f_mean and f_var element by
    element against oracle O-10 (one forward, 32 backward passes in fp64; about 20 s on 16 cores), at the
    bounds used for the 1 024-atom box.  PAPER.md:75-88 (Eq. 5, 6)."""
    w = wl.make_workload("config4")
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    ref = orc.ensemble(m, w.positions, w.species, w.cell, pairs)
    _, sysm, pos = _build(gm, w)
    e_mean, e_var, f_mean, f_var = (t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos))
    assert energy_atom_error(e_mean, ref.e_mean) <= 1.0
    assert force_error(f_mean, ref.f_mean) <= F_TOL
    assert np.abs(e_var - ref.e_var).max() <= 2e-4 * ref.e_var.max()
    assert np.abs(f_var - ref.f_var).max() <= 2e-4 * ref.f_var.max()
    assert np.all(e_var >= 0) and np.all(f_var >= 0)
    # the same call in bench.py's configuration (3xFP16 MLP on tcgen05, pair-buffer forces)
    _, sysm2, pos2 = _build(gm, w, mlp_precision=gm.GMNN_MLP_3XF16, force_mode=gm.GMNN_FORCE_PAIRBUF)
    e_mean, e_var, f_mean, f_var = (t.cpu().numpy().astype(np.float64) for t in sysm2.ensemble_energy_forces(pos2))
    assert energy_atom_error(e_mean, ref.e_mean) <= 1.0
    assert force_error(f_mean, ref.f_mean) <= F_TOL
    assert np.abs(e_var - ref.e_var).max() <= 2e-4 * ref.e_var.max()
    assert np.abs(f_var - ref.f_var).max() <= 2e-4 * ref.f_var.max()


def test_md_trajectory_and_energy_conservation(gm, orc):
    """Config-2-shaped NVE: trajectory parity for the first 10 steps (|dx| <= 1e-4 Ang), then state
    parity (oracle E, F at the GPU's own final positions), drift within 10x of the fp64 oracle's."""
    import torch

    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64))  # 384 atoms, L = 15.9 Ang: image path (2 cells)
    m = orc.Model(w.model)
    _, sysm, pos = _build(gm, w)
    vel = torch.from_numpy(w.velocities).cuda()
    mass = torch.from_numpy(w.masses).cuda()
    epot, ekin, nreb = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)
    ref = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, w.skin, w.dt_fs, 10)
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - ref.positions
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - ref.velocities).max() <= 1e-5
    ep, ek = epot.cpu().numpy(), ekin.cpu().numpy()
    assert np.abs(ep - ref.epot).max() <= 1e-5 * np.abs(ref.epot).max() + 1e-4
    assert np.abs(ek - ref.ekin).max() <= 1e-4 * np.abs(ref.ekin).max()
    # continue for 90 more steps, then check the state against the oracle at the GPU's own positions
    epot2, ekin2, nreb2 = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 90)
    x = pos.cpu().numpy()
    xw = (x.astype(np.float64) - np.floor(x.astype(np.float64) / L) * L).astype(np.float32)
    xw = np.where(xw >= w.cell[None, :], 0.0, xw).astype(np.float32)
    pairs = orc.auto_neighbors(xw, w.cell, w.pbc, w.model.r_cut)
    state = orc.energy_forces(m, xw, w.species, w.cell, pairs)
    assert abs(float(epot2[-1]) - state.energy) <= 2e-6 * np.abs(state.e_atom).sum()
    assert nreb + nreb2 >= 1  # hydrogens at 300 K cross skin/2 = 0.25 Ang within 100 steps
    ref100 = orc.nve(m, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, w.skin, w.dt_fs, 100)
    drift_ref = np.abs(ref100.epot + ref100.ekin - (ref100.epot[0] + ref100.ekin[0])).max()
    etot = np.concatenate([ep + ek, (epot2.cpu().numpy() + ekin2.cpu().numpy())[1:]])
    drift_gpu = np.abs(etot - etot[0]).max()
    assert drift_gpu <= 10 * drift_ref + 1e-3, (drift_gpu, drift_ref)


@pytest.mark.parametrize("force_mode", [0, 1])
def test_md_cell_list_rebuild_inside_the_loop(gm, orc, force_mode):
    """Config-5-shaped (Li3PO4, skin > 0, cell-list rebuild when max displacement > skin/2) at 8192
    atoms: fast atoms force several device-side rebuilds (k_wrap, two-part rows, reverse-pair index).
    (1) The list the loop left in the handle must be, as a sorted (i, j, n) set, bit for bit the oracle's
    list at the positions of the last rebuild (`xref`), at r_cut + skin; (2) the final state must match
    the oracle evaluated on the GPU's final positions within north_star's bounds."""
    import torch

    w = wl.li3po4_box(8192, hidden=(64, 64), skin=0.3)
    m = orc.Model(w.model)
    _, sysm, pos = _build(gm, w, force_mode=force_mode)  # 1: the reverse-pair index is rebuilt in the loop too
    vel = torch.from_numpy(w.velocities * 5.0).cuda()
    mass = torch.from_numpy(w.masses).cuda()
    epot, ekin, nreb = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 30)
    assert nreb >= 2
    # (1) neighbour set of the in-loop rebuild against the oracle at the rebuild's reference positions
    xref = sysm.debug_read("xref")
    assert (xref >= 0).all() and (xref < w.cell[None, :]).all()  # wrapped by k_wrap
    ref_pairs = orc.auto_neighbors(xref, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    assert np.array_equal(sysm.get_neighbors(), ref_pairs.as_set_array())
    # (2) state parity at the GPU's own final positions
    x = pos.cpu().numpy()
    L = w.cell.astype(np.float64)
    xw = (x.astype(np.float64) - np.floor(x.astype(np.float64) / L) * L).astype(np.float32)
    xw = np.where(xw >= w.cell[None, :], 0.0, xw).astype(np.float32)
    pairs = orc.auto_neighbors(xw, w.cell, w.pbc, w.model.r_cut)
    state = orc.energy_forces(m, xw, w.species, w.cell, pairs)
    assert abs(float(epot[-1]) - state.energy) <= 2e-6 * np.abs(state.e_atom).sum()
    # energy+forces on the returned (unwrapped-continuation) positions with the list left in the handle
    e, ea, f = sysm.energy_forces(pos)
    sysm.check()
    assert energy_atom_error(ea.cpu().numpy().astype(np.float64), state.e_atom) <= 1.0
    assert force_error(f.cpu().numpy().astype(np.float64), state.forces) <= F_TOL
    etot = (epot + ekin).cpu().numpy()
    assert np.abs(etot - etot[0]).max() <= 2e-3 * np.abs(ekin.cpu().numpy()).max()


def test_md_entry_with_moved_atoms_is_reported(gm):
    """gmnn_md_verlet_steps runs the skin test on its entry state too: positions that moved more than
    skin/2 since gmnn_build_neighbors give GMNN_STALE_NEIGHBORS, not a silently stale first step."""
    import torch

    w = wl.li3po4_box(1024, hidden=(32, 32), skin=0.4)
    _, sysm, pos = _build(gm, w)
    vel = torch.from_numpy(w.velocities).cuda()
    mass = torch.from_numpy(w.masses).cuda()
    moved = pos.clone()
    moved[7, 0] += 0.3  # > skin / 2 = 0.2
    with pytest.raises(gm.GmnnError) as e:
        sysm.md_verlet_steps(moved, vel, mass, w.dt_fs, 2)
    assert e.value.code == gm.GMNN_STALE_NEIGHBORS
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 2)  # a fresh list clears it


@pytest.mark.parametrize("mlp_precision", [1, 3])
@pytest.mark.parametrize("force_mode", [0, 1])
def test_md_graph_replay_is_bitwise_the_eager_loop(gm, force_mode, mlp_precision):
    """gmnn_md_verlet_steps replays the step as a CUDA graph (knob md_graph, default on): positions,
    velocities, both energy series and the rebuild count are bit-identical to the eager loop, across
    in-loop rebuilds and across a continued call."""
    import torch

    w = wl.li3po4_box(1024, hidden=(64, 64), skin=0.3)
    out = []
    for graph in (1, 0):
        _, sysm, pos = _build(gm, w, mlp_precision=mlp_precision, force_mode=force_mode)
        sysm.set_int("md_graph", graph)
        vel = torch.from_numpy(w.velocities * 6.0).cuda()
        mass = torch.from_numpy(w.masses).cuda()
        ep, ek, nreb = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 25)
        sysm.set_int("md_continue", 1)
        ep2, ek2, nreb2 = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 7)
        out.append((pos.cpu().numpy(), vel.cpu().numpy(), ep.cpu().numpy(), ek.cpu().numpy(), ep2.cpu().numpy(),
                    ek2.cpu().numpy(), nreb, nreb2))
    assert out[0][6] >= 2  # rebuilds happened inside the replayed steps
    for a, b in zip(out[0], out[1]):
        assert np.array_equal(a, b)
    assert np.isfinite(out[0][2]).all() and out[0][2].shape == (26,) and out[0][4].shape == (8,)
