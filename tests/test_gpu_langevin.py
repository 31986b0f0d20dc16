"""GPU parity for Langevin dynamics (BAOAB, reading R29) against oracle O-15."""
import numpy as np
import pytest

import workloads as wl

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


@pytest.mark.parametrize("gamma,first_step", [(0.02, 0), (2.0, 7)])
@pytest.mark.parametrize("name", ["ionic384", "li1024"])
def test_langevin_trajectory_matches_oracle(gm, orc, name, gamma, first_step):
    """Same seed, same counters: the GPU draws the oracle's normals, so the trajectories agree step by step."""
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64)) if name == "ionic384" else \
        wl.li3po4_box(1024, hidden=(64, 64), skin=0.5)
    T, n, seed = 600.0, 10, 2505221680
    x, v, ep, ek = orc.nvt_langevin(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell,
                                    w.pbc, w.dt_fs, n, T, gamma, seed, first_step)
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_langevin(T, gamma, seed, first_step)
    epot, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, n)
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - x
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - v).max() <= 1e-5
    assert np.abs(epot.cpu().numpy() - ep).max() <= 1e-5 * np.abs(ep).max() + 1e-4
    assert np.abs(ekin.cpu().numpy() - ek).max() <= 1e-4 * np.abs(ek).max()
    # the noise did act: a run without it ends elsewhere
    ref = orc.nve(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, w.skin, w.dt_fs, n)
    assert np.abs(vel.cpu().numpy() - ref.velocities).max() > 1e-3


def test_langevin_replay_continuation_and_switches(gm):
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64))
    runs = []
    for graph in (1, 0):
        sysm, pos, vel, mass = _system(gm, w)
        sysm.set_int("md_graph", graph)
        sysm.set_langevin(450.0, 0.05, 11)
        epot, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)
        runs.append((pos.cpu().numpy(), vel.cpu().numpy(), epot.cpu().numpy(), ekin.cpu().numpy()))
    for a, b in zip(runs[0], runs[1]):
        assert np.array_equal(a, b)  # graph replay = eager loop: the step counter lives on the device
    # two calls continue the same noise stream
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_int("md_continue", 1)
    sysm.set_langevin(450.0, 0.05, 11)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 4)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 6)
    assert np.array_equal(pos.cpu().numpy(), runs[0][0]) and np.array_equal(vel.cpu().numpy(), runs[0][1])
    # restarting at first_step = 4 from the state after 4 steps gives the same end state
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_langevin(450.0, 0.05, 11)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 4)
    sysm2 = gm.System(gm.Model(w.model), w.species)
    sysm2.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    sysm2.set_langevin(450.0, 0.05, 11, 4)
    sysm2.md_verlet_steps(pos, vel, mass, w.dt_fs, 6)
    assert np.abs(vel.cpu().numpy() - runs[0][1]).max() <= 2e-5  # new list order: equal up to summation order
    # another seed: another trajectory; gamma = 0: NVE bit for bit; off: NVE
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_langevin(450.0, 0.05, 12)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)
    assert not np.array_equal(vel.cpu().numpy(), runs[0][1])
    nve_sys, p0, v0, m0 = _system(gm, w)
    e_nve = nve_sys.md_verlet_steps(p0, v0, m0, w.dt_fs, 10)[0].cpu().numpy()
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_langevin(450.0, 0.05, 12)
    sysm.set_langevin(0.0)
    e_off = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)[0].cpu().numpy()
    assert np.array_equal(e_off, e_nve) and np.array_equal(pos.cpu().numpy(), p0.cpu().numpy())
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_langevin(450.0, 0.0, 12)  # c1 = 1, c2 = 0: two half drifts instead of one, same to rounding
    e_g0 = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)[0].cpu().numpy()
    assert np.abs(e_g0 - e_nve).max() <= 1e-5 * np.abs(e_nve).max() + 1e-4
    # one thermostat at a time
    sysm.set_langevin(300.0, 0.01, 1)
    with pytest.raises(gm.GmnnError):
        sysm.set_nose_hoover(300.0, 50.0)
    sysm.set_langevin(0.0)
    sysm.set_nose_hoover(300.0, 50.0)
    with pytest.raises(gm.GmnnError):
        sysm.set_langevin(300.0, 0.01, 1)
    with pytest.raises(gm.GmnnError):
        sysm.set_langevin(300.0, -1.0, 1)


def test_strong_friction_thermalises_at_the_target(gm):
    """gamma dt >> 1 on 8 192 atoms: E_kin = 3/2 N kT within a few standard deviations (0.9 % each)."""
    w = wl.li3po4_box(8192, hidden=(64, 64), skin=0.5)
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_langevin(500.0, 50.0, 3)
    _, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 8)
    target = 1.5 * 8192 * wl.KB_EV * 500.0
    assert abs(float(ekin[1:].mean()) / target - 1.0) < 0.03
