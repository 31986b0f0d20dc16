"""GPU parity for NVT with a Nose-Hoover chain against oracle O-14."""
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


@pytest.mark.parametrize("chain", [(3, 2, 3), (1, 1, 1), (4, 1, 5)])
@pytest.mark.parametrize("name", ["ionic384", "li1024"])
def test_nvt_trajectory_chain_state_and_conserved_energy(gm, orc, name, chain):
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64)) if name == "ionic384" else \
        wl.li3po4_box(1024, hidden=(64, 64), skin=0.5)
    T, tau, n = 600.0, 25.0, 12
    length, csteps, sy = chain
    x, v, ep, ek, cons = orc.nvt_nose_hoover(orc.Model(w.model), w.positions, w.velocities, w.masses, w.species,
                                             w.cell, w.pbc, w.dt_fs, n, T, tau, length, csteps, sy)
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_nose_hoover(T, tau, length, csteps, sy)
    epot, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, n)
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - x
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - v).max() <= 1e-5
    eg, kg = epot.cpu().numpy(), ekin.cpu().numpy()
    assert np.abs(eg - ep).max() <= 1e-5 * np.abs(ep).max() + 1e-4
    assert np.abs(kg - ek).max() <= 1e-4 * np.abs(ek).max()
    xi, pxi, e_thermo = sysm.get_nose_hoover()
    ref_thermo = cons[-1] - ep[-1] - ek[-1]
    assert len(xi) == length and abs(e_thermo - ref_thermo) <= 2e-4 * np.abs(ek).max()
    # extended energy: conserved as well as the fp64 oracle conserves it, up to fp32 round-off of the state
    cons_gpu = eg[-1] + kg[-1] + e_thermo - (eg[0] + kg[0])
    assert abs(cons_gpu) <= np.abs(cons - cons[0]).max() + 1e-4 * np.abs(ek).max()
    assert abs((eg + kg)[-1] - (eg + kg)[0]) > 20 * abs(cons_gpu)  # while E_pot + E_kin alone is not


def test_nvt_graph_replay_is_the_eager_loop_and_off_means_nve(gm):
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64))
    runs = []
    for graph in (1, 0):
        sysm, pos, vel, mass = _system(gm, w)
        sysm.set_int("md_graph", graph)
        sysm.set_nose_hoover(450.0, 30.0)
        epot, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)
        runs.append((pos.cpu().numpy(), vel.cpu().numpy(), epot.cpu().numpy(), ekin.cpu().numpy(), sysm.get_nose_hoover()))
    for a, b in zip(runs[0][:4], runs[1][:4]):
        assert np.array_equal(a, b)
    assert np.array_equal(runs[0][4][1], runs[1][4][1])
    # continuing in two calls is the same trajectory
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_int("md_continue", 1)
    sysm.set_nose_hoover(450.0, 30.0)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 4)
    sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 6)
    assert np.array_equal(pos.cpu().numpy(), runs[0][0])
    # off again: plain NVE
    sysm, pos, vel, mass = _system(gm, w)
    sysm.set_nose_hoover(450.0, 30.0)
    sysm.set_nose_hoover(0.0)
    e1 = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 10)[0].cpu().numpy()
    sysm2, pos2, vel2, mass2 = _system(gm, w)
    e2 = sysm2.md_verlet_steps(pos2, vel2, mass2, w.dt_fs, 10)[0].cpu().numpy()
    assert np.array_equal(e1, e2) and np.array_equal(pos.cpu().numpy(), pos2.cpu().numpy())
    with pytest.raises(gm.GmnnError):
        sysm.set_nose_hoover(300.0, 50.0, 9, 2, 3)
    with pytest.raises(gm.GmnnError):
        sysm.set_nose_hoover(300.0, 50.0, 3, 2, 4)


def test_nvt_with_switching_ensemble_md(gm, orc):
    """The thermostat composes with the switching-mode loop: samples do not disturb the chain."""
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64), n_heads=8)
    outs = []
    for rate in (4, 1000):
        sysm, pos, vel, mass = _system(gm, w)
        sysm.set_nose_hoover(450.0, 30.0)
        out = sysm.md_ensemble_steps(pos, vel, mass, w.dt_fs, 12, rate)
        outs.append((pos.cpu().numpy(), out["ekin"].cpu().numpy(), sysm.get_nose_hoover()[1]))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert np.array_equal(outs[0][2], outs[1][2])
