"""GPU parity for temperature schedules of the thermostats (reading R32) against
oracle O-19: Langevin and Nose-Hoover-chain trajectories under a piecewise-linear T(step), graph replay, removal."""
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


SCHEDULE = ([2, 6, 10], [300.0, 600.0, 300.0])  # one period of the paper's 300 <-> 600 K oscillation, in steps


@pytest.mark.parametrize("thermostat", ["langevin", "nose_hoover"])
@pytest.mark.parametrize("name", ["ionic384", "li1024"])
def test_scheduled_trajectory_matches_oracle(gm, orc, name, thermostat):
    w = wl.ionic_liquid_box(n_pairs=16, hidden=(64, 64)) if name == "ionic384" else \
        wl.li3po4_box(1024, hidden=(64, 64), skin=0.5)
    n = 12
    om = orc.Model(w.model)
    common = (om, w.positions, w.velocities, w.masses, w.species, w.cell, w.pbc, w.dt_fs, n)
    sysm, pos, vel, mass = _system(gm, w)
    if thermostat == "langevin":
        x, v, ep, ek = orc.nvt_langevin(*common, 300.0, 0.5, 424242, 0, schedule=SCHEDULE)
        flat = orc.nvt_langevin(*common, 300.0, 0.5, 424242, 0)
        sysm.set_langevin(300.0, 0.5, 424242, 0)
    else:
        x, v, ep, ek, _ = orc.nvt_nose_hoover(*common, 300.0, 10.0, schedule=SCHEDULE)
        flat = orc.nvt_nose_hoover(*common, 300.0, 10.0)
        sysm.set_nose_hoover(300.0, 10.0, 3, 2, 3)
    sysm.set_temperature_schedule(*SCHEDULE)
    epot, ekin, _ = sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, n)
    L = w.cell.astype(np.float64)
    d = pos.cpu().numpy().astype(np.float64) - x
    d -= np.round(d / L) * L
    assert np.abs(d).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - v).max() <= 1e-5
    assert np.abs(epot.cpu().numpy() - ep).max() <= 1e-5 * np.abs(ep).max() + 1e-4
    assert np.abs(ekin.cpu().numpy() - ek).max() <= 1e-4 * np.abs(ek).max()
    assert np.abs(v - flat[1]).max() > 20 * 1e-5  # the profile did act: the constant-target run ends elsewhere


def test_schedule_replay_continuation_and_removal(gm):
    """Graph replay = eager loop bit for bit under a schedule; two calls = one (the step counter lives on the device);
    removing the schedule gives back the constant-target trajectory."""
    w = wl.li3po4_box(1024, hidden=(64, 64), skin=0.5)
    runs = []
    for graph, split in ((1, False), (0, False), (1, True)):
        sysm, pos, vel, mass = _system(gm, w)
        sysm.set_int("md_graph", graph)
        sysm.set_langevin(300.0, 0.05, 5)
        sysm.set_temperature_schedule([0, 16], [300.0, 900.0])
        if split:
            sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 7)
            sysm.set_int("md_continue", 1)
            sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 9)
        else:
            sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 16)
        runs.append((pos.cpu().numpy(), vel.cpu().numpy()))
    for a, b in zip(runs[0], runs[1]):
        assert np.array_equal(a, b)
    for a, b in zip(runs[0], runs[2]):
        assert np.array_equal(a, b)
    out = []
    for remove in (False, True):
        sysm, pos, vel, mass = _system(gm, w)
        sysm.set_nose_hoover(400.0, 20.0, 3, 2, 3)
        if remove:
            sysm.set_temperature_schedule([0, 8], [400.0, 1200.0])
            sysm.set_temperature_schedule()
        sysm.md_verlet_steps(pos, vel, mass, w.dt_fs, 8)
        out.append(vel.cpu().numpy())
    assert np.array_equal(out[0], out[1])
    with pytest.raises(gm.GmnnError):
        sysm.set_temperature_schedule([5, 5], [300.0, 400.0])  # steps must ascend strictly
