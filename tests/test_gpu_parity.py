"""GPU parity: the CUDA path through the C ABI against the fp64 oracle on the same seeded inputs.
Neighbour lists bit-exact as sorted (i, j, n) sets; fp32 path: per-atom energies within 1e-5
relative, max |dF| / RMS F <= 1e-4 (north_star)."""
import numpy as np
import pytest

import workloads as wl
from parity_utils import (E_TOTAL_RTOL, F_TOL, energy_atom_error, force_error, r_list32, unique_from_full)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (they must not pass on a fallback)")
    import paper_2505_22168_b200 as pkg

    return pkg


def _oracle_ref(orc, w, intermediates=False):
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    return pairs, orc.energy_forces(m, w.positions, w.species, w.cell, pairs, intermediates=intermediates)


def _gpu_system(gm, w, **model_kw):
    import torch

    model = gm.Model(w.model, **model_kw)
    sysm = gm.System(model, w.species)
    pos = torch.from_numpy(w.positions).cuda()
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    return model, sysm, pos


# ------------------------------------------------------------------ neighbour sets: bit exact
@pytest.mark.parametrize("name", ["tiny", "ionic_liquid", "li1024", "li8192", "li8192_wide_skin", "cluster", "mixed_pbc", "ragged"])
def test_neighbor_sets_bit_exact(gm, orc, name):
    if name == "tiny":
        w = wl.tiny_box(hidden=(16, 16))  # image loop, duplicate-by-image pairs
    elif name == "ionic_liquid":
        w = wl.ionic_liquid_box(hidden=(16, 16))  # skin 0.5: exactly 3 cells per axis at r_list 6.5
    elif name == "li1024":
        w = wl.li3po4_box(1024, hidden=(16, 16))  # exactly 3 cells per axis
    elif name == "li8192":
        w = wl.li3po4_box(8192, hidden=(16, 16), skin=1.0)
    elif name == "li8192_wide_skin":
        w = wl.li3po4_box(8192, hidden=(16, 16), skin=4.0)  # ~330 shell entries per row: more than the build kernel stages
    elif name == "cluster":
        w = wl.cluster(24, 2)  # no periodic axis
    elif name == "mixed_pbc":
        w = wl.li3po4_box(1024, hidden=(16, 16))
        w.pbc = (1, 0, 1)
    else:
        w = wl.li3po4_box(1000, hidden=(16, 16))  # N not a multiple of any tile: ragged tails
    _, sysm, _ = _gpu_system(gm, w)
    got = sysm.get_neighbors()
    ref = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin)).as_set_array()
    assert got.shape == ref.shape and np.array_equal(got, ref)
    if name == "tiny":
        assert sysm.get_int("small_box") == 1
        ij = got[:, 0].astype(np.int64) * 64 + got[:, 1]
        assert np.unique(ij, return_counts=True)[1].max() >= 2


# ------------------------------------------------------------------ stage-by-stage intermediates
@pytest.mark.parametrize("name", ["tiny", "li1000"])
def test_stage_intermediates(gm, orc, name):
    w = wl.tiny_box() if name == "tiny" else wl.li3po4_box(1000)
    _, ref = _oracle_ref(orc, w, intermediates=True)
    _, sysm, pos = _gpu_system(gm, w)
    sysm.energy_forces(pos)
    perm = sysm.debug_read("perm")
    assert sorted(perm.tolist()) == list(range(w.n_atoms))
    psi_ref = unique_from_full(ref.P, summed=False)[perm]
    psi = sysm.debug_read("psi")
    assert np.abs(psi - psi_ref).max() <= 2e-6 * np.abs(psi_ref).max()
    # trace identities hold on the GPU tensors too: xx + yy + zz = P0; xxa + yya + zza = P1_a
    assert np.abs(psi[:, :, 4] + psi[:, :, 7] + psi[:, :, 9] - psi[:, :, 0]).max() <= 1e-5 * np.abs(psi).max()
    G_ref = ref.G[perm]
    G = sysm.debug_read("G")
    assert np.abs(G - G_ref).max() <= 5e-6 * np.abs(G_ref).max()
    sig = w.model.scale[w.species][perm][:, None]
    dG_ref = ref.dG[perm] / sig  # the CUDA path applies sigma_Z after the MLP backward
    dG = sysm.debug_read("dG")
    assert np.abs(dG - dG_ref).max() <= 1e-4 * np.abs(dG_ref).max()
    A_ref = unique_from_full(ref.Q, summed=True)[perm]
    A = sysm.debug_read("A")
    assert np.abs(A - A_ref).max() <= 1e-4 * np.abs(A_ref).max()


# ------------------------------------------------------------------ end-to-end energies and forces
def _check_energy_forces(gm, orc, w, **kw):
    _, ref = _oracle_ref(orc, w)
    _, sysm, pos = _gpu_system(gm, w, **kw)
    e, ea, f = sysm.energy_forces(pos)
    sysm.check()
    ea, f, e = ea.cpu().numpy().astype(np.float64), f.cpu().numpy().astype(np.float64), float(e.cpu()[0])
    assert energy_atom_error(ea, ref.e_atom) <= 1.0
    assert force_error(f, ref.forces) <= F_TOL
    assert abs(e - ref.energy) <= E_TOTAL_RTOL * np.abs(ref.e_atom).sum()
    assert np.abs(f.sum(0)).max() <= 1e-4 * np.abs(f).max() * np.sqrt(w.n_atoms)
    return sysm, pos, ref


def test_config1_tiny(gm, orc):
    _check_energy_forces(gm, orc, wl.make_workload("config1"))


def test_config2_ionic_liquid_initial_state(gm, orc):
    _check_energy_forces(gm, orc, wl.make_workload("config2"))  # list includes the 0.5 skin shell


@pytest.mark.parametrize("n", [1024, 8192])
def test_config3_li3po4(gm, orc, n):
    _check_energy_forces(gm, orc, wl.make_workload("config3_%d" % n))


def test_ragged_sizes_and_lane_groupings(gm, orc):
    """N = 1000 is a multiple of no tile; every lanes-per-atom grouping gives the same physics."""
    w = wl.li3po4_box(1000, hidden=(64, 48))
    _, ref = _oracle_ref(orc, w)
    _, sysm, pos = _gpu_system(gm, w)
    for lpa in (1, 2, 4, 8, 16, 32):
        sysm.set_int("lanes_per_atom", lpa)
        e, ea, f = sysm.energy_forces(pos)
        assert energy_atom_error(ea.cpu().numpy().astype(np.float64), ref.e_atom) <= 1.0, lpa
        assert force_error(f.cpu().numpy().astype(np.float64), ref.forces) <= F_TOL, lpa


def test_skin_shell_contributes_nothing(gm, orc):
    import torch

    w0 = wl.li3po4_box(1024, hidden=(32, 32), skin=0.0)
    w1 = wl.li3po4_box(1024, hidden=(32, 32), skin=1.0)
    out = []
    for w in (w0, w1):
        _, sysm, pos = _gpu_system(gm, w)
        e, ea, f = sysm.energy_forces(pos)
        out.append((float(e.cpu()[0]), f.cpu().numpy()))
    assert abs(out[0][0] - out[1][0]) <= 1e-6 * abs(out[0][0])
    assert np.abs(out[0][1] - out[1][1]).max() <= 1e-5 * np.abs(out[0][1]).max()


def test_bitwise_determinism(gm):
    """Segment-ordered force sums, fixed-order fp64 energy: two evaluations (and two independent
    builds) are bit-identical (SURVEY.md section 4 tier 5)."""
    w = wl.li3po4_box(8192, hidden=(64, 64))
    runs = []
    for _ in range(2):
        _, sysm, pos = _gpu_system(gm, w)
        for _ in range(2):
            e, ea, f = sysm.energy_forces(pos)
            runs.append((e.cpu().numpy().copy(), ea.cpu().numpy().copy(), f.cpu().numpy().copy()))
    for r in runs[1:]:
        assert np.array_equal(r[0], runs[0][0]) and np.array_equal(r[1], runs[0][1]) and np.array_equal(r[2], runs[0][2])


def test_host_entry_matches_device_entry(gm):
    import torch

    w = wl.li3po4_box(1024, hidden=(64, 64))
    _, sysm, pos = _gpu_system(gm, w)
    e, ea, f = sysm.energy_forces(pos)
    hp = torch.from_numpy(w.positions).pin_memory()
    hf = torch.empty(w.n_atoms, 3).pin_memory()
    he = torch.empty(w.n_atoms).pin_memory()
    e_host = sysm.energy_forces_host(hp.numpy(), hf.numpy(), he.numpy())
    assert e_host == float(e.cpu()[0])
    assert np.array_equal(hf.numpy(), f.cpu().numpy()) and np.array_equal(he.numpy(), ea.cpu().numpy())


# ------------------------------------------------------------------ errors, not fallbacks
def test_error_codes(gm):
    import torch

    w = wl.li3po4_box(1024, hidden=(16, 16), skin=0.5)
    model = gm.Model(w.model)
    sysm = gm.System(model, w.species)
    pos = torch.from_numpy(w.positions).cuda()
    with pytest.raises(gm.GmnnError) as e:
        sysm.energy_forces(pos)  # no list yet
    assert e.value.code == gm.GMNN_INVALID_ARG
    with pytest.raises(gm.GmnnError) as e:
        sysm.build_neighbors(pos, w.cell9, w.pbc, 5.0, 0.5)  # r_cut differs from the model's
    assert e.value.code == gm.GMNN_INVALID_ARG
    flat = w.cell9.copy()
    flat[3:6] = flat[0:3]  # b = a: no volume (sheared cells themselves are supported, tests/test_gpu_triclinic.py)
    with pytest.raises(gm.GmnnError) as e:
        sysm.build_neighbors(pos, flat, w.pbc, 6.0, 0.5)
    assert e.value.code == gm.GMNN_INVALID_ARG
    # a failed build leaves no list behind (never an old list beside a new geometry)
    with pytest.raises(gm.GmnnError) as e:
        sysm.energy_forces(pos)
    assert e.value.code == gm.GMNN_INVALID_ARG
    bad = pos.clone()
    bad[5, 0] = -0.25
    with pytest.raises(gm.GmnnError) as e:
        sysm.build_neighbors(bad, w.cell9, w.pbc, 6.0, 0.5)
    assert e.value.code == gm.GMNN_OUT_OF_BOX
    sysm.build_neighbors(pos, w.cell9, w.pbc, 6.0, 0.5)
    moved = pos.clone()
    moved[7, 1] += 0.3  # > skin / 2
    sysm.energy_forces(moved)
    with pytest.raises(gm.GmnnError) as e:
        sysm.check()
    assert e.value.code == gm.GMNN_STALE_NEIGHBORS
    sysm.energy_forces(pos)
    sysm.check()  # cleared
    # capacity too small: the library regrows and retries
    sysm.set_int("capacity", 32)
    sysm.build_neighbors(pos, w.cell9, w.pbc, 6.0, 0.5)
    assert sysm.get_int("capacity") >= 100
    with pytest.raises(gm.GmnnError) as e:
        gm.Model(w.model, mlp_precision=7)
    assert e.value.code == gm.GMNN_INVALID_ARG


def test_single_atom_and_isolated_atoms(gm, orc):
    """Degenerate inputs: one atom; atoms with no neighbour inside r_cut (G = 0, F = 0)."""
    import torch

    spec = wl.make_model(3, 2, r_cut=6.0, hidden=(16, 16))
    pos = np.array([[5.0, 5, 5], [25.0, 25, 25], [45.0, 45, 45]], np.float32)
    species = np.array([0, 1, 1], np.int32)
    cell9 = np.diag([60.0, 60, 60]).astype(np.float32).reshape(9)
    model = gm.Model(spec)
    for n in (1, 3):
        sysm = gm.System(model, species[:n])
        p = torch.from_numpy(pos[:n].copy()).cuda()
        sysm.build_neighbors(p, cell9, (1, 1, 1), 6.0, 0.0)
        assert sysm.get_neighbors().shape == (0, 5)
        e, ea, f = sysm.energy_forces(p)
        m = orc.Model(spec)
        ref = orc.energy_forces(m, pos[:n], species[:n], [60, 60, 60], orc.neighbors(pos[:n], [60, 60, 60], (1, 1, 1), 6.0))
        assert np.all(f.cpu().numpy() == 0)
        assert np.allclose(ea.cpu().numpy(), ref.e_atom, rtol=1e-5)


# ------------------------------------------------------------------ pair-buffer force reduction
@pytest.mark.parametrize("name", ["config1", "config2", "config3_1024", "config3_8192", "cluster", "ragged", "wide_skin"])
def test_pair_buffer_force_mode(gm, orc, name):
    """GMNN_FORCE_PAIRBUF: g_ij evaluated once per directed pair and delivered through the
    reverse-pair index; same tolerances as the gather form, bit-reproducible, and the two forms
    agree to round-off.  config1 has duplicate-by-image pairs and self images, cluster no PBC."""
    if name == "cluster":
        w = wl.cluster(24, 2)
    elif name == "ragged":
        w = wl.li3po4_box(1000, hidden=(64, 48), skin=0.7)
    elif name == "wide_skin":
        w = wl.li3po4_box(8192, hidden=(32, 32), skin=4.0)  # shell part of a row larger than the build kernel stages
    else:
        w = wl.make_workload(name)
    sysm, pos, ref = _check_energy_forces(gm, orc, w, force_mode=gm.GMNN_FORCE_PAIRBUF)
    e1, ea1, f1 = sysm.energy_forces(pos)
    e2, ea2, f2 = sysm.energy_forces(pos)
    assert np.array_equal(f1.cpu().numpy(), f2.cpu().numpy())
    _, sysg, _ = _gpu_system(gm, w)
    _, _, fg = sysg.energy_forces(pos)
    assert force_error(f1.cpu().numpy().astype(np.float64), fg.cpu().numpy().astype(np.float64)) <= 2e-5
    # switching the mode on a built system asks for a rebuild instead of using a stale index
    sysg.set_int("force_mode", gm.GMNN_FORCE_PAIRBUF)
    with pytest.raises(gm.GmnnError):
        sysg.energy_forces(pos)
    sysg.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    _, _, fp = sysg.energy_forces(pos)
    assert np.array_equal(fp.cpu().numpy(), f1.cpu().numpy())


@pytest.mark.parametrize("mlp_precision", [0, 3])
def test_energy_forces_graph_replay_is_bitwise_the_eager_call(gm, mlp_precision):
    """gmnn_energy_forces replays its inner launches as a CUDA graph from the third call of an unchanged configuration
    (knob "ef_graph"): same bits as the eager call, also at new positions, after a knob change, after a new list build
    and after MD steps that rebuilt the list inside their loop."""
    import torch

    w = wl.li3po4_box(2000, hidden=(64, 64))
    _, sysm, pos = _gpu_system(gm, w, mlp_precision=mlp_precision, force_mode=1)

    def call(p):
        e, ea, f = sysm.energy_forces(p)[:3]
        return float(e.cpu()[0]), ea.cpu().numpy().copy(), f.cpu().numpy().copy()

    def both(p, n=4):
        sysm.set_int("ef_graph", 0)
        ref = call(p)
        sysm.set_int("ef_graph", 1)
        n0 = gm.launch_count()
        outs = [call(p) for _ in range(n)]  # eager, capture, replay, replay
        per_call = (gm.launch_count() - n0) / n
        for o in outs:
            assert o[0] == ref[0] and np.array_equal(o[1], ref[1]) and np.array_equal(o[2], ref[2])
        return per_call

    launches = both(pos)
    assert launches > 10  # replayed launches are counted
    pos2 = pos + 0.02 * torch.randn_like(pos)  # inside the skin: same list, new positions through the same graph
    both(pos2, n=1)
    sysm.set_int("lanes_per_atom", 8)
    both(pos2)
    sysm.set_int("lanes_per_atom", 0)
    sysm.build_neighbors(pos2, w.cell9, w.pbc, w.model.r_cut, w.skin)
    both(pos2)
    vel = 0.05 * torch.randn_like(pos2)
    mass = torch.full((pos2.shape[0],), 10.0, device="cuda")
    p3 = pos2.clone()
    _, _, nreb = sysm.md_verlet_steps(p3, vel, mass, 1.0, 30)
    sysm.check()
    both(p3)
    sysm.check()


@pytest.mark.parametrize("n_weight_sets", [1, 3])
@pytest.mark.parametrize("mlp_precision", [0, 3])
def test_kept_state_survives_other_calls(gm, mlp_precision, n_weight_sets):
    """What gmnn_energy_forces keeps between calls (its CUDA graph, the backward seed of the constant mean-head weights)
    must not leak into or out of the calls that change the head weights or the buffers: an ensemble pass, a UDD-biased
    evaluation, a switch of the MLP mode.  Reference: a fresh system with the kept state off, same positions."""
    import torch

    w = wl.li3po4_box(1600, hidden=(64, 64), n_heads=8, n_weight_sets=n_weight_sets)
    _, sysm, pos = _gpu_system(gm, w, mlp_precision=mlp_precision, force_mode=1)
    _, ref_sys, _ = _gpu_system(gm, w, mlp_precision=mlp_precision, force_mode=1)
    ref_sys.set_int("ef_graph", 0)

    def out(system):
        e, ea, f = system.energy_forces(pos)[:3]
        return float(e.cpu()[0]), ea.cpu().numpy().copy(), f.cpu().numpy().copy()

    def same(a, b):
        return a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])

    ref = out(ref_sys)
    for _ in range(3):
        assert same(out(sysm), ref)  # eager, capture, replay
    ens = [t.cpu().numpy().copy() for t in sysm.ensemble_energy_forces(pos)]
    ens_ref = [t.cpu().numpy().copy() for t in ref_sys.ensemble_energy_forces(pos)]
    assert all(np.array_equal(a, b) for a, b in zip(ens, ens_ref))
    for _ in range(2):
        assert same(out(sysm), ref)  # after the ensemble pass (one-hot or stacked head weights) the mean-head seed is rebuilt
    ref_sys.set_udd_bias(0.5, 1.0)
    out(ref_sys)
    _, var_e = ref_sys.get_udd_bias()
    B = float(np.sqrt(var_e / (8 * pos.shape[0])))  # sigma_E^2 / (M N B^2) = 1: a bias force of the size of the forces
    sysm.set_udd_bias(0.5, B)
    ref_sys.set_udd_bias(0.5, B)
    biased_ref = out(ref_sys)
    assert not np.array_equal(biased_ref[2], ref[2])
    for _ in range(3):
        assert same(out(sysm), biased_ref)
    sysm.set_udd_bias(0.0, B)
    ref_sys.set_udd_bias(0.0, B)
    for _ in range(3):
        assert same(out(sysm), ref)
    other = 0 if mlp_precision == 3 else 3
    for system in (sysm, ref_sys):
        system.set_int("mlp_precision", other)
    ref_other = out(ref_sys)
    for _ in range(3):
        assert same(out(sysm), ref_other)
    for system in (sysm, ref_sys):
        system.set_int("mlp_precision", mlp_precision)
    for _ in range(3):
        assert same(out(sysm), ref)
    sysm.check()
