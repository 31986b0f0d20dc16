"""GPU parity of the tcgen05 tensor-core MLP (mlp_tc.cu) against the fp64 oracle.
mlp_precision = 1 (3xTF32) and 3 (3xFP16, the mode bench.py times) must meet the fp32 tolerances of
north_star (1e-5 per-atom energy, 1e-4 force measure).  mlp_precision = 2 (single-pass TF32, operands truncated by the tensor core) is
measured at 1e-2 .. 2.5e-2 on the force measure: it does NOT meet north_star's 2e-3 bound for a
reduced-precision variant, is not offered as one, and is only characterised here."""
import numpy as np
import pytest

import workloads as wl
from parity_utils import E_TOTAL_RTOL, F_TOL, energy_atom_error, force_error, r_list32, unique_from_full

F_TOL_TF32_MEASURED = 5e-2  # characterisation bound of the unclaimed single-pass mode

pytestmark = pytest.mark.gpu

P3X, PTF32, P3H = 1, 2, 3


@pytest.fixture(scope="module")
def gm():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (they must not pass on a fallback)")
    import paper_2505_22168_b200 as pkg

    return pkg


def _ref(orc, w, intermediates=False):
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    return orc.energy_forces(m, w.positions, w.species, w.cell, pairs, intermediates=intermediates)


def _system(gm, w, precision):
    import torch

    model = gm.Model(w.model, mlp_precision=precision)
    sysm = gm.System(model, w.species)
    pos = torch.from_numpy(w.positions).cuda()
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    return sysm, pos


def _run(sysm, pos):
    e, ea, f = sysm.energy_forces(pos)
    sysm.check()
    return float(e.cpu()[0]), ea.cpu().numpy().astype(np.float64), f.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("split_bk,flush_k", [(16, 32), (32, 64), (16, 128), (32, 128)])
@pytest.mark.parametrize("name", ["config1", "config2", "config3_1024", "config3_8192"])
def test_3xtf32_meets_fp32_tolerance(gm, orc, name, split_bk, flush_k):
    """Both stage shapes (64 B and 128 B swizzle) and several drain intervals of the hi.hi accumulator (128 = default)."""
    w = wl.make_workload(name)
    ref = _ref(orc, w)
    sysm, pos = _system(gm, w, P3X)
    sysm.set_int("tc_split_bk", split_bk)
    sysm.set_int("tc_flush_k", flush_k)
    try:
        e, ea, f = _run(sysm, pos)
    finally:
        sysm.set_int("tc_split_bk", 32)
        sysm.set_int("tc_flush_k", 128)
    print("3xTF32 %s bk %d flush %d: energy err %.3f x 1e-5, force err %.2e" % (
        name, split_bk, flush_k, energy_atom_error(ea, ref.e_atom), force_error(f, ref.forces)))
    assert energy_atom_error(ea, ref.e_atom) <= 1.0
    assert force_error(f, ref.forces) <= F_TOL
    assert abs(e - ref.energy) <= E_TOTAL_RTOL * np.abs(ref.e_atom).sum()


@pytest.mark.parametrize("h_bk,flush_k", [(64, 128), (64, 64), (32, 128), (32, 32)])
@pytest.mark.parametrize("name", ["config1", "config2", "config3_1024", "config3_8192"])
def test_3xf16_meets_fp32_tolerance(gm, orc, name, h_bk, flush_k):
    """3xFP16: both stage shapes (128 B and 64 B swizzle of the fp16 operand rows, 3 and 6 stages)."""
    w = wl.make_workload(name)
    ref = _ref(orc, w)
    sysm, pos = _system(gm, w, P3H)
    sysm.set_int("tc_h_bk", h_bk)
    sysm.set_int("tc_flush_k", flush_k)
    try:
        e, ea, f = _run(sysm, pos)
    finally:
        sysm.set_int("tc_h_bk", 64)
        sysm.set_int("tc_flush_k", 128)
    print("3xFP16 %s bk %d flush %d: energy err %.3f x 1e-5, force err %.2e" % (
        name, h_bk, flush_k, energy_atom_error(ea, ref.e_atom), force_error(f, ref.forces)))
    assert energy_atom_error(ea, ref.e_atom) <= 1.0
    assert force_error(f, ref.forces) <= F_TOL
    assert abs(e - ref.energy) <= E_TOTAL_RTOL * np.abs(ref.e_atom).sum()


@pytest.mark.parametrize("w0_scale,w1_scale", [(2.0 ** -12, 64.0), (16.0, 2.0 ** -9), (1e-3, 1e3)])
def test_3xf16_operand_scaling(gm, orc, w0_scale, w1_scale):
    """The fp16 split scales every GEMM operand by a power of two taken from its absolute maximum on the
    device: weights (and with them the activations and gradients) far outside the fp16 range keep the
    fp32 tolerance."""
    w = wl.li3po4_box(1000, hidden=(64, 48))
    w.model.W[0] = (w.model.W[0] * np.float32(w0_scale)).astype(np.float32)
    w.model.b[0] = (w.model.b[0] * np.float32(w0_scale)).astype(np.float32)
    w.model.W[1] = (w.model.W[1] * np.float32(w1_scale)).astype(np.float32)
    ref = _ref(orc, w)
    sysm, pos = _system(gm, w, P3H)
    e, ea, f = _run(sysm, pos)
    assert np.isfinite(f).all()
    assert energy_atom_error(ea, ref.e_atom) <= 1.0
    assert force_error(f, ref.forces) <= F_TOL
    # the fp32 SIMT path on the same weights: both within the tolerance of the oracle, hence of each other
    sysm.set_int("mlp_precision", 0)
    e0, ea0, f0 = _run(sysm, pos)
    assert force_error(f0, ref.forces) <= F_TOL and force_error(f, f0) <= 2 * F_TOL


@pytest.mark.parametrize("name", ["config1", "config3_1024", "config3_8192"])
def test_tf32_single_pass_characterised(gm, orc, name):
    w = wl.make_workload(name)
    ref = _ref(orc, w)
    sysm, pos = _system(gm, w, PTF32)
    e, ea, f = _run(sysm, pos)
    assert force_error(f, ref.forces) <= F_TOL_TF32_MEASURED
    assert np.abs(ea - ref.e_atom).max() <= 2e-2 * max(np.abs(ref.e_atom).max(), 1e-30)
    # and it really is a different arithmetic from the fp32 path (guards against a silent alias)
    sysm.set_int("mlp_precision", 0)
    _, _, f32 = _run(sysm, pos)
    assert np.abs(f32 - f).max() > 0


@pytest.mark.parametrize("precision", [P3X, PTF32, P3H])
@pytest.mark.parametrize("hidden", [(16, 16), (64, 48), (144, 272), (512, 512)])
def test_ragged_shapes(gm, orc, precision, hidden):
    """N = 1000 atoms (not a multiple of the 128-row tile), widths that are not multiples of the
    K stage (16 / 32) nor of the column tile; 272 > 256 forces two ragged column tiles."""
    w = wl.li3po4_box(1000, hidden=hidden)
    ref = _ref(orc, w, intermediates=True)
    sysm, pos = _system(gm, w, precision)
    e, ea, f = _run(sysm, pos)
    tol = F_TOL if precision != PTF32 else F_TOL_TF32_MEASURED
    assert force_error(f, ref.forces) <= tol
    perm = sysm.debug_read("perm")
    sig = w.model.scale[w.species][perm][:, None]
    dG_ref = ref.dG[perm] / sig
    dG = sysm.debug_read("dG")
    assert np.abs(dG - dG_ref).max() <= tol * np.abs(dG_ref).max()
    if precision != PTF32:
        assert energy_atom_error(ea, ref.e_atom) <= 1.0


@pytest.mark.parametrize("precision", [P3X, P3H])
def test_split_modes_match_fp32_simt_closely(gm, precision):
    """The fp32-accurate MLPs agree far inside the oracle tolerance, and each is bit-reproducible."""
    w = wl.li3po4_box(4096, hidden=(512, 512))
    sysm, pos = _system(gm, w, precision)
    e1, ea1, f1 = _run(sysm, pos)
    e1b, ea1b, f1b = _run(sysm, pos)
    assert e1 == e1b and np.array_equal(ea1, ea1b) and np.array_equal(f1, f1b)
    sysm.set_int("mlp_precision", 0)
    e0, ea0, f0 = _run(sysm, pos)
    assert force_error(f1, f0) <= 5e-5
    assert np.abs(ea1 - ea0).max() <= 1e-5 * np.abs(ea0).mean()  # each is within 1e-5 of the oracle (tests above)


@pytest.mark.parametrize("precision", [P3X, P3H])
def test_ensemble_heads_with_tc(gm, orc, precision):
    """Shallow ensemble (config 4 shape, smaller box): M backward passes through the TC MLP."""
    w = wl.li3po4_box(1024, n_heads=8)
    m = orc.Model(w.model)
    pairs = orc.auto_neighbors(w.positions, w.cell, w.pbc, r_list32(w.model.r_cut, w.skin))
    ref = orc.ensemble(m, w.positions, w.species, w.cell, pairs)
    sysm, pos = _system(gm, w, precision)
    e_mean, e_var, f_mean, f_var = (t.cpu().numpy().astype(np.float64) for t in sysm.ensemble_energy_forces(pos))
    assert energy_atom_error(e_mean, ref.e_mean) <= 1.0
    assert force_error(f_mean, ref.f_mean) <= F_TOL
    assert np.abs(f_var - ref.f_var).max() <= 2e-4 * ref.f_var.max()


@pytest.mark.parametrize("name", ["config2", "config3_8192", "ragged"])
def test_cta_pair_and_single_cta_kernels(gm, orc, name):
    """The 3xTF32 GEMM runs on CTA pairs (cta_group::2, default) or single CTAs: both meet the fp32
    tolerances; 'ragged' has an odd number of 128-atom tiles (a pair with an empty second tile)."""
    w = wl.li3po4_box(1000 + 128 * 2, hidden=(144, 272)) if name == "ragged" else wl.make_workload(name)
    ref = _ref(orc, w)
    sysm, pos = _system(gm, w, P3X)
    out = {}
    try:
        for pair in (1, 0):
            sysm.set_int("tc_pair", pair)
            e, ea, f = _run(sysm, pos)
            assert energy_atom_error(ea, ref.e_atom) <= 1.0, pair
            assert force_error(f, ref.forces) <= F_TOL, pair
            out[pair] = f
    finally:
        sysm.set_int("tc_pair", 1)
    assert force_error(out[0], out[1]) <= 5e-5


def test_contract_backward_odd_tile_count(gm, orc):
    """k_contract_backward (one 128-atom tile per block, orbit-representative body: a fifth of the adjoint's
    terms run five times with the channels shifted) on an odd tile count with a ragged last tile: the
    adjoints A = dE/dPsi against the oracle's, mapped to the symmetry-unique storage."""
    w = wl.li3po4_box(128 * 5 + 24, hidden=(32, 32))
    ref = _ref(orc, w, intermediates=True)
    sysm, pos = _system(gm, w, P3X)
    e, ea, f = _run(sysm, pos)
    assert force_error(f, ref.forces) <= F_TOL
    A = sysm.debug_read("A")
    perm = sysm.debug_read("perm")
    a_ref = unique_from_full(ref.Q, summed=True)[perm]  # adjoints with respect to the unique moments
    assert np.abs(A - a_ref).max() <= 1e-4 * np.abs(a_ref).max()
