"""gmnn_sum_energies_static: the allocation-free total-energy entry point (include/gmnn.h) against the existing path, the
total energy that gmnn_energy_forces returns for the same evaluation.  Its block partials sit in a file-scope device array
shared by all calls, so the check is made on two calls in a row with different sizes (the second reads fewer slots than the
first wrote).  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import workloads as wl
from parity_utils import E_TOTAL_RTOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gm():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (they must not pass on a fallback)")
    import paper_2505_22168_b200 as pkg

    return pkg


def _evaluate(gm, name):
    import torch

    w = wl.make_workload(name)
    sysm = gm.System(gm.Model(w.model), w.species)
    pos = torch.from_numpy(w.positions).cuda()
    sysm.build_neighbors(pos, w.cell9, w.pbc, w.model.r_cut, w.skin)
    e, e_atom, _ = sysm.energy_forces(pos)[:3]
    sysm.check()
    torch.cuda.synchronize()
    return float(e.cpu()[0]), e_atom


def test_static_sum_matches_energy_forces_twice_in_a_row(gm):
    import torch

    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    for name in ("config3_8192", "config3_1024", "config3_8192"):  # 32 blocks, then 4, then 32 again
        e_ref, e_atom = _evaluate(gm, name)
        before = gm.launch_count()
        gm.sum_energies_static(e_atom, out)
        torch.cuda.synchronize()
        assert gm.launch_count() - before == 2
        e = float(out.cpu()[0])
        ea = e_atom.cpu().numpy().astype(np.float64)
        bound = E_TOTAL_RTOL * np.abs(ea).sum()
        # the existing path sums the same fp32 E_i in the library's internal atom order, this one in the caller's order:
        # both are fp64 sums of identical terms, far inside the total-energy tolerance of the parity tests
        assert abs(e - e_ref) <= bound
        assert abs(e - ea.sum()) <= 1e-12 * np.abs(ea).sum()
        # a second call on the same input: identical bits (fixed reduction order, nothing kept from the call before)
        out2 = torch.zeros(1, dtype=torch.float64, device="cuda")
        gm.sum_energies_static(e_atom, out2)
        assert float(out2.cpu()[0]) == e


def test_static_sum_limits(gm):
    import torch

    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    x = torch.ones(1000, dtype=torch.float32, device="cuda")
    before = gm.launch_count()
    with pytest.raises(gm.GmnnError) as err:
        gm.sum_energies_static(x, out, n_atoms=gm.STATIC_SUM_MAX_ATOMS + 1)  # rejected before anything is read
    assert err.value.code == gm.GMNN_INVALID_ARG and "GMNN_STATIC_SUM_MAX_ATOMS" in str(err.value)
    assert gm.launch_count() == before
    gm.sum_energies_static(x, out)
    assert float(out.cpu()[0]) == 1000.0
    gm.sum_energies_static(x, out, n_atoms=0)
    assert float(out.cpu()[0]) == 0.0
