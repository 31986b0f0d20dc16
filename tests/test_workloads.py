"""The seeded generators: shapes, stoichiometry, determinism, minimum distances, calibration."""
import os

import numpy as np

import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


def test_splitmix64_reference_values():
    # splitmix64 with seed 0: first outputs of the published generator (Steele, Lea, Flood 2014;
    # the constants are the algorithm's own)
    z = wl.splitmix64(0, 3)
    assert [int(v) for v in z] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    u = wl.uniform01(123, 1000)
    assert u.min() >= 0 and u.max() < 1 and abs(u.mean() - 0.5) < 0.05
    n = wl.normal01(123, 20001)
    assert abs(n.mean()) < 0.03 and abs(n.std() - 1) < 0.03


def test_configs_shapes_and_stoichiometry():
    w = wl.tiny_box()
    assert w.n_atoms == 64 and np.bincount(w.species).tolist() == [32, 32]
    assert w.model.W[0].shape == (360, 512) and w.model.W[1].shape == (512, 512) and w.model.W[2].shape == (512, 1)
    assert abs(w.model.gamma - 1 / (2 * 0.75 ** 2)) < 1e-12
    w = wl.ionic_liquid_box()
    assert w.n_atoms == 1536 and np.bincount(w.species).tolist() == [704, 384, 128, 64, 256]
    assert abs(float(w.cell[0]) - 25.2947) < 1e-3  # 1.3 g/cm^3
    assert w.skin == 0.5 and w.dt_fs == 0.5 and w.n_steps == 1000 and w.model.r_cut == 6.0
    w = wl.li3po4_box(1024)
    assert np.bincount(w.species).tolist() == [384, 128, 512]
    assert abs(1024 / float(w.cell[0]) ** 3 - 0.09986) < 1e-4  # 2.4 g/cm^3
    w4 = wl.make_workload("config4")
    assert w4.n_atoms == 8192 and w4.model.n_heads == 32 and w4.model.W[2].shape == (512, 32)
    w3 = wl.make_workload("config3_8192")
    assert np.array_equal(w3.positions, w4.positions)  # "8192-atom box as above"
    assert all(np.array_equal(a, b) for a, b in zip(w3.model.W[:2], w4.model.W[:2]))


def test_determinism_and_wrapping():
    a, b = wl.ionic_liquid_box(), wl.ionic_liquid_box()
    assert np.array_equal(a.positions, b.positions) and np.array_equal(a.model.beta, b.model.beta)
    for w in (a, wl.tiny_box(), wl.li3po4_box(8192)):
        assert w.positions.dtype == np.float32
        assert np.all(w.positions >= 0) and np.all(w.positions < w.cell[None, :])
        p = (w.velocities.astype(np.float64) * w.masses[:, None]).sum(0)
        assert np.abs(p).max() < 1e-5


def _min_distance(pos, L):
    from scipy.spatial import cKDTree

    t = cKDTree(pos.astype(np.float64) % L.astype(np.float64), boxsize=L.astype(np.float64))
    d, _ = t.query(pos.astype(np.float64) % L.astype(np.float64), k=2)
    return d[:, 1].min()


def test_minimum_distances():
    w = wl.ionic_liquid_box()
    assert _min_distance(w.positions, w.cell) >= 0.9  # config 2: "0.9 A min distance"
    w = wl.li3po4_box(8192)
    assert _min_distance(w.positions, w.cell) >= 1.0
    w = wl.tiny_box()
    assert _min_distance(w.positions, w.cell) >= 2.125 - 0.6 * np.sqrt(3) - 1e-6


def test_force_scale_constants_follow_the_golden_file():
    rows = {}
    with open(os.path.join(HERE, "golden", "force_scale.txt")) as f:
        for line in f:
            if not line.startswith("#"):
                k, rms, fs, _ = line.split()
                rows[k] = float(fs)
    for fam in ("tiny", "ionic_liquid", "li3po4"):
        assert abs(wl.FORCE_SCALE[fam] / rows[fam] - 1) < 0.12, fam
