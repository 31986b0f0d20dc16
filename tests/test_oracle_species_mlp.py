"""Pins for O-5 with per-species weight sets (`n_weight_sets = n_species`; north_star: "the per-species atomic
MLP"; SURVEY.md 8(c-1) O-5 "the (W, b) used are those of set Z_i"; reading R11).  None of these
re-uses the oracle's per-species code path as its own reference: numpy matmuls with the set picked by hand,
the shared-NN path (pinned in test_oracle_descriptor.py), central finite differences."""
import dataclasses

import numpy as np

import workloads as wl


def _numpy_mlp(spec, G, wset):
    h = G
    for l in range(len(spec.hidden)):
        z = h @ spec.W[l][wset].astype(np.float64) + spec.b[l][wset].astype(np.float64)
        h = z / (1.0 + np.exp(-z))
    return h @ spec.W[-1][wset].astype(np.float64) + spec.b[-1][wset].astype(np.float64)


def test_first_set_of_the_generator_is_the_shared_model():
    a = wl.li3po4_box(64, hidden=(16, 16)).model
    b = wl.li3po4_box(64, hidden=(16, 16), n_weight_sets=3).model
    assert b.n_weight_sets == 3 and b.W[0].shape == (3, 360, 16) and b.b[1].shape == (3, 16)
    for l in range(3):
        assert np.array_equal(a.W[l], b.W[l][0]) and np.array_equal(a.b[l], b.b[l][0])
        assert not np.array_equal(b.W[l][0], b.W[l][1])


def test_per_atom_energy_is_the_numpy_mlp_of_the_atoms_own_set(orc):
    """E_i = sigma_Z NN_{Z_i}(G_i) + mu_Z with the weights of set Z_i, by numpy on the oracle's G_i."""
    w = wl.ionic_liquid_box(n_pairs=4, hidden=(24, 16), n_heads=3, n_weight_sets=5)  # 96 atoms, 5 species, 3 heads
    m = orc.Model(w.model)
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 6.0)
    res = orc.energy_forces(m, w.positions, w.species, w.cell, pairs, intermediates=True)
    for i in range(w.n_atoms):
        z = int(w.species[i])
        y = _numpy_mlp(w.model, res.G[i], z)
        e = float(w.model.scale[z]) * y + float(w.model.shift[z])
        assert np.allclose(res.e_heads[i], e, rtol=1e-12, atol=1e-12)
        other = _numpy_mlp(w.model, res.G[i], (z + 1) % 5)
        assert not np.allclose(y, other, rtol=1e-3)  # the sets do differ: a wrong set would show


def test_identical_sets_are_the_shared_network(orc):
    w1 = wl.li3po4_box(216, hidden=(32, 32))
    spec = w1.model
    rep = dataclasses.replace(spec, n_weight_sets=3, W=[np.repeat(x[None], 3, 0) for x in spec.W],
                              b=[np.repeat(x[None], 3, 0) for x in spec.b])
    pairs = orc.neighbors(w1.positions, w1.cell, w1.pbc, 6.0)
    a = orc.energy_forces(orc.Model(spec), w1.positions, w1.species, w1.cell, pairs)
    b = orc.energy_forces(orc.Model(rep), w1.positions, w1.species, w1.cell, pairs)
    assert np.array_equal(a.e_heads, b.e_heads) and np.array_equal(a.forces, b.forces)


def test_swapping_the_sets_of_two_species_swaps_which_network_they_see(orc):
    """With species-blind beta, sigma, mu the species enters only through the weight set: atoms of species 0
    under sets (A, B) have the energies that the shared network A gives them, atoms of species 1 those of B;
    under sets (B, A) the other way round."""
    w = wl.tiny_box(hidden=(16, 16), n_weight_sets=2)
    spec = w.model
    beta = np.repeat(np.repeat(spec.beta[:1, :1], 2, 0), 2, 1)
    blind = dataclasses.replace(spec, beta=beta, scale=np.full(2, 0.7, np.float32), shift=np.full(2, -0.2, np.float32))
    pairs = orc.neighbors(w.positions, w.cell, w.pbc, 5.0)

    def shared(k):
        return dataclasses.replace(blind, n_weight_sets=1, W=[x[k] for x in blind.W], b=[x[k] for x in blind.b])

    eA = orc.energy_forces(orc.Model(shared(0)), w.positions, w.species, w.cell, pairs, forces=False).e_atom
    eB = orc.energy_forces(orc.Model(shared(1)), w.positions, w.species, w.cell, pairs, forces=False).e_atom
    e_ab = orc.energy_forces(orc.Model(blind), w.positions, w.species, w.cell, pairs, forces=False).e_atom
    swapped = dataclasses.replace(blind, W=[x[::-1].copy() for x in blind.W], b=[x[::-1].copy() for x in blind.b])
    e_ba = orc.energy_forces(orc.Model(swapped), w.positions, w.species, w.cell, pairs, forces=False).e_atom
    is0 = w.species == 0
    assert np.allclose(e_ab[is0], eA[is0], rtol=0, atol=1e-13) and np.allclose(e_ab[~is0], eB[~is0], rtol=0, atol=1e-13)
    assert np.allclose(e_ba[is0], eB[is0], rtol=0, atol=1e-13) and np.allclose(e_ba[~is0], eA[~is0], rtol=0, atol=1e-13)
    assert np.abs(eA - eB).max() > 1e-3


def test_forces_equal_finite_differences_with_two_sets(orc):
    """The gradient pin on a 2-set box (config 1's image-loop box) and on a 3-set cell-list box."""
    for w, r_list, n in ((wl.tiny_box(hidden=(64, 64), n_weight_sets=2), 5.0, 64),
                         (wl.li3po4_box(216, hidden=(32, 32), n_weight_sets=3), 6.0, 216)):
        m = orc.Model(w.model)
        pos = w.positions.astype(np.float64)
        pairs = orc.neighbors(w.positions, w.cell, w.pbc, r_list)
        res = orc.energy_forces(m, pos, w.species, w.cell, pairs)
        scale = np.sqrt((res.forces ** 2).mean())
        rng = np.random.default_rng(5)
        for _ in range(12):
            i, a = int(rng.integers(n)), int(rng.integers(3))
            pp, pm = pos.copy(), pos.copy()
            pp[i, a] += 1e-5
            pm[i, a] -= 1e-5
            fd = -(orc.energy_forces(m, pp, w.species, w.cell, pairs, forces=False).energy
                   - orc.energy_forces(m, pm, w.species, w.cell, pairs, forces=False).energy) / 2e-5
            assert abs(fd - res.forces[i, a]) < 2e-7 * scale
        assert np.abs(res.forces.sum(0)).max() < 1e-12 * n * np.abs(res.forces).max()


def test_single_atom_calls_take_the_set(orc):
    """oracle.mlp_forward / mlp_backward with a set index: numpy forward, finite-difference backward."""
    spec = wl.li3po4_box(64, hidden=(16, 8), n_heads=2, n_weight_sets=3).model
    m = orc.Model(spec)
    rng = np.random.default_rng(3)
    G = rng.normal(size=360)
    for k in range(3):
        y, zs = orc.mlp_forward(m, G, k)
        assert np.allclose(y, _numpy_mlp(spec, G, k), rtol=1e-12, atol=1e-13)
        ybar = np.array([0.3, -1.1])
        gb = orc.mlp_backward(m, zs, ybar, 360, k)
        for f in (0, 17, 359):
            Gp, Gm = G.copy(), G.copy()
            Gp[f] += 1e-6
            Gm[f] -= 1e-6
            fd = (orc.mlp_forward(m, Gp, k)[0] - orc.mlp_forward(m, Gm, k)[0]) @ ybar / 2e-6
            assert abs(fd - gb[f]) < 1e-7 * max(1.0, abs(gb[f]))
