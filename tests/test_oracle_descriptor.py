"""Pins for O-2..O-5 (radial, moments, invariants, MLP): closed forms, identities, invariances.
SURVEY.md 8(c-3).  None of these re-types the oracle's own loops: they are special values,
textbook identities, numpy library routines, or symmetry statements."""
import numpy as np
import pytest

import workloads as wl

O1, O2, O3 = 1, 4, 13


def _model(orc, w):
    return orc.Model(w.model)


def _one_hot_beta_model(orc, n_species=1, k=3, r_cut=5.0):
    spec = wl.make_model(7, n_species, r_cut=r_cut, hidden=(8,))
    spec.beta[:] = 0.0
    spec.beta[..., :, k] = 1.0
    return spec, orc.Model(spec)


# ---------------------------------------------------------------- radial (O-2)
def test_radial_special_values(orc):
    spec, m = _one_hot_beta_model(orc, k=3)
    delta = (5.0 - 0.5) / 6
    mu3 = 0.5 + 3 * delta
    # at the Gaussian centre Phi = 1, so R = f_c(mu); f_c(r_cut/2) = 1/2
    R, _ = orc.radial(m, 0, 0, mu3)
    assert np.allclose(R, 0.5 * (1 + np.cos(np.pi * mu3 / 5.0)), rtol=0, atol=1e-15)
    spec2, m2 = _one_hot_beta_model(orc, k=0)
    spec2.r_min = 2.5  # centre 0 sits at r_cut / 2
    m2 = orc.Model(spec2)
    R, _ = orc.radial(m2, 0, 0, 2.5)
    assert np.allclose(R, 0.5, atol=1e-15)
    # f_c(0) = 1: R(0) = Phi_k(0) = exp(-gamma mu^2); gamma = 1/(2 Delta^2) (reading R2)
    R, dR = orc.radial(m, 0, 0, 0.0)
    assert np.allclose(R, np.exp(-mu3 ** 2 / (2 * delta ** 2)), rtol=1e-14)
    # at and beyond the cutoff everything vanishes, and R' -> 0 as r -> r_cut (C1)
    for r in (5.0, 5.5):
        R, dR = orc.radial(m, 0, 0, r)
        assert np.all(R == 0) and np.all(dR == 0)
    R, dR = orc.radial(m, 0, 0, 5.0 - 1e-7)
    assert np.all(np.abs(R) < 1e-13) and np.all(np.abs(dR) < 1e-6)


def test_radial_derivative_is_fd_of_radial(orc):
    w = wl.ionic_liquid_box(n_pairs=2, hidden=(8,))
    m = _model(orc, w)
    h = 1e-6
    for (zi, zj, r) in [(0, 1, 0.9), (4, 2, 2.345), (1, 1, 4.0), (3, 0, 5.9)]:
        _, dR = orc.radial(m, zi, zj, r)
        Rp, _ = orc.radial(m, zi, zj, r + h)
        Rm, _ = orc.radial(m, zi, zj, r - h)
        assert np.allclose(dR, (Rp - Rm) / (2 * h), rtol=1e-7, atol=1e-8)


def test_beta_is_ordered_centre_species_first(orc):
    w = wl.ionic_liquid_box(n_pairs=2, hidden=(8,))
    m = _model(orc, w)
    Rab, _ = orc.radial(m, 0, 1, 2.0)
    Rba, _ = orc.radial(m, 1, 0, 2.0)
    assert not np.allclose(Rab, Rba)  # general ordered table (reading R5)
    spec = w.model
    spec.beta[1, 0] = spec.beta[0, 1]
    Rba2, _ = orc.radial(orc.Model(spec), 1, 0, 2.0)
    assert np.allclose(Rab, Rba2)


# ---------------------------------------------------------------- moments (O-3)
def test_moment_trace_identities_and_symmetry(orc):
    w = wl.tiny_box(hidden=(8,))
    m = _model(orc, w)
    p = orc.neighbors(w.positions, w.cell, w.pbc, 5.0)
    P = orc.energy_forces(m, w.positions, w.species, w.cell, p, forces=False, intermediates=True).P
    P0 = P[:, :, 0]
    P1 = P[:, :, O1:O1 + 3]
    P2 = P[:, :, O2:O2 + 9].reshape(-1, 5, 3, 3)
    P3 = P[:, :, O3:O3 + 27].reshape(-1, 5, 3, 3, 3)
    assert np.abs(P0).max() > 1.0
    # u is a unit vector: sum_a P2_aa = P0, sum_b P3_abb = P1_a
    assert np.allclose(np.einsum("isaa->is", P2), P0, atol=1e-12)
    assert np.allclose(np.einsum("isabb->isa", P3), P1, atol=1e-12)
    assert np.allclose(P2, P2.transpose(0, 1, 3, 2), atol=1e-14)
    for perm in [(0, 1, 3, 2, 4), (0, 1, 2, 4, 3), (0, 1, 4, 3, 2), (0, 1, 3, 4, 2)]:
        assert np.allclose(P3, P3.transpose(perm), atol=1e-14)


def test_moments_of_a_single_neighbour(orc):
    """One neighbour at distance r along a known direction: Psi_L = R_s u^{(x)L} exactly."""
    spec, m = _one_hot_beta_model(orc, k=2)
    u = np.array([2.0, -1.0, 2.0]) / 3.0
    r = 2.2
    pos = np.array([[10.0, 10.0, 10.0], 10.0 + r * u])
    p = orc.neighbors(pos, [30, 30, 30], (0, 0, 0), 5.0)
    assert len(p) == 2
    res = orc.energy_forces(m, pos, [0, 0], [30, 30, 30], p, forces=False, intermediates=True)
    R, _ = orc.radial(m, 0, 0, r)
    P = res.P[0]
    assert np.allclose(P[:, 0], R, rtol=1e-13)
    assert np.allclose(P[:, O1:O1 + 3], R[:, None] * u, rtol=1e-12)
    assert np.allclose(P[:, O2:O2 + 9], R[:, None] * np.einsum("a,b->ab", u, u).reshape(-1), rtol=1e-12)
    assert np.allclose(P[:, O3:O3 + 27], R[:, None] * np.einsum("a,b,c->abc", u, u, u).reshape(-1), rtol=1e-12)
    # the other atom sees -u
    assert np.allclose(res.P[1][:, O1:O1 + 3], -R[:, None] * u, rtol=1e-12)


# ---------------------------------------------------------------- invariants (O-4)
def test_feature_count(orc):
    assert orc.n_features(5) == 360  # 5+15+15+15+35+75+75+125
    assert orc.n_features(1) == 1 + 3 + 1 + 2 + 1
    assert wl.inputs.n_features(5) == 360 and wl.inputs.n_features(3) == orc.n_features(3)


def _blocks_by_einsum(P):
    """Eq. 3 written with numpy.einsum on the full tensors, for ALL channel tuples (no uniqueness)."""
    n = P.shape[0]
    P0 = P[:, 0]
    P1 = P[:, O1:O1 + 3]
    P2 = P[:, O2:O2 + 9].reshape(n, 3, 3)
    P3 = P[:, O3:O3 + 27].reshape(n, 3, 3, 3)
    return dict(
        b0=P0,
        b1=np.einsum("sa,ta->st", P1, P1),  # first printed line of Eq. 3
        b2=np.einsum("sab,tab->st", P2, P2),
        b3=np.einsum("sabc,tabc->st", P3, P3),
        b4=np.einsum("sab,tbc,vca->stv", P2, P2, P2),
        b5=np.einsum("sa,tb,vab->stv", P1, P1, P2),
        b6=np.einsum("sabc,tabd,vcd->stv", P3, P3, P2),
        b7=np.einsum("sa,tabc,vbc->stv", P1, P3, P2),  # last printed line of Eq. 3
    )


def test_invariants_match_einsum_of_eq3_and_block_order(orc):
    rng = np.random.default_rng(5)
    n = 5
    P = rng.normal(size=(n, 40))
    # make P2, P3 symmetric as real moments are
    P2 = P[:, O2:O2 + 9].reshape(n, 3, 3)
    P[:, O2:O2 + 9] = (0.5 * (P2 + P2.transpose(0, 2, 1))).reshape(n, 9)
    P3 = P[:, O3:O3 + 27].reshape(n, 3, 3, 3)
    sym = sum(P3.transpose((0,) + tuple(1 + np.array(q))) for q in
              [(0, 1, 2), (0, 2, 1), (1, 0, 2), (1, 2, 0), (2, 0, 1), (2, 1, 0)]) / 6
    P[:, O3:O3 + 27] = sym.reshape(n, 27)
    G = orc.invariants(n, P)
    B = _blocks_by_einsum(P)
    exp = list(B["b0"])
    for key in ("b1", "b2", "b3"):
        exp += [B[key][s, t] for s in range(n) for t in range(s, n)]
    exp += [B["b4"][s, t, v] for s in range(n) for t in range(s, n) for v in range(t, n)]
    for key in ("b5", "b6"):
        exp += [B[key][s, t, v] for s in range(n) for t in range(s, n) for v in range(n)]
    exp += [B["b7"][s, t, v] for s in range(n) for t in range(n) for v in range(n)]
    assert len(exp) == 360
    assert np.allclose(G, np.array(exp), rtol=1e-12, atol=1e-12)


def test_dimer_closed_form(orc):
    """Two atoms: every feature is a plain product of R_s, independent of the direction."""
    w = wl.tiny_box(hidden=(8,))
    m = _model(orc, w)
    for u in (np.array([1.0, 0, 0]), np.array([1.0, 2.0, -2.0]) / 3.0):
        r = 3.1
        pos = np.array([[15.0, 15.0, 15.0], 15.0 + r * u])
        p = orc.neighbors(pos, [40, 40, 40], (0, 0, 0), 5.0)
        G = orc.energy_forces(m, pos, [0, 1], [40, 40, 40], p, forces=False, intermediates=True).G[0]
        R, _ = orc.radial(m, 0, 1, r)
        n = 5
        exp = list(R)
        for _ in range(3):
            exp += [R[s] * R[t] for s in range(n) for t in range(s, n)]
        exp += [R[s] * R[t] * R[v] for s in range(n) for t in range(s, n) for v in range(t, n)]
        for _ in range(2):
            exp += [R[s] * R[t] * R[v] for s in range(n) for t in range(s, n) for v in range(n)]
        exp += [R[s] * R[t] * R[v] for s in range(n) for t in range(n) for v in range(n)]
        assert np.allclose(G, exp, rtol=1e-11, atol=1e-13)


def test_simple_cubic_closed_form(orc):
    """One species on an unjittered simple-cubic lattice: P1 = P3 = 0 (inversion), P2 = P0/3 I
    (cubic) => blocks 1, 3, 5, 6, 7 vanish, block 2 = P0 P0 / 3, block 4 = P0 P0 P0 / 9;
    all forces vanish; all atomic energies are equal."""
    g, a = 4, 2.4
    idx = np.stack(np.meshgrid(*[np.arange(g)] * 3, indexing="ij"), -1).reshape(-1, 3)
    pos = (idx + 0.5) * a
    L = [g * a] * 3
    spec = wl.make_model(11, 1, r_cut=5.0, hidden=(16, 16))
    m = orc.Model(spec)
    p = orc.neighbors(pos, L, (1, 1, 1), 5.0)
    res = orc.energy_forces(m, pos, np.zeros(64, np.int32), L, p, intermediates=True)
    P0 = res.P[0, :, 0]
    G = res.G[0]
    n = 5
    pr = [(s, t) for s in range(n) for t in range(s, n)]
    tr = [(s, t, v) for s in range(n) for t in range(s, n) for v in range(t, n)]
    scale = np.abs(P0).max()
    assert np.allclose(G[0:5], P0)
    assert np.allclose(G[5:20], 0, atol=1e-12 * scale ** 2)
    assert np.allclose(G[20:35], [P0[s] * P0[t] / 3 for s, t in pr], rtol=1e-11)
    assert np.allclose(G[35:50], 0, atol=1e-12 * scale ** 2)
    assert np.allclose(G[50:85], [P0[s] * P0[t] * P0[v] / 9 for s, t, v in tr], rtol=1e-11)
    assert np.allclose(G[85:360], 0, atol=1e-11 * scale ** 3)
    assert np.abs(res.forces).max() < 1e-10
    assert np.ptp(res.e_atom) < 1e-10
    assert np.allclose(res.G, res.G[0][None, :], atol=1e-9)


def test_isolated_atom(orc):
    """No neighbours: Psi = 0 => G = 0 => E_i = sigma NN(0) + mu, F = 0."""
    spec = wl.make_model(3, 2, r_cut=5.0, hidden=(16, 16))
    spec.scale[:] = [1.5, 0.7]
    m = orc.Model(spec)
    pos = np.array([[5.0, 5, 5], [25.0, 25, 25]])
    p = orc.neighbors(pos, [50, 50, 50], (1, 1, 1), 5.0)
    assert len(p) == 0
    res = orc.energy_forces(m, pos, [0, 1], [50, 50, 50], p, intermediates=True)
    assert np.all(res.G == 0) and np.all(res.forces == 0)
    h = np.zeros(360)
    for W, b in zip(spec.W[:-1], spec.b[:-1]):
        z = h @ W.astype(np.float64) + b
        h = z / (1 + np.exp(-z))
    y0 = h @ spec.W[-1].astype(np.float64) + spec.b[-1]
    assert np.allclose(res.e_atom, spec.scale * y0[0] + spec.shift, rtol=1e-13)


def test_invariants_are_rotation_invariant(orc):
    """PAPER.md:49 'invariant under translations and rotations': every one of the 360 features,
    under a random proper rotation of a non-periodic cluster."""
    w = wl.cluster(24, 2)
    m = _model(orc, w)
    p = orc.neighbors(w.positions, w.cell, w.pbc, 5.0)
    G0 = orc.energy_forces(m, w.positions, w.species, w.cell, p, forces=False, intermediates=True).G
    rng = np.random.default_rng(1)
    A = rng.normal(size=(3, 3))
    Qm, _ = np.linalg.qr(A)
    if np.linalg.det(Qm) < 0:
        Qm[:, 0] *= -1
    c = w.positions.astype(np.float64).mean(0)
    pos = (w.positions.astype(np.float64) - c) @ Qm.T + c
    p2 = orc.neighbors(pos, w.cell, w.pbc, 5.0)
    assert len(p2) == len(p)
    G1 = orc.energy_forces(m, pos, w.species, w.cell, p2, forces=False, intermediates=True).G
    # positions handed to neighbors() are rounded to fp32 only for the predicate; G uses fp64 pos
    assert np.allclose(G0, G1, rtol=1e-9, atol=1e-9 * np.abs(G0).max())
    assert np.abs(G0[:, 85:]).max() > 1e-3  # the 4-body blocks are exercised


def test_invariants_bwd_is_gradient_of_invariants(orc):
    rng = np.random.default_rng(2)
    n = 3
    P = rng.normal(size=(n, 40))
    gbar = rng.normal(size=orc.n_features(n))
    Q = orc.invariants_bwd(n, P, gbar)
    h = 1e-6
    for (s, c) in [(0, 0), (1, 2), (2, 7), (0, 5), (1, 20), (2, 39), (0, 13), (2, 31)]:
        Pp, Pm = P.copy(), P.copy()
        Pp[s, c] += h
        Pm[s, c] -= h
        fd = (gbar @ orc.invariants(n, Pp) - gbar @ orc.invariants(n, Pm)) / (2 * h)
        assert abs(fd - Q[s, c]) < 1e-7 * max(1.0, abs(fd))


# ---------------------------------------------------------------- MLP (O-5, O-7)
def test_mlp_matches_numpy_matmul(orc):
    spec = wl.make_model(5, 2, r_cut=5.0, hidden=(512, 512), n_heads=4)
    m = orc.Model(spec)
    G = np.random.default_rng(3).normal(size=360) * 3
    y, zs = orc.mlp_forward(m, G)
    z1 = G @ spec.W[0].astype(np.float64) + spec.b[0]
    h1 = z1 / (1 + np.exp(-z1))
    z2 = h1 @ spec.W[1].astype(np.float64) + spec.b[1]
    h2 = z2 / (1 + np.exp(-z2))
    assert np.allclose(zs, np.concatenate([z1, z2]), rtol=1e-12, atol=1e-12)
    assert np.allclose(y, h2 @ spec.W[2].astype(np.float64) + spec.b[2], rtol=1e-12, atol=1e-12)


def test_mlp_without_hidden_layers_is_linear(orc):
    spec = wl.make_model(5, 1, r_cut=5.0, hidden=(), n_heads=1)
    m = orc.Model(spec)
    G = np.arange(360) / 100.0
    y, _ = orc.mlp_forward(m, G)
    assert np.allclose(y, G @ spec.W[0].astype(np.float64) + spec.b[0], rtol=1e-13)
    gb = orc.mlp_backward(m, np.zeros(1), [2.0], 360)
    assert np.allclose(gb, 2.0 * spec.W[0][:, 0], rtol=1e-13)


def test_swish_values_and_derivative(orc):
    assert orc.swish(0.0) == 0.0
    assert abs(orc.swish(40.0) - 40.0) < 1e-12 and abs(orc.swish(-40.0)) < 1e-12
    assert abs(orc.dswish(0.0) - 0.5) < 1e-15  # d/dx x sigmoid(x) at 0
    h = 1e-6
    for x in (-3.0, -0.5, 0.3, 2.0, 7.0):
        fd = (orc.swish(x + h) - orc.swish(x - h)) / (2 * h)
        assert abs(fd - orc.dswish(x)) < 1e-9


def test_mlp_backward_is_fd_of_forward(orc):
    spec = wl.make_model(9, 1, r_cut=5.0, hidden=(32, 24), n_heads=3)
    m = orc.Model(spec)
    G = np.random.default_rng(4).normal(size=360)
    ybar = np.array([0.3, -1.2, 0.8])
    _, zs = orc.mlp_forward(m, G)
    gb = orc.mlp_backward(m, zs, ybar, 360)
    h = 1e-6
    for k in (0, 17, 200, 359):
        Gp, Gm = G.copy(), G.copy()
        Gp[k] += h
        Gm[k] -= h
        fd = (ybar @ orc.mlp_forward(m, Gp)[0] - ybar @ orc.mlp_forward(m, Gm)[0]) / (2 * h)
        assert abs(fd - gb[k]) < 1e-8 * max(1.0, abs(fd))
