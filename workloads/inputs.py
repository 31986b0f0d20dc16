"""Seeded synthetic workloads shaped like the paper's systems.

Stand-ins, not data: the paper measures on EMIM+BF4- frames and on the
Li3PO4 dataset of its refs 5/8.  Neither is available here; these boxes
take their composition, density, cutoff and model shape only (BASELINE.json `configs`).

RNG: counter-based splitmix64, so every array is a pure function of (seed, index) and can be
regenerated on any machine; uniform = (x >> 11) * 2**-53, normals by Box-Muller.
Seeds: BASE_SEED + 10 * config + {0 positions, 1 species, 2 weights, 3 velocities}.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np

BASE_SEED = 250522168

# Units: Angstrom, eV, fs, amu.
KB_EV = 8.617333262e-5  # eV / K
ACC_CONV = 9.648533212e-3  # (eV/Ang/amu) -> Ang/fs^2 ; also eV/amu -> (Ang/fs)^2
AVOGADRO_CM3 = 0.602214076  # amu/Ang^3 per g/cm^3

# Per-family multiplier on scale_Z so the RMS force of the random-weight model is ~1 eV/Ang on the
# family's own initial positions (reading R17).  Written by
# tests/golden/calibrate_force_scale.py (calls only oracle/); values in
# tests/golden/force_scale.txt.  RMS force is per-atom (intensive), so one constant serves every
# N of a family.
FORCE_SCALE = {
    "tiny": 0.19,  # 1 / 5.317
    "ionic_liquid": 0.027,  # 1 / 37.13
    "li3po4": 0.02,  # 1 / 54.9 at N = 1024, 1 / 48.4 at N = 8192
}

_MASK = (1 << 64) - 1
_GAMMA = 0x9E3779B97F4A7C15


def splitmix64(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n outputs of splitmix64 seeded with `seed`, starting at draw `offset` (uint64)."""
    with np.errstate(over="ignore"):
        idx = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
        z = np.uint64(seed & _MASK) + idx * np.uint64(_GAMMA)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n doubles in [0, 1)."""
    return (splitmix64(seed, n, offset) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def normal01(seed: int, n: int) -> np.ndarray:
    """n standard normals (Box-Muller on consecutive uniform pairs)."""
    m = (n + 1) // 2
    u = uniform01(seed, 2 * m)
    u1 = 1.0 - u[0::2]  # (0, 1]
    u2 = u[1::2]
    r = np.sqrt(-2.0 * np.log(u1))
    out = np.empty(2 * m)
    out[0::2] = r * np.cos(2.0 * np.pi * u2)
    out[1::2] = r * np.sin(2.0 * np.pi * u2)
    return out[:n]


def _shuffle(seed: int, n: int) -> np.ndarray:
    """Seeded permutation of range(n): stable argsort of splitmix64 keys."""
    return np.argsort(splitmix64(seed, n), kind="stable")


def n_features(n_radial: int) -> int:
    """Length of the invariant vector G_i (shape only, blocks 0-7)."""
    n = n_radial
    return n + 3 * (n * (n + 1) // 2) + n * (n + 1) * (n + 2) // 6 + 2 * n * (n * (n + 1) // 2) + n ** 3


@dataclass
class ModelSpec:
    n_species: int
    n_basis: int
    n_radial: int
    r_cut: float
    r_min: float
    gamma: float
    hidden: Tuple[int, ...]
    n_heads: int
    beta: np.ndarray  # [S][S][n_radial][n_basis] f32, centre species first
    W: List[np.ndarray]  # layer l: [fan_in][fan_out] f32
    b: List[np.ndarray]  # layer l: [fan_out] f32
    scale: np.ndarray  # [S] f32  sigma_Z
    shift: np.ndarray  # [S] f32  mu_Z
    n_weight_sets: int = 1  # n_species: one NN per species, W[l] is [S][fan_in][fan_out], b[l] is [S][fan_out]
    basis_kind: int = 0  # 0 equidistant Gaussians, 1 Bessel-like functions of Kocer et al.
    zbl: bool = False  # add the ZBL repulsion
    zbl_r_max: float = 0.0  # Ang
    zbl_scale: float = 1.0
    atomic_numbers: "np.ndarray | None" = None  # [S] f32 nuclear charges for the ZBL term

    @property
    def n_features(self) -> int:
        return n_features(self.n_radial)


@dataclass
class Workload:
    name: str
    positions: np.ndarray  # [N][3] f32, wrapped into [0, L)
    species: np.ndarray  # [N] i32
    cell: np.ndarray  # [3] f32 orthorhombic edge lengths
    pbc: Tuple[int, int, int]
    masses: np.ndarray  # [N] f32 amu
    velocities: np.ndarray  # [N][3] f32 Ang/fs
    skin: float
    dt_fs: float
    n_steps: int
    model: ModelSpec
    species_names: Tuple[str, ...] = field(default_factory=tuple)
    lattice: "np.ndarray | None" = None  # [3][3] f32, rows = lattice vectors, for non-orthorhombic boxes (else None)

    @property
    def n_atoms(self) -> int:
        return int(self.positions.shape[0])

    @property
    def box(self) -> np.ndarray:
        """The cell as the oracle and the binding take it: [3][3] lattice if the box is triclinic, else [3] edges."""
        return self.cell if self.lattice is None else self.lattice

    @property
    def cell9(self) -> np.ndarray:
        """Row-major 3x3 lattice (rows = lattice vectors) as the C ABI takes it."""
        if self.lattice is not None:
            return np.ascontiguousarray(self.lattice, np.float32).reshape(9).copy()
        return np.diag(self.cell.astype(np.float32)).reshape(9).copy()


def make_model(
    seed: int,
    n_species: int,
    r_cut: float,
    n_basis: int = 7,
    n_radial: int = 5,
    r_min: float = 0.5,
    hidden: Sequence[int] = (512, 512),
    n_heads: int = 1,
    force_scale: float = 1.0,
    n_weight_sets: int = 1,
) -> ModelSpec:
    """Random-init GMNN weights: W ~ N(0, 1/fan_in), b ~ N(0, 0.1^2), beta ~ N(0, 1),
    shift ~ N(0, 1), scale = force_scale (BASELINE.json configs; R10, R17).

    The draws for beta, scale/shift and each layer come from separate seed streams, so a
    multi-head model (n_heads > 1) shares every tensor except the last layer with the
    single-head model of the same seed (config 4 "last MLP layer replaced by 32 heads").
    n_weight_sets = n_species draws one NN per species ("the per-species atomic MLP" of north_star): layer l is
    [S][fan_in][fan_out] from the same stream, so set 0 is the shared model of the same seed.
    """
    assert n_weight_sets in (1, n_species)
    delta = (r_cut - r_min) / (n_basis - 1)
    gamma = 1.0 / (2.0 * delta * delta)
    S = n_species
    beta = normal01(seed * 1000 + 1, S * S * n_radial * n_basis).reshape(S, S, n_radial, n_basis)
    dims = [n_features(n_radial), *hidden, n_heads]
    W, b = [], []
    for l in range(len(dims) - 1):
        fi, fo = dims[l], dims[l + 1]
        if n_weight_sets == 1:
            W.append((normal01(seed * 1000 + 10 + 2 * l, fi * fo).reshape(fi, fo) / np.sqrt(fi)).astype(np.float32))
            b.append((0.1 * normal01(seed * 1000 + 11 + 2 * l, fo)).astype(np.float32))
        else:
            T = n_weight_sets
            W.append((normal01(seed * 1000 + 10 + 2 * l, T * fi * fo).reshape(T, fi, fo) / np.sqrt(fi)).astype(np.float32))
            b.append((0.1 * normal01(seed * 1000 + 11 + 2 * l, T * fo).reshape(T, fo)).astype(np.float32))
    shift = normal01(seed * 1000 + 2, S).astype(np.float32)
    scale = np.full(S, force_scale, dtype=np.float32)
    return ModelSpec(
        n_species=S, n_basis=n_basis, n_radial=n_radial, r_cut=float(r_cut), r_min=float(r_min),
        gamma=float(gamma), hidden=tuple(int(h) for h in hidden), n_heads=int(n_heads),
        beta=beta.astype(np.float32), W=W, b=b, scale=scale, shift=shift, n_weight_sets=int(n_weight_sets),
    )


def _maxwell_boltzmann(seed: int, masses: np.ndarray, temperature: float) -> np.ndarray:
    n = masses.shape[0]
    sig = np.sqrt(KB_EV * temperature * ACC_CONV / masses.astype(np.float64))  # Ang/fs
    v = normal01(seed, 3 * n).reshape(n, 3) * sig[:, None]
    p = (v * masses[:, None].astype(np.float64)).sum(axis=0)
    v -= p[None, :] / masses.astype(np.float64).sum()
    return v.astype(np.float32)


def _wrap32(pos: np.ndarray, L: np.ndarray) -> np.ndarray:
    """Wrap into [0, L) and round to f32 such that the f32 value is still < f32(L)."""
    p = pos - np.floor(pos / L[None, :]) * L[None, :]
    p32 = p.astype(np.float32)
    L32 = L.astype(np.float32)
    p32 = np.where(p32 >= L32[None, :], np.float32(0.0), p32)
    p32 = np.where(p32 < 0, np.float32(0.0), p32)
    return p32


def _lattice_sites(seed: int, g: int, n: int) -> np.ndarray:
    """n of the g^3 simple-cubic sites, seeded choice, as integer triples [n][3]."""
    total = g ** 3
    assert n <= total
    pick = _shuffle(seed, total)[:n] if n < total else np.arange(total)
    pick = np.sort(pick)
    ix = pick // (g * g)
    iy = (pick // g) % g
    iz = pick % g
    return np.stack([ix, iy, iz], axis=1).astype(np.float64)


def _species_from_counts(seed: int, counts: Sequence[int]) -> np.ndarray:
    ids = np.concatenate([np.full(c, z, dtype=np.int32) for z, c in enumerate(counts)])
    return ids[_shuffle(seed, ids.shape[0])].astype(np.int32)


def tiny_box(hidden: Sequence[int] = (512, 512), n_heads: int = 1, seed_shift: int = 0,
             n_weight_sets: int = 1) -> Workload:
    """Config 1: 64 atoms, 8.5 Ang cube, 2 species 32/32, 4x4x4 lattice + U(-0.3, 0.3) jitter,
    r_cut 5 (box < 2 r_cut, so the same neighbour appears under several images)."""
    s = BASE_SEED + 10 * 1 + seed_shift
    L = np.array([8.5, 8.5, 8.5])
    a = 8.5 / 4
    sites = _lattice_sites(s, 4, 64)
    jit = uniform01(s, 3 * 64, offset=1 << 20).reshape(64, 3) * 0.6 - 0.3
    pos = _wrap32((sites + 0.5) * a + jit, L)
    species = _species_from_counts(s + 1, (32, 32))
    mass_table = np.array([12.011, 15.999], dtype=np.float32)
    masses = mass_table[species]
    model = make_model(s + 2, 2, r_cut=5.0, hidden=hidden, n_heads=n_heads, force_scale=FORCE_SCALE["tiny"],
                       n_weight_sets=n_weight_sets)
    vel = _maxwell_boltzmann(s + 3, masses, 300.0)
    return Workload("tiny", pos, species, L.astype(np.float32), (1, 1, 1), masses, vel,
                    skin=0.0, dt_fs=0.5, n_steps=0, model=model, species_names=("A", "B"))


def ionic_liquid_box(n_pairs: int = 64, hidden: Sequence[int] = (512, 512), n_heads: int = 1,
                     skin: float = 0.5, n_weight_sets: int = 1) -> Workload:
    """Config 2: EMIM+BF4- stoichiometry H11 C6 N2 B1 F4 per ion pair (24 atoms), 1.3 g/cm^3,
    jittered 12^3-type lattice with >= 0.9 Ang minimum distance, r_cut 6, skin 0.5, dt 0.5 fs."""
    s = BASE_SEED + 10 * 2
    per_pair = (11, 6, 2, 1, 4)  # H C N B F
    mass_table = np.array([1.008, 12.011, 14.007, 10.811, 18.998], dtype=np.float32)
    n = 24 * n_pairs
    pair_mass = float(sum(c * m for c, m in zip(per_pair, mass_table.astype(np.float64))))
    volume = n_pairs * pair_mass / (1.3 * AVOGADRO_CM3)
    Ls = volume ** (1.0 / 3.0)
    g = int(np.ceil((n * 1.125) ** (1.0 / 3.0) - 1e-9))  # 1536 atoms -> 12^3 = 1728 sites
    a = Ls / g
    jit_half = 0.5 * (a - 0.9) - 1e-3
    jit_half = min(jit_half, 0.6)
    assert a - 2 * jit_half >= 0.9
    L = np.array([Ls, Ls, Ls])
    sites = _lattice_sites(s, g, n)
    jit = (uniform01(s, 3 * n, offset=1 << 24).reshape(n, 3) * 2.0 - 1.0) * jit_half
    pos = _wrap32((sites + 0.5) * a + jit, L)
    species = _species_from_counts(s + 1, tuple(c * n_pairs for c in per_pair))
    masses = mass_table[species]
    model = make_model(s + 2, 5, r_cut=6.0, hidden=hidden, n_heads=n_heads,
                       force_scale=FORCE_SCALE["ionic_liquid"], n_weight_sets=n_weight_sets)
    vel = _maxwell_boltzmann(s + 3, masses, 300.0)
    return Workload("ionic_liquid", pos, species, L.astype(np.float32), (1, 1, 1), masses, vel,
                    skin=skin, dt_fs=0.5, n_steps=1000, model=model,
                    species_names=("H", "C", "N", "B", "F"))


def li3po4_box(n_atoms: int, hidden: Sequence[int] = (512, 512), n_heads: int = 1, skin: float = 0.0,
               n_steps: int = 0, config: int = 3, n_weight_sets: int = 1) -> Workload:
    """Configs 3, 4, 5: Li:P:O = 3:1:4 at 2.4 g/cm^3, jittered simple-cubic lattice with
    N(0, 0.1^2) noise clipped at +-0.4 Ang, r_cut 6.  Model weights depend only on the family
    (same seed for every N), positions on (config, N)."""
    assert n_atoms % 8 == 0
    s = BASE_SEED + 10 * config
    mass_table = np.array([6.94, 30.974, 15.999], dtype=np.float32)
    fu_mass = 3 * 6.94 + 30.974 + 4 * 15.999
    volume = (n_atoms // 8) * fu_mass / (2.4 * AVOGADRO_CM3)
    Ls = volume ** (1.0 / 3.0)
    g = int(np.ceil(n_atoms ** (1.0 / 3.0) - 1e-9))
    a = Ls / g
    L = np.array([Ls, Ls, Ls])
    sites = _lattice_sites(s + n_atoms, g, n_atoms)
    jit = np.clip(0.1 * normal01(s + n_atoms + 7, 3 * n_atoms).reshape(n_atoms, 3), -0.4, 0.4)
    pos = _wrap32((sites + 0.5) * a + jit, L)
    fu = n_atoms // 8
    species = _species_from_counts(s + n_atoms + 1, (3 * fu, fu, 4 * fu))
    masses = mass_table[species]
    # one weight seed for the whole Li3PO4 family (configs 3, 4, 5 share the model body)
    model = make_model(BASE_SEED + 10 * 3 + 2, 3, r_cut=6.0, hidden=hidden, n_heads=n_heads,
                       force_scale=FORCE_SCALE["li3po4"], n_weight_sets=n_weight_sets)
    vel = _maxwell_boltzmann(s + n_atoms + 3, masses, 300.0)
    return Workload("li3po4_%d" % n_atoms, pos, species, L.astype(np.float32), (1, 1, 1), masses, vel,
                    skin=skin, dt_fs=0.5, n_steps=n_steps, model=model, species_names=("Li", "P", "O"))


def triclinic_box(n_atoms: int = 1000, hidden: Sequence[int] = (64, 64), skin: float = 0.0, n_heads: int = 1,
                  shear: Sequence[float] = (0.25, 0.1, 0.35), stretch: Sequence[float] = (1.0, 1.1, 0.9)) -> Workload:
    """Li3PO4-shaped box (density, species ratio, r_cut, model family of config 3) in a sheared cell for the
    general-lattice path: lattice rows a = (s0 L, 0, 0), b = (shear0 L, s1 L, 0),
    c = (shear1 L, shear2 L, s2 L); atoms on a jittered grid in fractional coordinates, wrapped into the cell."""
    assert n_atoms % 8 == 0
    s = BASE_SEED + 10 * 6
    mass_table = np.array([6.94, 30.974, 15.999], dtype=np.float32)
    fu_mass = 3 * 6.94 + 30.974 + 4 * 15.999
    volume = (n_atoms // 8) * fu_mass / (2.4 * AVOGADRO_CM3)
    Ls = (volume / (stretch[0] * stretch[1] * stretch[2])) ** (1.0 / 3.0)
    h = np.array([[stretch[0] * Ls, 0.0, 0.0], [shear[0] * Ls, stretch[1] * Ls, 0.0],
                  [shear[1] * Ls, shear[2] * Ls, stretch[2] * Ls]])
    g = int(np.ceil(n_atoms ** (1.0 / 3.0) - 1e-9))
    sites = _lattice_sites(s + n_atoms, g, n_atoms)
    frac = (sites + 0.5) / g
    jit = np.clip(0.1 * normal01(s + n_atoms + 7, 3 * n_atoms).reshape(n_atoms, 3), -0.4, 0.4)
    h32 = h.astype(np.float32)
    hinv = np.linalg.inv(h32.astype(np.float64))
    f = frac + jit @ hinv
    f -= np.floor(f)
    pos = (f @ h32.astype(np.float64)).astype(np.float32)
    for _ in range(3):  # fp32 rounding may leave an atom a hair outside: fold again in the fp32 cell
        fr = pos.astype(np.float64) @ hinv
        k = np.floor(fr)
        if not k.any():
            break
        pos = (pos.astype(np.float64) - k @ h32.astype(np.float64)).astype(np.float32)
    fu = n_atoms // 8
    species = _species_from_counts(s + n_atoms + 1, (3 * fu, fu, 4 * fu))
    masses = mass_table[species]
    model = make_model(BASE_SEED + 10 * 3 + 2, 3, r_cut=6.0, hidden=hidden, n_heads=n_heads,
                       force_scale=FORCE_SCALE["li3po4"])
    vel = _maxwell_boltzmann(s + n_atoms + 3, masses, 300.0)
    edges = np.linalg.norm(h32, axis=1).astype(np.float32)
    return Workload("triclinic_%d" % n_atoms, pos, species, edges, (1, 1, 1), masses, vel, skin=skin, dt_fs=0.5,
                    n_steps=0, model=model, species_names=("Li", "P", "O"), lattice=h32)


def cluster(n_atoms: int = 24, n_species: int = 2, box: float = 40.0, radius: float = 3.5,
            hidden: Sequence[int] = (16, 16), n_heads: int = 1, seed_shift: int = 0,
            r_cut: float = 5.0) -> Workload:
    """Non-periodic blob of atoms (pbc = 0) centred in a big box: for rotation-invariance pins.
    Rejection-free: points on a jittered 3x3x3-ish grid scaled into a ball of `radius`."""
    s = BASE_SEED + 990 + seed_shift
    g = int(np.ceil(n_atoms ** (1.0 / 3.0)))
    sites = _lattice_sites(s, g, n_atoms)
    a = 2.0 * radius / g
    jit = (uniform01(s, 3 * n_atoms, offset=1 << 16).reshape(n_atoms, 3) - 0.5) * 0.5 * a
    pos = (sites + 0.5) * a - radius + jit + box / 2
    L = np.array([box, box, box])
    species = (splitmix64(s + 1, n_atoms) % np.uint64(n_species)).astype(np.int32)
    masses = (1.0 + 10.0 * species).astype(np.float32)
    model = make_model(s + 2, n_species, r_cut=r_cut, hidden=hidden, n_heads=n_heads)
    vel = _maxwell_boltzmann(s + 3, masses, 300.0)
    return Workload("cluster", pos.astype(np.float32), species, L.astype(np.float32), (0, 0, 0), masses, vel,
                    skin=0.0, dt_fs=0.5, n_steps=0, model=model)


def make_workload(name: str, **kw) -> Workload:
    """Named BASELINE.json configs: 'config1', 'config2', 'config3_<N>', 'config4', 'config5'."""
    if name == "config1":
        return tiny_box(**kw)
    if name == "config2":
        return ionic_liquid_box(**kw)
    if name.startswith("config3_"):
        return li3po4_box(int(name.split("_")[1]), **kw)
    if name == "config4":
        kw.setdefault("n_heads", 32)
        return li3po4_box(8192, config=3, **kw)
    if name == "config5":
        kw.setdefault("skin", 1.0)
        kw.setdefault("n_steps", 200)
        return li3po4_box(1048576, config=5, **kw)
    raise KeyError(name)
