"""ctypes face of oracle/gmnn_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2505_22168_b200/ and shares no code with it.
All floating point crosses this boundary as fp64 (fp32 inputs are promoted, never the reverse),
except the positions handed to the neighbour search, whose predicate is specified in fp32
(reading R20).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gmnn_oracle.c")
_LIB = os.path.join(_HERE, "libgmnn_oracle.so")
NC = 40  # components per channel: 1 + 3 + 9 + 27
GCC_FLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the shared object is missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", *GCC_FLAGS, _SRC, "-lm", "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


class _HParams(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32), ("n_basis", C.c_int32), ("n_radial", C.c_int32),
        ("r_cut", C.c_double), ("r_min", C.c_double), ("gamma", C.c_double),
        ("n_hidden", C.c_int32), ("hidden", C.c_int32 * 4), ("n_heads", C.c_int32), ("n_weight_sets", C.c_int32),
        ("basis_kind", C.c_int32), ("zbl_on", C.c_int32), ("zbl_r_max", C.c_double), ("zbl_scale", C.c_double),
    ]


class _Weights(C.Structure):
    _fields_ = [
        ("beta", C.c_void_p), ("W", C.c_void_p * 5), ("b", C.c_void_p * 5),
        ("scale", C.c_void_p), ("shift", C.c_void_p), ("atomic_number", C.c_void_p),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_neighbors_brute.restype = C.c_int64
        _lib.oracle_neighbors_cells.restype = C.c_int64
        _lib.oracle_swish.restype = C.c_double
        _lib.oracle_dswish.restype = C.c_double
        _lib.oracle_swish.argtypes = [C.c_double]
        _lib.oracle_dswish.argtypes = [C.c_double]
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a), dtype=np.int32)


def cell9(cell) -> np.ndarray:
    """The 3x3 lattice (rows = lattice vectors) as 9 doubles, from [3] edge lengths of an orthorhombic box,
    or a [3][3] / [9] matrix (O-16: general cells)."""
    c = np.asarray(cell, dtype=np.float64)
    if c.size == 3:
        return np.diag(c.reshape(3)).reshape(9).copy()
    assert c.size == 9
    return np.ascontiguousarray(c.reshape(9))


def wrap_positions(y, cell, pbc) -> np.ndarray:
    """Positions folded into the cell along the periodic axes (diag(L): y - floor(y / L) L; general lattice: in
    fractional coordinates)."""
    h = cell9(cell).reshape(3, 3)
    per = np.asarray(pbc).astype(bool)
    y = np.array(y, dtype=np.float64, copy=True)
    if np.count_nonzero(h - np.diag(np.diag(h))) == 0:
        L = np.diag(h)
        y[:, per] -= np.floor(y[:, per] / L[per]) * L[per]
        return y
    k = np.floor(y @ np.linalg.inv(h))
    k[:, ~per] = 0.0
    return y - k @ h


def to_fp32_inside(y, cell) -> np.ndarray:
    """fp32 copy of wrapped fp64 positions that is still inside the cell after rounding (the neighbour predicate
    is specified on fp32 positions in [0, 1) fractional; rounding up onto the far face folds to the near one)."""
    h = cell9(cell).reshape(3, 3)
    y32 = np.asarray(y).astype(np.float32)
    if np.count_nonzero(h - np.diag(np.diag(h))) == 0:
        L32 = np.diag(h).astype(np.float32)
        return np.where(y32 >= L32[None, :], np.float32(0), y32)
    frac = y32.astype(np.float64) @ np.linalg.inv(h.astype(np.float32).astype(np.float64))
    over = frac >= 1.0
    if over.any():
        y32 = (y32.astype(np.float64) - over.astype(np.float64) @ h).astype(np.float32)
    return y32


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(C.c_int(n))


def n_features(n_radial: int) -> int:
    return int(lib().oracle_n_features(C.c_int(n_radial)))


class Model:
    """fp64 copy of a model (any object with the attributes of workloads.ModelSpec)."""

    def __init__(self, spec):
        self.n_species = int(spec.n_species)
        self.n_basis = int(spec.n_basis)
        self.n_radial = int(spec.n_radial)
        self.r_cut = float(spec.r_cut)
        self.r_min = float(spec.r_min)
        self.gamma = float(spec.gamma)
        self.hidden = tuple(int(h) for h in spec.hidden)
        self.n_heads = int(spec.n_heads)
        # 1: one NN for all species (Eq. 4); n_species: W[l] is [S][fan_in][fan_out], b[l] is [S][fan_out] (O-5)
        self.n_weight_sets = int(getattr(spec, "n_weight_sets", 1))
        assert self.n_weight_sets in (1, int(spec.n_species))
        # O-17: radial basis 0 Gaussians / 1 Bessel-like; O-18: ZBL repulsion with nuclear charges per species
        self.basis_kind = int(getattr(spec, "basis_kind", 0))
        self.zbl_on = int(bool(getattr(spec, "zbl", False)))
        self.zbl_r_max = float(getattr(spec, "zbl_r_max", 0.0))
        self.zbl_scale = float(getattr(spec, "zbl_scale", 1.0))
        zn = getattr(spec, "atomic_numbers", None)
        self.atomic_numbers = _f64(zn if zn is not None else np.zeros(self.n_species))
        self.beta = _f64(spec.beta)
        self.W = [_f64(w) for w in spec.W]
        self.b = [_f64(b) for b in spec.b]
        self.scale = _f64(spec.scale)
        self.shift = _f64(spec.shift)
        assert len(self.W) == len(self.hidden) + 1
        self.n_features = n_features(self.n_radial)
        assert self.W[0].shape[-2] == self.n_features, (self.W[0].shape, self.n_features)
        if self.n_weight_sets > 1:
            assert all(w.shape[0] == self.n_weight_sets for w in self.W + self.b)
        self.hp = _HParams()
        self.hp.n_species, self.hp.n_basis, self.hp.n_radial = self.n_species, self.n_basis, self.n_radial
        self.hp.r_cut, self.hp.r_min, self.hp.gamma = self.r_cut, self.r_min, self.gamma
        self.hp.n_hidden = len(self.hidden)
        for l, h in enumerate(self.hidden):
            self.hp.hidden[l] = h
        self.hp.n_heads = self.n_heads
        self.hp.n_weight_sets = self.n_weight_sets
        self.hp.basis_kind, self.hp.zbl_on = self.basis_kind, self.zbl_on
        self.hp.zbl_r_max, self.hp.zbl_scale = self.zbl_r_max, self.zbl_scale
        self.w = _Weights()
        self.w.beta = _p(self.beta)
        for l in range(len(self.W)):
            self.w.W[l] = self.W[l].ctypes.data
            self.w.b[l] = self.b[l].ctypes.data
        self.w.scale = _p(self.scale)
        self.w.shift = _p(self.shift)
        self.w.atomic_number = _p(self.atomic_numbers)


@dataclass
class Pairs:
    i: np.ndarray  # [n] i32
    j: np.ndarray  # [n] i32
    n: np.ndarray  # [n][3] i32 image vector

    def __len__(self):
        return int(self.i.shape[0])

    def as_set_array(self) -> np.ndarray:
        """[n][5] int32 rows (i, j, nx, ny, nz), already sorted by the oracle."""
        return np.concatenate([self.i[:, None], self.j[:, None], self.n], axis=1)


def neighbors(positions, cell, pbc, r_list: float, method: str = "brute") -> Pairs:
    """O-1.  positions [N][3] are rounded to fp32 (the predicate's precision); cell [3] (orthorhombic edge
    lengths) or [3][3] (rows = lattice vectors, O-16), rounded to fp32 likewise."""
    pos = np.ascontiguousarray(np.asarray(positions), dtype=np.float32)
    c = np.asarray(cell, dtype=np.float32)
    L = np.ascontiguousarray(np.diag(c.reshape(3)).reshape(9) if c.size == 3 else c.reshape(9))
    pb = _i32(pbc)
    N = pos.shape[0]
    fn = {"brute": lib().oracle_neighbors_brute, "cells": lib().oracle_neighbors_cells}[method]
    cap = max(1024, 128 * N)
    while True:
        oi = np.empty(cap, np.int32)
        oj = np.empty(cap, np.int32)
        on = np.empty((cap, 3), np.int32)
        n = fn(C.c_int64(N), _p(pos), _p(L), _p(pb), C.c_float(r_list), C.c_int64(cap), _p(oi), _p(oj), _p(on))
        if n < 0:
            raise ValueError("cell list needs >= 3 cells on every periodic axis; use method='brute'")
        if n <= cap:
            return Pairs(oi[:n].copy(), oj[:n].copy(), on[:n].copy())
        cap = int(n)


def auto_neighbors(positions, cell, pbc, r_list: float) -> Pairs:
    """Brute force up to 8192 atoms, the oracle's own cell list above."""
    N = np.asarray(positions).shape[0]
    if N <= 8192:
        return neighbors(positions, cell, pbc, r_list, "brute")
    try:
        return neighbors(positions, cell, pbc, r_list, "cells")
    except ValueError:
        return neighbors(positions, cell, pbc, r_list, "brute")


def radial(model: Model, zi: int, zj: int, r: float):
    """O-2 for one pair: (R [n_radial], dR/dr [n_radial])."""
    R = np.zeros(model.n_radial)
    dR = np.zeros(model.n_radial)
    lib().oracle_radial(C.byref(model.hp), _p(model.beta), C.c_int(zi), C.c_int(zj), C.c_double(r), _p(R), _p(dR))
    return R, dR


def basis(model: Model, r: float):
    """O-2 / O-17: the raw basis functions of one distance and their derivatives, without the cutoff function."""
    phi = np.zeros(model.n_basis)
    dphi = np.zeros(model.n_basis)
    lib().oracle_basis(C.byref(model.hp), C.c_double(r), _p(phi), _p(dphi))
    return phi, dphi


def zbl_half(model: Model, z1: float, z2: float, r: float):
    """O-18: (V/2, d(V/2)/dr) of the ZBL repulsion for one directed pair."""
    e, de = C.c_double(0), C.c_double(0)
    lib().oracle_zbl_half(C.byref(model.hp), C.c_double(z1), C.c_double(z2), C.c_double(r), C.byref(e), C.byref(de))
    return float(e.value), float(de.value)


def invariants(n_radial: int, P) -> np.ndarray:
    """O-4 for one atom: P [n_radial][40] -> G [F]."""
    P = _f64(P)
    assert P.shape == (n_radial, NC)
    G = np.zeros(n_features(n_radial))
    lib().oracle_invariants(C.c_int(n_radial), _p(P), _p(G))
    return G


def invariants_bwd(n_radial: int, P, gbar) -> np.ndarray:
    """O-8 for one atom: Q [n_radial][40] = dE/dP given gbar = dE/dG."""
    P = _f64(P)
    gbar = _f64(gbar)
    Q = np.zeros((n_radial, NC))
    lib().oracle_invariants_bwd(C.c_int(n_radial), _p(P), _p(gbar), _p(Q))
    return Q


def mlp_forward(model: Model, G, wset: int = 0):
    """O-5 for one atom with weight set `wset`: (y [M], zs [sum hidden])."""
    G = _f64(G)
    zs = np.zeros(max(1, sum(model.hidden)))
    y = np.zeros(model.n_heads)
    lib().oracle_mlp_forward(C.byref(model.hp), C.byref(model.w), C.c_int(G.shape[0]), _p(G), _p(zs), _p(y), C.c_int(wset))
    return y, zs


def mlp_backward(model: Model, zs, ybar, n_in: int, wset: int = 0) -> np.ndarray:
    """O-7 for one atom with weight set `wset`: dE/dG given ybar [M]."""
    zs = _f64(zs)
    ybar = _f64(ybar)
    Gbar = np.zeros(n_in)
    lib().oracle_mlp_backward(C.byref(model.hp), C.byref(model.w), C.c_int(n_in), _p(zs), _p(ybar), _p(Gbar),
                              C.c_int(wset))
    return Gbar


def swish(x: float) -> float:
    return float(lib().oracle_swish(C.c_double(x)))


def dswish(x: float) -> float:
    return float(lib().oracle_dswish(C.c_double(x)))


@dataclass
class Result:
    energy: float  # sum_i sum_m head_w[m] E_i^(m)
    e_heads: np.ndarray  # [N][M]
    forces: Optional[np.ndarray]  # [N][3]
    P: Optional[np.ndarray] = None  # [N][n_radial][40]
    G: Optional[np.ndarray] = None  # [N][F]
    dG: Optional[np.ndarray] = None  # [N][F]
    Q: Optional[np.ndarray] = None  # [N][n_radial][40]
    virial: Optional[np.ndarray] = None  # [3][3]  W = -sum_pairs d (x) g = -dE/d strain (O-16); stress = -W / V

    @property
    def e_atom(self) -> np.ndarray:
        return self.e_heads[:, 0]


def energy_forces(model: Model, positions, species, cell, pairs: Pairs, head_w: Optional[Sequence[float]] = None,
                  forces: bool = True, intermediates: bool = False) -> Result:
    """O-2..O-9 on a pair list.  head_w: weights of the heads in the differentiated energy
    (default: 1 for a single head, 1/M each for an ensemble = gradient of the mean energy)."""
    pos = _f64(positions)
    sp = _i32(species)
    L = cell9(cell)
    N = pos.shape[0]
    M = model.n_heads
    hw = _f64(np.full(M, 1.0 / M) if head_w is None else head_w)
    assert hw.shape == (M,)
    F = model.n_features
    e_heads = np.zeros((N, M))
    f = np.zeros((N, 3)) if forces else None
    Pm = np.zeros((N, model.n_radial, NC)) if intermediates else None
    G = np.zeros((N, F)) if intermediates else None
    dG = np.zeros((N, F)) if (intermediates and forces) else None
    Q = np.zeros((N, model.n_radial, NC)) if (intermediates and forces) else None
    vir = np.zeros((3, 3)) if forces else None
    pi, pj, pn = _i32(pairs.i), _i32(pairs.j), _i32(pairs.n)
    rc = lib().oracle_energy_forces(
        C.byref(model.hp), C.byref(model.w), C.c_int64(N), _p(pos), _p(sp), _p(L), C.c_int64(len(pairs)),
        _p(pi), _p(pj), _p(pn), _p(hw), _p(e_heads), _p(f), _p(Pm), _p(G), _p(dG), _p(Q), _p(vir))
    if rc != 0:
        raise ValueError("oracle_energy_forces: bad argument")
    return Result(float((e_heads @ hw).sum()), e_heads, f, Pm, G, dG, Q, vir)


@dataclass
class EnsembleResult:
    e_heads: np.ndarray  # [N][M]
    e_mean: np.ndarray  # [N]
    e_var: np.ndarray  # [N]
    f_mean: np.ndarray  # [N][3]
    f_var: np.ndarray  # [N][3]
    f_heads: Optional[np.ndarray]  # [M][N][3]


def ensemble(model: Model, positions, species, cell, pairs: Pairs, keep_heads: bool = False) -> EnsembleResult:
    """O-10 (Eq. 5 with the 1/N_ens divisor, Eq. 6)."""
    pos = _f64(positions)
    sp = _i32(species)
    L = cell9(cell)
    N = pos.shape[0]
    M = model.n_heads
    e_heads = np.zeros((N, M))
    e_mean, e_var = np.zeros(N), np.zeros(N)
    f_mean, f_var = np.zeros((N, 3)), np.zeros((N, 3))
    fh = np.zeros((M, N, 3)) if keep_heads else None
    pi, pj, pn = _i32(pairs.i), _i32(pairs.j), _i32(pairs.n)
    rc = lib().oracle_ensemble(
        C.byref(model.hp), C.byref(model.w), C.c_int64(N), _p(pos), _p(sp), _p(L), C.c_int64(len(pairs)),
        _p(pi), _p(pj), _p(pn), _p(e_heads), _p(e_mean), _p(e_var), _p(f_mean), _p(f_var), _p(fh))
    if rc != 0:
        raise ValueError("oracle_ensemble: bad argument")
    return EnsembleResult(e_heads, e_mean, e_var, f_mean, f_var, fh)


@dataclass
class NVEResult:
    positions: np.ndarray
    velocities: np.ndarray
    epot: np.ndarray  # [n_steps + 1]
    ekin: np.ndarray  # [n_steps + 1]
    n_rebuilds: int


def nve(model: Model, positions, velocities, masses, species, cell, pbc, skin: float, dt_fs: float,
        n_steps: int) -> NVEResult:
    """O-11 velocity Verlet."""
    x = _f64(positions).copy()
    v = _f64(velocities).copy()
    m = _f64(masses)
    sp = _i32(species)
    L = cell9(cell)
    pb = _i32(pbc)
    epot = np.zeros(n_steps + 1)
    ekin = np.zeros(n_steps + 1)
    nreb = C.c_int64(0)
    rc = lib().oracle_nve(
        C.byref(model.hp), C.byref(model.w), C.c_int64(x.shape[0]), _p(x), _p(v), _p(m), _p(sp), _p(L), _p(pb),
        C.c_double(skin), C.c_double(dt_fs), C.c_int64(n_steps), _p(epot), _p(ekin), C.byref(nreb))
    if rc != 0:
        raise ValueError("oracle_nve: bad argument")
    return NVEResult(x, v, epot, ekin, int(nreb.value))


@dataclass
class SwitchingResult:
    positions: np.ndarray
    velocities: np.ndarray
    epot: np.ndarray  # [n_steps_done + 1], mean energy over the heads
    ekin: np.ndarray  # [n_steps_done + 1]
    sigma_e: np.ndarray  # [n_samples]
    sigma_f_max: np.ndarray  # [n_samples]
    f_var_last: np.ndarray  # [N][3] of the last sample (zeros if none was taken)
    n_steps_done: int
    n_rebuilds: int


def md_switching(model: Model, positions, velocities, masses, species, cell, pbc, skin: float, dt_fs: float,
                 n_steps: int, sampling_rate: int, f_sigma_stop: float = 0.0) -> SwitchingResult:
    """O-12 switching-mode shallow-ensemble MD (Eq. 5, 6)."""
    x = _f64(positions).copy()
    v = _f64(velocities).copy()
    m = _f64(masses)
    sp = _i32(species)
    L = cell9(cell)
    pb = _i32(pbc)
    epot = np.zeros(n_steps + 1)
    ekin = np.zeros(n_steps + 1)
    ns_max = max(n_steps // max(sampling_rate, 1), 1)
    se, sf = np.zeros(ns_max), np.zeros(ns_max)
    fv = np.zeros((x.shape[0], 3))
    done, nsamp, nreb = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    rc = lib().oracle_md_switching(
        C.byref(model.hp), C.byref(model.w), C.c_int64(x.shape[0]), _p(x), _p(v), _p(m), _p(sp), _p(L), _p(pb),
        C.c_double(skin), C.c_double(dt_fs), C.c_int64(n_steps), C.c_int64(sampling_rate), C.c_double(f_sigma_stop),
        _p(epot), _p(ekin), _p(se), _p(sf), _p(fv), C.byref(done), C.byref(nsamp), C.byref(nreb))
    if rc != 0:
        raise ValueError("oracle_md_switching: bad argument")
    d, k = int(done.value), int(nsamp.value)
    return SwitchingResult(x, v, epot[:d + 1], ekin[:d + 1], se[:k], sf[:k], fv, d, int(nreb.value))


@dataclass
class UDDResult:
    energy: float  # mean energy of the heads + bias
    e_mean: float
    e_bias: float
    var_e: float  # sigma_E^2 of Eq. 5 (total energies, 1/N_ens)
    forces: np.ndarray  # [N][3] = -d(energy)/dR


def udd_energy_forces(model: Model, positions, species, cell, pairs: Pairs, A: float, B: float) -> UDDResult:
    """O-13 uncertainty-driven-dynamics bias (Eq. 9):
    E_b = A [exp(-sigma_E^2 / (N_ens N_atoms B^2)) - 1], sigma_E^2 = 1/N_ens sum_m (E^(m) - mean)^2 of the TOTAL
    energies (Eq. 5, reading R27).  Forces of mean + E_b by the chain rule on the per-head forces of O-10:
    -grad sigma^2 = 2/N_ens sum_m (E^(m) - mean) (F^(m) - F_mean)."""
    ens = ensemble(model, positions, species, cell, pairs, keep_heads=True)
    M, N = model.n_heads, ens.e_heads.shape[0]
    tot = ens.e_heads.sum(0)
    mean = tot.mean()
    var = ((tot - mean) ** 2).mean()
    width = M * N * B * B
    e_b = A * (np.exp(-var / width) - 1.0)
    de_b = -A / width * np.exp(-var / width)  # dE_b / d sigma^2
    neg_grad_var = (2.0 / M) * np.einsum("m,mia->ia", tot - mean, ens.f_heads - ens.f_mean[None])
    forces = ens.f_mean + de_b * neg_grad_var
    return UDDResult(float(mean + e_b), float(mean), float(e_b), float(var), forces)


def nve_udd(model: Model, positions, velocities, masses, species, cell, pbc, dt_fs: float, n_steps: int,
            A: float, B: float):
    """O-11's velocity Verlet on the biased energy of O-13, with a fresh list of radius r_cut at every step
    (the trajectory does not depend on the skin: pinned for O-11).  Returns x, v, epot[n+1], ekin[n+1], e_bias[n+1]."""
    ACC = 9.648533212e-3
    x = _f64(positions).copy()
    v = _f64(velocities).copy()
    m = _f64(masses)[:, None]

    def wrap(y):
        return wrap_positions(y, cell, pbc)

    def evaluate(y):
        y32 = to_fp32_inside(y, cell)  # the neighbour predicate is specified in fp32 (R20); E and F use the fp64 y
        return udd_energy_forces(model, y, species, cell, auto_neighbors(y32, cell, pbc, model.r_cut), A, B)

    x = wrap(x)
    r = evaluate(x)
    epot, ekin, eb = [r.energy], [0.5 * (m * v * v).sum() / ACC], [r.e_bias]
    for _ in range(n_steps):
        v += 0.5 * dt_fs * r.forces / m * ACC
        x = wrap(x + dt_fs * v)
        r = evaluate(x)
        v += 0.5 * dt_fs * r.forces / m * ACC
        epot.append(r.energy)
        ekin.append(0.5 * (m * v * v).sum() / ACC)
        eb.append(r.e_bias)
    return x, v, np.array(epot), np.array(ekin), np.array(eb)


KB_EV = 8.617333262e-5  # Boltzmann constant, eV/K


def _sy_weights(sy_steps: int):
    """Suzuki-Yoshida weights of the chain sub-steps (1, 3 or 5)."""
    if sy_steps == 1:
        return [1.0]
    if sy_steps == 3:
        a = 1.0 / (2.0 - 2.0 ** (1.0 / 3.0))
        return [a, 1.0 - 2.0 * a, a]
    if sy_steps == 5:
        a = 1.0 / (4.0 - 4.0 ** (1.0 / 3.0))
        return [a, a, 1.0 - 4.0 * a, a, a]
    raise ValueError("sy_steps must be 1, 3 or 5")


def nhc_half_step(ke2: float, xi: np.ndarray, pxi: np.ndarray, Q: np.ndarray, dof: float, kT: float, dt: float,
                  chain_steps: int, sy_steps: int) -> float:
    """O-14a: the thermostat operator of a Nose-Hoover chain for half a time step (Martyna, Tuckerman, Tobias,
    Klein 1996; the `thermostat_chain` of PAPER.md:365-375: chain_length, chain_steps, sy_steps, tau).
    ke2 = sum m v^2 (eV).  Updates xi, pxi in place and returns the factor the velocities are scaled by."""
    Mc = len(xi)
    scale = 1.0
    delta = dt / chain_steps
    for _ in range(chain_steps):
        for wgt in _sy_weights(sy_steps):
            d2, d4, d8 = delta * wgt / 2, delta * wgt / 4, delta * wgt / 8
            G = (pxi[Mc - 2] ** 2 / Q[Mc - 2] - kT) if Mc > 1 else (ke2 - dof * kT)
            pxi[Mc - 1] += d4 * G
            for k in range(Mc - 2, -1, -1):
                G = (ke2 - dof * kT) if k == 0 else (pxi[k - 1] ** 2 / Q[k - 1] - kT)
                s = np.exp(-d8 * pxi[k + 1] / Q[k + 1])
                pxi[k] = s * (s * pxi[k] + d4 * G)
            s = np.exp(-d2 * pxi[0] / Q[0])
            scale *= s
            ke2 *= s * s
            xi += d2 * pxi / Q
            G = ke2 - dof * kT
            for k in range(Mc - 1):
                s = np.exp(-d8 * pxi[k + 1] / Q[k + 1])
                pxi[k] = s * (s * pxi[k] + d4 * G)
                G = pxi[k] ** 2 / Q[k] - kT
            pxi[Mc - 1] += d4 * G
    return scale


def schedule_temperature(schedule, n: int, default: float) -> float:
    """O-19: the thermostat's target at MD step n (0-based, counted from where the schedule was set) of a temperature
    schedule (steps [k] ascending, temps [k] in K): piecewise linear between the points, constant before the first and
    after the last ("temperature profiles oscillating between 300 K and 600 K"; reading R32).
    schedule None: the constant `default`."""
    if schedule is None:
        return float(default)
    steps, temps = schedule
    return float(np.interp(float(n), np.asarray(steps, np.float64), np.asarray(temps, np.float64)))


def nvt_nose_hoover(model: Model, positions, velocities, masses, species, cell, pbc, dt_fs: float, n_steps: int,
                    temperature: float, tau_fs: float, chain_length: int = 3, chain_steps: int = 2, sy_steps: int = 3,
                    schedule=None):
    """O-14: NVT with a Nose-Hoover chain: chain half step, velocity Verlet (O-11) on the mean
    energy, chain half step.  Q_0 = dof kT tau^2, Q_k = kT tau^2, dof = 3 N (reading R28).  Fresh list of radius
    r_cut every step.  Returns x, v, epot, ekin, conserved (all [n_steps + 1]; conserved = epot + ekin +
    sum pxi^2 / 2Q + dof kT xi_0 + kT sum_{k>0} xi_k).  With a `schedule` (O-19) both chain half steps of MD step n
    take kT = k_B T(n); the thermostat masses Q stay those of `temperature` (reading R32)."""
    ACC = 9.648533212e-3
    x = _f64(positions).copy()
    v = _f64(velocities).copy()
    m = _f64(masses)[:, None]
    N = x.shape[0]
    dof, kT = 3.0 * N, KB_EV * temperature
    Q = np.full(chain_length, kT * tau_fs ** 2)
    Q[0] *= dof
    xi, pxi = np.zeros(chain_length), np.zeros(chain_length)

    def wrap(y):
        return wrap_positions(y, cell, pbc)

    def evaluate(y):
        y32 = to_fp32_inside(y, cell)  # the neighbour predicate is specified in fp32 (R20); E and F use the fp64 y
        return energy_forces(model, y, species, cell, auto_neighbors(y32, cell, pbc, model.r_cut))

    def ke2():
        return float((m * v * v).sum() / ACC)

    def conserved(ep):
        return ep + 0.5 * ke2() + float((pxi ** 2 / (2 * Q)).sum()) + dof * kT * xi[0] + kT * float(xi[1:].sum())

    x = wrap(x)
    r = evaluate(x)
    epot, ekin, cons = [r.energy], [0.5 * ke2()], [conserved(r.energy)]
    for n in range(n_steps):
        kT = KB_EV * schedule_temperature(schedule, n, temperature)
        v *= nhc_half_step(ke2(), xi, pxi, Q, dof, kT, dt_fs, chain_steps, sy_steps)
        v += 0.5 * dt_fs * r.forces / m * ACC
        x = wrap(x + dt_fs * v)
        r = evaluate(x)
        v += 0.5 * dt_fs * r.forces / m * ACC
        v *= nhc_half_step(ke2(), xi, pxi, Q, dof, kT, dt_fs, chain_steps, sy_steps)
        epot.append(r.energy)
        ekin.append(0.5 * ke2())
        cons.append(conserved(r.energy))
    return x, v, np.array(epot), np.array(ekin), np.array(cons)


def _splitmix64(seed: int, counters: np.ndarray) -> np.ndarray:
    """Counter-based generator: output number `counter` (0-based) of the splitmix64 sequence started at `seed`."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (counters.astype(np.uint64) + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def langevin_normals(seed: int, step: int, n_atoms: int) -> np.ndarray:
    """O-15a: the standard normals xi [N][3] of MD step `step` (reading R29).  Atom i takes the two 64-bit words
    with counters (step N + i) 2 + {0, 1}; their four 32-bit halves (low first) give u = (h + 1) 2^-32 in (0, 1];
    Box-Muller: xi_x, xi_y = sqrt(-2 ln u1) (cos, sin)(2 pi u2), xi_z = sqrt(-2 ln u3) cos(2 pi u4)."""
    base = (np.uint64(step) * np.uint64(n_atoms) + np.arange(n_atoms, dtype=np.uint64)) * np.uint64(2)
    w0, w1 = _splitmix64(seed, base), _splitmix64(seed, base + np.uint64(1))
    lo, hi = np.uint64(0xFFFFFFFF), np.uint64(32)
    u = [((h.astype(np.float64)) + 1.0) * 2.0 ** -32 for h in (w0 & lo, w0 >> hi, w1 & lo, w1 >> hi)]
    r1, r2 = np.sqrt(-2.0 * np.log(u[0])), np.sqrt(-2.0 * np.log(u[2]))
    return np.stack([r1 * np.cos(2 * np.pi * u[1]), r1 * np.sin(2 * np.pi * u[1]), r2 * np.cos(2 * np.pi * u[3])], 1)


def nvt_langevin(model: Model, positions, velocities, masses, species, cell, pbc, dt_fs: float, n_steps: int,
                 temperature: float, gamma_per_fs: float, seed: int, first_step: int = 0, schedule=None):
    """O-15: Langevin dynamics ("Langevin thermostat") in the BAOAB splitting (reading R29):
    v += dt/2 a;  x += dt/2 v;  v = c1 v + sqrt(kT (1 - c1^2) / m) xi, c1 = exp(-gamma dt);  x += dt/2 v;
    forces;  v += dt/2 a.  Fresh list of radius r_cut every step.  Returns x, v, epot, ekin ([n_steps + 1]).
    With a `schedule` (O-19) the noise of MD step n takes kT = k_B T(n)."""
    ACC = 9.648533212e-3
    x = _f64(positions).copy()
    v = _f64(velocities).copy()
    m = _f64(masses)[:, None]
    N = x.shape[0]
    kT = KB_EV * temperature
    c1 = np.exp(-gamma_per_fs * dt_fs)

    def wrap(y):
        return wrap_positions(y, cell, pbc)

    def evaluate(y):
        y32 = to_fp32_inside(y, cell)  # the neighbour predicate is specified in fp32 (R20); E and F use the fp64 y
        return energy_forces(model, y, species, cell, auto_neighbors(y32, cell, pbc, model.r_cut))

    x = wrap(x)
    r = evaluate(x)
    epot, ekin = [r.energy], [0.5 * float((m * v * v).sum()) / ACC]
    for t in range(n_steps):
        v += 0.5 * dt_fs * r.forces / m * ACC
        x = x + 0.5 * dt_fs * v
        kT = KB_EV * schedule_temperature(schedule, t, temperature)
        c2 = np.sqrt(kT * (1.0 - c1 * c1) / m * ACC)  # Ang/fs
        v = c1 * v + c2 * langevin_normals(seed, first_step + t, N)
        x = wrap(x + 0.5 * dt_fs * v)
        r = evaluate(x)
        v += 0.5 * dt_fs * r.forces / m * ACC
        epot.append(r.energy)
        ekin.append(0.5 * float((m * v * v).sum()) / ACC)
    return x, v, np.array(epot), np.array(ekin)
