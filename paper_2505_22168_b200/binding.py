"""Thin ctypes binding of libgmnn_b200.so (include/gmnn.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch supplies device memory and
the stream.  There is no fallback: if the shared object is missing the import of this module
fails, and without a CUDA device every compute call raises GmnnError(GMNN_CUDA_ERROR).

Method names follow the C entry points (gmnn_build_neighbors -> System.build_neighbors, ...).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("GMNN_B200_LIB") or os.path.join(_HERE, "libgmnn_b200.so")

GMNN_OK = 0
GMNN_INVALID_ARG = -1
GMNN_UNSUPPORTED = -2
GMNN_NEIGHBOR_OVERFLOW = -3
GMNN_STALE_NEIGHBORS = -4
GMNN_CUDA_ERROR = -5
GMNN_OOM = -6
GMNN_OUT_OF_BOX = -7
GMNN_MLP_FP32, GMNN_MLP_3XTF32, GMNN_MLP_TF32, GMNN_MLP_3XF16 = 0, 1, 2, 3
GMNN_FORCE_GATHER, GMNN_FORCE_PAIRBUF = 0, 1

EXPORTS = (
    "gmnn_n_features", "gmnn_create", "gmnn_destroy", "gmnn_system_create", "gmnn_system_destroy",
    "gmnn_system_set_int", "gmnn_system_get_int", "gmnn_build_neighbors", "gmnn_get_neighbors", "gmnn_get_neighbor_rows",
    "gmnn_energy_forces", "gmnn_energy_forces_virial", "gmnn_energy_forces_host", "gmnn_ensemble_energy_forces", "gmnn_md_verlet_steps", "gmnn_md_ensemble_steps", "gmnn_system_set_langevin", "gmnn_system_set_temperature_schedule", "gmnn_system_set_nose_hoover", "gmnn_system_get_nose_hoover", "gmnn_system_set_udd_bias", "gmnn_system_get_udd_bias",
    "gmnn_check", "gmnn_measure_fp32_peak", "gmnn_sum_energies_static", "gmnn_stage_times", "gmnn_debug_read", "gmnn_launch_count", "gmnn_last_error",
)


class GmnnError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__("gmnn status %d: %s" % (code, message))
        self.code = code


class _HParams(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32), ("n_basis", C.c_int32), ("n_radial", C.c_int32), ("l_max", C.c_int32),
        ("r_cut", C.c_float), ("r_min", C.c_float), ("gauss_gamma", C.c_float),
        ("n_hidden", C.c_int32), ("hidden", C.c_int32 * 4), ("n_heads", C.c_int32),
        ("n_weight_sets", C.c_int32), ("mlp_precision", C.c_int32), ("force_mode", C.c_int32),
        ("radial_basis", C.c_int32), ("zbl", C.c_int32), ("zbl_r_max", C.c_float), ("zbl_scale", C.c_float),
    ]


class _Weights(C.Structure):
    _fields_ = [("beta", C.c_void_p), ("W", C.c_void_p * 5), ("b", C.c_void_p * 5),
                ("scale", C.c_void_p), ("shift", C.c_void_p), ("atomic_numbers", C.c_void_p)]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        try:  # build in-tree (nvcc cross-compiles sm_100a); never a fallback to other code
            from . import build as _build

            _build.build()
        except Exception:
            pass
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "%s is missing: build it with `python -m paper_2505_22168_b200.build` (nvcc, sm_100a). "
            "There is no CPU fallback." % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    lib.gmnn_last_error.restype = C.c_char_p
    lib.gmnn_launch_count.restype = C.c_int64
    lib.gmnn_n_features.restype = C.c_int32
    lib.gmnn_build_neighbors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p]
    lib.gmnn_md_verlet_steps.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_int32,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.gmnn_md_ensemble_steps.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_int32, C.c_int32,
                                           C.c_float] + [C.c_void_p] * 9
    lib.gmnn_system_set_langevin.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_uint64, C.c_uint64]
    lib.gmnn_system_set_nose_hoover.argtypes = [C.c_void_p, C.c_float, C.c_float, C.c_int32, C.c_int32, C.c_int32]
    lib.gmnn_system_get_nose_hoover.argtypes = [C.c_void_p] * 5
    lib.gmnn_system_set_udd_bias.argtypes = [C.c_void_p, C.c_float, C.c_float]
    lib.gmnn_system_set_temperature_schedule.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.gmnn_system_get_udd_bias.argtypes = [C.c_void_p] * 4
    lib.gmnn_energy_forces.argtypes = [C.c_void_p] * 6
    lib.gmnn_energy_forces_host.argtypes = [C.c_void_p] * 6
    lib.gmnn_energy_forces_virial.argtypes = [C.c_void_p] * 7
    lib.gmnn_ensemble_energy_forces.argtypes = [C.c_void_p] * 7
    lib.gmnn_system_create.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.gmnn_system_destroy.argtypes = [C.c_void_p]
    lib.gmnn_destroy.argtypes = [C.c_void_p]
    lib.gmnn_system_set_int.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
    lib.gmnn_system_get_int.argtypes = [C.c_void_p, C.c_char_p, C.c_void_p]
    lib.gmnn_get_neighbors.argtypes = [C.c_void_p] * 5
    lib.gmnn_get_neighbor_rows.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 5
    lib.gmnn_check.argtypes = [C.c_void_p, C.c_void_p]
    lib.gmnn_stage_times.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.gmnn_debug_read.argtypes = [C.c_void_p, C.c_char_p, C.c_void_p, C.c_int64]
    return lib


lib = _load()


def _check(rc: int) -> None:
    if rc != GMNN_OK:
        raise GmnnError(rc, (lib.gmnn_last_error() or b"").decode())


def measure_fp32_peak(stream=None) -> float:
    """TFLOP/s of fp32 FMA the current device sustains now (gmnn_measure_fp32_peak)."""
    v = C.c_double(0)
    _check(lib.gmnn_measure_fp32_peak(C.byref(v), _stream_ptr(stream)))
    return float(v.value)


STATIC_SUM_MAX_ATOMS = 16777216  # GMNN_STATIC_SUM_MAX_ATOMS of include/gmnn.h


def sum_energies_static(e_atom, energy_out, n_atoms: Optional[int] = None, stream=None) -> None:
    """energy_out[0] (device float64) = sum of e_atom (device float32 [n]) through gmnn_sum_energies_static: no
    allocation on the call path (the output tensor is the caller's); n_atoms <= STATIC_SUM_MAX_ATOMS."""
    import torch

    n = int(e_atom.numel()) if n_atoms is None else int(n_atoms)
    if n_atoms is None:
        _dev_ptr(e_atom, torch.float32, (n,))  # dtype / device / contiguity checks
    _check(lib.gmnn_sum_energies_static(C.c_void_p(e_atom.data_ptr()), C.c_int64(n), _dev_ptr(energy_out, torch.float64, (1,)),
                                        _stream_ptr(stream)))


def launch_count() -> int:
    return int(lib.gmnn_launch_count())


def n_features(n_radial: int) -> int:
    return int(lib.gmnn_n_features(C.c_int32(n_radial)))


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dev_ptr(t, dtype, shape=None):
    """data_ptr of a contiguous CUDA tensor of the given torch dtype (None passes through)."""
    if t is None:
        return None
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError("expected shape %s, got %s" % (tuple(shape), tuple(t.shape)))
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream=None):
    import torch

    st = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(st.cuda_stream)


class Model:
    """gmnn_create / gmnn_destroy.  `spec` is any object with the attributes of
    workloads.ModelSpec (host numpy arrays); weights are copied to the current CUDA device."""

    def __init__(self, spec, mlp_precision: int = GMNN_MLP_FP32, force_mode: int = GMNN_FORCE_GATHER,
                 n_weight_sets: Optional[int] = None, l_max: int = 3):
        if n_weight_sets is None:  # 1: one NN for all species; n_species: W[l] is [S][fan_in][fan_out], b[l] [S][fan_out]
            n_weight_sets = int(getattr(spec, "n_weight_sets", 1))
        dims = [n_features(spec.n_radial), *[int(h) for h in spec.hidden], int(spec.n_heads)]
        for l in range(min(len(spec.W), 5)):  # the library reads n_weight_sets x fan_in x fan_out floats per layer
            if n_weight_sets >= 1 and (np.asarray(spec.W[l]).size != n_weight_sets * dims[l] * dims[l + 1]
                                       or np.asarray(spec.b[l]).size != n_weight_sets * dims[l + 1]):
                raise ValueError("layer %d: weights do not hold %d set(s) of [%d][%d]" % (l, n_weight_sets, dims[l], dims[l + 1]))
        hp = _HParams()
        hp.n_species, hp.n_basis, hp.n_radial, hp.l_max = spec.n_species, spec.n_basis, spec.n_radial, l_max
        hp.r_cut, hp.r_min, hp.gauss_gamma = spec.r_cut, spec.r_min, spec.gamma
        self.hidden = tuple(int(h) for h in spec.hidden)
        hp.n_hidden = len(spec.hidden)
        for l, h in enumerate(spec.hidden[:4]):
            hp.hidden[l] = int(h)
        hp.n_heads = spec.n_heads
        hp.n_weight_sets, hp.mlp_precision, hp.force_mode = n_weight_sets, mlp_precision, force_mode
        hp.radial_basis = int(getattr(spec, "basis_kind", 0))  # 0 Gaussians, 1 Bessel-like
        hp.zbl = int(bool(getattr(spec, "zbl", False)))  # ZBL repulsion
        hp.zbl_r_max, hp.zbl_scale = float(getattr(spec, "zbl_r_max", 0.0)), float(getattr(spec, "zbl_scale", 1.0))
        self._keep = [np.ascontiguousarray(spec.beta, np.float32), np.ascontiguousarray(spec.scale, np.float32),
                      np.ascontiguousarray(spec.shift, np.float32)]
        w = _Weights()
        w.beta, w.scale, w.shift = (a.ctypes.data for a in self._keep)
        if getattr(spec, "atomic_numbers", None) is not None:
            zn = np.ascontiguousarray(spec.atomic_numbers, np.float32)
            self._keep.append(zn)
            w.atomic_numbers = zn.ctypes.data
        for l in range(min(len(spec.W), 5)):
            Wl = np.ascontiguousarray(spec.W[l], np.float32)
            bl = np.ascontiguousarray(spec.b[l], np.float32)
            self._keep += [Wl, bl]
            w.W[l], w.b[l] = Wl.ctypes.data, bl.ctypes.data
        self.handle = C.c_void_p()
        self.n_species, self.n_heads, self.n_radial = spec.n_species, spec.n_heads, spec.n_radial
        self.n_features = n_features(spec.n_radial)
        self.r_cut = float(spec.r_cut)
        _check(lib.gmnn_create(C.byref(hp), C.byref(w), C.byref(self.handle)))

    def destroy(self):
        if getattr(self, "handle", None):
            lib.gmnn_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class System:
    """gmnn_system_* and every per-system call.  Tensors are torch CUDA tensors unless a method
    says HOST."""

    def __init__(self, model: Model, species: Sequence[int]):
        sp = np.ascontiguousarray(np.asarray(species), np.int32)
        self.model = model
        self.n_atoms = int(sp.shape[0])
        self.handle = C.c_void_p()
        _check(lib.gmnn_system_create(model.handle, C.c_int64(self.n_atoms), _np_ptr(sp), C.byref(self.handle)))

    def destroy(self):
        if getattr(self, "handle", None):
            lib.gmnn_system_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # -- knobs
    def set_int(self, key: str, value: int) -> None:
        _check(lib.gmnn_system_set_int(self.handle, key.encode(), C.c_int64(value)))

    def get_int(self, key: str) -> int:
        v = C.c_int64(0)
        _check(lib.gmnn_system_get_int(self.handle, key.encode(), C.byref(v)))
        return int(v.value)

    # -- neighbours
    def build_neighbors(self, positions, cell9, pbc, r_cut: float, skin: float, stream=None) -> None:
        import torch

        cell = np.ascontiguousarray(np.asarray(cell9, np.float32).reshape(9))
        pb = np.ascontiguousarray(np.asarray(pbc, np.int32).reshape(3))
        _check(lib.gmnn_build_neighbors(self.handle, _dev_ptr(positions, torch.float32, (self.n_atoms, 3)),
                                        _np_ptr(cell), _np_ptr(pb), C.c_float(r_cut), C.c_float(skin),
                                        _stream_ptr(stream)))

    def get_neighbors(self) -> np.ndarray:
        """HOST [n_pairs][5] int32 rows (i, j, nx, ny, nz), sorted."""
        n = C.c_int64(0)
        _check(lib.gmnn_get_neighbors(self.handle, C.byref(n), None, None, None))
        oi = np.empty(n.value, np.int32)
        oj = np.empty(n.value, np.int32)
        on = np.empty((n.value, 3), np.int32)
        _check(lib.gmnn_get_neighbors(self.handle, C.byref(n), _np_ptr(oi), _np_ptr(oj), _np_ptr(on)))
        return np.concatenate([oi[:, None], oj[:, None], on], axis=1)

    def get_neighbor_rows(self, atoms) -> np.ndarray:
        """HOST [n_pairs][5] int32 rows (i, j, nx, ny, nz), sorted, of the chosen atoms (caller indices) only."""
        sel = np.ascontiguousarray(np.asarray(atoms), np.int32)
        n = C.c_int64(0)
        _check(lib.gmnn_get_neighbor_rows(self.handle, C.c_int64(sel.shape[0]), _np_ptr(sel), C.byref(n), None, None, None))
        oi = np.empty(n.value, np.int32)
        oj = np.empty(n.value, np.int32)
        on = np.empty((n.value, 3), np.int32)
        _check(lib.gmnn_get_neighbor_rows(self.handle, C.c_int64(sel.shape[0]), _np_ptr(sel), C.byref(n), _np_ptr(oi),
                                          _np_ptr(oj), _np_ptr(on)))
        return np.concatenate([oi[:, None], oj[:, None], on], axis=1)

    # -- energy and forces
    def energy_forces(self, positions, energy=None, energy_per_atom=None, forces=None, stream=None,
                      want_per_atom: bool = True):
        """Returns (energy f64[1], energy_per_atom f32[N] or None, forces f32[N][3]), all on device."""
        import torch

        dev = positions.device
        if energy is None:
            energy = torch.empty(1, dtype=torch.float64, device=dev)
        if energy_per_atom is None and want_per_atom:
            energy_per_atom = torch.empty(self.n_atoms, dtype=torch.float32, device=dev)
        if forces is None:
            forces = torch.empty(self.n_atoms, 3, dtype=torch.float32, device=dev)
        _check(lib.gmnn_energy_forces(self.handle, _dev_ptr(positions, torch.float32, (self.n_atoms, 3)),
                                      _dev_ptr(energy, torch.float64), _dev_ptr(energy_per_atom, torch.float32),
                                      _dev_ptr(forces, torch.float32, (self.n_atoms, 3)), _stream_ptr(stream)))
        return energy, energy_per_atom, forces

    def energy_forces_virial(self, positions, stream=None):
        """Returns (energy f64[1], energy_per_atom f32[N], forces f32[N][3], virial f64[3][3] = -dE/d strain), on device."""
        import torch

        dev, N = positions.device, self.n_atoms
        energy = torch.empty(1, dtype=torch.float64, device=dev)
        e_atom = torch.empty(N, dtype=torch.float32, device=dev)
        forces = torch.empty(N, 3, dtype=torch.float32, device=dev)
        virial = torch.empty(3, 3, dtype=torch.float64, device=dev)
        _check(lib.gmnn_energy_forces_virial(self.handle, _dev_ptr(positions, torch.float32, (N, 3)),
                                             _dev_ptr(energy, torch.float64), _dev_ptr(e_atom, torch.float32),
                                             _dev_ptr(forces, torch.float32, (N, 3)), _dev_ptr(virial, torch.float64),
                                             _stream_ptr(stream)))
        return energy, e_atom, forces, virial

    def energy_forces_host(self, positions: np.ndarray, forces: np.ndarray, energy_per_atom: Optional[np.ndarray] = None,
                           stream=None) -> float:
        """HOST numpy buffers (pinned recommended): copies in, computes, copies out, synchronises."""
        assert positions.dtype == np.float32 and positions.flags.c_contiguous and positions.shape == (self.n_atoms, 3)
        assert forces.dtype == np.float32 and forces.flags.c_contiguous and forces.shape == (self.n_atoms, 3)
        e = np.zeros(1, np.float64)
        _check(lib.gmnn_energy_forces_host(self.handle, _np_ptr(positions), _np_ptr(e),
                                           None if energy_per_atom is None else _np_ptr(energy_per_atom),
                                           _np_ptr(forces), _stream_ptr(stream)))
        return float(e[0])

    def ensemble_energy_forces(self, positions, stream=None):
        """Returns (e_mean[N], e_var[N], f_mean[N][3], f_var[N][3]) on device."""
        import torch

        dev = positions.device
        N = self.n_atoms
        e_mean = torch.empty(N, dtype=torch.float32, device=dev)
        e_var = torch.empty(N, dtype=torch.float32, device=dev)
        f_mean = torch.empty(N, 3, dtype=torch.float32, device=dev)
        f_var = torch.empty(N, 3, dtype=torch.float32, device=dev)
        _check(lib.gmnn_ensemble_energy_forces(self.handle, _dev_ptr(positions, torch.float32, (N, 3)),
                                               _dev_ptr(e_mean, torch.float32), _dev_ptr(e_var, torch.float32),
                                               _dev_ptr(f_mean, torch.float32), _dev_ptr(f_var, torch.float32),
                                               _stream_ptr(stream)))
        return e_mean, e_var, f_mean, f_var

    def md_verlet_steps(self, positions, velocities, masses, dt_fs: float, n_steps: int, want_series: bool = True,
                        stream=None) -> Tuple[Optional["object"], Optional["object"], int]:
        """In-place NVE; returns (epot[n_steps+1] f64, ekin[n_steps+1] f64, n_rebuilds)."""
        import torch

        N = self.n_atoms
        dev = positions.device
        epot = torch.zeros(n_steps + 1, dtype=torch.float64, device=dev) if want_series else None
        ekin = torch.zeros(n_steps + 1, dtype=torch.float64, device=dev) if want_series else None
        nreb = C.c_int32(0)
        _check(lib.gmnn_md_verlet_steps(self.handle, _dev_ptr(positions, torch.float32, (N, 3)),
                                        _dev_ptr(velocities, torch.float32, (N, 3)), _dev_ptr(masses, torch.float32, (N,)),
                                        C.c_float(dt_fs), C.c_int32(n_steps), _dev_ptr(epot, torch.float64),
                                        _dev_ptr(ekin, torch.float64), C.cast(C.byref(nreb), C.c_void_p),
                                        _stream_ptr(stream)))
        return epot, ekin, int(nreb.value)

    def md_ensemble_steps(self, positions, velocities, masses, dt_fs: float, n_steps: int, sampling_rate: int,
                          f_sigma_stop: float = 0.0, want_f_var: bool = False, stream=None):
        """In-place switching-mode ensemble MD; returns a dict: epot, ekin (f64 device, [n_steps_done + 1]),
        sigma_e, sigma_f_max (numpy f64 [n_samples]), f_var (device [N][3] or None), n_steps_done, n_rebuilds."""
        import torch

        N = self.n_atoms
        dev = positions.device
        epot = torch.zeros(n_steps + 1, dtype=torch.float64, device=dev)
        ekin = torch.zeros(n_steps + 1, dtype=torch.float64, device=dev)
        cap = max(n_steps // max(sampling_rate, 1), 1)
        se = np.zeros(cap, np.float64)
        sf = np.zeros(cap, np.float64)
        fvar = torch.zeros((N, 3), dtype=torch.float32, device=dev) if want_f_var else None
        done, nsamp, nreb = C.c_int32(0), C.c_int32(0), C.c_int32(0)
        _check(lib.gmnn_md_ensemble_steps(
            self.handle, _dev_ptr(positions, torch.float32, (N, 3)), _dev_ptr(velocities, torch.float32, (N, 3)),
            _dev_ptr(masses, torch.float32, (N,)), C.c_float(dt_fs), C.c_int32(n_steps), C.c_int32(sampling_rate),
            C.c_float(f_sigma_stop), _dev_ptr(epot, torch.float64), _dev_ptr(ekin, torch.float64),
            se.ctypes.data_as(C.c_void_p), sf.ctypes.data_as(C.c_void_p), _dev_ptr(fvar, torch.float32),
            C.cast(C.byref(done), C.c_void_p), C.cast(C.byref(nsamp), C.c_void_p), C.cast(C.byref(nreb), C.c_void_p),
            _stream_ptr(stream)))
        d, k = int(done.value), int(nsamp.value)
        return {"epot": epot[:d + 1], "ekin": ekin[:d + 1], "sigma_e": se[:k], "sigma_f_max": sf[:k], "f_var": fvar,
                "n_steps_done": d, "n_rebuilds": int(nreb.value)}

    def set_nose_hoover(self, temperature_K: float, tau_fs: float = 50.0, chain_length: int = 3, chain_steps: int = 2,
                        sy_steps: int = 3) -> None:
        """NVT for the MD entries (temperature_K <= 0: back to NVE); resets the chain."""
        _check(lib.gmnn_system_set_nose_hoover(self.handle, C.c_float(temperature_K), C.c_float(tau_fs),
                                               C.c_int32(chain_length), C.c_int32(chain_steps), C.c_int32(sy_steps)))
        self._nhc_len = chain_length if temperature_K > 0 else 0

    def get_nose_hoover(self, stream=None):
        """(xi[chain_length], p_xi[chain_length], thermostat energy in eV)."""
        n = getattr(self, "_nhc_len", 0)
        xi, pxi = np.zeros(max(n, 1)), np.zeros(max(n, 1))
        et = C.c_double(0)
        _check(lib.gmnn_system_get_nose_hoover(self.handle, xi.ctypes.data_as(C.c_void_p), pxi.ctypes.data_as(C.c_void_p),
                                               C.cast(C.byref(et), C.c_void_p), _stream_ptr(stream)))
        return xi[:n], pxi[:n], float(et.value)

    def set_langevin(self, temperature_K: float, gamma_per_fs: float = 0.01, seed: int = 0, first_step: int = 0) -> None:
        """Langevin (BAOAB) for the MD entries (temperature_K <= 0: off)."""
        _check(lib.gmnn_system_set_langevin(self.handle, C.c_float(temperature_K), C.c_float(gamma_per_fs),
                                            C.c_uint64(seed), C.c_uint64(first_step)))

    def set_temperature_schedule(self, steps=(), temperatures_K=()) -> None:
        """Piecewise-linear target temperature over the MD step count for the thermostat that is set (empty: none)."""
        st = np.ascontiguousarray(np.asarray(steps), np.int64)
        tk = np.ascontiguousarray(np.asarray(temperatures_K), np.float32)
        assert st.shape == tk.shape and st.ndim == 1
        _check(lib.gmnn_system_set_temperature_schedule(self.handle, C.c_int32(st.shape[0]), _np_ptr(st), _np_ptr(tk)))

    def set_udd_bias(self, A: float, B: float = 1.0) -> None:
        _check(lib.gmnn_system_set_udd_bias(self.handle, C.c_float(A), C.c_float(B)))

    def get_udd_bias(self, stream=None) -> Tuple[float, float]:
        """(E_b, sigma_E^2) of the latest biased evaluation."""
        eb, var = C.c_double(0), C.c_double(0)
        _check(lib.gmnn_system_get_udd_bias(self.handle, C.cast(C.byref(eb), C.c_void_p),
                                            C.cast(C.byref(var), C.c_void_p), _stream_ptr(stream)))
        return float(eb.value), float(var.value)

    def check(self, stream=None) -> None:
        _check(lib.gmnn_check(self.handle, _stream_ptr(stream)))

    def stage_times(self):
        """[(stage name, mean ms per occurrence, occurrences)] since set_int('profile', 1)."""
        names = (C.c_char_p * 64)()
        ms = (C.c_float * 64)()
        cnt = (C.c_int32 * 64)()
        n = lib.gmnn_stage_times(self.handle, C.c_int32(64), names, ms, cnt)
        if n < 0:
            _check(n)
        return [(names[k].decode(), float(ms[k]), int(cnt[k])) for k in range(n)]

    def debug_read(self, name: str) -> np.ndarray:
        N, m = self.n_atoms, self.model
        shapes = {
            "perm": ((N,), np.int32), "count": ((N,), np.int32), "xref": ((N, 3), np.float32),
            "psi": ((N, m.n_radial, 20), np.float32), "A": ((N, m.n_radial, 20), np.float32),
            "G": ((N, m.n_features), np.float32), "dG": ((N, m.n_features), np.float32),
            "e_heads": ((N, m.n_heads), np.float32),
            "H0": ((N, m.hidden[0]), np.float32), "D0": ((N, m.hidden[0]), np.float32),
        }
        shape, dt = shapes[name]
        out = np.empty(shape, dt)
        _check(lib.gmnn_debug_read(self.handle, name.encode(), _np_ptr(out), C.c_int64(out.nbytes)))
        return out
