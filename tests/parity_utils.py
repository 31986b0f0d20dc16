"""Helpers shared by the GPU parity tests: tolerances of DESIGN.md section 6 and the map between the
oracle's full tensors (1+3+9+27 per channel) and the CUDA path's symmetry-unique storage (20)."""
import numpy as np

E_ATOM_RTOL = 1e-5  # north_star: per-atom energies within 1e-5 relative (fp32 path)
F_TOL = 1e-4  # north_star: max |dF| / RMS(F) <= 1e-4 (fp32 path)
F_TOL_REDUCED = 2e-3  # reduced-precision MLP variant
E_TOTAL_RTOL = 1e-6  # total E against sum |E_i| (reading R21)

_T3 = [(0, 0, 0), (0, 0, 1), (0, 0, 2), (0, 1, 1), (0, 1, 2), (0, 2, 2), (1, 1, 1), (1, 1, 2), (1, 2, 2), (2, 2, 2)]


def idx2(a, b):
    lo, hi = min(a, b), max(a, b)
    return hi if lo == 0 else (2 + hi if lo == 1 else 5)


def idx3(a, b, c):
    return _T3.index(tuple(sorted((a, b, c))))


def unique_from_full(P, summed):
    """[N][n_r][40] -> [N][n_r][20].  summed=False: pick the (symmetric) component (moments);
    summed=True: add every full index that maps to the unique one (adjoints dE/dPsi)."""
    N, nr = P.shape[0], P.shape[1]
    U = np.zeros((N, nr, 20))
    U[:, :, 0] = P[:, :, 0]
    U[:, :, 1:4] = P[:, :, 1:4]
    for a in range(3):
        for b in range(3):
            if summed:
                U[:, :, 4 + idx2(a, b)] += P[:, :, 4 + 3 * a + b]
            else:
                U[:, :, 4 + idx2(a, b)] = P[:, :, 4 + 3 * a + b]
            for c in range(3):
                if summed:
                    U[:, :, 10 + idx3(a, b, c)] += P[:, :, 13 + 9 * a + 3 * b + c]
                else:
                    U[:, :, 10 + idx3(a, b, c)] = P[:, :, 13 + 9 * a + 3 * b + c]
    return U


def energy_atom_error(e_gpu, e_ref):
    """max_i |dE_i| / (1e-5 max(|E_i^ref|, mean |E^ref|)): <= 1 passes (reading R21)."""
    tol = E_ATOM_RTOL * np.maximum(np.abs(e_ref), np.abs(e_ref).mean())
    return float((np.abs(e_gpu - e_ref) / tol).max())


def force_error(f_gpu, f_ref):
    """max |dF| / sqrt(sum F_ref^2 / 3N)."""
    return float(np.abs(f_gpu - f_ref).max() / np.sqrt((f_ref ** 2).mean()))


def r_list32(r_cut, skin):
    """fl32(fl32(r_cut) + fl32(skin)): the list radius both sides use (reading R20)."""
    return float(np.float32(r_cut) + np.float32(skin))
