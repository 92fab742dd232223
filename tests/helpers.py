"""Shared test glue: workload -> oracle parameters, error norms."""
import numpy as np

import oracle as O


def oracle_params(w) -> O.Params:
    return O.Params(w.cell[0], w.cell[1], w.cell[2], w.nx, w.ny, w.n_slices, w.dz, w.voltage,
                    w.alpha, w.defocus, w.cs, w.f, w.det_step, w.det_max, tuple(w.aberrations))


def oracle_potential(w, phonon=0):
    lut_z, r_cut, lut_v = w.lut()
    return O.potential(oracle_params(w), w.atoms_for_phonon(phonon), w.z, lut_z, r_cut, lut_v)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128 if np.iscomplexobj(a) or np.iscomplexobj(b) else np.float64)
    b = np.asarray(b, dtype=a.dtype)
    den = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0))


def freq(n):
    """signed frequency index of each array slot (k in [-n/2, n/2))."""
    m = np.arange(n)
    return np.where(m < n // 2, m, m - n)
