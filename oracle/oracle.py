"""ctypes front end of ``prism_oracle.c`` -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; all arithmetic is in the C file, each function there
citing the passage of PAPER.md it follows.  ``build()`` compiles the C with gcc
(-O2, OpenMP over independent beams / probes).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "prism_oracle.c")
_HDR = os.path.join(_HERE, "prism_oracle.h")
_LIB = os.path.join(_HERE, "libprism_oracle.so")

__all__ = [
    "Params", "build", "constants", "dft_naive", "fft", "fft2", "dft2_naive",
    "potential", "transmission", "propagator", "slice_step", "multislice_wave",
    "num_aperture", "probe", "num_bins", "bin_intensity", "multislice_probe",
    "beams", "smatrix_layer", "smatrix", "prism_probe", "prism_probe_rows", "multislice_probes",
    "prism_probes", "num_threads",
]


class _CAberration(C.Structure):
    _fields_ = [("n", C.c_int32), ("m", C.c_int32), ("c", C.c_double), ("angle", C.c_double)]


class _CParams(C.Structure):
    _fields_ = [
        ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
        ("nx", C.c_int32), ("ny", C.c_int32), ("n_slices", C.c_int32),
        ("dz", C.c_double), ("voltage", C.c_double), ("alpha", C.c_double),
        ("defocus", C.c_double), ("cs", C.c_double), ("f", C.c_int32),
        ("det_step", C.c_double), ("det_max", C.c_double),
        ("n_aberr", C.c_int32), ("aberr", C.POINTER(_CAberration)),
    ]


@dataclass
class Params:
    """The paper's knobs (cell, grid, slices, voltage, semi-angle, f, detector)."""
    lx: float
    ly: float
    lz: float
    nx: int
    ny: int
    n_slices: int
    dz: float
    voltage: float
    alpha: float
    defocus: float = 0.0
    cs: float = 0.0
    f: int = 1
    det_step: float = 1e-3
    det_max: float = 0.1
    aberrations: tuple = ()     # further terms (n, m, c [Angstrom], angle [rad]) of the aberration function (R5b)

    def c(self) -> _CParams:
        cp = _CParams(self.lx, self.ly, self.lz, self.nx, self.ny, self.n_slices,
                      self.dz, self.voltage, self.alpha, self.defocus, self.cs,
                      self.f, self.det_step, self.det_max, 0, None)
        if self.aberrations:
            arr = (_CAberration * len(self.aberrations))(*[_CAberration(int(n), int(m), float(c), float(a))
                                                           for n, m, c, a in self.aberrations])
            cp.n_aberr, cp.aberr = len(self.aberrations), arr
            cp._keep = arr                      # the array must outlive the call
        return cp


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the shared object is missing or stale."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared",
                               "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.orc_num_aperture.restype = C.c_int
        lib.orc_num_bins.restype = C.c_int
        lib.orc_beams.restype = C.c_int
        lib.orc_potential.restype = C.c_int
        lib.orc_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_L().orc_num_threads())


def constants(voltage: float):
    lam, sig = C.c_double(), C.c_double()
    _L().orc_constants(C.c_double(voltage), C.byref(lam), C.byref(sig))
    return lam.value, sig.value


def dft_naive(x, sign: int):
    x = _c128(x)
    out = np.empty_like(x)
    _L().orc_dft_naive(_p(x), _p(out), C.c_int(x.size), C.c_int(sign))
    return out


def fft(x, sign: int):
    x = _c128(x).copy()
    _L().orc_fft(_p(x), C.c_int(x.size), C.c_int(sign))
    return x


def fft2(a, sign: int):
    a = _c128(a).copy()
    _L().orc_fft2(_p(a), C.c_int(a.shape[0]), C.c_int(a.shape[1]), C.c_int(sign))
    return a


def dft2_naive(a, sign: int):
    a = _c128(a).copy()
    _L().orc_dft2_naive(_p(a), C.c_int(a.shape[0]), C.c_int(a.shape[1]), C.c_int(sign))
    return a


def potential(p: Params, atoms_xyz, z, lut_z, r_cut: float, lut_v):
    """V[s][y][x] fp64.  lut_v[n_luts][lut_n] sampled on [0, r_cut]."""
    atoms_xyz = _f64(atoms_xyz).reshape(-1, 3)
    z = np.ascontiguousarray(z, dtype=np.int32)
    lut_z = np.ascontiguousarray(lut_z, dtype=np.int32)
    lut_v = _f64(lut_v).reshape(len(lut_z), -1)
    v = np.empty((p.n_slices, p.ny, p.nx), dtype=np.float64)
    cp = p.c()
    rc = _L().orc_potential(C.byref(cp), _p(atoms_xyz), _p(z), C.c_int64(len(z)), _p(lut_z),
                            C.c_int32(len(lut_z)), C.c_int32(lut_v.shape[1]),
                            C.c_double(r_cut), _p(lut_v), _p(v))
    if rc != 0:
        raise ValueError(f"orc_potential failed with code {rc}")
    return v


def transmission(v_slice, sigma: float):
    v_slice = _f64(v_slice)
    t = np.empty(v_slice.shape, dtype=np.complex128)
    _L().orc_transmission(_p(v_slice), C.c_double(sigma), C.c_int64(v_slice.size), _p(t))
    return t


def propagator(p: Params, dz: float | None = None):
    prop = np.empty((p.ny, p.nx), dtype=np.complex128)
    cp = p.c()
    _L().orc_propagator(C.byref(cp), C.c_double(p.dz if dz is None else dz), _p(prop))
    return prop


def slice_step(psi, t, prop, use_naive: bool = False):
    psi = _c128(psi).copy()
    t, prop = _c128(t), _c128(prop)
    _L().orc_slice_step(_p(psi), _p(t), _p(prop), C.c_int(psi.shape[0]), C.c_int(psi.shape[1]),
                        C.c_int(int(use_naive)))
    return psi


def multislice_wave(p: Params, v, psi, use_naive: bool = False):
    v = _f64(v)
    psi = _c128(psi).copy()
    cp = p.c()
    _L().orc_multislice_wave(C.byref(cp), _p(v), _p(psi), C.c_int(int(use_naive)))
    return psi


def num_aperture(p: Params) -> int:
    cp = p.c()
    return int(_L().orc_num_aperture(C.byref(cp)))


def probe(p: Params, xp: float, yp: float):
    psi = np.empty((p.ny, p.nx), dtype=np.complex128)
    cp = p.c()
    _L().orc_probe(C.byref(cp), C.c_double(xp), C.c_double(yp), _p(psi))
    return psi


def num_bins(p: Params) -> int:
    cp = p.c()
    return int(_L().orc_num_bins(C.byref(cp)))


def bin_intensity(p: Params, intensity, fy: int = 1, fx: int = 1):
    intensity = _f64(intensity)
    out = np.empty(num_bins(p), dtype=np.float64)
    cp = p.c()
    _L().orc_bin_intensity(C.byref(cp), _p(intensity), C.c_int(intensity.shape[0]),
                           C.c_int(intensity.shape[1]), C.c_int(fy), C.c_int(fx), _p(out))
    return out


def multislice_probe(p: Params, v, xp: float, yp: float, use_naive: bool = False,
                     want_pattern: bool = False):
    v = _f64(v)
    out = np.empty(num_bins(p), dtype=np.float64)
    pat = np.empty((p.ny, p.nx), dtype=np.float64) if want_pattern else None
    cp = p.c()
    _L().orc_multislice_probe(C.byref(cp), _p(v), C.c_double(xp), C.c_double(yp), _p(out),
                              _p(pat) if want_pattern else None, C.c_int(int(use_naive)))
    return (out, pat) if want_pattern else out


def beams(p: Params):
    cp = p.c()
    n = int(_L().orc_beams(C.byref(cp), None, C.c_int(0)))
    out = np.empty((n, 2), dtype=np.int32)
    _L().orc_beams(C.byref(cp), _p(out), C.c_int(n))
    return out


def smatrix_layer(p: Params, v, kx: int, ky: int, use_naive: bool = False):
    v = _f64(v)
    layer = np.empty((p.ny, p.nx), dtype=np.complex128)
    cp = p.c()
    _L().orc_smatrix_layer(C.byref(cp), _p(v), C.c_int(kx), C.c_int(ky), _p(layer),
                           C.c_int(int(use_naive)))
    return layer


def smatrix(p: Params, v, beam_list, use_naive: bool = False):
    v = _f64(v)
    beam_list = np.ascontiguousarray(beam_list, dtype=np.int32).reshape(-1, 2)
    s = np.empty((len(beam_list), p.ny, p.nx), dtype=np.complex128)
    cp = p.c()
    _L().orc_smatrix(C.byref(cp), _p(v), _p(beam_list), C.c_int(len(beam_list)), _p(s),
                     C.c_int(int(use_naive)))
    return s


def prism_probe(p: Params, s, beam_list, xp: float, yp: float, use_naive: bool = False,
                want_pattern: bool = False):
    s = _c128(s)
    beam_list = np.ascontiguousarray(beam_list, dtype=np.int32).reshape(-1, 2)
    out = np.empty(num_bins(p), dtype=np.float64)
    pat = np.empty((p.ny // p.f, p.nx // p.f), dtype=np.float64) if want_pattern else None
    cp = p.c()
    _L().orc_prism_probe(C.byref(cp), _p(s), _p(beam_list), C.c_int(len(beam_list)),
                         C.c_double(xp), C.c_double(yp), _p(out),
                         _p(pat) if want_pattern else None, C.c_int(int(use_naive)))
    return (out, pat) if want_pattern else out


def prism_probe_rows(p: Params, s_rows, row0: int, beam_list, xp: float, yp: float,
                     want_pattern: bool = False):
    """``prism_probe`` when only pixel rows ``[row0, row0 + n_rows)`` (mod ny) of every layer are in memory:
    ``s_rows[b][r]`` = pixel row ``(row0 + r) % ny`` of layer b (storage only; same loop and arithmetic)."""
    s_rows = _c128(s_rows)
    beam_list = np.ascontiguousarray(beam_list, dtype=np.int32).reshape(-1, 2)
    assert s_rows.ndim == 3 and s_rows.shape[0] == len(beam_list) and s_rows.shape[2] == p.nx
    out = np.empty(num_bins(p), dtype=np.float64)
    pat = np.empty((p.ny // p.f, p.nx // p.f), dtype=np.float64) if want_pattern else None
    cp = p.c()
    rc = _L().orc_prism_probe_rows(C.byref(cp), _p(s_rows), C.c_int(int(row0)), C.c_int(s_rows.shape[1]),
                                   _p(beam_list), C.c_int(len(beam_list)), C.c_double(xp), C.c_double(yp),
                                   _p(out), _p(pat) if want_pattern else None, C.c_int(0))
    if rc != 0:
        raise ValueError("the probe's window leaves the band of rows")
    return (out, pat) if want_pattern else out


def multislice_probes(p: Params, v, xy):
    v = _f64(v)
    xy = _f64(xy).reshape(-1, 2)
    out = np.empty((len(xy), num_bins(p)), dtype=np.float64)
    cp = p.c()
    _L().orc_multislice_probes(C.byref(cp), _p(v), _p(xy), C.c_int(len(xy)), _p(out))
    return out


def prism_probes(p: Params, s, beam_list, xy):
    s = _c128(s)
    beam_list = np.ascontiguousarray(beam_list, dtype=np.int32).reshape(-1, 2)
    xy = _f64(xy).reshape(-1, 2)
    out = np.empty((len(xy), num_bins(p)), dtype=np.float64)
    cp = p.c()
    _L().orc_prism_probes(C.byref(cp), _p(s), _p(beam_list), C.c_int(len(beam_list)), _p(xy),
                          C.c_int(len(xy)), _p(out))
    return out
