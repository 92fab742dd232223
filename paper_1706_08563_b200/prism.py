"""Thin ctypes binding of ``libprism_b200.so`` (C ABI: ``include/prism.h``).

Argument marshalling only -- every step of the path runs in the CUDA kernels of
``csrc/``.  PyTorch supplies device memory and the current CUDA stream; nothing
here computes.  There is no CPU fallback: if the library is missing, importing
this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libprism_b200.so")

PRISM_OK, PRISM_EINVAL, PRISM_ENOMEM, PRISM_ECUDA, PRISM_EUNSUPPORTED, PRISM_ENOLUT = 0, -1, -2, -3, -4, -5
WS_SMATRIX, WS_OUTPUT, WS_MULTISLICE, WS_POTENTIAL, WS_MULTISLICE_PATTERNS = 0, 1, 2, 3, 4

EXPORTS = ["prism_workspace_bytes", "prism_num_bins", "prism_num_beams", "prism_band_columns", "prism_constants",
           "prism_build_potential", "prism_build_potential_static", "prism_compute_smatrix", "prism_compute_output",
           "multislice_compute_output", "prism_compute_patterns", "multislice_compute_patterns",
           "prism_compute_detectors", "multislice_compute_detectors", "prism_accumulate", "prism_strerror", "prism_last_error", "prism_launch_count",
           "prism_timing_enable", "prism_timing_classes", "prism_timing_class_name", "prism_timing_read"]


class Aberration(C.Structure):
    """``prism_aberration`` of include/prism.h."""
    _fields_ = [("n", C.c_int32), ("m", C.c_int32), ("c", C.c_double), ("angle", C.c_double)]


class Params(C.Structure):
    """``prism_params`` of include/prism.h (same field order and types)."""
    _fields_ = [
        ("cell", C.c_double * 3), ("nx", C.c_int32), ("ny", C.c_int32),
        ("slice_thickness", C.c_double), ("n_slices", C.c_int32),
        ("voltage", C.c_double), ("alpha", C.c_double), ("defocus", C.c_double), ("cs", C.c_double),
        ("f", C.c_int32), ("probes_x", C.c_int32), ("probes_y", C.c_int32),
        ("probe_origin", C.c_double * 2), ("probe_step", C.c_double * 2),
        ("det_step", C.c_double), ("det_max", C.c_double),
        ("batch", C.c_int32), ("potential_on_host", C.c_int32), ("smatrix_on_host", C.c_int32),
        ("n_aberrations", C.c_int32), ("aberrations", C.POINTER(Aberration)),
    ]


class Lut(C.Structure):
    _fields_ = [("z", C.c_int32), ("n", C.c_int32), ("r_cut", C.c_double), ("v", C.POINTER(C.c_float))]


class PrismError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = _lib.prism_strerror(code).decode()
        detail = _lib.prism_last_error().decode() if code == PRISM_ECUDA else ""
        super().__init__(f"{where}: {msg} ({code}) {detail}".strip())


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is not built: run `python -m paper_1706_08563_b200.build` "
            "(nvcc, sm_100a).  There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t
    pp = C.POINTER(Params)
    lib.prism_workspace_bytes.restype = sz
    lib.prism_workspace_bytes.argtypes = [pp, i32]
    lib.prism_num_bins.restype = i32
    lib.prism_num_bins.argtypes = [pp]
    lib.prism_band_columns.restype = i32
    lib.prism_band_columns.argtypes = [pp]
    lib.prism_num_beams.restype = C.c_int
    lib.prism_num_beams.argtypes = [pp, C.POINTER(i32)]
    lib.prism_constants.restype = C.c_int
    lib.prism_constants.argtypes = [C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.prism_build_potential.restype = C.c_int
    lib.prism_build_potential.argtypes = [pp, vp, vp, i64, C.POINTER(Lut), i32, vp, vp, sz, vp]
    lib.prism_build_potential_static.restype = C.c_int
    lib.prism_build_potential_static.argtypes = [pp, vp, vp, i64, C.POINTER(Lut), i32, vp, vp]
    lib.prism_compute_smatrix.restype = C.c_int
    lib.prism_compute_smatrix.argtypes = [pp, vp, vp, vp, vp, sz, vp]
    lib.prism_compute_output.restype = C.c_int
    lib.prism_compute_output.argtypes = [pp, vp, vp, i32, vp, vp, sz, vp]
    lib.multislice_compute_output.restype = C.c_int
    lib.multislice_compute_output.argtypes = [pp, vp, vp, vp, sz, vp]
    lib.prism_compute_patterns.restype = C.c_int
    lib.prism_compute_patterns.argtypes = [pp, vp, vp, i32, vp, vp, sz, vp]
    lib.multislice_compute_patterns.restype = C.c_int
    lib.multislice_compute_patterns.argtypes = [pp, vp, vp, vp, sz, vp]
    lib.prism_compute_detectors.restype = C.c_int
    lib.prism_compute_detectors.argtypes = [pp, vp, vp, i32, vp, i32, vp, vp, sz, vp]
    lib.multislice_compute_detectors.restype = C.c_int
    lib.multislice_compute_detectors.argtypes = [pp, vp, vp, i32, vp, vp, sz, vp]
    lib.prism_accumulate.restype = C.c_int
    lib.prism_accumulate.argtypes = [vp, vp, i64, C.c_float, i32, vp]
    lib.prism_strerror.restype = C.c_char_p
    lib.prism_strerror.argtypes = [C.c_int]
    lib.prism_last_error.restype = C.c_char_p
    lib.prism_launch_count.restype = i64
    lib.prism_launch_count.argtypes = [i32]
    lib.prism_timing_enable.restype = i32
    lib.prism_timing_enable.argtypes = [i32]
    lib.prism_timing_classes.restype = i32
    lib.prism_timing_class_name.restype = C.c_char_p
    lib.prism_timing_class_name.argtypes = [i32]
    lib.prism_timing_read.restype = C.c_int
    lib.prism_timing_read.argtypes = [C.POINTER(C.c_double), C.POINTER(i64)]
    return lib


_lib = _load()


def _check(code: int, where: str):
    if code != PRISM_OK:
        raise PrismError(code, where)


def params_from_workload(w, **override) -> Params:
    """Fill ``prism_params`` from a ``workloads.Workload`` (plain field copy)."""
    p = Params()
    p.cell[:] = w.cell
    p.nx, p.ny = w.nx, w.ny
    p.slice_thickness, p.n_slices = w.dz, w.n_slices
    p.voltage, p.alpha, p.defocus, p.cs = w.voltage, w.alpha, w.defocus, w.cs
    p.f, p.probes_x, p.probes_y = w.f, w.probes_x, w.probes_y
    p.probe_origin[:] = w.probe_origin
    p.probe_step[:] = w.probe_step
    p.det_step, p.det_max = w.det_step, w.det_max
    p.batch, p.potential_on_host = w.batch, w.potential_on_host
    p.smatrix_on_host = getattr(w, "smatrix_on_host", 0)
    terms = tuple(getattr(w, "aberrations", ()))
    if terms:
        arr = (Aberration * len(terms))(*[Aberration(int(n), int(m), float(c), float(a)) for n, m, c, a in terms])
        p.n_aberrations, p.aberrations = len(terms), arr
        p._aberrations_keep = arr               # the host array must outlive the struct's use
    for k, v in override.items():
        setattr(p, k, v)
    return p


def _stream_ptr(stream=None) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _ptr(t) -> int:
    return int(t.data_ptr())


def workspace_bytes(p: Params, which: int, n_atoms: int = 0) -> int:
    n = int(_lib.prism_workspace_bytes(C.byref(p), which))
    if n == 0:
        raise PrismError(PRISM_EINVAL, "prism_workspace_bytes")
    return n + (32 * n_atoms + 256 if which == WS_POTENTIAL else 0)


def num_bins(p: Params) -> int:
    return int(_lib.prism_num_bins(C.byref(p)))


def band_columns(p: Params) -> int:
    return int(_lib.prism_band_columns(C.byref(p)))


def num_beams(p: Params) -> int:
    n = C.c_int32(0)
    _check(_lib.prism_num_beams(C.byref(p), C.byref(n)), "prism_num_beams")
    return n.value


def constants(voltage: float):
    lam, sig = C.c_double(), C.c_double()
    _check(_lib.prism_constants(voltage, C.byref(lam), C.byref(sig)), "prism_constants")
    return lam.value, sig.value


def launch_count(reset: bool = False) -> int:
    return int(_lib.prism_launch_count(1 if reset else 0))


def timing_enable(on: bool) -> bool:
    return bool(_lib.prism_timing_enable(1 if on else 0))


def timing_read() -> dict:
    """{kernel class: (total ms, launches)} of the launches recorded since the last read."""
    n = int(_lib.prism_timing_classes())
    ms = (C.c_double * n)()
    cnt = (C.c_int64 * n)()
    _check(_lib.prism_timing_read(ms, cnt), "prism_timing_read")
    return {_lib.prism_timing_class_name(i).decode(): (ms[i], int(cnt[i])) for i in range(n) if cnt[i]}


def build_potential(p: Params, atoms_xyz, z_number, lut_z, r_cut, lut_v, v_out, workspace, stream=None):
    """``prism_build_potential``.  atoms/z/luts are host numpy arrays; ``v_out`` is a CUDA tensor
    ``[n_slices][ny][nx]`` fp32, or a pinned host tensor when ``p.potential_on_host``."""
    atoms = np.ascontiguousarray(atoms_xyz, dtype=np.float64).reshape(-1, 3)
    zn = np.ascontiguousarray(z_number, dtype=np.int32)
    tabs = np.ascontiguousarray(lut_v, dtype=np.float32).reshape(len(lut_z), -1 if len(lut_z) else 0)
    luts = (Lut * len(lut_z))()
    for i, z in enumerate(lut_z):
        luts[i].z, luts[i].n, luts[i].r_cut = int(z), tabs.shape[1], float(r_cut)
        luts[i].v = tabs[i].ctypes.data_as(C.POINTER(C.c_float))
    _check(_lib.prism_build_potential(C.byref(p), atoms.ctypes.data, zn.ctypes.data, len(zn), luts, len(lut_z),
                                      _ptr(v_out), _ptr(workspace), workspace.numel() * workspace.element_size(),
                                      _stream_ptr(stream)), "prism_build_potential")
    return v_out


STATIC_SCRATCH_BYTES = 8 << 20       # PRISM_STATIC_SCRATCH_BYTES of include/prism.h


def build_potential_static(p: Params, atoms_xyz, z_number, lut_z, r_cut, lut_v, v_out, stream=None):
    """``prism_build_potential_static``: ``build_potential`` without a workspace, for callers that may not
    allocate device memory (they run inside another program's memory pool, or all of the device is already
    spoken for).  The kernel's scratch is an 8 MiB array built into the library, shared by every call on the
    device; requests that need more raise ``PrismError`` (``PRISM_EUNSUPPORTED``) with the byte counts.
    ``v_out`` must be a CUDA tensor.  Same result as ``build_potential``, bit for bit."""
    atoms = np.ascontiguousarray(atoms_xyz, dtype=np.float64).reshape(-1, 3)
    zn = np.ascontiguousarray(z_number, dtype=np.int32)
    tabs = np.ascontiguousarray(lut_v, dtype=np.float32).reshape(len(lut_z), -1 if len(lut_z) else 0)
    luts = (Lut * len(lut_z))()
    for i, z in enumerate(lut_z):
        luts[i].z, luts[i].n, luts[i].r_cut = int(z), tabs.shape[1], float(r_cut)
        luts[i].v = tabs[i].ctypes.data_as(C.POINTER(C.c_float))
    code = _lib.prism_build_potential_static(C.byref(p), atoms.ctypes.data, zn.ctypes.data, len(zn), luts,
                                             len(lut_z), _ptr(v_out), _stream_ptr(stream))
    if code == PRISM_EUNSUPPORTED:
        err = PrismError(code, "prism_build_potential_static")
        err.args = (f"{err.args[0]}: {_lib.prism_last_error().decode()}",)
        raise err
    _check(code, "prism_build_potential_static")
    return v_out


def compute_smatrix(p: Params, v, s_out, workspace, stream=None):
    """``prism_compute_smatrix``.  Returns the host beam list ``[n_beams][2]`` int32."""
    beams = np.empty((num_beams(p), 2), dtype=np.int32)
    _check(_lib.prism_compute_smatrix(C.byref(p), _ptr(v), beams.ctypes.data, _ptr(s_out), _ptr(workspace),
                                      workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "prism_compute_smatrix")
    return beams


def compute_output(p: Params, s, beams, out, workspace, stream=None):
    """``prism_compute_output``.  ``out`` fp32 ``[probes_y][probes_x][n_bins]``, CUDA or (pinned) host tensor."""
    beams = np.ascontiguousarray(beams, dtype=np.int32).reshape(-1, 2)
    _check(_lib.prism_compute_output(C.byref(p), _ptr(s), beams.ctypes.data, len(beams), _ptr(out), _ptr(workspace),
                                     workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "prism_compute_output")
    return out


def multislice_output(p: Params, v, out, workspace, stream=None):
    """``multislice_compute_output``."""
    _check(_lib.multislice_compute_output(C.byref(p), _ptr(v), _ptr(out), _ptr(workspace),
                                          workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "multislice_compute_output")
    return out


def accumulate(acc, x, weight: float = 1.0, first: bool = False, stream=None):
    """``prism_accumulate``: acc = (first ? 0 : acc) + weight * x on CUDA fp32 tensors of equal size."""
    assert acc.numel() == x.numel()
    _check(_lib.prism_accumulate(_ptr(acc), _ptr(x), acc.numel(), float(weight), 1 if first else 0,
                                 _stream_ptr(stream)), "prism_accumulate")
    return acc


def compute_patterns(p: Params, s, beams, patterns, workspace, stream=None):
    """``prism_compute_patterns``.  ``patterns`` fp32 CUDA tensor ``[probes_y * probes_x][ny / f][nx / f]``."""
    beams = np.ascontiguousarray(beams, dtype=np.int32).reshape(-1, 2)
    _check(_lib.prism_compute_patterns(C.byref(p), _ptr(s), beams.ctypes.data, len(beams), _ptr(patterns),
                                       _ptr(workspace), workspace.numel() * workspace.element_size(),
                                       _stream_ptr(stream)), "prism_compute_patterns")
    return patterns


def multislice_patterns(p: Params, v, patterns, workspace, stream=None):
    """``multislice_compute_patterns``.  ``patterns`` fp32 CUDA tensor ``[probes_y * probes_x][ny][nx]``."""
    _check(_lib.multislice_compute_patterns(C.byref(p), _ptr(v), _ptr(patterns), _ptr(workspace),
                                            workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "multislice_compute_patterns")
    return patterns


def compute_detectors(p: Params, s, beams, masks, out, workspace, stream=None):
    """``prism_compute_detectors``.  ``masks`` fp32 CUDA ``[n_masks][ny / f][nx / f]``, ``out`` fp32 CUDA
    ``[probes_y * probes_x][n_masks]``."""
    beams = np.ascontiguousarray(beams, dtype=np.int32).reshape(-1, 2)
    _check(_lib.prism_compute_detectors(C.byref(p), _ptr(s), beams.ctypes.data, len(beams), _ptr(masks),
                                        int(masks.shape[0]), _ptr(out), _ptr(workspace),
                                        workspace.numel() * workspace.element_size(), _stream_ptr(stream)),
           "prism_compute_detectors")
    return out


def multislice_detectors(p: Params, v, masks, out, workspace, stream=None):
    """``multislice_compute_detectors``.  ``masks`` fp32 CUDA ``[n_masks][ny][nx]``."""
    _check(_lib.multislice_compute_detectors(C.byref(p), _ptr(v), _ptr(masks), int(masks.shape[0]), _ptr(out),
                                             _ptr(workspace), workspace.numel() * workspace.element_size(),
                                             _stream_ptr(stream)), "multislice_compute_detectors")
    return out
