"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/prism.h
declares, and its host-side logic (constants, beam counts, ring counts, workspace sizes,
argument checks) agrees with the paper-derived oracle.  No compute call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle as O
from helpers import oracle_params
from paper_1706_08563_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def prism():
    from paper_1706_08563_b200 import build
    build.build()
    from paper_1706_08563_b200 import prism as mod
    return mod


def test_every_declared_symbol_is_exported(prism):
    header = open(os.path.join(ROOT, "include", "prism.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b((?:prism|multislice)_[a-z_]+)\s*\(", header))
    assert {"prism_build_potential", "prism_compute_smatrix", "prism_compute_output",
            "multislice_compute_output"} <= declared
    lib = C.CDLL(prism.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(prism.EXPORTS)


def test_params_struct_layout_matches_header(prism, tmp_path):
    # ask the C compiler for the layout of the real header and compare with the ctypes mirror
    src = tmp_path / "layout.c"
    fields = [f for f, _ in prism.Params._fields_]
    body = "".join(f'printf("{f} %zu\\n", offsetof(prism_params, {f}));' for f in fields)
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "prism.h"\nint main(void){'
                   + body + 'printf("sizeof %zu\\n", sizeof(prism_params));'
                   'printf("lut %zu %zu\\n", sizeof(prism_lut), offsetof(prism_lut, v)); return 0;}')
    exe = tmp_path / "layout"
    import subprocess
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    lines = dict(ln.split(None, 1) for ln in subprocess.check_output([str(exe)]).decode().splitlines())
    for f in fields:
        assert int(lines[f]) == getattr(prism.Params, f).offset, f
    assert int(lines["sizeof"]) == C.sizeof(prism.Params)
    assert lines["lut"].split() == [str(C.sizeof(prism.Lut)), str(prism.Lut.v.offset)]


@pytest.mark.parametrize("volt", [80e3, 200e3, 300e3])
def test_constants_agree_with_oracle(prism, volt):
    lam, sig = prism.constants(volt)
    lam_o, sig_o = O.constants(volt)
    assert abs(lam - lam_o) / lam_o < 1e-13 and abs(sig - sig_o) / sig_o < 1e-13


@pytest.mark.parametrize("name,n_beams", [("PR1", 89), ("P4", 529), ("P8", 509), ("P16", 1201)])
def test_beam_counts_and_bins(prism, name, n_beams):
    w = W.get(name)
    p = prism.params_from_workload(w)
    assert prism.num_beams(p) == n_beams == len(O.beams(oracle_params(w)))
    assert prism.num_bins(p) == O.num_bins(oracle_params(w))


@pytest.mark.parametrize("name", ["PR1", "MS2", "P4", "P8"])
def test_band_columns_cover_the_oracle_propagator(prism, name):
    """Every kx column in which the oracle's band-limited propagator is non-zero lies inside the column band
    the library moves through HBM, and the band is not wider than one 32-column rounding."""
    w = W.get(name)
    prop = O.propagator(oracle_params(w))
    live = np.flatnonzero(np.abs(prop).sum(axis=0) > 0)           # kx slots with any non-zero entry
    c = prism.band_columns(prism.params_from_workload(w))
    assert c % 32 == 0 and 0 < c <= w.nx // 2
    inside = (live < c) | (live >= w.nx - c)
    assert inside.all()
    kxmax = int(np.max(np.minimum(live, w.nx - live)))
    assert c == min(w.nx // 2, -(-(kxmax + 1) // 32) * 32)


def test_workspace_sizes_are_positive_and_scale(prism):
    w = W.get("P4")
    p = prism.params_from_workload(w)
    sizes = [prism.workspace_bytes(p, k) for k in range(5)]
    assert all(s > 0 for s in sizes)
    # 512^2 is a resident-multislice grid: ring output keeps a wave per SM, patterns / detectors a batch only
    assert sizes[prism.WS_MULTISLICE_PATTERNS] <= sizes[prism.WS_MULTISLICE]
    few = prism.params_from_workload(w, batch=4)
    assert (prism.workspace_bytes(few, prism.WS_MULTISLICE) - prism.workspace_bytes(few, prism.WS_MULTISLICE_PATTERNS)
            == (148 - 4) * 512 * 512 * 12)
    small = prism.params_from_workload(W.pr1())                     # 64^2 never runs resident: the two agree
    assert prism.workspace_bytes(small, prism.WS_MULTISLICE_PATTERNS) == prism.workspace_bytes(small, prism.WS_MULTISLICE)
    assert sizes[prism.WS_SMATRIX] < 64 << 20                       # tables + one t slice only
    p_host = prism.params_from_workload(w, potential_on_host=1)
    assert prism.workspace_bytes(p_host, prism.WS_SMATRIX) == sizes[0] + 3 * 512 * 512 * 4
    p_b = prism.params_from_workload(w, batch=16)
    assert prism.workspace_bytes(p_b, prism.WS_OUTPUT) < sizes[prism.WS_OUTPUT]


def test_argument_checks_without_a_gpu(prism):
    w = W.pr1()
    for bad in [dict(nx=96), dict(nx=32), dict(nx=4096), dict(f=3), dict(alpha=0.0), dict(alpha=0.09),
                dict(det_step=0.0), dict(n_slices=0), dict(voltage=-1.0)]:
        with pytest.raises(prism.PrismError):
            prism.num_beams(prism.params_from_workload(w, **bad))
    # malformed aberration terms (n outside 1..8, m beyond n + 1)
    for bad in [((0, 0, 1.0, 0.0),), ((9, 0, 1.0, 0.0),), ((2, 4, 1.0, 0.0),)]:
        with pytest.raises(prism.PrismError):
            prism.num_beams(prism.params_from_workload(w.with_(aberrations=bad)))
    assert prism.num_beams(prism.params_from_workload(w.with_(aberrations=((1, 2, 10.0, 0.3),)))) == 89
    # window smaller than 16 x 16 is outside this build
    p = prism.params_from_workload(w, f=8)
    with pytest.raises(prism.PrismError):
        prism.workspace_bytes(p, prism.WS_OUTPUT)
    # a window side above 128 points too, even when the window area is not (256 x 64 at 512 x 128, f = 2)
    wide = prism.params_from_workload(w, nx=512, ny=128, f=2)
    wide.cell[0], wide.cell[1] = 51.2, 12.8
    assert prism.num_beams(wide) > 0
    assert prism._lib.prism_workspace_bytes(C.byref(wide), prism.WS_OUTPUT) == 0
    assert prism._lib.prism_strerror(prism.PRISM_ENOMEM) == b"workspace too small"


def test_missing_library_fails_loudly(tmp_path, monkeypatch):
    import importlib
    import paper_1706_08563_b200.prism as mod
    monkeypatch.setattr(mod, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        mod._load()
    importlib.reload(mod)
