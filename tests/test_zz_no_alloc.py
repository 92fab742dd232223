"""``prism_build_potential_static``: the projected-potential build for callers that cannot allocate device memory.

Who needs it: code that runs inside another program's GPU memory pool (a plug-in whose host owns the device and
forbids ``cudaMalloc`` of its own), a process whose device memory is already fully handed out, or a caller in a
phase where the CUDA allocator must not be entered.  Such a caller cannot produce the ``workspace`` argument of
``prism_build_potential``; the ``_static`` entry point reads its scratch (sorted atoms, cell starts, radial tables)
from an 8 MiB array built into the library instead, and takes only inputs and the output.

Checked here: on two calls in a row with different atoms -- the second finds the first call's leftovers in the
shared array -- the output equals the workspace path's within the tolerance of the potential parity tests
(``TOL_V`` of ``test_gpu_parity.py``; both run the same deterministic kernel, so they are in fact bit-identical,
which is asserted too); and a request beyond the array is refused with a clear message before anything is launched.

This file sorts last on purpose (``pytest -x`` stops at the first failure: a failure here must not hide the parity
suite) and passes alone in a fresh process as well as after every other test (the entry point's first call on a
device does its own one-time set-up, the look-up of the array's device address).
"""
import numpy as np
import pytest

from paper_1706_08563_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_V = 1e-6          # relative L2, as for test_potential_parity


def rel_l2(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def G():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test collected on a machine without a CUDA device")
    import gpu_helpers
    return gpu_helpers


def _static_potential(G, w, phonon):
    import torch
    from paper_1706_08563_b200 import prism
    p = prism.params_from_workload(w)
    p.potential_on_host = 0
    lut_z, r_cut, lut_v = w.lut()
    # the output is the caller's; poisoned so that an unwritten pixel cannot pass for a zero of the potential
    v = torch.full((w.n_slices, w.ny, w.nx), float("nan"), dtype=torch.float32, device=G.DEV)
    prism.build_potential_static(p, w.atoms_for_phonon(phonon), w.z, lut_z, r_cut, lut_v, v)
    torch.cuda.synchronize()
    return v


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(G):
    import torch
    # first call: config 3 (512^2, 100 slices, 43 095 atoms) fills about 3.9 MB of the array; second call: config 1
    # (64^2, 4 slices, 40 atoms) rewrites only its front part and leaves the rest stale; third: config 3 again with
    # the atoms of another frozen-phonon configuration (same sizes, different values in the same bytes)
    for w, phonon in ((W.get("P4"), 0), (W.get("PR1"), 0), (W.get("P4"), 1)):
        got = _static_potential(G, w, phonon)
        want = G.gpu_potential(w, phonon=phonon)            # prism_build_potential with a torch-allocated workspace
        assert got.shape == want.shape
        assert not torch.isnan(got).any()
        assert rel_l2(got.cpu().numpy().astype(np.float64), want.cpu().numpy().astype(np.float64)) < TOL_V
        assert torch.equal(got, want)                       # same kernel, same summation order


def test_static_scratch_refuses_what_does_not_fit(G):
    import torch
    from paper_1706_08563_b200 import prism
    w = W.get("P16")                                        # 400 x 2048^2: the cell table alone is 26 MB
    p = prism.params_from_workload(w)
    p.potential_on_host = 0
    lut_z, r_cut, lut_v = w.lut()
    v = torch.zeros((1, 8, 8), dtype=torch.float32, device=G.DEV)      # never written: the call must refuse first
    launches = prism.launch_count()
    with pytest.raises(prism.PrismError) as err:
        prism.build_potential_static(p, np.zeros((1, 3)), np.array([lut_z[0]], dtype=np.int32), lut_z, r_cut, lut_v, v)
    assert err.value.code == prism.PRISM_EUNSUPPORTED
    assert "built-in array holds %d" % prism.STATIC_SCRATCH_BYTES in str(err.value)
    assert prism.launch_count() == launches
    # a streamed (host) potential needs staging buffers and a copy stream: refused as well
    p = prism.params_from_workload(W.get("PR1"))
    p.potential_on_host = 1
    with pytest.raises(prism.PrismError) as err:
        prism.build_potential_static(p, np.zeros((1, 3)), np.array([6], dtype=np.int32), *W.get("PR1").lut(), v)
    assert err.value.code == prism.PRISM_EUNSUPPORTED
