"""S-matrix in page-locked host memory (PAPER.md:136 streaming PRISM: the device holds only
"the current S-matrix subset").  Stage 1 propagates `batch` beams at a time in the workspace and copies their layers
out from alternating buffers; stage 2 keeps a ring of pixel rows of every layer in the workspace and brings in, on a
private copy stream, only the rows the next batch of probe rows adds while the current batch computes.  Both must
reproduce the resident path bit for bit, and through it the oracle."""
import numpy as np
import pytest

import oracle as O
from helpers import oracle_params, oracle_potential, rel_l2
from paper_1706_08563_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import gpu_helpers
    return gpu_helpers


CASES = {
    # Q = 8 lattice, off-pixel origin, 64^2 windows, 16 x 16 probes
    "L128f2q8": W.scaled_test_case(128, 3, 2, 16, alpha_mrad=25.0, defocus=30.0, seed_index=11,
                                   probe_offset=(0.137, 0.291)),
    # Q = 32, 128^2 windows, 64 x 64 probes with a 4-pixel step (the shape of configs 3-5); pipelined slice step
    "L256f2q32": W.scaled_test_case(256, 3, 2, 64, voltage=300e3, alpha_mrad=20.0, seed_index=12),
    # probe grid covering part of the cell, origin away from 0: slabs that wrap around the cell edge
    "L128f2part": W.scaled_test_case(128, 2, 2, 16, alpha_mrad=20.0, seed_index=15).with_(
        probes_x=5, probes_y=7, probe_origin=(1.2, 9.3)),
}


def _host_smatrix(G, w, v, batch):
    from paper_1706_08563_b200 import prism
    p = prism.params_from_workload(w, smatrix_on_host=1, batch=batch)
    s = torch.empty((prism.num_beams(p), w.ny, w.nx), dtype=torch.complex64).pin_memory()
    beams = prism.compute_smatrix(p, v, s, G.ws(p, prism.WS_SMATRIX))
    torch.cuda.synchronize()
    return s, beams


@pytest.mark.parametrize("name", list(CASES))
def test_host_resident_smatrix_reproduces_the_resident_path(G, name):
    from paper_1706_08563_b200 import prism
    w = CASES[name]
    v = G.gpu_potential(w)
    s_dev, beams = G.gpu_smatrix(w, v)
    out_dev = G.gpu_prism_output(w, s_dev, beams)
    for batch in (0, 1, 7):
        s_host, b2 = _host_smatrix(G, w, v, batch)
        assert np.array_equal(beams, b2)
        assert torch.equal(s_host, s_dev.cpu()), (name, batch)
    # stage 2 from host memory, several probe-row batch sizes (whole grid, one row, three rows and a ragged tail)
    for batch in (0, w.probes_x, 3 * w.probes_x + 1):
        p = prism.params_from_workload(w, smatrix_on_host=1, batch=batch)
        out = torch.empty((w.probes_y, w.probes_x, prism.num_bins(p)), dtype=torch.float32, device=G.DEV)
        prism.compute_output(p, s_host, beams, out, G.ws(p, prism.WS_OUTPUT))
        torch.cuda.synchronize()
        got = out.cpu().numpy().astype(np.float64).reshape(out_dev.shape)
        assert np.array_equal(got, out_dev), (name, batch)
    # and against the oracle end to end
    po = oracle_params(w)
    xy = w.probe_xy()
    pick = np.unique(np.linspace(0, len(xy) - 1, 25).astype(int))
    ref = O.prism_probes(po, O.smatrix(po, oracle_potential(w), beams), beams, xy[pick])
    assert rel_l2(got[pick], ref) < 1e-4


def test_streamed_potential_and_host_smatrix_together(G):
    w = CASES["L128f2q8"]
    v = G.gpu_potential(w)
    v_host = G.gpu_potential(w, on_host=True)
    s_dev, beams = G.gpu_smatrix(w, v)
    from paper_1706_08563_b200 import prism
    p = prism.params_from_workload(w, smatrix_on_host=1, potential_on_host=1, batch=5)
    s = torch.empty_like(s_dev, device="cpu").pin_memory()
    prism.compute_smatrix(p, v_host, s, G.ws(p, prism.WS_SMATRIX))
    torch.cuda.synchronize()
    assert torch.equal(s, s_dev.cpu())


def test_host_smatrix_needs_a_regular_probe_lattice(G):
    from paper_1706_08563_b200 import prism
    w = CASES["L128f2q8"].with_(probe_step=(0.83, 0.83))            # not a whole number of pixels
    v = G.gpu_potential(w)
    s_host, beams = _host_smatrix(G, w, v, 0)
    p = prism.params_from_workload(w, smatrix_on_host=1)
    out = torch.empty((w.probes_y, w.probes_x, prism.num_bins(p)), dtype=torch.float32, device=G.DEV)
    with pytest.raises(prism.PrismError) as e:
        prism.compute_output(p, s_host, beams, out, G.ws(p, prism.WS_OUTPUT))
    assert e.value.code == prism.PRISM_EUNSUPPORTED
