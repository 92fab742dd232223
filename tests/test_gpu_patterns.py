"""4-D output (SURVEY.md 8(f) NEXT-1; PAPER.md:82 "2D, 3D or 4D outputs", :90): the full diffraction pattern of every
probe from prism_compute_patterns / multislice_compute_patterns against the oracle's patterns, element by element.
Tolerance: relative L2 of a pattern <= 1e-4 (the ring tolerance of BASELINE.json: rings are sums of these pixels)."""
import numpy as np
import pytest

import oracle as O
from helpers import oracle_params, oracle_potential, rel_l2
from paper_1706_08563_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-4


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import gpu_helpers
    return gpu_helpers


CASES = {
    "PR1": W.pr1(),
    # off-pixel probes, defocus and Cs, 64^2 windows
    "T128f2": W.scaled_test_case(128, 4, 2, 5, alpha_mrad=25.0, defocus=40.0, cs=2.0e4, probe_offset=(0.137, 0.291),
                                 seed_index=1),
    # regular probe lattice (lattice-DFT path), 128^2 windows; pipelined 256-point slice step
    "L256f2q32": W.scaled_test_case(256, 3, 2, 64, voltage=300e3, alpha_mrad=20.0, seed_index=12),
    # rectangular window (128 x 16) from a 2048 x 256 grid on the packed kernels
    "R2048x256": W.scaled_test_case(256, 3, 4, 4, voltage=300e3, alpha_mrad=12.0, seed_index=31, density=0.03).with_(
        name="R2048x256", f=16, nx=2048, cell=(204.8, 25.6, 6.0), probe_step=(51.2, 6.4), alpha=6e-3),
}


def _prism_patterns(G, w, s, beams, p=None):
    from paper_1706_08563_b200 import prism
    p = p or prism.params_from_workload(w)
    pat = torch.empty((w.n_probes, w.ny // w.f, w.nx // w.f), dtype=torch.float32, device=G.DEV)
    prism.compute_patterns(p, s, beams, pat, G.ws(p, prism.WS_OUTPUT))
    torch.cuda.synchronize()
    return pat.cpu().numpy().astype(np.float64)


def _ms_patterns(G, w, v, p=None):
    from paper_1706_08563_b200 import prism
    p = p or prism.params_from_workload(w)
    pat = torch.empty((w.n_probes, w.ny, w.nx), dtype=torch.float32, device=G.DEV)
    prism.multislice_patterns(p, v, pat, G.ws(p, prism.WS_MULTISLICE_PATTERNS))
    torch.cuda.synchronize()
    return pat.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("name", list(CASES))
def test_prism_patterns_parity(G, name):
    w = CASES[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    pat = _prism_patterns(G, w, s, beams)
    s_ref = O.smatrix(p, oracle_potential(w), beams)
    xy = w.probe_xy()
    pick = np.unique(np.linspace(0, len(xy) - 1, 9).astype(int))
    for i in pick:
        _, ref = O.prism_probe(p, s_ref, beams, xy[i, 0], xy[i, 1], want_pattern=True)
        assert pat[i].shape == ref.shape
        assert rel_l2(pat[i], ref) < TOL, (name, i)
    # rings are sums of pattern pixels: the 3-D output of the same call path
    out = G.gpu_prism_output(w, s, beams)
    for i in pick:
        rings = O.bin_intensity(p, pat[i], w.f, w.f)
        assert np.allclose(rings, out[i], rtol=1e-5, atol=1e-9)


@pytest.mark.parametrize("name", ["PR1", "T128f2", "L256f2q32"])
def test_multislice_patterns_parity(G, name):
    w = CASES[name].with_(probes_x=3, probes_y=2)
    p = oracle_params(w)
    v = G.gpu_potential(w)
    pat = _ms_patterns(G, w, v)
    v_ref = oracle_potential(w)
    for i, (x, y) in enumerate(w.probe_xy()):
        _, ref = O.multislice_probe(p, v_ref, x, y, want_pattern=True)
        assert rel_l2(pat[i], ref) < TOL, (name, i)
    out = G.gpu_multislice(w, v)
    for i in range(len(pat)):
        assert np.allclose(O.bin_intensity(p, pat[i], 1, 1), out[i], rtol=1e-5, atol=1e-9)


def test_patterns_do_not_depend_on_batch(G):
    from paper_1706_08563_b200 import prism
    w = CASES["T128f2"]
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    a = _prism_patterns(G, w, s, beams)
    b = _prism_patterns(G, w, s, beams, prism.params_from_workload(w, batch=4))
    assert np.array_equal(a, b)
    m0 = _ms_patterns(G, w.with_(probes_x=3, probes_y=2), v)
    m1 = _ms_patterns(G, w.with_(probes_x=3, probes_y=2), v, prism.params_from_workload(w.with_(probes_x=3, probes_y=2), batch=1))
    assert np.array_equal(m0, m1)


def test_patterns_argument_checks(G):
    from paper_1706_08563_b200 import prism
    w = CASES["PR1"]
    p = prism.params_from_workload(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    host = torch.empty((w.n_probes, w.ny, w.nx), dtype=torch.float32)
    with pytest.raises(prism.PrismError) as e:
        prism.compute_patterns(p, s, beams, host, G.ws(p, prism.WS_OUTPUT))      # patterns must be device memory
    assert e.value.code == prism.PRISM_EINVAL


# ---- arbitrary virtual detectors (2-D output = one detector) ---------------------------------------------------
def _masks(w, p, my, mx, fy, fx, rng):
    """An annular detector built from the oracle's own angle convention (rings 3..7 of bin_intensity), a random
    weight mask, a half-plane (segmented) detector, and the all-ones mask."""
    lam, _ = O.constants(w.voltage)
    ky = np.where(np.arange(my) < my // 2, np.arange(my), np.arange(my) - my) * fy
    kx = np.where(np.arange(mx) < mx // 2, np.arange(mx), np.arange(mx) - mx) * fx
    ang = lam * np.sqrt((kx[None, :] / w.cell[0]) ** 2 + (ky[:, None] / w.cell[1]) ** 2)
    ring = np.floor(ang / w.det_step)
    annular = ((ring >= 3) & (ring < 8)).astype(np.float64)
    return np.stack([annular, rng.random((my, mx)), (kx[None, :] > 0) * np.ones((my, 1)), np.ones((my, mx))])


@pytest.mark.parametrize("name", ["PR1", "T128f2", "R2048x256"])
def test_prism_detectors_parity(G, name):
    from paper_1706_08563_b200 import prism
    w = CASES[name]
    p = oracle_params(w)
    pp = prism.params_from_workload(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    my, mx = w.ny // w.f, w.nx // w.f
    masks = _masks(w, p, my, mx, w.f, w.f, np.random.default_rng(5))
    m_dev = torch.as_tensor(masks, dtype=torch.float32, device=G.DEV).contiguous()
    out = torch.empty((w.n_probes, len(masks)), dtype=torch.float32, device=G.DEV)
    prism.compute_detectors(pp, s, beams, m_dev, out, G.ws(pp, prism.WS_OUTPUT))
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    s_ref = O.smatrix(p, oracle_potential(w), beams)
    xy = w.probe_xy()
    m32 = m_dev.cpu().numpy().astype(np.float64)             # the weights the kernel saw
    ref = np.empty_like(got)
    for i in range(len(xy)):
        bins, pat = O.prism_probe(p, s_ref, beams, xy[i, 0], xy[i, 1], want_pattern=True)
        ref[i] = (m32 * pat[None]).sum(axis=(1, 2))
        assert abs(ref[i, 0] - bins[3:8].sum()) < 1e-12          # the annular mask is rings 3..7 of the oracle
        assert abs(ref[i, 3] - pat.sum()) < 1e-12
    assert rel_l2(got, ref) < TOL
    for d in range(len(masks)):
        assert rel_l2(got[:, d], ref[:, d]) < 5 * TOL, d
    # one annular detector = a sum of rings of the 3-D output
    rings = G.gpu_prism_output(w, s, beams)
    assert np.allclose(got[:, 0], rings[:, 3:8].sum(axis=1), rtol=1e-5, atol=1e-9)
    # deterministic
    out2 = torch.empty_like(out)
    prism.compute_detectors(pp, s, beams, m_dev, out2, G.ws(pp, prism.WS_OUTPUT))
    assert torch.equal(out, out2)


def test_multislice_detectors_parity(G):
    from paper_1706_08563_b200 import prism
    w = CASES["L256f2q32"].with_(probes_x=3, probes_y=2)
    p = oracle_params(w)
    pp = prism.params_from_workload(w)
    v = G.gpu_potential(w)
    masks = _masks(w, p, w.ny, w.nx, 1, 1, np.random.default_rng(6))
    m_dev = torch.as_tensor(masks, dtype=torch.float32, device=G.DEV).contiguous()
    out = torch.empty((w.n_probes, len(masks)), dtype=torch.float32, device=G.DEV)
    prism.multislice_detectors(pp, v, m_dev, out, G.ws(pp, prism.WS_MULTISLICE_PATTERNS))
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    v_ref = oracle_potential(w)
    m32 = m_dev.cpu().numpy().astype(np.float64)
    ref = np.stack([(m32 * O.multislice_probe(p, v_ref, x, y, want_pattern=True)[1][None]).sum(axis=(1, 2))
                    for x, y in w.probe_xy()])
    assert rel_l2(got, ref) < TOL


def test_detector_argument_checks(G):
    from paper_1706_08563_b200 import prism
    w = CASES["PR1"]
    pp = prism.params_from_workload(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    too_many = torch.zeros((17, w.ny, w.nx), dtype=torch.float32, device=G.DEV)
    out = torch.empty((w.n_probes, 17), dtype=torch.float32, device=G.DEV)
    with pytest.raises(prism.PrismError) as e:
        prism.compute_detectors(pp, s, beams, too_many, out, G.ws(pp, prism.WS_OUTPUT))
    assert e.value.code == prism.PRISM_EUNSUPPORTED
