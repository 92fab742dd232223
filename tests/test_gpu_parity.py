"""Parity of the CUDA path (through the C ABI) with the fp64 oracle, element by element on
the same seeded inputs.  Tolerances: BASELINE.json north_star -- detector-ring intensities
within relative L2 1e-4 (1e-3 for 2048^2 with >= 400 slices); DESIGN.md derives the
per-stage bounds used for the potential (1e-6) and the S-matrix layers (2e-5)."""
import numpy as np
import pytest

import oracle as O
from helpers import oracle_params, oracle_potential, rel_l2
from paper_1706_08563_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_OUT = 1e-4
TOL_V = 1e-6
TOL_S = 2e-5


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import gpu_helpers
    return gpu_helpers


def _cases():
    return {
        "PR1": W.pr1(),
        # 128^2, f=2 -> 64^2 windows; off-pixel probe positions; defocus + Cs
        "T128f2": W.scaled_test_case(128, 6, 2, 5, alpha_mrad=25.0, defocus=40.0, cs=2.0e4,
                                     probe_offset=(0.137, 0.291), seed_index=1),
        # 128^2, f=4 -> 32^2 windows, 300 kV, heavy atoms
        "T128f4": W.scaled_test_case(128, 5, 4, 6, voltage=300e3, alpha_mrad=20.0, z_choices=(79, 33),
                                     seed_index=2),
        # 256^2, f=2 -> 128^2 windows (the window size of configs 3-5)
        "T256f2": W.scaled_test_case(256, 4, 2, 3, voltage=300e3, alpha_mrad=20.0, seed_index=3,
                                     probe_offset=(0.05, 0.0)),
        # 512^2: three-stage FFT plan, f=8 -> 64^2 windows
        "T512f8": W.scaled_test_case(512, 3, 8, 3, voltage=300e3, alpha_mrad=20.0, seed_index=4, density=0.02),
    }


CASES = _cases()


@pytest.mark.parametrize("name", list(CASES))
def test_potential_parity(G, name):
    w = CASES[name]
    v = G.gpu_potential(w).cpu().numpy().astype(np.float64)
    ref = oracle_potential(w)
    assert v.shape == ref.shape
    assert rel_l2(v, ref) < TOL_V
    assert np.array_equal(v == 0, ref == 0) or np.count_nonzero((v == 0) != (ref == 0)) <= 2


@pytest.mark.parametrize("name", list(CASES))
def test_smatrix_parity(G, name):
    w = CASES[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    ref_beams = O.beams(p)
    assert set(map(tuple, beams.tolist())) == set(map(tuple, ref_beams.tolist()))
    v_ref = oracle_potential(w)
    pick = np.unique(np.linspace(0, len(beams) - 1, 7).astype(int)) if name != "PR1" else np.arange(len(beams))
    s_host = s.cpu().numpy()
    for b in pick:
        ref = O.smatrix_layer(p, v_ref, int(beams[b, 0]), int(beams[b, 1]))
        assert rel_l2(s_host[b].astype(np.complex128), ref) < TOL_S, (name, b)


@pytest.mark.parametrize("name", list(CASES))
def test_prism_output_parity(G, name):
    w = CASES[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    out = G.gpu_prism_output(w, s, beams)
    v_ref = oracle_potential(w)
    s_ref = O.smatrix(p, v_ref, beams)
    ref = O.prism_probes(p, s_ref, beams, w.probe_xy())
    assert out.shape == ref.shape
    assert rel_l2(out, ref) < TOL_OUT
    d = G.dark_field(w, p)
    assert ref[:, d:].sum() > 0
    assert rel_l2(out[:, d:], ref[:, d:]) < 5 * TOL_OUT        # dark field alone (reading R22)


@pytest.mark.parametrize("name", ["PR1", "T128f2", "T256f2", "T512f8"])
def test_multislice_parity(G, name):
    w = CASES[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    out = G.gpu_multislice(w, v)
    ref = O.multislice_probes(p, oracle_potential(w), w.probe_xy())
    assert rel_l2(out, ref) < TOL_OUT
    d = G.dark_field(w, p)
    assert rel_l2(out[:, d:], ref[:, d:]) < 5 * TOL_OUT


def test_general_aberration_terms_parity(G):
    """Reading R5b: astigmatism, coma, three-fold astigmatism and C5 beside defocus, in the PRISM coefficients (per beam)
    and in the multislice probe spectrum (per aperture pixel), against the oracle."""
    terms = ((1, 2, 35.0, 0.4), (2, 1, 3.0e3, 1.1), (2, 3, 1.5e3, -0.6), (5, 0, 2.0e8, 0.0))
    w = W.scaled_test_case(128, 4, 2, 4, alpha_mrad=25.0, defocus=30.0, seed_index=31,
                           probe_offset=(0.21, 0.07)).with_(aberrations=terms)
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    v_ref = oracle_potential(w)
    ref = O.prism_probes(p, O.smatrix(p, v_ref, beams), beams, w.probe_xy())
    plain = O.prism_probes(oracle_params(w.with_(aberrations=())), O.smatrix(p, v_ref, beams), beams, w.probe_xy())
    assert rel_l2(plain, ref) > 1e-2                                   # the terms matter in this case
    out = G.gpu_prism_output(w, s, beams)
    d = G.dark_field(w, p)
    assert rel_l2(out, ref) < TOL_OUT and rel_l2(out[:, d:], ref[:, d:]) < 5 * TOL_OUT
    out_m = G.gpu_multislice(w, v)
    ref_m = O.multislice_probes(p, v_ref, w.probe_xy())
    assert rel_l2(out_m, ref_m) < TOL_OUT and rel_l2(out_m[:, d:], ref_m[:, d:]) < 5 * TOL_OUT
    # malformed terms are rejected
    from paper_1706_08563_b200 import prism
    for bad in [((0, 0, 1.0, 0.0),), ((9, 0, 1.0, 0.0),), ((2, 4, 1.0, 0.0),)]:
        with pytest.raises(prism.PrismError):
            prism.num_beams(prism.params_from_workload(w.with_(aberrations=bad)))


def test_frozen_phonon_average_parity(G):
    """Row FP of SURVEY.md 8(a) (images are averaged over frozen-phonon configurations): three
    thermally displaced configurations of a 128^2 case, each a full GPU run atoms -> rings, averaged on the device
    by prism_accumulate; against the mean of the oracle's three full runs."""
    from paper_1706_08563_b200 import prism
    w = W.scaled_test_case(128, 4, 2, 6, alpha_mrad=25.0, defocus=25.0, seed_index=21, density=0.25,
                           z_choices=(79, 33, 14), probe_offset=(0.05, 0.11)).with_(jitter=0.08, n_phonons=3)
    p = oracle_params(w)
    pp = prism.params_from_workload(w)
    n_bins = prism.num_bins(pp)
    acc = torch.full((w.probes_y, w.probes_x, n_bins), float("nan"), dtype=torch.float32, device=G.DEV)
    out = torch.empty_like(acc)
    refs, singles = [], []
    for ph in range(w.n_phonons):
        v = G.gpu_potential(w, phonon=ph)
        s, beams = G.gpu_smatrix(w, v)
        prism.compute_output(pp, s, beams, out, G.ws(pp, prism.WS_OUTPUT))
        prism.accumulate(acc, out, 1.0 / w.n_phonons, first=(ph == 0))
        singles.append(out.cpu().numpy().astype(np.float64).reshape(-1, n_bins))
        v_ref = oracle_potential(w, phonon=ph)
        refs.append(O.prism_probes(p, O.smatrix(p, v_ref, beams), beams, w.probe_xy()))
    torch.cuda.synchronize()
    got = acc.cpu().numpy().astype(np.float64).reshape(-1, n_bins)
    ref = np.mean(refs, axis=0)
    assert rel_l2(got, ref) < TOL_OUT
    d = G.dark_field(w, p)
    assert rel_l2(got[:, d:], ref[:, d:]) < 5 * TOL_OUT
    # the configurations differ, so the mean is not any single run (the test would pass trivially otherwise)
    assert rel_l2(singles[0], ref) > 20 * TOL_OUT
    assert np.allclose(got, np.mean(singles, axis=0), rtol=1e-5, atol=1e-10)


# ---- regular probe lattices: the lattice-DFT form of the beam sum -----------------
def _lattice_cases():
    return {
        # Q = 8, off-pixel origin, 64^2 windows
        "L128f2q8": W.scaled_test_case(128, 3, 2, 16, alpha_mrad=25.0, defocus=30.0, seed_index=11,
                                       probe_offset=(0.137, 0.291)),
        # Q = 32 with 128^2 windows and a 4-pixel step: the shape of BASELINE.json configs 3-5
        "L256f2q32": W.scaled_test_case(256, 3, 2, 64, voltage=300e3, alpha_mrad=20.0, seed_index=12),
        # Q = 16
        "L256f4q16": W.scaled_test_case(256, 2, 4, 64, voltage=300e3, alpha_mrad=20.0, seed_index=13, cs=1.0e4),
        # Q = 16 with beams folded onto the same lattice residue (25 beam indices per axis onto 16)
        "L128f1q16": W.scaled_test_case(128, 2, 1, 16, alpha_mrad=25.0, seed_index=14, density=0.03),
        # probe grid covering part of the cell only, rectangular, origin away from 0
        "L128f2part": W.scaled_test_case(128, 2, 2, 16, alpha_mrad=20.0, seed_index=15).with_(
            probes_x=5, probes_y=7, probe_origin=(1.2, 3.3)),
    }


LATTICE = _lattice_cases()


@pytest.mark.parametrize("name", list(LATTICE))
def test_prism_output_parity_regular_lattice(G, name):
    w = LATTICE[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    out = G.gpu_prism_output(w, s, beams)
    xy = w.probe_xy()
    pick = np.unique(np.linspace(0, len(xy) - 1, 97).astype(int))       # oracle on a spread of probes
    s_ref = O.smatrix(p, oracle_potential(w), beams)
    ref = O.prism_probes(p, s_ref, beams, xy[pick])
    assert rel_l2(out[pick], ref) < TOL_OUT
    d = G.dark_field(w, p)
    assert ref[:, d:].sum() > 0
    assert rel_l2(out[pick][:, d:], ref[:, d:]) < 5 * TOL_OUT
    # the stage in isolation: oracle stage 2 applied to the GPU's own S-matrix, every probe row touched
    rows = np.unique(np.concatenate([np.arange(0, len(xy), 53), [len(xy) - 1]]))
    ref2 = O.prism_probes(p, s.cpu().numpy().astype(np.complex128), beams, xy[rows])
    assert rel_l2(out[rows], ref2) < 2e-5


# ---- large grids: the pipelined slice-step kernels at 1024 and 2048 points per line ---
def _large_cases():
    return {
        # 1024^2 (one-exchange 32 x 32 transform), f=8 -> 128^2 windows, the grid of BASELINE.json config 4
        "T1024f8": W.scaled_test_case(1024, 3, 8, 4, voltage=200e3, alpha_mrad=12.0, defocus=50.0, seed_index=21,
                                      density=0.01),
        # 2048^2 (packed two-way transform, slice_pk.cu), f=16 -> 128^2 windows, the grid of config 5; small aperture keeps
        # the S-matrix of the test at a few GiB
        "T2048f16": W.scaled_test_case(2048, 2, 16, 4, voltage=300e3, alpha_mrad=6.0, seed_index=22,
                                       density=0.004),
    }


LARGE = _large_cases()


@pytest.mark.parametrize("name", list(LARGE))
def test_large_grid_parity(G, name):
    """Oracle by decomposition: sampled S-matrix layers, oracle stage 2 applied to the GPU
    S-matrix for sampled probes, and sampled multislice probes end to end."""
    w = LARGE[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    v_ref = oracle_potential(w)
    assert rel_l2(v.cpu().numpy().astype(np.float64), v_ref) < TOL_V
    s, beams = G.gpu_smatrix(w, v)
    assert set(map(tuple, beams.tolist())) == set(map(tuple, O.beams(p).tolist()))
    pick = np.unique(np.linspace(0, len(beams) - 1, 4).astype(int))
    for b in pick:
        ref = O.smatrix_layer(p, v_ref, int(beams[b, 0]), int(beams[b, 1]))
        assert rel_l2(s[b].cpu().numpy().astype(np.complex128), ref) < TOL_S, (name, b)
    out = G.gpu_prism_output(w, s, beams)
    xy = w.probe_xy()
    rows = np.array([0, 5, len(xy) - 1])
    ref2 = O.prism_probes(p, s.cpu().numpy().astype(np.complex128), beams, xy[rows])
    assert rel_l2(out[rows], ref2) < 2e-5
    if name == "T2048f16":
        # S-matrix in page-locked host memory on the blocked layout (ROW_FINAL staging chunks leave over the copy
        # stream, several beam batches): bit-identical to the resident path
        from paper_1706_08563_b200 import prism
        ph = prism.params_from_workload(w, smatrix_on_host=1, batch=5)
        s_host = torch.empty_like(s, device="cpu").pin_memory()
        b2 = prism.compute_smatrix(ph, v, s_host, G.ws(ph, prism.WS_SMATRIX))
        torch.cuda.synchronize()
        assert np.array_equal(beams, b2) and torch.equal(s_host, s.cpu())
        del s_host
    del s
    ms = G.gpu_multislice(w, v)
    ref3 = O.multislice_probes(p, v_ref, xy[rows])
    assert rel_l2(ms[rows], ref3) < TOL_OUT
    d = G.dark_field(w, p)
    assert rel_l2(ms[rows][:, d:], ref3[:, d:]) < 5 * TOL_OUT


def _odd_grid_cases():
    base = W.scaled_test_case(256, 3, 4, 4, voltage=300e3, alpha_mrad=12.0, seed_index=31, density=0.03)
    lz = base.cell[2]
    return {
        # 512 x 256 grid with square pixels: the pipelined column pass with a run-time row stride
        "R512x256": base.with_(name="R512x256", nx=512, cell=(51.2, 25.6, lz), probe_step=(12.8, 6.4)),
        # 256 x 512 grid
        "R256x512": base.with_(name="R256x512", ny=512, cell=(25.6, 51.2, lz), probe_step=(6.4, 12.8)),
        # 0.1 x 0.2 Angstrom pixels: the band-limit circle is narrower than the default column band in kx
        "A256": base.with_(name="A256", cell=(25.6, 51.2, lz), probe_step=(6.4, 12.8), alpha=8e-3),
        # 2048-point rows / columns on the packed kernels with the other axis short: run-time row stride, ragged
        # line counts, and (anisotropic pixels) a band that is not the compile-time default
        "R2048x256": base.with_(name="R2048x256", f=16, nx=2048, cell=(204.8, 25.6, lz), probe_step=(51.2, 6.4), alpha=6e-3),
        "R256x2048": base.with_(name="R256x2048", f=16, ny=2048, cell=(25.6, 204.8, lz), probe_step=(6.4, 51.2), alpha=6e-3),
        "A2048x256": base.with_(name="A2048x256", f=16, nx=2048, cell=(204.8, 51.2, lz), probe_step=(51.2, 12.8), alpha=5e-3),
        "A256x2048": base.with_(name="A256x2048", f=16, ny=2048, cell=(51.2, 204.8, lz), probe_step=(12.8, 51.2), alpha=5e-3),
    }


ODD = _odd_grid_cases()


@pytest.mark.parametrize("name", list(ODD))
def test_rectangular_grids_and_anisotropic_pixels(G, name):
    w = ODD[name]
    p = oracle_params(w)
    v = G.gpu_potential(w)
    v_ref = oracle_potential(w)
    assert rel_l2(v.cpu().numpy().astype(np.float64), v_ref) < TOL_V
    s, beams = G.gpu_smatrix(w, v)
    s_ref = O.smatrix(p, v_ref, beams)
    assert rel_l2(s.cpu().numpy().astype(np.complex128), s_ref) < TOL_S
    out = G.gpu_prism_output(w, s, beams)
    assert rel_l2(out, O.prism_probes(p, s_ref, beams, w.probe_xy())) < TOL_OUT
    ms = G.gpu_multislice(w, v)
    assert rel_l2(ms, O.multislice_probes(p, v_ref, w.probe_xy())) < TOL_OUT


def test_lattice_path_does_not_depend_on_batch(G):
    from paper_1706_08563_b200 import prism
    w = LATTICE["L128f2part"]
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    out0 = G.gpu_prism_output(w, s, beams)
    for b in [w.probes_x, 3 * w.probes_x + 2, 2]:           # one probe row, three rows, fewer than a row (direct sum)
        out1 = G.gpu_prism_output(w, s, beams, prism.params_from_workload(w, batch=b))
        if b >= w.probes_x:
            assert np.array_equal(out0, out1)
        else:
            assert rel_l2(out1, out0) < 2e-5


def test_prism_f1_equals_multislice_on_gpu(G):
    w = CASES["PR1"]
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    assert rel_l2(G.gpu_prism_output(w, s, beams), G.gpu_multislice(w, v)) < TOL_OUT


def test_results_do_not_depend_on_batch_or_memory_mode(G):
    from paper_1706_08563_b200 import prism
    w = CASES["T128f2"]
    v = G.gpu_potential(w)
    v_host = G.gpu_potential(w, on_host=True)
    assert torch.equal(v.cpu(), v_host)                              # same kernel, staged copy
    s0, beams = G.gpu_smatrix(w, v)
    for kw in [dict(batch=1), dict(batch=5), dict(batch=0)]:
        p = prism.params_from_workload(w, **kw)
        s1, b1 = G.gpu_smatrix(w, v, p)
        assert np.array_equal(beams, b1) and torch.equal(s0, s1)
    s2, _ = G.gpu_smatrix(w, v_host)                                  # streamed from pinned host memory
    assert torch.equal(s0, s2)
    s3, _ = G.gpu_smatrix(w, v_host, prism.params_from_workload(w, batch=7))
    assert torch.equal(s0, s3)
    out0 = G.gpu_prism_output(w, s0, beams)
    for b in [1, 4, 25]:
        assert np.array_equal(out0, G.gpu_prism_output(w, s0, beams, prism.params_from_workload(w, batch=b)))
    assert np.array_equal(out0, G.gpu_prism_output(w, s0, beams, host_out=True))
    m0 = G.gpu_multislice(w, v)
    for b in [1, 3]:
        assert np.array_equal(m0, G.gpu_multislice(w, v, prism.params_from_workload(w, batch=b)))
    assert np.array_equal(m0, G.gpu_multislice(w, v_host, prism.params_from_workload(w, batch=4)))
    assert np.array_equal(m0, G.gpu_multislice(w, v, host_out=True))


def test_empty_specimen_closed_form(G):
    w = CASES["T128f4"]
    w0 = w.with_(atoms=np.zeros((0, 3)), z=np.zeros(0, np.int32))
    p = oracle_params(w0)
    from paper_1706_08563_b200 import prism
    pp = prism.params_from_workload(w0)
    v = torch.zeros((w0.n_slices, w0.ny, w0.nx), dtype=torch.float32, device=G.DEV)
    s, beams = G.gpu_smatrix(w0, v, pp)
    out = G.gpu_prism_output(w0, s, beams, pp)
    lam, _ = O.constants(w0.voltage)
    ang = lam * np.hypot(beams[:, 0] / w0.cell[0], beams[:, 1] / w0.cell[1])
    want = np.bincount(np.floor(ang / w0.det_step).astype(int), minlength=out.shape[1])[:out.shape[1]] / len(beams)
    assert np.max(np.abs(out - want[None, :])) < 2e-6
    ms = G.gpu_multislice(w0, v, pp)
    ref = O.multislice_probes(p, np.zeros((w0.n_slices, w0.ny, w0.nx)), w0.probe_xy()[:1])
    assert np.max(np.abs(ms - ref)) < 2e-6
    # a potential builder call with zero atoms writes zeros
    assert torch.count_nonzero(G.gpu_potential(w0)) == 0


def test_single_slice_and_rectangular_probe_grid(G):
    w = W.scaled_test_case(64, 1, 2, 4, seed_index=5, density=0.2).with_(probes_x=3, probes_y=5,
                                                                       probe_step=(1.3, 0.7))
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    out = G.gpu_prism_output(w, s, beams)
    v_ref = oracle_potential(w)
    ref = O.prism_probes(p, O.smatrix(p, v_ref, beams), beams, w.probe_xy())
    assert out.shape == (15, O.num_bins(p)) and rel_l2(out, ref) < TOL_OUT
    assert rel_l2(G.gpu_multislice(w, v), O.multislice_probes(p, v_ref, w.probe_xy())) < TOL_OUT


def test_resident_multislice_edge_cases(G):
    """The resident multislice kernel (256^2 / 512^2 grids, one probe per SM): a single slice, more
    probes than SMs with a ragged last round, a rectangular probe grid off the pixel lattice, empty space, and
    agreement with the per-pass path (taken when the potential is streamed from host memory)."""
    from paper_1706_08563_b200 import prism
    w = W.scaled_test_case(256, 1, 2, 4, voltage=300e3, alpha_mrad=20.0, seed_index=41, density=0.1).with_(
        probes_x=3, probes_y=5, probe_step=(1.3, 0.7), probe_origin=(0.123, 0.456))
    p = oracle_params(w)
    v = G.gpu_potential(w)
    assert rel_l2(G.gpu_multislice(w, v), O.multislice_probes(p, oracle_potential(w), w.probe_xy())) < TOL_OUT
    # 13 x 13 = 169 probes > 148 SMs, three slices; the oracle on a sample of the probes, the per-pass path on all
    w2 = W.scaled_test_case(256, 3, 2, 13, voltage=300e3, alpha_mrad=20.0, seed_index=42, defocus=35.0)
    p2 = oracle_params(w2)
    v2 = G.gpu_potential(w2)
    out = G.gpu_multislice(w2, v2)
    pick = np.array([0, 1, 77, 147, 148, 149, 168])
    ref = O.multislice_probes(p2, oracle_potential(w2), w2.probe_xy()[pick])
    d = G.dark_field(w2, p2)
    assert rel_l2(out[pick], ref) < TOL_OUT and rel_l2(out[pick][:, d:], ref[:, d:]) < 5 * TOL_OUT
    v2_host = G.gpu_potential(w2, on_host=True)
    per_pass = G.gpu_multislice(w2, v2_host)                        # streamed potential: launch-per-pass kernels
    assert rel_l2(out, per_pass) < 2e-6
    # empty space: rings = aperture pixel counts (closed form through the oracle)
    w0 = w2.with_(atoms=np.zeros((0, 3)), z=np.zeros(0, np.int32))
    v0 = torch.zeros((w0.n_slices, w0.ny, w0.nx), dtype=torch.float32, device=G.DEV)
    ms0 = G.gpu_multislice(w0, v0)
    ref0 = O.multislice_probes(oracle_params(w0), np.zeros((w0.n_slices, w0.ny, w0.nx)), w0.probe_xy()[:1])
    assert np.max(np.abs(ms0 - ref0)) < 2e-6 and abs(ms0.sum(axis=1) - 1.0).max() < 1e-5


def test_error_codes(G):
    from paper_1706_08563_b200 import prism
    w = CASES["PR1"]
    p = prism.params_from_workload(w)
    v = torch.zeros((w.n_slices, w.ny, w.nx), dtype=torch.float32, device=G.DEV)
    s = torch.empty((prism.num_beams(p), w.ny, w.nx), dtype=torch.complex64, device=G.DEV)
    tiny = torch.empty(1024, dtype=torch.uint8, device=G.DEV)
    with pytest.raises(prism.PrismError) as e:
        prism.compute_smatrix(p, v, s, tiny)
    assert e.value.code == prism.PRISM_ENOMEM
    bad = prism.params_from_workload(w, nx=96)
    with pytest.raises(prism.PrismError) as e:
        prism.num_beams(bad)
    assert e.value.code == prism.PRISM_EINVAL
    bad = prism.params_from_workload(w, alpha=0.09)                   # beyond the 2/3 band-limit (83.6 mrad)
    with pytest.raises(prism.PrismError):
        prism.num_beams(bad)
    lut_z, r_cut, lut_v = w.lut()
    with pytest.raises(prism.PrismError) as e:
        prism.build_potential(p, [[1.0, 1.0, 1.0]], [13], lut_z, r_cut, lut_v, v, G.ws(p, prism.WS_POTENTIAL, 1))
    assert e.value.code == prism.PRISM_ENOLUT


def test_repeated_calls_are_bitwise_identical(G):
    """The path has no atomics and a fixed summation order, and the slice loop's kernels are chained by programmatic
    dependent launches: a missing dependency would show up as run-to-run differences."""
    cases = [CASES["T512f8"], LARGE["T1024f8"], ODD["R2048x256"], ODD["A256x2048"]]
    for w in cases:
        v = G.gpu_potential(w)
        assert torch.equal(v, G.gpu_potential(w))
        s0, beams = G.gpu_smatrix(w, v)
        out0 = G.gpu_prism_output(w, s0, beams)
        m0 = G.gpu_multislice(w, v)
        for _ in range(3):
            s1, _ = G.gpu_smatrix(w, v)
            assert torch.equal(s0, s1), w.name
            assert np.array_equal(out0, G.gpu_prism_output(w, s1, beams)), w.name
            assert np.array_equal(m0, G.gpu_multislice(w, v)), w.name
