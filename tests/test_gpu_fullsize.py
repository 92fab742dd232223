"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (whole beam set resident,
library-default batches, streamed potential for P16), on sampled outputs the oracle can compute one by one
(SURVEY.md 8(d) "parity by decomposition"):

  * the whole potential stack against the oracle's;
  * sampled S-matrix layers against oracle layers (each is one plane wave through every slice);
  * sampled probes of stage 2 against the oracle's stage 2 applied to the GPU S-matrix (fp64 copy);
  * sampled multislice probes end to end.

Tolerances: output rings 1e-4 relative L2 (1e-3 at 2048^2 with >= 400 slices), BASELINE.json north_star;
S-matrix layers 3e-7 sqrt(S) x 20; stage 2 in isolation 2e-5.

The 400-slice 2048^2 oracle costs ~5-10 core-minutes per wave, so config 5 is run twice: on its first 40 slices
(same grid, beams, streaming ring, kernels) with several layers, stage 2 and multislice probes, and at its full
400 slices on one S-matrix layer and one multislice probe (the two oracle waves run on host threads while the
GPU works).  Config 3 (P4) is also checked end to end, atoms -> rings, against the full oracle."""
import math
import threading

import numpy as np
import pytest

import oracle as O
from helpers import oracle_params, oracle_potential, rel_l2
from paper_1706_08563_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_OUT = 1e-4
TOL_V = 1e-6
TOL_STAGE2 = 2e-5


def tol_layer(n_slices):
    return 20.0 * 3e-7 * math.sqrt(n_slices)


@pytest.fixture(scope="module")
def G():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import gpu_helpers
    return gpu_helpers


def spread(n, k):
    return np.unique(np.linspace(0, n - 1, k).astype(int))


def check_prism(G, w, n_layers, n_probes, beam_filter=None, tol_out=TOL_OUT):
    """Potential, sampled layers, stage 2 on sampled probes.  beam_filter(beams) -> mask selects the layers
    stage 2 is run on when the fp64 copy of the whole S-matrix would not fit in host memory."""
    p = oracle_params(w)
    on_host = bool(w.potential_on_host)
    v = G.gpu_potential(w, on_host=on_host)
    v_ref = oracle_potential(w)
    v_gpu = v.cpu().numpy() if not on_host else v.numpy()
    assert rel_l2(v_gpu.astype(np.float64), v_ref) < TOL_V
    del v_gpu
    s, beams = G.gpu_smatrix(w, v)
    ref_beams = O.beams(p)
    assert set(map(tuple, beams.tolist())) == set(map(tuple, ref_beams.tolist()))
    pick = spread(len(beams), n_layers)
    layers = O.smatrix(p, v_ref, beams[pick])
    errs = [rel_l2(s[b].cpu().numpy().astype(np.complex128), layers[i]) for i, b in enumerate(pick)]
    assert max(errs) < tol_layer(w.n_slices), errs
    del layers
    # stage 2 in isolation on the layers the host can hold in fp64
    if beam_filter is None:
        sel = np.arange(len(beams))
        s_sel = s
    else:
        sel = np.nonzero(beam_filter(beams))[0]
        s_sel = s[torch.as_tensor(sel, device=s.device)].contiguous()
    out = G.gpu_prism_output(w, s_sel, np.ascontiguousarray(beams[sel]))
    xy = w.probe_xy()
    rows = spread(len(xy), n_probes)
    s64 = s_sel.cpu().numpy().astype(np.complex128)
    ref = O.prism_probes(p, s64, np.ascontiguousarray(beams[sel]), xy[rows])
    assert rel_l2(out[rows], ref) < TOL_STAGE2
    d = G.dark_field(w, p)
    assert ref[:, d:].sum() > 0
    assert rel_l2(out[rows][:, d:], ref[:, d:]) < 5 * tol_out
    # every probe of the grid: the rings hold about the incident current (PRISM's cropped window is not exactly
    # norm-conserving for f > 1, so this is a sanity band, not an identity)
    tot = out.sum(axis=1)
    assert np.all(tot > 0.5) and np.all(tot < 1.05)
    if beam_filter is not None:
        check_stage2_all_beams_on_row_bands(G, w, p, s, beams, tol_out)
    return v, v_ref, errs


def check_stage2_all_beams_on_row_bands(G, w, p, s, beams, tol_out, n_probes=8):
    """Stage 2 with EVERY beam at sizes where the fp64 copy of the whole S-matrix does not fit in host memory (80 GB at
    config 5): for one probe row, only the ny / f pixel rows its windows touch are brought to the host in fp64 (5 GB at
    config 5) and the oracle's band-of-rows entry (O.prism_probe_rows: the loop of O.prism_probe on that storage) gives
    the rings of sampled probes of the row.  Two probe rows: probe row 0, whose windows wrap the cell edge in y, and one
    in the middle of the grid."""
    out = G.gpu_prism_output(w, s, beams)                  # all beams, the launch configuration bench.py times
    xy = w.probe_xy().reshape(w.probes_y, w.probes_x, 2)
    my, py = w.ny // w.f, w.cell[1] / w.ny
    d = G.dark_field(w, p)
    for iy in (0, (w.probes_y // 2) + 3):
        jc = int(np.floor(xy[iy, 0, 1] / py + 0.5))
        row0 = (jc - my // 2) % w.ny
        if iy == 0:
            assert row0 + my > w.ny                        # this band wraps the cell edge
        idx = torch.as_tensor((row0 + np.arange(my)) % w.ny, device=s.device)
        band = s.index_select(1, idx).cpu().numpy().astype(np.complex128)
        cols = spread(w.probes_x, n_probes)
        ref = np.stack([O.prism_probe_rows(p, band, row0, beams, *xy[iy, ix]) for ix in cols])
        del band
        got = out.reshape(w.probes_y, w.probes_x, -1)[iy, cols]
        e, e_dark = rel_l2(got, ref), rel_l2(got[:, d:], ref[:, d:])
        print(f"{w.name} stage 2, all {len(beams)} beams, probe row {iy} (band from pixel row {row0}): "
              f"rings {e:.3e}, dark field {e_dark:.3e}")
        assert e < TOL_STAGE2, iy
        assert ref[:, d:].sum() > 0
        assert e_dark < 5 * tol_out, iy


def check_multislice(G, w, v, v_ref, n_probes, tol_out=TOL_OUT):
    p = oracle_params(w)
    out = G.gpu_multislice(w, v)
    xy = w.probe_xy()
    rows = spread(len(xy), n_probes)
    ref = O.multislice_probes(p, v_ref, xy[rows])
    e = rel_l2(out[rows], ref)
    assert e < tol_out, e
    d = G.dark_field(w, p)
    assert rel_l2(out[rows][:, d:], ref[:, d:]) < 5 * tol_out
    tot = out.sum(axis=1)
    assert np.all(tot > 0.0) and np.all(tot < 1.0 + 1e-4)
    return e


def test_ms2_full(G):
    """BASELINE.json configs[1]: 256^2, 50 slices, 32 x 32 probes.  The configuration's batch of 64 sizes the per-pass
    path only: on this grid the ring output takes the resident route (one launch, one probe per SM in flight), which
    ignores `batch`; results do not depend on the route (test_resident_multislice_edge_cases)."""
    w = W.ms2()
    assert w.batch == 64
    v = G.gpu_potential(w)
    v_ref = oracle_potential(w)
    assert rel_l2(v.cpu().numpy().astype(np.float64), v_ref) < TOL_V
    check_multislice(G, w, v, v_ref, 48)


def test_p4_full(G):
    """BASELINE.json configs[2]: 512^2, 100 slices, f = 4, 529 beams, 128 x 128 probes."""
    check_prism(G, W.p4(), n_layers=4, n_probes=12)


def test_p4_full_patterns(G):
    """4-D output at config 3's size (16384 patterns of 128^2): sampled patterns against the oracle's stage 2 applied
    to the GPU S-matrix, pixel by pixel, and the rings as sums of their pixels."""
    from paper_1706_08563_b200 import prism
    w = W.p4()
    p = oracle_params(w)
    pp = prism.params_from_workload(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    m = w.nx // w.f
    pat = torch.empty((w.n_probes, m, m), dtype=torch.float32, device=G.DEV)
    prism.compute_patterns(pp, s, beams, pat, G.ws(pp, prism.WS_OUTPUT))
    out = G.gpu_prism_output(w, s, beams)
    s64 = s.cpu().numpy().astype(np.complex128)
    xy = w.probe_xy()
    for i in spread(len(xy), 6):
        _, ref = O.prism_probe(p, s64, beams, xy[i, 0], xy[i, 1], want_pattern=True)
        got = pat[i].cpu().numpy().astype(np.float64)
        assert rel_l2(got, ref) < TOL_STAGE2, i
        assert np.allclose(O.bin_intensity(p, got, w.f, w.f), out[i], rtol=1e-5, atol=1e-9)
    tot = pat.sum(dim=(1, 2)).cpu().numpy()
    assert np.all(tot > 0.5) and np.all(tot < 1.05)


def test_p8_full(G):
    """BASELINE.json configs[3]: 1024^2, 50 slices, f = 8, 509 beams, 256 x 256 probes, defocus 50 A."""
    check_prism(G, W.p8(), n_layers=4, n_probes=12)


def p16_cases(n_slices):
    """Config 5 on its first n_slices slices: atoms above the truncated stack are dropped (not clamped into the
    last slice), everything else -- grid, beams, streamed potential, probe lattices -- is config 5."""
    w = W.p16_first_slices(n_slices)
    wm = w.with_(name="P16-MS", probes_x=64, probes_y=64, probe_step=(3.2, 3.2))
    return w, wm


def run_p16(G, n_slices, n_layers, n_ms_probes, tol_out):
    w, wm = p16_cases(n_slices)
    assert w.potential_on_host == 1 and w.nx == 2048 and w.f == 16
    # stage 2 on the three central rows of the beam lattice (|ky / f| <= 1): 39 beam columns fold onto the
    # 32 residues of the probe lattice, so the folded path of the lattice DFT is exercised (117 of 1201 layers)
    v, v_ref, errs = check_prism(G, w, n_layers=n_layers, n_probes=6,
                                 beam_filter=lambda b: np.abs(b[:, 1]) <= w.f, tol_out=tol_out)
    torch.cuda.empty_cache()
    e = check_multislice(G, wm, v, v_ref, n_ms_probes, tol_out=tol_out)
    print(f"P16 x {n_slices} slices: S-matrix layer errors {errs}, multislice rings {e:.3e}")


def test_p16_first_40_slices(G):
    """BASELINE.json configs[4] (2048^2, f = 16, 1201 beams, 512 x 512 probes, potential streamed from pinned
    host memory; multislice on 64 x 64 probes), first 40 of the 400 slices."""
    run_p16(G, 40, n_layers=2, n_ms_probes=2, tol_out=TOL_OUT)


class _P16OracleJob:
    """The 400-slice oracle waves of config 5: three S-matrix layers (the axial beam, an oblique one, one on the
    aperture edge) and two multislice probes, 4-9 min each on one core, each on its own host thread from the moment
    the module's first test begins, so that they overlap the other full-size tests."""

    def __init__(self):
        self.w, self.wm = p16_cases(400)
        self.p, self.pm = oracle_params(self.w), oracle_params(self.wm)
        self.beams_ref = O.beams(self.p)
        b = self.beams_ref.astype(np.int64)
        q2 = b[:, 0] ** 2 + b[:, 1] ** 2
        self.b_picks = {"axial": int(np.argmin(q2)), "oblique": len(b) // 3, "edge": int(np.argmax(q2))}
        assert q2[self.b_picks["axial"]] == 0 and len(set(self.b_picks.values())) == 3
        self.xy = self.wm.probe_xy()
        i_mid = int(spread(len(self.xy), 5)[2]) + 7        # away from the cell corner and from lattice symmetry points
        self.i_probes = [i_mid, int(spread(len(self.xy), 5)[1]) + 29]
        self.ref, self.v_ref, self.error = {}, None, None
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()

    def _run(self):
        try:
            self.v_ref = oracle_potential(self.w)          # ctypes releases the GIL inside the oracle calls

            def layer(name):
                kx, ky = (int(x) for x in self.beams_ref[self.b_picks[name]])
                self.ref["layer_" + name] = O.smatrix_layer(self.p, self.v_ref, kx, ky)

            def probe(i):
                self.ref["rings_%d" % i] = O.multislice_probe(self.pm, self.v_ref, *self.xy[i])

            ts = [threading.Thread(target=layer, args=(name,)) for name in self.b_picks]
            ts += [threading.Thread(target=probe, args=(i,)) for i in self.i_probes]
            for t in ts:
                t.start()
            for t in ts:
                t.join()
        except Exception as exc:                           # surfaced by the test that joins
            self.error = exc


_p16_job = None


@pytest.fixture(scope="module", autouse=True)
def p16_oracle_job(request, G):
    global _p16_job
    wanted = any("test_p16_full_400_slices" in item.nodeid for item in request.session.items)
    if wanted and _p16_job is None:
        _p16_job = _P16OracleJob()
    yield _p16_job


def test_p4_end_to_end_full_oracle(G):
    """BASELINE.json configs[2] end to end, atoms -> rings, against the FULL oracle (SURVEY.md 8(d) "Configs 1-4 get
    the full oracle"): the oracle's own potential, its own S-matrix of all 529 beams through all 100 slices, and its
    stage 2 on 24 probes spread over the grid; the GPU runs the whole path on its own.  Tolerance 1e-4 on the rings
    (BASELINE.json north_star), 5e-4 on the dark field alone."""
    w = W.p4()
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    out = G.gpu_prism_output(w, s, beams)
    del s
    torch.cuda.empty_cache()
    v_ref = oracle_potential(w)
    beams_ref = O.beams(p)
    assert len(beams_ref) == 529
    s_ref = O.smatrix(p, v_ref, beams_ref)              # 52 900 beam-slices at 512^2: ~2-4 min on 16 cores
    xy = w.probe_xy()
    rows = spread(len(xy), 24)
    ref = O.prism_probes(p, s_ref, beams_ref, xy[rows])
    e = rel_l2(out[rows], ref)
    d = G.dark_field(w, p)
    e_dark = rel_l2(out[rows][:, d:], ref[:, d:])
    print(f"P4 end to end vs full oracle: rings {e:.3e}, dark field {e_dark:.3e}")
    assert ref[:, d:].sum() > 0
    assert e < TOL_OUT, e
    assert e_dark < 5 * TOL_OUT, e_dark


def test_p8_end_to_end_full_oracle(G):
    """BASELINE.json configs[3] end to end for one frozen-phonon configuration, atoms -> rings, against the FULL oracle:
    its own potential, its own S-matrix of all 509 beams through all 50 slices at 1024^2 (25 450 beam-slices, a few
    minutes on 16 cores, 8.5 GB of complex128) and its stage 2 (defocus 50 A) on 12 probes spread over the grid."""
    w = W.p8()
    p = oracle_params(w)
    v = G.gpu_potential(w)
    s, beams = G.gpu_smatrix(w, v)
    out = G.gpu_prism_output(w, s, beams)
    del s, v
    torch.cuda.empty_cache()
    v_ref = oracle_potential(w)
    beams_ref = O.beams(p)
    assert len(beams_ref) == 509
    s_ref = O.smatrix(p, v_ref, beams_ref)
    xy = w.probe_xy()
    rows = spread(len(xy), 12)
    ref = O.prism_probes(p, s_ref, beams_ref, xy[rows])
    del s_ref
    e = rel_l2(out[rows], ref)
    d = G.dark_field(w, p)
    e_dark = rel_l2(out[rows][:, d:], ref[:, d:])
    print(f"P8 end to end vs full oracle: rings {e:.3e}, dark field {e_dark:.3e}")
    assert ref[:, d:].sum() > 0
    assert e < TOL_OUT, e
    assert e_dark < 5 * TOL_OUT, e_dark


def test_p16_prism_rings_against_stored_oracle_rings(G):
    """Config 5 end to end on its first slices -- atoms -> streamed potential -> all 1201 layers -> stage 2 -- against
    PRISM rings the ORACLE ALONE produced for sampled probes of two probe rows (tests/golden/p16_s10_rings.txt,
    written by tests/golden/make_p16_rings.py, which calls only oracle/ and workloads.py; 12 010 oracle beam-slices,
    ~45 min on 8 cores, hence 10 slices and not 400: the depth is covered layer by layer in test_p16_full_400_slices)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "p16_s10_rings.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    pick = np.array([[int(r[0]), int(r[1])] for r in rows])
    ref = np.array([[float(x) for x in r[2:]] for r in rows])
    w = W.p16_first_slices(10)
    p = oracle_params(w)
    assert ref.shape == (len(pick), O.num_bins(p)) and len(pick) >= 8
    v = G.gpu_potential(w, on_host=True)
    s, beams = G.gpu_smatrix(w, v)
    out = G.gpu_prism_output(w, s, beams).reshape(w.probes_y, w.probes_x, -1)
    got = out[pick[:, 0], pick[:, 1]]
    d = G.dark_field(w, p)
    e, e_dark = rel_l2(got, ref), rel_l2(got[:, d:], ref[:, d:])
    print(f"P16 x 10 slices end to end vs stored oracle rings ({len(pick)} probes): rings {e:.3e}, dark field {e_dark:.3e}")
    assert ref[:, d:].sum() > 0
    assert e < TOL_OUT and e_dark < 5 * TOL_OUT, (e, e_dark)
    for k in range(len(pick)):                              # and probe by probe
        assert rel_l2(got[k], ref[k]) < TOL_OUT, pick[k]


def test_p16_full_400_slices(G, p16_oracle_job):
    """Config 5 at its full depth (2048^2, all 400 slices streamed from pinned host memory, 1201 beams resident):
    three S-matrix layers (axial, oblique, aperture-edge beam) against the oracle's, and two probes of the 64 x 64
    multislice run end to end against the oracle's rings at the 1e-3 of BASELINE.json north_star ("1e-3 for 2048^2
    grids with >= 400 slices").  The five oracle waves (400 slices each, ~4-9 min on one core) run on host threads
    from the start of this module."""
    job = p16_oracle_job
    w, wm, p, pm = job.w, job.wm, job.p, job.pm
    assert w.n_slices == 400 and w.potential_on_host == 1
    beams_ref = job.beams_ref
    try:
        v = G.gpu_potential(w, on_host=True)
        s, beams = G.gpu_smatrix(w, v)
        assert np.array_equal(beams, beams_ref) or set(map(tuple, beams.tolist())) == set(map(tuple, beams_ref.tolist()))
        layers_gpu = {}
        for name, b_pick in job.b_picks.items():
            b_gpu = int(np.nonzero((beams == beams_ref[b_pick]).all(axis=1))[0][0])
            layers_gpu[name] = s[b_gpu].cpu().numpy().astype(np.complex128)
        del s
        torch.cuda.empty_cache()
        out = G.gpu_multislice(wm, v)
    finally:
        job.thread.join()
    assert job.error is None, job.error
    ref = job.ref
    assert rel_l2(v.numpy().astype(np.float64), job.v_ref) < TOL_V
    e_layers = {name: rel_l2(layers_gpu[name], ref["layer_" + name]) for name in job.b_picks}
    d = G.dark_field(wm, pm)
    e_rings = [rel_l2(out[i], ref["rings_%d" % i]) for i in job.i_probes]
    e_dark = [rel_l2(out[i][d:], ref["rings_%d" % i][d:]) for i in job.i_probes]
    print(f"P16 x 400 slices: S-matrix layers {e_layers}, multislice rings {e_rings}, dark field {e_dark}")
    assert max(e_layers.values()) < tol_layer(400), e_layers
    assert max(e_rings) < 1e-3 and max(e_dark) < 5e-3, (e_rings, e_dark)
    tot = out.sum(axis=1)
    assert np.all(tot > 0.0) and np.all(tot < 1.0 + 1e-3)
    job.v_ref = None
