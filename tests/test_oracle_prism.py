"""Pins for the oracle's multislice / PRISM drivers (O5-O12 of DESIGN.md):
closed forms for empty space, the PRISM(f=1) == multislice identity
(PAPER.md:84 linearity), brute force with the naive DFT, symmetry and
translation invariants, and window-placement checks with synthetic S-matrices.
CPU only."""
import os

import numpy as np
import pytest

import oracle as O
from helpers import freq, oracle_params, oracle_potential, rel_l2
from paper_1706_08563_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def params(n=64, **kw):
    base = dict(lx=0.1 * n, ly=0.1 * n, lz=8.0, nx=n, ny=n, n_slices=4, dz=2.0, voltage=200e3,
                alpha=20e-3, f=1, det_step=1e-3, det_max=60e-3)
    base.update(kw)
    return O.Params(**base)


def count_bins(p, kx, ky, fx=1, fy=1):
    """Independent (numpy) count of lattice points per detector ring."""
    lam, _ = O.constants(p.voltage)
    ang = lam * np.sqrt((kx * fx / p.lx) ** 2 + (ky * fy / p.ly) ** 2)
    b = np.floor(ang / p.det_step).astype(int)
    nb = int(round(p.det_max / p.det_step))
    return np.bincount(b[b < nb], minlength=nb)[:nb].astype(float)


# ----------------------------------------------------------------------------- beams (O8)
def test_beam_counts_match_golden_and_brute_force():
    for name, n, kv, a_mrad, f, n_b, _ in _rows("beam_counts.txt"):
        n, f = int(n), int(f)
        p = params(n, voltage=float(kv) * 1e3, alpha=float(a_mrad) * 1e-3, f=f)
        b = O.beams(p)
        assert len(b) == int(n_b), name
        lam, _ = O.constants(p.voltage)
        k = freq(n)
        kx, ky = np.meshgrid(k, k, indexing="xy")
        sel = (kx % f == 0) & (ky % f == 0) & ((kx / p.lx) ** 2 + (ky / p.ly) ** 2 <= (p.alpha / lam) ** 2)
        assert np.count_nonzero(sel) == len(b)
        assert set(map(tuple, b.tolist())) == set(zip(kx[sel].tolist(), ky[sel].tolist()))


def test_beams_lattice_properties():
    p = params(128, f=4, alpha=30e-3)
    b = O.beams(p)
    assert np.all(b % 4 == 0)
    s = set(map(tuple, b.tolist()))
    assert (0, 0) in s and len(s) == len(b)
    assert all((-kx, -ky) in s and (ky, kx) in s for kx, ky in s)


# ----------------------------------------------------------------------------- empty space
def test_empty_space_multislice_counts_aperture_pixels():
    p = params(64)
    v = np.zeros((4, 64, 64))
    k = freq(64)
    kx, ky = np.meshgrid(k, k, indexing="xy")
    lam, _ = O.constants(p.voltage)
    ap = (kx / p.lx) ** 2 + (ky / p.ly) ** 2 <= (p.alpha / lam) ** 2
    want = count_bins(p, kx[ap], ky[ap]) / np.count_nonzero(ap)
    for xp, yp in [(0.0, 0.0), (1.23, 4.56)]:
        out = O.multislice_probe(p, v, xp, yp)
        assert np.max(np.abs(out - want)) < 1e-12
        assert abs(out.sum() - 1.0) < 1e-12


@pytest.mark.parametrize("f", [1, 2, 4])
def test_empty_space_prism_counts_beams(f):
    p = params(64, f=f, alpha=30e-3)
    v = np.zeros((4, 64, 64))
    b = O.beams(p)
    s = O.smatrix(p, v, b)
    want = count_bins(p, b[:, 0].astype(float), b[:, 1].astype(float)) / len(b)
    for xp, yp in [(0.0, 0.0), (3.17, 0.42)]:
        out = O.prism_probe(p, s, b, xp, yp)
        assert np.max(np.abs(out - want)) < 1e-12


def test_smatrix_layer_empty_space_is_the_propagated_plane_wave():
    p = params(64, n_slices=3)
    lam, _ = O.constants(p.voltage)
    y, x = np.mgrid[0:64, 0:64]
    layer = O.smatrix_layer(p, np.zeros((3, 64, 64)), 4, -6)
    q2 = (16 + 36) / 6.4 ** 2
    want = np.exp(2j * np.pi * (4 * x - 6 * y) / 64) * np.exp(-1j * np.pi * lam * q2 * 6.0)
    assert np.max(np.abs(layer - want)) < 1e-12


# ----------------------------------------------------------------------------- identity and linearity
def test_prism_f1_equals_multislice_on_pr1():
    w = W.pr1()
    p = oracle_params(w)
    v = oracle_potential(w)
    b = O.beams(p)
    s = O.smatrix(p, v, b)
    xy = w.probe_xy()
    a = O.prism_probes(p, s, b, xy)
    m = O.multislice_probes(p, v, xy)
    assert rel_l2(a, m) < 1e-12
    dark = slice(21, None)                       # rings beyond the 20 mrad probe
    assert m[:, dark].sum() > 0
    assert rel_l2(a[:, dark], m[:, dark]) < 1e-10
    # exact (non-pixel) probe positions go into the phase (reading R9)
    out_p = O.prism_probe(p, s, b, 1.234, 5.678)
    out_m = O.multislice_probe(p, v, 1.234, 5.678)
    assert rel_l2(out_p, out_m) < 1e-12


def test_smatrix_is_linear_in_the_incident_wave():
    w = W.pr1()
    p = oracle_params(w)
    v = oracle_potential(w)
    b = O.beams(p)[:5]
    s = O.smatrix(p, v, b)
    rng = np.random.default_rng(8)
    c = rng.normal(size=5) + 1j * rng.normal(size=5)
    y, x = np.mgrid[0:64, 0:64]
    psi0 = sum(ci * np.exp(2j * np.pi * (kx * x + ky * y) / 64) for ci, (kx, ky) in zip(c, b))
    assert rel_l2(O.multislice_wave(p, v, psi0), np.tensordot(c, s, axes=1)) < 1e-12


def test_brute_force_naive_dft_everywhere():
    w = W.scaled_test_case(8, 2, 1, 2, alpha_mrad=40.0, density=0.6, det_max_mrad=160.0)
    w = w.with_(cell=(1.6, 1.6, 4.0))                     # 0.2 A pixels so the atoms fit
    p = oracle_params(w)
    lut_z, r_cut, lut_v = w.lut()
    xyz = w.atoms_for_phonon(0) * np.array([2.0, 2.0, 1.0])
    with pytest.raises(ValueError):
        O.potential(p, xyz, w.z, lut_z, r_cut, lut_v)     # 2 r_cut >= 1.6 A: refused
    lut_v = lut_v[:, :513]                                # same table cut at 0.5 A
    v = O.potential(p, xyz, w.z, lut_z, 0.5, lut_v)
    assert np.count_nonzero(v) > 20
    b = O.beams(p)
    s_fast, s_slow = O.smatrix(p, v, b), O.smatrix(p, v, b, use_naive=True)
    assert rel_l2(s_fast, s_slow) < 1e-12
    for xp, yp in w.probe_xy():
        assert rel_l2(O.multislice_probe(p, v, xp, yp), O.multislice_probe(p, v, xp, yp, use_naive=True)) < 1e-12
        assert rel_l2(O.prism_probe(p, s_fast, b, xp, yp), O.prism_probe(p, s_slow, b, xp, yp, use_naive=True)) < 1e-12


# ----------------------------------------------------------------------------- invariants
def test_translation_by_whole_pixels_changes_nothing():
    w = W.scaled_test_case(64, 3, 2, 2)
    p = oracle_params(w)
    lut_z, r_cut, lut_v = w.lut()
    xyz = w.atoms_for_phonon(0)
    shift = np.array([1.7, -2.3, 0.0])                    # 17 and -23 pixels
    moved = xyz + shift
    moved[:, :2] %= 6.4
    v0 = O.potential(p, xyz, w.z, lut_z, r_cut, lut_v)
    v1 = O.potential(p, moved, w.z, lut_z, r_cut, lut_v)
    b = O.beams(p)
    s0, s1 = O.smatrix(p, v0, b), O.smatrix(p, v1, b)
    for xp, yp in [(0.8, 3.1), (6.0, 0.1)]:
        xq, yq = (xp + 1.7) % 6.4, (yp - 2.3) % 6.4
        assert rel_l2(O.multislice_probe(p, v1, xq, yq), O.multislice_probe(p, v0, xp, yp)) < 1e-11
        assert rel_l2(O.prism_probe(p, s1, b, xq, yq), O.prism_probe(p, s0, b, xp, yp)) < 1e-11


def test_uniform_potential_offset_is_a_global_phase():
    w = W.pr1()
    p = oracle_params(w)
    v = oracle_potential(w)
    a = O.multislice_probe(p, v, 2.4, 3.2)
    b = O.multislice_probe(p, v + 1234.5, 2.4, 3.2)
    assert rel_l2(b, a) < 1e-11


def test_fourfold_symmetry_of_a_centred_atom():
    p = params(64, n_slices=2, alpha=30e-3)
    lut_z, r_cut, lut_v = np.array([79], np.int32), 1.0, (158.0 * np.exp(-(np.arange(1025) / 1024.0) ** 2 / 0.18))[None]
    v = O.potential(p, [[3.2, 3.2, 1.0]], [79], lut_z, r_cut, lut_v)
    _, pat = O.multislice_probe(p, v, 3.2, 3.2, want_pattern=True)
    k = freq(64)
    rot = np.empty_like(pat)                               # I(kx, ky) -> I(-ky, kx)
    for my in range(64):
        for mx in range(64):
            rot[my, mx] = pat[k[mx] % 64, (-k[my]) % 64]
    ok = np.ones((64, 64), bool)
    ok[32, :] = ok[:, 32] = False                          # the unpaired -N/2 line has no rotated partner
    assert pat[ok].max() > 0 and np.max(np.abs(rot - pat)[ok]) < 1e-12 * pat.max() + 1e-18
    assert np.count_nonzero(pat > 1e-9) > 200              # scattering beyond the bright disc exists


def test_single_slice_reduces_to_library_transform():
    w = W.pr1()
    p = oracle_params(w).__class__(**{**oracle_params(w).__dict__, "n_slices": 1})
    v = oracle_potential(w)[:1]
    _, sig = O.constants(p.voltage)
    psi0 = O.probe(p, 2.4, 1.6)
    spec = np.fft.fft2(psi0 * np.exp(1j * sig * v[0]))
    inten = np.where(O.propagator(p) != 0, abs(spec) ** 2, 0.0) / 64 ** 2
    out, pat = O.multislice_probe(p, v, 2.4, 1.6, want_pattern=True)
    assert np.max(np.abs(pat - inten)) < 1e-13
    assert rel_l2(out, O.bin_intensity(p, inten)) < 1e-12


def test_total_intensity_never_exceeds_one():
    w = W.scaled_test_case(64, 6, 2, 3, z_choices=(79,), density=0.08, det_max_mrad=200.0)
    p = oracle_params(w)
    v = oracle_potential(w)
    out = O.multislice_probes(p, v, w.probe_xy())
    assert np.all(out.sum(axis=1) <= 1.0 + 1e-12) and np.all(out.sum(axis=1) > 0.5)
    assert np.all(out >= 0)


# ----------------------------------------------------------------------------- PRISM window (O10)
def test_prism_window_placement_with_a_point_smatrix():
    n, f = 64, 4
    m = n // f                                            # 16-pixel window
    p = params(n, f=f, alpha=30e-3)
    b = O.beams(p)
    nb = len(b)

    def total(i0, j0, xp, yp):
        s = np.zeros((nb, n, n), complex)
        s[:, j0, i0] = 1.0
        return O.prism_probe(p, s, b, xp, yp, want_pattern=True)[1].sum()

    lam, _ = O.constants(p.voltage)
    xp, yp = 2.0, 3.0                                     # centre pixel (20, 30) -> window [12,28) x [22,38)
    coef = np.exp(-2j * np.pi * (b[:, 0] * xp + b[:, 1] * yp) / 6.4)
    inside = abs(coef.sum()) ** 2 / (nb * m * m)           # Parseval on the M x M window
    assert abs(total(12, 22, xp, yp) - inside) < 1e-12    # first pixel of the window
    assert abs(total(27, 37, xp, yp) - inside) < 1e-12    # last pixel of the window
    assert total(28, 30, xp, yp) == 0.0 and total(11, 30, xp, yp) == 0.0
    assert total(20, 38, xp, yp) == 0.0 and total(20, 21, xp, yp) == 0.0
    # periodic wrap: probe at the origin -> window [-8, 8) wraps to [56,64) U [0,8)
    assert total(60, 3, 0.0, 0.0) > 0 and total(3, 60, 0.0, 0.0) > 0 and total(8, 0, 0.0, 0.0) == 0.0
    # centre pixel is round-half-up: x = 0.25 A is pixel 2.5 -> 3 -> window [-5, 11)
    assert total(10, 0, 0.25, 0.0) > 0 and total(58, 0, 0.25, 0.0) == 0.0


def test_prism_pattern_location_and_aberration_coefficient():
    # S = plane waves (empty space): probe pattern has |coef_b|^2 / N_b at beam b's window frequency
    n, f = 64, 2
    p = params(n, f=f, alpha=30e-3, defocus=120.0, cs=1.0e6)
    b = O.beams(p)
    s = O.smatrix(p, np.zeros((4, n, n)), b)
    _, pat = O.prism_probe(p, s, b, 1.1, 2.2, want_pattern=True)
    want = np.zeros((32, 32))
    for kx, ky in b:
        want[(ky // f) % 32, (kx // f) % 32] += 1.0 / len(b)
    assert np.max(np.abs(pat - want)) < 1e-12
    # the aberration enters as a per-beam phase: two beams' interference fixes its sign and size
    lam, _ = O.constants(p.voltage)
    sel = np.array([[0, 0], [4, 2]], np.int32)
    s2 = np.zeros((2, n, n), complex)
    s2[:, 10, 12] = 1.0                                    # same pixel: |c0 + c1|^2 shows the relative phase
    xp, yp = 1.0, 1.0
    _, pat2 = O.prism_probe(p, s2, sel, xp, yp, want_pattern=True)
    q2 = (16 + 4) / 6.4 ** 2
    chi = np.pi * lam * q2 * 120.0 + 0.5 * np.pi * 1.0e6 * lam ** 3 * q2 ** 2
    c1 = np.exp(-1j * chi - 2j * np.pi * (4 * xp + 2 * yp) / 6.4)
    assert abs(pat2.sum() - abs(1.0 + c1) ** 2 / (2 * 32 * 32)) < 1e-13


def test_prism_f2_approaches_multislice_in_coarse_rings():
    # negligible error once the window holds most of the probe.  Not a gate on
    # accuracy, only a sanity bound (SURVEY measured 3.5e-3 on a 6.4 A cell).
    w = W.pr1()
    p2 = O.Params(**{**oracle_params(w).__dict__, "f": 2, "det_step": 10e-3})
    v = oracle_potential(w)
    b = O.beams(p2)
    s = O.smatrix(p2, v, b)
    a = O.prism_probes(p2, s, b, w.probe_xy()[:8])
    m = O.multislice_probes(p2, v, w.probe_xy()[:8])
    assert rel_l2(a, m) < 5e-2


def test_batched_drivers_equal_single_calls():
    w = W.pr1()
    p = oracle_params(w)
    v = oracle_potential(w)
    xy = w.probe_xy()[5:9]
    b = O.beams(p)
    s = O.smatrix(p, v, b)
    ms = O.multislice_probes(p, v, xy)
    pr = O.prism_probes(p, s, b, xy)
    for i, (xp, yp) in enumerate(xy):
        assert np.array_equal(ms[i], O.multislice_probe(p, v, xp, yp))
        assert np.array_equal(pr[i], O.prism_probe(p, s, b, xp, yp))
    assert np.array_equal(s[3], O.smatrix_layer(p, v, *b[3]))


# ----------------------------------------------------------------------------- band-of-rows storage (O10, storage only)
def _band(s, row0, n_rows):
    ny = s.shape[1]
    return np.ascontiguousarray(s[:, (row0 + np.arange(n_rows)) % ny, :])


@pytest.mark.parametrize("f", [1, 4])
def test_prism_probe_rows_is_bit_identical_to_the_whole_grid(f):
    """orc_prism_probe_rows sees only the pixel rows [row0, row0 + n_rows) of every layer; for any band that holds the
    probe's window it must give the whole-grid result bit for bit (same loop, same order): PR1 (f = 1: the band is the
    whole grid, rotated), an f = 4 window inside a band, and a band that wraps the cell edge."""
    w = W.pr1()
    p = oracle_params(w) if f == 1 else params(64, f=4, alpha=30e-3)
    rng = np.random.default_rng(99)
    b = O.beams(p)
    if f == 1:
        s = O.smatrix(p, oracle_potential(w), b)
    else:
        s = rng.normal(size=(len(b), 64, 64)) + 1j * rng.normal(size=(len(b), 64, 64))
    m = 64 // f
    for xp, yp in [(2.0, 3.0), (0.0, 0.0), (6.35, 0.25), (1.23, 5.9)]:
        want, want_pat = O.prism_probe(p, s, b, xp, yp, want_pattern=True)
        jc = int(np.floor(yp / 0.1 + 0.5))
        first = (jc - m // 2) % 64                         # first pixel row of the window (R8)
        bands = [(first, m), ((first - 3) % 64, min(64, m + 7))] if f > 1 else [(first, 64), (17, 64)]
        for row0, n_rows in bands:
            got, got_pat = O.prism_probe_rows(p, _band(s, row0, n_rows), row0, b, xp, yp, want_pattern=True)
            assert np.array_equal(got, want) and np.array_equal(got_pat, want_pat), (xp, yp, row0, n_rows)
    # the probe at the origin with f = 4: window rows [-8, 8) -> band starts at pixel row 56 and wraps through 0
    if f == 4:
        got = O.prism_probe_rows(p, _band(s, 56, 16), 56, b, 0.0, 0.0)
        assert np.array_equal(got, O.prism_probe(p, s, b, 0.0, 0.0))
        # a band that misses one window row is refused, not read out of bounds
        with pytest.raises(ValueError):
            O.prism_probe_rows(p, _band(s, 57, 16), 57, b, 0.0, 0.0)
        with pytest.raises(ValueError):
            O.prism_probe_rows(p, _band(s, 56, 15), 56, b, 0.0, 0.0)


def test_prism_probe_rows_placement_with_a_point_band():
    """Independent of the whole-grid routine: a single non-zero pixel at band row r stands for pixel row
    (row0 + r) mod ny; it contributes iff that pixel row lies in the probe's window, with the Parseval weight."""
    n, f = 64, 4
    m = n // f
    p = params(n, f=f, alpha=30e-3)
    b = O.beams(p)
    nb = len(b)
    xp, yp = 2.0, 0.3                                     # centre pixel (20, 3) -> window rows [-5, 11)
    row0, n_rows = 50, 30                                 # band = pixel rows 50 .. 63, 0 .. 15
    coef = np.exp(-2j * np.pi * (b[:, 0] * xp + b[:, 1] * yp) / 6.4)
    inside = abs(coef.sum()) ** 2 / (nb * m * m)

    def total(r, i0):
        s = np.zeros((nb, n_rows, n), complex)
        s[:, r, i0] = 1.0
        return O.prism_probe_rows(p, s, row0, b, xp, yp, want_pattern=True)[1].sum()

    assert abs(total(9, 20) - inside) < 1e-12             # pixel row 59 = -5: first row of the window
    assert abs(total(24, 27) - inside) < 1e-12            # pixel row 10: last row, last column [12, 28)
    assert total(8, 20) == 0.0 and total(25, 20) == 0.0   # pixel rows 58 and 11: just outside
    assert total(14, 28) == 0.0 and total(14, 11) == 0.0  # inside in y (pixel row 0), outside in x
