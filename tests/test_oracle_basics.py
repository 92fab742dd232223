"""Pins for the oracle's constants, transforms, potential, propagator, probe and
detector (O1-O7 of DESIGN.md).  None of these re-types the oracle's formula:
each compares with an independent derivation, a closed form, a library routine
or brute force.  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle as O
from helpers import freq, oracle_params, rel_l2
from paper_1706_08563_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def small_params(**kw):
    base = dict(lx=6.4, ly=6.4, lz=8.0, nx=64, ny=64, n_slices=4, dz=2.0, voltage=200e3,
                alpha=20e-3, f=1, det_step=1e-3, det_max=60e-3)
    base.update(kw)
    return O.Params(**base)


# ----------------------------------------------------------------------------- O1
def test_constants_match_printed_values():
    for v, lam, sig in _rows("constants.txt"):
        got_lam, got_sig = O.constants(float(v))
        assert abs(got_lam - float(lam)) < 0.6e-7       # printed to 7 decimals
        assert abs(got_sig - float(sig)) / float(sig) < 1e-6


@pytest.mark.parametrize("volt", [1.0, 80e3, 200e3, 300e3, 1e6])
def test_constants_from_relativistic_momentum(volt):
    # de Broglie lambda = h/p with E_total^2 = (pc)^2 + (mc^2)^2 ; sigma = 2 pi gamma m e lambda / h^2
    h, c, e, m = 6.62607015e-34, 299792458.0, 1.602176634e-19, 9.1093837015e-31
    etot = e * volt + m * c * c
    pmom = math.sqrt(etot ** 2 - (m * c * c) ** 2) / c
    lam_m = h / pmom
    gamma = etot / (m * c * c)
    sigma_si = 2 * math.pi * gamma * m * e * lam_m / h ** 2          # rad / (V m)
    lam, sig = O.constants(volt)
    tol = 1e-12 if volt > 1e3 else 1e-9     # E^2 - (mc^2)^2 cancels at 1 V in THIS form
    assert abs(lam - lam_m * 1e10) / lam < tol
    assert abs(sig - sigma_si * 1e-10) / sig < tol


def test_constants_nonrelativistic_limit():
    lam, _ = O.constants(1.0)       # 1 V: lambda = h / sqrt(2 m e V) = 12.2643 A
    assert abs(lam - 12.2643) < 2e-4


# ----------------------------------------------------------------------------- FFT
@pytest.mark.parametrize("n", [2, 4, 8, 16, 32, 64])
@pytest.mark.parametrize("sign", [-1, +1])
def test_fft_matches_naive_dft_and_library(n, sign):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    lib = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
    assert rel_l2(O.dft_naive(x, sign), lib) < 1e-12
    assert rel_l2(O.fft(x, sign), lib) < 1e-12
    assert rel_l2(O.fft(x, sign), O.dft_naive(x, sign)) < 1e-12


def test_fft_closed_forms_fix_the_sign():
    n, n0, k0 = 32, 5, 7
    delta = np.zeros(n, complex)
    delta[n0] = 1.0
    k = np.arange(n)
    assert np.allclose(O.fft(delta, -1), np.exp(-2j * np.pi * k * n0 / n), atol=1e-13)
    assert np.allclose(O.fft(delta, +1), np.exp(+2j * np.pi * k * n0 / n), atol=1e-13)
    wave = np.exp(2j * np.pi * k0 * k / n)
    expect = np.zeros(n, complex)
    expect[k0] = n
    assert np.allclose(O.fft(wave, -1), expect, atol=1e-12)
    assert np.allclose(O.dft_naive(wave, -1), expect, atol=1e-12)


def test_fft_parseval_and_roundtrip():
    rng = np.random.default_rng(3)
    x = rng.normal(size=256) + 1j * rng.normal(size=256)
    fx = O.fft(x, -1)
    assert abs(np.sum(abs(fx) ** 2) / 256 - np.sum(abs(x) ** 2)) < 1e-10
    assert rel_l2(O.fft(fx, +1) / 256, x) < 1e-13


def test_fft2_axes_scale_and_library():
    rng = np.random.default_rng(4)
    a = rng.normal(size=(8, 32)) + 1j * rng.normal(size=(8, 32))      # non-square: catches swapped axes
    assert rel_l2(O.fft2(a, -1), np.fft.fft2(a)) < 1e-12
    assert rel_l2(O.fft2(a, +1), np.fft.ifft2(a)) < 1e-12              # inverse carries 1/(nx ny)
    assert rel_l2(O.dft2_naive(a, -1), np.fft.fft2(a)) < 1e-12
    assert rel_l2(O.dft2_naive(a, +1), np.fft.ifft2(a)) < 1e-12
    ky0, kx0 = 3, 11
    y, x = np.mgrid[0:8, 0:32]
    wave = np.exp(2j * np.pi * (kx0 * x / 32 + ky0 * y / 8))
    out = O.fft2(wave, -1)
    expect = np.zeros((8, 32), complex)
    expect[ky0, kx0] = 8 * 32
    assert np.allclose(out, expect, atol=1e-10)


# ----------------------------------------------------------------------------- O2
def _lut(zs, kind="gauss", n=1025, r_cut=1.0):
    r = np.arange(n) * r_cut / (n - 1)
    if kind == "gauss":
        v = np.stack([2.0 * z * np.exp(-r ** 2 / 0.18) for z in zs])
    else:                              # linear table: the interpolant is exact
        v = np.stack([z * (1.0 - r / r_cut) for z in zs])
    return np.array(zs, np.int32), r_cut, v


def test_potential_single_atom_on_a_pixel():
    p = small_params()
    lz, rc, lv = _lut([6])
    v = O.potential(p, [[3.2, 1.6, 2.5]], [6], lz, rc, lv)
    assert v.shape == (4, 64, 64)
    assert np.count_nonzero(v[0]) == 0 and np.count_nonzero(v[2:]) == 0   # z=2.5 -> slice 1
    s = v[1]
    assert s[16, 32] == 12.0                                              # v(0) = 2Z exactly
    jj, ii = np.mgrid[0:64, 0:64]
    d2 = (ii - 32) ** 2 + (jj - 16) ** 2                                  # integer pixel offsets
    strictly_inside, on_cut = d2 < 100, d2 == 100                         # the 12 lattice points with d2 == 100
    assert np.count_nonzero(strictly_inside) == 305 and np.count_nonzero(on_cut) == 12
    assert np.all(s[strictly_inside] > 0) and np.all(s[d2 > 100] == 0)    # ties on the cut are fp-decided
    expect = 12.0 * np.exp(-d2 * 0.01 / 0.18)
    ok = strictly_inside
    assert np.max(np.abs(s[ok] - expect[ok])) / 12.0 < 2e-6               # table interpolation error only
    assert np.all((s[on_cut] == 0) | (np.abs(s[on_cut] - expect[on_cut]) < 1e-4))


def test_potential_subpixel_position_and_linear_table_exact():
    p = small_params()
    lz, rc, lv = _lut([10], kind="linear")
    ax, ay = 3.237, 2.911
    v = O.potential(p, [[ax, ay, 0.1]], [10], lz, rc, lv)[0]
    jj, ii = np.mgrid[0:64, 0:64]
    r = np.hypot(ii * 0.1 - ax, jj * 0.1 - ay)
    expect = np.where(r <= 1.0, 10.0 * (1.0 - r), 0.0)
    assert np.max(np.abs(v - expect)) < 1e-12


def test_potential_slice_assignment_and_clamp():
    p = small_params()
    lz, rc, lv = _lut([6])
    for zc, want in [(0.0, 0), (1.999999, 0), (2.0, 1), (5.9, 2), (7.99, 3), (8.0, 3), (11.0, 3), (-0.3, 0)]:
        v = O.potential(p, [[1.0, 1.0, zc]], [6], lz, rc, lv)
        hit = [s for s in range(4) if np.count_nonzero(v[s])]
        assert hit == [want], (zc, hit)


def test_potential_periodic_wrap_and_translation():
    p = small_params()
    lz, rc, lv = _lut([8])
    centre = O.potential(p, [[3.23, 3.21, 1.0]], [8], lz, rc, lv)[0]
    moved = O.potential(p, [[(3.23 + 3.5) % 6.4, (3.21 - 3.3) % 6.4, 1.0]], [8], lz, rc, lv)[0]
    assert np.max(np.abs(np.roll(centre, (-33, 35), axis=(0, 1)) - moved)) < 1e-12
    edge = O.potential(p, [[0.02, 6.39, 1.0]], [8], lz, rc, lv)[0]
    assert edge[0, 63] > 0 and edge[63, 0] > 0 and edge[0, 0] > 0          # wrapped on both axes
    assert abs(edge.sum() - centre.sum()) / centre.sum() < 2e-3


def test_potential_superposition_and_integral():
    w = W.pr1()
    p = oracle_params(w)
    lz, rc, lv = w.lut()
    xyz = w.atoms_for_phonon(0)
    v = O.potential(p, xyz, w.z, lz, rc, lv)
    parts = sum(O.potential(p, xyz[i:i + 1], w.z[i:i + 1], lz, rc, lv) for i in range(len(w.z)))
    assert np.max(np.abs(v - parts)) < 1e-10
    # integral of 2Z exp(-r^2/0.18) over the disc r <= 1: 2Z * 2 pi * 0.09 * (1 - exp(-1/0.18))
    closed = sum(2.0 * z * 2 * np.pi * 0.09 * (1 - np.exp(-1 / 0.18)) for z in w.z)
    assert abs(v.sum() * 0.01 - closed) / closed < 5e-5


def test_potential_errors():
    p = small_params()
    lz, rc, lv = _lut([6])
    with pytest.raises(ValueError):
        O.potential(p, [[1, 1, 1]], [7], lz, rc, lv)                       # no table for Z=7
    with pytest.raises(ValueError):
        O.potential(small_params(lx=1.5), [[1, 1, 1]], [6], lz, rc, lv)    # 2 r_cut >= cell


# ----------------------------------------------------------------------------- O3, O4, O5
def test_transmission_is_a_pure_phase():
    sig = 0.5
    t = O.transmission(np.array([[0.0, np.pi, 2 * np.pi, 3.0]]), sig)
    assert np.allclose(t, [[1.0, 1j, -1.0, np.exp(1.5j)]], atol=1e-15)
    assert np.allclose(abs(t), 1.0, atol=1e-15)


def test_propagator_closed_form_mask_and_axes():
    p = small_params(lx=6.4, ly=12.8, nx=64, ny=128)      # non-square cell, equal pixels
    lam, _ = O.constants(p.voltage)
    prop = O.propagator(p)
    assert prop[0, 0] == 1.0
    kx, ky = freq(64), freq(128)
    q2 = (kx[None, :] / 6.4) ** 2 + (ky[:, None] / 12.8) ** 2
    qcut = (2.0 / 3.0) * min(64 / (2 * 6.4), 128 / (2 * 12.8))
    mask = q2 < qcut ** 2
    assert np.array_equal(prop != 0, mask)
    assert np.allclose(prop[mask], np.exp(-1j * np.pi * lam * q2[mask] * 2.0), atol=1e-12)
    # one specific off-axis slot, by hand: slot (my=125, mx=3) is k=(3,-3)
    q2h = (3 / 6.4) ** 2 + (-3 / 12.8) ** 2
    assert abs(prop[125, 3] - np.exp(-1j * np.pi * lam * q2h * 2.0)) < 1e-13


@pytest.mark.parametrize("n", [64, 256, 512])
def test_propagator_band_limit_count_is_the_integer_test(n):
    p = small_params(lx=0.1 * n, ly=0.1 * n, nx=n, ny=n)
    k = freq(n).astype(np.int64)
    want = np.count_nonzero(9 * (k[None, :] ** 2 + k[:, None] ** 2) < n * n)
    assert np.count_nonzero(O.propagator(p)) == want


def test_propagators_compose():
    p = small_params()
    a, b, ab = O.propagator(p, 1.5), O.propagator(p, 2.5), O.propagator(p, 4.0)
    assert np.max(np.abs(a * b - ab)) < 1e-12


def test_slice_step_plane_wave_closed_form_and_band_limit():
    p = small_params()
    lam, _ = O.constants(p.voltage)
    prop = O.propagator(p)
    t = np.ones((64, 64), complex)
    y, x = np.mgrid[0:64, 0:64]
    for kx0, ky0 in [(3, -5), (0, 0), (-20, 2), (25, 0), (16, 16)]:
        wave = np.exp(2j * np.pi * (kx0 * x + ky0 * y) / 64)
        out = O.slice_step(wave, t, prop)
        q2 = (kx0 ** 2 + ky0 ** 2) / 6.4 ** 2
        if 9 * (kx0 ** 2 + ky0 ** 2) < 64 * 64:
            assert np.max(np.abs(out - wave * np.exp(-1j * np.pi * lam * q2 * 2.0))) < 1e-12
        else:
            assert np.max(np.abs(out)) < 1e-12


def test_slice_step_naive_equals_fft_and_norm_budget():
    rng = np.random.default_rng(5)
    p = small_params(nx=16, ny=16, lx=1.6, ly=1.6)
    psi = rng.normal(size=(16, 16)) + 1j * rng.normal(size=(16, 16))
    t = np.exp(1j * rng.normal(size=(16, 16)))
    prop = O.propagator(p)
    a, b = O.slice_step(psi, t, prop, use_naive=False), O.slice_step(psi, t, prop, use_naive=True)
    assert rel_l2(a, b) < 1e-12
    spec = np.fft.fft2(psi * t)
    in_band = np.sum(abs(spec[prop != 0]) ** 2) / 256
    assert abs(np.sum(abs(a) ** 2) - in_band) / in_band < 1e-12
    assert np.sum(abs(a) ** 2) <= np.sum(abs(psi) ** 2) * (1 + 1e-12)


def test_two_empty_slices_equal_one_thick_slice():
    rng = np.random.default_rng(6)
    p2 = small_params(n_slices=2, dz=2.0)
    p1 = small_params(n_slices=1, dz=4.0)
    psi = rng.normal(size=(64, 64)) + 1j * rng.normal(size=(64, 64))
    a = O.multislice_wave(p2, np.zeros((2, 64, 64)), psi)
    b = O.multislice_wave(p1, np.zeros((1, 64, 64)), psi)
    assert rel_l2(a, b) < 1e-12


def test_multislice_wave_order_of_slices():
    # transmission before propagation, slices in ascending order: compare with library FFTs
    rng = np.random.default_rng(7)
    p = small_params(nx=32, ny=32, lx=3.2, ly=3.2, n_slices=3)
    _, sig = O.constants(p.voltage)
    v = rng.random((3, 32, 32)) * 300.0
    psi = rng.normal(size=(32, 32)) + 1j * rng.normal(size=(32, 32))
    prop = O.propagator(p)
    ref = psi.copy()
    for s in range(3):
        ref = np.fft.ifft2(prop * np.fft.fft2(ref * np.exp(1j * sig * v[s])))
    assert rel_l2(O.multislice_wave(p, v, psi), ref) < 1e-12
    assert rel_l2(O.multislice_wave(p, v[::-1], psi), ref) > 1e-3          # order matters


# ----------------------------------------------------------------------------- O6
def test_probe_norm_peak_position_and_shift():
    p = small_params()
    n_a = O.num_aperture(p)
    assert n_a == 89
    psi = O.probe(p, 0.0, 0.0)
    assert abs(np.sum(abs(psi) ** 2) - 1.0) < 1e-12
    assert abs(psi[0, 0] - math.sqrt(n_a) / 64) < 1e-12                    # all aperture terms in phase
    assert np.max(np.abs(psi.imag)) < 1e-12                               # symmetric aperture, no aberration
    psi2 = O.probe(p, 1.3, 4.2)                                            # integer pixels (13, 42)
    assert np.unravel_index(np.argmax(abs(psi2)), psi2.shape) == (42, 13)
    assert rel_l2(psi2, np.roll(psi, (42, 13), axis=(0, 1))) < 1e-12


def test_probe_aperture_counts_match_golden():
    for name, n, kv, a_mrad, f, n_b, n_a in _rows("beam_counts.txt"):
        if int(n_a) < 0:
            continue
        p = small_params(lx=0.1 * int(n), ly=0.1 * int(n), nx=int(n), ny=int(n),
                         voltage=float(kv) * 1e3, alpha=float(a_mrad) * 1e-3)
        assert O.num_aperture(p) == int(n_a)


def test_probe_aberration_phase():
    p = small_params(defocus=80.0, cs=2.0e6)
    lam, _ = O.constants(p.voltage)
    spec = np.fft.fft2(O.probe(p, 0.0, 0.0))
    n_a = O.num_aperture(p)
    for ky0, kx0 in [(0, 4), (3, -2), (-5, 0)]:
        q2 = (kx0 ** 2 + ky0 ** 2) / 6.4 ** 2
        chi = np.pi * lam * q2 * 80.0 + 0.5 * np.pi * 2.0e6 * lam ** 3 * q2 ** 2
        want = np.exp(-1j * chi) * 64 / math.sqrt(n_a)
        assert abs(spec[ky0 % 64, kx0 % 64] - want) < 1e-10
    assert abs(spec[0, 20]) < 1e-10                                        # outside 20 mrad


# ----------------------------------------------------------------------------- O7
def test_detector_bins_by_hand():
    p = small_params(lx=6.4, ly=12.8, nx=64, ny=128, det_step=1e-3, det_max=60e-3)
    lam, _ = O.constants(p.voltage)
    assert O.num_bins(p) == 60
    for (my, mx), amp in [((0, 0), 1.0), ((3, 61), 2.0), ((120, 5), 0.5), ((64, 32), 7.0)]:
        img = np.zeros((128, 64))
        img[my, mx] = amp
        ky = my if my < 64 else my - 128
        kx = mx if mx < 32 else mx - 64
        angle = lam * math.hypot(kx / 6.4, ky / 12.8)
        b = int(angle / 1e-3)
        out = O.bin_intensity(p, img)
        if b < 60:
            assert out[b] == amp and np.count_nonzero(out) == 1
        else:
            assert np.count_nonzero(out) == 0


def test_detector_bins_prism_grid_uses_f_times_index():
    p = small_params(lx=12.8, ly=12.8, nx=128, ny=128, f=4)
    lam, _ = O.constants(p.voltage)
    img = np.zeros((32, 32))
    img[2, 31] = 1.0                                    # k = (-1, 2) on the window grid -> q = 4 k / L
    angle = lam * math.hypot(-4 / 12.8, 8 / 12.8)
    out = O.bin_intensity(p, img, fy=4, fx=4)
    assert out[int(angle / 1e-3)] == 1.0 and np.count_nonzero(out) == 1
