"""Pins of the oracle's general aberration terms (reading R5b): chi gains
(2 pi / lambda) c (lambda q)^(n+1) / (n+1) cos(m (phi - angle)) per listed term.  PAPER.md:86 names defocus and
spherical aberration; the two rotationally symmetric terms (1,0) and (3,0) must reduce to them, and the azimuthal
part is fixed by symmetry: none of these checks retypes the formula."""
import numpy as np

import oracle as O
from helpers import freq


def params(n=64, **kw):
    base = dict(lx=0.1 * n, ly=0.1 * n, lz=8.0, nx=n, ny=n, n_slices=4, dz=2.0, voltage=200e3,
                alpha=30e-3, f=1, det_step=1e-3, det_max=60e-3)
    base.update(kw)
    return O.Params(**base)


def spectrum(p):
    """Probe spectrum at position 0 (aperture pixels carry exp(-i chi) up to one real scale)."""
    return np.fft.fft2(O.probe(p, 0.0, 0.0))


def test_terms_1_0_and_3_0_are_defocus_and_spherical_aberration():
    a = O.probe(params(defocus=85.0, cs=2.0e6), 1.3, 2.1)
    b = O.probe(params(aberrations=((1, 0, 85.0, 0.0), (3, 0, 2.0e6, 0.7))), 1.3, 2.1)      # angle is irrelevant at m = 0
    assert np.max(np.abs(a - b)) < 1e-12
    # and they add to the fixed terms
    c = O.probe(params(defocus=40.0, aberrations=((1, 0, 45.0, 0.0), (3, 0, 2.0e6, 0.0))), 1.3, 2.1)
    assert np.max(np.abs(a - c)) < 1e-12


def test_twofold_astigmatism_is_plus_and_minus_defocus_on_its_axes():
    # cos(2 (phi - angle)): +1 along the axis `angle`, -1 at right angles, 0 on the diagonals between them
    c = 60.0
    plus, minus, none = spectrum(params(defocus=c)), spectrum(params(defocus=-c)), spectrum(params())
    for angle, ax_plus in [(0.0, "x"), (np.pi / 2, "y")]:
        s = spectrum(params(aberrations=((1, 2, c, angle),)))
        on_x, on_y = (slice(0, 1), slice(1, 9)), (slice(1, 9), slice(0, 1))           # kx = 1..8 at ky = 0, and vice versa
        a, b = (on_x, on_y) if ax_plus == "x" else (on_y, on_x)
        assert np.max(np.abs(s[a] - plus[a])) < 1e-10
        assert np.max(np.abs(s[b] - minus[b])) < 1e-10
        k = np.arange(1, 6)
        assert np.max(np.abs(s[k, k] - none[k, k])) < 1e-10                             # 45 degrees: no phase at all
    # a rotation of the axis by 45 degrees moves the +defocus line onto the diagonal
    s = spectrum(params(aberrations=((1, 2, c, np.pi / 4),)))
    k = np.arange(1, 6)
    assert np.max(np.abs(s[k, k] - plus[k, k])) < 1e-10
    assert np.max(np.abs(s[k, -k] - minus[k, -k])) < 1e-10


def test_rotating_the_aberration_axis_by_90_degrees_rotates_the_probe():
    # on a square grid a quarter turn is exact: psi'(x, y) = psi(y, -x)
    for n_, m_ in [(2, 1), (2, 3), (3, 2), (4, 5)]:
        c = {2: 4.0e3, 3: 1.5e6, 4: 2.0e8}[n_]
        a = O.probe(params(aberrations=((n_, m_, c, 0.3),)), 0.0, 0.0)
        b = O.probe(params(aberrations=((n_, m_, c, 0.3 + np.pi / 2),)), 0.0, 0.0)
        # b[y][x] = a[-x][y]  (array indices modulo n)
        rot = np.roll(a[::-1, :], 1, axis=0).T
        assert np.max(np.abs(b - rot)) < 1e-10, (n_, m_)
        assert np.max(np.abs(b - a)) > 1e-3                                             # and it is not a no-op


def test_m_fold_symmetry_of_the_probe_intensity():
    # (with defocus beside it: a pure m = 2 term alone gives a four-fold intensity, because a quarter turn only flips
    # the sign of chi)
    def inten(m_, n_=3):
        return np.abs(O.probe(params(defocus=60.0, aberrations=((n_, m_, 3.0e6, 0.2),)), 0.0, 0.0)) ** 2
    quarter = lambda a: np.roll(a[::-1, :], 1, axis=0).T                               # noqa: E731
    half = lambda a: np.roll(np.roll(a[::-1, ::-1], 1, axis=0), 1, axis=1)             # noqa: E731
    i4, i2 = inten(4), inten(2)
    assert np.max(np.abs(i4 - quarter(i4))) < 1e-12 * i4.max() + 1e-15                # m = 4: invariant under 90 degrees
    assert np.max(np.abs(i2 - half(i2))) < 1e-12 * i2.max() + 1e-15                   # m = 2: invariant under 180 ...
    assert np.max(np.abs(i2 - quarter(i2))) > 1e-3 * i2.max()                          # ... but not under 90


def test_radial_power_and_the_one_over_n_plus_one():
    # along one axis the phase of term (n, 0) grows as q^(n+1); against the pinned C3 term it fixes the 1/(n+1):
    # (2 pi / lambda) c5 (lambda q)^6 / 6  ==  (pi / 2) c3 lambda^3 q^4  at  c5 = 1.5 c3 / (lambda q)^2
    p0 = params()
    lam, _ = O.constants(p0.voltage)
    k = 6
    q = k / p0.lx
    c3 = 1.0e6
    a = spectrum(params(cs=c3))[0, k]
    b = spectrum(params(aberrations=((5, 0, 1.5 * c3 / (lam * q) ** 2, 0.0),)))[0, k]
    assert abs(a - b) < 1e-10 * abs(a)
    # q^(n+1): the phase at 2 q is 2^6 times the phase at q (kept below pi so that no branch is crossed)
    c5 = 4.0e8
    s = spectrum(params(aberrations=((5, 0, c5, 0.0),)))
    ph1, ph2 = -np.angle(s[0, 3] / np.abs(s[0, 3])), -np.angle(s[0, 6] / np.abs(s[0, 6]))
    assert 0.0 < ph1 < ph2 < np.pi
    assert abs(ph2 / ph1 - 64.0) < 1e-6


def test_prism_and_multislice_agree_at_f1_with_general_aberrations():
    # the same chi enters the multislice probe and the PRISM coefficients: f = 1 makes the two paths identical
    rng = np.random.default_rng(5)
    p = params(n=32, alpha=25e-3, lx=3.2, ly=3.2, aberrations=((1, 2, 30.0, 0.4), (2, 1, 2.0e3, 1.1), (2, 3, 1.0e3, 0.2)))
    v = rng.random((p.n_slices, 32, 32)) * 40.0
    b = O.beams(p)
    s = O.smatrix(p, v, b)
    xy = np.array([[0.7, 1.9]])
    assert np.max(np.abs(O.prism_probes(p, s, b, xy) - O.multislice_probes(p, v, xy))) < 1e-12
    k = freq(32)
    assert k[0] == 0
