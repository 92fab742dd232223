"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module holds NO arithmetic of the method (no FFT, no potential
summation, no wavelength): it only draws atoms, fills the caller-supplied
per-Z radial table and lists the run parameters.  It is the one module both the
CUDA tests / bench and the oracle tests read their inputs from; it imports
neither the CUDA binding nor ``oracle``.

The inputs stand in for the paper's workloads (amorphous carbon blocks,
PAPER.md:158,182,200; the layered oxide of PAPER.md:212; the nanoparticle of
PAPER.md:222), whose atomic models are not available; shapes, sizes and
structure follow BASELINE.json ``configs`` and SURVEY.md section 8(d).  The
recipe is restated in DESIGN.md ("Input recipe").

Random numbers: ``numpy.random.Generator(PCG64(seed))``;
structure seed = 170608563 + 1000*config_index + 999,
frozen-phonon jitter seed = 170608563 + 1000*config_index + phonon_index.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

SEED_BASE = 170608563
MRAD = 1e-3

# BASELINE.json config 1: "projected potential per atom = 2D Gaussian amplitude
# 2*Z V*A^2, sigma=0.3 A, cut at 1 A" (reading R15: peak value 2Z, hard cut).
LUT_SAMPLES = 1025
LUT_RCUT = 1.0
LUT_SIGMA = 0.3

CARBON_DENSITY = 0.100277  # atoms / A^3  (2 g/cm^3, Z=6)


@dataclass
class Workload:
    """One simulation input: the paper's parameters, atoms, tables, probe grid."""
    name: str
    cell: tuple            # (lx, ly, lz) Angstrom
    nx: int
    ny: int
    n_slices: int
    dz: float              # slice thickness, Angstrom
    voltage: float         # volt
    alpha: float           # probe semi-angle, rad
    defocus: float = 0.0   # C1, Angstrom
    cs: float = 0.0        # C3, Angstrom
    aberrations: tuple = ()  # further terms (n, m, c [Angstrom], angle [rad]) of the aberration function
    f: int = 1             # PRISM interpolation factor
    probes_x: int = 1
    probes_y: int = 1
    probe_origin: tuple = (0.0, 0.0)
    probe_step: tuple = (0.0, 0.0)
    det_step: float = 1.0 * MRAD
    det_max: float = 100.0 * MRAD
    batch: int = 0
    potential_on_host: int = 0
    smatrix_on_host: int = 0
    n_phonons: int = 1
    jitter: float = 0.0
    config_index: int = 0
    atoms: np.ndarray = field(default=None, repr=False)   # [n][3] fp64, un-jittered
    z: np.ndarray = field(default=None, repr=False)       # [n] int32

    # -- derived inputs -------------------------------------------------------
    def lut(self):
        """(lut_z int32[n_luts], r_cut, lut_v fp64[n_luts][LUT_SAMPLES])."""
        zs = np.unique(self.z).astype(np.int32)
        r = np.arange(LUT_SAMPLES, dtype=np.float64) * (LUT_RCUT / (LUT_SAMPLES - 1))
        v = 2.0 * zs[:, None].astype(np.float64) * np.exp(-(r[None, :] ** 2) / (2.0 * LUT_SIGMA ** 2))
        return zs, LUT_RCUT, v

    def atoms_for_phonon(self, phonon: int = 0) -> np.ndarray:
        """Atom positions of one frozen-phonon configuration (reading R20):
        iid Gaussian displacement per axis, wrap x,y into the cell, clamp z."""
        xyz = self.atoms.copy()
        if self.jitter > 0.0:
            rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1000 * self.config_index + phonon))
            xyz += rng.normal(0.0, self.jitter, size=xyz.shape)
        lx, ly, _ = self.cell
        xyz[:, 0] = np.mod(xyz[:, 0], lx)
        xyz[:, 1] = np.mod(xyz[:, 1], ly)
        zmax = self.n_slices * self.dz
        xyz[:, 2] = np.clip(xyz[:, 2], 0.0, np.nextafter(zmax, 0.0))
        return xyz

    def probe_xy(self) -> np.ndarray:
        """[probes_y*probes_x][2] positions, x fastest (reading R10)."""
        xs = self.probe_origin[0] + np.arange(self.probes_x) * self.probe_step[0]
        ys = self.probe_origin[1] + np.arange(self.probes_y) * self.probe_step[1]
        return np.stack(np.meshgrid(xs, ys, indexing="xy"), axis=-1).reshape(-1, 2).astype(np.float64)

    @property
    def n_probes(self) -> int:
        return self.probes_x * self.probes_y

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


def _structure_rng(config_index: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + 1000 * config_index + 999))


def amorphous(rng, lx, ly, z_lo, z_hi, density, zval):
    n = int(round(density * lx * ly * (z_hi - z_lo)))
    xyz = rng.random((n, 3)) * np.array([lx, ly, z_hi - z_lo]) + np.array([0.0, 0.0, z_lo])
    return xyz, np.full(n, zval, dtype=np.int32)


def lattice(a, reps, basis, origin):
    """All basis sites of an a-cubic lattice with reps=(nx,ny,nz) cells."""
    ix, iy, iz = np.meshgrid(*[np.arange(r) for r in reps], indexing="ij")
    cells = np.stack([ix, iy, iz], axis=-1).reshape(-1, 1, 3).astype(np.float64)
    sites = (cells + np.asarray(basis, dtype=np.float64)[None, :, :]) * a
    return sites.reshape(-1, 3) + np.asarray(origin, dtype=np.float64)


# ---------------------------------------------------------------------------
def pr1() -> Workload:
    """Config 1 (PR1): 6.4x6.4x8 A, 64^2, 4 slices, 40 atoms Z in {6,8}, 200 kV."""
    rng = _structure_rng(1)
    xyz = rng.random((40, 3)) * np.array([6.4, 6.4, 8.0])
    z = rng.choice(np.array([6, 8], dtype=np.int32), size=40)
    return Workload("PR1", (6.4, 6.4, 8.0), 64, 64, 4, 2.0, 200e3, 20 * MRAD, f=1,
                    probes_x=8, probes_y=8, probe_step=(0.8, 0.8), det_max=60 * MRAD,
                    config_index=1, atoms=xyz, z=z.astype(np.int32))


def ms2() -> Workload:
    """Config 2 (MS2): 25.6^2 x 100 A amorphous carbon, 256^2, 50 slices, 300 kV."""
    rng = _structure_rng(2)
    xyz, z = amorphous(rng, 25.6, 25.6, 0.0, 100.0, CARBON_DENSITY, 6)
    return Workload("MS2", (25.6, 25.6, 100.0), 256, 256, 50, 2.0, 300e3, 20 * MRAD,
                    probes_x=32, probes_y=32, probe_step=(0.8, 0.8), batch=64,
                    config_index=2, atoms=xyz, z=z)


def p4() -> Workload:
    """Config 3 (P4): 51.2^2 x 200 A cubic perovskite-like lattice, 512^2, f=4."""
    a = 3.9
    reps = (13, 13, 51)
    origin = ((51.2 - reps[0] * a) / 2, (51.2 - reps[1] * a) / 2, (200.0 - reps[2] * a) / 2)
    basis = [(0, 0, 0), (0.5, 0.5, 0.5), (0.5, 0.5, 0), (0.5, 0, 0.5), (0, 0.5, 0.5)]
    zb = np.array([38, 22, 8, 8, 8], dtype=np.int32)
    xyz = lattice(a, reps, basis, origin)
    z = np.tile(zb, reps[0] * reps[1] * reps[2])
    return Workload("P4", (51.2, 51.2, 200.0), 512, 512, 100, 2.0, 300e3, 20 * MRAD, f=4,
                    probes_x=128, probes_y=128, probe_step=(0.4, 0.4), jitter=0.08,
                    config_index=3, atoms=xyz, z=z)


def p8() -> Workload:
    """Config 4 (P8): 102.4 A cube, fcc Z=79 particle on amorphous carbon, 1024^2, f=8."""
    rng = _structure_rng(4)
    a = 4.08
    centre = np.array([51.2, 51.2, 57.0])
    radius = 42.0
    n_cells = int(np.ceil(2 * radius / a)) + 2
    basis = [(0, 0, 0), (0.5, 0.5, 0), (0.5, 0, 0.5), (0, 0.5, 0.5)]
    origin = centre - 0.5 * n_cells * a
    au = lattice(a, (n_cells,) * 3, basis, origin)
    rel = au - centre
    keep = np.sum(rel ** 2, axis=1) <= radius ** 2
    normals = rng.normal(size=(12, 3))
    normals /= np.linalg.norm(normals, axis=1, keepdims=True)
    dist = rng.uniform(0.75, 1.0, size=12) * radius
    keep &= np.all(rel @ normals.T <= dist[None, :], axis=1)
    au = au[keep]
    carbon, zc = amorphous(rng, 102.4, 102.4, 0.0, 14.0, CARBON_DENSITY, 6)
    xyz = np.concatenate([au, carbon])
    z = np.concatenate([np.full(len(au), 79, dtype=np.int32), zc])
    return Workload("P8", (102.4, 102.4, 102.4), 1024, 1024, 50, 2.0, 200e3, 25 * MRAD,
                    defocus=50.0, cs=0.0, f=8, probes_x=256, probes_y=256,
                    probe_step=(0.4, 0.4), jitter=0.08, n_phonons=4,
                    config_index=4, atoms=xyz, z=z)


def p16() -> Workload:
    """Config 5 (P16): 204.8^2 x 800 A multi-element slab, 2048^2, f=16, streamed slices."""
    rng = _structure_rng(5)
    a = 5.65
    reps = (36, 36, 141)
    origin = ((204.8 - reps[0] * a) / 2, (204.8 - reps[1] * a) / 2, (800.0 - reps[2] * a) / 2)
    fcc = np.array([(0, 0, 0), (0.5, 0.5, 0), (0.5, 0, 0.5), (0, 0.5, 0.5)], dtype=np.float64)
    basis = np.concatenate([fcc, fcc + 0.25])
    xyz = lattice(a, reps, basis, origin)
    z = rng.choice(np.array([14, 31, 33, 79], dtype=np.int32), size=len(xyz),
                   p=[0.3, 0.3, 0.3, 0.1]).astype(np.int32)
    return Workload("P16", (204.8, 204.8, 800.0), 2048, 2048, 400, 2.0, 300e3, 30 * MRAD, f=16,
                    probes_x=512, probes_y=512, probe_step=(0.4, 0.4), jitter=0.1,
                    n_phonons=8, potential_on_host=1, config_index=5, atoms=xyz, z=z)


def p16_multislice() -> Workload:
    """Config 5's comparison run: the same grid/slices as plain multislice on 64x64 probes."""
    w = p16()
    return w.with_(name="P16-MS", probes_x=64, probes_y=64, probe_step=(3.2, 3.2))


def p16_first_slices(n_slices: int) -> Workload:
    """Config 5 cut to its first `n_slices` slices (for oracle runs that cannot afford all 400): atoms above the
    truncated stack are dropped (not clamped into the last slice), the cell height follows; grid, beams, probe
    lattice and the streamed potential are config 5's."""
    w = p16()
    if n_slices >= w.n_slices:
        return w
    keep = w.atoms[:, 2] < n_slices * w.dz - 1.0
    return w.with_(n_slices=n_slices, atoms=w.atoms[keep], z=w.z[keep],
                   cell=(w.cell[0], w.cell[1], n_slices * w.dz))


CONFIGS = {"PR1": pr1, "MS2": ms2, "P4": p4, "P8": p8, "P16": p16, "P16-MS": p16_multislice}


def get(name: str) -> Workload:
    return CONFIGS[name]()


def scaled_test_case(n: int, n_slices: int, f: int, probes: int, voltage: float = 200e3,
                     alpha_mrad: float = 20.0, seed_index: int = 7, det_max_mrad: float = 100.0,
                     defocus: float = 0.0, cs: float = 0.0, z_choices=(6, 14, 31, 79),
                     density: float = 0.05, probe_offset=(0.0, 0.0)) -> Workload:
    """Mid-size parity case: an n x n grid at 0.1 A pixels filled with a seeded
    random multi-element gas (same distribution family as the configs), sized
    so the oracle finishes in seconds."""
    rng = _structure_rng(100 + seed_index)
    length = 0.1 * n
    lz = 2.0 * n_slices
    n_atoms = max(1, int(round(density * length * length * lz)))
    xyz = rng.random((n_atoms, 3)) * np.array([length, length, lz])
    z = rng.choice(np.array(z_choices, dtype=np.int32), size=n_atoms).astype(np.int32)
    step = length / probes
    return Workload(f"T{n}", (length, length, lz), n, n, n_slices, 2.0, voltage,
                    alpha_mrad * MRAD, defocus=defocus, cs=cs, f=f, probes_x=probes,
                    probes_y=probes, probe_origin=probe_offset, probe_step=(step, step),
                    det_max=det_max_mrad * MRAD, config_index=100 + seed_index, atoms=xyz, z=z)
