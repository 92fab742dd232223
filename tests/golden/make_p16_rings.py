"""Writes tests/golden/p16_s<S>_rings.txt: PRISM rings of config 5 (BASELINE.json configs[4]: 2048^2, f = 16, 1201
beams, 512 x 512 probes) on its first S slices, end to end through the ORACLE ONLY -- atoms -> potential -> all 1201
S-matrix layers -> stage 2 -- for sampled probes of two probe rows (SURVEY.md 8(d) plan (ii)).

Calls only `oracle/` and the seeded input generator `workloads.py`; nothing of the CUDA path.  The fp64 S-matrix of
config 5 is 80 GB, so only the 128 pixel rows each of the two probe rows touches are kept of every layer
(O.prism_probe_rows: the loop of the whole-grid routine on that storage).  Cost: about 0.23 s per beam-slice on 8
cores, i.e. S = 10 in ~50 min, S = 40 in ~3 h.

    python tests/golden/make_p16_rings.py [--slices 10] [--probes 8] [--chunk 8]
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle as O                                               # noqa: E402
from paper_1706_08563_b200 import workloads as W                 # noqa: E402

PROBE_ROWS = (0, 259)          # probe row 0: windows wrap the cell edge in y; 259: mid-grid, off the lattice symmetry


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--slices", type=int, default=10)
    ap.add_argument("--probes", type=int, default=8)
    ap.add_argument("--chunk", type=int, default=8, help="layers per oracle call (one per thread)")
    args = ap.parse_args()

    w = W.p16_first_slices(args.slices)
    p = O.Params(w.cell[0], w.cell[1], w.cell[2], w.nx, w.ny, w.n_slices, w.dz, w.voltage, w.alpha, w.defocus, w.cs,
                 w.f, w.det_step, w.det_max, tuple(w.aberrations))
    lut_z, r_cut, lut_v = w.lut()
    v = O.potential(p, w.atoms_for_phonon(0), w.z, lut_z, r_cut, lut_v)
    beams = O.beams(p)
    my, py = w.ny // w.f, w.cell[1] / w.ny
    xy = w.probe_xy().reshape(w.probes_y, w.probes_x, 2)
    row0 = {iy: (int(np.floor(xy[iy, 0, 1] / py + 0.5)) - my // 2) % w.ny for iy in PROBE_ROWS}
    bands = {iy: np.empty((len(beams), my, w.nx), dtype=np.complex128) for iy in PROBE_ROWS}
    t0 = time.time()
    for b0 in range(0, len(beams), args.chunk):
        layers = O.smatrix(p, v, beams[b0:b0 + args.chunk])
        for iy in PROBE_ROWS:
            bands[iy][b0:b0 + len(layers)] = layers[:, (row0[iy] + np.arange(my)) % w.ny, :]
        print(f"layers {b0 + len(layers)} / {len(beams)}  {time.time() - t0:.0f} s", flush=True)
    cols = np.unique(np.linspace(0, w.probes_x - 1, args.probes).astype(int))
    path = os.path.join(HERE, f"p16_s{args.slices}_rings.txt")
    with open(path + ".tmp", "w") as fh:
        fh.write(f"# PRISM rings of config 5 (P16) on its first {args.slices} slices, frozen-phonon configuration 0, from the fp64 oracle alone.\n"
                 f"# Written by: python tests/golden/make_p16_rings.py --slices {args.slices} --probes {args.probes}\n"
                 "# Source: the algorithm of PAPER.md:44 (Eq. 1), :80 (Eq. 2), :86, :120, :128 as restated in oracle/prism_oracle.c\n"
                 "# (O1-O11 of SURVEY.md 8(c)); inputs: workloads.p16_first_slices (seeded).\n"
                 f"# columns: probe_row probe_col  then {O.num_bins(p)} ring values (1 mrad rings from 0)\n")
        for iy in PROBE_ROWS:
            for ix in cols:
                rings = O.prism_probe_rows(p, bands[iy], row0[iy], beams, *xy[iy, ix])
                fh.write(f"{iy} {ix} " + " ".join(f"{r:.12e}" for r in rings) + "\n")
    os.replace(path + ".tmp", path)
    print("wrote", path, f"{time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
