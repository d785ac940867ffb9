"""Writes tests/golden/c1_oracle_samples.txt: sampled values of the ORACLE's reconstruction of config C1.

    python tests/golden/make_golden.py

Calls only oracle/ (double precision CPU) and the seeded input generator synthgen/ -- never the CUDA path.  The
paper (arXiv 2209.08450) prints no worked numerical example of the method (no formulas, no tables of values other
than timings and SSIM on data that is not available), so there are no paper values to store; this fixture instead
freezes the oracle's own output on BASELINE.json's config C1 (128^2 x 8 slices, 180 angles, centre 64.0, Shepp-Logan
window; stages S1-S7 after PAPER.md:57-65, :173 as read in DESIGN.md section 2), so that a later change to the
oracle's arithmetic cannot pass unnoticed: tests/test_oracle_pins.py::test_golden_c1_oracle_samples re-computes and
compares.  What makes the oracle RIGHT is pinned elsewhere (P1-P11: closed forms, definitions, brute force)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle as orc  # noqa: E402
import synthgen as sg  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle_samples.txt")
SLICES = (0, 3, 7)
PIXELS = ((64, 64), (40, 70), (90, 52), (64, 20), (10, 10), (100, 96), (57, 81), (127, 0))   # (iy, ix)


def compute():
    w = sg.make_workload("C1")
    rows = list(SLICES)
    raw, _ = sg.make_counts(w, rows)
    flat, dark, _, _ = sg.make_flat_dark(w, rows)
    vals = {}
    for method, m in (("grid", 3), ("grid", 4), ("exact", 3), ("lin", 3)):
        out = orc.recon(raw, flat, dark, w.theta, w.center, w.filter, m, method)
        for si, z in enumerate(SLICES):
            for (iy, ix) in PIXELS:
                vals[(method, m, z, iy, ix)] = float(out[si, iy, ix])
    return vals


def main():
    vals = compute()
    with open(OUT, "w") as f:
        f.write("# oracle reconstruction of BASELINE.json config C1 (seed 20220908 + 0), written by tests/golden/make_golden.py\n")
        f.write("# (calls only oracle/ and synthgen/).  Stages S1-S7: PAPER.md:57-65, :173; readings: DESIGN.md section 2.\n")
        f.write("# columns: method  m  slice  iy  ix  value (attenuation per pixel, double precision, %.17e)\n")
        for (method, m, z, iy, ix), v in sorted(vals.items()):
            f.write("%s %d %d %d %d %.17e\n" % (method, m, z, iy, ix, v))
    print("wrote", OUT, len(vals), "values")


if __name__ == "__main__":
    main()
