#!/usr/bin/env python
"""Writes the stored oracle values of tests/golden/ (see README.md).  Calls only oracle/ and the seeded input generators."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle as O                       # noqa: E402
from paper_2202_03411_b200 import workloads as W     # noqa: E402  (input generators: no method arithmetic)


def cfg1_pixels():
    w = W.config(0)
    pix = W.sample_pixels(12345, w.npix, 24, always=[0, w.npix - 1, w.npy // 2 * w.npx + w.npx // 2])
    I = O.simulate(w.grid(0), (w.dx, w.dy, w.dz), w.lam, w.npx, w.npy, w.theta_max_deg, pixels=pix)
    return w, pix, I


def main():
    w, pix, I = cfg1_pixels()
    with open(os.path.join(HERE, "cfg1_oracle_pixels.txt"), "w") as f:
        f.write("# FP64 oracle (oracle/msft_oracle.c, direct triple sum of Eq. 2/9) on BASELINE.json config 1: sphere R = 60 nm on a 32^3 grid\n"
                "# (4 nm voxels), delta = 0.01, beta = 0.001, lambda = 20 nm, 64 x 64 flat detector to +-30 degrees.  Written by make_golden.py.\n"
                "# columns: pixel index (iy * 64 + ix), intensity I (nm^6)\n")
        for p, v in zip(pix, I):
            f.write(f"{int(p)} {float(v)!r}\n")
    print("wrote cfg1_oracle_pixels.txt", len(pix), "pixels")


if __name__ == "__main__":
    main()
