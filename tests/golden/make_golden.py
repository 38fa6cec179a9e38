"""Writes tests/golden/nudft_tiny16.txt: path-A (exact NUDFT, Eq. 7 + Eq. 3 filter) output on a
seeded 16x16x8 case.  Calls only oracle/ and numpy.  Run:  python tests/golden/make_golden.py
The stored values guard the pinned oracle against silent later changes; they are never produced by the CUDA path."""
import math
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import lam_oracle as O  # noqa: E402


def case():
    rng = np.random.default_rng(20240111)
    n, nz, h, w, nth = 16, 8, 16, 16, 10
    theta = 2 * np.pi * np.arange(nth) / nth
    d = rng.standard_normal((nth, h, w)).round(3)
    geom = O.Geometry(n=n, nz=nz, h=h, w=w, theta=theta, phi=math.radians(20.0), filter="ramp")
    return geom, d


if __name__ == "__main__":
    geom, d = case()
    vol = O.fbp_nudft(geom, d)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "nudft_tiny16.txt")
    with open(out, "w") as f:
        f.write("# path A (oracle/lam_oracle.cpp orc_fbp_nudft) on tests/golden/make_golden.py:case();"
                " Eq. 7 PAPER.md:128, filter Eq. 3 PAPER.md:103,109; vol[nz=8][16][16], %.17g\n")
        np.savetxt(f, vol.reshape(geom.nz, -1), fmt="%.17g")
    print("wrote", out)
