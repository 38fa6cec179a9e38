"""Parity gates shared by the GPU tests (DESIGN.md section 2 "Tolerances").

Two levels.  The north_star gates are hard ceilings: rel L2 <= 2e-4 against the exact path A on configs[0]-sized
cases, <= 1e-3 on larger cases.  The TIGHT gates sit about 10x above what the arithmetic gives (Kaiser-Bessel W = 6,
sigma = 2 aliasing ~4e-6, fp32 FFT round-off ~1e-6, fp32 accumulation of N_theta W^2 taps per cell ~1e-6 sqrt(taps),
uint16 inputs: the -log in fp32): a wrong tile edge, a mis-merged tile or a wrong Nyquist column in a few voxels moves
the max-abs figure by orders of magnitude long before it moves a whole-array norm, so every comparison checks both.
"""
import numpy as np

NORTH_TINY = 2e-4    # north_star: configs[0] against the exact oracle
NORTH_LARGE = 1e-3   # north_star: larger configs against the gridded oracle / exact columns
L2_CLEAN = 5e-5      # tight: noise-free fp32 inputs (measured 6e-7 .. 9.4e-6, white noise the largest)
L2_NOISY = 2e-4      # tight: noisy / uint16 / full-size inputs (measured 1e-5 .. 2.4e-5)
L2_RAW_SPARSE = 4e-4 # tight: full-size uint16 scans with data at 1-4 % of the angles (measured 6e-5 .. 1.5e-4: the
                     #        signal is K/N_theta of a dense scan's, the fp32 -log and FFT round-off floor is not)
MAXABS_CLEAN = 1e-4  # max |got - ref| <= c max |ref|   (measured 1e-6 .. 1.3e-5)
MAXABS_NOISY = 1e-3


def rel(a, b):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def maxabs(a, b):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.abs(a - b).max() / np.abs(b).max())


def check(got, ref, l2, linf, what=""):
    """Both gates; returns (rel L2, max-abs / max |ref|) for the log."""
    got = np.asarray(got)
    assert np.isfinite(got).all(), what
    e2, ei = rel(got, ref), maxabs(got, ref)
    assert e2 <= l2, f"{what}: rel L2 {e2:.3e} > {l2:.1e} (max-abs {ei:.3e})"
    assert ei <= linf, f"{what}: max-abs {ei:.3e} > {linf:.1e} (rel L2 {e2:.3e})"
    return e2, ei
