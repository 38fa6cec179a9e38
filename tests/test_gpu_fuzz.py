"""Randomised GPU parity sweep: shapes, angle sets, tilts, filters, kernel widths, axis offsets, padding, spectral
multiplier and batch sizes drawn at random (seeded), white-noise or ramp-like projections, ten random x3-columns each
against the exact path A (Eq. 7).  Gates per kernel width (path A has no gridding kernel: Kaiser-Bessel at
sigma = 2 aliases at ~1e-3 for W = 4, ~5e-6 for W = 6, ~1e-7 for W = 8, where fp32 takes over)."""
import math

import numpy as np
import pytest
import torch

from oracle import lam_oracle as O
from paper_2401_11101_b200 import lam

pytestmark = pytest.mark.gpu
TOL = {4: 5e-3, 6: 1e-4, 8: 5e-5}


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_configurations_against_exact_columns(seed):
    rng = np.random.default_rng(seed)
    worst = 0.0
    for it in range(16):
        n = int(rng.choice([32, 64, 128]))
        nz = int(rng.choice([16, 32, 64]))
        h = int(rng.choice([32, 64, 128, 256]))
        w = int(rng.choice([32, 64, 128, 256]))
        nth = int(rng.choice([1, 2, 7, 33, 100, 257, 300, 600]))   # > 256 lines: tiles split over several jobs
        phi = float(rng.uniform(0, math.radians(60)))
        theta = rng.uniform(0, 2 * np.pi, nth) if rng.random() < 0.4 else np.linspace(0, 2 * np.pi, nth, endpoint=False)
        filt = str(rng.choice(["ramp", "none", "shepp-logan", "parzen"]))
        cu = w / 2 + (float(rng.uniform(-3, 3)) if rng.random() < 0.5 else 0.0)
        cv = h / 2 + (float(rng.uniform(-2, 2)) if rng.random() < 0.3 else 0.0)
        Wk = int(rng.choice([4, 6, 6, 6, 8]))
        pad = bool(rng.random() < 0.2) and filt != "none"
        alpha = float(rng.choice([0.0, 0.0, 30.0]))
        if rng.random() < 0.5:
            proj = rng.normal(size=(nth, h, w)).astype(np.float32)                         # full band: wrap and Nyquist bins
        else:
            proj = (np.abs(rng.normal(size=(nth, h, w))).cumsum(axis=2) / w).astype(np.float32)  # does not vanish at the edge
        plan = lam.Plan(n, h, w, theta, phi, nz=nz, filter=filt, center_u=cu, center_v=cv, width=Wk, pad_u=pad,
                        spectral_alpha=alpha, plane_batch=int(rng.choice([0, 1, 3])), theta_chunk=int(rng.choice([0, 1, 5])))
        vol = plan.backproject(torch.from_numpy(proj).cuda()).cpu().numpy()
        plan.close()
        g = O.Geometry(n, h, w, theta, phi, nz=nz, filter=filt, cu=cu, cv=cv, pad=2 if pad else 1, alpha=alpha)
        cols = rng.integers(0, n, size=(10, 2)).astype(np.int32)
        ref = O.fbp_nudft(g, proj, cols=cols)
        got = np.stack([vol[:, c[1], c[0]] for c in cols])
        e = float(np.linalg.norm(got - ref) / (np.linalg.norm(ref) + 1e-300))
        what = (f"seed {seed} case {it}: n={n} nz={nz} h={h} w={w} nth={nth} phi={math.degrees(phi):.1f} {filt} W={Wk} "
                f"pad={pad} alpha={alpha} cu={cu - w / 2:+.2f} cv={cv - h / 2:+.2f}")
        assert np.isfinite(got).all(), what
        assert e <= TOL[Wk], f"{what}: rel L2 {e:.3e} > {TOL[Wk]:.0e}"
        worst = max(worst, e / TOL[Wk])
    print(f"seed {seed}: worst error / gate = {worst:.2f}")


@pytest.mark.parametrize("seed", [11, 12])
def test_random_configurations_adjoint_identity(seed):
    """<L f, d> = <f, L* d> ("adjoint") on random shapes: lam_forward (tile-staged gather on the k_spread work
    lists) against lam_backproject with filter none, random f and d, relative 2e-5 (fp32 sums of ~1e6 terms)."""
    rng = np.random.default_rng(seed)
    for it in range(10):
        n = int(rng.choice([32, 64, 128]))
        nz = int(rng.choice([16, 32, 64]))
        h = int(rng.choice([32, 64, 128, 256]))
        w = int(rng.choice([32, 64, 128, 256]))
        nth = int(rng.choice([1, 3, 40, 257, 400]))
        phi = float(rng.uniform(0, math.radians(60)))
        theta = rng.uniform(0, 2 * np.pi, nth) if rng.random() < 0.5 else np.linspace(0, 2 * np.pi, nth, endpoint=False)
        Wk = int(rng.choice([4, 6, 8]))
        cu = w / 2 + (float(rng.uniform(-3, 3)) if rng.random() < 0.5 else 0.0)
        plan = lam.Plan(n, h, w, theta, phi, nz=nz, filter="none", width=Wk, center_u=cu, plane_batch=int(rng.choice([0, 2])))
        f = torch.from_numpy(rng.normal(size=(nz, n, n)).astype(np.float32)).cuda()
        d = torch.from_numpy(rng.normal(size=(nth, h, w)).astype(np.float32)).cuda()
        Lf = plan.forward(f)
        LTd = plan.backproject(d)
        plan.close()
        a = float((Lf.double() * d.double()).sum())
        b = float((f.double() * LTd.double()).sum())
        scale = float(Lf.double().norm() * d.double().norm())
        assert abs(a - b) <= 2e-5 * scale, f"seed {seed} case {it}: n={n} nz={nz} h={h} w={w} nth={nth} W={Wk}: {a} vs {b} (scale {scale})"
