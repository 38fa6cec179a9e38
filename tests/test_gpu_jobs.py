"""Work lists of the (xi1, xi2) gridding on angle lists that are not a monotone sweep (include/lam.h: theta may hold
"any values").  A theta range of a job record has an 11-bit length; a tile that is crossed by every 10th angle of a long
single-orientation list keeps one range open across the misses in between (up to 32 are tolerated), so the range grows
past 2047 thetas unless k_jobs closes it in time.  Compared on exact x3-columns of path A (Eq. 7, PAPER.md:128;
frequencies of Eq. 6)."""
import math

import numpy as np
import pytest
import torch

from oracle import lam_oracle as O
from paper_2401_11101_b200 import lam

from gates import L2_CLEAN, MAXABS_CLEAN, check

pytestmark = pytest.mark.gpu


def interlaced_angles(nth, rng):
    """Every 10th angle lies in a narrow fan around 40 degrees, the nine in between in a fan around 5 degrees: all of one
    orientation (|cos| > |sin|), so the outer tiles near the 40-degree diagonal are hit with stride 10 from the first
    angle to the last."""
    theta = np.radians(rng.uniform(-5.0, 15.0, nth))
    theta[::10] = np.radians(rng.uniform(38.0, 43.0, len(theta[::10])))
    return theta


@pytest.mark.parametrize("nth,filt", [(4100, "ramp"), (2300, "none")])
def test_theta_ranges_longer_than_the_length_field(nth, filt):
    rng = np.random.default_rng(nth)
    n, nz, h, w, phi = 64, 16, 32, 64, math.radians(20.0)
    theta = interlaced_angles(nth, rng)
    proj = rng.normal(size=(nth, h, w)).astype(np.float32)
    plan = lam.Plan(n, h, w, theta, phi, nz=nz, filter=filt)
    vol = plan.backproject(torch.from_numpy(proj).cuda()).cpu().numpy()
    if filt == "none":   # the transpose walks the same job records
        f = torch.from_numpy(rng.normal(size=(nz, n, n)).astype(np.float32)).cuda()
        d = torch.from_numpy(proj).cuda()
        a = float((plan.forward(f).double() * d.double()).sum())
        b = float((f.double() * torch.from_numpy(vol).cuda().double()).sum())
        assert abs(a - b) <= 2e-5 * float(plan.forward(f).double().norm() * d.double().norm()), (a, b)
    plan.close()
    cols = rng.integers(0, n, size=(12, 2)).astype(np.int32)
    cols[:4] = [[60, 58], [57, 61], [3, 5], [6, 2]]          # inside the tiles the 40-degree fan reaches
    ref = O.fbp_nudft(O.Geometry(n, h, w, theta, phi, nz=nz, filter=filt), proj, cols=cols)
    got = np.stack([vol[:, c[1], c[0]] for c in cols])
    print(f"interlaced {nth} angles, {filt}:", check(got, ref, L2_CLEAN, MAXABS_CLEAN, "long theta ranges"))
