"""lam_forward, lam_backproject_slice and lam_admm_tv at the transform lengths and launch shapes bench.py times them at
(configs[2]: sigma*n = 2048, h = w = 1024, sigma*nz = 512) and at every long FFT length of configs[3]/[4], against the
fp64 oracle.  The small-size parity of the same entry points is in test_gpu_parity.py / test_gpu_next.py /
test_gpu_admm.py; the template instantiations k_fft_x1_T<11..13>, k_fft_x2_T<11..13>, k_cols_T<10..12>,
k_rows_T<10..11>, k_zstage_T<9..10>, k_gather on the tiles of a 2048^2 .. 8192^2 plane and k_slice_reduce over 513 planes
only exist at these sizes.

How the exact oracle reaches these sizes:
  * lam_forward (Eq. 5).  For a volume f supported on a few x3-columns and any projection-space vector d,
    <L f, d> = <f, L* d> = sum over those columns of f . (L* d), and the columns of L* d are what the oracle's exact
    path A evaluates (O.fbp_nudft(..., cols), filter none; Eq. 7).  With d a unit sample this is ONE
    detector value of L f, exactly; with d dense it is a weighted sum of all of them.  The spectrum of a few columns is
    full-band plane waves: every tile of every plane carries data.  Dense random f is covered by the adjoint identity
    against lam_backproject, whose columns the oracle checks at the same shapes (test_gpu_parity.py).
  * lam_backproject_slice: sampled voxels of the slice against exact path-A columns computed with
    the shifted axis, on the DENSE configs[2] scan at full size.
  * lam_admm_tv (Eqs. 10-20): oracle/admm_tv.py runs the paper's iterations in fp64 numpy with the
    operator pair handed in; at these sizes its exact pair is out of reach, so it is given the GPU's lam_forward /
    lam_backproject (each checked against the exact pair at this shape above and in test_gpu_parity.py).  What is
    compared is everything else: TV gradient / divergence, shrinkage, the fp64 reductions, the CG recurrences.
"""
import math

import numpy as np
import pytest
import torch

from oracle import admm_tv as A
from oracle import lam_oracle as O
from paper_2401_11101_b200 import inputs, lam

from gates import L2_NOISY, MAXABS_NOISY, check

pytestmark = pytest.mark.gpu
# one detector value of L f against max |L f| (measured <= 2e-6: Kaiser-Bessel W = 6 aliasing + fp32 transforms), and a
# dense weighted sum against ||L f|| ||d|| (measured <= 4e-7); both 10x above what was measured
SAMPLE_GATE, SUM_GATE = 2e-5, 5e-6

#         n    nz     h     w  nth
SHAPES = [(2048, 32, 64, 64, 6),       # sigma*n = 4096
          (1024, 32, 2048, 64, 6),     # h = 2048
          (256, 512, 64, 2048, 6),     # w = 2048, sigma*nz = 1024
          (4096, 16, 32, 32, 4),       # sigma*n = 8192
          (256, 16, 4096, 32, 4),      # h = 4096
          (1024, 16, 1024, 1024, 6),   # configs[2]: sigma*n = 2048, h = w = 1024 (bench.py next_rows)
          (64, 256, 64, 64, 6)]        # configs[2]: sigma*nz = 512


@pytest.mark.parametrize("n,nz,h,w,nth", SHAPES)
def test_forward_at_long_transform_lengths(n, nz, h, w, nth):
    rng = np.random.default_rng(n + h + w)
    theta = 2 * np.pi * np.arange(nth) / nth + 0.07
    phi = math.radians(20.0)
    cu = w / 2 + 0.3
    plan = lam.Plan(n, h, w, theta, phi, nz=nz, filter="none", center_u=cu)
    geom = O.Geometry(n, h, w, theta, phi, nz=nz, filter="none", cu=cu)

    # (1) exact detector samples and exact weighted sums of L f, f on four columns
    r = min(n // 4, w // 3)
    cols = (n // 2 + rng.integers(-r, r, size=(4, 2))).astype(np.int32)
    fcols = rng.normal(size=(len(cols), nz))
    f = torch.zeros((nz, n, n), dtype=torch.float32)
    for c, v in zip(cols, fcols):
        f[:, int(c[1]), int(c[0])] += torch.from_numpy(v.astype(np.float32))
    fcols = np.stack([f[:, int(c[1]), int(c[0])].numpy().astype(np.float64) for c in cols])   # what the GPU reads
    Lf = plan.forward(f.cuda()).cpu().numpy().astype(np.float64)
    top = np.abs(Lf).max()
    worst = 0.0
    for k in range(6):
        d = np.zeros((nth, h, w), dtype=np.float32)
        if k < 4:      # one detector sample: near the axis, at the detector edges, anywhere
            t, jv, ju = [(0, h // 2, w // 2 + 1), (nth - 1, 0, w - 1), (1, h - 1, 0),
                         (int(rng.integers(nth)), int(rng.integers(h)), int(rng.integers(w)))][k]
            d[t, jv, ju] = 1.0
        else:
            d = rng.normal(size=(nth, h, w)).astype(np.float32)
        LTd = O.fbp_nudft(geom, d, cols=cols)                      # exact columns of L* d, [ncols][nz]
        ref = float((fcols * LTd).sum())
        got = float((Lf * d.astype(np.float64)).sum())
        scale = top if k < 4 else float(np.linalg.norm(Lf) * np.linalg.norm(d))
        err = abs(got - ref) / scale
        assert err <= (SAMPLE_GATE if k < 4 else SUM_GATE), f"n={n} nz={nz} h={h} w={w}: d #{k}: {got} vs {ref} (scale {scale})"
        worst = max(worst, err / (SAMPLE_GATE if k < 4 else SUM_GATE))

    # (2) dense random f, d: exact transposes stage by stage
    fd = torch.from_numpy(rng.normal(size=(nz, n, n)).astype(np.float32)).cuda()
    dd = torch.from_numpy(rng.normal(size=(nth, h, w)).astype(np.float32)).cuda()
    Lfd = plan.forward(fd)
    LTd = plan.backproject(dd)
    a, b = float((Lfd.double() * dd.double()).sum()), float((fd.double() * LTd.double()).sum())
    scale = float(Lfd.double().norm() * dd.double().norm())
    plan.close()
    assert abs(a - b) <= 1e-5 * scale, (a, b, scale)
    print(f"lam_forward n={n} nz={nz} h={h} w={w}: exact samples / sums worst error/gate {worst:.2f}, "
          f"adjoint identity {abs(a - b) / scale:.1e}")


def test_slice_search_on_configs2_at_full_size():
    """`try` on the dense configs[2] scan as bench.py next_rows times it: 513 planes reduced onto one 2048^2 grid."""
    cfg = inputs.config(2)
    d = inputs.projections(cfg, device="cuda")
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample)
    shifted = cfg.w / 2 + 2.5
    slices = [cfg.nz // 2 - 3, cfg.nz // 2 + 40]
    got = {i3: plan.backproject_slice(d["proj"], i3, [cfg.w / 2, shifted]).cpu().numpy() for i3 in slices}
    vol = plan.backproject(d["proj"])
    torch.cuda.synchronize()
    for i3 in slices:    # the plan's own axis: the slice of the full volume (itself checked on exact columns at full size)
        print(f"slice {i3} vs full volume:", check(got[i3][0], vol[i3].cpu().numpy(), 1e-4, 5e-4, f"slice {i3} vs full volume"))
    del vol
    plan.close()
    proj = d["proj"].cpu().numpy()
    del d
    torch.cuda.empty_cache()
    rng = np.random.default_rng(22)
    rr, aa = 0.45 * cfg.n * np.sqrt(rng.uniform(size=32)), rng.uniform(0, 2 * np.pi, size=32)
    cols = np.stack([cfg.n // 2 + np.round(rr * np.cos(aa)), cfg.n // 2 + np.round(rr * np.sin(aa))], axis=1).astype(np.int32)
    ref = O.fbp_nudft(O.Geometry(cfg.n, cfg.h, cfg.w, cfg.theta(), cfg.phi, nz=cfg.nz, cu=shifted), proj, cols=cols)
    for i3 in slices:    # the shifted axis: exact path A with that axis, 32 voxels of the slice
        pts = np.array([got[i3][1][int(c[1]), int(c[0])] for c in cols])
        print(f"slice {i3}, axis +2.5 px, 32 exact voxels:", check(pts, ref[:, i3], L2_NOISY, MAXABS_NOISY, f"slice {i3} shifted axis"))
    # the shift is visible: the own-axis slice fails the same comparison by a wide margin
    own = np.array([got[slices[0]][0][int(c[1]), int(c[0])] for c in cols])
    assert np.linalg.norm(own - ref[:, slices[0]]) > 0.05 * np.linalg.norm(ref[:, slices[0]])


def test_admm_tv_at_configs2_transform_lengths():
    """2 x 2 iterations at sigma*n = 2048, h = w = 1024 against the oracle's iterations on the same operator pair."""
    n, nz, h, w, nth, phi = 1024, 16, 1024, 1024, 6, 0.4
    theta = np.linspace(0, 2 * np.pi, nth, endpoint=False)
    rng = np.random.default_rng(5)
    plan = lam.Plan(n, h, w, theta, phi, nz=nz, filter="none")

    def L(f):
        return plan.forward(torch.from_numpy(np.ascontiguousarray(f, dtype=np.float32)).cuda()).cpu().numpy().astype(np.float64)

    def LT(r):
        return plan.backproject(torch.from_numpy(np.ascontiguousarray(r, dtype=np.float32)).cuda()).cpu().numpy().astype(np.float64)

    mu_true = np.zeros((nz, n, n))
    mu_true[5:11, 300:700, 260:640] = 1.0
    mu_true[6:9, 420:560, 700:860] = 0.5
    d = (L(mu_true) + 0.05 * rng.normal(size=(nth, h, w))).astype(np.float32)
    alpha, rho, n_outer, n_cg = 0.3, 1.0, 2, 2
    vol, hist = plan.admm_tv(torch.from_numpy(d).cuda(), alpha, rho, n_outer, n_cg)
    got = vol.cpu().numpy().astype(np.float64)
    geom = O.Geometry(n, h, w, theta, phi, nz=nz, filter="none")
    mu_ref, href = A.admm_tv(geom, d.astype(np.float64), alpha, rho, n_outer, n_cg, L=L, LT=LT, track=False)
    plan.close()
    e = np.linalg.norm(got - mu_ref) / np.linalg.norm(mu_ref)
    print("admm-tv at n = 1024:", e, "||grad F|| gpu", hist, "oracle iterations", href["gnorm_steps"])
    assert e <= 5e-5, e
    assert np.abs(got - mu_ref).max() <= 2e-4 * np.abs(mu_ref).max()
    assert np.allclose(hist, href["gnorm_steps"], rtol=1e-3)
