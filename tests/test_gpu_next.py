"""GPU parity of the SURVEY.md 8(f) rows built after the hot path: f3 single-slice `try` / `try-lamino` search
 and f4 Parzen window, u-padding, 2-D spectral multiplier, each against the
CPU fp64 oracle's exact path A (Eq. 7) on the same seeded inputs, through the C ABI."""
import math

import numpy as np
import pytest
import torch

from oracle import lam_oracle as O
from paper_2401_11101_b200 import inputs, lam

from gates import L2_CLEAN, L2_NOISY, MAXABS_CLEAN, MAXABS_NOISY, check

pytestmark = pytest.mark.gpu


def _geom(cfg, d, **kw):
    dark = d["dark"].numpy() if d["dark"] is not None else None
    flat = d["flat"].numpy() if d["flat"] is not None else None
    return O.Geometry(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, dark=dark, flat=flat, **kw)


def _plan(cfg, d, **kw):
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample,
                    input="u16" if cfg.raw16 else "f32", **kw)
    if cfg.raw16:
        plan.set_darkflat(d["dark"].cuda(), d["flat"].cuda())
    return plan


def _run(cfg, d, **kw):
    plan = _plan(cfg, d, **kw)
    vol = plan.backproject(d["proj"].cuda())
    torch.cuda.synchronize()
    plan.close()
    return vol.cpu().numpy()


# ---- f4 ----------------------------------------------------------------------------------------------------------------
def test_parzen_filter_against_exact_nudft():
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    vol = _run(cfg, d, filter="parzen")
    ref = O.fbp_nudft(_geom(cfg, d, filter="parzen"), d["proj"].numpy())
    print("parzen:", check(vol, ref, L2_CLEAN, MAXABS_CLEAN, "parzen"))
    ramp = O.fbp_nudft(_geom(cfg, d), d["proj"].numpy())
    assert np.linalg.norm(ref - ramp) > 0.05 * np.linalg.norm(ramp)   # the window is not a no-op


@pytest.mark.parametrize("alpha", [40.0, 900.0])
def test_spectral_multiplier_against_exact_nudft(alpha):
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    vol = _run(cfg, d, spectral_alpha=alpha)
    ref = O.fbp_nudft(_geom(cfg, d, alpha=alpha), d["proj"].numpy())
    print("alpha", alpha, check(vol, ref, L2_CLEAN, MAXABS_CLEAN, "spectral multiplier"))
    plain = O.fbp_nudft(_geom(cfg, d), d["proj"].numpy())
    assert np.linalg.norm(ref - plain) > 0.02 * np.linalg.norm(plain)


@pytest.mark.parametrize("idx,n,filt", [(0, 64, "ramp"), (0, 64, "shepp-logan"), (3, 128, "ramp"), (2, 256, "parzen")])
def test_padded_rows_against_exact_nudft_columns(idx, n, filt):
    """pad_u (reading Q11b): rows edge-extended to 2w before the filter.  w = 64 (two-pass transforms), 128 (uint16
    input) and 256; compared on exact x3-columns of path A with the oracle's padded filtering."""
    cfg = inputs.config(0) if idx == 0 else inputs.scaled(idx, n)
    d = inputs.projections(cfg)
    if not cfg.raw16:   # a background that does not vanish at the detector edge: padding then changes the result visibly
        d["proj"] = d["proj"] + 0.5
    vol = _run(cfg, d, filter=filt, pad_u=True)
    rng = np.random.default_rng(3)
    cols = rng.integers(2, cfg.n - 2, size=(24, 2)).astype(np.int32)
    ref = O.fbp_nudft(_geom(cfg, d, filter=filt, pad=2), d["proj"].numpy(), cols=cols)
    got = np.stack([vol[:, c[1], c[0]] for c in cols])
    gate = (L2_NOISY, MAXABS_NOISY) if cfg.raw16 else (L2_CLEAN, MAXABS_CLEAN)
    print("pad_u", cfg.name, filt, check(got, ref, gate[0], gate[1], "pad_u"))
    nopad = O.fbp_nudft(_geom(cfg, d, filter=filt), d["proj"].numpy(), cols=cols)
    assert np.linalg.norm(ref - nopad) > 1e-3 * np.linalg.norm(nopad)   # teeth: padding is visible in the oracle


# ---- f3 ----------------------------------------------------------------------------------------------------------------
def test_try_slices_for_several_rotation_axes_against_exact_nudft():
    """`try`: one slice, several rotation axes.  Every (centre, slice) against the full exact path A
    with that axis, and against the oracle's own single-slice path C' (Eq. 9 with the exact x3 phase)."""
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    centers = [cfg.w / 2 - 1.5, cfg.w / 2, cfg.w / 2 + 0.75, cfg.w / 2 + 3.0]
    plan = _plan(cfg, d)
    for i3 in (cfg.nz // 2, cfg.nz // 2 + 5, 3):
        out = plan.backproject_slice(d["proj"].cuda(), i3, centers).cpu().numpy()
        for c, img in zip(centers, out):
            g = _geom(cfg, d, cu=c)
            ref = O.fbp_nudft(g, d["proj"].numpy())[i3]
            # slice 3 lies outside the object (|x3| <= 8): only missing-cone tails, 200x weaker than the central slices,
            # so the same absolute error is a larger fraction of that slice's own norm
            l2, li = (L2_CLEAN, MAXABS_CLEAN) if abs(i3 - cfg.nz // 2) <= 8 else (L2_NOISY, MAXABS_NOISY)
            e = check(img, ref, l2, li, f"try slice {i3} centre {c}")
            ref_c = O.fbp_gridded_slice(g, d["proj"].numpy(), i3)
            check(img, ref_c, l2, li, f"try slice {i3} centre {c} vs C'")
        print("try slice", i3, e)
    # the plan's own axis, no list
    own = plan.backproject_slice(d["proj"].cuda(), cfg.nz // 2).cpu().numpy()[0]
    check(own, O.fbp_nudft(_geom(cfg, d), d["proj"].numpy())[cfg.nz // 2], L2_CLEAN, MAXABS_CLEAN, "own axis")
    # and the full volume of the same plan is unchanged by the search (S is rebuilt by every call)
    vol = plan.backproject(d["proj"].cuda()).cpu().numpy()
    check(vol[cfg.nz // 2], own, 1e-4, 5e-4, "slice mode vs full volume")
    plan.close()


def test_try_lamino_slices_for_several_tilts_against_exact_nudft():
    """`try-lamino`: one slice for several tilt angles = one plan per phi."""
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    i3 = cfg.nz // 2 + 6
    for dphi in (-2.0, -0.5, 1.0):
        phi = cfg.phi + math.radians(dphi)
        plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], phi, nz=cfg.nz)
        img = plan.backproject_slice(d["proj"].cuda(), i3).cpu().numpy()[0]
        plan.close()
        ref = O.fbp_nudft(O.Geometry(cfg.n, cfg.h, cfg.w, d["theta"], phi, nz=cfg.nz), d["proj"].numpy())[i3]
        print("try-lamino", dphi, check(img, ref, L2_CLEAN, MAXABS_CLEAN, f"try-lamino {dphi}"))


def test_try_on_a_raw_uint16_scan_with_many_angles():
    """scaled configs[3] (uint16 + dark/flat, multi-writer tiles around the axis) through the slice path."""
    cfg = inputs.scaled(3, 128)
    d = inputs.projections(cfg)
    plan = _plan(cfg, d)
    centers = [cfg.w / 2 + 0.5, cfg.w / 2 - 2.0]
    out = plan.backproject_slice(d["proj"].cuda(), cfg.nz // 2 + 1, centers).cpu().numpy()
    plan.close()
    for c, img in zip(centers, out):
        ref = O.fbp_gridded_slice(_geom(cfg, d, cu=c), d["proj"].numpy(), cfg.nz // 2 + 1)
        print("raw try", c, check(img, ref, L2_NOISY, MAXABS_NOISY, "raw try"))


def test_slice_entry_point_rejects_bad_arguments():
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    plan = _plan(cfg, d)
    out = torch.empty((1, cfg.n, cfg.n), device="cuda")
    with pytest.raises(lam.LamError) as e:
        lam.lam_backproject_slice(plan._plan, d["proj"].cuda().data_ptr(), cfg.nz, None, out.data_ptr())
    assert e.value.status == lam.LAM_EINVAL
    with pytest.raises(lam.LamError) as e:
        lam.lam_backproject_slice(plan._plan, d["proj"].numpy().ctypes.data, 0, None, out.data_ptr())
    assert e.value.status == lam.LAM_EUNSUPPORTED
    plan.close()
