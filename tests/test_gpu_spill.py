"""S5 for real (SURVEY.md 8(a) row S5, PAPER.md:172 "> 64 GB for 2048^3", :181-191): params.device_bytes decides between
the in-core workspace and the SPILLED schedule (spectra in bands of planes, cropped planes through plan-owned pinned
host memory, x3 stage per slab).  The spilled result must equal the in-core one and match the oracle."""
import numpy as np
import pytest
import torch

from oracle import lam_oracle as O
from paper_2401_11101_b200 import inputs, lam

from gates import L2_CLEAN, L2_NOISY, MAXABS_CLEAN, MAXABS_NOISY, check

pytestmark = pytest.mark.gpu


def _plan(cfg, d, **kw):
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, input="u16" if cfg.raw16 else "f32", **kw)
    if cfg.raw16:
        plan.set_darkflat(d["dark"].cuda(), d["flat"].cuda())
    return plan


def _geom(cfg, d):
    dark = d["dark"].numpy() if d["dark"] is not None else None
    flat = d["flat"].numpy() if d["flat"] is not None else None
    return O.Geometry(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, dark=dark, flat=flat)


@pytest.mark.parametrize("idx,n,host", [(4, 128, False), (4, 128, True), (2, 128, False), (4, 256, True)])
def test_capped_device_budget_runs_the_spilled_schedule(idx, n, host):
    cfg = inputs.scaled(idx, n)
    d = inputs.projections(cfg)
    ref_plan = _plan(cfg, d)
    full = ref_plan.info()["device_bytes"]
    vol_ref = ref_plan.backproject(d["proj"].cuda()).cpu().numpy()
    assert ref_plan.info()["out_of_core"] & 2 == 0
    ref_plan.close()
    # a budget well under the in-core workspace: several bands of planes, several plane batches, several slabs
    plan = _plan(cfg, d, device_bytes=int(0.35 * full))
    info = plan.info()
    assert info["out_of_core"] & 2, info
    assert info["pinned_bytes"] >= info["planes"] * cfg.n * cfg.n * 8
    assert info["device_bytes"] <= 0.5 * full, (info, full)
    if host:
        hp = d["proj"].pin_memory()
        hv = torch.empty((cfg.nz, cfg.n, cfg.n), dtype=torch.float32).pin_memory()
        plan.backproject(hp, hv)
        vol = hv.numpy().copy()
    else:
        vol = plan.backproject(d["proj"].cuda()).cpu().numpy()
    torch.cuda.synchronize()
    # repeat call: the double buffers and events are reusable
    vol2 = plan.backproject(d["proj"].cuda()).cpu().numpy()
    plan.close()
    assert np.abs(vol - vol_ref).max() <= 2e-6 * np.abs(vol_ref).max(), "spilled and in-core schedules differ"
    assert np.abs(vol2 - vol_ref).max() <= 2e-6 * np.abs(vol_ref).max()
    rng = np.random.default_rng(11)
    cols = rng.integers(2, cfg.n - 2, size=(16, 2)).astype(np.int32)
    ref = O.fbp_nudft(_geom(cfg, d), d["proj"].numpy(), cols=cols)
    got = np.stack([vol[:, c[1], c[0]] for c in cols])
    gate = (L2_NOISY, MAXABS_NOISY) if cfg.raw16 else (L2_CLEAN, MAXABS_CLEAN)
    print("spilled", cfg.name, info, check(got, ref, *gate, "spilled vs exact columns"))


def test_budget_too_small_even_for_the_spilled_schedule_fails_cleanly():
    cfg = inputs.scaled(4, 128)
    d = inputs.projections(cfg)
    with pytest.raises(lam.LamError) as e:
        _plan(cfg, d, device_bytes=1 << 20)
    assert e.value.status == lam.LAM_ENOMEM_DEVICE


def test_forward_and_slice_need_the_in_core_workspace():
    cfg = inputs.scaled(2, 128)
    d = inputs.projections(cfg)
    probe = _plan(cfg, d)
    full = probe.info()["device_bytes"]
    probe.close()
    plan = _plan(cfg, d, device_bytes=int(0.35 * full))
    with pytest.raises(lam.LamError) as e:
        plan.backproject_slice(d["proj"].cuda(), 3)
    assert e.value.status == lam.LAM_EUNSUPPORTED
    plan.close()
