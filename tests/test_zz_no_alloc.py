"""lam_backproject_slice_static: the rotation-axis search for callers that cannot allocate device memory.

Some users of this library build their plans once, while their program starts, and from then on must keep away from
cudaMalloc: a preview service that re-runs the axis search between detector frames (cudaMalloc synchronises the whole
device and takes as long as it likes), or a process whose own memory pool (PyTorch, CuPy) has by then taken every free
byte, so that the five first-use allocations of lam_backproject_slice would fail.  lam_backproject_slice_static does the
same work on a 16 MiB scratch array that is part of liblam.so's device image (sigma*n <= 1024), shared by all calls.

What is checked here, against the allocating entry point on the same inputs and at the gates the slice tests use:
two calls one straight after the other (the second starts from the first one's leftovers in the shared scratch), a
third call from a plan of another shape (different sub-buffer offsets over the same bytes), that the plan's device
byte count does not move, and that a plan too large for the scratch is refused with a message instead of overrunning it.

This file sorts last on purpose (pytest -x stops at the first failure): it needs nothing from the tests before it and
passes on its own in a fresh process as well.
"""
import numpy as np
import pytest
import torch

from paper_2401_11101_b200 import inputs, lam

from gates import L2_CLEAN, L2_NOISY, MAXABS_CLEAN, MAXABS_NOISY, check

pytestmark = pytest.mark.gpu


def _plan(cfg, d):
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample,
                    input="u16" if cfg.raw16 else "f32")
    if cfg.raw16:
        plan.set_darkflat(d["dark"].cuda(), d["flat"].cuda())
    return plan


def test_static_scratch_slices_match_the_allocating_entry_point_on_consecutive_calls():
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    proj = d["proj"].cuda()
    calls = [(cfg.nz // 2, [cfg.w / 2 - 1.5, cfg.w / 2, cfg.w / 2 + 3.0]),
             (cfg.nz // 2 + 5, [cfg.w / 2 + 0.75, cfg.w / 2 - 2.0])]
    # the existing path, on a plan of its own: the plan under test never gets slice buffers of its own
    ref_plan = _plan(cfg, d)
    refs = [ref_plan.backproject_slice(proj, i3, c).cpu().numpy() for i3, c in calls]
    ref_plan.close()

    plan = _plan(cfg, d)
    outs = [torch.full((len(c), cfg.n, cfg.n), float("nan"), device="cuda") for _, c in calls]
    bytes_before = plan.info()["device_bytes"]
    free = []
    for (i3, c), out in zip(calls, outs):      # two calls in a row, nothing in between
        plan.backproject_slice(proj, i3, c, out=out, static_scratch=True)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    assert plan.info()["device_bytes"] == bytes_before, "the static entry point grew the plan's device workspace"
    print("free device bytes after call 1 / 2:", free)
    for k, ((i3, c), out, ref) in enumerate(zip(calls, outs, refs)):
        e = check(out.cpu().numpy(), ref, L2_CLEAN, MAXABS_CLEAN, f"static scratch, call {k + 1} (slice {i3})")
        print(f"static vs allocating, call {k + 1}:", e)
    assert np.linalg.norm(refs[0][0] - refs[1][0]) > 0.05 * np.linalg.norm(refs[0][0])   # the two calls differ

    # a plan of another shape (uint16 input, n = 128) lays its buffers out differently over the same scratch, then the
    # first plan again: stale contents of either must not leak into the other
    cfg2 = inputs.scaled(3, 128)
    d2 = inputs.projections(cfg2)
    proj2 = d2["proj"].cuda()
    plan2 = _plan(cfg2, d2)
    c2 = [cfg2.w / 2 + 0.5]
    got2 = plan2.backproject_slice(proj2, cfg2.nz // 2 + 1, c2, static_scratch=True).cpu().numpy()
    ref2 = plan2.backproject_slice(proj2, cfg2.nz // 2 + 1, c2).cpu().numpy()      # same plan, allocating path
    print("other shape:", check(got2, ref2, L2_NOISY, MAXABS_NOISY, "static scratch, n = 128 raw plan"))
    plan2.close()
    again = plan.backproject_slice(proj, calls[0][0], calls[0][1], static_scratch=True).cpu().numpy()
    print("first plan again:", check(again, refs[0], L2_CLEAN, MAXABS_CLEAN, "static scratch after another plan"))
    assert plan.info()["device_bytes"] == bytes_before
    plan.close()


def test_static_scratch_refuses_plans_that_do_not_fit():
    n = 1024                                    # sigma * n = 2048: 56 MiB of slice scratch against 16 MiB
    theta = np.linspace(0.0, 2.0 * np.pi, 8, endpoint=False)
    plan = lam.Plan(n, 32, 64, theta, 0.35, nz=16)
    proj = torch.zeros((8, 32, 64), device="cuda")
    out = torch.zeros((1, n, n), device="cuda")
    with pytest.raises(lam.LamError) as e:
        plan.backproject_slice(proj, 8, out=out, static_scratch=True)
    assert e.value.status == lam.LAM_EUNSUPPORTED
    assert "static" in str(e.value) and "lam_backproject_slice" in str(e.value)
    plan.backproject_slice(proj, 8, out=out)    # the allocating path still serves it
    torch.cuda.synchronize()
    plan.close()
