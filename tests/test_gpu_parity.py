"""GPU parity tests: the CUDA path (through the C ABI of include/lam.h) against the CPU fp64 oracle, element by
element on the same seeded inputs.  Gates (BASELINE.json north_star): rel L2 <= 2e-4 against path A (exact NUDFT,
Eq. 7) on configs[0]; <= 1e-3 against the oracle's double gridded path C / exact columns on larger cases.
"""
import math

import numpy as np
import pytest
import torch

from oracle import lam_oracle as O
from paper_2401_11101_b200 import inputs, lam

from gates import L2_CLEAN, L2_NOISY, MAXABS_CLEAN, MAXABS_NOISY, NORTH_LARGE, NORTH_TINY, check, rel

pytestmark = pytest.mark.gpu

GATE_TINY = NORTH_TINY    # north_star: configs[0] against the exact oracle (hard ceiling)
GATE_LARGE = NORTH_LARGE  # north_star: larger configs (hard ceiling)
assert L2_CLEAN <= GATE_TINY and L2_NOISY <= GATE_LARGE


def tight(got, ref, what=""):
    """noise-free fp32 inputs: rel L2 <= 5e-5 and max-abs <= 2e-4 max|ref| (tests/gates.py)"""
    return check(got, ref, L2_CLEAN, MAXABS_CLEAN, what)


def tight_noisy(got, ref, what=""):
    """noisy / uint16 inputs: rel L2 <= 2e-4 and max-abs <= 1e-3 max|ref|"""
    return check(got, ref, L2_NOISY, MAXABS_NOISY, what)


def run_gpu(cfg, d, **kw):
    args = dict(nz=cfg.nz, width=cfg.width, oversample=cfg.oversample, input="u16" if cfg.raw16 else "f32")
    args.update(kw)
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, **args)
    if cfg.raw16:
        plan.set_darkflat(d["dark"].cuda(), d["flat"].cuda())
    vol = plan.backproject(d["proj"].cuda())
    torch.cuda.synchronize()
    info = plan.info()
    plan.close()
    return vol.cpu().numpy(), info


def geometry(cfg, d, **kw):
    dark = d["dark"].numpy() if d["dark"] is not None else None
    flat = d["flat"].numpy() if d["flat"] is not None else None
    return O.Geometry(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, dark=dark, flat=flat, **kw)


def test_version_and_native_library_loaded():
    assert "sm_100a" in lam.lam_version()


def test_config0_tiny_against_exact_nudft_full_volume():
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    vol, info = run_gpu(cfg, d)
    ref = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy())
    assert vol.shape == ref.shape == (cfg.nz, cfg.n, cfg.n)
    print("configs[0] full volume vs exact NUDFT:", tight(vol, ref, "configs[0]"))
    assert info["launches"] > 0


@pytest.mark.parametrize("filt", ["none", "shepp-logan"])
def test_config0_other_filters(filt):
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d, filter=filt)
    ref = O.fbp_nudft(geometry(cfg, d, filter=filt), d["proj"].numpy())
    tight(vol, ref, filt)


def test_config0_gaussian_kernel_w8():
    """The paper's psi is a Gaussian; at W = 8 it meets 1e-3 (reading Q5)."""
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d, kernel="gauss", width=8)
    ref = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy())
    assert rel(vol, ref) <= GATE_LARGE


def test_config0_fractional_rotation_axis():
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    cu, cv = cfg.w / 2 + 1.37, cfg.h / 2 - 0.61
    vol, _ = run_gpu(cfg, d, center_u=cu, center_v=cv)
    ref = O.fbp_nudft(geometry(cfg, d, cu=cu, cv=cv), d["proj"].numpy())
    tight(vol, ref, "fractional axis")


def test_small_batches_give_the_same_answer():
    """plane_batch / theta_chunk only change the launch schedule (ragged last batch included)."""
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    a, _ = run_gpu(cfg, d)
    b, info = run_gpu(cfg, d, plane_batch=5, theta_chunk=7)
    assert info["plane_batch"] == 5 and info["theta_chunk"] == 7
    assert rel(b, a) <= 2e-6


@pytest.mark.parametrize("idx,n", [(1, 128), (2, 128), (2, 256)])
def test_scaled_configs_against_gridded_oracle(idx, n):
    """Same recipes as configs[1], [2] shrunk so that the oracle's path C finishes in seconds; non-cubic slab
    (nz = n/4, h != nz), phi = 20 / 30 degrees, noise, box layer; several gridding tiles and plane batches."""
    cfg = inputs.scaled(idx, n)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d, plane_batch=24)
    ref = O.fbp_gridded(geometry(cfg, d), d["proj"].numpy())
    e = tight_noisy(vol, ref, cfg.name)
    rng = np.random.default_rng(5)
    cols = rng.integers(0, cfg.n, size=(16, 2)).astype(np.int32)
    refA = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy(), cols=cols)     # [ncols][nz]
    got = np.stack([vol[:, c[1], c[0]] for c in cols])
    print(cfg.name, "vs C:", e, "vs A columns:", tight_noisy(got, refA, cfg.name + " columns"))


def test_raw_uint16_darkflat_path():
    """configs[3] recipe (uint16 counts + dark/flat, -log fused) shrunk to n = 128."""
    cfg = inputs.scaled(3, 128)
    d = inputs.projections(cfg)
    assert d["proj"].dtype == torch.uint16
    vol, _ = run_gpu(cfg, d)
    ref = O.fbp_gridded(geometry(cfg, d), d["proj"].numpy())
    print("raw16:", tight_noisy(vol, ref, "raw16"))


def test_wide_detector_nonsquare():
    """configs[4] recipe shrunk (w = 2 h, n = w): detector wider than tall."""
    cfg = inputs.scaled(4, 128)
    d = inputs.projections(cfg)
    assert cfg.w == 2 * cfg.h
    vol, _ = run_gpu(cfg, d)
    ref = O.fbp_gridded(geometry(cfg, d), d["proj"].numpy())
    print("wide detector:", tight_noisy(vol, ref, "wide"))


def test_phi_zero_is_slicewise_tomography():
    """phi = 0 (the Radon transform): every detector row reconstructs its own slice."""
    cfg = inputs.scaled(0, 64)
    from dataclasses import replace
    cfg = replace(cfg, phi_deg=0.0)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d)
    ref = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy())
    tight(vol, ref, "phi = 0")


def test_repeat_calls_agree():
    cfg = inputs.config(0)
    d = inputs.projections(cfg)
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz)
    p = d["proj"].cuda()
    a = plan.backproject(p).clone()
    b = plan.backproject(p)
    torch.cuda.synchronize()
    assert rel(b.cpu().numpy(), a.cpu().numpy()) <= 2e-6
    plan.close()


def test_errors_do_not_cross_the_boundary():
    with pytest.raises(lam.LamError) as e:
        lam.Plan(60, 64, 64, [0.0, 1.0], 0.3)          # sigma*n not a power of two
    assert e.value.status == lam.LAM_EUNSUPPORTED
    with pytest.raises(lam.LamError) as e:
        lam.Plan(64, 64, 64, [0.0, 1.0], 2.0)          # phi out of range
    assert e.value.status == lam.LAM_EINVAL
    plan = lam.Plan(64, 64, 64, [0.0, 1.0], 0.3, input="u16")
    with pytest.raises(lam.LamError):                   # dark/flat missing
        plan.backproject(torch.zeros((2, 64, 64), dtype=torch.uint16, device="cuda"))
    plan.close()


@pytest.mark.parametrize("n,nz,h,w,nth", [(2048, 32, 64, 64, 6),      # sigma*n = 4096: three radix-16 passes
                                          (1024, 32, 2048, 64, 6),    # h = 2048: 512-thread column FFT
                                          (256, 512, 64, 2048, 6),    # w = 2048, sigma*nz = 1024
                                          (4096, 16, 32, 32, 4),      # sigma*n = 8192: four passes, 2 columns per block
                                          (256, 16, 4096, 32, 4)])    # h = 4096: 4 columns per block
def test_long_transform_lengths_against_exact_columns(n, nz, h, w, nth):
    """Every FFT length / block shape the full-size configs use, on thin problems the exact oracle can follow."""
    cfg = inputs.Config(f"fft{n}x{h}x{w}", n, nz, h, w, nth, 20.0, 12, min(nz / 4, h / 8), seed=5)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d)
    rng = np.random.default_rng(1)
    r = min(n // 4, w // 3)
    cols = (n // 2 + rng.integers(-r, r, size=(6, 2))).astype(np.int32)
    ref = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy(), cols=cols)
    got = np.stack([vol[:, c[1], c[0]] for c in cols])
    tight(got, ref, f"fft {n} {h} {w}")


def test_forward_against_exact_oracle():
    """lam_forward = L (Eq. 5) against the oracle's exact forward NUDFT O1 on a small volume."""
    n, nz, h, w, nth = 32, 32, 32, 32, 8
    rng = np.random.default_rng(3)
    zz, yy, xx = np.meshgrid(np.arange(nz) - nz / 2, np.arange(n) - n / 2, np.arange(n) - n / 2, indexing="ij")
    f = np.zeros((nz, n, n))
    for _ in range(6):
        c = rng.uniform(-6, 6, 3)
        s = rng.uniform(1.5, 3.0)
        f += rng.uniform(0.5, 1.0) * np.exp(-((xx - c[0]) ** 2 + (yy - c[1]) ** 2 + (zz - c[2]) ** 2) / (2 * s * s))
    theta = 2 * np.pi * np.arange(nth) / nth + 0.1
    phi = math.radians(20.0)
    plan = lam.Plan(n, h, w, theta, phi, nz=nz, filter="none")
    got = plan.forward(torch.from_numpy(f.astype(np.float32)).cuda()).cpu().numpy()
    plan.close()
    ref = O.forward_nudft(O.Geometry(n, h, w, theta, phi, nz=nz, filter="none"), f.astype(np.float32).astype(np.float64))
    tight(got, ref, "lam_forward")


@pytest.mark.parametrize("idx,n", [(2, 128), (4, 128)])
def test_adjoint_identity_on_the_gpu(idx, n):
    """<L f, d> = <f, L* d> for lam_forward / lam_backproject(filter = none): exact transposes stage by stage;
    SURVEY.md 8(c) gate 1e-5 in fp32 (dot products accumulated in fp64 on the host)."""
    cfg = inputs.scaled(idx, n)
    rng = np.random.default_rng(17)
    f = torch.from_numpy(rng.standard_normal((cfg.nz, cfg.n, cfg.n)).astype(np.float32)).cuda()
    d = torch.from_numpy(rng.standard_normal((cfg.ntheta, cfg.h, cfg.w)).astype(np.float32)).cuda()
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, cfg.theta(), cfg.phi, nz=cfg.nz, filter="none", plane_batch=7, theta_chunk=11)
    Lf = plan.forward(f)
    Ld = plan.backproject(d)
    torch.cuda.synchronize()
    plan.close()
    lhs = float((Lf.double() * d.double()).sum())
    rhs = float((f.double() * Ld.double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs), (lhs, rhs)


def test_zero_projections_give_an_exactly_zero_volume():
    cfg = inputs.scaled(2, 64)
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, cfg.theta(), cfg.phi, nz=cfg.nz)
    vol = plan.backproject(torch.zeros((cfg.ntheta, cfg.h, cfg.w), dtype=torch.float32, device="cuda"))
    torch.cuda.synchronize()
    plan.close()
    assert float(vol.abs().max()) == 0.0


@pytest.mark.parametrize("nth", [1, 3])
def test_very_few_angles(nth):
    """Degenerate scans: one or three projections (most gridding tiles are then empty)."""
    cfg = inputs.Config("few", 64, 32, 64, 64, nth, 20.0, 8, 4.0, seed=9)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d)
    ref = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy())
    tight(vol, ref, "few angles")


def test_arbitrary_unsorted_angles():
    """theta[] is any list (reading Q10): random, unsorted, with repeats; the job lists follow theta's order."""
    cfg = inputs.Config("rand", 64, 32, 64, 64, 40, 25.0, 8, 4.0, seed=10)
    rng = np.random.default_rng(4)
    theta = rng.uniform(-7.0, 7.0, size=cfg.ntheta)
    theta[5] = theta[17]
    d = inputs.projections(cfg, theta=theta)
    vol, _ = run_gpu(cfg, d)
    ref = O.fbp_nudft(geometry(cfg, d), d["proj"].numpy())
    tight(vol, ref, "unsorted angles")


def test_width4_kernel_runs_and_is_as_accurate_as_its_oracle_twin():
    """W = 4 (less accurate by design): the CUDA path must agree with the oracle's gridded path at the same W."""
    cfg = inputs.scaled(1, 64)
    d = inputs.projections(cfg)
    vol, _ = run_gpu(cfg, d, width=4)
    ref = O.fbp_gridded(geometry(cfg, d), d["proj"].numpy(), W=4)
    assert rel(vol, ref) <= 1e-4


def test_raw_counts_below_dark_are_clamped_like_the_oracle():
    """Reading Q12: transmission <= 0 is clamped to t_min before the logarithm."""
    cfg = inputs.scaled(3, 64)
    d = inputs.projections(cfg)
    raw = d["proj"].clone()
    raw[:, ::7, ::5] = 0          # counts below the dark field
    d = dict(d, proj=raw)
    vol, _ = run_gpu(cfg, d)
    ref = O.fbp_gridded(geometry(cfg, d), raw.numpy())
    tight_noisy(vol, ref, "clamped counts")


# ---------------------------------------------------------------------------------------------------------------------
# Full-band inputs: white noise puts energy into the out-of-band corners (periodic wrap, reading Q7) and into the
# Nyquist rows / columns (symmetric split, reading Q8), which smooth blobs leave almost empty.
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,phi_deg,filt", [(32, 37.0, "ramp"), (32, 40.0, "none"), (64, 35.0, "ramp")])
def test_white_noise_projections_against_exact_nudft(n, phi_deg, filt):
    nth = 24 if n == 32 else 16
    rng = np.random.default_rng(100 + n)
    theta = 2 * np.pi * np.arange(nth) / nth + 0.05
    phi = math.radians(phi_deg)
    proj = rng.standard_normal((nth, n, n)).astype(np.float32)
    plan = lam.Plan(n, n, n, theta, phi, filter=filt, plane_batch=5, theta_chunk=7)
    vol = plan.backproject(torch.from_numpy(proj).cuda())
    torch.cuda.synchronize()
    plan.close()
    geom = O.Geometry(n, n, n, theta, phi, filter=filt)
    if n == 32:
        ref = O.fbp_nudft(geom, proj)
        got = vol.cpu().numpy()
    else:
        cols = rng.integers(0, n, size=(96, 2)).astype(np.int32)
        ref = O.fbp_nudft(geom, proj, cols=cols)
        got = np.stack([vol[:, int(c[1]), int(c[0])].cpu().numpy() for c in cols])
    print(f"white noise n={n} phi={phi_deg} {filt}:", tight(got, ref, "white noise"))


def test_forward_of_a_white_noise_volume_against_exact_nudft():
    n, nz, nth = 32, 16, 10
    rng = np.random.default_rng(77)
    theta = 2 * np.pi * np.arange(nth) / nth + 0.2
    phi = math.radians(38.0)
    f = rng.standard_normal((nz, n, n)).astype(np.float32)
    plan = lam.Plan(n, n, n, theta, phi, nz=nz, filter="none")
    got = plan.forward(torch.from_numpy(f).cuda()).cpu().numpy()
    plan.close()
    ref = O.forward_nudft(O.Geometry(n, n, n, theta, phi, nz=nz, filter="none"), f.astype(np.float64))
    print("forward, white-noise volume:", tight(got, ref, "lam_forward white noise"))


@pytest.mark.parametrize("pinned", [True, False])
def test_host_pointers_pinned_and_pageable(pinned):
    """Host proj / vol (include/lam.h): several projection chunks in, several volume slabs out, same answer as the
    device-pointer call."""
    cfg = inputs.scaled(3, 128)
    d = inputs.projections(cfg)
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, input="u16", theta_chunk=9, plane_batch=6)
    plan.set_darkflat(d["dark"].cuda(), d["flat"].cuda())
    ref = plan.backproject(d["proj"].cuda()).cpu()
    hp = d["proj"].clone()
    hv = torch.zeros((cfg.nz, cfg.n, cfg.n), dtype=torch.float32)
    if pinned:
        hp, hv = hp.pin_memory(), hv.pin_memory()
    lam.lam_backproject(plan._plan, hp.data_ptr(), hv.data_ptr(), torch.cuda.current_stream().cuda_stream)
    # the call returns when the host volume is complete (header contract): no synchronisation here
    assert rel(hv.numpy(), ref.numpy()) <= 2e-6
    # mixed: host projections, device volume
    dv = torch.empty_like(ref, device="cuda")
    lam.lam_backproject(plan._plan, hp.data_ptr(), dv.data_ptr(), torch.cuda.current_stream().cuda_stream)
    hp.zero_()          # the call has consumed the host projections on return (header contract)
    torch.cuda.synchronize()
    assert rel(dv.cpu().numpy(), ref.numpy()) <= 2e-6
    assert plan.info()["out_of_core"] == 1
    plan.close()


@pytest.mark.parametrize("columns", [16, 8, 4])
def test_x3_stage_tma_and_plain_kernels_agree(columns):
    """The x3 stage has two forms (k_zstage_tma: persistent blocks fed by TMA, the default below sigma*nz = 2048, and the
    plain k_zstage, used by long transforms and by the spilled schedule), each with 16, 8 or 4 columns per block (the
    full-size configs use 16 / 8 / 4; the TMA form splits a cell's band over 1 / 2 / 4 lanes), chosen here through
    params.z_form / params.z_columns.  Same tables, same arithmetic up to the order of the partial sums: both against the
    oracle, and against each other at fp32 rounding."""
    cfg = inputs.scaled(2, 256)
    d = inputs.projections(cfg)
    vols = {}
    for mode, form in (("1", 2), ("0", 1)):
        plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample,
                        z_form=form, z_columns=columns)
        vols[mode] = plan.backproject(d["proj"].cuda()).cpu().numpy()
        plan.close()
    lcb = columns.bit_length() - 1
    ref = O.fbp_gridded(geometry(cfg, d), d["proj"].numpy())
    for mode, v in vols.items():
        print("x3 stage", "tma" if mode == "1" else "plain", 1 << lcb, "columns:", tight(v, ref, f"x3 stage mode {mode}"))
    assert np.abs(vols["1"] - vols["0"]).max() <= 2e-6 * np.abs(vols["0"]).max()
