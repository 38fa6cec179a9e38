#!/usr/bin/env python
"""bench.py — reconstructed GVoxel/s of lam_backproject (laminography FBP, Eq. 3 / :128 Eq. 7) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One "step" = one whole lam_backproject (S0..S4 of DESIGN.md) over one synthetic scan of the chosen config.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
  value     device-resident input and output, CUDA events on the launching stream, max over ranks
  e2e       the same call with HOST (pinned) buffers: H2D of the projections and D2H of the volume inside the timed region
  roofline  the dominant kernel group against its binding ceiling, plus `stages`: every stage against the HBM roofline
  cpu_baseline / --impl reference: the CPU fp64 oracle (oracle/), as it stands, on a bounded sample of the same workload
  all_configs  configs[2] and configs[4] (host-resident, PCIe inside) measured in the same run, with their stage tables
  next_rows    lam_forward, lam_backproject_slice and lam_admm_tv timed on configs[2]
N > 1: the path does not shard without an exchange step: N independent replicas, weak scaling.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "reconstructed GVoxel/s (laminography FBP, lam_backproject)"
UNIT = "GVoxel/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3,
                    help="index into BASELINE.json configs (default 3: the largest HBM-resident one, 2048x2048x512 from uint16)")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the all_configs block (configs[2], [4] measured beside the headline)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-full-config", type=int, default=-1,
                    help="also run oracle path C in full on this config (0..2; minutes of host time) into all_configs[...].cpu_baseline")
    ap.add_argument("--cpu-angles", type=int, default=0, help="angles in the oracle's sample (0: auto)")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = max([int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()] or [0])
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any(len(r) > 2 + i and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": reasons,
                "samples": len(sm)}


def stage_model(cfg):
    """ALGORITHMIC bytes / flops per step of each stage."""
    esz = 2 if cfg.raw16 else 4
    M, M3 = int(cfg.oversample * cfg.n), int(cfg.oversample * cfg.nz)
    NP = cfg.h // 2 + 1
    inp = cfg.ntheta * cfg.h * cfg.w * esz
    S = NP * cfg.ntheta * (cfg.w + 1) * 8
    G = NP * M * M * 8
    A = NP * cfg.n * cfg.n * 8
    vol = cfg.voxels * 4
    samples = NP * cfg.ntheta * (cfg.w + 1)
    W = cfg.width
    return {
        "s1_prep_filter_fft2d": {"bytes": inp + S},
        "s2_gridding_xy": {"bytes": S + G, "flops": samples * (4 * W * W + 2 * W)},
        "s3_ifft_xy": {"bytes": G + A},
        "s4_z_grid_ifft_deapodise": {"bytes": A + vol},
    }


# SURVEY.md section 8(d) "Which roofline binds": ALGORITHMIC GB per step on the Hermitian-half 3-D grid (S3 there is the
# whole pruned three-pass transform, S4 the deapodise pass; here the x3 pass lives in stage 4, so S3 + S4 are given as one
# figure).  The factored method of Eq. 9 grids (h/2+1) planes of M^2 cells where the 3-D grid has sigma*nz/2: its own
# work is what stage_model() counts; the survey's figure is printed beside it so both fractions are in the line.
SURVEY_GB = {2: {"s1": 10.1, "s2": 13.6, "s3_s4": 22.5 + 2.1, "step": 48.4},
             3: {"s1": 45.3, "s2": 98.9, "s3_s4": 180.0 + 17.2, "step": 342.0},
             4: {"s1": 151.0, "s2": 650.0, "s3_s4": 1443.0 + 137.0, "step": 2382.0}}


def survey_report(idx, stage, ms_step, hbm):
    """Per-stage and whole-step HBM fractions on SURVEY.md 8(d)'s byte counts (None for configs it does not tabulate)."""
    g = SURVEY_GB.get(idx)
    if g is None:
        return None
    f = lambda gb, ms: round(gb / (ms * 1e-3) / hbm, 4) if ms > 0 else None
    return {"algorithmic_GB_survey": g,
            "hbm_frac_survey": {"s1": f(g["s1"], stage[0]), "s2": f(g["s2"], stage[1]), "s3_s4": f(g["s3_s4"], stage[2] + stage[3]),
                                "step": f(g["step"], ms_step)}}


def cpu_sample(cfg, nangles=None, slab=4, mult=3):
    """The oracle as it stands, path C (the double-precision gridded USFFT of PAPER.md:130-142: 3-D gridding with
    W^3 taps per sample, 3-D inverse FFT, deapodisation), on a BOUNDED sample of the config: the full detector and the
    full lateral grid, but a slab of `slab` x3-slices and `nangles` / mult*`nangles` of the scan's angles.
    Every sample still spreads its W^3 taps (the thin fine grid is periodic in xi3), so the per-angle cost is the
    whole job's; the fixed cost (3-D inverse FFT + deapodisation of M x M x sigma*slab cells) grows with the slab as
    nz/slab * log2(M M sigma nz)/log2(M M sigma slab).  Whole job = ntheta * t_angle + t_fix(nz), extrapolated."""
    import math
    from dataclasses import replace
    import numpy as np
    from oracle import lam_oracle as O
    from paper_2401_11101_b200 import inputs
    if nangles is None:
        nangles = max(1, min(cfg.ntheta // (2 * mult), int(round(8 * (1024 * 1024) / (cfg.h * cfg.w)))))
    times, used = [], []
    for na in (nangles, mult * nangles):
        idx = np.linspace(0, cfg.ntheta - 1, na).astype(int)
        d = inputs.projections(cfg, device="cpu", theta=cfg.theta()[idx])
        proj = d["proj"].contiguous().numpy()
        g = O.Geometry(cfg.n, cfg.h, cfg.w, cfg.theta()[idx], cfg.phi, nz=slab,
                       dark=None if d["dark"] is None else d["dark"].numpy(), flat=None if d["flat"] is None else d["flat"].numpy())
        t0 = time.perf_counter()
        O.fbp_gridded(g, proj, W=cfg.width, sigma=cfg.oversample)
        times.append(time.perf_counter() - t0)
        used.append(na)
        if len(used) == 1:
            g_b, proj_b = g, proj
    # path B (direct "Linerec" discretisation, O(N^4)): the same slab and the smaller angle subset (its row filter
    # is a space-domain convolution, w^2 per row); its cost is
    # proportional to voxels x angles, so the whole job is the sample's time scaled by (nz / slab) (ntheta / angles)
    t0 = time.perf_counter()
    O.fbp_direct(g_b, proj_b)
    t_b = time.perf_counter() - t0
    path_b = {"seconds": round(t_b, 2), "whole_job_seconds_extrapolated": round(t_b * (cfg.nz / slab) * (cfg.ntheta / used[0]), 1),
              "value": cfg.voxels / (t_b * (cfg.nz / slab) * (cfg.ntheta / used[0])) / 1e9,
              "sample": f"oracle path B (direct back-projection with linear interpolation) on the same slab, {used[0]} angles"}
    t_angle = max(1e-9, (times[1] - times[0]) / (used[1] - used[0]))
    t_fix = max(0.0, times[0] - used[0] * t_angle)
    M = cfg.oversample * cfg.n
    grow = (cfg.nz / slab) * math.log2(M * M * cfg.oversample * cfg.nz) / math.log2(M * M * cfg.oversample * slab)
    total = cfg.ntheta * t_angle + t_fix * grow
    return {"seconds": sum(times) + t_b, "value": cfg.voxels / total / 1e9, "cores": O.threads(), "path_b": path_b,
            "whole_job_seconds_extrapolated": total,
            "sample": f"oracle path C (fp64 3-D gridded USFFT, W^3 taps per sample) on the full {cfg.h}x{cfg.w} detector and "
                      f"{cfg.n}x{cfg.n} lateral grid, a slab of {slab} of {cfg.nz} x3-slices, {used[0]} and {used[1]} of "
                      f"{cfg.ntheta} angles: t_angle={t_angle:.3f}s, t_fix(slab)={t_fix:.2f}s; whole job = ntheta*t_angle + "
                      f"t_fix*{grow:.1f} (extrapolated)"}


def cpu_full_path_c(idx, device="cpu"):
    """Oracle path C IN FULL on one config (no sampling, no extrapolation): SURVEY.md 8(d) names it for configs[0]-[2]
    (the fp64 fine grid of configs[2] is 34 GB).  Minutes of host time, so bench.py runs it only with --cpu-full-config."""
    from oracle import lam_oracle as O
    from paper_2401_11101_b200 import inputs
    cfg = inputs.config(idx)
    d = inputs.projections(cfg, device=device)
    proj = d["proj"].cpu().contiguous().numpy()
    g = O.Geometry(cfg.n, cfg.h, cfg.w, cfg.theta(), cfg.phi, nz=cfg.nz,
                   dark=None if d["dark"] is None else d["dark"].cpu().numpy(), flat=None if d["flat"] is None else d["flat"].cpu().numpy())
    del d
    t0 = time.perf_counter()
    O.fbp_gridded(g, proj, W=cfg.width, sigma=cfg.oversample)
    dt = time.perf_counter() - t0
    return {"value": float(f"{cfg.voxels / dt / 1e9:.6g}"), "unit": UNIT, "cores": O.threads(), "kind": "oracle",
            "seconds": round(dt, 1), "sample": f"oracle path C in full on configs[{idx}] {cfg.name} (all {cfg.ntheta} angles, whole volume): measured, not extrapolated"}


def max_over_ranks(ms, world, device):
    """Replicas: the job's time is the slowest rank's (MAX all-reduce; identity at world = 1)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gvoxels(world, voxels_per_rank, ms_step):
    """N independent scans (one per rank, weak scaling) finished in ms_step: aggregate GVoxel/s."""
    return world * voxels_per_rank / (ms_step * 1e-3) / 1e9


def measure(idx, steps, warmup, world, barrier, want_e2e=True, want_overlap=False):
    """One config: plan, K timed whole back-projections, per-stage times, optional end-to-end (host buffers) leg."""
    import statistics
    import torch
    from paper_2401_11101_b200 import inputs, lam
    cfg = inputs.config(idx)
    hostmode = cfg.out_of_core  # configs[4]: input + output + workspace exceed HBM; projections and volume live in pinned host memory
    if hostmode:
        out = torch.empty((cfg.ntheta, cfg.h, cfg.w), dtype=torch.uint16 if cfg.raw16 else torch.float32, pin_memory=True)
        d = inputs.projections(cfg, device="cuda", out=out)
    else:
        d = inputs.projections(cfg, device="cuda")
    proj = d["proj"]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample,
                    input="u16" if cfg.raw16 else "f32")
    torch.cuda.synchronize()
    plan_ms = (time.perf_counter() - t0) * 1e3
    if cfg.raw16:
        plan.set_darkflat(d["dark"], d["flat"])
    vol = (torch.empty((cfg.nz, cfg.n, cfg.n), dtype=torch.float32, pin_memory=True) if hostmode else
           torch.empty((cfg.nz, cfg.n, cfg.n), dtype=torch.float32, device="cuda"))
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        plan.backproject(proj, vol)
    barrier()
    # ---- timed region: K whole back-projections, CUDA events on the launching stream (one pair brackets all K; one
    # event between calls gives the per-call times for the median)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for i in range(steps):
        plan.backproject(proj, vol)
        ev[i + 1].record(stream)
    barrier()
    ms_total = ev[0].elapsed_time(ev[steps])
    per_call = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
    launches = plan.info()["launches"] * steps
    # ---- per-stage device times, live, over K further calls (events inside the plan; not the headline number)
    plan.set_profiling(True)
    stage = [0.0] * 6
    for _ in range(steps):
        plan.backproject(proj, vol)
        stage = [a + b for a, b in zip(stage, plan.stage_ms())]
    plan.set_profiling(False)
    stage = [x / steps for x in stage]
    res = {"cfg": cfg, "ms_total": ms_total, "per_call": per_call, "median_ms": statistics.median(per_call),
           "stage": stage, "launches": launches, "plan_ms": plan_ms, "info": plan.info(), "hostmode": hostmode,
           "proj_bytes": proj.numel() * proj.element_size(), "e2e": None, "overlap": None}
    # ---- e2e: the same call with host (pinned) buffers; H2D + D2H inside the timed region
    if want_e2e and not hostmode:
        hproj = torch.empty(proj.shape, dtype=proj.dtype, pin_memory=True)
        hproj.copy_(proj)
        hvol = torch.empty(vol.shape, dtype=torch.float32, pin_memory=True)
        for _ in range(2):
            lam.lam_backproject(plan._plan, hproj.data_ptr(), hvol.data_ptr(), stream.cuda_stream)
        barrier()
        ksteps = max(1, min(steps, 5))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(ksteps):
            lam.lam_backproject(plan._plan, hproj.data_ptr(), hvol.data_ptr(), stream.cuda_stream)
        e1.record(stream)
        barrier()
        wall = (time.perf_counter() - t0) * 1e3
        ems = max(e0.elapsed_time(e1), wall if world == 1 else 0.0) / ksteps
        err = float((hvol.cuda() - vol).norm() / vol.norm())
        res["e2e"] = {"ms": ems, "steps": ksteps, "h2d": hproj.numel() * hproj.element_size(), "d2h": hvol.numel() * 4, "err": err}
        del hproj, hvol
    if hostmode:
        res["e2e"] = {"ms": ms_total / steps, "steps": steps, "h2d": res["proj_bytes"], "d2h": vol.numel() * 4, "err": None}
    if want_overlap and hostmode:
        # t_total (host -> host call), t_copy_only (the same chunked copies on two copy streams, no
        # kernels), t_compute_only (the device stages of the profiled call), overlap ratio
        # copy-only: the library's own copies (same chunks, slabs, streams and events), kernels skipped
        lam.lam_set_profiling(plan._plan, 2)
        plan.backproject(proj, vol)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(2):
            plan.backproject(proj, vol)
        torch.cuda.synchronize()
        t_copy = (time.perf_counter() - t0) * 1e3 / 2
        lam.lam_set_profiling(plan._plan, 0)
        t_compute = sum(stage[:4])
        t_total = ms_total / steps
        res["overlap"] = {"t_total_ms": round(t_total, 2), "t_copy_only_ms": round(t_copy, 2),
                          "t_compute_only_ms": round(t_compute, 2),
                          "overlap_ratio": round((t_copy + t_compute - t_total) / min(t_copy, t_compute), 4),
                          "note": "copy-only: the same call with every kernel skipped (lam_set_profiling(plan, 2)); "
                                  "compute-only: sum of the device stages of the profiled host-buffer call"}
    plan.close()
    del plan, proj, vol, d
    torch.cuda.empty_cache()
    return res


def measure_next_rows(idx, reps=3):
    """SURVEY.md 8(f) rows timed on one config (fp32 input): lam_forward, one lam_backproject_slice centre, one CG step of
    lam_admm_tv.  CUDA events on the launching stream; not part of `value`."""
    import torch
    from paper_2401_11101_b200 import inputs, lam
    cfg = inputs.config(idx)
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, cfg.theta(), cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample, filter="none")
    vol = torch.rand((cfg.nz, cfg.n, cfg.n), device="cuda")
    proj = torch.empty((cfg.ntheta, cfg.h, cfg.w), device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn, k):
        fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(k):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / k

    out = {"workload": f"{cfg.name}: volume {cfg.n}x{cfg.n}x{cfg.nz}, {cfg.ntheta} angles, detector {cfg.h}x{cfg.w} fp32"}
    t = timed(lambda: plan.forward(vol, proj), reps)
    # correctness beside the timing: <L f, d> = <f, L* d> on this very plan (L* = lam_backproject, filter none, whose
    # columns the tests compare with the exact oracle at this size)
    dd = torch.randn((cfg.ntheta, cfg.h, cfg.w), device="cuda")
    ltd = plan.backproject(dd)
    a, b = float((proj.double() * dd.double()).sum()), float((vol.double() * ltd.double()).sum())
    out["lam_forward"] = {"ms": round(t, 3), "GVoxel_per_s": round(cfg.voxels / t / 1e6, 3),
                          "adjoint_identity_rel": float(f"{abs(a - b) / float(proj.double().norm() * dd.double().norm()):.3e}")}
    centers = [cfg.w / 2 - 1.0, cfg.w / 2, cfg.w / 2 + 1.0]
    sl = torch.empty((3, cfg.n, cfg.n), device="cuda")
    t3 = timed(lambda: plan.backproject_slice(proj, cfg.nz // 2, centers, sl), 1)
    t1 = timed(lambda: plan.backproject_slice(proj, cfg.nz // 2, centers[:1], sl[:1]), 1)
    plan.backproject_slice(proj, cfg.nz // 2, None, sl[:1])
    plan.backproject(proj, ltd)
    ref = ltd[cfg.nz // 2]
    out["lam_backproject_slice"] = {"ms_first_centre": round(t1, 3), "ms_per_further_centre": round((t3 - t1) / 2, 3),
                                    "slice_vs_full_volume_rel_l2": float(f"{float((sl[0] - ref).norm() / ref.norm()):.3e}")}
    del dd, ltd
    # one CG step = one lam_forward + one lam_backproject + TV kernels and reductions: warm-up call first (it allocates
    # the workspace), then the difference of a 4-step and a 2-step call, each timed with CUDA events
    plan.admm_tv(proj, 0.1, 1.0, 1, 1, vol)
    hist = []
    t2 = timed(lambda: hist.append(plan.admm_tv(proj, 0.1, 1.0, 1, 2, vol)[1]), 1)
    t4 = timed(lambda: hist.append(plan.admm_tv(proj, 0.1, 1.0, 1, 4, vol)[1]), 1)
    out["lam_admm_tv"] = {"ms_per_cg_step": round((t4 - t2) / 2, 3), "ms_2_steps": round(t2, 3), "ms_4_steps": round(t4, 3),
                          "gradF_norm_after_each_step": [float(f"{x:.4e}") for x in hist[-1]],
                          "note": "one lam_forward + one lam_backproject + TV kernels and reductions per step"}
    plan.close()
    del vol, proj, sl
    torch.cuda.empty_cache()
    return out


def stage_report(cfg, stage, hbm):
    model = stage_model(cfg)
    out = {}
    for i, nm in enumerate(model.keys()):
        gbs = model[nm]["bytes"] / (stage[i] * 1e-3) / 1e9 if stage[i] > 0 else None
        out[nm] = {"ms": round(stage[i], 4), "algorithmic_GB": round(model[nm]["bytes"] / 1e9, 4),
                   "achieved_GBs": round(gbs, 1) if gbs else None, "hbm_frac": round(gbs / hbm, 4) if gbs else None}
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2401_11101_b200 import inputs, lam

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warmup = max(args.warmup, 3)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    r = measure(args.config, args.steps, warmup, world, barrier, want_e2e=not args.no_e2e, want_overlap=True)
    clocks = sampler.stop() if rank == 0 else None
    cfg = r["cfg"]
    ms = max_over_ranks(r["ms_total"], world, "cuda")
    ms_step = ms / args.steps
    value = whole_job_gvoxels(world, cfg.voxels, ms_step)
    stage = r["stage"]
    e2e = None
    if r["e2e"] is not None:
        ems = max_over_ranks(r["e2e"]["ms"], world, "cuda")
        e2e = {"value": whole_job_gvoxels(world, cfg.voxels, ems), "unit": UNIT, "ms_per_step": round(ems, 3),
               "steps": r["e2e"]["steps"], "h2d_bytes_per_step": r["e2e"]["h2d"], "d2h_bytes_per_step": r["e2e"]["d2h"]}
        if r["e2e"]["err"] is not None:
            e2e["host_vs_device_result_rel_l2"] = r["e2e"]["err"]
        if r["hostmode"]:
            e2e["note"] = "configs[4] does not fit HBM: value and e2e are the same host-buffer run"
    # ---- the other single-GPU configs, measured in the same run (rank 0 of a 1-GPU run only): fewer calls
    others = {}
    if world == 1 and not args.no_all_configs:
        free, _ = torch.cuda.mem_get_info()
        for idx in (2, 3, 4):
            if idx == args.config:
                continue
            c = inputs.config(idx)
            try:
                if idx == 4:
                    import psutil
                    if free < 150e9 or psutil.virtual_memory().available < c.ntheta * c.h * c.w * 2 + c.voxels * 4 + 30e9:
                        others[f"configs[{idx}]"] = {"skipped": "needs ~145 GB of device and ~135 GB of pinned host memory"}
                        continue
                k = 3 if idx == 4 else min(args.steps, 5)
                o = measure(idx, k, 3 if idx != 4 else 2, world, barrier, want_e2e=False, want_overlap=True)
                hbm, _ = peaks()
                oms = o["ms_total"] / k
                others[f"configs[{idx}]"] = {
                    "workload": f"{c.name}: volume {c.n}x{c.n}x{c.nz}, {c.ntheta} angles, detector {c.h}x{c.w} "
                                f"{'uint16 raw + dark/flat' if c.raw16 else 'fp32'}" + (", host-resident buffers (PCIe inside)" if o["hostmode"] else ""),
                    "value": round(c.voxels / (oms * 1e-3) / 1e9, 4), "unit": UNIT, "ms_per_step": round(oms, 3),
                    "ms_per_step_median": round(o["median_ms"], 3), "steps": k, "warmup": 3 if idx != 4 else 2,
                    "plan_ms": round(o["plan_ms"], 1), "stages": stage_report(c, o["stage"], hbm),
                    "copies_ms": round(o["stage"][4], 2), "overlap": o["overlap"], "plan": o["info"]}
                sv = survey_report(idx, o["stage"], oms, hbm)
                if sv:
                    others[f"configs[{idx}]"].update(sv)
            except Exception as e:  # a config that does not fit this box must not void the headline line
                others[f"configs[{idx}]"] = {"error": str(e)[:200]}
                torch.cuda.empty_cache()
    next_rows = None
    if world == 1 and not args.no_all_configs:
        try:
            next_rows = measure_next_rows(2)
        except Exception as e:
            next_rows = {"error": str(e)[:200]}
            torch.cuda.empty_cache()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- rooflines
    hbm, src = peaks()
    model = stage_model(cfg)
    names = list(model.keys())
    stages = stage_report(cfg, stage, hbm)
    dom = max(range(4), key=lambda i: stage[i])
    ach = model[names[dom]]["bytes"] / (stage[dom] * 1e-3) / 1e9
    roof = {"kernel": "k_spread (+k_zero_tiles)" if names[dom] == "s2_gridding_xy" else names[dom], "stage": names[dom],
            "bound": "hbm", "achieved": round(ach, 1), "peak": hbm, "unit": "GB/s", "frac": round(ach / hbm, 4),
            "traffic": None, "peak_source": src}
    if names[dom] == "s2_gridding_xy":
        # With the factored gridding of Eq. 9 (W^2 = 36 taps per sample instead of W^3 = 216) the fp32-ALU floor of S2
        # (samples x 36 taps x 3 lane-instr / 3.72e13 per s) lies BELOW its HBM floor, so HBM is the binding roofline and
        # `frac` is taken against it.  What the kernel actually saturates is the shared-memory (LSU) data pipe
        # (DESIGN.md section 5); the ALU and LSU-pipe figures are kept here as context.
        samples = model[names[dom]]["flops"] / (4 * cfg.width * cfg.width + 2 * cfg.width)
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
        alu_ach = model[names[dom]]["flops"] / (stage[dom] * 1e-3) / 1e12
        lsu_floor_ms = samples * cfg.width * cfg.width * 16 / (148 * 128 * 1.965e9) * 1e3
        roof["alu"] = {"achieved_TFLOPs": round(alu_ach, 3), "peak_TFLOPs": round(alu_peak, 2), "frac": round(alu_ach / alu_peak, 4),
                       "floor_ms": round(samples * cfg.width * cfg.width * 3 / (148 * 128 * 1.965e9) * 1e3, 2),
                       "peak_source": "derived: 148 SM x 128 fp32 lanes x 2 flop x 1.965 GHz"}
        roof["lsu_pipe"] = {"floor_ms": round(lsu_floor_ms, 2), "frac": round(lsu_floor_ms / stage[dom], 4),
                            "note": "samples x W^2 taps x 16 B of shared-memory read-modify-write at 128 B/clk/SM"}
        roof["hbm_floor_ms"] = round(model[names[dom]]["bytes"] / hbm / 1e6, 2)
    # traffic: dram bytes per launch of the dominant kernel from a committed ncu --set full capture, used only when that
    # capture was taken on THIS build and THIS launch shape (library version, config, plane batch); otherwise null
    try:
        import csv
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "r03_traffic.csv"))):
            if (int(row["config"]) == args.config and row["stage"] == names[dom] and row["lib_version"] == lam.lam_version()
                    and int(row["plane_batch"]) == r["info"]["plane_batch"]):
                roof["traffic"] = float(row["dram_bytes_per_launch"])
                roof["traffic_source"] = row["source"]
    except Exception:
        pass
    roof["stages"] = stages
    roof["share_of_step"] = round(stage[dom] / max(1e-9, sum(stage[:4])), 4)
    total_bytes = sum(m["bytes"] for m in model.values())
    roof["whole_step_hbm_frac"] = round(total_bytes / (ms_step * 1e-3) / 1e9 / hbm, 4)
    roof["whole_step_algorithmic_GB"] = round(total_bytes / 1e9, 2)
    sv = survey_report(args.config, stage, ms_step, hbm)
    if sv:
        roof.update(sv)
    out = {"metric": METRIC, "value": round(value, 4), "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": warmup, "ms_per_step": round(ms_step, 4), "ms_per_step_median": round(r["median_ms"], 4),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"configs[{args.config}] {cfg.name}: volume {cfg.n}x{cfg.n}x{cfg.nz} fp32, "
                                  f"{cfg.ntheta} angles, phi={cfg.phi_deg} deg, detector {cfg.h}x{cfg.w} "
                                  f"{'uint16 raw + dark/flat' if cfg.raw16 else 'fp32'}, KB W={cfg.width} sigma={cfg.oversample}",
                      "l2": "inputs larger than L2 (projections %.2f GB, spectra + fine grid %.2f GB per step)" % (
                          r["proj_bytes"] / 1e9, model["s2_gridding_xy"]["bytes"] / 1e9),
                      "parallelism": "replicas only" if world > 1 else "single GPU",
                      "plan": r["info"], "plan_ms": round(r["plan_ms"], 1), "lib": lam.lam_version()},
           "clocks": clocks, "e2e": e2e, "gpu_launches": r["launches"], "roofline": roof}
    if r["overlap"]:
        out["overlap"] = r["overlap"]
    if others:
        out["all_configs"] = others
    if next_rows:
        out["next_rows"] = next_rows
    if 0 <= args.cpu_full_config <= 2:
        torch.cuda.empty_cache()
        out.setdefault("all_configs", {}).setdefault(f"configs[{args.cpu_full_config}]", {})["cpu_baseline"] = cpu_full_path_c(args.cpu_full_config, "cuda")
    if not args.no_cpu_baseline:
        cb = cpu_sample(cfg)
        out["cpu_baseline"] = {"value": float(f"{cb['value']:.6g}"), "unit": UNIT, "cores": cb["cores"], "kind": "oracle",
                               "sample": cb["sample"], "seconds": round(cb["seconds"], 2),
                               "path_b": {k: (float(f"{v:.6g}") if isinstance(v, float) else v) for k, v in cb["path_b"].items()}}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_reference(args):
    """The reference arm of this tier = the CPU oracle, as it stands, on the host cores (rank 0 only).
    One step = one bounded sample (cpu_sample: path C on a thin slab at two angle counts); the step's value is the
    whole-job throughput the sample's two cost terms give."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import lam_oracle as O
    from paper_2401_11101_b200 import inputs
    cfg = inputs.config(args.config)
    vals, secs, last = [], [], None
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        # 13 samples at the default --steps 10 --warmup 3: one and two angles on a 2-slice slab keep a step near 10 s
        last = cpu_sample(cfg, nangles=args.cpu_angles or 1, slab=2, mult=2)
        if it >= args.warmup:
            vals.append(last["value"])
            secs.append(time.perf_counter() - t0)
    value = len(vals) / sum(1.0 / v for v in vals)
    out = {"impl": "reference", "metric": METRIC, "value": float(f"{value:.6g}"), "unit": UNIT,
           "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": round(1e3 * sum(secs) / len(secs), 2), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"configs[{args.config}] {cfg.name} (bounded sample per step, see cpu_baseline.sample)"},
           "cpu_baseline": {"value": float(f"{value:.6g}"), "unit": UNIT, "cores": O.threads(), "kind": "oracle",
                            "sample": last["sample"]},
           "e2e": {"value": float(f"{value:.6g}"), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
