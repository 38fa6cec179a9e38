#!/usr/bin/env python
"""bench.py — reconstructed GVoxel/s of lam_backproject (laminography FBP, Eq. 3 / :128 Eq. 7) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One "step" = one whole lam_backproject (S0..S4 of DESIGN.md) over one synthetic scan of the chosen config.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
  value     device-resident input and output, CUDA events on the launching stream, max over ranks
  e2e       the same call with HOST (pinned) buffers: H2D of the projections and D2H of the volume inside the timed region
  roofline  the dominant kernel group against its binding ceiling, plus `stages`: every stage against the HBM roofline
  cpu_baseline / --impl reference: the CPU fp64 oracle (oracle/), as it stands, on a bounded sample of the same workload
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
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2: slab 1024x1024x256)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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


def cpu_sample(cfg, d, nangles, nslices=1, theta=None, mult=3):
    """The oracle as it stands (path C': exact x3 transform + double-precision 2-D gridding, Eq. 9)
    on one x3-slice, timed with `nangles` and with mult*`nangles` of the scan's angles.  A slice costs
    t(na) = t_fix + na * t_angle (t_fix: the 2-D inverse FFT of the fine grid and the crop; t_angle: 2-D FFT + gridding of
    one projection), so the two timings give both terms and the whole job is nz * (t_fix + ntheta * t_angle)."""
    import numpy as np
    from oracle import lam_oracle as O
    dark = d["dark"].cpu().numpy() if d["dark"] is not None else None
    flat = d["flat"].cpu().numpy() if d["flat"] is not None else None
    th_all = np.asarray(d["theta"] if theta is None else theta)
    nav = len(th_all)
    times, used = [], []
    for na in (nangles, mult * nangles):
        na = max(1, min(nav, na))
        idx = np.linspace(0, nav - 1, na).astype(int)
        proj = d["proj"][idx].cpu().contiguous().numpy()
        g = O.Geometry(cfg.n, cfg.h, cfg.w, th_all[idx], cfg.phi, nz=cfg.nz, dark=dark, flat=flat)
        t0 = time.perf_counter()
        for s in range(nslices):
            O.fbp_gridded_slice(g, proj, cfg.nz // 2 + s, W=cfg.width, sigma=cfg.oversample)
        times.append((time.perf_counter() - t0) / nslices)
        used.append(na)
    if used[1] > used[0]:
        t_angle = max(0.0, (times[1] - times[0]) / (used[1] - used[0]))
        t_fix = max(0.0, times[0] - used[0] * t_angle)
    else:
        t_angle, t_fix = times[0] / used[0], 0.0
    total = cfg.nz * (t_fix + cfg.ntheta * t_angle)
    return {"seconds": sum(times) * nslices, "value": cfg.voxels / total / 1e9, "cores": O.threads(),
            "whole_job_seconds_extrapolated": total,
            "sample": f"1 of {cfg.nz} x3-slices through oracle path C' (fp64 exact-x3 + 2-D gridded USFFT) with {used[0]} and "
                      f"{used[1]} of {cfg.ntheta} angles; per-slice cost t_fix={t_fix:.3f}s + {t_angle:.4f}s/angle, "
                      f"whole job = nz*(t_fix + ntheta*t_angle) extrapolated"}


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
    cfg = inputs.config(args.config)
    hostmode = cfg.out_of_core  # configs[4]: input + workspace exceed HBM; projections and volume live in pinned host memory
    if hostmode:
        out = torch.empty((cfg.ntheta, cfg.h, cfg.w), dtype=torch.uint16 if cfg.raw16 else torch.float32, pin_memory=True)
        d = inputs.projections(cfg, device="cuda", out=out)
    else:
        d = inputs.projections(cfg, device="cuda")
    proj = d["proj"]
    plan = lam.Plan(cfg.n, cfg.h, cfg.w, d["theta"], cfg.phi, nz=cfg.nz, width=cfg.width, oversample=cfg.oversample,
                    input="u16" if cfg.raw16 else "f32")
    if cfg.raw16:
        plan.set_darkflat(d["dark"], d["flat"])
    vol = (torch.empty((cfg.nz, cfg.n, cfg.n), dtype=torch.float32, pin_memory=True) if hostmode else
           torch.empty((cfg.nz, cfg.n, cfg.n), dtype=torch.float32, device="cuda"))
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        plan.backproject(proj, vol)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    # ---- timed region: K whole back-projections, device-resident input/output, CUDA events on the launching stream
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        plan.backproject(proj, vol)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = plan.info()["launches"] * args.steps
    # ---- per-stage device times, live, over the same K steps again (events inside the plan; not the headline number)
    plan.set_profiling(True)
    stage = [0.0] * 6
    for _ in range(args.steps):
        plan.backproject(proj, vol)
        stage = [a + b for a, b in zip(stage, plan.stage_ms())]
    plan.set_profiling(False)
    stage = [s / args.steps for s in stage]
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(ms, world, "cuda")
    ms_step = ms / args.steps
    value = whole_job_gvoxels(world, cfg.voxels, ms_step)

    # ---- e2e: the same call with host (pinned) buffers; H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e and not hostmode:
        hproj = torch.empty(proj.shape, dtype=proj.dtype, pin_memory=True)
        hproj.copy_(proj)
        hvol = torch.empty(vol.shape, dtype=torch.float32, pin_memory=True)
        for _ in range(2):
            lam.lam_backproject(plan._plan, hproj.data_ptr(), hvol.data_ptr(), stream.cuda_stream)
        barrier()
        ksteps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(ksteps):
            lam.lam_backproject(plan._plan, hproj.data_ptr(), hvol.data_ptr(), stream.cuda_stream)
        e1.record(stream)
        barrier()
        wall = (time.perf_counter() - t0) * 1e3
        ems = max(e0.elapsed_time(e1), wall if world == 1 else 0.0)
        ems = max_over_ranks(ems, world, "cuda") / ksteps
        err = float((hvol.cuda() - vol).norm() / vol.norm())
        e2e = {"value": whole_job_gvoxels(world, cfg.voxels, ems), "unit": UNIT, "ms_per_step": ems, "steps": ksteps,
               "h2d_bytes_per_step": hproj.numel() * hproj.element_size(),
               "d2h_bytes_per_step": hvol.numel() * 4, "host_vs_device_result_rel_l2": err}
        del hproj, hvol
    if hostmode:  # the timed call above already ran host -> host
        e2e = {"value": value, "unit": UNIT, "ms_per_step": ms_step, "steps": args.steps,
               "h2d_bytes_per_step": proj.numel() * proj.element_size(), "d2h_bytes_per_step": vol.numel() * 4,
               "note": "configs[4] does not fit HBM: value and e2e are the same host-buffer run"}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- rooflines
    hbm, src = peaks()
    model = stage_model(cfg)
    names = list(model.keys())
    stages = {}
    for i, nm in enumerate(names):
        gbs = model[nm]["bytes"] / (stage[i] * 1e-3) / 1e9 if stage[i] > 0 else None
        stages[nm] = {"ms": round(stage[i], 4), "algorithmic_GB": round(model[nm]["bytes"] / 1e9, 4),
                      "achieved_GBs": round(gbs, 1) if gbs else None, "hbm_frac": round(gbs / hbm, 4) if gbs else None}
    dom = max(range(4), key=lambda i: stage[i])
    if names[dom] == "s2_gridding_xy":
        peak = 148 * 128 * 2 * 1.965e9 / 1e12   # fp32 FMA lanes x 2 flop x max SM clock
        ach = model[names[dom]]["flops"] / (stage[dom] * 1e-3) / 1e12
        roof = {"kernel": "k_spread (+k_zero_tiles)", "stage": names[dom], "bound": "alu", "achieved": round(ach, 3),
                "peak": round(peak, 2), "unit": "TFLOP/s", "frac": round(ach / peak, 4), "traffic": None,
                "peak_source": "derived: 148 SM x 128 fp32 lanes x 2 flop x 1.965 GHz"}
    else:
        ach = model[names[dom]]["bytes"] / (stage[dom] * 1e-3) / 1e9
        roof = {"kernel": names[dom], "stage": names[dom], "bound": "hbm", "achieved": round(ach, 1), "peak": hbm,
                "unit": "GB/s", "frac": round(ach / hbm, 4), "traffic": None, "peak_source": src}
    # traffic: dram bytes per launch of the dominant kernel from the committed ncu --set full capture (profiles/), if any
    try:
        import csv
        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "r01_traffic.csv"))):
            if int(row["config"]) == args.config and row["stage"] == names[dom]:
                roof["traffic"] = float(row["dram_bytes_per_launch"])
                roof["traffic_note"] = row["source"]
                if row.get("issue_active_pct"):  # what binds the kernel under ncu: issue slots and the shared-memory pipe
                    roof["ncu_issue_active_pct"] = float(row["issue_active_pct"])
                    roof["ncu_l1tex_throughput_pct"] = float(row["l1tex_throughput_pct"])
    except Exception:
        pass
    roof["stages"] = stages
    roof["share_of_step"] = round(stage[dom] / max(1e-9, sum(stage[:4])), 4)
    total_bytes = sum(m["bytes"] for m in model.values())
    roof["whole_step_hbm_frac"] = round(total_bytes / (ms_step * 1e-3) / 1e9 / hbm, 4)
    out = {"metric": METRIC, "value": round(value, 4), "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": round(ms_step, 4), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"configs[{args.config}] {cfg.name}: volume {cfg.n}x{cfg.n}x{cfg.nz} fp32, "
                                  f"{cfg.ntheta} angles, phi={cfg.phi_deg} deg, detector {cfg.h}x{cfg.w} "
                                  f"{'uint16 raw + dark/flat' if cfg.raw16 else 'fp32'}, KB W={cfg.width} sigma={cfg.oversample}",
                      "l2": "inputs larger than L2 (projections %.2f GB, spectra %.2f GB per step)" % (
                          proj.numel() * proj.element_size() / 1e9, model["s2_gridding_xy"]["bytes"] / 1e9),
                      "parallelism": "replicas only" if world > 1 else "single GPU",
                      "plan": plan.info()},
           "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof}
    if not args.no_cpu_baseline:
        na = args.cpu_angles or max(1, min(cfg.ntheta // 3, int(round(16 * (256 * 256) / (cfg.h * cfg.w)))))
        cb = cpu_sample(cfg, d, na)
        out["cpu_baseline"] = {"value": float(f"{cb['value']:.6g}"), "unit": UNIT, "cores": cb["cores"], "kind": "oracle",
                               "sample": cb["sample"], "seconds": round(cb["seconds"], 2)}
    print(json.dumps(out), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def run_reference(args):
    """The reference arm of this tier = the CPU oracle, as it stands, on the host cores (rank 0 only).
    One step = one bounded sample (cpu_sample: one x3-slice at two angle counts); the step's value is the whole-job
    throughput the sample's two cost terms give."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import numpy as np
    import torch
    from oracle import lam_oracle as O
    from paper_2401_11101_b200 import inputs
    cfg = inputs.config(args.config)
    na = args.cpu_angles or max(1, min(cfg.ntheta // 3, int(round(4 * (256 * 256) / (cfg.h * cfg.w)))))
    # only the sampled angles are generated (same recipe, same seed; the angle subset is part of the stated sample)
    idx = np.linspace(0, cfg.ntheta - 1, 2 * na).astype(int)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    d = inputs.projections(cfg, device=dev, theta=cfg.theta()[idx])
    d = {k: (v.cpu() if hasattr(v, "cpu") else v) for k, v in d.items()}
    vals, secs, last = [], [], None
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        last = cpu_sample(cfg, d, na, theta=d["theta"], mult=2)
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
