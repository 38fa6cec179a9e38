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


def cpu_sample(cfg, d, nangles, nslices=1):
    """The oracle as it stands (path C': exact x3 transform + double-precision 2-D gridding, Eq. 9)
    on `nslices` x3-slices and the first-of-every-k angles; throughput scaled to the whole workload
    (cost is linear in both slices and angles)."""
    import numpy as np
    from oracle import lam_oracle as O
    step = max(1, cfg.ntheta // max(1, nangles))
    idx = np.arange(0, cfg.ntheta, step)[:nangles]
    proj = d["proj"][idx].cpu().contiguous().numpy()
    dark = d["dark"].cpu().numpy() if d["dark"] is not None else None
    flat = d["flat"].cpu().numpy() if d["flat"] is not None else None
    g = O.Geometry(cfg.n, cfg.h, cfg.w, d["theta"][idx], cfg.phi, nz=cfg.nz, dark=dark, flat=flat)
    t0 = time.perf_counter()
    for s in range(nslices):
        O.fbp_gridded_slice(g, proj, cfg.nz // 2 + s, W=cfg.width, sigma=cfg.oversample)
    dt = time.perf_counter() - t0
    frac = (nslices / cfg.nz) * (len(idx) / cfg.ntheta)
    return {"seconds": dt, "value": cfg.voxels * frac / dt / 1e9, "cores": O.threads(),
            "sample": f"{nslices} of {cfg.nz} x3-slices x {len(idx)} of {cfg.ntheta} angles through oracle path C' "
                      f"(fp64 exact-x3 + 2-D gridded USFFT); GVoxel/s scaled by both fractions (cost is linear in each)"}
