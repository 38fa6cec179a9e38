"""Seeded synthetic inputs shaped like the paper's slab scans.

This module serves BOTH the oracle-side tests and the CUDA path with the same arrays.  It holds none of
the reconstruction method's arithmetic: it only evaluates closed-form line integrals of Gaussian blobs and
of one box layer in the geometry of Eq. 2, adds noise, and encodes raw 16-bit counts with
the detector model of PAPER.md:99.  The TomoBank brain scans and the Table 1 HDF5
sets are not available; these inputs take their shapes, bit depths and value ranges and
stand in for them.

Works on CPU (float64 arithmetic) or on a CUDA device (float32 arithmetic) through plain torch ops; the
result is float32 (or uint16), and whatever is produced is what both sides read.
"""
import math
from dataclasses import dataclass, field, replace

import numpy as np
import torch

SEED0 = 20240111


@dataclass(frozen=True)
class Config:
    name: str
    n: int
    nz: int
    h: int
    w: int
    ntheta: int
    phi_deg: float
    nblobs: int
    blob_zmax: float            # blob centres have |x3| <= blob_zmax
    layer: bool = False         # thin dense box layer (configs[2]..)
    noise: float = 0.0          # additive Gaussian noise, fraction of max(d) (configs[1])
    raw16: bool = False         # uint16 counts + dark/flat (configs[3], [4])
    dmax: float = 0.0           # raw16: rescale so that max line integral = dmax
    out_of_core: bool = False
    seed: int = SEED0
    width: int = 6
    oversample: float = 2.0

    @property
    def phi(self):
        return math.radians(self.phi_deg)

    def theta(self):
        """Uniform angles over the whole circle, float64."""
        return 2.0 * np.pi * np.arange(self.ntheta, dtype=np.float64) / self.ntheta

    @property
    def voxels(self):
        return self.n * self.n * self.nz


CONFIGS = [
    Config("tiny64", 64, 64, 64, 64, 64, 20.0, 20, 8.0, seed=SEED0 + 0),
    Config("cube256", 256, 256, 256, 256, 400, 20.0, 200, 32.0, noise=0.01, seed=SEED0 + 1),
    Config("slab1024", 1024, 256, 1024, 1024, 1200, 30.0, 2000, 120.0, layer=True, seed=SEED0 + 2),
    Config("slab2048_raw", 2048, 512, 2048, 2048, 1800, 20.0, 4000, 240.0, layer=True, raw16=True,
           dmax=1.9, seed=SEED0 + 3),
    Config("ooc4096_raw", 4096, 1024, 2048, 4096, 3000, 20.0, 8000, 480.0, layer=True, raw16=True,
           dmax=1.9, out_of_core=True, seed=SEED0 + 4),
]


def config(idx):
    return CONFIGS[idx]


def scaled(idx, n, ntheta=None, name=None):
    """The same recipe as configs[idx] shrunk to lateral size n (aspect ratios, phi, blob density kept):
    parity-test cases the oracle finishes in seconds."""
    c = CONFIGS[idx]
    f = n / c.n
    return replace(c, name=name or f"{c.name}@{n}", n=n, nz=max(2, int(round(c.nz * f / 2)) * 2),
                   h=max(2, int(round(c.h * f / 2)) * 2), w=max(2, int(round(c.w * f / 2)) * 2),
                   ntheta=ntheta or max(8, int(round(c.ntheta * f))),
                   nblobs=max(4, int(round(c.nblobs * f))), blob_zmax=max(2.0, c.blob_zmax * f))


def phantom(cfg):
    """Blob list (centres uniform in the disc r <= 0.45 n and |x3| <= blob_zmax, s ~ U[1,4], A ~ U[0.5,1])
    kept inside the measured region r sin(phi) + |x3| cos(phi) + 3 s < h/2 (reading Q9), plus the layer."""
    rng = np.random.default_rng(cfg.seed)
    cs, ss, As = [], [], []
    sp, cp = math.sin(cfg.phi), math.cos(cfg.phi)
    smax = min(4.0, max(1.0, cfg.n / 16))
    while len(cs) < cfg.nblobs:
        r = 0.45 * cfg.n * math.sqrt(rng.uniform())
        a = rng.uniform(0, 2 * math.pi)
        z = rng.uniform(-cfg.blob_zmax, cfg.blob_zmax)
        s = rng.uniform(1.0, smax)
        A = rng.uniform(0.5, 1.0)
        if r * sp + abs(z) * cp + 3 * s < cfg.h / 2 and r + 3 * s < cfg.w / 2:
            cs.append((r * math.cos(a), r * math.sin(a), z))
            ss.append(s)
            As.append(A)
    ph = {"c": np.array(cs), "s": np.array(ss), "A": np.array(As), "layer": None}
    if cfg.layer:
        ph["layer"] = {"a": 0.32 * cfg.n, "b": max(1.0, cfg.n / 64.0), "mu": 0.2 / (2 * max(1.0, cfg.n / 64.0))}
    return ph


def _line_integrals(cfg, ph, theta, device, dtype):
    """d[theta][j_v][j_u]: closed-form line integrals along e_b of the blobs and the layer (Eqs. 1-2).

    A Gaussian blob A exp(-|x-c|^2/(2 s^2)) integrates along any unit-speed line to
    A s sqrt(2 pi) exp(-((u - c.e_u)^2 + (v - c.e_v)^2)/(2 s^2)): separable in (u, v), so one projection is
    Gv^T Gu with Gu[b][j_u], Gv[b][j_v]."""
    T = len(theta)
    th = torch.as_tensor(theta, device=device, dtype=dtype)
    ct, st = torch.cos(th), torch.sin(th)
    sp, cp = math.sin(cfg.phi), math.cos(cfg.phi)
    c = torch.as_tensor(ph["c"], device=device, dtype=dtype)
    s = torch.as_tensor(ph["s"], device=device, dtype=dtype)
    A = torch.as_tensor(ph["A"], device=device, dtype=dtype)
    u = torch.arange(cfg.w, device=device, dtype=dtype) - cfg.w / 2
    v = torch.arange(cfg.h, device=device, dtype=dtype) - cfg.h / 2
    cu = c[None, :, 0] * ct[:, None] + c[None, :, 1] * st[:, None]                       # c.e_u  [T][B]
    cv = (c[None, :, 0] * st[:, None] - c[None, :, 1] * ct[:, None]) * sp + c[None, :, 2] * cp
    Gu = torch.exp(-(u[None, None, :] - cu[:, :, None]) ** 2 / (2 * s[None, :, None] ** 2))
    Gv = torch.exp(-(v[None, None, :] - cv[:, :, None]) ** 2 / (2 * s[None, :, None] ** 2))
    Gv = Gv * (A * s * math.sqrt(2 * math.pi))[None, :, None]
    d = torch.bmm(Gv.transpose(1, 2), Gu)                                                # [T][h][w]
    if ph["layer"] is not None:
        a, b, mu = ph["layer"]["a"], ph["layer"]["b"], ph["layer"]["mu"]
        # ray: p + t e_b, p = u e_u + v e_v, e_b = (sin t cos p, -cos t cos p, -sin p); exact chord in the box
        P1 = u[None, None, :] * ct[:, None, None] + v[None, :, None] * (st * sp)[:, None, None]
        P2 = u[None, None, :] * st[:, None, None] - v[None, :, None] * (ct * sp)[:, None, None]
        P3 = (v * cp)[None, :, None].expand(T, cfg.h, cfg.w)
        E = [st * cp, -ct * cp, torch.full_like(ct, -sp)]
        lo = torch.full((T, cfg.h, cfg.w), -float("inf"), device=device, dtype=dtype)
        hi = torch.full((T, cfg.h, cfg.w), float("inf"), device=device, dtype=dtype)
        for P, e, lim in ((P1, E[0], a), (P2, E[1], a), (P3, E[2], b)):
            e = e[:, None, None].expand_as(P)
            par = e.abs() < 1e-12
            es = torch.where(par, torch.ones_like(e), e)
            t0, t1 = (-lim - P) / es, (lim - P) / es
            tlo, thi = torch.minimum(t0, t1), torch.maximum(t0, t1)
            inside = P.abs() <= lim
            tlo = torch.where(par, torch.where(inside, -float("inf"), float("inf")), tlo)
            thi = torch.where(par, torch.where(inside, float("inf"), -float("inf")), thi)
            lo, hi = torch.maximum(lo, tlo), torch.minimum(hi, thi)
        d = d + mu * torch.clamp(hi - lo, min=0.0)
    return d


def detector_fields(cfg, device="cpu"):
    """Fixed-pattern dark (mean 100) and flat (mean 30000, 30 % vertical roll-off) fields, float32 [h][w]."""
    gen = torch.Generator(device="cpu").manual_seed(cfg.seed + 7919)
    dark = 100.0 + 2.0 * torch.randn(cfg.h, cfg.w, generator=gen)
    vv = (torch.arange(cfg.h, dtype=torch.float32) - cfg.h / 2) * 2 / cfg.h
    flat = 30000.0 * (1 - 0.3 * vv[:, None] ** 2) * (1 + 0.01 * torch.randn(cfg.h, cfg.w, generator=gen))
    return dark.float().to(device), flat.float().to(device)


def projections(cfg, device="cpu", out=None, chunk=None, theta=None):
    """Full input of a config.

    Returns dict(proj=..., dark=..., flat=..., theta=float64 numpy):
      fp32 configs : proj float32 [ntheta][h][w] line integrals (+ noise for configs[1])
      raw16 configs: proj uint16 counts, dark/flat float32 [h][w]
    `out` may be a preallocated tensor (e.g. pinned host memory for the out-of-core config).
    `theta` (optional): generate only these angles (a bounded sample of the scan; global scales are still taken
    from the full angle set, the noise stream is the sample's own)."""
    device = torch.device(device)
    dtype = torch.float64 if device.type == "cpu" else torch.float32
    ph = phantom(cfg)
    full_theta = cfg.theta()
    theta = full_theta if theta is None else np.ascontiguousarray(theta, dtype=np.float64)
    ntheta = len(theta)
    if chunk is None:
        chunk = max(1, int(2 ** 26 // max(1, cfg.nblobs * max(cfg.h, cfg.w) + cfg.h * cfg.w * 8)))
    odt = torch.uint16 if cfg.raw16 else torch.float32
    if out is None:
        out = torch.empty((ntheta, cfg.h, cfg.w), dtype=odt, device=device)
    dark = flat = None
    scale = 1.0
    if cfg.raw16:
        dark, flat = detector_fields(cfg, device)
        # one global scale so that max d = dmax (transmission >= 15 %); found on a theta subset
        sub = full_theta[:: max(1, cfg.ntheta // 16)]
        scale = cfg.dmax / float(_line_integrals(cfg, ph, sub, device, dtype).max())
    gen = torch.Generator(device=device).manual_seed(cfg.seed + 104729)
    dmax = None
    if cfg.noise > 0:
        sub = full_theta[:: max(1, cfg.ntheta // 16)]
        dmax = float(_line_integrals(cfg, ph, sub, device, dtype).max())
    for t0 in range(0, ntheta, chunk):
        t1 = min(ntheta, t0 + chunk)
        d = _line_integrals(cfg, ph, theta[t0:t1], device, dtype) * scale
        if cfg.noise > 0:
            d = d + cfg.noise * dmax * torch.randn(d.shape, generator=gen, device=device, dtype=dtype)
        if cfg.raw16:
            cnt = (flat - dark).to(dtype)[None] * torch.exp(-d)
            cnt = cnt + torch.sqrt(cnt.clamp(min=0)) * torch.randn(d.shape, generator=gen, device=device, dtype=dtype)
            raw = torch.clamp(torch.round(cnt + dark.to(dtype)[None]), 0, 65535)
            out[t0:t1].copy_(raw.to(torch.int32).to(torch.uint16))
        else:
            out[t0:t1].copy_(d.to(torch.float32))
    return {"proj": out, "dark": dark, "flat": flat, "theta": theta, "phantom": ph, "scale": scale}
