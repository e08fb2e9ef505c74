"""Seeded synthetic DECam-shaped image stacks (input generation only).

This module serves BOTH the CUDA path and the CPU oracle with inputs.  It holds none of
the method's arithmetic: no psi/phi, no trajectory sampling, no scoring.  It only draws
noise, variance planes, masks, PSF kernels, injected sources, timestamps and velocity
grids with the shapes and value structure of the paper's workload (PAPER.md:221-231:
DECam 2K x 4K CCDs / 4K x 4K patches, 0.26"/px, ~1.6 h cadence over 3-4 nights, Gaussian
PSF, 1-5.7"/hr = 92-526 px/day) as laid out per config in DESIGN.md ("Input recipe").

The real HiTS data are not available; these stacks stand in for them.

Draw order (one numpy Generator per stack, seed = config number unless overridden):
times -> per-image variance -> per-image PSF parameters -> masks -> sources -> noise.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np


# --------------------------------------------------------------------------------------
# configuration
# --------------------------------------------------------------------------------------
@dataclass(frozen=True)
class StackConfig:
    name: str
    N: int
    H: int
    W: int
    seed: int
    # times
    times_kind: str = "nights"          # "explicit" | "nights" | "uniform"
    times_explicit: tuple = ()
    epochs_per_night: int = 4
    epoch_spacing: float = 0.0625
    t_span: float = 4.0                 # for "uniform"
    # variance
    var_lo: float = 100.0
    var_hi: float = 100.0
    var_gradient: float = 0.0           # +/- fraction of a smooth plane
    # psf
    psf_kind: str = "gauss"             # "gauss" | "elliptical"
    sigma_lo: float = 1.0
    sigma_hi: float = 1.0
    # mask
    mask_frac: float = 0.0
    mask_static: bool = False           # config 4: bad columns + saturated discs
    # sources
    n_sources: int = 0
    flux_lo: float = 100.0
    flux_hi: float = 2000.0
    flux_from_nu: tuple = ()            # (nu_lo, nu_hi): config 4
    sources_explicit: tuple = ()        # ((x, y, vx, vy, F), ...)
    # velocity grid
    n_angles: int = 8
    n_speeds: int = 8
    ang_lo: float = -math.pi / 4
    ang_hi: float = math.pi / 4
    speed_lo: float = 5.0
    speed_hi: float = 25.0
    # search
    K: int = 4
    min_obs: int = 3

    @property
    def V(self) -> int:
        return self.n_angles * self.n_speeds

    @property
    def trajectories(self) -> int:
        return self.H * self.W * self.V

    @property
    def evals(self) -> int:
        return self.trajectories * self.N


def config(k: int, **over) -> StackConfig:
    """BASELINE.json configs[k-1] (k = 1..5).  Config 5 is a sweep: pass N=..., and
    n_angles/n_speeds for the grid point (defaults: N=10, 32x20).  k = 6 is not a BASELINE.json
    config: it is the paper's own production search (13 images over three nights,
    128 angles within +-12 degrees x 250 speeds over 1-5.7 arcsec/hour = 92.3-526 px/day at 0.26
    arcsec/px, 32 000 velocities per start pixel, threshold nu >= 10), the workload of row N4."""
    if k == 1:
        c = StackConfig(
            name="c1_tiny", N=5, H=64, W=64, seed=1,
            times_kind="explicit", times_explicit=(0.0, 0.1, 0.2, 1.0, 1.1),
            var_lo=100.0, var_hi=100.0, sigma_lo=1.0, sigma_hi=1.0,
            sources_explicit=((20.0, 30.0, 12.0, -4.0, 500.0),),
            n_angles=8, n_speeds=8, speed_lo=5.0, speed_hi=25.0, K=4, min_obs=3)
    elif k == 2:
        c = StackConfig(
            name="c2_ccd_pair", N=8, H=2048, W=4096, seed=2,
            var_lo=80.0, var_hi=150.0, sigma_lo=1.2, sigma_hi=1.8, mask_frac=0.005,
            n_sources=50, flux_lo=100.0, flux_hi=2000.0,
            n_angles=32, n_speeds=16, speed_lo=90.0, speed_hi=500.0, K=8, min_obs=5)
    elif k == 3:
        c = StackConfig(
            name="c3_paper_scale", N=15, H=4096, W=4096, seed=3,
            var_lo=80.0, var_hi=150.0, var_gradient=0.2, sigma_lo=1.2, sigma_hi=2.0,
            mask_frac=0.01, n_sources=200, flux_lo=50.0, flux_hi=1000.0,
            n_angles=32, n_speeds=20, speed_lo=90.0, speed_hi=500.0, K=8, min_obs=8)
    elif k == 4:
        c = StackConfig(
            name="c4_stress", N=12, H=4096, W=4096, seed=4,
            times_kind="uniform", t_span=4.0,
            var_lo=50.0, var_hi=400.0, psf_kind="elliptical", sigma_lo=1.0, sigma_hi=2.5,
            mask_frac=0.10, mask_static=True, n_sources=500, flux_from_nu=(5.0, 10.0),
            n_angles=64, n_speeds=32, speed_lo=50.0, speed_hi=600.0, K=16, min_obs=6)
    elif k == 5:
        N = over.pop("N", 10)
        c = StackConfig(
            name=f"c5_sweep_N{N}", N=N, H=4096, W=4096, seed=5,
            var_lo=80.0, var_hi=150.0, sigma_lo=1.2, sigma_hi=1.8, mask_frac=0.005,
            n_sources=100, flux_lo=100.0, flux_hi=2000.0,
            n_angles=32, n_speeds=20, ang_lo=-math.pi / 2, ang_hi=math.pi / 2,
            speed_lo=50.0, speed_hi=800.0, K=8, min_obs=(N + 1) // 2)
    elif k == 6:
        c = StackConfig(
            name="c6_hits_production", N=13, H=4096, W=4096, seed=6,
            epochs_per_night=5, epoch_spacing=0.0625,                  # 5 + 5 + 3 epochs over three nights
            var_lo=80.0, var_hi=150.0, sigma_lo=1.2, sigma_hi=1.8, mask_frac=0.01,
            n_sources=200, flux_lo=100.0, flux_hi=2000.0,
            n_angles=128, n_speeds=250, ang_lo=-math.radians(12.0), ang_hi=math.radians(12.0),
            speed_lo=24.0 / 0.26, speed_hi=5.7 * 24.0 / 0.26, K=8, min_obs=7)
    else:
        raise ValueError(f"no config {k}")
    return replace(c, **over) if over else c


SWEEP_GRIDS = {256: (16, 16), 640: (32, 20), 2048: (64, 32), 8192: (128, 64)}


# --------------------------------------------------------------------------------------
# pieces
# --------------------------------------------------------------------------------------
def make_times(cfg: StackConfig, rng: np.random.Generator) -> np.ndarray:
    if cfg.times_kind == "explicit":
        t = np.asarray(cfg.times_explicit, dtype=np.float64)
        assert t.shape == (cfg.N,)
        return t
    if cfg.times_kind == "uniform":
        return np.sort(rng.uniform(0.0, cfg.t_span, size=cfg.N))
    # nights x epochs, truncated to N (config 3: 4 nights x 4 epochs, last dropped)
    e = cfg.epochs_per_night
    t = [float(i // e) + (i % e) * cfg.epoch_spacing for i in range(cfg.N)]
    return np.asarray(t, dtype=np.float64)


def velocity_grid(n_angles, n_speeds, ang_lo, ang_hi, speed_lo, speed_hi) -> np.ndarray:
    """[V,2] fp32 (vx, vy) px/day; j = a * n_speeds + s; angles and speeds linearly
    spaced, end points included (PAPER.md:231 'linearly-spaced grid'); built in double,
    rounded once to fp32."""
    ang = np.linspace(ang_lo, ang_hi, n_angles, dtype=np.float64)
    spd = np.linspace(speed_lo, speed_hi, n_speeds, dtype=np.float64)
    a, s = np.meshgrid(ang, spd, indexing="ij")
    v = np.stack([s * np.cos(a), s * np.sin(a)], axis=-1).reshape(-1, 2)
    return np.ascontiguousarray(v.astype(np.float32))


def gaussian_psf_kernels(sig_x, sig_y, theta, P: int) -> np.ndarray:
    """[N,P,P] fp32, psf[i][r+dy][r+dx] = T_i(dx,dy): Gaussian point-sampled at pixel
    centres, unit sum in double, then cast to fp32."""
    r = (P - 1) // 2
    d = np.arange(-r, r + 1, dtype=np.float64)
    dx, dy = np.meshgrid(d, d, indexing="xy")          # dx varies along columns
    out = []
    for sx, sy, th in zip(sig_x, sig_y, theta):
        c, s = math.cos(th), math.sin(th)
        u = c * dx + s * dy
        v = -s * dx + c * dy
        g = np.exp(-0.5 * ((u / sx) ** 2 + (v / sy) ** 2))
        out.append(g / g.sum())
    return np.ascontiguousarray(np.stack(out).astype(np.float32))


def _blob_mask(rng, H, W, frac) -> np.ndarray:
    """Cosmic-ray-like 1-3 px blobs covering about `frac` of the plane."""
    m = np.zeros((H, W), dtype=np.uint8)
    if frac <= 0:
        return m
    n = int(round(frac * H * W / 2.0))                 # mean blob length 2
    y = rng.integers(0, H, size=n)
    x = rng.integers(0, W, size=n)
    length = rng.integers(1, 4, size=n)
    direction = rng.integers(0, 4, size=n)             # E, S, SE, NE
    ddx = np.array([1, 0, 1, 1])[direction]
    ddy = np.array([0, 1, 1, -1])[direction]
    for k in range(3):
        sel = length > k
        yy = np.clip(y[sel] + k * ddy[sel], 0, H - 1)
        xx = np.clip(x[sel] + k * ddx[sel], 0, W - 1)
        m[yy, xx] = 1
    return m


def _static_mask(rng, H, W) -> np.ndarray:
    """Bad columns + saturated-star discs of radius 5-30 px (same in every image)."""
    m = np.zeros((H, W), dtype=np.uint8)
    ncol = max(1, W // 400)
    for cx in rng.integers(0, W, size=ncol):
        m[:, cx:cx + int(rng.integers(1, 3))] = 1
    ndisc = max(1, int(0.04 * H * W / (math.pi * 17.5 ** 2)))
    cy = rng.integers(0, H, size=ndisc)
    cx = rng.integers(0, W, size=ndisc)
    rr = rng.uniform(5.0, 30.0, size=ndisc)
    for y0, x0, r in zip(cy, cx, rr):
        ri = int(math.ceil(r))
        ya, yb = max(0, y0 - ri), min(H, y0 + ri + 1)
        xa, xb = max(0, x0 - ri), min(W, x0 + ri + 1)
        yy, xx = np.ogrid[ya:yb, xa:xb]
        m[ya:yb, xa:xb] |= (((yy - y0) ** 2 + (xx - x0) ** 2) <= r * r).astype(np.uint8)
    return m


def _inject(sci_i, x, y, flux, sx, sy, th):
    """Add flux * (unit-sum Gaussian sampled at pixel centres) at sub-pixel (x, y)."""
    H, W = sci_i.shape
    rad = int(math.ceil(5.0 * max(sx, sy))) + 1
    x0, y0 = int(math.floor(x + 0.5)), int(math.floor(y + 0.5))
    xa, xb = x0 - rad, x0 + rad + 1
    ya, yb = y0 - rad, y0 + rad + 1
    if xb <= 0 or yb <= 0 or xa >= W or ya >= H:
        return
    xs = np.arange(xa, xb, dtype=np.float64) - x
    ys = np.arange(ya, yb, dtype=np.float64) - y
    dx, dy = np.meshgrid(xs, ys, indexing="xy")
    c, s = math.cos(th), math.sin(th)
    u = c * dx + s * dy
    v = -s * dx + c * dy
    g = np.exp(-0.5 * ((u / sx) ** 2 + (v / sy) ** 2))
    g *= flux / g.sum()
    cxa, cxb = max(xa, 0), min(xb, W)
    cya, cyb = max(ya, 0), min(yb, H)
    sci_i[cya:cyb, cxa:cxb] += g[cya - ya:cyb - ya, cxa - xa:cxb - xa].astype(np.float32)


# --------------------------------------------------------------------------------------
# the stack
# --------------------------------------------------------------------------------------
@dataclass
class Stack:
    cfg: StackConfig
    sci: np.ndarray        # [N,H,W] f32
    var: np.ndarray        # [N,H,W] f32
    mask: np.ndarray       # [N,H,W] u8 (nonzero = masked)
    psf: np.ndarray        # [N,P,P] f32
    times: np.ndarray      # [N] f64 days
    vel_grid: np.ndarray   # [V,2] f32 px/day
    sources: np.ndarray    # [S,5] f64 (x, y, vx, vy, flux) at times[0]
    psf_sigma: np.ndarray  # [N,3] f64 (sigma_x, sigma_y, theta)
    var_level: np.ndarray = field(default_factory=lambda: np.zeros(0))


def make_stack(cfg: StackConfig, seed: Optional[int] = None, noise: bool = True) -> Stack:
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    N, H, W = cfg.N, cfg.H, cfg.W

    times = make_times(cfg, rng)

    # per-image variance level (+ smooth plane gradient)
    lvl = rng.uniform(cfg.var_lo, cfg.var_hi, size=N) if cfg.var_hi > cfg.var_lo \
        else np.full(N, cfg.var_lo)
    var = np.empty((N, H, W), dtype=np.float32)
    if cfg.var_gradient > 0:
        phi = rng.uniform(0.0, 2 * math.pi, size=N)
        yy = np.linspace(-1.0, 1.0, H, dtype=np.float64)[:, None]
        xx = np.linspace(-1.0, 1.0, W, dtype=np.float64)[None, :]
        for i in range(N):
            g = (math.cos(phi[i]) * xx + math.sin(phi[i]) * yy) / \
                (abs(math.cos(phi[i])) + abs(math.sin(phi[i])))
            var[i] = (lvl[i] * (1.0 + cfg.var_gradient * g)).astype(np.float32)
    else:
        for i in range(N):
            var[i] = np.float32(lvl[i])

    # per-image PSF
    if cfg.psf_kind == "elliptical":
        sx = rng.uniform(cfg.sigma_lo, cfg.sigma_hi, size=N)
        sy = rng.uniform(cfg.sigma_lo, cfg.sigma_hi, size=N)
        th = rng.uniform(0.0, math.pi, size=N)
    else:
        sx = rng.uniform(cfg.sigma_lo, cfg.sigma_hi, size=N) if cfg.sigma_hi > cfg.sigma_lo \
            else np.full(N, cfg.sigma_lo)
        sy = sx.copy()
        th = np.zeros(N)
    r = int(math.ceil(5.0 * max(cfg.sigma_hi, cfg.sigma_lo)))
    P = 2 * r + 1
    psf = gaussian_psf_kernels(sx, sy, th, P)

    # masks
    mask = np.zeros((N, H, W), dtype=np.uint8)
    if cfg.mask_frac > 0:
        static = _static_mask(rng, H, W) if cfg.mask_static else None
        for i in range(N):
            if static is not None:
                rest = max(0.0, cfg.mask_frac - float(static.mean()))
                mask[i] = static | _blob_mask(rng, H, W, rest)
            else:
                mask[i] = _blob_mask(rng, H, W, cfg.mask_frac)

    # sources (x, y, vx, vy, F) at times[0]
    if cfg.sources_explicit:
        src = np.asarray(cfg.sources_explicit, dtype=np.float64)
    elif cfg.n_sources > 0:
        S = cfg.n_sources
        x = rng.uniform(0, W, size=S)
        y = rng.uniform(0, H, size=S)
        ang = rng.uniform(cfg.ang_lo, cfg.ang_hi, size=S)
        spd = rng.uniform(cfg.speed_lo, cfg.speed_hi, size=S)
        if cfg.flux_from_nu:
            nu_t = rng.uniform(cfg.flux_from_nu[0], cfg.flux_from_nu[1], size=S)
            t2 = (psf.astype(np.float64) ** 2).sum(axis=(1, 2))
            F = nu_t / math.sqrt(float((t2 / lvl).sum()))
        else:
            F = np.exp(rng.uniform(math.log(cfg.flux_lo), math.log(cfg.flux_hi), size=S))
        src = np.stack([x, y, spd * np.cos(ang), spd * np.sin(ang), F], axis=1)
    else:
        src = np.zeros((0, 5), dtype=np.float64)

    # noise + sources
    sci = np.empty((N, H, W), dtype=np.float32)
    for i in range(N):
        if noise:
            sci[i] = rng.standard_normal(size=(H, W), dtype=np.float32)
            sci[i] *= np.sqrt(var[i])
        else:
            sci[i] = 0.0
        dt = times[i] - times[0]
        for (x, y, vx, vy, F) in src:
            _inject(sci[i], x + vx * dt, y + vy * dt, F, sx[i], sy[i], th[i])

    vel = velocity_grid(cfg.n_angles, cfg.n_speeds, cfg.ang_lo, cfg.ang_hi,
                        cfg.speed_lo, cfg.speed_hi)
    return Stack(cfg=cfg, sci=sci, var=var, mask=mask, psf=psf, times=times, vel_grid=vel,
                 sources=src, psf_sigma=np.stack([sx, sy, th], axis=1), var_level=lvl)


def random_psiphi(N, H, W, seed, invalid_frac=0.02) -> np.ndarray:
    """Seeded psi/phi stack for search-only tests: psi ~ N(0,1)*sqrt(phi), phi ~ U[0.5,1.5]*0.01,
    a fraction of pixels set to the invalid marker (NaN, 0).  [N,H,W,2] f32."""
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0.005, 0.015, size=(N, H, W)).astype(np.float32)
    psi = (rng.standard_normal(size=(N, H, W)).astype(np.float32) * np.sqrt(phi)).astype(np.float32)
    bad = rng.random(size=(N, H, W)) < invalid_frac
    psi[bad] = np.nan
    phi[bad] = 0.0
    return np.ascontiguousarray(np.stack([psi, phi], axis=-1))
