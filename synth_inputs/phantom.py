"""Seeded ellipse phantoms, analytic fan-beam sinograms and Poisson counts (see package docstring)."""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Dict, List, Tuple

import numpy as np

MU_WATER = 0.0070  # /mm  ("approximately 0.07 [cm^-1]" in the water area)


@dataclass(frozen=True)
class ScanConfig:
    """One BASELINE.json config."""
    name: str
    nx: int
    ny: int
    pixel_mm: float
    n_views: int
    n_channels: int
    sad_mm: float = 850.0
    sdd_mm: float = 1450.0
    dgamma_rad: float = 0.0       # 0 -> channels span the FOV circle: 2*asin(R_FOV/SAD)/C
    channel_offset: float = 0.0
    theta0_rad: float = 0.0
    i0: float = 2e4
    betas: Tuple[float, ...] = (0.005,)
    n_subsets: int = 1
    n_iters: int = 10
    seed: int = 0
    n_ellipses: int = 5
    mix: str = "uniform"          # how insert values are drawn
    batch: int = 1


CONFIGS: Dict[str, ScanConfig] = {
    # BASELINE.json configs[0..4]; seeds from SURVEY.md 8(d)
    "1": ScanConfig("1", 64, 64, 1.0, 90, 96, i0=1e4, betas=(0.01,), n_subsets=1, n_iters=10, seed=1001,
                    n_ellipses=5),
    "2": ScanConfig("2", 256, 256, 1.5, 400, 384, i0=5e4, betas=(0.005,), n_subsets=10, n_iters=100, seed=2001,
                    n_ellipses=10),
    "3": ScanConfig("3", 512, 512, 0.78125, 800, 738, i0=2e4, betas=(0.001, 0.005, 0.02), n_subsets=20,
                    n_iters=500, seed=3001, n_ellipses=20, mix="mvct"),
    "4": ScanConfig("4", 512, 512, 0.78125, 800, 738, i0=2e4, betas=(0.005,), n_subsets=20, n_iters=500,
                    seed=4001, n_ellipses=20, mix="mvct", batch=64),
    "5a": ScanConfig("5a", 512, 512, 0.78125, 800, 738, seed=5001),
    "5b": ScanConfig("5b", 1024, 1024, 0.390625, 1600, 1476, seed=5002),
}


def scan_config(name: str, **overrides) -> ScanConfig:
    return replace(CONFIGS[str(name)], **overrides)


def dgamma(cfg: ScanConfig) -> float:
    if cfg.dgamma_rad > 0:
        return cfg.dgamma_rad
    rfov = 0.5 * min(cfg.nx, cfg.ny) * cfg.pixel_mm
    return 2.0 * np.arcsin(rfov / cfg.sad_mm) / cfg.n_channels


def ray_geometry(cfg: ScanConfig):
    """Where the scanner puts its rays: source s_v = SAD(cos th_v, sin th_v), th_v = th0 + 2 pi v / V;
    channel c looks along d = -(cos(th_v+ga_c), sin(th_v+ga_c)), ga_c = (c-(C-1)/2+off) dgamma.
    Returns sx, sy [V,1] and dx, dy [V,C] (float64)."""
    th = cfg.theta0_rad + 2.0 * np.pi * np.arange(cfg.n_views) / cfg.n_views
    ga = (np.arange(cfg.n_channels) - 0.5 * (cfg.n_channels - 1) + cfg.channel_offset) * dgamma(cfg)
    ang = th[:, None] + ga[None, :]
    return (cfg.sad_mm * np.cos(th)[:, None], cfg.sad_mm * np.sin(th)[:, None], -np.cos(ang), -np.sin(ang))


def draw_ellipses(cfg: ScanConfig, seed: int) -> List[Tuple[float, float, float, float, float, float]]:
    """List of (x0, y0, A, B, phi, density) in mm and /mm; densities add.  First entry is the water disk."""
    rng = np.random.default_rng(seed)
    rfov = 0.5 * min(cfg.nx, cfg.ny) * cfg.pixel_mm
    ell = [(0.0, 0.0, 0.85 * rfov, 0.85 * rfov, 0.0, MU_WATER)]
    for _ in range(cfg.n_ellipses):
        rad = 0.55 * rfov * np.sqrt(rng.uniform())
        ang = rng.uniform(0.0, 2.0 * np.pi)
        a, b = rng.uniform(0.05, 0.22, size=2) * rfov
        phi = rng.uniform(0.0, np.pi)
        u = rng.uniform()
        if cfg.mix == "mvct":       # 60 % low-contrast (+-1..3 % of water), 20 % fat-like, 20 % bone-like
            if u < 0.6:
                val = MU_WATER * (1.0 + rng.choice([-1.0, 1.0]) * rng.uniform(0.01, 0.03))
            elif u < 0.8:
                val = rng.uniform(0.0060, 0.0068)
            else:
                val = rng.uniform(0.0100, 0.0130)
        else:
            val = rng.uniform(0.0050, 0.0130)
        ell.append((rad * np.cos(ang), rad * np.sin(ang), a, b, phi, val - MU_WATER))
    return ell


def ellipse_sinogram(cfg: ScanConfig, ellipses) -> np.ndarray:
    """Exact line integrals [V,C] of a sum of constant-density ellipses along the fan's rays (the
    textbook chord of a line through an ellipse: map the ellipse to the unit circle, solve the
    quadratic)."""
    sx, sy, dx, dy = ray_geometry(cfg)
    out = np.zeros(dx.shape, dtype=np.float64)
    for (x0, y0, A, B, phi, rho) in ellipses:
        cp, sp = np.cos(phi), np.sin(phi)
        px, py = sx - x0, sy - y0
        qx, qy = (cp * px + sp * py) / A, (-sp * px + cp * py) / B
        ex, ey = (cp * dx + sp * dy) / A, (-sp * dx + cp * dy) / B
        a = ex * ex + ey * ey
        b = qx * ex + qy * ey
        c = qx * qx + qy * qy - 1.0
        disc = b * b - a * c
        out += rho * 2.0 * np.sqrt(np.maximum(disc, 0.0)) / a
    return out


def rasterize(cfg: ScanConfig, ellipses, supersample: int = 8) -> np.ndarray:
    """The phantom on the pixel grid [ny,nx] (mean over supersample^2 points per pixel), float64."""
    ss = supersample
    sub = (np.arange(ss) + 0.5) / ss - 0.5
    xs = ((np.arange(cfg.nx) - 0.5 * (cfg.nx - 1))[:, None] + sub[None, :]).reshape(-1) * cfg.pixel_mm
    ys = ((np.arange(cfg.ny) - 0.5 * (cfg.ny - 1))[:, None] + sub[None, :]).reshape(-1) * cfg.pixel_mm
    img = np.zeros((cfg.ny * ss, cfg.nx * ss), dtype=np.float64)
    X, Y = xs[None, :], ys[:, None]
    for (x0, y0, A, B, phi, rho) in ellipses:
        cp, sp = np.cos(phi), np.sin(phi)
        u = (cp * (X - x0) + sp * (Y - y0)) / A
        v = (-sp * (X - x0) + cp * (Y - y0)) / B
        img += rho * ((u * u + v * v) <= 1.0)
    return img.reshape(cfg.ny, ss, cfg.nx, ss).mean(axis=(1, 3))


def make_counts(cfg: ScanConfig, sinogram: np.ndarray, seed: int) -> np.ndarray:
    """y ~ Poisson(I0 exp(-l)) as float32 [V,C] (integers < 2^24, exact in float32)."""
    rng = np.random.default_rng(seed + 7919)
    return rng.poisson(cfg.i0 * np.exp(-sinogram)).astype(np.float32)


def make_case(cfg: ScanConfig, slice_index: int = 0, noisy: bool = True):
    """(ellipses, line integrals [V,C] float64, counts [V,C] float32) for slice `slice_index` of a config."""
    seed = cfg.seed + slice_index
    ell = draw_ellipses(cfg, seed)
    sino = ellipse_sinogram(cfg, ell)
    if noisy:
        counts = make_counts(cfg, sino, seed)
    else:
        counts = (cfg.i0 * np.exp(-sino)).astype(np.float32)
    return ell, sino, counts


def uniform_image(cfg: ScanConfig, seed: int = None, hi: float = 0.013) -> np.ndarray:
    """config 5: uniform-random image in [0, 0.013] /mm, float32 [ny,nx]"""
    rng = np.random.default_rng(cfg.seed if seed is None else seed)
    return rng.uniform(0.0, hi, size=(cfg.ny, cfg.nx)).astype(np.float32)


def uniform_sinogram(cfg: ScanConfig, n_views: int = None, seed: int = None) -> np.ndarray:
    """config 5: uniform-random sinogram in [0,1], float32 [n_views,C] (seed+1 by default)"""
    rng = np.random.default_rng((cfg.seed + 1) if seed is None else seed)
    nv = cfg.n_views if n_views is None else n_views
    return rng.uniform(0.0, 1.0, size=(nv, cfg.n_channels)).astype(np.float32)


def insert_phantom(cfg: ScanConfig, n_inserts: int = 11):
    """Insert phantom for the parameter study (stands in for the Gammex phantom of PAPER.md:96, whose
    scans and ROI definitions are not available): a water disk of radius 0.8 R_FOV with `n_inserts` circular rods of
    radius 0.075 R_FOV on a ring of radius 0.5 R_FOV, contrasts from -30 % to +60 % of water in equal steps (the rod
    nearest 0 % is given +2 %).  Returns (ellipses, rois): ellipses as in draw_ellipses (densities add), rois = list of
    (x0, y0, radius, mu) in mm and /mm, plus the background ROI at the centre as the last entry."""
    rfov = 0.5 * min(cfg.nx, cfg.ny) * cfg.pixel_mm
    ell = [(0.0, 0.0, 0.8 * rfov, 0.8 * rfov, 0.0, MU_WATER)]
    rois = []
    rad = 0.075 * rfov
    for i in range(n_inserts):
        ang = 2.0 * np.pi * i / n_inserts
        contrast = -0.30 + 0.90 * i / max(n_inserts - 1, 1)
        if abs(contrast) < 0.02:
            contrast = 0.02
        x0, y0 = 0.5 * rfov * np.cos(ang), 0.5 * rfov * np.sin(ang)
        ell.append((x0, y0, rad, rad, 0.0, MU_WATER * contrast))
        rois.append((x0, y0, rad, MU_WATER * (1.0 + contrast)))
    rois.append((0.0, 0.0, 2.0 * rad, MU_WATER))
    return ell, rois
