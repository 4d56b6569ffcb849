"""Parameter-study harness: the paper picks the TV weight by the signal-to-noise ratio, the
contrast-to-noise ratio and the blurring of edges on an insert phantom (its ROI definitions are
in a supplement that is not available, so the definitions below are this repository's, stated in DESIGN.md section 3).

The reconstructions run through the library (``Handle.reconstruct``); the figures of merit are plain numpy on the
returned images -- analysis, not the hot path.

    snr(roi)        = mean / standard deviation of the pixels within 0.7 radius of the ROI centre
    cnr(roi, bg)    = |mean(roi) - mean(bg)| / standard deviation(bg)
    edge_width(roi) = 10 % - 90 % rise distance [mm] of the mean radial profile across the rod's edge
"""
from __future__ import annotations

from typing import Dict, List, Sequence

import numpy as np


def _grid(shape, pixel_mm: float):
    ny, nx = shape
    x = (np.arange(nx) - 0.5 * (nx - 1)) * pixel_mm
    y = (np.arange(ny) - 0.5 * (ny - 1)) * pixel_mm
    return x[None, :], y[:, None]


def roi_pixels(img: np.ndarray, pixel_mm: float, roi, shrink: float = 0.7) -> np.ndarray:
    X, Y = _grid(img.shape, pixel_mm)
    x0, y0, rad = roi[0], roi[1], roi[2]
    return img[(X - x0) ** 2 + (Y - y0) ** 2 <= (shrink * rad) ** 2]


def snr(img: np.ndarray, pixel_mm: float, roi) -> float:
    p = roi_pixels(img, pixel_mm, roi).astype(np.float64)
    return float(p.mean() / p.std())


def cnr(img: np.ndarray, pixel_mm: float, roi, bg) -> float:
    p = roi_pixels(img, pixel_mm, roi).astype(np.float64)
    b = roi_pixels(img, pixel_mm, bg).astype(np.float64)
    return float(abs(p.mean() - b.mean()) / b.std())


def edge_width(img: np.ndarray, pixel_mm: float, roi, n_bins_per_pixel: int = 4) -> float:
    """10-90 % rise distance of the rod's mean radial profile (binned by distance from the rod's centre)."""
    X, Y = _grid(img.shape, pixel_mm)
    x0, y0, rad = roi[0], roi[1], roi[2]
    r = np.sqrt((X - x0) ** 2 + (Y - y0) ** 2)
    sel = r <= 2.0 * rad
    step = pixel_mm / n_bins_per_pixel
    idx = (r[sel] / step).astype(int)
    prof = np.bincount(idx, weights=img[sel].astype(np.float64)) / np.maximum(np.bincount(idx), 1)
    rr = (np.arange(len(prof)) + 0.5) * step
    inner = prof[rr <= 0.5 * rad].mean()
    outer = prof[(rr >= 1.5 * rad) & (rr <= 2.0 * rad)].mean()
    t = (prof - outer) / (inner - outer)                        # 1 inside the rod, 0 outside
    band = (rr > 0.5 * rad) & (rr < 1.5 * rad)
    rb, tb = rr[band], t[band]

    def crossing(level: float) -> float:
        below = np.nonzero(tb < level)[0]
        if len(below) == 0 or below[0] == 0:
            return float("nan")
        i = below[0]
        return float(rb[i - 1] + (tb[i - 1] - level) / (tb[i - 1] - tb[i]) * (rb[i] - rb[i - 1]))

    return crossing(0.1) - crossing(0.9)


def figures_of_merit(img: np.ndarray, pixel_mm: float, rois: Sequence) -> Dict[str, object]:
    """rois as from synth_inputs.insert_phantom: the rods, then the background ROI."""
    bg = rois[-1]
    rods = rois[:-1]
    return {"snr_background": snr(img, pixel_mm, bg),
            "noise_background": float(roi_pixels(img, pixel_mm, bg).astype(np.float64).std()),
            "cnr": [cnr(img, pixel_mm, r, bg) for r in rods],
            "edge_width_mm": [edge_width(img, pixel_mm, r) for r in rods],
            "mean": [float(roi_pixels(img, pixel_mm, r).astype(np.float64).mean()) for r in rods]}


def beta_sweep(handle, counts, blank, betas: Sequence[float], params, pixel_mm: float, rois: Sequence) -> List[Dict]:
    """One reconstruction per TV weight (``params`` with ``beta`` replaced) of the same counts [1][V][C] (device
    tensor); returns one figures_of_merit dict per beta, with the beta and the final monitor value."""
    from dataclasses import replace
    out = []
    for beta in betas:
        img, trace = handle.reconstruct(counts, blank, replace(params, beta=float(beta)), trace=True)
        fom = figures_of_merit(img[0].detach().cpu().numpy(), pixel_mm, rois)
        fom.update(beta=float(beta), D_final=float(trace[0, -1, 0]), lambda_final=float(trace[0, -1, 1]))
        out.append(fom)
    return out
