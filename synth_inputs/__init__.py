"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no projector, no chord weights, no
residual, no TV, no update): it only *describes the scan* (where the source and the detector
channels are -- the data-acquisition geometry of SURVEY.md 8(c) C1 / BASELINE.json), draws
ellipse phantoms, evaluates their textbook closed-form line integrals, and samples Poisson
counts.  It imports neither ``oracle`` nor ``paper_1903_10088_b200``.

The inputs stand in for the paper's Gammex / Cheese / patient MVCT scans, which
are not available; shapes follow BASELINE.json ``configs``, the attenuation scale PAPER.md:140
(water 0.07 /cm = 0.0070 /mm).  Recipe (also stated in DESIGN.md):

  phantom  = water disk, radius 0.85 R_FOV, mu = 0.0070 /mm, plus K ellipses whose densities ADD
             (centre uniform in the disk of radius 0.55 R_FOV, semi-axes U(0.05,0.22) R_FOV, angle
             U(0,pi), insert value drawn per config; an ellipse contributes (value - 0.0070))
  sinogram = exact line integrals of those ellipses along the zero-width rays of the fan
  counts   = Poisson(I0 * exp(-sinogram)) stored as float32, blank scan b = I0 (scalar)
"""
from .phantom import (  # noqa: F401
    CONFIGS, MU_WATER, ScanConfig, scan_config, dgamma, ray_geometry, draw_ellipses, ellipse_sinogram,
    rasterize, make_counts, make_case, uniform_image, uniform_sinogram, insert_phantom,
)
