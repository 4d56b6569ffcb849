"""Parameter-study harness: the figures of merit against closed forms (CPU), and the beta sweep on
the GPU against the same figures computed from the oracle's reconstruction."""
import numpy as np
import pytest

import synth_inputs as si


def test_figures_of_merit_closed_forms():
    from paper_1903_10088_b200 import study
    from scipy.ndimage import gaussian_filter
    cfg = si.ScanConfig("t", 256, 256, 1.0, 8, 8, seed=1)
    ell, rois = si.insert_phantom(cfg)
    assert len(rois) == 12 and abs(rois[-1][3] - si.MU_WATER) < 1e-15
    clean = si.rasterize(cfg, ell, supersample=4)
    rng = np.random.default_rng(0)
    sigma = 2e-4
    noisy = clean + sigma * rng.standard_normal(clean.shape)
    fom = study.figures_of_merit(noisy, cfg.pixel_mm, rois)
    assert abs(fom["snr_background"] - si.MU_WATER / sigma) < 0.08 * si.MU_WATER / sigma
    for (x0, y0, rad, mu), c, m in zip(rois[:-1], fom["cnr"], fom["mean"]):
        assert abs(m - mu) < 8e-5
        want = abs(mu - si.MU_WATER) / sigma
        assert abs(c - want) < 0.1 * want + 0.5
    # a Gaussian blur of width s turns the rod's edge into an error-function profile: 10-90 % = 2.563 s
    # (a straight edge; the rod's curvature and the radial binning shorten it somewhat)
    ws = [study.edge_width(gaussian_filter(clean, s), cfg.pixel_mm, rois[-2]) for s in (1.5, 2.0, 3.0)]
    assert ws[0] < ws[1] < ws[2]
    for s, w in zip((1.5, 2.0, 3.0), ws):
        assert abs(w - 2.563 * s) < 0.25 * 2.563 * s
    assert study.edge_width(clean, cfg.pixel_mm, rois[-2]) < 1.2            # the rasterised edge itself: about a pixel


@pytest.mark.gpu
def test_beta_sweep_on_the_gpu_and_against_the_oracle():
    torch = pytest.importorskip("torch")
    import oracle
    import paper_1903_10088_b200 as osiv
    from paper_1903_10088_b200 import study
    cfg = si.ScanConfig("t", 128, 128, 2.0, 200, 192, i0=3e4, seed=41)
    ell, rois = si.insert_phantom(cfg)
    counts = si.make_counts(cfg, si.ellipse_sinogram(cfg, ell), cfg.seed)
    gg = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm)
    prm = osiv.Params(n_subsets=10, n_iters=150)
    betas = [0.0, 0.005, 0.02, 0.08]
    with osiv.Handle(gg, max_batch=1) as h:
        rows = study.beta_sweep(h, torch.from_numpy(counts)[None].cuda(), cfg.i0, betas, prm, cfg.pixel_mm, rois)
    noise = [r["noise_background"] for r in rows]
    assert all(a > b for a, b in zip(noise, noise[1:]))                     # more TV, less noise ...
    assert rows[-1]["snr_background"] > 2.0 * rows[0]["snr_background"]
    assert all(b > a for a, b in zip(rows[0]["cnr"], rows[2]["cnr"]))       # ... and every rod stands out more
    assert all(np.isfinite(w) and 1.0 < w < 12.0 for r in rows[2:] for w in r["edge_width_mm"][-2:])  # reported, in mm
    # the same figures from the oracle's image for one beta
    og = oracle.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm)
    ref, _, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(beta=betas[2], n_subsets=10, n_iters=150))
    want = study.figures_of_merit(ref, cfg.pixel_mm, rois)
    assert abs(rows[2]["snr_background"] - want["snr_background"]) < 1e-3 * want["snr_background"]
    assert np.allclose(rows[2]["cnr"], want["cnr"], rtol=2e-3, atol=1e-3)
