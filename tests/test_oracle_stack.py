"""Pins of the oracle's stack-of-slices extension (readings H1-H3); CPU only.

H1 (gantry angle of slice s advanced by k views) is pinned by the exact view-shift invariance of the projector, H2 (3-D
smoothed TV) by central finite differences of the TV value written out here and by its 2-D special case, H3 (per-slice
monitor and step, joint update) by a replay of the step rule on every slice's trace, by the reduction to independent
2-D reconstructions when the coupling is off, and by the coupling's effect on neighbouring slices.
"""
import numpy as np
import pytest

import oracle
import synth_inputs as si


def tv3_by_definition(mu, eps, wz):
    S, ny, nx = mu.shape
    dx = np.zeros_like(mu); dy = np.zeros_like(mu); dz = np.zeros_like(mu)
    dx[:, :, :-1] = mu[:, :, 1:] - mu[:, :, :-1]
    dy[:, :-1, :] = mu[:, 1:, :] - mu[:, :-1, :]
    dz[:-1] = wz * (mu[1:] - mu[:-1])
    return float(np.sqrt(eps * eps + dx * dx + dy * dy + dz * dz).sum())


@pytest.mark.parametrize("eps,wz", [(1e-5, 1.0), (1e-4, 0.6)])
def test_H2_tv3_value_and_gradient(eps, wz):
    rng = np.random.default_rng(2)
    mu = 0.007 + 1e-3 * rng.uniform(size=(4, 7, 9))
    mu[1:3, 2:5, 3:7] = 0.0075                                  # a flat patch: the smoothing eps matters there
    assert abs(oracle.tv3_value(mu, eps, wz) - tv3_by_definition(mu, eps, wz)) < 1e-14
    g = oracle.tv3_grad(mu, eps, wz)
    assert abs(g.sum()) < 1e-12                                 # TV is invariant under a constant shift
    h = 1e-9
    worst = 0.0
    for idx in [(0, 0, 0), (3, 6, 8), (1, 3, 4), (2, 2, 3), (0, 6, 0), (3, 0, 8), (2, 4, 6), (1, 1, 1)]:
        p, m = mu.copy(), mu.copy()
        p[idx] += h; m[idx] -= h
        fd = (tv3_by_definition(p, eps, wz) - tv3_by_definition(m, eps, wz)) / (2 * h)
        worst = max(worst, abs(fd - g[idx]) / max(1.0, abs(fd)))
    assert worst < 2e-6


def test_H2_one_slice_or_no_coupling_is_the_2d_prior():
    mu = 0.007 + 1e-3 * np.random.default_rng(3).uniform(size=(3, 6, 5))
    g0 = oracle.tv3_grad(mu, 1e-5, 0.0)
    for s in range(3):
        assert np.abs(g0[s] - oracle.tv_grad(mu[s], 1e-5)).max() < 1e-14
    assert np.abs(oracle.tv3_grad(mu[:1], 1e-5, 1.0)[0] - oracle.tv_grad(mu[0], 1e-5)).max() < 1e-14


def test_H1_view_shift_is_a_roll_of_the_view_axis():
    g = oracle.Geometry(nx=16, ny=16, pixel_mm=1.25, n_views=24, n_channels=20, sad_mm=90.0, theta0_rad=0.1)
    x = np.random.default_rng(4).uniform(size=(16, 16))
    full = oracle.forward(g, x)
    for k in (1, 5):
        gs = oracle.Geometry(nx=16, ny=16, pixel_mm=1.25, n_views=24, n_channels=20, sad_mm=90.0,
                             theta0_rad=0.1 + 2 * np.pi * k / 24)
        assert np.abs(oracle.forward(gs, x) - np.roll(full, -k, axis=0)).max() < 1e-11


def small_stack(S=3, seed=31, i0=2e4):
    cfg = si.ScanConfig("t", 16, 16, 1.25, 24, 24, i0=i0, seed=seed, n_ellipses=3, sad_mm=90.0)
    g = oracle.Geometry(nx=16, ny=16, pixel_mm=1.25, n_views=24, n_channels=24, sad_mm=90.0)
    return cfg, g


def shifted_counts(cfg, g, S, k, rng):
    """Poisson counts of S different phantoms, slice s seen from gantry angles advanced by k*s views."""
    out, truths = [], []
    for s in range(S):
        truth = si.rasterize(cfg, si.draw_ellipses(cfg, cfg.seed + s))
        gs = oracle.Geometry(nx=g.nx, ny=g.ny, pixel_mm=g.pixel_mm, n_views=g.n_views, n_channels=g.n_channels,
                             sad_mm=g.sad_mm, theta0_rad=2 * np.pi * k * s / g.n_views)
        out.append(rng.poisson(cfg.i0 * np.exp(-oracle.forward(gs, truth))).astype(np.float64))
        truths.append(truth)
    return np.stack(out), np.stack(truths)


def test_H3_uncoupled_stack_is_independent_slices_at_shifted_angles():
    cfg, g = small_stack(i0=1e6)
    k, S = 5, 3
    counts, truths = shifted_counts(cfg, g, S, k, np.random.default_rng(5))
    prm = oracle.Params(beta=0.003, n_subsets=3, n_iters=90)
    img, tr, status = oracle.reconstruct_stack(g, counts, cfg.i0, prm, view_shift=k, tv_z=0.0)
    assert status == 0
    for s in range(S):
        gs = oracle.Geometry(nx=16, ny=16, pixel_mm=1.25, n_views=24, n_channels=24, sad_mm=90.0,
                             theta0_rad=2 * np.pi * k * s / 24)
        one, tr1, _ = oracle.reconstruct(gs, counts[s], cfg.i0, prm)
        assert np.array_equal(img[s], one) and np.array_equal(tr[s], tr1)
    # with the wrong shift a slice comes out rotated against its phantom (the monitor cannot tell: a rotated image
    # fits the rotated data just as well), so the error against the truth is what separates the two
    bad, _, _ = oracle.reconstruct_stack(g, counts, cfg.i0, prm, view_shift=0, tv_z=0.0)
    yy, xx = np.mgrid[0:16, 0:16] - 7.5
    inside = (xx ** 2 + yy ** 2) < 6.0 ** 2
    err = lambda a, s: np.linalg.norm((a[s] - truths[s])[inside]) / np.linalg.norm(truths[s][inside])
    assert np.array_equal(bad[0], img[0])
    for s in (1, 2):
        assert err(bad, s) > 1.5 * err(img, s)


def test_H3_coupled_stack_step_rule_replay_and_smoothing_across_slices():
    cfg, g = small_stack()
    S = 4
    rng = np.random.default_rng(6)
    truth = si.rasterize(cfg, si.draw_ellipses(cfg, cfg.seed))
    counts = np.stack([rng.poisson(cfg.i0 * np.exp(-oracle.forward(g, truth))).astype(np.float64) for _ in range(S)])
    prm = oracle.Params(beta=0.02, n_subsets=2, n_iters=60)
    free, _, _ = oracle.reconstruct_stack(g, counts, cfg.i0, prm, tv_z=0.0)
    tied, tr, status = oracle.reconstruct_stack(g, counts, cfg.i0, prm, tv_z=1.0)
    assert status == 0
    for s in range(S):                                           # Eq. 4-5 on every slice's own monitor
        lam = np.zeros(60)
        for n in range(60):
            if n == 0:
                lam[n] = prm.lambda0
            elif tr[s, n, 0] < tr[s, n - 1, 0]:
                lam[n] = lam[n - 1] + prm.lambda_up
            else:
                lam[n] = max(lam[n - 1] - prm.lambda_down, prm.lambda_min)
        assert np.array_equal(lam, tr[s, :, 1])
    # same object in every slice, independent noise: the z-coupling pulls the slices together
    spread = lambda v: float(np.abs(np.diff(v, axis=0)).sum())
    assert spread(tied) < 0.7 * spread(free)
    assert not np.array_equal(tied[0], free[0])
