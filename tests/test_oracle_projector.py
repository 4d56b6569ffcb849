"""Pins P1-P5, P8 of the float64 oracle's projector pair; CPU only.

Every check compares the oracle with something that is NOT the oracle: polygon clipping written
here, textbook ellipse integrals (synth_inputs), exact symmetries, the adjoint identity between two
differently structured loops, and an eigenvalue bound.
"""
import numpy as np
import pytest

import oracle
import synth_inputs as si


def clip_length(sx, sy, dx, dy, x0, x1, y0, y1):
    """Liang-Barsky: length of the infinite line s+t*d (|d|=1) inside the box [x0,x1]x[y0,y1]."""
    t0, t1 = -np.inf, np.inf
    for s, d, lo, hi in ((sx, dx, x0, x1), (sy, dy, y0, y1)):
        if d == 0.0:
            if s < lo or s > hi:
                return 0.0
            continue
        ta, tb = (lo - s) / d, (hi - s) / d
        if ta > tb:
            ta, tb = tb, ta
        t0, t1 = max(t0, ta), min(t1, tb)
    return max(t1 - t0, 0.0)


def small_geom(nx=16, ny=16, pixel=1.25, V=24, C=20, **kw):
    return oracle.Geometry(nx=nx, ny=ny, pixel_mm=pixel, n_views=V, n_channels=C, sad_mm=kw.pop("sad", 90.0), **kw)


@pytest.mark.parametrize("theta0,off", [(0.0, 0.0), (0.3, 0.25)])
def test_P1_weight_vs_polygon_clipping(theta0, off):
    g = small_geom(theta0_rad=theta0, channel_offset=off)
    worst = 0.0
    nz = 0
    for v in range(g.n_views):
        for c in range(g.n_channels):
            sx, sy, dx, dy = oracle.ray(g, v, c)
            for iy in range(g.ny):
                for ix in range(g.nx):
                    cx = (ix - (g.nx - 1) / 2) * g.pixel_mm
                    cy = (iy - (g.ny - 1) / 2) * g.pixel_mm
                    h = g.pixel_mm / 2
                    ref = clip_length(sx, sy, dx, dy, cx - h, cx + h, cy - h, cy + h)
                    a = oracle.weight(g, v, c, ix, iy)
                    worst = max(worst, abs(a - ref))
                    nz += ref > 0
    assert nz > 5000
    assert worst < 1e-11


def test_P1_ray_geometry_convention():
    # C1: source on the circle of radius SAD at angle theta_v; central ray (gamma=0) points at the isocentre;
    # distance of ray (v,c) from the isocentre is SAD*|sin gamma_c| for every view
    g = small_geom(C=21)
    dg = oracle.dgamma(g)
    assert dg == pytest.approx(2 * np.arcsin(0.5 * 16 * 1.25 / 90.0) / 21, rel=1e-14)
    for v in (0, 5, 13):
        th = 2 * np.pi * v / g.n_views
        for c in (0, 10, 20):
            sx, sy, dx, dy = oracle.ray(g, v, c)
            assert sx == pytest.approx(90.0 * np.cos(th), abs=1e-12)
            assert sy == pytest.approx(90.0 * np.sin(th), abs=1e-12)
            assert dx * dx + dy * dy == pytest.approx(1.0, abs=1e-14)
            dist = abs(sx * dy - sy * dx)
            assert dist == pytest.approx(90.0 * abs(np.sin((c - 10) * dg)), abs=1e-11)
            if c == 10:
                assert dx == pytest.approx(-np.cos(th), abs=1e-14) and dy == pytest.approx(-np.sin(th), abs=1e-14)


@pytest.mark.parametrize("shape", [(16, 16), (20, 12)])
def test_P2_forward_of_ones_is_chord_through_grid(shape):
    nx, ny = shape
    g = small_geom(nx=nx, ny=ny, V=36, C=40, theta0_rad=0.1)
    l = oracle.forward(g, np.ones((ny, nx)))
    ref = np.zeros_like(l)
    for v in range(g.n_views):
        for c in range(g.n_channels):
            sx, sy, dx, dy = oracle.ray(g, v, c)
            ref[v, c] = clip_length(sx, sy, dx, dy, -nx * g.pixel_mm / 2, nx * g.pixel_mm / 2,
                                    -ny * g.pixel_mm / 2, ny * g.pixel_mm / 2)
    assert ref.max() > 10
    assert np.abs(l - ref).max() < 1e-11


def test_P3_forward_vs_analytic_ellipses_error_falls_with_pixel_size():
    errs = []
    for n in (32, 64, 128):
        cfg = si.ScanConfig("t", n, n, 64.0 / n, 60, 96, seed=77, n_ellipses=4)
        ell = si.draw_ellipses(cfg, cfg.seed)
        exact = si.ellipse_sinogram(cfg, ell)
        g = oracle.Geometry(nx=n, ny=n, pixel_mm=cfg.pixel_mm, n_views=60, n_channels=96)
        l = oracle.forward(g, si.rasterize(cfg, ell))
        errs.append(np.linalg.norm(l - exact) / np.linalg.norm(exact))
    assert errs[0] < 0.03 and errs[2] < 0.008
    assert errs[0] > errs[1] > errs[2]
    assert errs[2] < 0.6 * errs[0]


@pytest.mark.parametrize("subset,M", [(-1, 1), (1, 3), (0, 2)])
def test_P4_adjoint_identity_and_brute_force(subset, M):
    rng = np.random.default_rng(5)
    g = small_geom(nx=18, ny=14, V=24, C=22, theta0_rad=0.05, channel_offset=0.25)
    nv = g.n_views if subset < 0 else g.n_views // M
    x = rng.uniform(size=(g.ny, g.nx))
    y = rng.uniform(size=(nv, g.n_channels))
    Ax = oracle.forward(g, x, subset, M)
    Aty = oracle.backward(g, y, subset, M)
    lhs, rhs = float((Ax * y).sum()), float((x * Aty).sum())
    assert abs(lhs - rhs) / abs(lhs) < 1e-12
    assert np.abs(Ax - oracle.forward_brute(g, x, subset, M)).max() < 1e-11
    assert np.abs(Aty - oracle.backward_brute(g, y, subset, M)).max() < 1e-11


def test_P4_adjoint_identity_config1_geometry():
    cfg = si.scan_config("1")
    g = oracle.Geometry(nx=cfg.nx, ny=cfg.ny, pixel_mm=cfg.pixel_mm, n_views=cfg.n_views, n_channels=cfg.n_channels)
    rng = np.random.default_rng(6)
    x = rng.uniform(size=(g.ny, g.nx))
    y = rng.uniform(size=(g.n_views, g.n_channels))
    lhs = float((oracle.forward(g, x) * y).sum())
    rhs = float((x * oracle.backward(g, y)).sum())
    assert abs(lhs - rhs) / abs(lhs) < 1e-12


def test_P4_subsets_partition_the_views():
    # C11 / PAPER.md:118: S_m = {v : v mod M = m}; the M subset projections interleave to the full one
    g = small_geom(V=24, C=20)
    x = np.random.default_rng(1).uniform(size=(g.ny, g.nx))
    full = oracle.forward(g, x)
    M = 4
    for m in range(M):
        assert np.array_equal(oracle.forward(g, x, m, M), full[m::M])
    y = np.random.default_rng(2).uniform(size=full.shape)
    acc = sum(oracle.backward(g, y[m::M].copy(), m, M) for m in range(M))
    assert np.abs(acc - oracle.backward(g, y)).max() < 1e-11


def test_P5_rotation_and_mirror_symmetry():
    g = small_geom(nx=24, ny=24, V=16, C=20)
    x = np.random.default_rng(3).uniform(size=(24, 24))
    l = oracle.forward(g, x)
    # rotate the object by +90 deg about the grid centre: new[iy, ix] = old[n-1-ix, iy]  (x' = -y, y' = x)
    xr = np.empty_like(x)
    for iy in range(24):
        for ix in range(24):
            xr[iy, ix] = x[23 - ix, iy]
    lr = oracle.forward(g, xr)
    d_plus = np.abs(lr - np.roll(l, +4, axis=0)).max()     # object turned +90 deg == views advanced by V/4
    d_minus = np.abs(lr - np.roll(l, -4, axis=0)).max()
    assert min(d_plus, d_minus) < 1e-10 and max(d_plus, d_minus) > 1e-2
    assert d_plus < 1e-10
    # mirror in y: ray (v,c) -> ((V-v) mod V, C-1-c)
    lm = oracle.forward(g, x[::-1, :].copy())
    ref = l[(-np.arange(16)) % 16][:, ::-1]
    assert np.abs(lm - ref).max() < 1e-10


def test_P8_step_scale_bounds_the_subset_hessian():
    # C6: L_geo = V_S N Delta^3 / delta_iso bounds ||A_S^T A_S||; SURVEY SCRATCH saw 0.957-0.962
    for (n, V, C, M) in ((32, 48, 48, 1), (32, 60, 64, 3)):
        g = oracle.Geometry(nx=n, ny=n, pixel_mm=1.0, n_views=V, n_channels=C, sad_mm=850.0)
        x = np.random.default_rng(0).uniform(size=(n, n))
        lam = 0.0
        for _ in range(40):
            x /= np.linalg.norm(x)
            y = oracle.backward(g, oracle.forward(g, x, 0, M), 0, M)
            lam = float((x * y).sum())
            x = y
        L_geo = (V // M) * n * 1.0 ** 3 / (850.0 * oracle.dgamma(g))
        assert 0.9 < lam / L_geo < 1.0
        assert oracle.tau(g, M, 100.0) == pytest.approx(100.0 / L_geo, rel=1e-13)


def test_candidate_range_is_complete():
    # the gather backprojector's K must cover every touching channel: compare with brute force on a
    # geometry with a short SAD (strong fan divergence) and a non-square grid
    g = oracle.Geometry(nx=12, ny=20, pixel_mm=2.0, n_views=20, n_channels=64, sad_mm=30.0, channel_offset=-0.4)
    y = np.random.default_rng(4).uniform(size=(20, 64))
    assert np.abs(oracle.backward(g, y) - oracle.backward_brute(g, y)).max() < 1e-11
