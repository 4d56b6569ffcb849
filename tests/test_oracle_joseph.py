"""Pins of the oracle's second system matrix (model = 1, Joseph's interpolating projector; SURVEY.md 8(f)-2,
DESIGN.md section 3 reading J1); CPU only.

Each check compares the oracle with something that is not the oracle: the textbook definition of Joseph's method
written out here (sample the image by linear interpolation on every line of the ray's major axis), the partition of
unity of the interpolation weights, analytic ellipse integrals, the adjoint identity between the ray loop and the
pixel gather, brute force over all (ray, pixel) pairs, and the scan's symmetries.
"""
import numpy as np
import pytest

import oracle
import synth_inputs as si


def geom(nx=16, ny=16, pixel=1.25, V=24, C=20, **kw):
    return oracle.Geometry(nx=nx, ny=ny, pixel_mm=pixel, n_views=V, n_channels=C, sad_mm=kw.pop("sad", 90.0), model=1, **kw)


def joseph_by_definition(g, img):
    """Joseph (1982): march along the major axis, one sample per image line at the line's centre, linear interpolation
    between the two neighbouring pixel centres of that line (zero outside the grid), step length D/max(|dx|,|dy|)."""
    out = np.zeros((g.n_views, g.n_channels))
    D = g.pixel_mm
    xs = (np.arange(g.nx) - 0.5 * (g.nx - 1)) * D
    ys = (np.arange(g.ny) - 0.5 * (g.ny - 1)) * D
    for v in range(g.n_views):
        for c in range(g.n_channels):
            sx, sy, dx, dy = oracle.ray(g, v, c)
            acc = 0.0
            if abs(dy) >= abs(dx):
                for iy in range(g.ny):
                    x = sx + (ys[iy] - sy) / dy * dx
                    f = (x - xs[0]) / D                     # position in pixel-centre units
                    i0 = int(np.floor(f))
                    w1 = f - i0
                    for i, w in ((i0, 1.0 - w1), (i0 + 1, w1)):
                        if 0 <= i < g.nx:
                            acc += w * img[iy, i]
                acc *= D / abs(dy)
            else:
                for ix in range(g.nx):
                    y = sy + (xs[ix] - sx) / dx * dy
                    f = (y - ys[0]) / D
                    i0 = int(np.floor(f))
                    w1 = f - i0
                    for i, w in ((i0, 1.0 - w1), (i0 + 1, w1)):
                        if 0 <= i < g.ny:
                            acc += w * img[i, ix]
                acc *= D / abs(dx)
            out[v, c] = acc
    return out


@pytest.mark.parametrize("theta0,off", [(0.0, 0.0), (0.3, 0.25)])
def test_J1_forward_is_josephs_definition(theta0, off):
    g = geom(nx=14, ny=18, theta0_rad=theta0, channel_offset=off)
    x = np.random.default_rng(11).uniform(size=(g.ny, g.nx))
    assert np.abs(oracle.forward(g, x) - joseph_by_definition(g, x)).max() < 1e-11


def test_J1_weight_differs_from_the_exact_chord_and_is_a_tent():
    g = geom()
    g0 = oracle.Geometry(nx=g.nx, ny=g.ny, pixel_mm=g.pixel_mm, n_views=g.n_views, n_channels=g.n_channels, sad_mm=g.sad_mm)
    v, c = 0, 9                                  # nearly axis-aligned: box (exact chord) against tent (Joseph)
    sx, sy, dx, dy = oracle.ray(g, v, c)
    m = max(abs(dx), abs(dy))
    diff = 0.0
    for iy in range(g.ny):
        for ix in range(g.nx):
            px, py = (ix - 0.5 * (g.nx - 1)) * g.pixel_mm, (iy - 0.5 * (g.ny - 1)) * g.pixel_mm
            p = (px - sx) * dy - (py - sy) * dx
            want = g.pixel_mm / m * max(0.0, 1.0 - abs(p) / (g.pixel_mm * m))
            assert abs(oracle.weight(g, v, c, ix, iy) - want) < 1e-13
            diff = max(diff, abs(oracle.weight(g, v, c, ix, iy) - oracle.weight(g0, v, c, ix, iy)))
    assert diff > 0.05 * g.pixel_mm


def test_J2_partition_of_unity():
    # a ray whose crossings all lie between the first and the last pixel centre of every line sees weights that sum to
    # h per line: A.1 = (number of lines) * D / max(|dx|,|dy|)
    g = geom(nx=40, ny=40, pixel=1.0, V=4, C=6, sad=200.0, dgamma_rad=0.004, theta0_rad=0.1)
    l = oracle.forward(g, np.ones((g.ny, g.nx)))
    for v in range(g.n_views):
        for c in range(g.n_channels):
            sx, sy, dx, dy = oracle.ray(g, v, c)
            assert abs(l[v, c] - 40 * 1.0 / max(abs(dx), abs(dy))) < 1e-10


def test_J3_forward_vs_analytic_ellipses_error_falls_with_pixel_size():
    errs = []
    for n in (32, 64, 128):
        cfg = si.ScanConfig("t", n, n, 64.0 / n, 60, 96, seed=77, n_ellipses=4)
        ell = si.draw_ellipses(cfg, cfg.seed)
        exact = si.ellipse_sinogram(cfg, ell)
        g = oracle.Geometry(nx=n, ny=n, pixel_mm=cfg.pixel_mm, n_views=60, n_channels=96, model=1)
        l = oracle.forward(g, si.rasterize(cfg, ell))
        errs.append(np.linalg.norm(l - exact) / np.linalg.norm(exact))
    assert errs[0] < 0.03 and errs[2] < 0.008
    assert errs[0] > errs[1] > errs[2]


@pytest.mark.parametrize("subset,M", [(-1, 1), (1, 3)])
def test_J4_adjoint_identity_and_brute_force(subset, M):
    rng = np.random.default_rng(5)
    g = geom(nx=18, ny=14, V=24, C=22, theta0_rad=0.05, channel_offset=0.25)
    nv = g.n_views if subset < 0 else g.n_views // M
    x = rng.uniform(size=(g.ny, g.nx))
    y = rng.uniform(size=(nv, g.n_channels))
    Ax = oracle.forward(g, x, subset, M)
    Aty = oracle.backward(g, y, subset, M)
    lhs, rhs = float((Ax * y).sum()), float((x * Aty).sum())
    assert abs(lhs - rhs) / abs(lhs) < 1e-12
    assert np.abs(Ax - oracle.forward_brute(g, x, subset, M)).max() < 1e-11
    assert np.abs(Aty - oracle.backward_brute(g, y, subset, M)).max() < 1e-11


def test_J4_candidate_range_is_complete_for_the_wider_footprint():
    g = oracle.Geometry(nx=12, ny=20, pixel_mm=2.0, n_views=20, n_channels=64, sad_mm=30.0, channel_offset=-0.4, model=1)
    y = np.random.default_rng(4).uniform(size=(20, 64))
    assert np.abs(oracle.backward(g, y) - oracle.backward_brute(g, y)).max() < 1e-11


def test_J5_rotation_symmetry():
    g = geom(nx=24, ny=24, V=16, C=20)
    x = np.random.default_rng(3).uniform(size=(24, 24))
    l = oracle.forward(g, x)
    xr = np.empty_like(x)
    for iy in range(24):
        for ix in range(24):
            xr[iy, ix] = x[23 - ix, iy]
    assert np.abs(oracle.forward(g, xr) - np.roll(l, +4, axis=0)).max() < 1e-10


def test_J6_iteration_runs_and_converges_noise_free():
    # the loop is model-agnostic: noise-free, beta = 0 data made with the Joseph matrix are fitted by it
    cfg = si.ScanConfig("t", 16, 16, 1.25, 48, 32, i0=1e5, seed=21, n_ellipses=3, sad_mm=90.0)
    g = oracle.Geometry(nx=16, ny=16, pixel_mm=1.25, n_views=48, n_channels=32, sad_mm=90.0, model=1)
    truth = si.rasterize(cfg, si.draw_ellipses(cfg, cfg.seed))
    counts = cfg.i0 * np.exp(-oracle.forward(g, truth))
    img, trace, status = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=0.0, n_subsets=1, n_iters=2000))
    yy, xx = np.mgrid[0:16, 0:16] - 7.5
    inside = (xx ** 2 + yy ** 2) < (0.8 * 8) ** 2         # the corners lie outside the fan and are not determined
    err = np.linalg.norm((img - truth)[inside]) / np.linalg.norm(truth[inside])
    assert status == 0 and trace[-1, 0] < 1e-20 * trace[0, 0] and err < 1e-10
