"""GPU parity tests (run with -m gpu on the B200): the CUDA path, called through the C ABI, against the
float64 oracle on the same seeded inputs.

Bars (BASELINE.json north_star): projector outputs within 1e-5 relative L2, the
reconstructed image within 1e-3 relative L2; lambda traces are compared exactly (both sides keep lambda and
D in float64 and no decision flips are expected below the stability limit); the monitor D
within 1e-5 relative (float32 line integrals, float64 accumulation)."""
import numpy as np
import pytest

import oracle
import synth_inputs as si

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

PROJ_TOL = 1e-5
IMG_TOL = 1e-3


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def geoms(cfg):
    import paper_1903_10088_b200 as osiv
    og = oracle.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.dgamma_rad,
                         cfg.channel_offset, cfg.theta0_rad)
    gg = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm,
                       cfg.dgamma_rad, cfg.channel_offset, cfg.theta0_rad)
    return og, gg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    return t.detach().cpu().numpy()


ODD = si.ScanConfig("odd", 37, 29, 1.3, 24, 45, sad_mm=120.0, theta0_rad=0.3, channel_offset=0.25, seed=7)
WIDE = si.ScanConfig("wide", 48, 40, 2.0, 30, 70, sad_mm=75.0, seed=8)           # wide fan: atanf branch
TINY = si.ScanConfig("tiny", 3, 5, 1.0, 4, 3, sad_mm=20.0, seed=9)
SYM = si.ScanConfig("sym", 36, 36, 1.3, 24, 45, sad_mm=120.0, theta0_rad=0.3, channel_offset=0.25, seed=11)  # quarter-turn path
NEAR_AXIS = si.ScanConfig("axis", 64, 64, 1.0, 90, 97, theta0_rad=1e-7, seed=10)  # G10: central ray ~ on pixel edges


@pytest.fixture(scope="module")
def osiv():
    import paper_1903_10088_b200 as m
    assert torch.cuda.is_available()
    m.lib()                      # raises if libosiv.so is missing: there is no fallback
    return m


# ------------------------------------------------------------------ projector pair

@pytest.mark.parametrize("cfg,subsets", [
    (si.scan_config("1"), [(-1, 1), (0, 3), (2, 3)]),
    (ODD, [(-1, 1), (1, 2), (5, 6)]),
    (WIDE, [(-1, 1), (4, 5)]),
    (TINY, [(-1, 1), (1, 2)]),
    (si.scan_config("2"), [(-1, 1), (7, 10)]),
    (SYM, [(-1, 1), (1, 2), (2, 3), (0, 4)]),          # V_S = 24, 12, 8 take the quarter-turn kernels, V_S = 6 the general
], ids=["config1", "odd", "wide", "tiny", "config2", "sym"])
def test_forward_and_back_match_oracle(osiv, cfg, subsets):
    og, gg = geoms(cfg)
    rng = np.random.default_rng(cfg.seed)
    img = rng.uniform(0.0, 0.013, size=(cfg.ny, cfg.nx)).astype(np.float32)
    with osiv.Handle(gg, max_batch=1) as h:
        for sub, M in subsets:
            ref = oracle.forward(og, img, sub, M)
            got = host(h.forward(dev(img)[None], sub, M))[0]
            assert got.shape == ref.shape
            assert rel(got, ref) < PROJ_TOL, (cfg.name, sub, M)
            sino = rng.uniform(0.0, 1.0, size=ref.shape).astype(np.float32)
            refb = oracle.backward(og, sino, sub, M)
            gotb = host(h.backward(dev(sino)[None], sub, M))[0]
            assert rel(gotb, refb) < PROJ_TOL, (cfg.name, sub, M)
            # fp32 adjoint identity <Ax,y> = <x,A^T y>, dot products in float64 (oracle bound is 1e-12, P4)
            lhs = np.dot(got.astype(np.float64).ravel(), sino.astype(np.float64).ravel())
            rhs = np.dot(img.astype(np.float64).ravel(), gotb.astype(np.float64).ravel())
            assert abs(lhs - rhs) / abs(lhs) < 2e-6


def test_quarter_turn_path_is_taken_and_agrees_with_the_general_path(osiv):
    """The NS = 4 kernels (one chord weight per quarter-turn orbit) against the NS = 1 kernels on the same inputs:
    equal up to float32 rounding, and the plan reports which one runs."""
    for cfg, sub, M in [(SYM, 1, 2), (si.scan_config("2"), 7, 10), (si.scan_config("2"), -1, 1)]:
        _, gg = geoms(cfg)
        rng = np.random.default_rng(cfg.seed + 1)
        img = rng.uniform(0.0, 0.013, size=(2, cfg.ny, cfg.nx)).astype(np.float32)
        vs = cfg.n_views if sub < 0 else cfg.n_views // M
        sino = rng.uniform(0.0, 1.0, size=(2, vs, cfg.n_channels)).astype(np.float32)
        with osiv.Handle(gg, max_batch=2) as h:
            plan = h.plan(M if sub >= 0 else 0, 2)
            assert plan["k1_orbit"] == 4 and plan["k2_orbit"] == 4
            f4, b4 = host(h.forward(dev(img), sub, M)), host(h.backward(dev(sino), sub, M))
            h.set_symmetry(False)
            plan = h.plan(M if sub >= 0 else 0, 2)
            assert plan["k1_orbit"] == 1 and plan["k2_orbit"] == 1
            f1, b1 = host(h.forward(dev(img), sub, M)), host(h.backward(dev(sino), sub, M))
        assert rel(f4, f1) < 2e-6 and rel(b4, b1) < 2e-6
    _, gg = geoms(si.scan_config("1"))                  # V = 90: no quarter-turn orbits
    with osiv.Handle(gg, max_batch=1) as h:
        assert h.plan(1, 1)["k1_orbit"] == 1


SYM8 = si.ScanConfig("sym8", 40, 40, 1.3, 24, 45, sad_mm=120.0, theta0_rad=0.3, channel_offset=0.25, seed=12)   # side % 8 == 0: staged K2
SYM64 = si.ScanConfig("sym64", 64, 64, 1.0, 88, 97, theta0_rad=0.05, seed=13)


@pytest.mark.parametrize("cfg,subsets,model", [
    (SYM8, [(-1, 1), (1, 2), (2, 3)], 0),                 # V_S = 24, 12, 8
    (SYM64, [(-1, 1), (3, 11), (1, 2)], 0),               # V_S = 88 (several staging rounds), 8, 44
    (si.scan_config("2"), [(-1, 1), (7, 10)], 0),         # all 400 views: 100 base views in rounds; 40 views: one round
    (SYM64, [(-1, 1), (0, 2)], 1),                        # Joseph's matrix through the same kernel
], ids=["sym8", "sym64", "config2", "sym64-joseph"])
def test_staged_back_kernel_matches_oracle_and_general_kernel(osiv, cfg, subsets, model):
    """K2 with its windows staged in shared memory (csrc/osiv_back_staged.cuh: 4 x 2 tiles, 8-byte ray entries with a
    per-window orientation flag, bulk-copied constants) against the oracle's A^T and against the general gather K2."""
    og = oracle.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.dgamma_rad,
                         cfg.channel_offset, cfg.theta0_rad, model=model)
    gg = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm,
                       cfg.dgamma_rad, cfg.channel_offset, cfg.theta0_rad, model=model)
    rng = np.random.default_rng(cfg.seed + 5)
    with osiv.Handle(gg, max_batch=3) as h:
        for sub, M in subsets:
            vs = cfg.n_views if sub < 0 else cfg.n_views // M
            sino = rng.uniform(0.0, 1.0, size=(3, vs, cfg.n_channels)).astype(np.float32)
            h.set_back_kernel(staged_rounds=True)                 # also the subsets that take several staging rounds
            assert h.back_kernel(M if sub >= 0 else 0, 3) == "staged"
            got = host(h.backward(dev(sino), sub, M))
            h.set_back_kernel(general_only=True)
            assert h.back_kernel(M if sub >= 0 else 0, 3) == "general"
            gen = host(h.backward(dev(sino), sub, M))
            h.set_back_kernel(staged_rounds=True)
            for s in range(3):
                assert rel(got[s], oracle.backward(og, sino[s], sub, M)) < PROJ_TOL, (cfg.name, sub, M, s)
            assert rel(got, gen) < 2e-6
            again = host(h.backward(dev(sino), sub, M))
            assert np.array_equal(got, again)                     # no atomics on data, fixed-order sums


@pytest.mark.parametrize("N,V,C", [(8, 8, 13), (16, 12, 25), (24, 16, 40), (72, 20, 101), (136, 24, 190)])
def test_staged_back_kernel_region_partition_edge_sizes(osiv, N, V, C):
    """The staged K2's block regions on small and awkward grids (one or two tiles in all, fewer regions than SMs, rows of
    regions of unequal height): backprojection and a short reconstruction against the oracle."""
    cfg = si.ScanConfig(f"edge{N}", N, N, 1.1, V, C, sad_mm=max(120.0, 2.0 * N), theta0_rad=0.11, channel_offset=-0.3, seed=100 + N,
                        i0=5e4, n_subsets=1, n_iters=6, betas=(0.01,))
    og, gg = geoms(cfg)
    rng = np.random.default_rng(cfg.seed)
    with osiv.Handle(gg, max_batch=2) as h:
        h.set_back_kernel(staged_rounds=True)
        assert h.back_kernel(0, 2) == "staged"
        sino = rng.uniform(0.0, 1.0, size=(2, V, C)).astype(np.float32)
        got = host(h.backward(dev(sino)))
        for s in range(2):
            assert rel(got[s], oracle.backward(og, sino[s])) < PROJ_TOL
        _, _, counts = si.make_case(cfg)
        prm = dict(beta=0.01, n_subsets=1, n_iters=6)
        img, tr = h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(**prm), trace=True)
        ref, tr_ref, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(**prm))
        assert np.array_equal(tr[0, :, 1], tr_ref[:, 1])
        assert rel(host(img)[0], ref) < IMG_TOL


def test_staged_back_kernel_in_the_iteration(osiv):
    """The whole iteration with the staged K2 against the general K2 (same K1): equal lambda traces, images equal to
    rounding order; with return_best, a per-channel blank scan and three slices per launch."""
    cfg = si.scan_config("2")
    _, gg = geoms(cfg)
    counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(3)])
    blank = (cfg.i0 * (1.0 + 0.05 * np.cos(np.arange(cfg.n_channels)))).astype(np.float32)
    prm = osiv.Params(beta=0.005, n_subsets=10, n_iters=40, return_best=1)
    with osiv.Handle(gg, max_batch=3) as h:
        assert h.back_kernel(10, 3) == "staged"
        a, ta = h.reconstruct(dev(counts), dev(blank), prm, trace=True)
        h.set_back_kernel(general_only=True)
        b, tb = h.reconstruct(dev(counts), dev(blank), prm, trace=True)
    a, b = host(a), host(b)
    assert np.array_equal(ta[:, :, 1], tb[:, :, 1])
    assert np.allclose(ta[:, :, 0], tb[:, :, 0], rtol=1e-5)
    assert rel(a, b) < 5e-6


def test_projector_near_axis_rays(osiv):
    """G10 stress: theta0 = 1e-7 puts the central ray of views 0 and V/2 (and, with V = 4k, V/4 and 3V/4) within
    1e-7 rad of a pixel edge.  The chord of such a ray is a ramp 1e-7 pixel wide, which float32 positions
    (ulp(32) = 4e-6 pixel) cannot resolve: the result stays finite and the damage is confined to those rays."""
    cfg = NEAR_AXIS
    og, gg = geoms(cfg)
    rng = np.random.default_rng(cfg.seed)
    img = rng.uniform(0.0, 0.013, size=(cfg.ny, cfg.nx)).astype(np.float32)
    _, _, dx, dy = si.ray_geometry(cfg)
    ok = np.minimum(np.abs(dx), np.abs(dy)) > 1e-4
    assert 0 < (~ok).sum() < 40
    with osiv.Handle(gg, max_batch=1) as h:
        ref = oracle.forward(og, img)
        got = host(h.forward(dev(img)[None]))[0]
        assert np.all(np.isfinite(got))
        assert rel(got[ok], ref[ok]) < PROJ_TOL
        assert np.abs(got - ref).max() < 0.013 * 2.0 * cfg.pixel_mm      # at most ~two pixels' worth on a bad ray
        sino = rng.uniform(0.0, 1.0, size=ref.shape).astype(np.float32) * ok
        gotb = host(h.backward(dev(sino)[None]))[0]
        assert rel(gotb, oracle.backward(og, sino)) < PROJ_TOL


def test_projector_degenerate_inputs(osiv):
    cfg = ODD
    og, gg = geoms(cfg)
    with osiv.Handle(gg, max_batch=2) as h:
        z = torch.zeros((2, cfg.ny, cfg.nx), device="cuda")
        assert float(h.forward(z).abs().max()) == 0.0
        zs = torch.zeros((2, cfg.n_views, cfg.n_channels), device="cuda")
        assert float(h.backward(zs).abs().max()) == 0.0
        # A*1 = chord of each ray through the whole grid rectangle (P2), a single-pixel image = one matrix column
        ones = np.ones((cfg.ny, cfg.nx), dtype=np.float32)
        assert rel(host(h.forward(dev(ones)[None]))[0], oracle.forward(og, ones)) < PROJ_TOL
        e = np.zeros((cfg.ny, cfg.nx), dtype=np.float32)
        e[cfg.ny - 1, 0] = 1.0
        got = host(h.forward(dev(e)[None]))[0]
        ref = np.array([[oracle.weight(og, v, c, 0, cfg.ny - 1) for c in range(cfg.n_channels)]
                        for v in range(cfg.n_views)])
        assert np.abs(got - ref).max() < 2e-5 * cfg.pixel_mm
        # single-ray sinogram = one matrix row, scattered by the gather backprojector
        s1 = np.zeros((cfg.n_views, cfg.n_channels), dtype=np.float32)
        s1[5, 20] = 1.0
        gotb = host(h.backward(dev(s1)[None]))[0]
        refb = np.array([[oracle.weight(og, 5, 20, ix, iy) for ix in range(cfg.nx)] for iy in range(cfg.ny)])
        assert np.abs(gotb - refb).max() < 2e-5 * cfg.pixel_mm


def test_batched_projectors_equal_single_slice_calls_bitwise(osiv):
    cfg = ODD
    _, gg = geoms(cfg)
    rng = np.random.default_rng(3)
    imgs = rng.uniform(0.0, 0.013, size=(3, cfg.ny, cfg.nx)).astype(np.float32)
    sinos = rng.uniform(0.0, 1.0, size=(3, cfg.n_views // 2, cfg.n_channels)).astype(np.float32)
    with osiv.Handle(gg, max_batch=3) as h:
        fb = host(h.forward(dev(imgs), 1, 2))
        bb = host(h.backward(dev(sinos), 1, 2))
        for s in range(3):
            assert np.array_equal(fb[s], host(h.forward(dev(imgs[s:s + 1]), 1, 2))[0])
            assert np.array_equal(bb[s], host(h.backward(dev(sinos[s:s + 1]), 1, 2))[0])


def test_projector_pair_full_size_config5a(osiv):
    """512x512, 800 x 738: the launch configuration bench.py times; the oracle needs ~2 s for it."""
    cfg = si.scan_config("5a")
    og, gg = geoms(cfg)
    img = si.uniform_image(cfg)
    with osiv.Handle(gg, max_batch=1) as h:
        ref = oracle.forward(og, img)
        got = host(h.forward(dev(img)[None]))[0]
        assert rel(got, ref) < PROJ_TOL
        sino = si.uniform_sinogram(cfg)
        refb = oracle.backward(og, sino)
        gotb = host(h.backward(dev(sino)[None]))[0]
        assert rel(gotb, refb) < PROJ_TOL
        lhs = np.dot(got.astype(np.float64).ravel(), sino.astype(np.float64).ravel())
        rhs = np.dot(img.astype(np.float64).ravel(), gotb.astype(np.float64).ravel())
        assert abs(lhs - rhs) / abs(lhs) < 2e-6
        # one 40-view subset (the per-iteration launch of config 3)
        ref = oracle.forward(og, img, 3, 20)
        assert rel(host(h.forward(dev(img)[None], 3, 20))[0], ref) < PROJ_TOL
        s40 = si.uniform_sinogram(cfg, n_views=40)
        assert rel(host(h.backward(dev(s40)[None], 3, 20))[0], oracle.backward(og, s40, 3, 20)) < PROJ_TOL


def test_projector_pair_max_size_config5b_subset(osiv):
    """1024x1024, 1600 x 1476 (the largest configuration): one 40-view subset against the oracle, plus sampled
    rays / pixels of the all-view operators computed one by one from oracle.weight."""
    cfg = si.scan_config("5b")
    og, gg = geoms(cfg)
    img = si.uniform_image(cfg)
    with osiv.Handle(gg, max_batch=1) as h:
        ref = oracle.forward(og, img, 7, 40)
        assert rel(host(h.forward(dev(img)[None], 7, 40))[0], ref) < PROJ_TOL
        s40 = si.uniform_sinogram(cfg, n_views=40)
        assert rel(host(h.backward(dev(s40)[None], 7, 40))[0], oracle.backward(og, s40, 7, 40)) < PROJ_TOL
        full = host(h.forward(dev(img)[None]))[0]
        rng = np.random.default_rng(0)
        for v, c in zip(rng.integers(0, cfg.n_views, 6), rng.integers(0, cfg.n_channels, 6)):
            one = oracle.forward(og, img, int(v), cfg.n_views)          # subset {v} of V subsets = a single view
            assert abs(full[v, c] - one[0, c]) < 2e-5 * abs(one[0, c]) + 1e-7


# ------------------------------------------------------------------ second system matrix (Joseph, 8(f)-2)
@pytest.mark.parametrize("cfg,subsets", [
    (si.scan_config("1"), [(-1, 1), (2, 5)]),           # general path (V = 90)
    (si.scan_config("2"), [(-1, 1), (3, 10)]),          # quarter-turn path
    (ODD, [(-1, 1), (1, 3)]),
    (WIDE, [(-1, 1)]),
    (NEAR_AXIS, [(-1, 1)]),
])
def test_joseph_model_forward_and_back_match_oracle(osiv, cfg, subsets):
    from dataclasses import replace
    og, gg = geoms(cfg)
    og, gg = replace(og, model=1), replace(gg, model=1)
    rng = np.random.default_rng(cfg.seed + 5)
    with osiv.Handle(gg, max_batch=1) as h:
        for sub, M in subsets:
            img = rng.uniform(0.0, 0.013, size=(cfg.ny, cfg.nx)).astype(np.float32)
            vs = cfg.n_views if sub < 0 else cfg.n_views // M
            sino = rng.uniform(0.0, 1.0, size=(vs, cfg.n_channels)).astype(np.float32)
            f = host(h.forward(dev(img)[None], sub, M))[0]
            b = host(h.backward(dev(sino)[None], sub, M))[0]
            assert rel(f, oracle.forward(og, img, sub, M)) < PROJ_TOL
            assert rel(b, oracle.backward(og, sino, sub, M)) < PROJ_TOL
            lhs = np.dot(f.astype(np.float64).ravel(), sino.astype(np.float64).ravel())
            rhs = np.dot(img.astype(np.float64).ravel(), b.astype(np.float64).ravel())
            assert abs(lhs - rhs) / abs(lhs) < 5e-6


def test_joseph_model_reconstruct_config2(osiv):
    from dataclasses import replace
    cfg = si.scan_config("2")
    og, gg = geoms(cfg)
    og, gg = replace(og, model=1), replace(gg, model=1)
    counts = si.make_case(cfg)[2]
    kw = dict(beta=cfg.betas[0], n_subsets=cfg.n_subsets, n_iters=cfg.n_iters)
    ref, tr_ref, status = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(**kw))
    with osiv.Handle(gg, max_batch=1) as h:
        got, tr = h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(**kw), trace=True)
    assert status == 0 and np.array_equal(tr[0, :, 1], tr_ref[:, 1])
    assert np.all(np.abs(tr[0, :, 0] - tr_ref[:, 0]) <= 1e-5 * tr_ref[:, 0])
    assert rel(host(got)[0], ref) < IMG_TOL


# ------------------------------------------------------------------ TV gradient

@pytest.mark.parametrize("shape", [(29, 37), (64, 64), (5, 3), (1, 7)])
def test_tv_gradient_matches_oracle(osiv, shape):
    ny, nx = shape
    gg = osiv.Geometry(nx, ny, 1.0, 8, 8, sad_mm=200.0)
    rng = np.random.default_rng(11)
    img = (0.007 + 1e-4 * rng.standard_normal((ny, nx))).astype(np.float32)
    if ny > 8 and nx > 8:
        img[2:6, 3:8] = 0.007                                           # flat patch: t = eps
    with osiv.Handle(gg, max_batch=1) as h:
        for eps in (1e-5, 1e-3):
            ref = oracle.tv_grad(img, eps)
            got = host(h.tv_gradient(dev(img)[None], eps))[0]
            assert rel(got, ref) < 5e-6
        const = np.full((ny, nx), 0.005, dtype=np.float32)
        assert float(h.tv_gradient(dev(const)[None], 1e-5).abs().max()) == 0.0


# ------------------------------------------------------------------ the iteration

def run_pair(osiv, cfg, prm_kw, blank=None, batch_counts=None):
    og, gg = geoms(cfg)
    ell, sino, counts = si.make_case(cfg)
    b = cfg.i0 if blank is None else blank
    ref, tr_ref, st = oracle.reconstruct(og, counts, b, oracle.Params(**prm_kw))
    with osiv.Handle(gg, max_batch=1) as h:
        bd = b if np.isscalar(b) else dev(b)
        got, tr = h.reconstruct(dev(counts)[None], bd, osiv.Params(**prm_kw), trace=True)
    return host(got)[0], tr[0], ref, tr_ref, st


def check_run(got, tr, ref, tr_ref, exact_lambda=True):
    assert rel(got, ref) < IMG_TOL
    assert np.all(np.abs(tr[:, 0] - tr_ref[:, 0]) <= 1e-5 * tr_ref[:, 0])
    if exact_lambda:
        assert np.array_equal(tr[:, 1], tr_ref[:, 1])
    assert got.min() >= 0.0


def test_reconstruct_config1(osiv):
    cfg = si.scan_config("1")
    got, tr, ref, tr_ref, st = run_pair(osiv, cfg, dict(beta=0.01, n_subsets=1, n_iters=10))
    assert st == 0
    check_run(got, tr, ref, tr_ref)
    assert rel(got, ref) < 1e-5                    # far inside the bar on this small case


def test_reconstruct_config2(osiv):
    cfg = si.scan_config("2")
    got, tr, ref, tr_ref, st = run_pair(osiv, cfg, dict(beta=0.005, n_subsets=10, n_iters=100))
    check_run(got, tr, ref, tr_ref)


def test_reconstruct_first_iteration_monitor_and_residual(osiv):
    """n_iters=1 isolates A1-A6 once: D(0) is the monitor of the homogeneous image, the image is one Eq. 3 step."""
    cfg = ODD
    cfg = si.ScanConfig("odd1", 37, 29, 4.0, 24, 45, sad_mm=400.0, theta0_rad=0.3, channel_offset=0.25, seed=7, i0=3e4)
    got, tr, ref, tr_ref, st = run_pair(osiv, cfg, dict(beta=0.02, n_subsets=3, n_iters=1))
    check_run(got, tr, ref, tr_ref)
    assert tr[0, 1] == 0.01


def test_reconstruct_odd_geometry_with_channel_blank_and_zero_counts(osiv):
    cfg = si.ScanConfig("odd2", 37, 29, 4.0, 24, 45, sad_mm=400.0, theta0_rad=0.3, channel_offset=0.25, seed=17, i0=3.0)
    og, gg = geoms(cfg)
    ell, sino, counts = si.make_case(cfg)
    assert (counts == 0).any()                     # G11: max(y,1) only matters for the monitor
    blank = (cfg.i0 * (1.0 + 0.2 * np.sin(np.arange(cfg.n_channels)))).astype(np.float32)
    prm = dict(beta=0.01, n_subsets=4, n_iters=40)
    ref, tr_ref, st = oracle.reconstruct(og, counts, blank, oracle.Params(**prm))
    with osiv.Handle(gg, max_batch=1) as h:
        got, tr = h.reconstruct(dev(counts)[None], dev(blank), osiv.Params(**prm), trace=True)
    check_run(host(got)[0], tr[0], ref, tr_ref)


def test_reconstruct_forced_lambda_and_constant_lambda(osiv):
    cfg = si.scan_config("1")
    lam = 0.01 + 0.001 * np.arange(30)          # stays below the stability limit: rounding noise is not amplified
    got, tr, ref, tr_ref, _ = run_pair(osiv, cfg, dict(beta=0.01, n_subsets=2, n_iters=30, forced_lambda=lam))
    check_run(got, tr, ref, tr_ref)
    assert np.array_equal(tr[:, 1], lam)
    # constant-lambda comparator of PAPER.md:140 (Fig. 3): up = down = 0
    got, tr, ref, tr_ref, _ = run_pair(osiv, cfg, dict(beta=0.0, n_subsets=1, n_iters=25, lambda_up=0.0, lambda_down=0.0))
    check_run(got, tr, ref, tr_ref)
    assert np.all(tr[:, 1] == 0.01)


def test_reconstruct_through_the_oscillation_with_return_best(osiv):
    """lambda overshoots, D turns upward, Eq. 5 pulls it back; the image at the minimum of D is
    returned.  Eq. 4-5 compare D(n) with D(n-1): the float32 path carries ~1e-6 relative rounding noise in D
    (DESIGN.md section 7), so DECISION parity is asserted where the oracle's relative change of D exceeds 2e-5,
    ARITHMETIC parity beyond that by replaying the oracle's lambda trace (forced_lambda), and past the blow-up
    (where rounding noise is amplified and parity is undefined) only the paper's qualitative
    behaviour."""
    cfg = si.ScanConfig("osc", 16, 16, 4.0, 24, 24, i0=2e4, seed=5)
    og, gg = geoms(cfg)
    ell, sino, counts = si.make_case(cfg)
    N = 1200
    ref, tr_ref, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(beta=0.002, n_iters=N, return_best=1))
    relchg = np.abs(np.diff(tr_ref[:, 0])) / tr_ref[1:, 0]
    robust = int(np.argmax(relchg < 2e-5)) + 1            # decisions up to here are far above the noise
    ups = np.diff(tr_ref[:, 0]) >= 0
    assert ups.any() and 100 < robust < int(np.argmax(ups))
    first = int(np.argmax(ups)) + 1
    with osiv.Handle(gg, max_batch=1) as h:
        got, tr = h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(beta=0.002, n_iters=N, return_best=1), trace=True)
        tr = tr[0]
        assert np.array_equal(tr[:robust, 1], tr_ref[:robust, 1])
        assert np.all(np.abs(tr[:robust, 0] - tr_ref[:robust, 0]) <= 1e-5 * tr_ref[:robust, 0])
        # qualitative: the step rule is obeyed, lambda was pulled back, floor respected, the
        # returned image is finite, non-negative and its monitor is the smallest one seen
        lam_replay = np.empty(N)
        for n in range(N):
            lam_replay[n] = 0.01 if n == 0 else (lam_replay[n - 1] + 1e-4 if tr[n, 0] < tr[n - 1, 0]
                                                 else max(lam_replay[n - 1] - 2e-4, 1e-4))
        assert np.array_equal(tr[:, 1], lam_replay)
        assert (np.diff(tr[:, 1]) < 0).any() and tr[:, 1].min() >= 1e-4
        g = host(got)[0]
        assert np.all(np.isfinite(g)) and g.min() >= 0.0
        _, D_g = oracle.residual(og, oracle.forward(og, g), counts.astype(np.float64), cfg.i0)
        assert D_g <= tr[:, 0].min() * (1 + 1e-5)
        # return_best inside the robust region
        kw = dict(beta=0.002, n_iters=robust, return_best=1)
        ref2, tr2, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(**kw))
        got2 = host(h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(**kw)))[0]
        assert rel(got2, ref2) < IMG_TOL
        # forced replay of the oracle's lambda beyond the robust region but below the stability limit (the
        # oracle blows up at lambda ~ 0.048; float32 noise seeds the unstable mode earlier, so stop at 0.04)
        n3 = int(np.argmax(tr_ref[:, 1] >= 0.04))
        assert robust < n3 < first
        kw = dict(beta=0.002, n_iters=n3, return_best=1, forced_lambda=tr_ref[:n3, 1].copy())
        ref3, tr3, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(**kw))
        got3, trg3 = h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(**kw), trace=True)
        assert np.array_equal(trg3[0, :, 1], tr3[:, 1])
        assert np.all(np.abs(trg3[0, :, 0] - tr3[:, 0]) <= 1e-5 * tr3[:, 0])
        assert rel(host(got3)[0], ref3) < IMG_TOL


def test_reconstruct_batch_is_independent_and_deterministic(osiv):
    cfg = si.scan_config("1")
    _, gg = geoms(cfg)
    counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(3)])
    prm = osiv.Params(beta=0.01, n_subsets=3, n_iters=12)
    with osiv.Handle(gg, max_batch=3) as h:
        a, tra = h.reconstruct(dev(counts), cfg.i0, prm, trace=True)
        b, trb = h.reconstruct(dev(counts), cfg.i0, prm, trace=True)
        assert torch.equal(a, b) and np.array_equal(tra, trb)          # atomic-free, fixed-order reductions
        for s in range(3):
            # a launch that carries several slices splits rays and views differently (two half-size blocks per SM), so a
            # slice reconstructed alone agrees up to the rounding order of the sums, with the same lambda decisions
            one, tr1 = h.reconstruct(dev(counts[s:s + 1]), cfg.i0, prm, trace=True)
            assert rel(host(one)[0], host(a)[s].astype(np.float64)) < 2e-6
            assert np.array_equal(tr1[0, :, 1], tra[s, :, 1]) and np.allclose(tr1[0, :, 0], tra[s, :, 0], rtol=1e-6, atol=0)
        assert not torch.equal(a[0], a[1])
        # the host-buffer entry point gives the same bits
        hst = h.reconstruct_host(counts, cfg.i0, prm)
        assert np.array_equal(hst, host(a))
        n0 = h.launch_count()
        h.reconstruct(dev(counts), cfg.i0, prm)
        assert h.launch_count() - n0 >= 2 * prm.n_iters


def test_reconstruct_same_subset_monitor_variant(osiv):
    """monitor_mode = 1 (reading G3): Eq. 4-5 compare D(n) with D(n-M).  Config 2 (10 subsets) and an
    odd geometry in a batch of two; lambda traces equal to the oracle's, images within the bar."""
    cfg = si.scan_config("2")
    og, gg = geoms(cfg)
    counts = si.make_case(cfg)[2]
    kw = dict(beta=cfg.betas[0], n_subsets=cfg.n_subsets, n_iters=cfg.n_iters, monitor_mode=1, return_best=1)
    ref, tr_ref, status = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(**kw))
    assert status == 0 and not np.array_equal(
        tr_ref[:, 1], oracle.reconstruct(og, counts, cfg.i0, oracle.Params(**dict(kw, monitor_mode=0)))[1][:, 1])
    with osiv.Handle(gg, max_batch=1) as h:
        got, tr = h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(**kw), trace=True)
    assert np.array_equal(tr[0, :, 1], tr_ref[:, 1])
    assert np.all(np.abs(tr[0, :, 0] - tr_ref[:, 0]) <= 1e-5 * tr_ref[:, 0])
    assert rel(host(got)[0], ref) < IMG_TOL
    og, gg = geoms(ODD)
    cs = np.stack([si.make_case(ODD, slice_index=s)[2] for s in range(2)])
    kw = dict(beta=0.003, n_subsets=4, n_iters=30, monitor_mode=1)
    with osiv.Handle(gg, max_batch=2) as h:
        got, tr = h.reconstruct(dev(cs), ODD.i0, osiv.Params(**kw), trace=True)
    for s in range(2):
        ref, tr_ref, _ = oracle.reconstruct(og, cs[s], ODD.i0, oracle.Params(**kw))
        assert np.array_equal(tr[s, :, 1], tr_ref[:, 1]) and rel(host(got)[s], ref) < IMG_TOL


@pytest.mark.parametrize("cfg,M", [(si.scan_config("1"), 3), (SYM, 2), (ODD, 4)])
def test_pairs_of_slices_path_matches_oracle(osiv, cfg, M):
    """Launches with >= 4 slices serve a pair of slices per block (interleaved images, shared chord weights): an odd
    batch (the last pair half empty) of different slices against the oracle, slice by slice -- projector pair,
    reconstruction with return_best, traces -- on the general path (config 1, ODD) and the quarter-turn path (SYM)."""
    og, gg = geoms(cfg)
    B = 5
    rng = np.random.default_rng(cfg.seed + 9)
    with osiv.Handle(gg, max_batch=B) as h:
        assert h.plan(M, B)["k2_threads"] <= 448            # the pair path is the one being planned
        img = rng.uniform(0.0, 0.013, size=(B, cfg.ny, cfg.nx)).astype(np.float32)
        vs = cfg.n_views // M
        sino = rng.uniform(0.0, 1.0, size=(B, vs, cfg.n_channels)).astype(np.float32)
        f, b = host(h.forward(dev(img), 1, M)), host(h.backward(dev(sino), 1, M))
        for s in range(B):
            assert rel(f[s], oracle.forward(og, img[s], 1, M)) < PROJ_TOL
            assert rel(b[s], oracle.backward(og, sino[s], 1, M)) < PROJ_TOL
        counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(B)])
        kw = dict(beta=0.004, n_subsets=M, n_iters=24, return_best=1)
        got, tr = h.reconstruct(dev(counts), cfg.i0, osiv.Params(**kw), trace=True)
        again, tr2 = h.reconstruct(dev(counts), cfg.i0, osiv.Params(**kw), trace=True)
        assert torch.equal(got, again) and np.array_equal(tr, tr2)
        for s in range(B):
            ref, tr_ref, _ = oracle.reconstruct(og, counts[s], cfg.i0, oracle.Params(**kw))
            assert np.array_equal(tr[s, :, 1], tr_ref[:, 1])
            assert np.all(np.abs(tr[s, :, 0] - tr_ref[:, 0]) <= 1e-5 * tr_ref[:, 0])
            assert rel(host(got)[s], ref) < IMG_TOL
        # a single slice on the same handle afterwards (the image buffers change their layout back)
        one = h.reconstruct(dev(counts[:1]), cfg.i0, osiv.Params(**kw))
        assert rel(host(one)[0], host(got)[0].astype(np.float64)) < 2e-6


@pytest.mark.parametrize("cfg,M,k,tvz", [(SYM, 2, 5, 0.8), (si.scan_config("1"), 3, 7, 1.0), (ODD, 4, -3, 0.5),
                                         (SYM, 2, 0, 1.0), (SYM, 2, 5, 0.0)])
def test_stack_of_slices_matches_oracle(osiv, cfg, M, k, tvz):
    """SURVEY.md 8(f)-3 (readings H1-H3): the slices of a call as one volume -- the gantry advanced by k views per slice,
    3-D TV coupling neighbouring slices, per-slice monitor and step -- against oracle.reconstruct_stack."""
    og, gg = geoms(cfg)
    S = 4
    counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(S)])
    kw = dict(beta=0.01, n_subsets=M, n_iters=30)
    ref, tr_ref, status = oracle.reconstruct_stack(og, counts, cfg.i0, oracle.Params(**kw), view_shift=k, tv_z=tvz)
    assert status == 0
    with osiv.Handle(gg, max_batch=S) as h:
        got, tr = h.reconstruct(dev(counts), cfg.i0, osiv.Params(view_shift=k, tv_z=tvz, **kw), trace=True)
        for s in range(S):
            assert np.array_equal(tr[s, :, 1], tr_ref[s, :, 1])
            assert np.all(np.abs(tr[s, :, 0] - tr_ref[s, :, 0]) <= 1e-5 * tr_ref[s, :, 0])
            assert rel(host(got)[s], ref[s]) < IMG_TOL
        if tvz > 0:                                             # the coupling is really on: not the independent slices
            free = h.reconstruct(dev(counts), cfg.i0, osiv.Params(view_shift=k, **kw))
            assert rel(host(free)[1], ref[1]) > 1e-3
        with pytest.raises(osiv.OsivError):                     # stacks offer neither return_best nor forced lambda
            h.reconstruct(dev(counts), cfg.i0, osiv.Params(view_shift=k, tv_z=tvz, return_best=1, **kw))


def test_dependent_launch_chain_gives_the_same_bits_as_stream_order(osiv):
    """K1/K2 chained by programmatic dependent launch (default) vs plain stream order: the overlap moves only
    constant-dependent prologues ahead of the wait, so images and traces must be identical bit for bit."""
    cfg = si.scan_config("2")
    _, gg = geoms(cfg)
    counts = si.make_case(cfg)[2]
    prm = osiv.Params(beta=cfg.betas[0], n_subsets=cfg.n_subsets, n_iters=60, return_best=1)
    with osiv.Handle(gg, max_batch=1) as h:
        a, tra = h.reconstruct(dev(counts)[None], cfg.i0, prm, trace=True)
        h.set_overlap(False)
        b, trb = h.reconstruct(dev(counts)[None], cfg.i0, prm, trace=True)
        h.set_overlap(True)
        c2, trc = h.reconstruct(dev(counts)[None], cfg.i0, prm, trace=True)
    assert torch.equal(a, b) and np.array_equal(tra, trb)
    assert torch.equal(a, c2) and np.array_equal(tra, trc)


def test_reconstruct_zero_iterations_and_errors(osiv):
    cfg = si.scan_config("1")
    _, gg = geoms(cfg)
    counts = dev(si.make_case(cfg)[2])[None]
    with osiv.Handle(gg, max_batch=1) as h:
        img = h.reconstruct(counts, cfg.i0, osiv.Params(n_iters=0, mu0=0.004))
        assert torch.all(img == np.float32(0.004))
        for bad in (dict(n_subsets=7), dict(n_subsets=0), dict(n_iters=-1)):
            with pytest.raises(osiv.OsivError) as e:
                h.reconstruct(counts, cfg.i0, osiv.Params(**bad))
            assert e.value.status == osiv.OSIV_ERR_INVALID_ARG
        with pytest.raises(osiv.OsivError):
            h.forward(torch.zeros((2, cfg.ny, cfg.nx), device="cuda"))          # batch > max_batch
        with pytest.raises(osiv.OsivError):
            h.forward(torch.zeros((1, cfg.ny, cfg.nx), device="cuda"), 3, 3)    # subset >= n_subsets
        # a monitor that is not finite is reported, not hidden
        bad_counts = counts.clone()
        bad_counts[0, 0, 0] = float("inf")        # ln(b/inf) = -inf -> D = inf
        with pytest.raises(osiv.OsivError) as e:
            h.reconstruct(bad_counts, cfg.i0, osiv.Params(n_iters=2), trace=True)
        assert e.value.status == osiv.OSIV_ERR_NOT_FINITE


def test_reconstruct_config3_full(osiv):
    """BASELINE.json configs[2] in full (512x512, 800 x 738, 20 subsets, 500 iterations, beta = 0.005): the
    launch configuration bench.py times.  The oracle needs about a minute on the GPU box's host cores."""
    cfg = si.scan_config("3")
    got, tr, ref, tr_ref, st = run_pair(osiv, cfg, dict(beta=0.005, n_subsets=20, n_iters=500))
    assert st == 0
    check_run(got, tr, ref, tr_ref)
    truth = si.rasterize(cfg, si.draw_ellipses(cfg, cfg.seed))
    assert rel(got, truth) < 0.06                  # sanity only: noisy data, parity unpinned against truth


@pytest.mark.parametrize("beta", [0.001, 0.02])
def test_reconstruct_config3_other_betas_full(osiv, beta):
    """BASELINE.json configs[2]: "beta swept over {0.001, 0.005, 0.02}", each for the full 500 iterations (the oracle
    needs well under a minute per run on the GPU box's host cores); lambda peaks near 0.025 and decays."""
    cfg = si.scan_config("3")
    got, tr, ref, tr_ref, st = run_pair(osiv, cfg, dict(beta=beta, n_subsets=20, n_iters=500))
    assert st == 0
    check_run(got, tr, ref, tr_ref)
    assert 0.02 < tr[:, 1].max() < 0.03 and tr[-1, 1] < tr[:, 1].max()


@pytest.mark.parametrize("M,n_iters", [(1, 3), (2, 6), (5, 15), (10, 30), (40, 120)])
def test_reconstruct_config3_at_the_papers_other_thinning_parameters(osiv, M, n_iters):
    """PAPER.md:158-164 Table I times one 512 x 512 slice at thinning 1, 1/2, 1/5, 1/10, 1/20 and 1/40 (1/20 is config 3
    itself, above); bench.py's `extra.table1` times the same six.  Each is another launch plan at full size (K1's rays per
    block and segments; K2: the general kernel for M <= 10, where a subset's windows need several staging rounds, the
    staged one for 20 and 40), checked here against the oracle for about 2400 view-iterations (three passes over the
    subsets for M = 40), with the paper's regulariser scaling beta / M."""
    cfg = si.scan_config("3")
    with osiv.Handle(geoms(cfg)[1], max_batch=1) as h:
        assert h.back_kernel(M, 1) == ("staged" if M >= 20 else "general")
    got, tr, ref, tr_ref, st = run_pair(osiv, cfg, dict(beta=0.005, n_subsets=M, n_iters=n_iters))
    assert st == 0
    check_run(got, tr, ref, tr_ref)


def test_pairs_of_slices_path_at_config4_size(osiv):
    """A8 where the clock runs (BASELINE.json configs[3]: slices of 512x512, 800 x 738, 20 subsets): the launch plan of the
    pair-of-slices path at this size (K1 two 512-thread blocks per SM, K2 view shares of 56 tiles) is another regime
    than the toy sizes of test_pairs_of_slices_path_matches_oracle.  An odd batch (7: the last pair half empty) and an
    even batch (6) for 60 iterations (three passes over the 20 subsets), slice by slice against the oracle with equal
    lambda traces; projector pair of the batch as well."""
    cfg = si.scan_config("4")
    og, gg = geoms(cfg)
    B, N, M = 7, 60, cfg.n_subsets
    counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(B)])
    kw = dict(beta=cfg.betas[0], n_subsets=M, n_iters=N)
    refs = [oracle.reconstruct(og, counts[s], cfg.i0, oracle.Params(**kw)) for s in range(B)]
    rng = np.random.default_rng(cfg.seed + 9)
    with osiv.Handle(gg, max_batch=B) as h:
        plan = h.plan(M, B)
        assert plan["k1_orbit"] == 4 and plan["k2_threads"] <= 448      # the pair path, quarter-turn kernels
        for batch in (B, B - 1):
            got, tr = h.reconstruct(dev(counts[:batch]), cfg.i0, osiv.Params(**kw), trace=True)
            for s in range(batch):
                ref, tr_ref, st = refs[s]
                assert st == 0
                assert np.array_equal(tr[s, :, 1], tr_ref[:, 1]), (batch, s)
                assert np.all(np.abs(tr[s, :, 0] - tr_ref[:, 0]) <= 1e-5 * tr_ref[:, 0])
                assert rel(host(got)[s], ref) < IMG_TOL
            if batch == B:
                first = host(got)
        # one slice alone agrees with the same slice inside the batch up to the rounding order of the sums
        one, tr1 = h.reconstruct(dev(counts[2:3]), cfg.i0, osiv.Params(**kw), trace=True)
        assert rel(host(one)[0], first[2].astype(np.float64)) < 2e-6 and np.array_equal(tr1[0, :, 1], refs[2][1][:, 1])
        # the batch's projector pair on one subset
        img = rng.uniform(0.0, 0.013, size=(B, cfg.ny, cfg.nx)).astype(np.float32)
        sino = rng.uniform(0.0, 1.0, size=(B, cfg.n_views // M, cfg.n_channels)).astype(np.float32)
        f, b = host(h.forward(dev(img), 3, M)), host(h.backward(dev(sino), 3, M))
        for s in (0, 3, B - 1):
            assert rel(f[s], oracle.forward(og, img[s], 3, M)) < PROJ_TOL
            assert rel(b[s], oracle.backward(og, sino[s], 3, M)) < PROJ_TOL


def test_projector_pair_max_size_config5b_all_views(osiv):
    """1024x1024, 1600 x 1476, all views (BASELINE.json configs[4], the launch bench.py --workload 5b times): forward
    and back in full against the oracle (about 2.9e9 weights per pass: some tens of seconds on the host cores)."""
    cfg = si.scan_config("5b")
    og, gg = geoms(cfg)
    img, sino = si.uniform_image(cfg), si.uniform_sinogram(cfg)
    with osiv.Handle(gg, max_batch=1) as h:
        got = host(h.forward(dev(img)[None]))[0]
        gotb = host(h.backward(dev(sino)[None]))[0]
    assert rel(got, oracle.forward(og, img)) < PROJ_TOL
    assert rel(gotb, oracle.backward(og, sino)) < PROJ_TOL
    lhs = np.dot(got.astype(np.float64).ravel(), sino.astype(np.float64).ravel())
    rhs = np.dot(img.astype(np.float64).ravel(), gotb.astype(np.float64).ravel())
    assert abs(lhs - rhs) / abs(lhs) < 2e-6


def test_stack_of_slices_at_256(osiv):
    """8(f)-3 beyond toy sizes: config 2's geometry (256x256, 400 x 384, 10 subsets, quarter-turn kernels) as a stack of
    5 slices with the gantry advanced 7 views per slice and the 3-D TV on, 30 iterations."""
    cfg = si.scan_config("2")
    og, gg = geoms(cfg)
    S, k, tvz = 5, 7, 0.8
    counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(S)])
    kw = dict(beta=0.01, n_subsets=cfg.n_subsets, n_iters=30)
    ref, tr_ref, status = oracle.reconstruct_stack(og, counts, cfg.i0, oracle.Params(**kw), view_shift=k, tv_z=tvz)
    assert status == 0
    with osiv.Handle(gg, max_batch=S) as h:
        got, tr = h.reconstruct(dev(counts), cfg.i0, osiv.Params(view_shift=k, tv_z=tvz, **kw), trace=True)
        free = h.reconstruct(dev(counts), cfg.i0, osiv.Params(view_shift=k, **kw))
    for s in range(S):
        assert np.array_equal(tr[s, :, 1], tr_ref[s, :, 1])
        assert np.all(np.abs(tr[s, :, 0] - tr_ref[s, :, 0]) <= 1e-5 * tr_ref[s, :, 0])
        assert rel(host(got)[s], ref[s]) < IMG_TOL
    assert rel(host(free)[2], ref[2]) > 10 * rel(host(got)[2], ref[2])          # the coupling is really on


def test_stack_of_slices_at_512(osiv):
    """8(f)-3 at the size the clock runs at (PAPER.md:51 helical acquisition): config 3's geometry (512x512, 800 x 738, 20
    subsets) as a stack of 3 slices, the gantry advanced 11 views per slice, 3-D TV on, 20 iterations (one pass over the
    subsets) against the oracle's stack."""
    cfg = si.scan_config("3")
    og, gg = geoms(cfg)
    S, k, tvz = 3, 11, 0.6
    counts = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(S)])
    kw = dict(beta=0.005, n_subsets=cfg.n_subsets, n_iters=20)
    ref, tr_ref, status = oracle.reconstruct_stack(og, counts, cfg.i0, oracle.Params(**kw), view_shift=k, tv_z=tvz)
    assert status == 0
    with osiv.Handle(gg, max_batch=S) as h:
        got, tr = h.reconstruct(dev(counts), cfg.i0, osiv.Params(view_shift=k, tv_z=tvz, **kw), trace=True)
    for s in range(S):
        assert np.array_equal(tr[s, :, 1], tr_ref[s, :, 1])
        assert np.all(np.abs(tr[s, :, 0] - tr_ref[s, :, 0]) <= 1e-5 * tr_ref[s, :, 0])
        assert rel(host(got)[s], ref[s]) < IMG_TOL


def test_forced_lambda_ramp_up_to_the_oracles_stability_limit(osiv):
    """G12: arithmetic parity under a forced step is defined while the iteration is stable.  Where that ends is taken from
    the oracle, not assumed: under the steep ramp lambda(n) = 0.01 + 0.002 n the oracle's monitor falls until the step
    crosses the stability limit and then grows; the CUDA path must agree with the oracle up to two iterations before that
    turn (beyond it rounding noise is amplified on both sides and the trajectories separate)."""
    cfg = si.scan_config("1")
    og, gg = geoms(cfg)
    counts = si.make_case(cfg)[2]
    lam = 0.01 + 0.002 * np.arange(40)
    kw = dict(beta=0.01, n_subsets=2)
    _, tr_all, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(n_iters=40, forced_lambda=lam, **kw))
    D = tr_all[:, 0]
    per = D[0::2]                                            # subset 0's visits
    turn = 2 * (int(np.argmax(np.diff(per) > 0)) + 1) if (np.diff(per) > 0).any() else 40
    n_ok = max(turn - 2, 1)
    assert 10 <= n_ok <= 40, turn                            # the ramp does reach the limit inside the window
    ref, tr_ref, _ = oracle.reconstruct(og, counts, cfg.i0, oracle.Params(n_iters=n_ok, forced_lambda=lam[:n_ok].copy(), **kw))
    with osiv.Handle(gg, max_batch=1) as h:
        got, tr = h.reconstruct(dev(counts)[None], cfg.i0, osiv.Params(n_iters=n_ok, forced_lambda=lam[:n_ok].copy(), **kw), trace=True)
    check_run(host(got)[0], tr[0], ref, tr_ref)


def test_not_finite_is_reported_by_the_host_call_without_a_trace(osiv):
    cfg = si.scan_config("1")
    _, gg = geoms(cfg)
    counts = si.make_case(cfg)[2][None].copy()
    counts[0, 0, 0] = np.inf
    with osiv.Handle(gg, max_batch=1) as h:
        with pytest.raises(osiv.OsivError) as e:
            h.reconstruct_host(counts, cfg.i0, osiv.Params(n_iters=2))
        assert e.value.status == osiv.OSIV_ERR_NOT_FINITE
        with pytest.raises(osiv.OsivError) as e:
            h.reconstruct(dev(counts), cfg.i0, osiv.Params(n_iters=2, tv_eps=0.0))
        assert e.value.status == osiv.OSIV_ERR_INVALID_ARG


def test_checked_build_finds_no_out_of_range_index():
    """compute-sanitizer is closed on the development pool, so the gathers that rely on clamped indices, zero padding and
    slack behind a row are checked by the library itself: the same sources built with -DOSIV_CHECKED compare every such
    index with its buffer's extent on the device (include/osiv.h `osiv_debug_checks`).  Runs in a child process because
    the build is chosen when the library is loaded."""
    import os
    import subprocess
    import sys
    code = r'''
import numpy as np, torch
import synth_inputs as si
import paper_1903_10088_b200 as osiv
def geom(c, **kw):
    return osiv.Geometry(c.nx, c.ny, c.pixel_mm, c.n_views, c.n_channels, c.sad_mm, c.sdd_mm, c.dgamma_rad, c.channel_offset, c.theta0_rad, **kw)
cases = [(si.scan_config("1"), 1, 1), (si.scan_config("2"), 10, 1), (si.scan_config("2"), 10, 5),
         (si.ScanConfig("sym8", 40, 40, 1.3, 24, 45, sad_mm=120.0, theta0_rad=0.3, channel_offset=0.25, seed=12), 2, 3),
         (si.ScanConfig("odd", 37, 29, 1.3, 24, 45, sad_mm=120.0, theta0_rad=0.3, channel_offset=0.25, seed=7), 2, 4)]
for c, M, B in cases:
    counts = torch.from_numpy(np.stack([si.make_case(c, slice_index=s)[2] for s in range(B)])).cuda()
    with osiv.Handle(geom(c), max_batch=B) as h:
        h.reconstruct(counts, c.i0, osiv.Params(beta=0.005, n_subsets=M, n_iters=12, return_best=1))
        img = torch.rand((B, c.ny, c.nx), device="cuda") * 0.013
        sino = h.forward(img)
        h.backward(sino)
        if B >= 3:
            h.reconstruct(counts, c.i0, osiv.Params(beta=0.005, n_subsets=M, n_iters=6, view_shift=1, tv_z=0.5))
        h.set_back_kernel(True)
        h.reconstruct(counts, c.i0, osiv.Params(beta=0.005, n_subsets=M, n_iters=6))
    torch.cuda.synchronize()
r = osiv.debug_checks()
print("CHECKS", r)
assert r["violations"] == 0 and r["checks"] > 100000, r
'''
    env = dict(os.environ, OSIV_CHECK_BUILD="1")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    res = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, res.stdout[-2000:] + res.stderr[-2000:]
    assert "CHECKS" in res.stdout


def test_graph_replay_gives_the_same_bits_as_launch_by_launch(osiv):
    """osiv_reconstruct as one CUDA graph (captured when a call repeats the previous call's arguments, with the dependent
    launches as programmatic edges) against the same call enqueued launch by launch: identical images and traces, on the
    staged-K2 path (config 2), the general path (config 1), with return_best and with several slices."""
    for cfg, M, B, rb in [(si.scan_config("2"), 10, 1, 0), (si.scan_config("1"), 1, 2, 1), (si.scan_config("2"), 10, 5, 1)]:
        _, gg = geoms(cfg)
        counts = dev(np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(B)]))
        prm = osiv.Params(beta=0.005, n_subsets=M, n_iters=30, return_best=rb)
        out = torch.empty((B, cfg.ny, cfg.nx), dtype=torch.float32, device="cuda")
        with osiv.Handle(gg, max_batch=B) as h:
            h.set_graph(False)
            ref, tr_ref = h.reconstruct(counts, cfg.i0, prm, out=out, trace=True)
            ref = host(ref).copy()
            assert h.graph_replays() == 0
            h.set_graph(True)
            n0 = h.launch_count()
            imgs = []
            for _ in range(3):                         # first call: launch by launch; second: capture + replay; third: replay
                got, tr = h.reconstruct(counts, cfg.i0, prm, out=out, trace=True)
                imgs.append(host(got).copy())
                assert np.array_equal(tr, tr_ref)
            assert h.graph_replays() == 2
            assert (h.launch_count() - n0) % 3 == 0      # replays account for the same launches
            for im in imgs:
                assert np.array_equal(im, ref)
            # other arguments: back to launch by launch, and still the same arithmetic
            prm2 = osiv.Params(beta=0.005, n_subsets=M, n_iters=29, return_best=rb)
            h.reconstruct(counts, cfg.i0, prm2, out=out)
            assert h.graph_replays() == 2
