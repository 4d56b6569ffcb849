"""Pins P6, P7, P9-P12 of the float64 oracle's iteration; CPU only."""
import os

import numpy as np
import pytest

import oracle
import synth_inputs as si

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")


def paper_constants():
    out = {}
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            name, val = line.split()[:2]
            out[name] = float(val)
    return out


def tv_plain(mu, eps):
    """TV_eps written out with numpy slices (C8): forward differences, zero across the border."""
    dx = np.zeros_like(mu)
    dy = np.zeros_like(mu)
    dx[:, :-1] = mu[:, 1:] - mu[:, :-1]
    dy[:-1, :] = mu[1:, :] - mu[:-1, :]
    return float(np.sqrt(eps * eps + dx * dx + dy * dy).sum())


@pytest.mark.parametrize("eps", [1e-5, 1e-3])
def test_P6_tv_gradient_finite_difference(eps):
    rng = np.random.default_rng(11)
    mu = 0.007 + 1e-3 * rng.standard_normal((9, 12))
    mu[2:5, 3:8] = 0.0071            # a flat patch: where |grad| = 0 only eps keeps TV smooth
    assert oracle.tv_value(mu, eps) == pytest.approx(tv_plain(mu, eps), rel=1e-14)
    g = oracle.tv_grad(mu, eps)
    assert abs(g.sum()) < 1e-12 * np.abs(g).sum() + 1e-13     # TV is shift invariant
    h = 1e-9 if eps < 1e-4 else 1e-7
    worst = 0.0
    for (iy, ix) in [(0, 0), (0, 5), (8, 11), (4, 0), (3, 4), (2, 3), (5, 8), (8, 0), (4, 11), (6, 6), (1, 9)]:
        e = np.zeros_like(mu)
        e[iy, ix] = h
        fd = (tv_plain(mu + e, eps) - tv_plain(mu - e, eps)) / (2 * h)
        worst = max(worst, abs(fd - g[iy, ix]) / max(1.0, abs(g[iy, ix])))
    assert worst < 2e-6


def test_P6_tv_gradient_of_constant_image_is_zero():
    assert np.abs(oracle.tv_grad(np.full((7, 5), 0.01), 1e-5)).max() == 0.0


def small_case(n=16, V=48, C=32, i0=1e4, seed=21, noisy=True):
    cfg = si.ScanConfig("t", n, n, 1.0, V, C, i0=i0, seed=seed, n_ellipses=3)
    g = oracle.Geometry(nx=n, ny=n, pixel_mm=1.0, n_views=V, n_channels=C)
    return cfg, g


def test_P7_likelihood_gradient_finite_difference():
    cfg, g = small_case()
    rng = np.random.default_rng(8)
    mu = 0.004 + 0.004 * rng.uniform(size=(16, 16))
    counts = rng.poisson(cfg.i0 * np.exp(-oracle.forward(g, 0.006 * np.ones((16, 16))))).astype(np.float64)
    blank = cfg.i0 * (1.0 + 0.1 * rng.uniform(size=g.n_channels))        # per-channel blank scan
    for (m, M) in ((-1, 1), (2, 4)):
        l = oracle.forward(g, mu, m, M)
        r, D = oracle.residual(g, l, counts, blank, m, M)
        grad = oracle.backward(g, r, m, M)                             # dL/dmu / b_ref  (C4)
        for _ in range(3):
            d = rng.standard_normal(mu.shape)
            h = 1e-5
            fd =(oracle.loglik(g, mu + h * d, counts, blank, m, M) - oracle.loglik(g, mu - h * d, counts, blank, m, M)) / (2 * h)
            assert fd == pytest.approx(float((grad * d).sum()), rel=2e-6)
        # monitor (C5): D = sum (l - ln(b/max(y,1)))^2 on the subset's rays
        ys = counts if m < 0 else counts[m::M]
        p = np.log(blank[None, :] / np.maximum(ys, 1.0))
        assert D == pytest.approx(float(((l - p) ** 2).sum()), rel=1e-13)
        # residual definition
        assert np.allclose(r, (blank[None, :] * np.exp(-l) - ys) / blank.mean(), rtol=0, atol=1e-13)


def test_golden_paper_constants_are_the_oracle_defaults():
    k = paper_constants()
    p = oracle.Params()
    assert p.lambda0 == k["lambda0"] and p.lambda_up == k["lambda_up"] and p.lambda_down == k["lambda_down"]
    assert p.mu0 == pytest.approx(k["mu0_per_cm"] / 10.0)              # /cm -> /mm
    g = oracle.Geometry(nx=8, ny=8, pixel_mm=1.0, n_views=int(k["views"]), n_channels=8)
    for M in (2, 5, 10, 20, 40):
        l = oracle.forward(g, np.ones((8, 8)), 0, M)
        assert l.shape[0] == k["subset_views_%d" % M]


def replay_step_rule(D, prm):
    lam = np.zeros(len(D))
    for n in range(len(D)):
        if n == 0:
            lam[n] = prm.lambda0
        elif D[n] < D[n - 1]:
            lam[n] = lam[n - 1] + prm.lambda_up
        else:
            lam[n] = max(lam[n - 1] - prm.lambda_down, prm.lambda_min)
    return lam


def test_P9_noise_free_beta0_converges_to_truth():
    cfg, g = small_case()
    ell = si.draw_ellipses(cfg, cfg.seed)
    truth = si.rasterize(cfg, ell)
    counts = cfg.i0 * np.exp(-oracle.forward(g, truth))               # un-sampled, in the model's range
    errs = {}
    for its in (100, 200, 3000):
        prm = oracle.Params(beta=0.0, n_subsets=1, n_iters=its)
        img, trace, status = oracle.reconstruct(g, counts, cfg.i0, prm)
        assert status == 0
        errs[its] = np.linalg.norm(img - truth) / np.linalg.norm(truth)
        if its == 200:
            # Eq. 4: D falls monotonically here, so lambda climbs by 1e-4 per iteration from 0.01
            assert np.all(np.diff(trace[:, 0]) < 0)
            assert trace[-1, 1] == pytest.approx(0.01 + 1e-4 * 199, rel=1e-12)
    # SURVEY SCRATCH saw 2e-3 @100, 6e-5 @200, 4e-16 @3000 on this geometry (after the oscillation of P10)
    assert errs[100] < 5e-3 and errs[200] < 1e-4 and errs[3000] < 1e-12


def test_P10_step_rule_replay_and_oscillation():
    # lambda grows (Eq. 4) until D turns upward, Eq. 5 pulls it back -> oscillation
    cfg, g = small_case(n=16, V=24, C=24, i0=2e4, seed=5)
    ell, sino, counts = si.make_case(cfg)
    prm = oracle.Params(beta=0.002, n_subsets=1, n_iters=1200)
    img, trace, status = oracle.reconstruct(g, counts, cfg.i0, prm)
    assert status == 0 and np.all(np.isfinite(img)) and img.min() >= 0.0
    assert np.array_equal(trace[:, 1], replay_step_rule(trace[:, 0], prm))
    ups = np.diff(trace[:, 0]) >= 0
    assert ups.any(), "lambda never overshot: the test does not reach the oscillatory regime"
    first = int(np.argmax(ups)) + 1
    assert first > 50 and np.all(np.diff(trace[:first, 0]) < 0)
    assert trace[:, 1].max() > 0.02 and trace[:, 1].min() >= prm.lambda_min
    # forced-lambda replay reproduces the adaptive run bit for bit
    prm2 = oracle.Params(beta=0.002, n_subsets=1, n_iters=1200, forced_lambda=trace[:, 1].copy())
    img2, trace2, _ = oracle.reconstruct(g, counts, cfg.i0, prm2)
    assert np.array_equal(img, img2) and np.array_equal(trace, trace2)
    # minimum-of-oscillation image: return_best yields an image whose D is the trace minimum
    prm3 = oracle.Params(beta=0.002, n_subsets=1, n_iters=first + 40, return_best=1)
    img3, trace3, _ = oracle.reconstruct(g, counts, cfg.i0, prm3)
    l3 = oracle.forward(g, img3)
    _, D3 = oracle.residual(g, l3, counts.astype(np.float64), cfg.i0)
    assert D3 <= trace3[:, 0].min() * (1 + 1e-12)


def replay_step_rule_same_subset(D, prm):
    M, lam = prm.n_subsets, np.zeros(len(D))
    for n in range(len(D)):
        if n < M:
            lam[n] = prm.lambda0
        elif D[n] < D[n - M]:
            lam[n] = lam[n - 1] + prm.lambda_up
        else:
            lam[n] = max(lam[n - 1] - prm.lambda_down, prm.lambda_min)
    return lam


def test_P10b_same_subset_monitor_variant():
    # reading G3's alternative: D(n) is compared with D(n-M), the last visit of the same subset.  With one subset the
    # two rules are the same rule; with M > 1 lambda stays at lambda0 for the first pass, the trace replays from its own
    # D values, and the step no longer collapses under strong thinning (the literal rule compares different subsets'
    # D, which differ by more than one update changes them; "the oscillation behavior is emphasized").
    cfg, g = small_case(n=16, V=24, C=24, i0=2e4, seed=5)
    _, _, counts = si.make_case(cfg)
    a = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=0.002, n_subsets=1, n_iters=300))
    b = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=0.002, n_subsets=1, n_iters=300, monitor_mode=1))
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    for M in (3, 6):
        prm = oracle.Params(beta=0.002, n_subsets=M, n_iters=240, monitor_mode=1)
        img, trace, status = oracle.reconstruct(g, counts, cfg.i0, prm)
        assert status == 0
        assert np.all(trace[:M, 1] == prm.lambda0)
        assert np.array_equal(trace[:, 1], replay_step_rule_same_subset(trace[:, 0], prm))
        lit = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=0.002, n_subsets=M, n_iters=240))[1]
        assert not np.array_equal(lit[:, 1], trace[:, 1])
        # per-subset D falls pass after pass at first, so lambda climbs by lambda_up every iteration after the first pass
        per = trace[:, 0].reshape(-1, M)
        assert np.all(np.diff(per[:5], axis=0) < 0) and abs(trace[5 * M - 1, 1] - (prm.lambda0 + 4 * M * prm.lambda_up)) < 1e-12


def test_P11_adaptive_lambda_is_about_three_times_faster():
    # "a similar degree of convergence is achieved with 500 iterations compared to 1500
    # iterations using a constant convergence parameter" -- same counts, on a 32x32 body-sized phantom
    cfg = si.ScanConfig("t", 32, 32, 4.0, 64, 48, i0=2e4, seed=9, n_ellipses=4)
    g = oracle.Geometry(nx=32, ny=32, pixel_mm=4.0, n_views=64, n_channels=48)
    ell, sino, counts = si.make_case(cfg)

    def final_D(prm):
        img, trace, _ = oracle.reconstruct(g, counts, cfg.i0, prm)
        _, D = oracle.residual(g, oracle.forward(g, img), counts.astype(np.float64), cfg.i0)
        return D

    base = dict(beta=0.0, n_subsets=1)
    D_adapt_500 = final_D(oracle.Params(n_iters=500, **base))
    D_const_500 = final_D(oracle.Params(n_iters=500, lambda_up=0.0, lambda_down=0.0, **base))
    D_const_1500 = final_D(oracle.Params(n_iters=1500, lambda_up=0.0, lambda_down=0.0, **base))
    assert D_adapt_500 < D_const_500
    assert D_adapt_500 < 1.1 * D_const_1500


def test_P12_initial_image_matters_little_and_subsets_run():
    cfg = si.ScanConfig("t", 32, 32, 4.0, 60, 48, i0=2e4, seed=10, n_ellipses=4)
    g = oracle.Geometry(nx=32, ny=32, pixel_mm=4.0, n_views=60, n_channels=48)
    ell, sino, counts = si.make_case(cfg)
    Ds = []
    for mu0 in (0.0, 0.005, 0.01):                                      # 0, 0.05, 0.1 /cm
        img, trace, _ = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=0.001, n_iters=200, mu0=mu0))
        _, D = oracle.residual(g, oracle.forward(g, img), counts.astype(np.float64), cfg.i0)
        Ds.append(D)
    assert max(Ds) / min(Ds) < 1.1                                      # "the difference was so small"
    # ordered subsets: one iteration = one subset; water reconstructs to ~0.0070 /mm
    img, trace, status = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=0.002, n_subsets=5, n_iters=200))
    assert status == 0 and trace.shape == (200, 2)
    truth = si.rasterize(cfg, ell)
    assert np.linalg.norm(img - truth) / np.linalg.norm(truth) < 0.15


# ---- pins of the update itself: thinning scale beta/M, subset order (C11), sign of the prior
# (Eq. 2-3), positivity, zero counts in the monitor (G11).  None of these replays
# the oracle's own trace: every expected value is composed here, in numpy, from the individually pinned pieces
# (forward P2-P5, backward P4, residual P7, tv_grad P6, tau P8). ----

def asymmetric_case():
    # no symmetry of the phantom or the scan maps one subset onto another: every subset sees different data
    cfg = si.ScanConfig("t", 20, 20, 1.0, 36, 30, i0=5e3, seed=31, n_ellipses=4, theta0_rad=0.13, channel_offset=0.25)
    g = oracle.Geometry(nx=20, ny=20, pixel_mm=1.0, n_views=36, n_channels=30, theta0_rad=0.13, channel_offset=0.25)
    _, _, counts = si.make_case(cfg)
    return cfg, g, counts.astype(np.float64)


def one_update(g, mu, counts, blank, m, M, lam, beta, eps, kappa=100.0):
    """Eq. 3 on subset m with the regulariser weight multiplied by the thinning 1/M,
    then mu >= 0; returns (mu_next, D, unclamped)."""
    l = oracle.forward(g, mu, m, M)
    r, D = oracle.residual(g, l, counts, blank, m, M)
    grad = oracle.backward(g, r, m, M)
    u = mu + lam * oracle.tau(g, M, kappa) * (grad - (beta / M) * oracle.tv_grad(mu, eps))
    return np.maximum(u, 0.0), D, u


@pytest.mark.parametrize("M", [3, 4])
def test_update_replay_pins_thinning_scale_and_subset_order(M):
    cfg, g, counts = asymmetric_case()
    beta, eps = 0.5, 1e-4                 # strong prior: the beta/M term is far above rounding in every step
    N = M + 2
    # mu0 = 0 with a doubled first step: some pixels overshoot below zero in most steps, so the clamp is exercised
    base = dict(beta=beta, n_subsets=M, mu0=0.0, lambda0=0.02, tv_eps=eps)
    prm = oracle.Params(n_iters=N, **base)
    runs = [oracle.reconstruct(g, counts, cfg.i0, oracle.Params(n_iters=n, **base)) for n in range(1, N + 1)]
    trace = runs[-1][1]
    mu = np.zeros((g.ny, g.nx))
    lam, D_prev = prm.lambda0, None
    clamp_bites = 0
    for n in range(N):
        m = n % M                                                      # C11: natural order
        D = oracle.residual(g, oracle.forward(g, mu, m, M), counts, cfg.i0, m, M)[1]
        if n > 0:                                                      # Eq. 4-5 from the D values composed here
            lam = lam + prm.lambda_up if D < D_prev else max(lam - prm.lambda_down, prm.lambda_min)
        D_prev = D
        assert trace[n, 0] == pytest.approx(D, rel=1e-13)              # D(n) is the monitor of subset n mod M ...
        assert trace[n, 1] == lam
        for other in range(M):                                         # ... and of no other subset
            if other != m:
                Do = oracle.residual(g, oracle.forward(g, mu, other, M), counts, cfg.i0, other, M)[1]
                assert abs(Do - D) > 1e-6 * D
        nxt, _, u = one_update(g, mu, counts, cfg.i0, m, M, lam, beta, eps)
        assert np.allclose(runs[n][0], nxt, rtol=0, atol=1e-15)
        clamp_bites += int((u < 0).sum())
        assert (u < 0).sum() < u.size // 2                             # the clamp acts on a part of the image only
        if n > 0:
            # the readings the paper excludes must be visibly different updates of this very step:
            # un-thinned weight beta instead of beta/M, another subset's data, the prior with the other sign
            for alt in (one_update(g, mu, counts, cfg.i0, m, M, lam, beta * M, eps)[0],
                        one_update(g, mu, counts, cfg.i0, (m + 1) % M, M, lam, beta, eps)[0],
                        one_update(g, mu, counts, cfg.i0, m, M, lam, -beta, eps)[0]):
                assert np.abs(alt - nxt).max() > 1e-4 * np.abs(nxt).max()
        mu = nxt
    assert clamp_bites > 0, "the positivity clamp never acted: the case does not pin it"


def test_zero_counts_only_touch_the_monitor():
    # G11: p_i = ln(b_i / max(y_i, 1)).  A ray that counted nothing has the monitor term of a ray that counted one
    # photon, stays finite, and enters the gradient with its true count 0.
    cfg, g, counts = asymmetric_case()
    mu = np.full((g.ny, g.nx), 0.004)
    l = oracle.forward(g, mu, 1, 3)
    ys = counts[1::3].copy()
    zero = np.zeros_like(ys, dtype=bool)
    zero[2, 5] = zero[7, 11] = zero[0, 0] = True
    c0, c1 = counts.copy(), counts.copy()
    c0[1::3][zero] = 0.0
    c1[1::3][zero] = 1.0
    r0, D0 = oracle.residual(g, l, c0, cfg.i0, 1, 3)
    r1, D1 = oracle.residual(g, l, c1, cfg.i0, 1, 3)
    assert np.isfinite(D0) and D0 == D1
    assert np.allclose((r0 - r1)[zero], 1.0 / cfg.i0, rtol=1e-12) and np.array_equal(r0[~zero], r1[~zero])
    # the term itself: (l - ln b)^2 for those rays
    base = counts.copy()
    base[1::3][zero] = 1.0
    expect = ((l - np.log(cfg.i0 / np.maximum(base[1::3], 1.0))) ** 2).sum()
    assert D0 == pytest.approx(float(expect), rel=1e-13)
    # a whole reconstruction on data with dead rays stays finite
    img, trace, status = oracle.reconstruct(g, c0, cfg.i0, oracle.Params(beta=0.01, n_subsets=3, n_iters=12))
    assert status == 0 and np.all(np.isfinite(trace)) and np.all(np.isfinite(img))


def test_prior_sign_more_beta_means_less_total_variation():
    # Eq. 2-3: the prior enters the ascent as +alpha*R with R = -TV, so a larger weight must give an
    # image of smaller total variation from the same data, at equal data iterations, and at beta = 0 the TV term is absent
    cfg, g, counts = asymmetric_case()
    tvs = []
    for beta in (0.0, 0.05, 0.5):
        img, _, _ = oracle.reconstruct(g, counts, cfg.i0, oracle.Params(beta=beta, n_subsets=3, n_iters=60, tv_eps=1e-4))
        tvs.append(tv_plain(img, 1e-4))
    assert tvs[0] > tvs[1] > tvs[2] and tvs[2] < 0.8 * tvs[0]
