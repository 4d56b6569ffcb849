"""CPU-only checks of the C-ABI boundary: the library builds with nvcc, loads without a GPU, exports every
symbol include/osiv.h declares, validates arguments before touching CUDA, and its host-side A0 tables
reproduce the oracle's chord weights.  No kernel runs here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import paper_1903_10088_b200 as osiv

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "osiv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(osiv_[a-z_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    L = osiv.lib()
    names = declared_functions()
    assert len(names) >= 13
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/osiv.h but not exported"
    assert sorted(osiv.EXPORTED_SYMBOLS) == names
    assert osiv.version() >= 100
    assert osiv.strerror(0) == "ok" and "invalid" in osiv.strerror(-1) and "CUDA" in osiv.strerror(-2)


def test_default_params_are_the_papers_constants():
    p = osiv.default_params()
    k = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_constants.txt")):
        if line.strip() and not line.startswith("#"):
            name, val = line.split()[:2]
            k[name] = float(val)
    assert p.lambda0 == k["lambda0"] and p.lambda_up == k["lambda_up"] and p.lambda_down == k["lambda_down"]
    assert p.mu0 == pytest.approx(k["mu0_per_cm"] / 10.0)
    assert p.kappa == 100.0 and p.tv_eps == 1e-5 and p.lambda_min == 1e-4 and p.return_best == 0


def test_argument_validation_happens_before_cuda():
    L = osiv.lib()
    h = C.c_void_p()
    good = osiv.Geometry(64, 64, 1.0, 90, 96).c()
    assert L.osiv_create(None, 1, 0, C.byref(h)) == osiv.OSIV_ERR_INVALID_ARG
    assert L.osiv_create(C.byref(good), 0, 0, C.byref(h)) == osiv.OSIV_ERR_INVALID_ARG
    assert L.osiv_create(C.byref(good), 1, -1, C.byref(h)) == osiv.OSIV_ERR_INVALID_ARG
    for bad in (dict(nx=0), dict(n_views=0), dict(n_channels=-3), dict(pixel_mm=0.0), dict(sad_mm=40.0),
                dict(pixel_mm=float("nan")), dict(dgamma_rad=0.1)):        # 96 * 0.1 rad > pi
        kw = dict(nx=64, ny=64, pixel_mm=1.0, n_views=90, n_channels=96)
        kw.update(bad)
        g = osiv.Geometry(**kw).c()
        assert L.osiv_create(C.byref(g), 1, 0, C.byref(h)) == osiv.OSIV_ERR_INVALID_ARG, bad
        assert L.osiv_ray_table(C.byref(g), None, None) == osiv.OSIV_ERR_INVALID_ARG, bad
    # null handles
    assert L.osiv_forward(None, None, None, 1, -1, 1, None) == osiv.OSIV_ERR_INVALID_ARG
    assert L.osiv_backward(None, None, None, 1, -1, 1, None) == osiv.OSIV_ERR_INVALID_ARG
    assert L.osiv_tv_gradient_static(None, None, None, 1, 1e-5, None) == osiv.OSIV_ERR_INVALID_ARG
    assert "OSIV_STATIC_SCRATCH_BYTES" in osiv.strerror(osiv.OSIV_ERR_SCRATCH_LIMIT)
    assert L.osiv_reconstruct(None, None, None, 1.0, None, 1, None, None, None) == osiv.OSIV_ERR_INVALID_ARG
    assert L.osiv_reconstruct_host(None, None, None, 1.0, None, 1, None, None, None) == osiv.OSIV_ERR_INVALID_ARG
    assert L.osiv_destroy(None) == osiv.OSIV_OK
    assert L.osiv_launch_count(None) == 0


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(osiv.OsivError) as e:
        osiv.Handle(osiv.Geometry(64, 64, 1.0, 90, 96))
    assert e.value.status == osiv.OSIV_ERR_CUDA


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1903_10088_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "osiv_oracle" not in text and "liboracle" not in text, f
    for f in ("oracle.py", "osiv_oracle.c", "__init__.py"):
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert not re.search(r"^\s*(import|from)\s+paper_1903_10088_b200\b", text, flags=re.M), f
        assert "osiv.h" not in text and "libosiv" not in text


@pytest.mark.parametrize("kw", [
    dict(nx=16, ny=16, pixel_mm=1.25, n_views=24, n_channels=20, sad_mm=90.0),
    dict(nx=20, ny=12, pixel_mm=0.8, n_views=36, n_channels=33, sad_mm=70.0, theta0_rad=0.3, channel_offset=0.25),
])
def test_A0_ray_table_reproduces_the_oracle_chord(kw):
    """Host logic: the {alpha,beta,g0,h} coefficients, evaluated in float64 with the formula the header states,
    give the oracle's a(i,r) (itself pinned to polygon clipping, P1) up to the float32 rounding of the table."""
    gg = osiv.Geometry(**kw)
    og = oracle.Geometry(**kw)
    rays, views = osiv.ray_table(gg)
    V, Cn = gg.n_views, gg.n_channels
    assert rays.shape == (V, Cn, 4) and views.shape == (V, 2)
    th = gg.theta0_rad + 2 * np.pi * np.arange(V) / V
    assert np.allclose(views[:, 0], np.cos(th), atol=1e-7) and np.allclose(views[:, 1], np.sin(th), atol=1e-7)
    # one coefficient is exactly +-1 (-1 only in the rotated quarter turns of a V % 4 == 0 scan), the other >= 1 in magnitude
    a, b = rays[..., 0].astype(np.float64), rays[..., 1].astype(np.float64)
    assert np.all((np.abs(a) == 1.0) | (np.abs(b) == 1.0)) and np.all(np.maximum(np.abs(a), np.abs(b)) >= 1.0)
    xc = np.arange(gg.nx) - 0.5 * (gg.nx - 1)
    yc = np.arange(gg.ny) - 0.5 * (gg.ny - 1)
    worst, nz = 0.0, 0
    for v in range(0, V, 5):
        for c in range(Cn):
            al, be, g0, h = rays[v, c].astype(np.float64)
            q = al * xc[None, :] + be * yc[:, None] + g0
            w = h * np.clip(0.5 * (abs(al) + abs(be)) - np.abs(q), 0.0, 1.0)
            ref = np.array([[oracle.weight(og, v, c, ix, iy) for ix in range(gg.nx)] for iy in range(gg.ny)])
            worst = max(worst, np.abs(w - ref).max())
            nz += int((ref > 0).sum())
    assert nz > 500
    assert worst < 5e-5 * gg.pixel_mm      # float32 coefficients: position error ~1e-6 pixel on a ramp of slope <= |k|
