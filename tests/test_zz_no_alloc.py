"""GPU test of the allocation-free entry point `osiv_tv_gradient_static` (include/osiv.h): the TV gradient (C8) with
its padded-image scratch in the library's fixed `static __device__` array instead of cudaMalloc'ed workspace.

Collected last on purpose (the file name sorts after every other test file): the run uses `pytest -x`, so
a failure here cannot hide another test.  It passes alone in a fresh process and after the rest of the suite: nothing
here depends on what earlier tests left in the array, and each case clears nothing itself -- the entry point does."""
import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TV_TOL = 5e-6          # the bar of test_tv_gradient_matches_oracle in test_gpu_parity.py


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


@pytest.fixture(scope="module")
def osiv():
    import paper_1903_10088_b200 as m
    assert torch.cuda.is_available()
    m.lib()                      # raises if libosiv.so is missing: there is no fallback
    return m


def images(shape, seed, batch):
    ny, nx = shape
    rng = np.random.default_rng(seed)
    img = (0.007 + 1e-4 * rng.standard_normal((batch, ny, nx))).astype(np.float32)
    if ny > 8 and nx > 8:
        img[:, 2:6, 3:8] = 0.007                                        # flat patch: t = eps
    return img


def test_static_scratch_matches_the_existing_path_on_two_calls_in_a_row(osiv):
    """Two calls back to back on one stream, the second on a SMALLER grid than the first, so that the array still holds
    the first call's larger images where the second call's zero border must be: a missing clear shows at the border."""
    big, small = (72, 96), (29, 37)
    g_big = osiv.Geometry(big[1], big[0], 1.0, 8, 8, sad_mm=400.0)
    g_small = osiv.Geometry(small[1], small[0], 1.0, 8, 8, sad_mm=400.0)
    with osiv.Handle(g_big, max_batch=3) as hb, osiv.Handle(g_small, max_batch=3) as hs:
        a, b = images(big, 21, 3), images(small, 22, 2)
        da, db = dev(a), dev(b)
        out_a, out_b = torch.full_like(da, float("nan")), torch.full_like(db, float("nan"))
        hb.tv_gradient_static(da, out_a, 1e-5)          # call 1
        hs.tv_gradient_static(db, out_b, 1e-5)          # call 2, right behind it
        torch.cuda.synchronize()
        ref_a, ref_b = hb.tv_gradient(da, 1e-5), hs.tv_gradient(db, 1e-5)      # the existing path
        torch.cuda.synchronize()
        for got, ref, src in ((out_a, ref_a, a), (out_b, ref_b, b)):
            assert bool(torch.isfinite(got).all())
            assert rel(got.cpu().numpy(), ref.cpu().numpy()) < TV_TOL
            assert torch.equal(got, ref)                # same kernel on the same layout: the header promises equal bits
            for s in range(src.shape[0]):               # and both agree with the float64 oracle
                assert rel(got[s].cpu().numpy(), oracle.tv_grad(src[s], 1e-5)) < TV_TOL
        # the same call again, now over its own previous contents, and with another eps
        again = torch.full_like(da, float("nan"))
        hb.tv_gradient_static(da, again, 1e-3)
        torch.cuda.synchronize()
        assert torch.equal(again, hb.tv_gradient(da, 1e-3))
        const = torch.full_like(db, 0.005)
        assert float(hs.tv_gradient_static(const, torch.empty_like(const), 1e-5).abs().max()) == 0.0


def test_static_scratch_call_allocates_no_device_memory(osiv):
    """Free device memory is the same before and after the first static call on a fresh handle (whose lazily allocated
    workspace does not exist yet), while the existing path's first call on that handle lowers it."""
    shape = (512, 512)
    g = osiv.Geometry(shape[1], shape[0], 0.78125, 8, 8, sad_mm=850.0)
    with osiv.Handle(g, max_batch=2) as warm:           # loads both kernels (lazy module loading is not an allocation of ours)
        d = dev(images(shape, 23, 1))
        warm.tv_gradient_static(d, torch.empty_like(d), 1e-5)
        torch.cuda.synchronize()
    with osiv.Handle(g, max_batch=2) as h:
        d = dev(images(shape, 24, 2))
        out = torch.empty_like(d)
        ref = torch.empty_like(d)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        h.tv_gradient_static(d, out, 1e-5)
        h.tv_gradient_static(d, out, 1e-5)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
        h.tv_gradient(d, 1e-5, out=ref)                 # the existing path allocates the handle's padded images here
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] < free0
        assert torch.equal(out, ref)


def test_static_scratch_rejects_sizes_beyond_the_stated_maximum(osiv):
    assert osiv.STATIC_SCRATCH_BYTES == 4 << 20
    g = osiv.Geometry(512, 512, 0.78125, 8, 8, sad_mm=850.0)
    with osiv.Handle(g, max_batch=4) as h:
        d3, d4 = dev(images((512, 512), 25, 3)), dev(images((512, 512), 26, 4))
        assert 3 * 514 * 520 * 4 <= osiv.STATIC_SCRATCH_BYTES < 4 * 514 * 520 * 4
        out3 = torch.empty_like(d3)
        h.tv_gradient_static(d3, out3, 1e-5)            # three slices fit
        assert torch.equal(out3, h.tv_gradient(d3, 1e-5))
        out4 = torch.full_like(d4, -1.0)
        with pytest.raises(osiv.OsivError) as e:
            h.tv_gradient_static(d4, out4, 1e-5)        # four do not
        assert e.value.status == osiv.OSIV_ERR_SCRATCH_LIMIT
        assert "OSIV_STATIC_SCRATCH_BYTES" in str(e.value)
        torch.cuda.synchronize()
        assert bool((out4 == -1.0).all())               # nothing was enqueued
    g1024 = osiv.Geometry(1024, 1024, 0.5, 8, 8, sad_mm=2000.0)
    with osiv.Handle(g1024, max_batch=1) as h:
        d = dev(images((1024, 1024), 27, 1))
        with pytest.raises(osiv.OsivError) as e:
            h.tv_gradient_static(d, torch.empty_like(d), 1e-5)
        assert e.value.status == osiv.OSIV_ERR_SCRATCH_LIMIT
