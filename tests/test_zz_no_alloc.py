"""GPU test (-m gpu) of imager_hogbom_static, the minor cycle for callers that are not allowed to allocate device memory
(include/imager.h: a pipeline whose HBM was all handed out at start-up, a process whose caching allocator owns the
device, a real-time loop that cannot take the allocator's locks or implicit waits).  The entry point uses a 128 KB scratch
array built into libimager.so instead of cudaMallocAsync, so what has to hold is: (1) it gives the results of the
allocating path, imager_hogbom -- bit for bit, the bar tests/test_gpu_clean.py sets for the minor cycle, since both run
the same one-IEEE-operation-per-step arithmetic and the peak search does not depend on how many blocks share the image;
(2) it still does so on a SECOND call, when the shared array holds the first call's leftovers (a finished control block,
component counts, peak records of a larger image); (3) an image beyond IMAGER_HOGBOM_STATIC_MAX_N is refused with a message
that names the limit, and nothing is touched.

This file is named so that pytest collects it after every other test file: under `pytest -x` a failure here cannot hide
another test's result.  It needs nothing from the other tests and passes alone in a fresh process as well as at the end of
the whole suite (the set-up of the scratch address happens inside the first call, whenever that is)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _psf_and_sky(n, seed, n_src=10):
    """A PSF with sidelobes (peak 1 at the centre) and a sky of point sources convolved with it plus noise: synthetic and
    seeded, float32 like the images the minor cycle works on."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[:n, :n] - n // 2
    r2 = (x * x + y * y).astype(np.float64)
    psf = np.exp(-r2 / 6.0) + 0.07 * np.cos(0.4 * x + 0.1) * np.cos(0.33 * y) * np.exp(-r2 / 700.0) * (r2 > 0)
    psf[n // 2, n // 2] = 1.0
    psf = psf.astype(np.float32)
    sky = (1e-3 * rng.standard_normal((n, n))).astype(np.float32)
    c = n // 2
    for _ in range(n_src):
        py, px = int(rng.integers(n // 4, 3 * n // 4)), int(rng.integers(n // 4, 3 * n // 4))
        a = np.float32(rng.uniform(-2, 3))
        qy0, qy1, qx0, qx1 = max(0, py - c), min(n, py - c + n), max(0, px - c), min(n, px - c + n)
        sky[qy0:qy1, qx0:qx1] += (a * psf[qy0 - py + c:qy1 - py + c, qx0 - px + c:qx1 - px + c]).astype(np.float32)
    return psf, sky


def _run(fn, sky, psf, window, gain, thr, cf, n_iter):
    import torch
    n = sky.shape[0]
    res = torch.from_numpy(sky.copy()).cuda()
    model = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    comps = torch.zeros((max(n_iter, 1), 3), dtype=torch.float32, device="cuda")
    count = torch.full((1,), -7, dtype=torch.int32, device="cuda")
    fn(res, torch.from_numpy(psf).cuda(), model, window, gain, thr, cf, n_iter, comps, count)
    torch.cuda.synchronize()
    return res.cpu().numpy(), model.cpu().numpy(), comps.cpu().numpy(), int(count.item())


def test_static_scratch_minor_cycle_matches_the_allocating_one_twice_in_a_row():
    import torch
    assert torch.cuda.is_available()
    from paper_2206_15117_b200 import imager_hogbom, imager_hogbom_static
    # first call: 200 x 200 (40 blocks), ends on the cycle factor with components found; second call: a smaller image
    # (9 blocks, n not a multiple of the block's 1024 pixels), another window, runs all its iterations -- it starts
    # from a scratch array that still says "done", carries the first call's count and 31 stale peak records; third
    # call: an empty window, which must report zero components whatever the array held
    cases = [(200, (50, 50, 150, 150), 0.2, 0.0, 0.3, 400),
             (93, (5, 11, 80, 90), 0.1, 0.0, 0.0, 150),
             (93, (10, 10, 10, 40), 0.1, 0.0, 0.0, 50)]
    for k, (n, window, gain, thr, cf, n_iter) in enumerate(cases):
        psf, sky = _psf_and_sky(n, seed=100 + k)
        want = _run(imager_hogbom, sky, psf, window, gain, thr, cf, n_iter)
        got = _run(imager_hogbom_static, sky, psf, window, gain, thr, cf, n_iter)
        assert got[3] == want[3], f"call {k}: number of components"
        assert (got[3] > 5) == (k < 2)
        assert np.array_equal(got[2], want[2]), f"call {k}: components (y, x, a)"
        assert np.array_equal(got[0], want[0]), f"call {k}: residual image"
        assert np.array_equal(got[1], want[1]), f"call {k}: model image"
        if k < 2:
            assert not np.array_equal(got[0], sky)


def test_static_scratch_minor_cycle_refuses_an_image_beyond_its_limit():
    import torch
    from paper_2206_15117_b200 import ImagerError, imager_hogbom_static
    from paper_2206_15117_b200.binding import HOGBOM_STATIC_MAX_N
    n = HOGBOM_STATIC_MAX_N + 8
    img = torch.ones((n, n), dtype=torch.float32, device="cuda")
    model = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    with pytest.raises(ImagerError, match="IMAGER_HOGBOM_STATIC_MAX_N = 4096"):
        imager_hogbom_static(img, img, model, (0, 0, n, n), 0.1, 0.0, 0.0, 3)
    torch.cuda.synchronize()
    assert torch.count_nonzero(model).item() == 0 and bool((img == 1).all())
    # the limit itself is accepted (one block per 1024 pixels: all 16384 peak records in use)
    n = HOGBOM_STATIC_MAX_N
    psf = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    psf[n // 2, n // 2] = 1.0
    res = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    res[n - 1, n - 1] = 2.0                                   # the peak sits in the last block's last pixel
    res[7, 5] = -1.5
    model = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    count = torch.zeros(1, dtype=torch.int32, device="cuda")
    imager_hogbom_static(res, psf, model, (0, 0, n, n), 1.0, 0.5, 0.0, 5, None, count)
    torch.cuda.synchronize()
    assert int(count.item()) == 2
    assert float(model[n - 1, n - 1]) == 2.0 and float(model[7, 5]) == -1.5 and torch.count_nonzero(res).item() == 0
