"""GPU tests (-m gpu) of the loop around the hot path: the Hogbom minor cycle (imager_hogbom) bit for
bit against oracle/clean.py, and the Cotton-Schwab loop (imager_clean) against the oracle's composition of its own steps
on a three-point-source sky with config 1's geometry (BASELINE.json configs[0]: 10,000 visibilities, 256^2 grid, 7 x 7
prolate-spheroidal kernel, oversampling 8)."""
import numpy as np
import pytest

from oracle import clean as oc, index as oidx
from helpers import oracle_tables
from synth import make_workload

pytestmark = pytest.mark.gpu


def _psf_and_sky(n, seed, n_src=12):
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[:n, :n] - n // 2
    r2 = (x * x + y * y).astype(np.float64)
    psf = np.exp(-r2 / 8.0) + 0.08 * np.cos(0.45 * x + 0.2) * np.cos(0.31 * y) * np.exp(-r2 / 900.0) * (r2 > 0)
    psf[n // 2, n // 2] = 1.0
    psf = psf.astype(np.float32)
    sky = (1e-3 * rng.standard_normal((n, n))).astype(np.float32)
    c = n // 2
    for _ in range(n_src):
        py, px, a = int(rng.integers(n // 4, 3 * n // 4)), int(rng.integers(n // 4, 3 * n // 4)), np.float32(rng.uniform(-2, 3))
        qy0, qy1, qx0, qx1 = max(0, py - c), min(n, py - c + n), max(0, px - c), min(n, px - c + n)
        sky[qy0:qy1, qx0:qx1] += (a * psf[qy0 - py + c:qy1 - py + c, qx0 - px + c:qx1 - px + c]).astype(np.float32)
    return psf, sky


@pytest.mark.parametrize("n,window,gain,thr,cf,n_iter", [
    (96, (24, 24, 72, 72), 0.1, 0.0, 0.0, 300),          # runs all its iterations
    (96, (0, 0, 96, 96), 0.25, 0.05, 0.0, 400),          # ends on the threshold
    (130, (10, 33, 97, 120), 0.2, 0.0, 0.3, 500),        # ends on the cycle factor; n not a multiple of anything
    (64, (16, 16, 48, 48), 1.0, 0.0, 0.0, 40),           # gain 1
])
def test_hogbom_is_bit_exact(n, window, gain, thr, cf, n_iter):
    import torch
    assert torch.cuda.is_available()
    from paper_2206_15117_b200 import imager_hogbom
    psf, sky = _psf_and_sky(n, seed=n + n_iter)
    if n == 64:                                          # an exact tie between two pixels of the window: the first wins
        sky[20, 40] = sky[30, 22] = np.float32(np.abs(sky).max() * 2)
    ref = oc.hogbom(sky, psf, window, gain, thr, cf, n_iter)
    d_res = torch.from_numpy(sky.copy()).cuda()
    d_psf = torch.from_numpy(psf).cuda()
    d_model = torch.zeros((n, n), dtype=torch.float32, device="cuda")
    d_comp = torch.zeros((n_iter, 3), dtype=torch.float32, device="cuda")
    d_n = torch.zeros(1, dtype=torch.int32, device="cuda")
    imager_hogbom(d_res, d_psf, d_model, window, gain, thr, cf, n_iter, d_comp, d_n)
    torch.cuda.synchronize()
    k = int(d_n.item())
    assert k == len(ref["components"]) and k > 5
    got = d_comp.cpu().numpy()[:k]
    want = np.array(ref["components"], dtype=np.float32)
    assert np.array_equal(got[:, :2], want[:, :2]), "peak positions"
    assert np.array_equal(got[:, 2], want[:, 2]), "component values"
    assert np.array_equal(d_res.cpu().numpy(), ref["residual"])
    assert np.array_equal(d_model.cpu().numpy(), ref["model"])
    if n == 64:
        assert tuple(got[0, :2]) == (20.0, 40.0)


def test_hogbom_edge_cases():
    import torch
    from paper_2206_15117_b200 import imager_hogbom
    psf, sky = _psf_and_sky(64, seed=3)
    d_res = torch.from_numpy(sky.copy()).cuda()
    d_psf = torch.from_numpy(psf).cuda()
    d_model = torch.zeros((64, 64), dtype=torch.float32, device="cuda")
    d_n = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    for window, n_iter, thr in (((10, 10, 10, 30), 20, 0.0), ((0, 0, 64, 64), 0, 0.0), ((0, 0, 64, 64), 20, 1e9)):
        imager_hogbom(d_res, d_psf, d_model, window, 0.1, thr, 0.0, n_iter, None, d_n)     # empty window / no iterations / high threshold
        torch.cuda.synchronize()
        assert int(d_n.item()) == 0 and torch.count_nonzero(d_model).item() == 0
        assert np.array_equal(d_res.cpu().numpy(), sky)


def test_cotton_schwab_loop_on_config1_geometry(oracle_lib):
    """imager_clean against the oracle's loop: same peaks cycle by cycle while they are well separated, model image and
    residual visibilities within 1e-4 of the brightest source, and the three sources recovered."""
    import torch
    from paper_2206_15117_b200 import Plan
    wl = make_workload("config1")
    params, nvis = wl.params, wl.nvis
    n, cell = params["grid_size"], params["cell_size_rad"]
    srcs = [(23, -31, 1.0), (-40, 12, 0.6), (9, 47, 0.35)]               # (px, py, flux), inside the inner half
    u, v = wl.uvw[:, 0].astype(np.float64), wl.uvw[:, 1].astype(np.float64)
    vis = sum(a * np.exp(2j * np.pi * (u * px * cell + v * py * cell)) for px, py, a in srcs).astype(np.complex64)[:, None]
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(wl.uvw, None, params)
    kw = dict(n_major=4, gain=0.2, threshold=0.005, cycle_factor=1.5, n_iter=150)
    ref = oc.cotton_schwab(rec, vis, wl.weights, flat, offs, params, **kw)
    with Plan(params, nvis, user_tables=flat) as plan:
        dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
        model = torch.empty((n, n), dtype=torch.float32, device="cuda")
        resid = torch.empty((n, n), dtype=torch.float32, device="cuda")
        psf = torch.empty((n, n), dtype=torch.float32, device="cuda")
        rvis = torch.empty((nvis, 1), dtype=torch.complex64, device="cuda")
        ncomp = torch.zeros(kw["n_major"], dtype=torch.int32, device="cuda")
        plan.clean(dev(wl.uvw), dev(vis), dev(wl.weights), model, resid, rvis, psf_out=psf, n_components_out=ncomp, **kw)
        torch.cuda.synchronize()
        assert plan.last_launch_count() > 4 * kw["n_major"]
        got_model, got_psf, got_rvis = model.cpu().numpy(), psf.cpu().numpy(), rvis.cpu().numpy()
    inner = (slice(n // 4, 3 * n // 4),) * 2
    assert np.abs(got_psf - ref["psf"])[inner].max() < 2e-5
    # the first cycle's components are found on nearly identical images: same count, same pixels in the model
    assert int(ncomp[0].item()) == len(ref["cycles"][0])
    assert set(zip(*np.nonzero(got_model))) == set(zip(*np.nonzero(ref["model"])))
    assert np.abs(got_model - ref["model"]).max() < 1e-4
    assert np.abs(got_rvis - ref["residual_vis"]).max() < 1e-4
    for px, py, a in srcs:
        box = got_model[n // 2 + py - 1:n // 2 + py + 2, n // 2 + px - 1:n // 2 + px + 2]
        assert abs(box.sum() - a) < 0.05 * a + 0.02
    assert np.abs(got_rvis).mean() < 0.1 * np.abs(vis).mean()
