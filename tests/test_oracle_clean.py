"""Pins for the minor-cycle / Cotton-Schwab oracle (oracle/clean.py, readings R18-R20): closed forms,
exact deconvolution of shifted PSFs, flux conservation, window / threshold / cycle-factor behaviour, and recovery of a
three-point-source sky through the whole major-cycle loop."""
import numpy as np

from oracle import clean as oc, index as oidx
from helpers import base_params, random_vis, oracle_tables


def _gauss_psf(n, width=2.0, sidelobe=0.1):
    y, x = np.mgrid[:n, :n] - n // 2
    r2 = x * x + y * y
    b = np.exp(-r2 / (2 * width ** 2)) + sidelobe * np.cos(0.9 * x) * np.cos(0.7 * y) * (r2 > 0) * np.exp(-r2 / 300.0)
    b[n // 2, n // 2] = 1.0
    return b.astype(np.float32)


def test_delta_psf_closed_form():
    """B = delta: one pixel v0 decays geometrically, model = v0 (1 - (1 - g)^k), residual = v0 (1 - g)^k."""
    n = 16
    psf = np.zeros((n, n), np.float32)
    psf[8, 8] = 1.0
    r = np.zeros((n, n), np.float32)
    r[5, 9] = -3.0
    out = oc.hogbom(r, psf, (0, 0, n, n), gain=0.25, threshold=0.0, cycle_factor=0.0, n_iter=10)
    assert [c[:2] for c in out["components"]] == [(5, 9)] * 10
    assert np.isclose(out["residual"][5, 9], -3.0 * 0.75 ** 10, rtol=1e-6)
    assert np.isclose(out["model"][5, 9], -3.0 * (1 - 0.75 ** 10), rtol=1e-6)
    assert np.count_nonzero(out["residual"]) == 1 and np.count_nonzero(out["model"]) == 1


def test_shifted_psfs_are_deconvolved_exactly_at_gain_one():
    n = 64
    psf = _gauss_psf(n)
    assert oc.psf_sidelobe(psf) < 0.7
    srcs = [(20, 41, 2.0), (44, 17, -1.25), (30, 30, 0.5)]
    r = np.zeros((n, n), np.float32)
    c = n // 2
    for py, px, a in srcs:                                              # built with the oracle's own float32 steps
        qy0, qy1, qx0, qx1 = max(0, py - c), min(n, py - c + n), max(0, px - c), min(n, px - c + n)
        r[qy0:qy1, qx0:qx1] += (np.float32(a) * psf[qy0 - py + c:qy1 - py + c, qx0 - px + c:qx1 - px + c]).astype(np.float32)
    r0 = r.copy()
    out = oc.hogbom(r, psf, (0, 0, n, n), gain=1.0, threshold=1e-3, cycle_factor=0.0, n_iter=50)
    got = {(y, x): v for y, x, v in out["components"][:3]}
    assert set(got) == {(y, x) for y, x, _ in srcs}                     # strongest first: 2.0, -1.25, 0.5
    assert [c[:2] for c in out["components"][:2]] == [(20, 41), (44, 17)]
    # conservation: residual + model (*) PSF = the input, to float32 rounding
    rebuilt = out["residual"].astype(np.float64)
    for py, px, a in out["components"]:
        qy0, qy1, qx0, qx1 = max(0, py - c), min(n, py - c + n), max(0, px - c), min(n, px - c + n)
        rebuilt[qy0:qy1, qx0:qx1] += a * psf[qy0 - py + c:qy1 - py + c, qx0 - px + c:qx1 - px + c].astype(np.float64)
    assert np.abs(rebuilt - r0).max() < 1e-5
    assert np.abs(out["residual"]).max() < 1e-3                         # cleaned down to the threshold
    for py, px, a in srcs:
        assert abs(out["model"][py, px] - a) < 0.1                      # overlapping wings shift the fluxes a little


def test_window_threshold_cycle_factor_and_ties():
    n = 32
    psf = _gauss_psf(n, width=1.0, sidelobe=0.2)
    side = oc.psf_sidelobe(psf)
    r = np.zeros((n, n), np.float32)
    r[4, 4] = 10.0                                                      # outside the window: never picked
    r[12, 20] = r[12, 10] = r[20, 10] = 3.0                             # a three-way tie: row-major first wins
    out = oc.hogbom(r, psf, (8, 8, 24, 24), gain=0.5, threshold=0.0, cycle_factor=0.0, n_iter=1)
    assert out["components"] == [(12, 10, 1.5)] and out["residual"][4, 4] > 9.0
    # cycle factor: stop = cycle_factor * sidelobe * first peak (on a sky that IS a sum of shifted PSFs)
    sky = np.zeros((n, n), np.float32)
    for py, px, a in [(12, 10, 3.0), (19, 21, 2.0)]:
        yy, xx = np.mgrid[:n, :n]
        ok = (np.abs(yy - py) <= n // 2 - 1) & (np.abs(xx - px) <= n // 2 - 1)
        sky[ok] += (np.float32(a) * psf[(yy - py + n // 2)[ok], (xx - px + n // 2)[ok]]).astype(np.float32)
    out = oc.hogbom(sky, psf, (8, 8, 24, 24), gain=0.5, threshold=0.0, cycle_factor=2.0, n_iter=100)
    peak0 = np.abs(sky[8:24, 8:24]).max()
    assert np.isclose(out["stop"], np.float32(np.float32(2.0) * np.float32(side)) * peak0, rtol=1e-6)
    win = np.abs(out["residual"][8:24, 8:24])
    assert win.max() < out["stop"] <= peak0 and 0 < len(out["components"]) < 100
    # threshold above the peak: nothing happens
    out = oc.hogbom(r, psf, (8, 8, 24, 24), gain=0.5, threshold=5.0, cycle_factor=0.0, n_iter=10)
    assert out["components"] == [] and np.array_equal(out["residual"], r)


def test_cotton_schwab_recovers_three_point_sources(oracle_lib):
    """The whole loop on a small w = 0 data set: three point sources inside the inner half are found at their pixels
    and their fluxes recovered to a few per cent; the residual visibilities shrink by an order of magnitude."""
    n, fov = 64, 0.05
    params = base_params(grid_size=n, cell_size_rad=fov / n, oversample=16)
    uvw, _, _, _ = random_vis(params, 1500, seed=21, frac=0.4)
    uvw[:, 2] = 0
    cell = fov / n
    srcs = [(6, -9, 1.0), (-11, 4, 0.6), (3, 12, 0.35)]                 # (px, py, flux)
    u, v = uvw[:, 0].astype(np.float64), uvw[:, 1].astype(np.float64)
    vis = sum(a * np.exp(2j * np.pi * (u * px * cell + v * py * cell)) for px, py, a in srcs).astype(np.complex64)[:, None]
    wts = np.ones((1500, 1), np.float32)
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, None, params)
    out = oc.cotton_schwab(rec, vis, wts, flat, offs, params, n_major=5, gain=0.2, threshold=0.01, cycle_factor=1.5,
                           n_iter=200)
    assert abs(out["psf"][n // 2, n // 2] - 1.0) < 1e-3 and out["sumwt"] == 1500.0
    for px, py, a in srcs:
        box = out["model"][n // 2 + py - 1:n // 2 + py + 2, n // 2 + px - 1:n // 2 + px + 2]
        assert abs(box.sum() - a) < 0.05 * a + 0.02, (px, py, box.sum())
        assert abs(out["model"][n // 2 + py, n // 2 + px] - a) < 0.1 * a + 0.02
    assert np.abs(out["residual_vis"]).mean() < 0.1 * np.abs(vis).mean()
    assert len(out["cycles"]) == 5 and len(out["cycles"][0]) > 3


def test_float64_pixel_loop_finds_the_same_peaks():
    """The oracle works in float32 on purpose (the peak search decides an integer; header of oracle/clean.py).  Pin its
    decisions against R18 written out once more in float64 with plain pixel loops: while successive peaks are separated
    by far more than float32 rounding, both must find the same pixels in the same order, and values within 1e-5."""
    n, c = 24, 12
    psf = _gauss_psf(n, width=1.5, sidelobe=0.15)
    r32 = np.zeros((n, n), np.float32)
    for py, px, a in [(7, 15, 3.0), (16, 6, -2.2), (11, 11, 1.3)]:
        for y in range(n):
            for x in range(n):
                if 0 <= y - py + c < n and 0 <= x - px + c < n:
                    r32[y, x] += np.float32(a) * psf[y - py + c, x - px + c]
    gain, n_iter = 0.35, 12
    out = oc.hogbom(r32, psf, (2, 2, 22, 22), gain=gain, threshold=0.0, cycle_factor=0.0, n_iter=n_iter)
    r, b, found = r32.astype(np.float64), psf.astype(np.float64), []
    for _ in range(n_iter):
        best, p = -1.0, None
        for y in range(2, 22):
            for x in range(2, 22):
                if abs(r[y, x]) > best:                                  # strict: the first maximum in row-major order
                    best, p = abs(r[y, x]), (y, x)
        a = gain * r[p]
        found.append((p[0], p[1], a))
        for y in range(n):
            for x in range(n):
                if 0 <= y - p[0] + c < n and 0 <= x - p[1] + c < n:
                    r[y, x] -= a * b[y - p[0] + c, x - p[1] + c]
    assert [k[:2] for k in out["components"]] == [k[:2] for k in found]
    assert len({k[:2] for k in found}) >= 3
    assert np.allclose([k[2] for k in out["components"]], [k[2] for k in found], rtol=0, atol=1e-5)
    assert np.abs(out["residual"] - r).max() < 1e-5
