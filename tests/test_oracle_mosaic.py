"""Pins for the image-domain mosaic oracle (oracle/mosaic.py, readings R21-R23): identities of the bilinear
reprojection, the flat-sky closed form, reduction to plain imaging, and agreement of the image-domain mosaic with the
UV-domain mosaic (two independent chains of the oracle) on the same sky."""
import numpy as np

from oracle import mosaic as om, kernels as ok, imaging as oi, index as oidx, gridder as og
from helpers import base_params, random_vis, oracle_tables, MODE_MOSAIC_PB


def test_reprojection_identities():
    rng = np.random.default_rng(1)
    n, cell = 32, 1e-3
    img = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    assert np.array_equal(om.reproject(img, cell, n, cell, (0.0, 0.0)), img)                  # identity
    sh = om.reproject(img, cell, n, cell, (3 * cell, -5 * cell))                               # whole pixels: a shift
    assert np.allclose(sh[:27, 3:], img[5:, :29], atol=1e-12) and np.all(sh[27:, :] == 0) and np.all(sh[:, :3] == 0)
    y, x = np.mgrid[:n, :n]
    ramp = (2.0 * x - 3.0 * y + 0.5).astype(np.complex128)                                      # bilinear is exact on planes
    half = om.reproject(ramp, cell, n, cell, (0.5 * cell, 0.25 * cell))
    assert np.allclose(half[1:, 1:], (2.0 * (x - 0.5) - 3.0 * (y - 0.25) + 0.5)[1:, 1:], atol=1e-10)
    # a finer target grid samples between the source pixels; l is the LAST axis
    fine = om.reproject(ramp, cell, 2 * n, cell / 2, (0.0, 0.0))
    assert np.isclose(fine[n, n + 1], ramp[n // 2, n // 2] + 1.0) and np.isclose(fine[n + 1, n], ramp[n // 2, n // 2] - 1.5)
    # beam factors: "src" is centred on the source frame (moves with the shift), "dst" on the target frame
    ones = np.ones((n, n), np.complex128)
    b_src = om.reproject(ones, cell, n, cell, (4 * cell, 0.0), "src", 12.0, 30e9)
    b_dst = om.reproject(ones, cell, n, cell, (4 * cell, 0.0), "dst", 12.0, 30e9)
    e2 = lambda l, m: ok.airy(np.hypot(l, m), 12.0, 30e9) ** 2
    assert np.isclose(b_src[n // 2, n // 2 + 4], 1.0) and np.isclose(b_src[n // 2 + 2, n // 2 + 7], e2(3 * cell, 2 * cell))
    assert np.isclose(b_dst[n // 2, n // 2 + 4], e2(4 * cell, 0.0)) and np.isclose(b_dst[n // 2, n // 2], 1.0)


def test_flat_sky_mosaic_is_the_weighted_sum_of_beams():
    """Component images that are identically 1 (a unit visibility at the origin, P6) mosaic to sum_i w_i B_i(l - l_i): the
    beam-weighted sum that Eq. 1 then corrects."""
    n_c, n_m, cell = 48, 64, 5e-4
    pts = [(0.0, 0.0), (6.3 * cell, -2.2 * cell), (-4.5 * cell, 7.75 * cell)]
    sw = [100.0, 50.0, 50.0]
    imgs = [np.ones((n_c, n_c), np.complex128)] * 3
    mos = om.mosaic_image(imgs, sw, cell, pts, n_m, cell, 12.0, 60e9)
    ax = (np.arange(n_m) - n_m // 2) * cell
    ll, mm = np.meshgrid(ax, ax)
    want = sum(w / 200.0 * ok.airy(np.hypot(ll - a, mm - b), 12.0, 60e9) ** 2 for w, (a, b) in zip(sw, pts))
    inside = (slice(n_m // 2 - 4, n_m // 2 + 4),) * 2                  # covered by the inner halves of all three frames
    assert np.allclose(mos[inside], want[inside], rtol=1e-12)
    beams = np.stack([ok.airy(np.hypot(ll - a, mm - b), 12.0, 60e9) ** 2 for a, b in pts])
    gamma = oi.mosaic_gamma(beams)                                       # Eq. 1 applies to the result as it stands
    assert np.all(np.isfinite(gamma[inside]))


def test_one_central_pointing_without_beam_is_plain_imaging(oracle_lib):
    params = base_params(grid_size=64, cell_size_rad=0.05 / 64, oversample=8)
    uvw, vis, wts, _ = random_vis(params, 200, seed=4, frac=0.3)
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, None, params)
    g = og.grid(rec, vis, wts, flat, offs, params)
    img = oi.grid_to_image(g["grid"][0], g["sumwt"][0])
    mos = om.mosaic_image([img], [g["sumwt"][0]], params["cell_size_rad"], [(0.0, 0.0)], 64, params["cell_size_rad"], 0.0, 1e9)
    half = (slice(16, 48),) * 2
    assert np.allclose(mos[half], img[half], rtol=1e-12, atol=1e-14)
    mos[half] = 0
    assert np.all(mos == 0)                                               # only the inner half of a component image is used
    back = om.component_model(img, params["cell_size_rad"], 64, params["cell_size_rad"], (0.0, 0.0), 0.0, 1e9)
    assert np.allclose(back, img, rtol=1e-12, atol=1e-14)


def test_image_domain_mosaic_agrees_with_uv_domain_mosaic(oracle_lib):
    """Two independent chains of the oracle on the same sky: (a) UV-domain mosaic, all pointings on one grid with their
    beams as gridding kernels (MOSAIC_PB tables); (b) image-domain mosaic, each pointing imaged at its own
    phase centre with the plain anti-aliasing kernel, beam-weighted, reprojected and summed.  Both estimate
    sum_i w_i B_i(l) [dirty beam_i * (B_i I)](l); they agree to the approximation error of the beam kernels' finite
    support and the bilinear interpolation.  A sign error in the shift, a beam centred on the wrong frame, missing weights
    or a transposed axis is off by tens of per cent."""
    n, fov = 96, 0.03
    cell = fov / n
    freq, dish = 4e9, 12.0
    pts = [(0.0, 0.0), (8 * cell, -5 * cell), (-7 * cell, 6 * cell)]          # whole pixels: reprojection is then exact
    srcs = [(3, -4, 1.0), (-9, 7, 0.7), (10, 2, 0.5)]                          # (px, py, flux) on the mosaic frame
    rng = np.random.default_rng(8)
    p_uv = base_params(grid_size=n, cell_size_rad=cell, oversample=16, support_min=24, support_max=24, n_aplanes=3,
                       pa_rad=[0] * 3, pointing_lm=[list(p) for p in pts], kernel_mode=MODE_MOSAIC_PB, freq_hz=freq,
                       dish_diameter_m=dish)
    p_img = base_params(grid_size=n, cell_size_rad=cell, oversample=16)
    uvws, vis_common, vis_own, a_idx = [], [], [], []
    for i, (li, mi) in enumerate(pts):
        uvw, _, _, _ = random_vis(p_img, 400, seed=30 + i, frac=0.3)
        uvw[:, 2] = 0
        u, v = uvw[:, 0].astype(np.float64), uvw[:, 1].astype(np.float64)
        vc = np.zeros(400, np.complex128)
        for px, py, a in srcs:
            l, m = px * cell, py * cell
            vc += a * ok.airy(np.hypot(l - li, m - mi), dish, freq) ** 2 * np.exp(2j * np.pi * (u * l + v * m))
        uvws.append(uvw)
        vis_common.append(vc)
        vis_own.append(vc * np.exp(-2j * np.pi * (u * li + v * mi)))         # phase centre moved to the pointing (R21)
        a_idx.append(np.full(400, i, np.int32))
    wts = np.ones((1200, 1), np.float32)
    # (a) UV-domain
    _, _, flat_uv, offs_uv = oracle_tables(p_uv)
    rec = oidx.index_visibilities(np.concatenate(uvws), np.concatenate(a_idx), p_uv)
    assert not rec["drop"].any()
    g = og.grid(rec, np.concatenate(vis_common).astype(np.complex64)[:, None], wts, flat_uv, offs_uv, p_uv)
    uv_mosaic = oi.grid_to_image(g["grid"][0], g["sumwt"][0]).real
    # (b) image-domain
    _, _, flat_i, offs_i = oracle_tables(p_img)
    imgs, sws = [], []
    for uvw, vo in zip(uvws, vis_own):
        r = oidx.index_visibilities(uvw, None, p_img)
        gi = og.grid(r, vo.astype(np.complex64)[:, None], wts[:400], flat_i, offs_i, p_img)
        imgs.append(oi.grid_to_image(gi["grid"][0], gi["sumwt"][0]))
        sws.append(gi["sumwt"][0])
    img_mosaic = om.mosaic_image(imgs, sws, cell, pts, n, cell, dish, freq).real
    inner = (slice(n // 2 - 14, n // 2 + 14),) * 2                     # inside the inner half of every component frame
    peak = np.abs(uv_mosaic[inner]).max()
    assert peak > 0.2
    assert np.abs(img_mosaic - uv_mosaic)[inner].max() < 0.03 * peak
    wrong = om.mosaic_image(imgs, sws, cell, [(-a, -b) for a, b in pts], n, cell, dish, freq).real
    assert np.abs(wrong - uv_mosaic)[inner].max() > 0.3 * peak
