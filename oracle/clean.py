"""Oracle for the minor cycle and the Cotton-Schwab loop.  TEST INFRASTRUCTURE (oracle/__init__.py).

Paper: "The output images are cleaned using an implementation of the Cotton-Schwab algorithm [6], which accepts many of
the usual parameters such as the number of clean cycles, the loop gain, the cycle factor, and a threshold stopping
criterion".  Of the minor cycle the paper says only that "more iterative processes such as Högbom cleaning
[10] are less able to take full advantage of parallelisation".  The paper gives neither algorithm in
symbols; what follows is the textbook statement (readings R18-R20):

  Hogbom minor cycle (R18) on a real residual image R, a PSF B with B[c, c] = 1 at c = N/2, inside a window W:
      repeat up to n_iter times:
          p = first pixel (row-major) of W with the largest |R|;   stop if |R[p]| < stop
          a = gain * R[p];   model[p] += a;   R[q] -= a * B[q - p + c]  for every q whose PSF sample exists
  Cycle threshold (R19):  stop = max(threshold, cycle_factor * sidelobe * |R[p_0]|), p_0 the cycle's first peak,
      sidelobe = the largest |B| outside the PSF's main lobe (here: outside the 3 x 3 pixels around its centre).
  Cotton-Schwab major cycle (R20):  residual visibilities V - V_model (model image -> grid -> degrid) are gridded and
      transformed into the next residual image; the minor cycle runs on it; n_major times.

Precision: the peak search decides an integer, so both sides take it in the kernel's precision (float32): every
arithmetic step below is ONE IEEE float32 operation (a product, then a difference: no fused multiply-add), in the order
written, which the CUDA kernels reproduce with __fmul_rn / __fsub_rn.  Peak positions and component values are then
comparable bit for bit.
"""
from __future__ import annotations

import numpy as np


def psf_sidelobe(psf: np.ndarray) -> float:
    """Largest |B| outside the 3 x 3 pixels around the PSF centre (R19)."""
    n = psf.shape[0]
    c = n // 2
    a = np.abs(np.asarray(psf, dtype=np.float32)).copy()
    a[c - 1:c + 2, c - 1:c + 2] = 0.0
    return float(a.max())


def hogbom(residual: np.ndarray, psf: np.ndarray, window: tuple[int, int, int, int], gain: float, threshold: float,
           cycle_factor: float, n_iter: int) -> dict:
    """R18 + R19.  residual, psf: float32 [N][N]; window = (y0, x0, y1, x1), half-open.  Returns the updated residual,
    the model image of this cycle (float32), and the component list (y, x, value) in the order found."""
    r = np.array(residual, dtype=np.float32, copy=True)
    b = np.asarray(psf, dtype=np.float32)
    n = r.shape[0]
    c = n // 2
    y0, x0, y1, x1 = window
    model = np.zeros_like(r)
    comps = []
    stop = np.float32(threshold)
    side = np.float32(psf_sidelobe(b))
    g32 = np.float32(gain)
    for it in range(int(n_iter)):
        win = np.abs(r[y0:y1, x0:x1])
        k = int(np.argmax(win))                                  # first maximum in row-major order
        py, px = y0 + k // (x1 - x0), x0 + k % (x1 - x0)
        peak = r[py, px]
        if it == 0:
            stop = max(np.float32(threshold), np.float32(np.float32(cycle_factor) * side) * np.abs(peak))
        if not (np.abs(peak) >= stop):
            break
        a = np.float32(g32 * peak)
        model[py, px] = np.float32(model[py, px] + a)
        comps.append((py, px, float(a)))
        # R[q] -= a * B[q - p + c] wherever that PSF sample exists
        qy0, qy1 = max(0, py - c), min(n, py - c + n)
        qx0, qx1 = max(0, px - c), min(n, px - c + n)
        sub = b[qy0 - py + c:qy1 - py + c, qx0 - px + c:qx1 - px + c]
        r[qy0:qy1, qx0:qx1] = (r[qy0:qy1, qx0:qx1] - (a * sub).astype(np.float32)).astype(np.float32)
    return dict(residual=r, model=model, components=comps, stop=float(stop))


def cotton_schwab(rec: dict, vis: np.ndarray, weights: np.ndarray, tables: np.ndarray, offsets: np.ndarray, params: dict,
                  n_major: int, gain: float, threshold: float, cycle_factor: float, n_iter: int) -> dict:
    """R20, single polarisation: the major-cycle loop as a composition of the oracle's own steps (O4 gridding, O7
    grid -> image, R18/R19 minor cycle, O7 image -> grid, O5 degridding).  The PSF is the dirty image of unit
    visibilities; the window is the inner half of the field (where the taper correction is valid, S20).
    Returns the model image (float32), the last dirty residual image, the PSF, the residual visibilities and the
    component lists of every cycle."""
    from . import gridder as og, imaging as oi
    assert int(params["n_pol"]) == 1 and int(params["n_corr"]) == 1
    n = int(params["grid_size"])
    s_ps = int(params.get("pswf_support", 7))
    ones = np.ones_like(vis)
    g_psf = og.grid(rec, ones, weights, tables, offsets, params)
    sumwt = float(g_psf["sumwt"][0])
    psf = oi.grid_to_image(g_psf["grid"][0], sumwt, s_ps).real.astype(np.float32)
    q = n // 4
    window = (q, q, 3 * q, 3 * q)
    model = np.zeros((n, n), np.float32)
    res_vis = np.array(vis, dtype=np.complex64, copy=True)
    cycles, dirty = [], None
    for _ in range(int(n_major)):
        g = og.grid(rec, res_vis, weights, tables, offsets, params)
        dirty = oi.grid_to_image(g["grid"][0], sumwt, s_ps).real.astype(np.float32)
        out = hogbom(dirty, psf, window, gain, threshold, cycle_factor, n_iter)
        cycles.append(out["components"])
        model = (model + out["model"]).astype(np.float32)
        mg = oi.image_to_grid(model.astype(np.complex128), s_ps)
        pred = og.degrid(rec, mg[None].astype(np.complex64), tables, offsets, params)
        res_vis = (vis.astype(np.complex128) - pred["vis"]).astype(np.complex64)
    return dict(model=model, dirty=dirty, psf=psf, residual_vis=res_vis, cycles=cycles, sumwt=sumwt)
