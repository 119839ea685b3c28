"""Oracle for the image-domain mosaic.  TEST INFRASTRUCTURE (oracle/__init__.py).

Paper (section 2.2): "For image-domain mosaics, an image of each mosaic component is generated with the phase
position at its centre, and image-plane reprojection is used to construct the mosaic at a common phase position.  Prior to
the degridding stage of cleaning the model image is reprojected to the phase position of each mosaic component, and
multiple FFT and degridding steps are performed."  The paper names no interpolant, no weighting and no projection; the
readings (R21-R23):

  R21  frames: component i is imaged on its own tangent plane, pixel (n/2, n/2) at its pointing; in the small-field limit
       its coordinates (l', m') relate to the mosaic's by the translation l = l' + l_i, m = m' + m_i (the pointing offsets
       are those of the UV-domain mosaic kernels, R11; curvature and w between tangent planes are out of scope).
  R22  reprojection = bilinear interpolation of the source image at the target pixel's position, zero outside the source.
       A component image (forward direction) is used only inside its inner half, where the taper-corrected image is valid
       (S20: 1 / psi psi reaches 2.7e7 in the corners); a model image (backward direction) is used whole.
  R23  mosaic = sum_i w_i B_i(l - l_i, m - m_i) * reproject_i[I_i],  w_i = sum of weights of component i / total, B the power
       beam E^2 of an Airy dish: the linear mosaic that the UV-domain mosaic forms with its beam kernels, so
       that the same Eq. 1 correction gamma(l, m) applies afterwards.  Prediction is the adjoint chain without the
       weights: model -> reproject to component i -> times B(l', m') -> image -> grid (O7) -> degrid (O5).
"""
from __future__ import annotations

import numpy as np

from .kernels import airy


def reproject(src: np.ndarray, cell_src: float, n_dst: int, cell_dst: float, shift_lm: tuple[float, float],
              beam: str | None = None, dish_diameter_m: float = 0.0, freq_hz: float = 0.0,
              inner_half: bool = False) -> np.ndarray:
    """R22.  dst(l, m) = B * bilinear(src at (l - shift_l, m - shift_m)); pixel (n/2, n/2) is the origin of either frame,
    x (l) along the last axis.  beam = None, "src" (B evaluated at the source-frame position l - shift: the forward
    direction, the beam is centred on the component image) or "dst" (at the target-frame position l: the backward
    direction).  inner_half: only source pixels n/4 <= x, y < 3n/4 count (R22).  complex128 in, complex128 out."""
    n_src = src.shape[-1]
    lo, hi = (n_src // 4, 3 * (n_src // 4)) if inner_half else (0, n_src)
    ax = (np.arange(n_dst) - n_dst // 2) * cell_dst
    ll, mm = np.meshgrid(ax, ax)                                   # [m index][l index]
    ls, ms = ll - shift_lm[0], mm - shift_lm[1]
    fx = ls / cell_src + n_src // 2
    fy = ms / cell_src + n_src // 2
    x0 = np.floor(fx).astype(np.int64)
    y0 = np.floor(fy).astype(np.int64)
    tx, ty = fx - x0, fy - y0
    out = np.zeros((n_dst, n_dst), np.complex128)
    for dy, wy in ((0, 1.0 - ty), (1, ty)):
        for dx, wx in ((0, 1.0 - tx), (1, tx)):
            yy, xx = y0 + dy, x0 + dx
            ok = (yy >= lo) & (yy < hi) & (xx >= lo) & (xx < hi)
            out[ok] += (wy * wx)[ok] * src[yy[ok], xx[ok]]
    if beam == "src":
        out *= airy(np.hypot(ls, ms), dish_diameter_m, freq_hz) ** 2
    elif beam == "dst":
        out *= airy(np.hypot(ll, mm), dish_diameter_m, freq_hz) ** 2
    return out


def mosaic_image(component_images: list[np.ndarray], sum_weights: list[float], cell_comp: float, pointing_lm,
                 n_mosaic: int, cell_mosaic: float, dish_diameter_m: float, freq_hz: float) -> np.ndarray:
    """R23 forward: sum_i w_i B_i reproject_i[I_i] on the mosaic frame."""
    total = float(np.sum(sum_weights))
    out = np.zeros((n_mosaic, n_mosaic), np.complex128)
    for img, sw, (li, mi) in zip(component_images, sum_weights, pointing_lm):
        out += (sw / total) * reproject(img, cell_comp, n_mosaic, cell_mosaic, (li, mi), "src", dish_diameter_m, freq_hz,
                                        inner_half=True)
    return out


def component_model(model: np.ndarray, cell_mosaic: float, n_comp: int, cell_comp: float, pointing_lm_i,
                    dish_diameter_m: float, freq_hz: float) -> np.ndarray:
    """R23 backward: the model image as component i sees it, B(l', m') * model(l' + l_i, m' + m_i), on its own frame."""
    li, mi = pointing_lm_i
    return reproject(model, cell_mosaic, n_comp, cell_comp, (-li, -mi), "dst", dish_diameter_m, freq_hz)
