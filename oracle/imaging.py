"""Oracle steps O0 / O7: grid <-> image with taper correction, the direct DFT, and Eq. 1.
TEST INFRASTRUCTURE (see oracle/__init__.py).

Sign convention from the visibility equation, Eq. 2:  V(u,v,w) = sum_pix I(l,m)
exp[+2 pi i (u l + v m + w (n-1))], n = sqrt(1 - l^2 - m^2).  Hence grid -> image is the FORWARD DFT
(kernel e^{-2 pi i ...}) and image -> grid the unnormalised inverse DFT, both centred: pixel (N/2, N/2)
is l = m = 0 and grid cell (N/2, N/2) is u = v = 0 (R1).
"""
from __future__ import annotations

import numpy as np
from .kernels import pswf


def taper_image(n: int, pswf_support: int = 7) -> np.ndarray:
    """psi(2(x-N/2)/N) psi(2(y-N/2)/N): the image-domain anti-aliasing function the kernels were built from."""
    t = pswf(2.0 * (np.arange(n) - n // 2) / n, pswf_support)
    return np.outer(t, t)


def grid_to_image(grid: np.ndarray, sum_weights: float, pswf_support: int = 7) -> np.ndarray:
    """O7 forward: centred forward DFT of each [N][N] plane, divided by the taper and by sum of weights."""
    n = grid.shape[-1]
    img = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(grid, axes=(-2, -1))), axes=(-2, -1))
    return img / taper_image(n, pswf_support) / sum_weights


def image_to_grid(image: np.ndarray, pswf_support: int = 7) -> np.ndarray:
    """O7 inverse: divide by the taper first, then the centred UNNORMALISED inverse DFT."""
    n = image.shape[-1]
    pre = image / taper_image(n, pswf_support)
    return np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(pre, axes=(-2, -1))), axes=(-2, -1)) * (n * n)


def direct_dft_image(uvw: np.ndarray, vis: np.ndarray, weights: np.ndarray, n: int, cell: float) -> np.ndarray:
    """Dirty image by the definition the gridder approximates (adjoint of Eq. 2, one polarisation):
    I(l,m) = sum_k w_k V_k exp[-2 pi i (u l + v m + w (n-1))] / sum_k w_k.  Tiny inputs only."""
    x = (np.arange(n) - n // 2) * cell
    ll, mm = np.meshgrid(x, x)
    nn = np.sqrt(1.0 - ll * ll - mm * mm) - 1.0
    img = np.zeros((n, n), dtype=np.complex128)
    for (u, v, w), vk, wk in zip(uvw.astype(np.float64), vis, weights):
        img += wk * vk * np.exp(-2j * np.pi * (u * ll + v * mm + w * nn))
    return img / np.sum(weights)


def mosaic_gamma(beams: np.ndarray) -> np.ndarray:
    """Eq. 1: gamma = [sqrt(sum B_i^2) / max sqrt(sum B_i^2)]_PBP * [1 / sum B_i^2]_WC."""
    ssq = np.sum(np.asarray(beams, dtype=np.float64) ** 2, axis=0)
    root = np.sqrt(ssq)
    return (root / root.max()) * (1.0 / ssq)
