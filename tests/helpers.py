"""Shared test helpers: small random workloads and thin wrappers that run the ORACLE end to end."""
import numpy as np

from oracle import index as oidx, kernels as okern, gridder as ogrid

MODE_DELTA, MODE_PSWF, MODE_WPROJ, MODE_AWPROJ_ADJOINT, MODE_AWPROJ_PAPER, MODE_MOSAIC_PB, MODE_USER = range(7)


def base_params(**kw):
    p = dict(grid_size=64, cell_size_rad=1.0e-3, n_corr=1, n_pol=1, n_wplanes=1, w_max=0.0, support_min=7,
             support_max=7, oversample=8, n_aplanes=1, kernel_mode=MODE_PSWF, dish_diameter_m=12.0,
             freq_hz=1.0e9, leakage=[0j, 0j], pa_rad=[0.0], pointing_lm=[[0.0, 0.0]], pswf_support=7)
    p.update(kw)
    return p


def random_vis(params, nvis, seed, frac=0.3, a_planes=False):
    rng = np.random.default_rng(seed)
    n, cell = params["grid_size"], params["cell_size_rad"]
    du = 1.0 / (n * cell)
    uvw = np.empty((nvis, 3), np.float32)
    uvw[:, 0] = (rng.random(nvis) * 2 - 1) * frac * n * du
    uvw[:, 1] = (rng.random(nvis) * 2 - 1) * frac * n * du
    uvw[:, 2] = (rng.random(nvis) * 2 - 1) * params["w_max"]
    nc = params["n_corr"]
    vis = (rng.standard_normal((nvis, nc)) + 1j * rng.standard_normal((nvis, nc))).astype(np.complex64)
    wts = (0.5 + rng.random((nvis, nc))).astype(np.float32)
    a = rng.integers(0, params["n_aplanes"], nvis).astype(np.int32) if a_planes else None
    return uvw, vis, wts, a


def oracle_tables(params, which="grid"):
    tabs, supports = okern.make_tables(params, which)
    flat, offs = okern.flatten_tables(tabs)
    return tabs, supports, flat, offs


def oracle_grid(params, uvw, vis, wts, a_index=None, flat=None, offs=None, **kw):
    rec = oidx.index_visibilities(uvw, a_index, params)
    if flat is None:
        _, _, flat, offs = oracle_tables(params)
    return ogrid.grid(rec, vis, wts, flat, offs, params, **kw), rec


def oracle_degrid(params, uvw, grid_c64, a_index=None, flat=None, offs=None, **kw):
    rec = oidx.index_visibilities(uvw, a_index, params)
    if flat is None:
        _, _, flat, offs = oracle_tables(params, "degrid")
    return ogrid.degrid(rec, grid_c64, flat, offs, params, **kw), rec
