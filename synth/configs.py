"""The five synthetic workloads of BASELINE.json (`configs[0..4]`, called config 1..5 here).

Only data layout and random draws live here; see DESIGN.md "Input recipe".  The paper's own
measurement sets (ASKAP / ALMA) are not available, so these stand in for them.

Draw order (numpy `default_rng(seed)`): antenna radii, antenna azimuths, leakage phases,
visibilities.  uvw: textbook ENU -> (u, v, w) rotation for latitude phi, declination delta,
hour angle H, scaled by nu/c per channel, cast to float32, order [time][baseline][channel].

Chunks: `make_workload(name, time_range=(t0, t1))` builds only the (strided) time steps t0 <= t < t1 of an ASKAP-like
workload (configs 2, 3, 5) with the cell size, w_max and parallactic-angle bins of the FULL track; the chunk's
visibilities come from their own generator, `default_rng([seed, t0])`, so that config 5 (181 M visibilities x 4
correlations, 11.6 GB of inputs) can be produced and fed chunk by chunk without ever being held whole.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

C_LIGHT = 299792458.0

# kernel_mode values mirror include/imager.h (plain integers, no code shared)
MODE_DELTA, MODE_PSWF, MODE_WPROJ, MODE_AWPROJ_ADJOINT, MODE_AWPROJ_PAPER, MODE_MOSAIC_PB, MODE_USER = range(7)


@dataclass
class Workload:
    name: str
    params: dict                      # fields of imager_params (include/imager.h)
    uvw: np.ndarray                   # float32 [nvis, 3], wavelengths
    vis: np.ndarray                   # complex64 [nvis, n_corr]
    weights: np.ndarray               # float32 [nvis, n_corr]
    a_index: np.ndarray | None        # int32 [nvis] or None
    notes: dict = field(default_factory=dict)

    @property
    def nvis(self) -> int:
        return int(self.uvw.shape[0])


def _array_xyz(n_ant: int, radius_m: float, lat_deg: float, rng) -> tuple[np.ndarray, ...]:
    r = radius_m * np.sqrt(rng.random(n_ant))
    th = 2.0 * np.pi * rng.random(n_ant)
    east, north = r * np.cos(th), r * np.sin(th)
    lat = np.deg2rad(lat_deg)
    x = -np.sin(lat) * north
    y = east
    z = np.cos(lat) * north
    i, j = np.triu_indices(n_ant, 1)
    return x[j] - x[i], y[j] - y[i], z[j] - z[i]


def uvw_tracks(bx, by, bz, dec_deg: float, hour_angles_h: np.ndarray, freqs_hz: np.ndarray) -> np.ndarray:
    """float32 [ntime, nbl, nchan, 3] in wavelengths for baselines (bx,by,bz) in metres."""
    dec = np.deg2rad(dec_deg)
    h = np.deg2rad(15.0 * np.asarray(hour_angles_h, dtype=np.float64))[:, None]
    u = np.sin(h) * bx + np.cos(h) * by
    v = -np.sin(dec) * np.cos(h) * bx + np.sin(dec) * np.sin(h) * by + np.cos(dec) * bz
    w = np.cos(dec) * np.cos(h) * bx - np.cos(dec) * np.sin(h) * by + np.sin(dec) * bz
    s = (np.asarray(freqs_hz, dtype=np.float64) / C_LIGHT)[None, None, :]
    out = np.empty(u.shape + (s.shape[-1], 3), dtype=np.float32)
    out[..., 0] = u[:, :, None] * s
    out[..., 1] = v[:, :, None] * s
    out[..., 2] = w[:, :, None] * s
    return out


def _parallactic(hour_angles_h, lat_deg, dec_deg):
    h = np.deg2rad(15.0 * np.asarray(hour_angles_h, dtype=np.float64))
    lat, dec = np.deg2rad(lat_deg), np.deg2rad(dec_deg)
    return np.arctan2(np.sin(h) * np.cos(lat), np.sin(lat) * np.cos(dec) - np.cos(lat) * np.sin(dec) * np.cos(h))


def _normal_vis(rng, nvis: int, n_corr: int) -> np.ndarray:
    out = np.empty((nvis, n_corr), dtype=np.complex64)
    step = 1 << 22
    for a in range(0, nvis, step):
        b = min(nvis, a + step)
        z = rng.standard_normal((b - a, n_corr, 2), dtype=np.float32)
        out[a:b] = z[..., 0] + 1j * z[..., 1]
    return out


def _cell_from_uv(uvw: np.ndarray, n: int) -> float:
    umax = float(max(np.abs(uvw[..., 0]).max(), np.abs(uvw[..., 1]).max()))
    du = umax / (0.4 * n)
    return 1.0 / (n * du)


def _askap_like(name, seed, n_time, n_chan, hours, grid, n_corr, n_wplanes, smin, smax, mode,
                n_aplanes, time_stride, time_range=None):
    rng = np.random.default_rng(seed)
    lat, dec = -26.7, -30.0
    bx, by, bz = _array_xyz(36, 3000.0, lat, rng)
    leak_phase = 2.0 * np.pi * rng.random(2)
    hs = np.linspace(-hours / 2, hours / 2, n_time)
    freqs = 1.0e9 + 1.0e6 * np.arange(n_chan)
    # cell size and w_max always come from the FULL track so that a strided subset keeps the geometry
    umax = wmax = 0.0
    for a in range(0, n_time, 50):
        t = uvw_tracks(bx, by, bz, dec, hs[a:a + 50], freqs[[0, -1]])
        umax = max(umax, float(np.abs(t[..., :2]).max()))
        wmax = max(wmax, float(np.abs(t[..., 2]).max()))
    cell = 1.0 / (grid * (umax / (0.4 * grid)))
    hs_used = hs[::time_stride]
    t0, t1 = (0, len(hs_used)) if time_range is None else (int(time_range[0]), min(int(time_range[1]), len(hs_used)))
    n_time_all = len(hs_used)
    hs_used = hs_used[t0:t1]
    uvw = np.concatenate([uvw_tracks(bx, by, bz, dec, hs_used[a:a + 25], freqs).reshape(-1, 3)
                          for a in range(0, len(hs_used), 25)])
    nvis = uvw.shape[0]
    a_index, pa_centres = None, np.zeros(n_aplanes)
    if n_aplanes > 1:
        chi = _parallactic(hs, lat, dec)
        lo, hi = float(chi.min()), float(chi.max())
        width = (hi - lo) / n_aplanes
        bins = np.minimum(n_aplanes - 1, np.floor((chi - lo) / width).astype(np.int64))
        pa_centres = lo + (np.arange(n_aplanes) + 0.5) * width
        per_time = bins[::time_stride][t0:t1].astype(np.int32)
        a_index = np.repeat(per_time, bx.size * n_chan)
    vis = _normal_vis(rng if time_range is None else np.random.default_rng([seed, t0]), nvis, n_corr)
    params = dict(grid_size=grid, cell_size_rad=cell, n_corr=n_corr, n_pol=n_corr, n_wplanes=n_wplanes,
                  w_max=wmax, support_min=smin, support_max=smax, oversample=4, n_aplanes=n_aplanes,
                  kernel_mode=mode, dish_diameter_m=12.0, freq_hz=1.0e9,
                  leakage=[0.01 * np.exp(1j * leak_phase[0]), 0.01 * np.exp(1j * leak_phase[1])],
                  pa_rad=[float(x) for x in pa_centres], pointing_lm=[[0.0, 0.0]] * n_aplanes,
                  pswf_support=7)
    return Workload(name, params, uvw, vis, np.ones((nvis, n_corr), np.float32), a_index,
                    notes=dict(n_time=len(hs_used), n_time_all=n_time_all, n_chan=n_chan, n_baselines=int(bx.size), umax=umax))


def _hex_pointings(n_point: int, spacing: float) -> np.ndarray:
    pts = []
    for j in range(-8, 9):
        for i in range(-8, 9):
            pts.append((i * i + i * j + j * j, j, i))
    pts.sort()
    out = np.array([[spacing * (i + 0.5 * j), spacing * (np.sqrt(3.0) / 2.0) * j] for _, j, i in pts[:n_point]])
    return out


def _config1(seed):
    rng = np.random.default_rng(seed)
    n, nvis, cell = 256, 10000, 2.0e-4
    du = 1.0 / (n * cell)
    u = (rng.random(nvis) * 2 - 1) * 0.4 * n * du
    v = (rng.random(nvis) * 2 - 1) * 0.4 * n * du
    uvw = np.stack([u, v, np.zeros(nvis)], axis=1).astype(np.float32)
    vis = _normal_vis(rng, nvis, 1)
    params = dict(grid_size=n, cell_size_rad=cell, n_corr=1, n_pol=1, n_wplanes=1, w_max=0.0, support_min=7,
                  support_max=7, oversample=8, n_aplanes=1, kernel_mode=MODE_PSWF, dish_diameter_m=12.0,
                  freq_hz=1.0e9, leakage=[0j, 0j], pa_rad=[0.0], pointing_lm=[[0.0, 0.0]], pswf_support=7)
    return Workload("config1_tiny", params, uvw, vis, np.ones((nvis, 1), np.float32), None)


def _config4(seed, time_stride):
    rng = np.random.default_rng(seed)
    lat, dec, n, n_point, n_int = -23.0, -30.0, 512, 50, 82
    bx, by, bz = _array_xyz(50, 500.0, lat, rng)
    hs = np.linspace(-1.0, 1.0, n_point * n_int)            # pointings interleaved: step t -> pointing t % 50
    freqs = np.array([100.0e9])
    full = uvw_tracks(bx, by, bz, dec, hs, freqs)
    cell = _cell_from_uv(full, n)
    keep = np.arange(0, hs.size, time_stride)
    uvw = full[keep].reshape(-1, 3)
    a_index = np.repeat((keep % n_point).astype(np.int32), bx.size)
    nvis = uvw.shape[0]
    vis = _normal_vis(rng, nvis, 1)
    field_rad = n * cell
    pointings = _hex_pointings(n_point, field_rad / 12.0)
    params = dict(grid_size=n, cell_size_rad=cell, n_corr=1, n_pol=1, n_wplanes=1, w_max=0.0, support_min=64,
                  support_max=64, oversample=4, n_aplanes=n_point, kernel_mode=MODE_MOSAIC_PB,
                  dish_diameter_m=12.0, freq_hz=100.0e9, leakage=[0j, 0j], pa_rad=[0.0] * n_point,
                  pointing_lm=[[float(a), float(b)] for a, b in pointings], pswf_support=7)
    return Workload("config4_mosaic", params, uvw, vis, np.ones((nvis, 1), np.float32), a_index,
                    notes=dict(n_time=len(keep), n_baselines=int(bx.size)))


CONFIGS = ("config1", "config2", "config3", "config4", "config5")


def make_workload(name: str, seed: int = 0, time_stride: int = 1, time_range=None) -> Workload:
    """Build one of the five workloads.  `time_stride` > 1 keeps every n-th time step (a smaller
    workload with the same geometry, cell size and w_max) for tests and bounded CPU samples; `time_range` = (t0, t1)
    keeps the (strided) time steps t0 <= t < t1 only (configs 2, 3, 5: chunked feeding, see the module docstring)."""
    if time_range is not None and name not in ("config2", "config3", "config5"):
        raise ValueError("time_range applies to the ASKAP-like workloads only")
    if name == "config1":
        return _config1(seed)
    if name == "config2":
        return _askap_like("config2_wproj", seed, 300, 64, 8.0, 2048, 1, 32, 15, 63, MODE_WPROJ, 1, time_stride, time_range)
    if name == "config3":
        return _askap_like("config3_aproj", seed, 300, 64, 8.0, 4096, 4, 8, 31, 31, MODE_AWPROJ_ADJOINT, 4,
                           time_stride, time_range)
    if name == "config4":
        return _config4(seed, time_stride)
    if name == "config5":
        return _askap_like("config5_major", seed, 1000, 288, 8.0, 8192, 4, 64, 15, 127, MODE_AWPROJ_ADJOINT, 4,
                           time_stride, time_range)
    raise ValueError(f"unknown workload {name!r}")
