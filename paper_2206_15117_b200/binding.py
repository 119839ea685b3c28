"""Thin ctypes binding of libimager.so (include/imager.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; torch is used for device memory and
streams.  There is no CPU fallback: if the shared library is missing or no CUDA device is present, calls fail
loudly (`ImagerError`).
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_float, c_int32, c_int64, c_uint32, c_void_p)

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("IMAGER_LIBRARY") or os.path.join(_HERE, "libimager.so")   # IMAGER_LIBRARY: e.g. the checked build

MODE_DELTA, MODE_PSWF, MODE_WPROJ, MODE_AWPROJ_ADJOINT, MODE_AWPROJ_PAPER, MODE_MOSAIC_PB, MODE_USER = range(7)
REUSE_INDEX = 1
PATH_REFERENCE = 2
DEGRID_RESIDUAL = 16

EXPORTS = ("imager_plan_create", "imager_index", "imager_grid", "imager_degrid", "imager_plan_destroy",
           "imager_grid_image_transform", "imager_mosaic_correct", "imager_debug_index", "imager_debug_kernels", "imager_plan_info", "imager_plan_path",
           "imager_index_stats", "imager_hogbom", "imager_hogbom_static", "imager_clean", "imager_reproject", "imager_mosaic_grid",
           "imager_mosaic_degrid",
           "imager_last_launch_count", "imager_debug_violations", "imager_debug_probe", "imager_last_error")


class ImagerError(RuntimeError):
    pass


class ImagerParams(Structure):
    _fields_ = [("grid_size", c_int32), ("n_corr", c_int32), ("n_pol", c_int32), ("n_wplanes", c_int32),
                ("support_min", c_int32), ("support_max", c_int32), ("oversample", c_int32), ("n_aplanes", c_int32),
                ("kernel_mode", c_int32), ("pswf_support", c_int32), ("cell_size_rad", c_double), ("w_max", c_double),
                ("dish_diameter_m", c_double), ("freq_hz", c_double), ("leakage", c_double * 4), ("beam_eps", c_double),
                ("pa_rad", POINTER(c_double)), ("pointing_lm", POINTER(c_double)), ("user_tables", POINTER(c_float)),
                ("user_tables_degrid", POINTER(c_float)), ("max_nvis", c_int64)]


class ImagerCleanParams(Structure):
    _fields_ = [("n_major", c_int32), ("n_iter", c_int32), ("gain", c_float), ("threshold", c_float), ("cycle_factor", c_float)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libimager.so (built in-tree by paper_2206_15117_b200.build).  Raises ImagerError if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImagerError(f"{LIB_PATH} is missing: run `python -m paper_2206_15117_b200.build` (there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    lib.imager_last_error.restype = c_char_p
    lib.imager_plan_create.argtypes = [POINTER(ImagerParams), c_void_p, POINTER(c_void_p)]
    lib.imager_grid.argtypes = [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_uint32,
                                c_void_p]
    lib.imager_index.argtypes = [c_void_p, c_int64, c_void_p, c_void_p, c_void_p]
    lib.imager_degrid.argtypes = [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, c_uint32, c_void_p]
    lib.imager_plan_destroy.argtypes = [c_void_p]
    lib.imager_grid_image_transform.argtypes = [c_void_p, c_void_p, c_int32, c_double, c_void_p]
    lib.imager_mosaic_correct.argtypes = [c_void_p, c_void_p, c_void_p]
    lib.imager_debug_index.argtypes = [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                       POINTER(c_int64), c_void_p]
    lib.imager_debug_kernels.argtypes = [c_void_p, c_int32, c_int32, c_void_p, POINTER(c_int32)]
    lib.imager_plan_info.argtypes = [c_void_p, POINTER(c_int64)]
    lib.imager_plan_path.argtypes = [c_void_p, c_char_p, c_int32]
    lib.imager_index_stats.argtypes = [c_void_p, POINTER(c_int64), c_void_p]
    lib.imager_reproject.argtypes = [c_void_p, c_int32, c_double, c_void_p, c_int32, c_double, c_double, c_double, c_int32,
                                     c_double, c_double, c_int32, c_int32, c_void_p]
    lib.imager_mosaic_grid.argtypes = [c_void_p, c_int32, POINTER(c_int64), POINTER(c_void_p), POINTER(c_void_p), POINTER(c_void_p),
                                       POINTER(c_double), c_void_p, c_int32, c_double, c_void_p, c_void_p]
    lib.imager_mosaic_degrid.argtypes = [c_void_p, c_int32, POINTER(c_int64), POINTER(c_void_p), POINTER(c_double), c_void_p,
                                         c_int32, c_double, POINTER(c_void_p), c_uint32, c_void_p]
    lib.imager_hogbom.argtypes = [c_void_p, c_void_p, c_void_p, c_int32, POINTER(c_int32), c_float, c_float, c_float, c_int32,
                                  c_void_p, c_void_p, c_void_p]
    lib.imager_hogbom_static.argtypes = lib.imager_hogbom.argtypes
    lib.imager_clean.argtypes = [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, POINTER(ImagerCleanParams), c_void_p,
                                 c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.imager_last_launch_count.argtypes = [c_void_p]
    lib.imager_debug_violations.argtypes = [POINTER(c_int64)]
    lib.imager_debug_probe.argtypes = [POINTER(c_double), c_void_p]
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != 0:
        msg = load_library().imager_last_error().decode()
        raise ImagerError(f"{what} failed with status {rc}: {msg}")


def _dev_ptr(t, dtype, what):
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise ImagerError(f"{what} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise ImagerError(f"{what} must be a contiguous {dtype} tensor")
    return c_void_p(t.data_ptr())


def _stream_ptr(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return c_void_p(s.cuda_stream)


class Plan:
    """imager_plan_create / imager_plan_destroy.  `params` is a dict with the fields of imager_params
    (synth.Workload.params has exactly those); `user_tables` (complex64 numpy, canonical layout) selects USER mode."""

    def __init__(self, params: dict, max_nvis: int, user_tables: np.ndarray | None = None,
                 user_tables_degrid: np.ndarray | None = None, stream=None):
        lib = load_library()
        p = ImagerParams()
        for name in ("grid_size", "n_corr", "n_pol", "n_wplanes", "support_min", "support_max", "oversample", "n_aplanes",
                     "kernel_mode"):
            setattr(p, name, int(params[name]))
        p.pswf_support = int(params.get("pswf_support", 7))
        p.cell_size_rad = float(params["cell_size_rad"])
        p.w_max = float(params.get("w_max", 0.0))
        p.dish_diameter_m = float(params.get("dish_diameter_m", 0.0))
        p.freq_hz = float(params.get("freq_hz", 0.0))
        leak = params.get("leakage", [0j, 0j])
        p.leakage = (c_double * 4)(complex(leak[0]).real, complex(leak[0]).imag, complex(leak[1]).real, complex(leak[1]).imag)
        p.beam_eps = float(params.get("beam_eps", 0.0))
        self._keep = []
        if params.get("pa_rad") is not None:
            pa = np.ascontiguousarray(params["pa_rad"], dtype=np.float64)
            self._keep.append(pa)
            p.pa_rad = pa.ctypes.data_as(POINTER(c_double))
        if params.get("pointing_lm") is not None:
            lm = np.ascontiguousarray(params["pointing_lm"], dtype=np.float64).reshape(-1)
            self._keep.append(lm)
            p.pointing_lm = lm.ctypes.data_as(POINTER(c_double))
        if user_tables is not None:
            p.kernel_mode = MODE_USER
            ut = np.ascontiguousarray(user_tables, dtype=np.complex64)
            self._keep.append(ut)
            p.user_tables = ut.ctypes.data_as(POINTER(c_float))
            if user_tables_degrid is not None:
                ud = np.ascontiguousarray(user_tables_degrid, dtype=np.complex64)
                self._keep.append(ud)
                p.user_tables_degrid = ud.ctypes.data_as(POINTER(c_float))
        p.max_nvis = int(max_nvis)
        self.params = dict(params)
        self.n_corr, self.n_pol, self.grid_size = p.n_corr, p.n_pol, p.grid_size
        self._h = c_void_p()
        _check(lib.imager_plan_create(byref(p), _stream_ptr(stream), byref(self._h)), "imager_plan_create")
        self._keep = []

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            load_library().imager_plan_destroy(self._h)
            self._h = c_void_p()

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- hot path -------------------------------------------------------------------------------------------
    def index(self, uvw, a_index=None, stream=None):
        """A1 + A2 ahead of time; follow with grid / degrid calls that pass REUSE_INDEX."""
        import torch
        nvis = int(uvw.shape[0])
        _check(load_library().imager_index(self._h, nvis, _dev_ptr(uvw, torch.float32, "uvw"),
                                           _dev_ptr(a_index, torch.int32, "a_index"), _stream_ptr(stream)), "imager_index")

    def grid(self, uvw, vis, weights, grid, a_index=None, sum_weights=None, flags: int = 0, stream=None):
        """imager_grid: accumulates into `grid` (complex64 [n_pol,N,N] CUDA tensor)."""
        import torch
        nvis = int(uvw.shape[0]) if uvw is not None else int(vis.shape[0])
        _check(load_library().imager_grid(
            self._h, nvis, _dev_ptr(uvw, torch.float32, "uvw"), _dev_ptr(vis, torch.complex64, "vis"),
            _dev_ptr(weights, torch.float32, "weights"), _dev_ptr(a_index, torch.int32, "a_index"),
            _dev_ptr(grid, torch.complex64, "grid"), _dev_ptr(sum_weights, torch.float64, "sum_weights"),
            flags, _stream_ptr(stream)), "imager_grid")

    def degrid(self, uvw, grid, vis_out, a_index=None, flags: int = 0, stream=None):
        """imager_degrid: overwrites `vis_out` (complex64 [nvis,n_corr] CUDA tensor)."""
        import torch
        nvis = int(vis_out.shape[0])
        _check(load_library().imager_degrid(
            self._h, nvis, _dev_ptr(uvw, torch.float32, "uvw"), _dev_ptr(a_index, torch.int32, "a_index"),
            _dev_ptr(grid, torch.complex64, "grid"), _dev_ptr(vis_out, torch.complex64, "vis_out"), flags,
            _stream_ptr(stream)), "imager_degrid")

    # ---- surrounding stages ---------------------------------------------------------------------------------
    def grid_image_transform(self, data, direction: int, norm: float = 1.0, stream=None):
        import torch
        _check(load_library().imager_grid_image_transform(self._h, _dev_ptr(data, torch.complex64, "data"), direction,
                                                          float(norm), _stream_ptr(stream)), "imager_grid_image_transform")

    def mosaic_correct(self, image, stream=None):
        """Eq. 1: multiply the image planes by gamma(l, m) in place (MOSAIC_PB plans)."""
        import torch
        _check(load_library().imager_mosaic_correct(self._h, _dev_ptr(image, torch.complex64, "image"), _stream_ptr(stream)),
               "imager_mosaic_correct")

    def clean(self, uvw, vis, weights, model_image, residual_image, residual_vis, n_major: int, n_iter: int, gain: float,
              threshold: float, cycle_factor: float, a_index=None, psf_out=None, n_components_out=None, stream=None):
        """imager_clean: Cotton-Schwab major cycles around the hot path (single-polarisation plans)."""
        import torch
        cp = ImagerCleanParams(int(n_major), int(n_iter), float(gain), float(threshold), float(cycle_factor))
        _check(load_library().imager_clean(
            self._h, int(uvw.shape[0]), _dev_ptr(uvw, torch.float32, "uvw"), _dev_ptr(vis, torch.complex64, "vis"),
            _dev_ptr(weights, torch.float32, "weights"), _dev_ptr(a_index, torch.int32, "a_index"), byref(cp),
            _dev_ptr(model_image, torch.float32, "model_image"), _dev_ptr(residual_image, torch.float32, "residual_image"),
            _dev_ptr(residual_vis, torch.complex64, "residual_vis"), _dev_ptr(psf_out, torch.float32, "psf_out"),
            _dev_ptr(n_components_out, torch.int32, "n_components_out"), _stream_ptr(stream)), "imager_clean")

    @staticmethod
    def _ptr_array(tensors, dtype, what):
        return (c_void_p * len(tensors))(*[_dev_ptr(t, dtype, what).value for t in tensors])

    def mosaic_grid(self, uvw_list, vis_list, weights_list, pointing_lm, mosaic_image, cell_mosaic: float, sum_weights=None,
                    stream=None):
        """imager_mosaic_grid: image-domain mosaic of components given at their own phase centres (lists of CUDA tensors)."""
        import torch
        k = len(uvw_list)
        nv = (c_int64 * k)(*[int(u.shape[0]) for u in uvw_list])
        lm = np.ascontiguousarray(pointing_lm, dtype=np.float64).reshape(-1)
        _check(load_library().imager_mosaic_grid(
            self._h, k, nv, self._ptr_array(uvw_list, torch.float32, "uvw"), self._ptr_array(vis_list, torch.complex64, "vis"),
            self._ptr_array(weights_list, torch.float32, "weights"), lm.ctypes.data_as(POINTER(c_double)),
            _dev_ptr(mosaic_image, torch.complex64, "mosaic_image"), int(mosaic_image.shape[-1]), float(cell_mosaic),
            _dev_ptr(sum_weights, torch.float64, "sum_weights"), _stream_ptr(stream)), "imager_mosaic_grid")

    def mosaic_degrid(self, uvw_list, pointing_lm, model_image, cell_mosaic: float, vis_out_list, flags: int = 0, stream=None):
        """imager_mosaic_degrid: predicts every component's visibilities from a model image on the mosaic frame."""
        import torch
        k = len(uvw_list)
        nv = (c_int64 * k)(*[int(u.shape[0]) for u in uvw_list])
        lm = np.ascontiguousarray(pointing_lm, dtype=np.float64).reshape(-1)
        _check(load_library().imager_mosaic_degrid(
            self._h, k, nv, self._ptr_array(uvw_list, torch.float32, "uvw"), lm.ctypes.data_as(POINTER(c_double)),
            _dev_ptr(model_image, torch.complex64, "model_image"), int(model_image.shape[-1]), float(cell_mosaic),
            self._ptr_array(vis_out_list, torch.complex64, "vis_out"), flags, _stream_ptr(stream)), "imager_mosaic_degrid")

    def last_launch_count(self) -> int:
        return int(load_library().imager_last_launch_count(self._h))

    # ---- debug exports --------------------------------------------------------------------------------------
    def info(self) -> dict:
        out = (c_int64 * 8)()
        _check(load_library().imager_plan_info(self._h, out), "imager_plan_info")
        names = ("n_sets", "bucket_tile", "n_buckets", "key_bits", "n_dropped", "last_launches", "table_elems", "n_kept")
        return dict(zip(names, [int(x) for x in out]))

    def path(self) -> tuple[str, str]:
        """imager_plan_path: ("tiled", "") or ("reference", why the tiled kernels cannot run this plan)."""
        buf = ctypes.create_string_buffer(256)
        rc = load_library().imager_plan_path(self._h, buf, len(buf))
        if rc < 0:
            _check(rc, "imager_plan_path")
        return ("tiled" if rc == 1 else "reference", buf.value.decode())

    def index_stats(self, stream=None) -> dict:
        out = (c_int64 * 8)()
        _check(load_library().imager_index_stats(self._h, out, _stream_ptr(stream)), "imager_index_stats")
        names = ("n_kept", "n_dropped", "n_merged", "nominal_cmacs", "executed_cmacs", "n_hits", "n_items")
        return dict(zip(names, [int(x) for x in out]))

    def debug_index(self, uvw, a_index=None, stream=None) -> dict:
        import torch
        nvis = int(uvw.shape[0])
        nb = self.info()["n_buckets"]
        rec = np.empty((nvis, 4), np.int32)
        perm = np.empty(nvis, np.int32)
        keys = np.empty(nvis, np.uint32)
        boff = np.empty(nb + 1, np.int32)
        n_kept = c_int64()
        _check(load_library().imager_debug_index(
            self._h, nvis, _dev_ptr(uvw, torch.float32, "uvw"), _dev_ptr(a_index, torch.int32, "a_index"),
            rec.ctypes.data_as(c_void_p), perm.ctypes.data_as(c_void_p), keys.ctypes.data_as(c_void_p),
            boff.ctypes.data_as(c_void_p), byref(n_kept), _stream_ptr(stream)), "imager_debug_index")
        return dict(records=rec, perm=perm, sorted_keys=keys, bucket_offset=boff, n_kept=int(n_kept.value))

    def debug_kernels(self, kset: int, which: int = 0) -> np.ndarray:
        s = c_int32()
        _check(load_library().imager_debug_kernels(self._h, kset, which, None, byref(s)), "imager_debug_kernels")
        o = int(self.params["oversample"])
        out = np.empty((self.n_pol, self.n_corr, o, o, s.value, s.value), np.complex64)
        _check(load_library().imager_debug_kernels(self._h, kset, which, out.ctypes.data_as(c_void_p), byref(s)),
               "imager_debug_kernels")
        return out


def hogbom(residual, psf, model, window, gain: float, threshold: float, cycle_factor: float, n_iter: int, components_out=None,
           n_components_out=None, stream=None):
    """imager_hogbom: the minor cycle on float32 CUDA images [n][n]; window = (y0, x0, y1, x1)."""
    import torch
    n = int(residual.shape[-1])
    win = (c_int32 * 4)(*[int(v) for v in window])
    _check(load_library().imager_hogbom(
        _dev_ptr(residual, torch.float32, "residual"), _dev_ptr(psf, torch.float32, "psf"), _dev_ptr(model, torch.float32, "model"),
        n, win, float(gain), float(threshold), float(cycle_factor), int(n_iter), _dev_ptr(components_out, torch.float32, "components_out"),
        _dev_ptr(n_components_out, torch.int32, "n_components_out"), _stream_ptr(stream)), "imager_hogbom")


def debug_probe(stream=None) -> dict:
    """imager_debug_probe: clocks per warp instruction per SM of LDS.64 (32 and 16 active lanes) and FFMA2."""
    out = (c_double * 4)()
    _check(load_library().imager_debug_probe(out, _stream_ptr(stream)), "imager_debug_probe")
    return {"lds64_clk": out[0], "lds64_half_mask_clk": out[1], "ffma2_clk": out[2], "n_sm": int(out[3])}


HOGBOM_STATIC_MAX_N = 4096


def hogbom_static(residual, psf, model, window, gain: float, threshold: float, cycle_factor: float, n_iter: int,
                  components_out=None, n_components_out=None, stream=None):
    """imager_hogbom_static: the minor cycle of `hogbom`, same arguments and bit-identical results, for callers that may not
    allocate device memory (all HBM handed out at start-up, a caching allocator that owns the device, a real-time loop).
    The library calls no allocator here: its scratch is a 128 KB array built into libimager.so and shared by every call on
    that GPU, so images are limited to HOGBOM_STATIC_MAX_N pixels a side (ImagerError otherwise) and two calls that can
    overlap on one GPU race.  The first call on a device also looks up the array's address: make it before any stream
    capture.  (This Python wrapper itself allocates nothing on the device; the tensors are the caller's.)"""
    import torch
    n = int(residual.shape[-1])
    win = (c_int32 * 4)(*[int(v) for v in window])
    _check(load_library().imager_hogbom_static(
        _dev_ptr(residual, torch.float32, "residual"), _dev_ptr(psf, torch.float32, "psf"), _dev_ptr(model, torch.float32, "model"),
        n, win, float(gain), float(threshold), float(cycle_factor), int(n_iter), _dev_ptr(components_out, torch.float32, "components_out"),
        _dev_ptr(n_components_out, torch.int32, "n_components_out"), _stream_ptr(stream)), "imager_hogbom_static")


def reproject(src, cell_src: float, dst, cell_dst: float, shift_lm, beam: int = 0, dish_diameter_m: float = 0.0,
              freq_hz: float = 0.0, inner_half: bool = False, accumulate: bool = False, stream=None):
    """imager_reproject: bilinear image-plane reprojection between complex64 CUDA images (R22)."""
    import torch
    _check(load_library().imager_reproject(
        _dev_ptr(src, torch.complex64, "src"), int(src.shape[-1]), float(cell_src), _dev_ptr(dst, torch.complex64, "dst"),
        int(dst.shape[-1]), float(cell_dst), float(shift_lm[0]), float(shift_lm[1]), int(beam), float(dish_diameter_m),
        float(freq_hz), int(bool(inner_half)), int(bool(accumulate)), _stream_ptr(stream)), "imager_reproject")
