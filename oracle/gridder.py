"""ctypes wrapper of oracle/gridder.c (O4 gridding, O5 degridding).  TEST INFRASTRUCTURE (oracle/__init__.py).

`build()` compiles gridder.c with gcc into oracle/_build/liboracle.so (done on first use and by
`__graft_entry__.build()`).  Nothing here touches CUDA.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "_build", "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "gridder.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        os.makedirs(os.path.dirname(_SO), exist_ok=True)
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _SO, src, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_max_threads.restype = ctypes.c_int
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _rec_arrays(rec):
    names = ("gx", "gy", "ox", "oy", "kset", "support")
    arrs = [np.ascontiguousarray(rec[n], dtype=np.int64) for n in names]
    arrs.append(np.ascontiguousarray(rec["drop"], dtype=np.uint8))
    return arrs


def grid(rec: dict, vis: np.ndarray, weights: np.ndarray, tables: np.ndarray, offsets: np.ndarray,
         params: dict, n_threads: int | None = None, sample_cells: np.ndarray | None = None) -> dict:
    """O4.  rec from oracle.index.index_visibilities; tables/offsets from oracle.kernels.flatten_tables.
    Returns grid complex128 [n_pol][N][N], norm float64, sumwt [n_corr]; or, with sample_cells int [n,2] (y,x),
    `samples` complex128 [n_pol][n] and `sample_norm` in the order given."""
    lib = _load()
    n, n_corr, n_pol, o = (int(params[k]) for k in ("grid_size", "n_corr", "n_pol", "oversample"))
    nvis = len(rec["gx"])
    arrs = _rec_arrays(rec)
    vis = np.ascontiguousarray(vis, dtype=np.complex64).reshape(nvis, n_corr)
    weights = np.ascontiguousarray(weights, dtype=np.float32).reshape(nvis, n_corr)
    tables = np.ascontiguousarray(tables, dtype=np.complex64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    sumwt = np.zeros(n_corr)
    nt = n_threads or max_threads()
    if sample_cells is None:
        g = np.zeros((n_pol, n, n), dtype=np.complex128)
        a = np.zeros((n_pol, n, n))
        lib.oracle_grid(ctypes.c_int64(nvis), n, n_corr, n_pol, o, *map(_p, arrs), _p(vis), _p(weights),
                        _p(tables), _p(offsets), _p(g), _p(a), _p(sumwt), None, None, ctypes.c_int64(0),
                        None, None, nt)
        return dict(grid=g, norm=a, sumwt=sumwt)
    cells = np.asarray(sample_cells, dtype=np.int64)
    order = np.lexsort((cells[:, 1], cells[:, 0]))
    sy, sx = cells[order, 0], np.ascontiguousarray(cells[order, 1])
    rowptr = np.searchsorted(sy, np.arange(n + 1), side="left").astype(np.int64)
    out = np.zeros((n_pol, len(cells)), dtype=np.complex128)
    onorm = np.zeros((n_pol, len(cells)))
    lib.oracle_grid(ctypes.c_int64(nvis), n, n_corr, n_pol, o, *map(_p, arrs), _p(vis), _p(weights),
                    _p(tables), _p(offsets), None, None, _p(sumwt), _p(rowptr), _p(sx),
                    ctypes.c_int64(len(cells)), _p(out), _p(onorm), nt)
    inv = np.empty_like(order)
    inv[order] = np.arange(len(order))
    return dict(samples=out[:, inv], sample_norm=onorm[:, inv], sumwt=sumwt)


def degrid(rec: dict, grid_c64: np.ndarray, tables: np.ndarray, offsets: np.ndarray, params: dict,
           n_threads: int | None = None) -> dict:
    """O5.  grid_c64 complex64 [n_pol][N][N].  Returns vis complex128 [nvis][n_corr] and norm float64."""
    lib = _load()
    n, n_corr, n_pol, o = (int(params[k]) for k in ("grid_size", "n_corr", "n_pol", "oversample"))
    nvis = len(rec["gx"])
    arrs = _rec_arrays(rec)
    g = np.ascontiguousarray(grid_c64, dtype=np.complex64).reshape(n_pol, n, n)
    tables = np.ascontiguousarray(tables, dtype=np.complex64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    out = np.zeros((nvis, n_corr), dtype=np.complex128)
    onorm = np.zeros((nvis, n_corr))
    lib.oracle_degrid(ctypes.c_int64(nvis), n, n_corr, n_pol, o, *map(_p, arrs), _p(g), _p(tables), _p(offsets),
                      _p(out), _p(onorm), n_threads or max_threads())
    return dict(vis=out, norm=onorm)
