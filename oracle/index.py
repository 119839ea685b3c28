"""Oracle steps O1 (index) and O2 (bucketing).  TEST INFRASTRUCTURE (see oracle/__init__.py).

The paper names gridding but gives no uv -> cell mapping; the reading
followed here is DESIGN.md R2-R5/R8 (= SURVEY.md section 8(c) O1, S2-S5, S8):

  uv_scale = O * N * cell            (double; O*N is exact, one rounding)
  q   = rint(double(u) * uv_scale)   (one IEEE multiply, round-half-to-even)  -- fine lattice, O per cell
  i   = floor((q + O/2) / O),  o = q - i*O  in [-O/2, O/2-1],  g = i + N/2
  p   = min(P-1, rint(|w| * (P-1)/w_max)),  sp = -p if w < 0 else p     (signed w-plane)
  kset = a_index * (2P-1) + (sp + P-1)
  S_p = support_min + 2*rint(((support_max-support_min)/2) * p/(P-1));  taps d in [-h_lo, h_hi],
        h_lo = S//2, h_hi = S-1-h_lo;  drop if the footprint leaves the grid.
  R17 (invalid input): u, v or w not finite, |u * uv_scale| or |v * uv_scale| >= 2^30, or a_index outside
        [0, n_aplanes)  ->  dropped, with the fixed record gx = gy = 0, ox = oy = -O/2, sp = 0, kset = 0.

Integer outputs: compared BIT-EXACTLY with the CUDA path.
"""
from __future__ import annotations

import numpy as np

KEY_DROP = np.uint32(0xFFFFFFFF)


def support_schedule(support_min: int, support_max: int, n_wplanes: int) -> np.ndarray:
    """S_p for p = 0..P-1 (R5).  Parity of support_min is preserved."""
    if n_wplanes == 1:
        return np.array([support_min], dtype=np.int64)
    if (support_max - support_min) % 2:
        raise ValueError("support_max - support_min must be even")
    half = (support_max - support_min) // 2
    return np.array([support_min + 2 * int(np.rint(half * p / (n_wplanes - 1))) for p in range(n_wplanes)],
                    dtype=np.int64)


def index_visibilities(uvw: np.ndarray, a_index: np.ndarray | None, params: dict) -> dict:
    """O1.  uvw float32 [nvis,3].  Returns int64 arrays gx, gy, ox, oy, sp, a, kset, support and bool drop."""
    n = int(params["grid_size"])
    o = int(params["oversample"])
    p_count = int(params["n_wplanes"])
    uv_scale = float(o) * float(n) * float(params["cell_size_rad"])
    w_scale = (p_count - 1) / float(params["w_max"]) if p_count > 1 else 0.0
    u = uvw[:, 0].astype(np.float64)
    v = uvw[:, 1].astype(np.float64)
    w = uvw[:, 2].astype(np.float64)
    a = np.zeros(len(u), dtype=np.int64) if a_index is None else np.asarray(a_index, dtype=np.int64)
    with np.errstate(invalid="ignore"):
        invalid = ~(np.isfinite(u) & np.isfinite(v) & np.isfinite(w))
        invalid |= ~(np.abs(u * uv_scale) < 2.0 ** 30) | ~(np.abs(v * uv_scale) < 2.0 ** 30)
    invalid |= (a < 0) | (a >= int(params["n_aplanes"]))                # R17
    u, v, w, a = (np.where(invalid, 0, x) for x in (u, v, w, a))
    qx = np.rint(u * uv_scale).astype(np.int64)
    qy = np.rint(v * uv_scale).astype(np.int64)
    half_o = o // 2
    ix = (qx + half_o) // o           # numpy // on integers is floor division
    iy = (qy + half_o) // o
    ox = qx - ix * o
    oy = qy - iy * o
    gx = ix + n // 2
    gy = iy + n // 2
    p = np.minimum(p_count - 1, np.rint(np.abs(w) * w_scale).astype(np.int64))
    sp = np.where(w < 0, -p, p)
    kset = a * (2 * p_count - 1) + (sp + p_count - 1)
    sched = support_schedule(int(params["support_min"]), int(params["support_max"]), p_count)
    support = sched[p]
    h_lo = support // 2
    h_hi = support - 1 - h_lo
    drop = (gx - h_lo < 0) | (gx + h_hi >= n) | (gy - h_lo < 0) | (gy + h_hi >= n) | invalid
    zero = np.int64(0)
    gx, gy, sp, kset = (np.where(invalid, zero, x) for x in (gx, gy, sp, kset))
    ox, oy = np.where(invalid, -half_o, ox), np.where(invalid, -half_o, oy)
    return dict(gx=gx, gy=gy, ox=ox, oy=oy, sp=sp, a=a, kset=kset, support=support, drop=drop)


def pack_records(rec: dict, oversample: int) -> np.ndarray:
    """The 16-byte record the C-ABI debug export returns (include/imager.h `imager_record`):
    int32 gx, int32 gy, uint32 sub = (ox+O/2) | (oy+O/2) << 8 | drop << 16, int32 kset."""
    half_o = oversample // 2
    out = np.empty((len(rec["gx"]), 4), dtype=np.int32)
    out[:, 0] = rec["gx"]
    out[:, 1] = rec["gy"]
    out[:, 2] = (rec["ox"] + half_o) | ((rec["oy"] + half_o) << 8) | (rec["drop"].astype(np.int64) << 16)
    out[:, 3] = rec["kset"]
    return out


def bucket_keys(rec: dict, params: dict, tile: int) -> np.ndarray:
    """O2 key: a pure integer function of the record,
        key = ((kset * nty + gy // tile) * ntx + gx // tile) * O*O + (oy+O/2)*O + (ox+O/2),
    nty = ntx = ceil(N / tile); dropped visibilities get KEY_DROP so that they sort last."""
    n = int(params["grid_size"])
    o = int(params["oversample"])
    nt = -(-n // tile)
    half_o = o // 2
    sub = (rec["oy"] + half_o) * o + (rec["ox"] + half_o)
    key = ((rec["kset"] * nt + rec["gy"] // tile) * nt + rec["gx"] // tile) * (o * o) + sub
    if np.any(key[~rec["drop"]] >= int(KEY_DROP)) or np.any(key[~rec["drop"]] < 0):
        raise ValueError("bucket key does not fit 32 bits")
    return np.where(rec["drop"], np.int64(KEY_DROP), key).astype(np.uint32)


def bucket_sort(keys: np.ndarray, params: dict, tile: int) -> dict:
    """Stable sort by key; bucket b = key // O^2 (= (kset * nty + ty) * ntx + tx), dropped excluded.
    Returns perm (int32, sorted position -> input index), the sorted keys, n_kept, and the dense
    bucket_offset[n_buckets + 1] (bucket b occupies sorted positions bucket_offset[b] .. bucket_offset[b+1])."""
    o = int(params["oversample"])
    nt = -(-int(params["grid_size"]) // tile)
    n_sets = int(params["n_aplanes"]) * (2 * int(params["n_wplanes"]) - 1)
    n_buckets = n_sets * nt * nt
    perm = np.argsort(keys, kind="stable").astype(np.int32)
    skeys = keys[perm]
    n_kept = int(np.searchsorted(skeys, KEY_DROP, side="left"))
    edges = np.arange(n_buckets + 1, dtype=np.int64) * (o * o)
    offsets = np.searchsorted(skeys[:n_kept].astype(np.int64), edges, side="left").astype(np.int32)
    return dict(perm=perm, sorted_keys=skeys, n_kept=n_kept, bucket_offset=offsets)
