"""Pins for oracle step O1/O2 (index, bucketing): P1 (cell mapping), P10 (exact-arithmetic properties)."""
from fractions import Fraction

import numpy as np
from hypothesis import given, settings, strategies as st

from oracle import index as oidx
from helpers import base_params, MODE_WPROJ


def test_support_schedule_matches_baseline_configs():
    # BASELINE.json configs[1]: "support growing 15->63"; configs[4]: "support up to 127"
    s2 = oidx.support_schedule(15, 63, 32)
    assert s2[0] == 15 and s2[-1] == 63 and np.all(s2 % 2 == 1) and np.all(np.diff(s2) >= 0)
    s5 = oidx.support_schedule(15, 127, 64)
    assert s5[0] == 15 and s5[-1] == 127 and np.all(s5 % 2 == 1)
    assert list(oidx.support_schedule(64, 64, 1)) == [64]


@settings(max_examples=300, deadline=None)
@given(st.floats(-3.0e4, 3.0e4, width=32), st.floats(-3.0e4, 3.0e4, width=32), st.floats(-2.0e4, 2.0e4, width=32),
       st.sampled_from([1, 2, 4, 8]), st.sampled_from([64, 256, 2048]))
def test_index_against_exact_rational_arithmetic(u, v, w, o, n):
    """P10: the float pipeline equals exact rational arithmetic on the same float inputs
    (round-half-even of u*uv_scale where the product is the correctly rounded double)."""
    params = base_params(grid_size=n, oversample=o, cell_size_rad=1.0 / (n * 23.5), n_wplanes=32, w_max=16400.0,
                         support_min=15, support_max=63, kernel_mode=MODE_WPROJ)
    uvw = np.array([[u, v, w]], dtype=np.float32)
    r = oidx.index_visibilities(uvw, None, params)
    uv_scale = float(o) * float(n) * params["cell_size_rad"]
    for axis, (g, off) in enumerate(((r["gx"], r["ox"]), (r["gy"], r["oy"]))):
        prod = float(np.float64(uvw[0, axis])) * uv_scale           # correctly rounded IEEE product
        fr = Fraction(prod)
        q = round(fr)                                                # Python round(Fraction) is half-to-even
        assert abs(fr - q) <= Fraction(1, 2)
        i = (q + o // 2) // o
        assert int(g[0]) == i + n // 2
        assert int(off[0]) == q - i * o
        assert -(o // 2) <= int(off[0]) <= o - o // 2 - 1
        assert (int(g[0]) - n // 2) * o + int(off[0]) == q
    p = min(31, round(Fraction(abs(float(np.float64(uvw[0, 2]))) * (31 / 16400.0))))
    assert int(r["sp"][0]) == (-p if uvw[0, 2] < 0 else p)
    assert int(r["kset"][0]) == int(r["sp"][0]) + 31


def test_round_half_even_ties_and_symmetry():
    """Exact ties: u*uv_scale = k + 0.5 must round to the even neighbour, and q(-u) = -q(u) (needed by P3)."""
    n, o = 64, 4
    params = base_params(grid_size=n, oversample=o, cell_size_rad=1.0 / 256.0)   # uv_scale = 4*64/256 = 1.0 exactly
    u = np.array([0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 3.5], dtype=np.float32)
    uvw = np.stack([u, -u, np.zeros_like(u)], axis=1)
    r = oidx.index_visibilities(uvw, None, params)
    q = (r["gx"] - n // 2) * o + r["ox"]
    assert list(q) == [0, 2, 2, 0, -2, -2, 4]
    qy = (r["gy"] - n // 2) * o + r["oy"]
    assert np.array_equal(qy, -q)


def test_drop_flag_is_footprint_leaving_grid():
    n = 64
    params = base_params(grid_size=n, oversample=1, cell_size_rad=1.0 / n, support_min=7, support_max=7)  # uv_scale=1
    # gx = u + 32; footprint gx-3 .. gx+3 must stay in [0, 63]
    u = np.array([-29, -30, 28, 29, 0], dtype=np.float32)
    uvw = np.stack([u, np.zeros_like(u), np.zeros_like(u)], axis=1)
    r = oidx.index_visibilities(uvw, None, params)
    assert list(r["drop"]) == [False, True, False, True, False]
    # even support 4: taps -2..+1
    params = base_params(grid_size=n, oversample=1, cell_size_rad=1.0 / n, support_min=4, support_max=4)
    u = np.array([-30, -31, 30, 31], dtype=np.float32)
    uvw = np.stack([u, np.zeros_like(u), np.zeros_like(u)], axis=1)
    assert list(oidx.index_visibilities(uvw, None, params)["drop"]) == [False, True, False, True]


def test_bucket_sort_is_stable_and_partitions():
    rng = np.random.default_rng(5)
    params = base_params(grid_size=256, oversample=4, cell_size_rad=1.0 / (256 * 20.0), n_wplanes=4, w_max=100.0,
                         support_min=7, support_max=13, kernel_mode=MODE_WPROJ, n_aplanes=2)
    nvis = 5000
    uvw = ((rng.random((nvis, 3)) * 2 - 1) * np.array([2600.0, 2600.0, 100.0])).astype(np.float32)
    a = rng.integers(0, 2, nvis).astype(np.int32)
    rec = oidx.index_visibilities(uvw, a, params)
    assert rec["drop"].any() and not rec["drop"].all()
    keys = oidx.bucket_keys(rec, params, tile=32)
    b = oidx.bucket_sort(keys, params, tile=32)
    perm = b["perm"]
    assert sorted(perm.tolist()) == list(range(nvis))
    sk = keys[perm]
    assert np.all(np.diff(sk.astype(np.int64)) >= 0)
    same = sk[1:] == sk[:-1]
    assert np.all(perm[1:][same] > perm[:-1][same])                 # stability
    assert b["n_kept"] == int((~rec["drop"]).sum())
    off = b["bucket_offset"]
    nt = 8
    assert len(off) == 2 * 7 * nt * nt + 1 and off[0] == 0 and off[-1] == b["n_kept"]
    for bucket in np.flatnonzero(np.diff(off))[:200]:               # every bucket is one (kset, tile) pair
        seg = perm[off[bucket]:off[bucket + 1]]
        assert np.all(rec["kset"][seg] == bucket // (nt * nt))
        assert np.all(rec["gy"][seg] // 32 == (bucket // nt) % nt)
        assert np.all(rec["gx"][seg] // 32 == bucket % nt)


def test_invalid_input_is_dropped_with_a_fixed_record():
    """R17: non-finite uvw, positions beyond 2^30 fine cells and out-of-range a_index are dropped (never indexed)."""
    params = dict(grid_size=64, cell_size_rad=1e-3, n_wplanes=4, w_max=50.0, support_min=5, support_max=9, oversample=4,
                  n_aplanes=3)
    uvw = np.array([[1.0, 2.0, 3.0], [np.nan, 0, 0], [0, np.inf, 0], [0, 0, -np.inf], [3e38, 0, 0], [1.0, 2.0, 3.0],
                    [1.0, 2.0, 3.0], [5.0, -4.0, -20.0]], np.float32)
    a = np.array([0, 0, 0, 0, 0, 3, -1, 2], np.int32)
    rec = oidx.index_visibilities(uvw, a, params)
    assert list(rec["drop"]) == [False, True, True, True, True, True, True, False]
    bad = slice(1, 7)
    for name, val in (("gx", 0), ("gy", 0), ("ox", -2), ("oy", -2), ("sp", 0), ("kset", 0)):
        assert np.all(rec[name][bad] == val), name
    packed = oidx.pack_records(rec, 4)
    assert np.all(packed[bad] == np.array([0, 0, 1 << 16, 0]))
    assert rec["kset"][7] == 2 * 7 + (-1 + 3) and rec["kset"][0] == 0 * 7 + (0 + 3)
    keys = oidx.bucket_keys(rec, params, tile=32)
    assert np.all(keys[bad] == oidx.KEY_DROP)
