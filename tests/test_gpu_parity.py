"""GPU parity tests (-m gpu): the CUDA path, called through the C-ABI binding, against the CPU oracle on the
same seeded inputs.  Bar (BASELINE.json north_star): index / bucketing bit-exact; grids and degridded
visibilities within 1e-5 of the oracle, normalised by sum |kernel . vis| per output element.

The hot-path cases feed the ORACLE's kernel tables (rounded to complex64) to the library (USER mode), so that
the comparison isolates indexing, bucketing, gridding and degridding; the library's own table generator is
compared with the oracle's tables separately (test_gpu_tables.py)."""
import numpy as np
import pytest

from oracle import index as oidx, gridder as og
from helpers import (base_params, random_vis, oracle_tables, MODE_DELTA, MODE_PSWF, MODE_WPROJ, MODE_AWPROJ_ADJOINT,
                     MODE_AWPROJ_PAPER, MODE_MOSAIC_PB)

pytestmark = pytest.mark.gpu
TOL = 1e-5


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    return torch


def _to_dev(torch, uvw, vis, wts, a):
    d = lambda x: None if x is None else torch.from_numpy(np.ascontiguousarray(x)).cuda()
    return d(uvw), d(vis), d(wts), d(a)


def grid_error(g_gpu, oracle_out):
    """max |G_gpu - G_oracle| / A[cell]; cells the oracle never touched must be exactly zero."""
    g, a = oracle_out["grid"], oracle_out["norm"]
    untouched = a == 0
    assert np.all(g_gpu[untouched] == 0), "GPU wrote cells the oracle did not touch"
    return float(np.max(np.abs(g_gpu[~untouched] - g[~untouched]) / a[~untouched])) if (~untouched).any() else 0.0


def vis_error(v_gpu, oracle_out, drop):
    v, b = oracle_out["vis"], oracle_out["norm"]
    assert np.all(v_gpu[drop] == 0), "dropped visibilities must predict 0"
    ok = b > 0
    return float(np.max(np.abs(v_gpu[ok] - v[ok]) / b[ok])) if ok.any() else 0.0


CASES = {
    "pswf": lambda: base_params(grid_size=128, oversample=8),
    "wproj": lambda: base_params(grid_size=256, oversample=4, n_wplanes=8, w_max=90.0, support_min=7, support_max=21,
                                 kernel_mode=MODE_WPROJ, cell_size_rad=0.1 / 256),
    "wproj_big_support": lambda: base_params(grid_size=256, oversample=2, n_wplanes=3, w_max=30.0, support_min=33,
                                             support_max=67, kernel_mode=MODE_WPROJ, cell_size_rad=0.05 / 256),
    "awproj": lambda: base_params(grid_size=128, oversample=4, n_wplanes=3, w_max=30.0, support_min=7, support_max=11,
                                  n_corr=4, n_pol=4, n_aplanes=3, pa_rad=[0.0, 0.5, 1.0], pointing_lm=[[0, 0]] * 3,
                                  leakage=[0.01j, -0.01], kernel_mode=MODE_AWPROJ_ADJOINT, cell_size_rad=0.04 / 128),
    "mosaic_even": lambda: base_params(grid_size=128, oversample=4, support_min=16, support_max=16, n_aplanes=5,
                                       pa_rad=[0] * 5, pointing_lm=[[0, 0], [0.003, 0.001], [-0.002, 0.004], [0.001, -0.003],
                                                                    [0.0, 0.002]],
                                       kernel_mode=MODE_MOSAIC_PB, cell_size_rad=0.03 / 128, freq_hz=3.0e9),
}


@pytest.mark.parametrize("case", sorted(CASES))
@pytest.mark.parametrize("flags", [0, 2], ids=["default", "reference"])
def test_grid_and_degrid_parity_small(torch_cuda, oracle_lib, case, flags):
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    params = CASES[case]()
    nvis = 6000
    uvw, vis, wts, a = random_vis(params, nvis, seed=31, frac=0.52, a_planes=params["n_aplanes"] > 1)
    wts[::17] = 0.0                                                  # zero weights contribute nothing (R9)
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    assert rec["drop"].any() and (~rec["drop"]).sum() > nvis // 4      # frac 0.52 pushes some footprints off the grid
    n, npol, nc = params["grid_size"], params["n_pol"], params["n_corr"]
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, d_wts, d_a = _to_dev(torch, uvw, vis, wts, a)
        grid = torch.zeros((npol, n, n), dtype=torch.complex64, device="cuda")
        sumwt = torch.zeros(nc, dtype=torch.float64, device="cuda")
        plan.grid(d_uvw, d_vis, d_wts, grid, d_a, sumwt, flags=flags)
        torch.cuda.synchronize()
        ref = og.grid(rec, vis, wts, flat, offs, params)
        err = grid_error(grid.cpu().numpy(), ref)
        assert err <= TOL, f"grid parity {err:.3e}"
        assert np.allclose(sumwt.cpu().numpy(), ref["sumwt"], rtol=1e-12)
        assert plan.info()["n_dropped"] == int(rec["drop"].sum())
        # warm call (index reuse) accumulates a second copy
        plan.grid(d_uvw, d_vis, d_wts, grid, d_a, None, flags=flags | 1)
        torch.cuda.synchronize()
        ref2 = dict(grid=2 * ref["grid"], norm=2 * ref["norm"])
        assert grid_error(grid.cpu().numpy(), ref2) <= TOL
        # degridding from a random grid
        rng = np.random.default_rng(9)
        g = (rng.standard_normal((npol, n, n)) + 1j * rng.standard_normal((npol, n, n))).astype(np.complex64)
        d_g = torch.from_numpy(g).cuda()
        out = torch.full((nvis, nc), 7.0 + 7.0j, dtype=torch.complex64, device="cuda")
        plan.degrid(d_uvw, d_g, out, d_a, flags=flags)
        torch.cuda.synchronize()
        refd = og.degrid(rec, g, flat, offs, params)
        errd = vis_error(out.cpu().numpy(), refd, rec["drop"])
        assert errd <= TOL, f"degrid parity {errd:.3e}"


@pytest.mark.parametrize("case", sorted(CASES))
def test_index_and_bucketing_bit_exact(torch_cuda, case):
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    params = CASES[case]()
    nvis = 50000
    uvw, _, _, a = random_vis(params, nvis, seed=41, frac=0.55, a_planes=params["n_aplanes"] > 1)
    # exact ties on the fine lattice (q + 0.5) in both signs
    uv_scale = float(params["oversample"]) * float(params["grid_size"]) * params["cell_size_rad"]
    uvw[:64, 0] = ((np.arange(64) - 32) + 0.5) / uv_scale
    uvw[:64, 1] = -uvw[:64, 0]
    _, _, flat, _ = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    keys = oidx.bucket_keys(rec, params, tile=32)
    ref = oidx.bucket_sort(keys, params, tile=32)
    with Plan(params, nvis, user_tables=flat) as plan:
        assert plan.info()["bucket_tile"] == 32
        d_uvw, _, _, d_a = _to_dev(torch, uvw, None, None, a)
        got = plan.debug_index(d_uvw, d_a)
    assert np.array_equal(got["records"], oidx.pack_records(rec, params["oversample"]))
    assert np.array_equal(got["sorted_keys"], ref["sorted_keys"])
    assert np.array_equal(got["perm"], ref["perm"])
    assert got["n_kept"] == ref["n_kept"]
    assert np.array_equal(got["bucket_offset"], ref["bucket_offset"])


def test_delta_kernel_single_visibility(torch_cuda):
    """P1 on the GPU: one visibility, delta kernel, lands on the expected cell with value w*V."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    n, cell = 64, 1.0e-3
    du = 1.0 / (n * cell)
    params = base_params(grid_size=n, cell_size_rad=cell, support_min=1, support_max=1, oversample=1, kernel_mode=MODE_DELTA)
    with Plan(params, 4) as plan:
        uvw = torch.tensor([[3.2 * du, -7.6 * du, 0.0]], dtype=torch.float32, device="cuda")
        vis = torch.tensor([[2.0 - 3.0j]], dtype=torch.complex64, device="cuda")
        wts = torch.tensor([[0.25]], dtype=torch.float32, device="cuda")
        grid = torch.zeros((1, n, n), dtype=torch.complex64, device="cuda")
        plan.grid(uvw, vis, wts, grid)
        g = grid.cpu().numpy()[0]
        assert np.count_nonzero(g) == 1 and g[n // 2 - 8, n // 2 + 3] == np.complex64(0.25 * (2 - 3j))


def test_edge_cases_empty_and_all_dropped(torch_cuda):
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan, ImagerError
    params = CASES["wproj"]()
    _, _, flat, _ = oracle_tables(params)
    n = params["grid_size"]
    with Plan(params, 100, user_tables=flat) as plan:
        grid = torch.zeros((1, n, n), dtype=torch.complex64, device="cuda")
        empty = lambda *s, dt=torch.float32: torch.zeros(s, dtype=dt, device="cuda")
        plan.grid(empty(0, 3), empty(0, 1, dt=torch.complex64), empty(0, 1), grid)
        plan.degrid(empty(0, 3), grid, empty(0, 1, dt=torch.complex64))
        torch.cuda.synchronize()
        assert torch.count_nonzero(grid).item() == 0
        far = torch.full((100, 3), 1.0e7, dtype=torch.float32, device="cuda")       # every footprint leaves the grid
        plan.grid(far, torch.ones((100, 1), dtype=torch.complex64, device="cuda"), torch.ones((100, 1), device="cuda"), grid)
        out = torch.ones((100, 1), dtype=torch.complex64, device="cuda")
        plan.degrid(far, grid, out)
        torch.cuda.synchronize()
        assert torch.count_nonzero(grid).item() == 0 and torch.count_nonzero(out).item() == 0
        assert plan.info()["n_dropped"] == 100
        with pytest.raises(ImagerError):
            plan.grid(empty(101, 3), empty(101, 1, dt=torch.complex64), empty(101, 1), grid)   # TOO_MANY_VIS


def test_adjointness_on_gpu(torch_cuda):
    """<G v, g> = <v, G^H g> to 1e-6 relative (BASELINE.json north_star) on the CUDA path."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    for case in ("wproj", "awproj", "mosaic_even"):
        params = CASES[case]()
        nvis = 20000
        uvw, vis, _, a = random_vis(params, nvis, seed=51, frac=0.3, a_planes=params["n_aplanes"] > 1)
        _, _, flat, _ = oracle_tables(params)
        n, npol, nc = params["grid_size"], params["n_pol"], params["n_corr"]
        with Plan(params, nvis, user_tables=flat) as plan:
            d_uvw, d_vis, _, d_a = _to_dev(torch, uvw, vis, None, a)
            ones = torch.ones((nvis, nc), dtype=torch.float32, device="cuda")
            gv = torch.zeros((npol, n, n), dtype=torch.complex64, device="cuda")
            plan.grid(d_uvw, d_vis, ones, gv, d_a)
            noise = torch.randn((npol, n, n), dtype=torch.complex64, device="cuda")
            # (1) a generic random g: the defect is bounded against the size of the terms of the sum, 1e-6 sum |g_i| |(Gv)_i|
            #     (<g, Gv> itself is a cancelling random sum; FP32 accumulation order differs from run to run: atomics);
            # (2) g = noise + a multiple of G v, where <g, Gv> has a large coherent part: 1e-6 relative to |<g, Gv>| itself.
            for g, coherent in ((noise, False), (noise + gv * (torch.linalg.vector_norm(noise) / torch.linalg.vector_norm(gv)), True)):
                hg = torch.zeros((nvis, nc), dtype=torch.complex64, device="cuda")
                plan.degrid(d_uvw, g, hg, d_a, flags=1)
                lhs = torch.vdot(g.to(torch.complex128).flatten(), gv.to(torch.complex128).flatten()).item()
                rhs = torch.vdot(hg.to(torch.complex128).flatten(), d_vis.to(torch.complex128).flatten()).item()
                size = abs(lhs) if coherent else float((g.abs().double() * gv.abs().double()).sum().item())
                assert abs(lhs - rhs) <= 1e-6 * size, (case, coherent, lhs, rhs, size)


def test_index_ahead_of_grid(torch_cuda, oracle_lib):
    """imager_index (A1 + A2 on their own) followed by REUSE_INDEX calls gives what the one-call path gives."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan, REUSE_INDEX
    params = CASES["wproj"]()
    nvis = 5000
    uvw, vis, wts, a = random_vis(params, nvis, seed=7, frac=0.45)
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    ref = og.grid(rec, vis, wts, flat, offs, params)
    n = params["grid_size"]
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, d_wts, _ = _to_dev(torch, uvw, vis, wts, None)
        plan.index(d_uvw)
        assert plan.last_launch_count() > 0
        grid = torch.zeros((1, n, n), dtype=torch.complex64, device="cuda")
        plan.grid(d_uvw, d_vis, d_wts, grid, flags=REUSE_INDEX)
        out = torch.empty((nvis, 1), dtype=torch.complex64, device="cuda")
        plan.degrid(d_uvw, grid, out, flags=REUSE_INDEX)
        torch.cuda.synchronize()
        g = grid.cpu().numpy()
        assert grid_error(g, ref) <= TOL
        refd = og.degrid(rec, g, flat, offs, params)
        assert vis_error(out.cpu().numpy(), refd, rec["drop"]) <= TOL


@pytest.mark.parametrize("flags", [0, 2], ids=["default", "reference"])
def test_degrid_residual_flag(torch_cuda, oracle_lib, flags):
    """IMAGER_DEGRID_RESIDUAL: vis_out := vis_out - V_model (the major-cycle update), against the oracle's prediction."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan, DEGRID_RESIDUAL
    params = CASES["awproj"]()
    nvis = 4000
    uvw, vis, _, a = random_vis(params, nvis, seed=13, frac=0.5, a_planes=True)
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    n, npol = params["grid_size"], params["n_pol"]
    rng = np.random.default_rng(3)
    g = (rng.standard_normal((npol, n, n)) + 1j * rng.standard_normal((npol, n, n))).astype(np.complex64)
    refd = og.degrid(rec, g, flat, offs, params)
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, _, d_a = _to_dev(torch, uvw, vis, None, a)
        d_g = torch.from_numpy(g).cuda()
        res = d_vis.clone()
        plan.degrid(d_uvw, d_g, res, d_a, flags=flags | DEGRID_RESIDUAL)
        torch.cuda.synchronize()
        got = res.cpu().numpy()
    want = vis.astype(np.complex128) - refd["vis"]
    assert np.array_equal(got[rec["drop"]], vis[rec["drop"]])             # dropped: predicted 0, left as they are
    ok = refd["norm"] > 0
    assert float(np.max(np.abs(got[ok] - want[ok]) / (refd["norm"][ok] + np.abs(vis[ok])))) <= TOL


@pytest.mark.parametrize("case", ["wproj", "awproj"])
def test_duplicate_visibilities_are_presummed_exactly(torch_cuda, oracle_lib, case):
    """Visibilities with the same (kernel set, cell, sub-cell) are merged by the library (their weighted values summed
    before gridding, one prediction copied to all of them in degridding): results must stay those of the oracle, which
    treats every visibility on its own.  Half of the inputs here are exact duplicates in uvw with their own values,
    weights (some zero) and, for the residual, observed visibilities."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan, DEGRID_RESIDUAL
    params = CASES[case]()
    n0 = 3000
    uvw, vis, wts, a = random_vis(params, n0, seed=77, frac=0.45, a_planes=params["n_aplanes"] > 1)
    rng = np.random.default_rng(78)
    pick = rng.integers(0, n0, 3000)
    uvw = np.concatenate([uvw, uvw[pick]])
    a = None if a is None else np.concatenate([a, a[pick]])
    extra = (rng.standard_normal((3000,) + vis.shape[1:]) + 1j * rng.standard_normal((3000,) + vis.shape[1:])).astype(np.complex64)
    vis = np.concatenate([vis, extra])
    wts = np.concatenate([wts, rng.random((3000,) + wts.shape[1:]).astype(np.float32)])
    wts[::13] = 0.0
    nvis = uvw.shape[0]
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    ref = og.grid(rec, vis, wts, flat, offs, params)
    n, npol, nc = params["grid_size"], params["n_pol"], params["n_corr"]
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, d_wts, d_a = _to_dev(torch, uvw, vis, wts, a)
        grid = torch.zeros((npol, n, n), dtype=torch.complex64, device="cuda")
        plan.grid(d_uvw, d_vis, d_wts, grid, d_a)
        out = torch.empty((nvis, nc), dtype=torch.complex64, device="cuda")
        plan.degrid(d_uvw, grid, out, d_a, flags=1)
        res = d_vis.clone()
        plan.degrid(d_uvw, grid, res, d_a, flags=1 | DEGRID_RESIDUAL)
        torch.cuda.synchronize()
        g = grid.cpu().numpy()
        assert grid_error(g, ref) <= TOL
        refd = og.degrid(rec, g, flat, offs, params)
        v = out.cpu().numpy()
        assert vis_error(v, refd, rec["drop"]) <= TOL
        ok = refd["norm"] > 0
        same = ok[n0:] & ok[pick]                  # a duplicate gets its original's prediction (bit-equal when merged)
        assert float(np.max(np.abs(v[n0:][same] - v[pick][same]) / refd["norm"][n0:][same])) <= TOL
        want = vis.astype(np.complex128) - refd["vis"]
        assert float(np.max(np.abs(res.cpu().numpy()[ok] - want[ok]) / (refd["norm"][ok] + np.abs(vis[ok])))) <= TOL


def test_paper_mode_grids_and_degrids_with_distinct_tables(torch_cuda, oracle_lib):
    """The paper's own mode: gridding with the (M^S')^-1 tables (Eq. 6), degridding with the M^S tables.
    The oracle's two table sets go in as user_tables / user_tables_degrid; both directions element-wise <= 1e-5, and the
    two table sets really differ (a library that degrids with the gridding tables fails)."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    params = base_params(grid_size=128, oversample=4, n_wplanes=3, w_max=30.0, support_min=7, support_max=11, n_corr=4,
                         n_pol=4, n_aplanes=2, pa_rad=[0.0, 0.6], pointing_lm=[[0, 0]] * 2, leakage=[0.01j, -0.01],
                         kernel_mode=MODE_AWPROJ_PAPER, beam_eps=0.2, cell_size_rad=0.04 / 128)
    nvis = 6000
    uvw, vis, wts, a = random_vis(params, nvis, seed=61, frac=0.45, a_planes=True)
    _, _, flat_g, offs = oracle_tables(params, "grid")
    _, _, flat_d, offs_d = oracle_tables(params, "degrid")
    assert np.array_equal(offs, offs_d) and np.abs(flat_g - flat_d).max() > 0.1 * np.abs(flat_d).max()
    rec = oidx.index_visibilities(uvw, a, params)
    n, npol, nc = params["grid_size"], 4, 4
    with Plan(params, nvis, user_tables=flat_g, user_tables_degrid=flat_d) as plan:
        d_uvw, d_vis, d_wts, d_a = _to_dev(torch, uvw, vis, wts, a)
        for flags in (0, 2):
            grid = torch.zeros((npol, n, n), dtype=torch.complex64, device="cuda")
            plan.grid(d_uvw, d_vis, d_wts, grid, d_a, flags=flags)
            out = torch.empty((nvis, nc), dtype=torch.complex64, device="cuda")
            plan.degrid(d_uvw, grid, out, d_a, flags=flags | 1)
            torch.cuda.synchronize()
            g = grid.cpu().numpy()
            assert grid_error(g, og.grid(rec, vis, wts, flat_g, offs, params)) <= TOL
            refd = og.degrid(rec, g, flat_d, offs, params)
            assert vis_error(out.cpu().numpy(), refd, rec["drop"]) <= TOL
            wrong = og.degrid(rec, g, flat_g, offs, params)           # degridding with the gridding tables is far off
            ok = refd["norm"] > 0
            assert np.max(np.abs(wrong["vis"][ok] - refd["vis"][ok]) / refd["norm"][ok]) > 1e-2


def test_duplicates_across_dedupe_chunks(torch_cuda, oracle_lib):
    """Duplicate pre-summation works on chunks of 4096 consecutive sorted visibilities: (a) 9000 copies of ONE geometry
    span three chunks (several representatives), (b) pairs of duplicates whose sorted positions are more than 4096
    apart (same bucket key, thousands of other visibilities of that key between them in input order: the sort is stable)
    are not merged at all.  Either way the results are the oracle's."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    params = base_params(grid_size=128, oversample=2, cell_size_rad=1.0e-3)
    rng = np.random.default_rng(5)
    du = 1.0 / (128 * 1.0e-3)
    # (b) 30000 visibilities inside one 32 x 32 tile: ~7500 per (tile, sub-cell) key; the first 500 repeated at the end
    base = np.zeros((30000, 3), np.float32)
    base[:, 0] = (4 + 24 * rng.random(30000)) * du
    base[:, 1] = (4 + 24 * rng.random(30000)) * du
    one = np.tile(np.array([[-20.3 * du, 11.2 * du, 0.0]], np.float32), (9000, 1))           # (a)
    uvw = np.concatenate([base, one, base[:500]])
    nvis = uvw.shape[0]
    vis = (rng.standard_normal((nvis, 1)) + 1j * rng.standard_normal((nvis, 1))).astype(np.complex64)
    wts = (0.5 + rng.random((nvis, 1))).astype(np.float32)
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, None, params)
    keys = oidx.bucket_keys(rec, params, tile=32)
    srt = oidx.bucket_sort(keys, params, tile=32)
    where = np.empty(nvis, np.int64)
    where[srt["perm"]] = np.arange(nvis)
    assert np.min(np.abs(where[30000 + 9000:] - where[:500])) > 4096      # (b) holds on these inputs
    ref = og.grid(rec, vis, wts, flat, offs, params)
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, d_wts, _ = _to_dev(torch, uvw, vis, wts, None)
        grid = torch.zeros((1, 128, 128), dtype=torch.complex64, device="cuda")
        plan.grid(d_uvw, d_vis, d_wts, grid)
        out = torch.empty((nvis, 1), dtype=torch.complex64, device="cuda")
        plan.degrid(d_uvw, grid, out, flags=1)
        torch.cuda.synchronize()
        g = grid.cpu().numpy()
        assert grid_error(g, ref) <= TOL
        refd = og.degrid(rec, g, flat, offs, params)
        assert vis_error(out.cpu().numpy(), refd, rec["drop"]) <= TOL


def test_invalid_input_is_dropped_not_indexed(torch_cuda, oracle_lib):
    """R17: NaN / infinite uvw rows and a_index outside [0, n_aplanes) are dropped and counted; records bit-exact with the
    oracle; the grid is the oracle's (which never sees them) and nothing outside it is written."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    params = CASES["awproj"]()
    nvis = 4000
    uvw, vis, wts, a = random_vis(params, nvis, seed=91, frac=0.4, a_planes=True)
    uvw[10] = [np.nan, 1.0, 2.0]
    uvw[11] = [1.0, np.inf, 2.0]
    uvw[12] = [1.0, 2.0, -np.inf]
    uvw[13] = [3.0e38, 0.0, 0.0]
    a[20], a[21], a[22] = params["n_aplanes"], -1, 2 ** 30
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    assert rec["drop"][[10, 11, 12, 13, 20, 21, 22]].all()
    ref = og.grid(rec, vis, wts, flat, offs, params)
    n, npol, nc = params["grid_size"], 4, 4
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, d_wts, d_a = _to_dev(torch, uvw, vis, wts, a)
        got = plan.debug_index(d_uvw, d_a)
        assert np.array_equal(got["records"], oidx.pack_records(rec, params["oversample"]))
        keys = oidx.bucket_keys(rec, params, tile=32)
        srt = oidx.bucket_sort(keys, params, tile=32)
        assert np.array_equal(got["sorted_keys"], srt["sorted_keys"]) and np.array_equal(got["perm"], srt["perm"])
        for flags in (0, 2):
            guard = torch.zeros((npol + 2, n, n), dtype=torch.complex64, device="cuda")     # a plane of slack on either side
            grid = guard[1:npol + 1]
            sumwt = torch.zeros(nc, dtype=torch.float64, device="cuda")
            plan.grid(d_uvw, d_vis, d_wts, grid, d_a, sumwt, flags=flags)
            out = torch.full((nvis, nc), 3.0 + 0j, dtype=torch.complex64, device="cuda")
            plan.degrid(d_uvw, grid, out, d_a, flags=flags | 1)
            torch.cuda.synchronize()
            assert plan.info()["n_dropped"] == int(rec["drop"].sum())
            assert grid_error(grid.cpu().numpy(), ref) <= TOL
            assert torch.count_nonzero(guard[0]).item() == 0 and torch.count_nonzero(guard[-1]).item() == 0
            assert np.allclose(sumwt.cpu().numpy(), ref["sumwt"], rtol=1e-12)
            assert np.all(out.cpu().numpy()[rec["drop"]] == 0)


@pytest.mark.parametrize("case", ["wproj", "awproj"])
def test_flagged_samples_contribute_nothing(torch_cuda, oracle_lib, case):
    """R24: samples with zero weight or a non-finite weight / value (flagged data often carry NaN) add nothing -- on both
    kernel paths, with and without duplicates of the flagged visibility (whose pre-summed value must stay clean), and
    nothing outside the footprints is written (the tiled kernel multiplies values into zero padding)."""
    torch = torch_cuda
    from paper_2206_15117_b200 import Plan
    params = CASES[case]()
    nvis, nc, npol, n = 6000, params["n_corr"], params["n_pol"], params["grid_size"]
    uvw, vis, wts, a = random_vis(params, nvis, seed=123, frac=0.35, a_planes=params["n_aplanes"] > 1)
    uvw[100:104] = uvw[7]                                                  # duplicates of a visibility that gets flagged
    if a is not None:
        a[100:104] = a[7]
    bad = [(7, 0, np.nan + 0j, 0.0), (9, nc - 1, complex(np.inf, 1.0), 0.0), (101, 0, complex(1.0, np.nan), 0.0),
           (500, 0, complex(np.nan, np.nan), 1.0), (501, nc - 1, 1.0 + 1.0j, np.nan), (502, 0, 1.0 - 2.0j, np.inf)]
    for k, c, v, w in bad:
        vis[k, c], wts[k, c] = v, w
    _, _, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    ref = og.grid(rec, vis, wts, flat, offs, params)
    assert np.isfinite(ref["grid"]).all()
    with Plan(params, nvis, user_tables=flat) as plan:
        d_uvw, d_vis, d_wts, d_a = _to_dev(torch, uvw, vis, wts, a)
        for flags in (0, 2):
            guard = torch.zeros((npol + 2, n, n), dtype=torch.complex64, device="cuda")
            grid = guard[1:npol + 1]
            sumwt = torch.zeros(nc, dtype=torch.float64, device="cuda")
            plan.grid(d_uvw, d_vis, d_wts, grid, d_a, sumwt, flags=flags)
            torch.cuda.synchronize()
            g = grid.cpu().numpy()
            assert np.isfinite(g).all(), "a flagged sample reached the grid"
            assert grid_error(g, ref) <= TOL
            assert torch.count_nonzero(guard[0]).item() == 0 and torch.count_nonzero(guard[-1]).item() == 0
            assert np.allclose(sumwt.cpu().numpy(), ref["sumwt"], rtol=1e-12)
