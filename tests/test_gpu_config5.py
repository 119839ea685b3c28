"""GPU parity on BASELINE.json configs[4] ("config 5": 36 antennas, 288 channels x 1000 time steps = 181,440,000
visibilities x 4 correlations, 8192^2 x 4 grids, 64 w-planes with supports 15..127, A-projection with 4 parallactic-angle
bins) AS STATED: the visibilities are fed through the public API in chunks of whole time steps (gridding accumulates into
the caller's grid; one call holds fewer than 2^31 hits), then grid -> cuFFT -> (clean-model window) -> cuFFT -> degrid
(PAPER.md:46 puts the FFT between the two; the model is the dirty image inside the inner half of the field, which is
where a taper-corrected image is valid: psi(+-1) = 1.9e-4).

Checked against the oracle, chunk by chunk:
  * index records, sorted keys, permutation, bucket offsets of EVERY chunk: bit-exact;
  * 3000 sampled grid cells after all chunks (the oracle's `sample_cells` mode accumulates them over the chunks) and
    300 sampled degridded visibilities per chunk (oracle O5 on the grid the library degrids from): <= 1e-5, normalised
    by sum |kernel . vis| per output element; sum of weights to 1e-12.

Default: every 10th time step (100 of the 1000 steps: 18,144,000 visibilities x 4 in 2 chunks, the same grid, tables and
call sequence; about 8 minutes, 5 of them the oracle building 508 kernel sets).  IMAGER_CONFIG5_FULL=1 runs all 1000 time
steps in 10 chunks (about 20 minutes; the record of that run is profiles/r2_config5.md).  IMAGER_SKIP_SLOW=1 skips."""
import os

import numpy as np
import pytest

from oracle import index as oidx, kernels as okern, gridder as og
from synth import make_workload

pytestmark = [pytest.mark.gpu, pytest.mark.slow]
TOL = 1e-5


def test_config5_chunked_grid_fft_degrid_round_trip(oracle_lib):
    if os.environ.get("IMAGER_SKIP_SLOW") == "1":
        pytest.skip("IMAGER_SKIP_SLOW=1")
    import torch
    assert torch.cuda.is_available()
    from paper_2206_15117_b200 import Plan
    full = os.environ.get("IMAGER_CONFIG5_FULL") == "1"
    stride, steps_per_chunk = (1, 100) if full else (10, 50)
    probe = make_workload("config5", time_stride=stride, time_range=(0, 1))
    params, n_time = probe.params, probe.notes["n_time_all"]
    per_step = probe.nvis
    n, npol, nc = params["grid_size"], params["n_pol"], params["n_corr"]
    assert (n, npol, nc, params["support_max"], params["n_wplanes"]) == (8192, 4, 4, 127, 64)
    assert n_time * per_step * stride == 181_440_000
    tabs, _ = okern.make_tables(params)
    flat, offs = okern.flatten_tables(tabs)
    del tabs
    chunks = [(t0, min(t0 + steps_per_chunk, n_time)) for t0 in range(0, n_time, steps_per_chunk)]
    rng = np.random.default_rng(2025)
    with Plan(params, steps_per_chunk * per_step, user_tables=flat) as plan:
        assert plan.path() == ("tiled", ""), f"config 5 would run on the reference kernels: {plan.path()[1]}"
        grid = torch.zeros((npol, n, n), dtype=torch.complex64, device="cuda")
        sumwt = torch.zeros(nc, dtype=torch.float64, device="cuda")
        cells = acc = acc_norm = None
        ref_sumwt = np.zeros(nc)
        keep = []                                                   # per chunk: (uvw, a_index) for the degridding pass
        for t0, t1 in chunks:
            wl = make_workload("config5", time_stride=stride, time_range=(t0, t1))
            rec = oidx.index_visibilities(wl.uvw, wl.a_index, params)
            uvw = torch.from_numpy(wl.uvw).cuda()
            a = torch.from_numpy(wl.a_index).cuda()
            got = plan.debug_index(uvw, a)
            assert np.array_equal(got["records"], oidx.pack_records(rec, params["oversample"]))
            ref = oidx.bucket_sort(oidx.bucket_keys(rec, params, tile=32), params, tile=32)
            assert np.array_equal(got["sorted_keys"], ref["sorted_keys"]) and np.array_equal(got["perm"], ref["perm"])
            assert np.array_equal(got["bucket_offset"], ref["bucket_offset"]) and got["n_kept"] == ref["n_kept"]
            del got, ref
            vis = torch.from_numpy(wl.vis).cuda()
            wts = torch.from_numpy(wl.weights).cuda()
            plan.grid(uvw, vis, wts, grid, a, sumwt, flags=1)        # accumulates: the index is the one just built
            torch.cuda.synchronize()
            assert plan.index_stats()["n_hits"] > 0, "support 127 must run on the tiled path (its slice has to fit the table budget)"
            del vis, wts, uvw, a
            if cells is None:                                       # half at visibility positions, half across the coverage
                pick = rng.integers(0, wl.nvis, 1500)
                near = np.stack([rec["gy"][pick] + rng.integers(-3, 4, 1500), rec["gx"][pick] + rng.integers(-3, 4, 1500)], 1)
                r = 0.42 * n * np.sqrt(rng.random(1500))
                th = 2 * np.pi * rng.random(1500)
                spread = np.stack([n // 2 + r * np.sin(th), n // 2 + r * np.cos(th)], 1).astype(np.int64)
                cells = np.unique(np.clip(np.concatenate([near, spread]), 0, n - 1), axis=0)
                acc = np.zeros((npol, len(cells)), np.complex128)
                acc_norm = np.zeros((npol, len(cells)))
            sm = og.grid(rec, wl.vis, wl.weights, flat, offs, params, sample_cells=cells)
            acc += sm["samples"]
            acc_norm += sm["sample_norm"]
            ref_sumwt += sm["sumwt"]
            keep.append((wl.uvw, wl.a_index))
            del wl, rec, sm
        g = grid[:, torch.from_numpy(cells[:, 0]).cuda(), torch.from_numpy(cells[:, 1]).cuda()].cpu().numpy()
        touched = acc_norm > 0
        assert touched.mean() > 0.5 and np.all(g[~touched] == 0)
        err = np.max(np.abs(g[touched] - acc[touched]) / acc_norm[touched])
        assert err <= TOL, f"config5: sampled grid parity {err:.3e}"
        assert np.allclose(sumwt.cpu().numpy(), ref_sumwt, rtol=1e-12)
        # grid -> image -> clean-model window -> grid
        plan.grid_image_transform(grid, +1, float(ref_sumwt[0]))
        q = n // 4
        model = torch.zeros_like(grid)
        model[:, q:3 * q, q:3 * q] = grid[:, q:3 * q, q:3 * q]
        del grid
        plan.grid_image_transform(model, -1)
        torch.cuda.synchronize()
        model_host = model.cpu().numpy()
        assert np.isfinite(model_host.view(np.float32)).all() and np.abs(model_host).max() > 0
        for uvw_h, a_h in keep:
            nv = uvw_h.shape[0]
            uvw, a = torch.from_numpy(uvw_h).cuda(), torch.from_numpy(a_h).cuda()
            out = torch.empty((nv, nc), dtype=torch.complex64, device="cuda")
            plan.degrid(uvw, model, out, a)                          # re-indexes this chunk
            torch.cuda.synchronize()
            ks = np.sort(rng.choice(nv, 300, replace=False))
            sub = oidx.index_visibilities(uvw_h[ks], a_h[ks], params)
            refd = og.degrid(sub, model_host, flat, offs, params)
            v = out[torch.from_numpy(ks).cuda()].cpu().numpy()
            ok = refd["norm"] > 0
            errd = np.max(np.abs(v[ok] - refd["vis"][ok]) / refd["norm"][ok])
            assert errd <= TOL, f"config5: sampled degrid parity {errd:.3e}"
            assert np.all(v[sub["drop"]] == 0)
            del uvw, a, out
