"""GPU tests (-m gpu) of the image-domain mosaic (readings R21-R23): the reprojection
kernel against oracle/mosaic.py element by element, and the per-component loops (imager_mosaic_grid / imager_mosaic_degrid:
grid -> cuFFT -> beam -> reproject, and back) against the oracle's composition of its own steps on a 50-pointing cut of
config 4 (BASELINE.json configs[3]: 50 antennas, 100 GHz, 50 hexagonal pointings, 512^2 grid), every third time step."""
import numpy as np
import pytest

from oracle import mosaic as om, index as oidx, gridder as og, imaging as oi
from helpers import base_params, oracle_tables
from synth import make_workload

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_src,n_dst,cs,cd,shift,beam,inner,acc", [
    (64, 64, 1e-3, 1e-3, (0.0, 0.0), 0, False, False),
    (64, 96, 1e-3, 0.7e-3, (3.3e-3, -5.1e-3), 1, True, False),
    (80, 50, 0.9e-3, 1.3e-3, (-7.77e-3, 2.5e-3), 2, False, True),
    (33, 131, 2e-3, 0.5e-3, (1e-2, 1e-2), 1, True, True),
])
def test_reproject_matches_oracle(n_src, n_dst, cs, cd, shift, beam, inner, acc):
    import torch
    assert torch.cuda.is_available()
    from paper_2206_15117_b200 import imager_reproject
    rng = np.random.default_rng(n_src + n_dst)
    src = (rng.standard_normal((n_src, n_src)) + 1j * rng.standard_normal((n_src, n_src))).astype(np.complex64)
    prev = (rng.standard_normal((n_dst, n_dst)) + 1j * rng.standard_normal((n_dst, n_dst))).astype(np.complex64)
    dish, freq = 12.0, 20e9
    ref = om.reproject(src.astype(np.complex128), cs, n_dst, cd, shift, {0: None, 1: "src", 2: "dst"}[beam], dish, freq, inner)
    if acc:
        ref = ref + prev
    d_dst = torch.from_numpy(prev.copy()).cuda()
    imager_reproject(torch.from_numpy(src).cuda(), cs, d_dst, cd, shift, beam, dish, freq, inner, acc)
    torch.cuda.synchronize()
    got = d_dst.cpu().numpy()
    assert np.abs(got - ref).max() <= 2e-6 * np.abs(ref).max()
    assert np.all(got[ref == 0] == 0)                                   # outside the source: exactly nothing


def test_image_domain_mosaic_on_a_cut_of_config4(oracle_lib):
    import torch
    from paper_2206_15117_b200 import Plan
    wl = make_workload("config4", time_stride=3)
    p4 = wl.params
    n, cell = p4["grid_size"], p4["cell_size_rad"]
    pts = np.asarray(p4["pointing_lm"], dtype=np.float64)
    params = base_params(grid_size=n, cell_size_rad=cell, oversample=4, dish_diameter_m=p4["dish_diameter_m"],
                         freq_hz=p4["freq_hz"])                          # the component plan: plain 7 x 7 anti-aliasing kernel
    _, _, flat, offs = oracle_tables(params)
    groups = [np.nonzero(wl.a_index == i)[0] for i in range(len(pts))]
    assert all(len(g) > 1000 for g in groups)
    nmax = max(len(g) for g in groups)
    # oracle: every component through O1, O4, O7, then R23
    imgs, sws = [], []
    for g in groups:
        rec = oidx.index_visibilities(wl.uvw[g], None, params)
        out = og.grid(rec, wl.vis[g], wl.weights[g], flat, offs, params)
        imgs.append(oi.grid_to_image(out["grid"][0], out["sumwt"][0]))
        sws.append(out["sumwt"][0])
    ref = om.mosaic_image(imgs, sws, cell, pts, n, cell, params["dish_diameter_m"], params["freq_hz"])
    rng = np.random.default_rng(6)
    model = np.zeros((n, n), np.complex64)
    q = n // 4
    model[q:3 * q, q:3 * q] = (rng.standard_normal((2 * q, 2 * q)) * (rng.random((2 * q, 2 * q)) < 0.01)).astype(np.complex64)
    with Plan(params, nmax, user_tables=flat) as plan:
        dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
        uvw_l = [dev(wl.uvw[g]) for g in groups]
        vis_l = [dev(wl.vis[g]) for g in groups]
        wts_l = [dev(wl.weights[g]) for g in groups]
        mosaic = torch.full((n, n), 5.0 + 5.0j, dtype=torch.complex64, device="cuda")        # overwritten
        total = torch.zeros(1, dtype=torch.float64, device="cuda")
        plan.mosaic_grid(uvw_l, vis_l, wts_l, pts, mosaic, cell, total)
        torch.cuda.synchronize()
        assert plan.last_launch_count() > 4 * len(pts)
        got = mosaic.cpu().numpy()
        assert np.isclose(total.item(), float(np.sum(sws)), rtol=1e-12)
        assert np.abs(got - ref).max() <= 2e-5 * np.abs(ref).max()
        # backward: predict five of the components from a sparse model image
        sel = [0, 7, 19, 33, 49]
        outs = [torch.empty((len(groups[i]), 1), dtype=torch.complex64, device="cuda") for i in sel]
        plan.mosaic_degrid([uvw_l[i] for i in sel], pts[sel], dev(model), cell, outs)
        torch.cuda.synchronize()
        for i, o in zip(sel, outs):
            ks = np.sort(rng.choice(len(groups[i]), 400, replace=False))
            comp = om.component_model(model.astype(np.complex128), cell, n, cell, pts[i], params["dish_diameter_m"], params["freq_hz"])
            mg = oi.image_to_grid(comp)
            sub = oidx.index_visibilities(wl.uvw[groups[i]][ks], None, params)
            refd = og.degrid(sub, mg[None].astype(np.complex64), flat, offs, params)
            v = o.cpu().numpy()[ks]
            assert np.abs(v - refd["vis"]).max() <= 2e-5 * np.abs(refd["vis"]).max(), i


def test_plan_with_a_beam_in_its_kernels_is_refused():
    """The image-domain mosaic applies the primary beam in the image plane; a MOSAIC_PB plan already holds it in its gridding
    kernels and would apply it twice, so imager_mosaic_grid / _degrid refuse it (include/imager.h).  A grid too narrow for the
    tiled kernels also shows up in imager_plan_path with its reason."""
    import torch
    from paper_2206_15117_b200 import ImagerError, Plan, MODE_MOSAIC_PB, MODE_PSWF
    base = dict(grid_size=128, cell_size_rad=0.03 / 128, n_corr=1, n_pol=1, n_wplanes=1, w_max=0.0, support_min=16, support_max=16,
                oversample=4, n_aplanes=1, dish_diameter_m=12.0, freq_hz=3.0e9, pointing_lm=[[0.0, 0.0]], pa_rad=[0.0])
    uvw = torch.zeros((4, 3), dtype=torch.float32, device="cuda")
    vis = torch.ones((4, 1), dtype=torch.complex64, device="cuda")
    wts = torch.ones((4, 1), dtype=torch.float32, device="cuda")
    mosaic = torch.zeros((64, 64), dtype=torch.complex64, device="cuda")
    with Plan(dict(base, kernel_mode=MODE_MOSAIC_PB), 4) as plan:
        assert plan.path() == ("tiled", "")
        with pytest.raises(ImagerError, match="carries the primary beam"):
            plan.mosaic_grid([uvw], [vis], [wts], [[0.0, 0.0]], mosaic, 0.03 / 128)
        with pytest.raises(ImagerError, match="carries the primary beam"):
            plan.mosaic_degrid([uvw], [[0.0, 0.0]], mosaic, 0.03 / 128, [vis])
        torch.cuda.synchronize()
        assert torch.count_nonzero(mosaic).item() == 0
    with Plan(dict(base, kernel_mode=MODE_PSWF, grid_size=80, support_min=7, support_max=7), 4) as plan:
        path, why = plan.path()
        assert path == "reference" and "multiple of the 32-cell strip" in why
