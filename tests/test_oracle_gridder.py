"""Pins for oracle steps O4/O5/O7 (gridding, degridding, imaging): P1, P2, P3, P4, P6, P9, P11, P13."""
import numpy as np

from oracle import index as oidx, kernels as ok, gridder as og, imaging as oi
from helpers import (base_params, random_vis, oracle_tables, oracle_grid, oracle_degrid, MODE_DELTA, MODE_WPROJ,
                     MODE_AWPROJ_ADJOINT, MODE_MOSAIC_PB)


def test_P1_delta_kernel_lands_on_expected_cell(oracle_lib):
    """BASELINE.json north_star: "a single visibility with a delta kernel lands on the expected cell"."""
    n, cell = 64, 1.0e-3
    du = 1.0 / (n * cell)
    params = base_params(grid_size=n, cell_size_rad=cell, support_min=1, support_max=1, oversample=1,
                         kernel_mode=MODE_DELTA)
    for u, v in ((3.2 * du, -7.6 * du), (-12.49 * du, 0.51 * du), (0.0, 0.0)):
        uvw = np.array([[u, v, 0.0]], np.float32)
        vis = np.array([[2.0 - 3.0j]], np.complex64)
        wts = np.array([[0.25]], np.float32)
        out, _ = oracle_grid(params, uvw, vis, wts)
        g = out["grid"][0]
        ey, ex = int(np.rint(v / du)) + n // 2, int(np.rint(u / du)) + n // 2
        assert np.count_nonzero(g) == 1 and g[ey, ex] == 0.25 * (2.0 - 3.0j)
        assert out["sumwt"][0] == 0.25 and out["norm"][0, ey, ex] == 0.25 * abs(2 - 3j)


def _point_source_vis(uvw, cell, sources):
    u, v, w = (uvw[:, i].astype(np.float64) for i in range(3))
    vis = np.zeros(len(u), np.complex128)
    for px, py, amp in sources:
        l, m = px * cell, py * cell
        vis += amp * np.exp(2j * np.pi * (u * l + v * m + w * (np.sqrt(1 - l * l - m * m) - 1)))   # Eq. 2 sign
    return vis.astype(np.complex64)[:, None]


def test_P2_dirty_image_matches_direct_dft_w0(oracle_lib):
    n, fov = 64, 0.05
    params = base_params(grid_size=n, cell_size_rad=fov / n, oversample=64)
    uvw, _, _, _ = random_vis(params, 300, seed=1, frac=0.35)
    uvw[:, 2] = 0
    vis = _point_source_vis(uvw, fov / n, [(5, -7, 1.0), (-9, 3, 0.5), (0, 0, 0.3)])
    wts = np.ones((300, 1), np.float32)
    out, _ = oracle_grid(params, uvw, vis, wts)
    img = oi.grid_to_image(out["grid"][0], out["sumwt"][0]).real
    ref = oi.direct_dft_image(uvw, vis[:, 0], wts[:, 0], n, fov / n).real
    q = n // 4
    inner = (slice(n // 2 - q, n // 2 + q),) * 2
    assert ref.max() > 0.9
    assert np.abs(img - ref)[inner].max() < 3e-3 * ref.max()       # SURVEY probe: 1.1e-3 at O = 64
    assert np.unravel_index(np.argmax(ref), ref.shape) == (n // 2 - 7, n // 2 + 5)   # source 1 at (x=+5, y=-7)


def test_P2_dirty_image_matches_direct_dft_with_w(oracle_lib):
    """Wide field + significant w: pins the w-term sign and the signed-plane lookup (a flipped sign gives ~0.9)."""
    n, fov = 64, 0.2
    params = base_params(grid_size=n, cell_size_rad=fov / n, oversample=16, n_wplanes=16, w_max=200.0,
                         support_min=19, support_max=19, kernel_mode=MODE_WPROJ)
    uvw, _, _, _ = random_vis(params, 300, seed=3, frac=0.3)
    vis = _point_source_vis(uvw, fov / n, [(12, -10, 1.0), (-9, 13, 0.5)])
    wts = np.ones((300, 1), np.float32)
    out, rec = oracle_grid(params, uvw, vis, wts)
    assert rec["sp"].min() < -10 and rec["sp"].max() > 10
    img = oi.grid_to_image(out["grid"][0], out["sumwt"][0]).real
    ref = oi.direct_dft_image(uvw, vis[:, 0], wts[:, 0], n, fov / n).real
    q = n // 4
    inner = (slice(n // 2 - q, n // 2 + q),) * 2
    err = np.abs(img - ref)[inner].max() / ref.max()
    assert err < 2.5e-2, err
    # ignoring w in the reference must be far worse: the test is sensitive to the w-term
    flat = oi.direct_dft_image(uvw * np.array([1, 1, 0], np.float32), vis[:, 0], wts[:, 0], n, fov / n).real
    assert np.abs(img - flat)[inner].max() / ref.max() > 10 * err


def test_P6_flat_field(oracle_lib):
    """One visibility at u = v = w = 0 with V = 1 images to a flat field of 1 over the inner half (O6 scalar, O7)."""
    params = base_params(grid_size=64, oversample=8)
    out, _ = oracle_grid(params, np.zeros((1, 3), np.float32), np.ones((1, 1), np.complex64), np.ones((1, 1), np.float32))
    img = oi.grid_to_image(out["grid"][0], out["sumwt"][0])
    inner = (slice(16, 48),) * 2
    assert np.abs(img[inner] - 1.0).max() < 2e-4


def test_P3_hermitian_symmetry(oracle_lib):
    """Gridding {(u,v,w,V)} and {(-u,-v,-w,V*)} gives G'[N-gy][N-gx] = conj(G[gy][gx])."""
    params = base_params(grid_size=64, oversample=4, n_wplanes=8, w_max=80.0, support_min=7, support_max=11,
                         kernel_mode=MODE_WPROJ, cell_size_rad=0.1 / 64)
    uvw, vis, wts, _ = random_vis(params, 400, seed=7)
    _, _, flat, offs = oracle_tables(params)
    g1, rec = oracle_grid(params, uvw, vis, wts, flat=flat, offs=offs)
    g2, rec2 = oracle_grid(params, -uvw, np.conj(vis), wts, flat=flat, offs=offs)
    assert np.array_equal(rec2["sp"], -rec["sp"])
    a, b = g1["grid"][0], g2["grid"][0]
    mirrored = np.conj(a[1:, 1:][::-1, ::-1])
    # exact (up to rounding) unless a sub-cell offset is -O/2, which has no mirror partner: then the
    # mismatch is bounded by the edge taps
    edge = (rec["ox"] == -2) | (rec["oy"] == -2)
    assert edge.any()
    assert np.abs(b[1:, 1:] - mirrored).max() < 2e-2 * np.abs(a).max()
    keep = ~edge
    g1k, _ = oracle_grid(params, uvw[keep], vis[keep], wts[keep], flat=flat, offs=offs)
    g2k, _ = oracle_grid(params, -uvw[keep], np.conj(vis[keep]), wts[keep], flat=flat, offs=offs)
    assert np.abs(g2k["grid"][0][1:, 1:] - np.conj(g1k["grid"][0][1:, 1:][::-1, ::-1])).max() < 1e-12


def test_P4_adjointness(oracle_lib):
    """<G v, g> = <v, G^H g> (BASELINE.json north_star), all modes that share one table for both directions."""
    cases = [
        base_params(grid_size=64, oversample=4, n_wplanes=6, w_max=60.0, support_min=7, support_max=13,
                    kernel_mode=MODE_WPROJ, cell_size_rad=0.1 / 64),
        base_params(grid_size=64, oversample=2, n_wplanes=3, w_max=30.0, support_min=7, support_max=9, n_corr=4,
                    n_pol=4, n_aplanes=3, pa_rad=[0.0, 0.5, 1.0], pointing_lm=[[0, 0]] * 3,
                    leakage=[0.01j, -0.01], kernel_mode=MODE_AWPROJ_ADJOINT, cell_size_rad=0.04 / 64),
        base_params(grid_size=64, oversample=4, support_min=8, support_max=8, n_aplanes=2, pa_rad=[0, 0],
                    pointing_lm=[[0, 0], [0.003, 0.001]], kernel_mode=MODE_MOSAIC_PB, cell_size_rad=0.03 / 64),
    ]
    for params in cases:
        rng = np.random.default_rng(11)
        uvw, vis, _, a = random_vis(params, 200, seed=13, a_planes=params["n_aplanes"] > 1)
        ones = np.ones_like(vis, dtype=np.float32)
        _, _, flat, offs = oracle_tables(params)
        shape = (params["n_pol"], 64, 64)
        g = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
        gv, _ = oracle_grid(params, uvw, vis, ones, a, flat=flat, offs=offs)
        hg, _ = oracle_degrid(params, uvw, g, a, flat=flat, offs=offs)
        lhs = np.vdot(g.astype(np.complex128), gv["grid"])
        rhs = np.vdot(hg["vis"], vis.astype(np.complex128))
        assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_P9_brute_force_dense_matrix(oracle_lib):
    """Tiny case against a dense matrix A[(k,c), (s,y,x)] written straight from O1/O3/O6: grid = A^T (w V),
    degrid = conj(A) g.  Catches a transposed operand, a wrong index order or a wrong conjugate."""
    n = 16
    params = base_params(grid_size=n, oversample=2, n_wplanes=2, w_max=10.0, support_min=3, support_max=5, n_corr=4,
                         n_pol=4, n_aplanes=2, pa_rad=[0.2, 0.9], pointing_lm=[[0, 0]] * 2, leakage=[0.02j, 0.01],
                         kernel_mode=MODE_AWPROJ_ADJOINT, cell_size_rad=0.05 / n)
    uvw, vis, wts, a = random_vis(params, 20, seed=17, frac=0.2, a_planes=True)
    tabs, supports, flat, offs = oracle_tables(params)
    rec = oidx.index_visibilities(uvw, a, params)
    assert not rec["drop"].any()
    amat = np.zeros((20, 4, 4, n, n), np.complex128)
    for k in range(20):
        s_k = int(supports[rec["kset"][k]])
        t = tabs[rec["kset"][k]].astype(np.complex64).astype(np.complex128)
        h = s_k // 2
        for dy in range(s_k):
            for dx in range(s_k):
                amat[k, :, :, rec["gy"][k] - h + dy, rec["gx"][k] - h + dx] = \
                    t[:, :, rec["oy"][k] + 1, rec["ox"][k] + 1, dy, dx].T          # [c][s]
    wv = wts.astype(np.float64) * vis.astype(np.complex128)
    expect_grid = np.einsum("kcsyx,kc->syx", amat, wv)
    out = og.grid(rec, vis, wts, flat, offs, params)
    assert np.abs(out["grid"] - expect_grid).max() < 1e-13
    rng = np.random.default_rng(3)
    g = (rng.standard_normal((4, n, n)) + 1j * rng.standard_normal((4, n, n))).astype(np.complex64)
    expect_vis = np.einsum("kcsyx,syx->kc", np.conj(amat), g.astype(np.complex128))
    dv = og.degrid(rec, g, flat, offs, params)
    assert np.abs(dv["vis"] - expect_vis).max() < 1e-13
    # sampled-cell mode equals the dense result
    cells = np.array([[rec["gy"][0], rec["gx"][0]], [3, 4], [rec["gy"][5] + 1, rec["gx"][5] - 1], [15, 15]])
    sm = og.grid(rec, vis, wts, flat, offs, params, sample_cells=cells)
    assert np.abs(sm["samples"] - out["grid"][:, cells[:, 0], cells[:, 1]]).max() < 1e-15
    assert np.abs(sm["sample_norm"] - out["norm"][:, cells[:, 0], cells[:, 1]]).max() < 1e-15
    # thread count must not change anything (each output element has one owner)
    out1 = og.grid(rec, vis, wts, flat, offs, params, n_threads=1)
    assert np.array_equal(out1["grid"], out["grid"])


def test_P11_identity_mueller_is_four_single_pol_runs(oracle_lib):
    """AWPROJ with J = I (no beam, no leakage, chi = 0): Stokes grids = (S^-1)^H applied to the four
    correlations gridded independently with the plain w-kernel."""
    common = dict(grid_size=64, oversample=4, n_wplanes=4, w_max=40.0, support_min=7, support_max=11,
                  cell_size_rad=0.08 / 64)
    p4 = base_params(n_corr=4, n_pol=4, kernel_mode=MODE_AWPROJ_ADJOINT, dish_diameter_m=0.0, **common)
    p1 = base_params(kernel_mode=MODE_WPROJ, **common)
    uvw, vis, wts, _ = random_vis(p4, 150, seed=23)
    g4, _ = oracle_grid(p4, uvw, vis, wts)
    _, _, flat1, offs1 = oracle_tables(p1)
    singles = np.array([oracle_grid(p1, uvw, vis[:, c:c + 1], wts[:, c:c + 1], flat=flat1, offs=offs1)[0]["grid"][0]
                        for c in range(4)])
    mix = np.conj(np.linalg.inv(ok.STOKES).T)                      # (S^-1)^H  [s][c]
    scale = mix[0, 0]                                              # global normalisation makes element (0,0) unity
    expect = np.einsum("sc,cyx->syx", mix / scale, singles)
    assert np.abs(g4["grid"] - expect).max() < 1e-5 * np.abs(expect).max()   # tables are rounded to complex64


def _model_image(n, sources):
    img = np.zeros((n, n), np.complex128)
    for px, py, amp in sources:
        img[n // 2 + py, n // 2 + px] = amp                    # pixel (N/2, N/2) is l = m = 0; x (l) is the last axis
    return img


def test_P13_image_to_grid_then_degrid_is_the_visibility_equation(oracle_lib):
    """O7 inverse (`image_to_grid`) pinned against Eq. 2: a model image of point sources, pre-corrected by
    the taper and inverse-transformed, then degridded (O5) at random uvw, reproduces V = sum I exp[+2 pi i (ul + vm +
    w (n - 1))] within the method's own approximation error PER VISIBILITY (no averaging over visibilities as in P2):
    nearest sub-cell lookup moves a visibility by at most du / (2 O) per axis (phase 2 pi du/(2O) (|l| + |m|)), nearest
    w-plane by at most w_max / (2 (P - 1)) (phase 2 pi dw |n - 1|), plus 3e-3 for the finite support (P2's bound at
    O = 64).  A dropped n*n, a wrong shift, a wrong sign of the exponent or of the w-term, a transposed image, or a taper
    applied after the transform is off by order one.  Cases: w = 0 (PSWF tables) and a wide field with w (WPROJ)."""
    cases = [
        (base_params(grid_size=64, cell_size_rad=0.05 / 64, oversample=64), 0.05, True,
         [(5, -7, 1.0), (-9, 3, 0.5), (0, 0, 0.3)]),
        (base_params(grid_size=64, cell_size_rad=0.2 / 64, oversample=16, n_wplanes=16, w_max=60.0, support_min=19,
                     support_max=19, kernel_mode=MODE_WPROJ), 0.2, False, [(12, -10, 1.0), (-9, 13, 0.5)]),
    ]
    for params, fov, zero_w, sources in cases:
        n, o = params["grid_size"], params["oversample"]
        cell = fov / n
        uvw, _, _, _ = random_vis(params, 300, seed=5, frac=0.3)
        if zero_w:
            uvw[:, 2] = 0
        dw = 0.0 if zero_w else params["w_max"] / (2 * (params["n_wplanes"] - 1))
        bound = 0.0
        for px, py, amp in sources:
            l, m = px * cell, py * cell
            bound += abs(amp) * (2 * np.pi * (1.0 / fov) / (2 * o) * (abs(l) + abs(m))
                                 + 2 * np.pi * dw * abs(np.sqrt(1 - l * l - m * m) - 1) + 3e-3)
        expect = _point_source_vis(uvw, cell, sources)[:, 0].astype(np.complex128)
        model_grid = oi.image_to_grid(_model_image(n, sources))
        pred, rec = oracle_degrid(params, uvw, model_grid[None].astype(np.complex64))
        assert not rec["drop"].any()
        err = np.abs(pred["vis"][:, 0] - expect).max()
        assert bound < 0.15 and 0.3 * bound < err < bound, (err, bound)      # the bound is tight, not a loose allowance
        # sensitivity: the conjugate (wrong exponent sign), the transposed image (l <-> m) and, with w, a flipped w-term
        assert np.abs(pred["vis"][:, 0] - np.conj(expect)).max() > 5 * bound
        wrong, _ = oracle_degrid(params, uvw, oi.image_to_grid(_model_image(n, sources).T)[None].astype(np.complex64))
        assert np.abs(wrong["vis"][:, 0] - expect).max() > 5 * bound
        if not zero_w:
            flipped = _point_source_vis(uvw * np.array([1, 1, -1], np.float32), cell, sources)[:, 0]
            assert np.abs(pred["vis"][:, 0] - flipped).max() > 5 * bound


def test_P13_grid_to_image_inverts_image_to_grid_up_to_taper_squared():
    """grid_to_image(image_to_grid(x), sum_weights = N^2) * psi^2 = x: both directions divide by the taper (A4 corrects
    the dirty image, A5 pre-corrects the model), and the inverse DFT is unnormalised."""
    n = 32
    rng = np.random.default_rng(2)
    x = np.zeros((2, n, n), np.complex128)
    x[:, n // 4:3 * n // 4, n // 4:3 * n // 4] = rng.standard_normal((2, n // 2, n // 2)) + 1j * rng.standard_normal((2, n // 2, n // 2))
    back = oi.grid_to_image(oi.image_to_grid(x), float(n * n)) * oi.taper_image(n) ** 2
    assert np.abs(back - x).max() < 1e-9 * np.abs(x).max()
    # a single centred unit pixel transforms to a constant grid of 1 / psi(0)^2 = 1 (DC and scale)
    one = np.zeros((n, n), np.complex128)
    one[n // 2, n // 2] = 1.0
    assert np.allclose(oi.image_to_grid(one), 1.0, atol=1e-12)


def test_P21_flagged_samples_contribute_nothing(oracle_lib):
    """Reading R24 (extends R9, "omega = 0 contributes 0"): a sample whose weight is zero, or whose weight or value is not
    finite, adds nothing to the grid and nothing to the sum of weights.  Pinned against what that sentence fixes: the grid of
    a data set with flagged samples (NaN / Inf values at zero weight, a NaN at weight 1, a NaN weight) is, bit for bit, the
    grid of the same data set with those samples replaced by value 0 and weight 0 -- and is finite everywhere."""
    from helpers import MODE_AWPROJ_ADJOINT
    params = base_params(grid_size=64, oversample=4, n_wplanes=3, w_max=30.0, support_min=7, support_max=11, n_corr=4, n_pol=4,
                         n_aplanes=2, pa_rad=[0.0, 0.7], pointing_lm=[[0, 0]] * 2, leakage=[0.01j, -0.01],
                         kernel_mode=MODE_AWPROJ_ADJOINT, cell_size_rad=0.04 / 64)
    uvw, vis, wts, a = random_vis(params, 300, seed=5, a_planes=True)
    clean_vis, clean_wts = vis.copy(), wts.copy()
    for k, c, v, w in [(3, 0, np.nan + 0j, 0.0), (3, 2, complex(np.inf, 1.0), 0.0), (17, 1, complex(2.0, -np.inf), 0.0),
                       (40, 3, complex(np.nan, np.nan), 1.0), (41, 0, 1.0 + 1.0j, np.nan), (42, 2, 1.0 - 2.0j, np.inf)]:
        vis[k, c], wts[k, c] = v, w
        clean_vis[k, c], clean_wts[k, c] = 0.0, 0.0
    wts[50, 1] = clean_wts[50, 1] = 0.0                                   # a plain zero weight with a finite value
    out, _ = oracle_grid(params, uvw, vis, wts, a)
    ref, _ = oracle_grid(params, uvw, clean_vis, clean_wts, a)
    assert np.isfinite(out["grid"]).all() and np.isfinite(out["norm"]).all()
    assert np.array_equal(out["grid"], ref["grid"]) and np.array_equal(out["norm"], ref["norm"])
    assert np.array_equal(out["sumwt"], ref["sumwt"])
    assert np.allclose(out["sumwt"], clean_wts.astype(np.float64).sum(axis=0), rtol=1e-12)
