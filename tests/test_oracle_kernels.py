"""Pins for oracle step O6 (kernel tables) and the paper's Eq. 1-6: P5, P7, P8."""
import os

import numpy as np
from scipy import integrate

from oracle import kernels as ok, imaging as oi
from helpers import base_params, MODE_WPROJ, MODE_AWPROJ_ADJOINT, MODE_AWPROJ_PAPER, MODE_MOSAIC_PB

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_pswf_is_eigenfunction_of_sinc_kernel():
    """The order-0 prolate spheroidal function is the eigenfunction of the finite Fourier transform:
    int_{-1}^{1} psi(t) exp(i c x t) dt = mu * psi(x) on [-1,1]  (textbook definition; pins pswf() against
    something other than scipy's own evaluation of it)."""
    c = np.pi * 7 / 2.0
    xs = np.array([0.0, 0.2, 0.5, 0.8, 0.95])
    vals = np.array([integrate.quad(lambda t: ok.pswf(t, 7) * np.cos(c * x * t), -1, 1, epsabs=1e-12)[0] for x in xs])
    ratio = vals / ok.pswf(xs, 7)
    assert np.allclose(ratio, ratio[0], rtol=2e-7)
    assert ok.pswf(0.0, 7) == 1.0 and abs(ok.pswf(1.0, 7) - 1.92e-4) < 2e-6      # SURVEY 8(c) probe value


def test_P5_pswf_table_is_self_fourier():
    """P5: the PSWF kernel table equals mu' * psi(2 d / S) at tap offset d cells (self-Fourier property), so the
    generator's sampling, sub-cell direction (d - o/O) and crop are right."""
    params = base_params(support_min=7, support_max=7, oversample=8)
    tabs, supports = ok.make_tables(params)
    t = tabs[0][0, 0]                                   # [oy][ox][dy][dx]
    assert list(supports) == [7] and t.shape == (8, 8, 7, 7)
    assert np.max(np.abs(t.imag)) < 1e-12
    d = np.arange(-3, 4)
    peak = abs(t).max()
    for oy in range(-4, 4):
        for ox in range(-4, 4):
            py = ok.pswf(2.0 * (d - oy / 8.0) / 7.0, 7)
            px = ok.pswf(2.0 * (d - ox / 8.0) / 7.0, 7)
            model = np.outer(np.where(np.abs(d - oy / 8.0) <= 3.5, py, 0), np.where(np.abs(d - ox / 8.0) <= 3.5, px, 0))
            got = t[oy + 4, ox + 4].real
            scale = got[3, 3] / model[3, 3]
            assert np.max(np.abs(got - scale * model)) < 3e-3 * peak
    # normalisation: zero-offset taps sum to 1; other offsets within the truncation error
    assert abs(t[4, 4].sum() - 1.0) < 1e-12
    assert np.max(np.abs(t.sum(axis=(2, 3)) - 1.0)) < 3e-4      # SURVEY probe: 1.000007 .. 0.99991 (worst at o = -O/2)


def test_P7_w_kernel_identities():
    params = base_params(grid_size=256, cell_size_rad=0.2 / 256, n_wplanes=4, w_max=150.0, support_min=9,
                         support_max=15, oversample=4, kernel_mode=MODE_WPROJ)
    tabs, supports = ok.make_tables(params)
    assert list(supports) == [15, 13, 11, 9, 11, 13, 15]
    pswf_tabs, _ = ok.make_tables(base_params(grid_size=256, cell_size_rad=0.2 / 256, support_min=9, support_max=9,
                                              oversample=4))
    assert np.array_equal(tabs[3], pswf_tabs[0])                   # plane 0 == plain PSWF kernel, bit for bit
    # T_{-p}(delta) = conj(T_{+p}(-delta)): mirrored taps and mirrored sub-cell offsets (ox=-2 has no partner)
    for p in (1, 2, 3):
        tp, tm = tabs[3 + p][0, 0], tabs[3 - p][0, 0]
        for oy in (-1, 0, 1):
            for ox in (-1, 0, 1):
                assert np.allclose(tm[oy + 2, ox + 2], np.conj(tp[-oy + 2, -ox + 2][::-1, ::-1]), atol=1e-13)
    # Parseval: uncropped sum |Tfine|^2 is independent of w because |exp(i phi)| = 1
    funcs = {k: f for k, _, f in ok.image_functions(params)}
    e = [np.sum(np.abs(ok._fine_kernel(funcs[k][0, 0], 4)) ** 2) for k in (3, 4, 6)]
    assert np.allclose(e, e[0], rtol=1e-12)
    # w-term sign (Eq. 2): the kernel's image-domain phase at (l,m) is exp(-2 pi i w (n-1))
    k, s, f = next(x for x in ok.image_functions(params) if x[0] == 6)
    nk = f.shape[-1]
    j = nk // 2 + 5
    l = 5 * 0.2 / nk
    expected = np.exp(-2j * np.pi * 150.0 * (np.sqrt(1 - 2 * l * l) - 1))
    assert np.allclose(f[0, 0, j, j] / abs(f[0, 0, j, j]), expected, atol=1e-12)


def test_P8_mueller_and_stokes():
    ident = np.eye(2)
    assert np.array_equal(ok.mueller(ident, ident), np.eye(4))                     # J = I  =>  M = I4
    ji, jj = np.diag([1.2 + 0.1j, 0.9]), np.diag([1.1, 0.8 - 0.2j])
    m = ok.mueller(ji, jj)
    assert np.count_nonzero(m - np.diag(np.diag(m))) == 0                          # zero leakage => diagonal
    assert np.allclose(np.diag(m), [ji[0, 0] * np.conj(jj[0, 0]), ji[0, 0] * np.conj(jj[1, 1]),
                                    ji[1, 1] * np.conj(jj[0, 0]), ji[1, 1] * np.conj(jj[1, 1])])
    # leakage lands off the diagonal at first order
    jl = ok.jones_matrix([0.01, 0.02j], 0.0)
    ml = ok.mueller(jl, jl)
    assert abs(ml[0, 1] - np.conj(0.01)) < 1e-15 and abs(ml[0, 2] - 0.01) < 1e-15
    # Eq. 4: unpolarised source XX = YY = 1, XY = YX = 0  ->  I = 1, Q = U = V = 0; pure XX -> I = Q = 1/2
    assert np.allclose(ok.STOKES @ [1, 0, 0, 1], [1, 0, 0, 0])
    assert np.allclose(ok.STOKES @ [1, 0, 0, 0], [0.5, 0.5, 0, 0])
    assert np.allclose(ok.STOKES @ [0, 1, 1, 0], [0, 0, 1, 0])                     # U (reading G3)
    assert np.allclose(ok.STOKES @ [0, -1j, 1j, 0], [0, 0, 0, -1])                 # V = i(YX - XY)/2
    assert np.allclose(ok.STOKES @ np.linalg.inv(ok.STOKES), np.eye(4))
    # Eq. 5: identity Mueller stays identity in the Stokes basis
    assert np.allclose(ok.mueller_stokes(np.eye(4)), np.eye(4))


def test_P8_eq6_closed_forms_and_fig1():
    """Eq. 6: |B'| = |B| + beta/|B| >= 2 sqrt(beta) = eps max|B|, 1/B' = B*/(|B|^2+beta);
    Fig. 1 numbers (tests/golden/fig1_eq6_divergence.txt)."""
    x = np.linspace(-3, 3, 6001)
    beam = np.sinc(x) ** 2                                         # np.sinc = sin(pi x)/(pi x)
    eps = 0.02
    mod = ok.eq6_modify(beam, eps)
    beta = (eps / 2) ** 2
    assert np.all(np.abs(mod) >= eps * 1.0 - 1e-12)
    assert abs(np.abs(mod).min() - eps) < 1e-4                     # equality where |B| = (eps/2) max|B|
    nz = beam > 1e-9
    assert np.allclose(1 / mod[nz], beam[nz] / (beam[nz] ** 2 + beta), rtol=1e-12)
    assert np.all(np.isfinite(1 / mod))                            # finite at the nulls x = +-1, +-2, +-3
    golden = {}
    for line in open(os.path.join(GOLDEN, "fig1_eq6_divergence.txt")):
        if not line.startswith("#") and line.strip():
            name, val, used = line.split()
            golden[name] = (float(val), used == "yes")
    div = 1 - (1 / mod) / (1 / np.where(nz, beam, 1))              # fractional divergence of the inverse
    centre = div[3000]
    assert golden["centre"][1] and abs(centre / golden["centre"][0] - 1) < 0.01
    side = (x > 1.2) & (x < 1.7)
    k = np.argmax(np.where(side, beam, 0))                         # first sidelobe peak of sinc^2
    assert golden["first_sidelobe"][1] and abs(div[k] / golden["first_sidelobe"][0] - 1) < 0.15
    half = np.argmin(np.abs(beam - 0.5) + (x < 0))
    assert abs(div[half] - 4e-4) < 2e-5 and not golden["half_power"][1]     # printed 4e-3 is a typo (G7)


def test_eq1_single_pointing_and_airy():
    b = ok.airy(np.linspace(0, 0.02, 50), 12.0, 1.0e9) ** 2
    g = oi.mosaic_gamma(b[None])
    assert np.allclose(g, (b / b.max()) / b ** 2)
    assert ok.airy(0.0, 12.0, 1e9) == 1.0
    first_null = 1.2196699 * 0.299792458 / 12.0                    # 1.22 lambda / D
    assert abs(ok.airy(first_null, 12.0, 1e9)) < 1e-6


def test_eq1_several_pointings_by_hand():
    """Eq. 1 with N > 1, where sum B_i^2, (sum B_i)^2 and the max term can be told apart.  Values worked by
    hand from the printed formula gamma = [sqrt(sum B_i^2) / max sqrt(sum B_i^2)] [1 / sum B_i^2]."""
    # two flat beams B_1 = 1, B_2 = b: sum B^2 = 1 + b^2 everywhere, the first bracket is 1, gamma = 1 / (1 + b^2)
    # ((sum B)^2 would give 1 / (1 + b)^2 = 0.4444, a plain mean 1 / ((1 + b^2) / 2) = 1.6)
    b = 0.5
    g = oi.mosaic_gamma(np.array([np.ones((3, 4)), np.full((3, 4), b)]))
    assert g.shape == (3, 4) and np.allclose(g, 0.8, rtol=0, atol=1e-15)
    # two pixels, two beams: B_1 = (1, 1/2), B_2 = (1/2, 1/5)  =>  sum B^2 = (5/4, 29/100); the maximum of the root is at
    # pixel 0, so gamma_0 = 1 / (5/4) = 0.8 and gamma_1 = sqrt(29/100) / sqrt(5/4) / (29/100) = sqrt(0.232) / 0.29
    g = oi.mosaic_gamma(np.array([[1.0, 0.5], [0.5, 0.2]]))
    assert abs(g[0] - 0.8) < 1e-15
    assert abs(g[1] - 1.6609095970747993) < 1e-14                  # 0.48166378315169184 / 0.29, by hand calculator
    # three beams that never overlap: each pixel sees one beam, gamma = 1 / (B max B) as for a single pointing
    beams = np.array([[0.9, 0.0, 0.0], [0.0, 0.6, 0.0], [0.0, 0.0, 0.3]])
    assert np.allclose(oi.mosaic_gamma(beams), 1.0 / (np.array([0.9, 0.6, 0.3]) * 0.9), rtol=1e-15)


def test_R10_rotation_sense_and_eq5_on_a_rotation():
    """Reading R10 (J = E D R(chi)) and Eq. 5 pinned on what the mathematics fixes: a rotation of the feeds
    by chi, R = [[cos, -sin], [sin, cos]] acting on (E_x, E_y), leaves Stokes I and V alone and turns (Q, U) by +2 chi:
    a field along x (XX = 1: I = Q = 1/2, U = 0) becomes (cos chi, sin chi), i.e. XX = cos^2, YY = sin^2, XY = YX =
    sin cos, so Q = cos(2 chi)/2 and U = +sin(2 chi)/2.  A transposed rotation flips the sign of the U term; S and S^-1
    swapped in Eq. 5 does not give a real rotation at all."""
    chi = 0.3
    j = ok.jones_matrix([0.0, 0.0], chi)
    assert np.allclose(j @ np.array([1.0, 0.0]), [np.cos(chi), np.sin(chi)], atol=1e-15)
    ms = ok.mueller_stokes(ok.mueller(j, j))
    c2, s2 = 0.8253356149096783, 0.5646424733950354                # cos 0.6, sin 0.6
    want = np.array([[1, 0, 0, 0], [0, c2, -s2, 0], [0, s2, c2, 0], [0, 0, 0, 1]], dtype=np.complex128)
    assert np.allclose(ms, want, atol=1e-15)
    assert np.allclose(ms @ [0.5, 0.5, 0, 0], [0.5, 0.5 * c2, +0.5 * s2, 0], atol=1e-15)     # the worked example above
    # Eq. 5 on a matrix that is not a rotation: pure gain difference g_x = 1, g_y = k mixes I and Q only, as
    # I' = (1 + k^2)/2 I + (1 - k^2)/2 Q and Q' = (1 - k^2)/2 I + (1 + k^2)/2 Q, and scales U and V by k
    k = 0.8
    jg = np.diag([1.0, k])
    mg = ok.mueller_stokes(ok.mueller(jg, jg))
    p, m = (1 + k * k) / 2, (1 - k * k) / 2
    assert np.allclose(mg, [[p, m, 0, 0], [m, p, 0, 0], [0, 0, k, 0], [0, 0, 0, k]], atol=1e-15)
    # leakage enters on the left of the rotation (D R), so at chi = pi/2 it is the SECOND column of D that meets E_x
    jl = ok.jones_matrix([0.01, 0.02j], np.pi / 2)
    assert np.allclose(jl @ np.array([1.0, 0.0]), [0.01, 1.0], atol=1e-15)


def test_awproj_tables_structure():
    """ADJOINT tables are (M S^-1)^H element by element times the scalar w-kernel; PAPER-mode gridding tables
    invert the regularised Stokes Mueller matrix: with zero leakage and a flat beam they reduce to S itself."""
    common = dict(grid_size=128, cell_size_rad=0.02 / 128, n_corr=4, n_pol=4, n_wplanes=2, w_max=50.0,
                  support_min=7, support_max=9, oversample=2, n_aplanes=2, pa_rad=[0.1, 0.7],
                  pointing_lm=[[0, 0]] * 2, leakage=[0.01 * np.exp(0.3j), 0.01 * np.exp(2.1j)])
    pa = base_params(kernel_mode=MODE_AWPROJ_ADJOINT, dish_diameter_m=0.0, **common)      # D = 0: E = 1
    tabs, supports = ok.make_tables(pa)
    assert len(tabs) == 6 and list(supports) == [9, 7, 9, 9, 7, 9]
    wp = base_params(kernel_mode=MODE_WPROJ, **{**common, "n_corr": 1, "n_pol": 1, "n_aplanes": 1,
                                                   "pa_rad": [0.0], "pointing_lm": [[0, 0]]})
    wt, _ = ok.make_tables(wp)
    for a in range(2):
        jm = ok.jones_matrix(pa["leakage"], pa["pa_rad"][a])
        f = np.conj((ok.mueller(jm, jm) @ np.linalg.inv(ok.STOKES)).T)
        for k in range(3):
            scale = tabs[1][0, 0, 1, 1].sum() / wt[1][0, 0, 1, 1].sum() / f0(pa)          # global normalisation
            for s in range(4):
                for c in range(4):
                    assert np.allclose(tabs[a * 3 + k][s, c], f[s, c] * wt[k][0, 0] * scale, atol=1e-13)
    pp = base_params(kernel_mode=MODE_AWPROJ_PAPER, dish_diameter_m=0.0, beam_eps=0.2,
                     **{**common, "leakage": [0j, 0j], "pa_rad": [0.0, 0.0]})
    tg, _ = ok.make_tables(pp, "grid")
    # flat beam B = 1: Eq. 6 gives B' = 1 + (eps/2)^2, so (M^S')^-1 S = S / 1.01 up to the global scale
    ratio = tg[1] / tg[1][0, 0][None, None]
    for s in range(4):
        for c in range(4):
            assert np.allclose(ratio[s, c][abs(tg[1][0, 0]) > 1e-9], ok.STOKES[s, c] / ok.STOKES[0, 0], atol=1e-9)
    td, _ = ok.make_tables(pp, "degrid")
    ta, _ = ok.make_tables(dict(pp, kernel_mode=MODE_AWPROJ_ADJOINT))
    assert all(np.array_equal(x, y) for x, y in zip(td, ta))


def f0(params):
    jm = ok.jones_matrix(params["leakage"], params["pa_rad"][0])
    return np.conj((ok.mueller(jm, jm) @ np.linalg.inv(ok.STOKES)).T)[0, 0]


def test_P12_mosaic_flat_beam_equals_pswf():
    pm = base_params(kernel_mode=MODE_MOSAIC_PB, dish_diameter_m=0.0)
    pp = base_params()
    tm, _ = ok.make_tables(pm)
    tp, _ = ok.make_tables(pp)
    assert np.array_equal(tm[0], tp[0])
    # an off-centre pointing multiplies the image-domain function by the shifted power beam
    pm2 = base_params(kernel_mode=MODE_MOSAIC_PB, n_aplanes=2, pa_rad=[0, 0], pointing_lm=[[0, 0], [0.004, -0.002]],
                      freq_hz=3e9)
    fs = list(ok.image_functions(pm2))
    nk = fs[0][2].shape[-1]
    l1 = (np.arange(nk) - nk // 2) * 0.064 / nk
    ll, mm = np.meshgrid(l1, l1)
    ratio = fs[1][2][0, 0][1:, 1:] / fs[0][2][0, 0][1:, 1:] * ok.airy(np.hypot(ll, mm), 12, 3e9)[1:, 1:] ** 2
    assert np.allclose(ratio, ok.airy(np.hypot(ll - 0.004, mm + 0.002), 12, 3e9)[1:, 1:] ** 2, rtol=1e-9, atol=1e-12)


def test_P14_paper_gridding_function_with_airy_beam_and_leakage():
    """`_paper_gridding_function` (Eq. 6) pinned with an Airy beam and 1 % leakage, where nothing
    degenerates: per pixel F_g S^-1 is the inverse of a matrix M^S' that (a) has the off-diagonal cells of
    M^S = S M S^-1 untouched ("from the diagonal elements"), (b) has Eq. 6 applied to each diagonal beam
    with ITS OWN max|B_p| (a global maximum, or Eq. 6 applied to M instead of M^S, fails), so that
    |B'_p| >= eps max|B_p| everywhere including the nulls of the Airy pattern."""
    nk, eps = 48, 0.2
    l1 = (np.arange(nk) - nk // 2) * 0.12 / nk                     # out to the second null of a 12 m dish at 1 GHz
    ll, mm = np.meshgrid(l1, l1)
    e = ok.airy(np.hypot(ll, mm), 12.0, 1.0e9)
    assert (e < 0).any() and np.abs(e).min() < 2e-3                # sidelobes and a near-null are inside the field
    jm = ok.jones_matrix([0.01 * np.exp(0.4j), 0.01 * np.exp(2.0j)], 0.6)
    m_field = (e * e)[None, None] * ok.mueller(jm, jm)[:, :, None, None]
    fg = ok._paper_gridding_function(m_field, eps)                 # [s][c][y][x]
    s_mat, s_inv = ok.STOKES, np.linalg.inv(ok.STOKES)
    ms = np.einsum("sc,cdyz,dt->styz", s_mat, m_field, s_inv)      # M^S per pixel from the pinned helpers (P8)
    implied = np.linalg.inv(np.einsum("scyz,ct->yzst", fg, s_inv))  # (F_g S^-1)^-1 = M^S' as the oracle built it
    maxima = [np.abs(ms[p, p]).max() for p in range(4)]
    assert max(maxima) / min(maxima) > 1.5                         # the four beams differ: a global maximum would show
    for s in range(4):
        for t in range(4):
            if s != t:
                assert np.allclose(implied[..., s, t], ms[s, t], rtol=1e-9, atol=1e-12)
    for p in range(4):
        b = ms[p, p]
        beta = ((eps / 2.0) * maxima[p]) ** 2
        want = b / np.abs(b) * (np.abs(b) + beta / np.abs(b))      # Eq. 6 with this beam's own maximum
        assert np.allclose(implied[..., p, p], want, rtol=1e-9)
        assert np.abs(implied[..., p, p]).min() >= eps * maxima[p] * (1 - 1e-9)
    # and the defining identity: F_g S^-1 M^S' = I_4 at every pixel
    ident = np.einsum("scyz,ct,yztu->yzsu", fg, s_inv, implied)
    assert np.allclose(ident, np.eye(4)[None, None], atol=1e-9)
