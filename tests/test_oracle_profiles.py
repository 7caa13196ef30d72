"""Pins for the oracle's radial profiles and ellipse geometry (not gpu).

Identities and special cases the paper states (P:69 n=0.5/n=1, P:121-125 Ferrer,
P:152 King, P:160 and Eq. 14 FWHM, P:174 Moffat limit, P:220 theta at q=1) and
the geometric readings G1-G3 of DESIGN.md.
"""
import math

import numpy as np
import pytest
from scipy import special

import oracle

CF = 2 * math.sqrt(2 * math.log(2))


def comp(kind, xc=0.0, yc=0.0, theta=0.0, q=1.0, amp=1.0, shape=(), box=0.0):
    return np.array([xc, yc, theta, q, amp, *shape, *([0.0] * (3 - len(shape))), box])


def val(kind, p, x, y):
    return oracle.component_at(kind, p, x, y)[0]


def test_sersic_value_at_re_and_centre():
    p = comp("sersic", amp=2.5, shape=(4.0, 3.0))
    assert val("sersic", p, 4.0, 0.0) == pytest.approx(2.5, rel=1e-14)          # I(re) = Ie
    nu = special.gammaincinv(6.0, 0.5)
    assert val("sersic", p, 0.0, 0.0) == pytest.approx(2.5 * math.exp(nu), rel=1e-13)   # S4
    r = 7.3
    assert val("sersic", p, r, 0.0) == pytest.approx(2.5 * math.exp(-nu * ((r / 4.0) ** (1 / 3.0) - 1)), rel=1e-13)


@pytest.mark.parametrize("r", [0.0, 0.3, 1.0, 2.2, 5.0, 9.0])
def test_sersic_half_is_gaussian(r):
    # n = 0.5 is a Gaussian: FWHM = 2 re, I0 = 2 Ie
    re, Ie = 2.2, 0.9
    a = val("sersic", comp("sersic", amp=Ie, shape=(re, 0.5)), r, 0.0)
    b = val("gaussian", comp("gaussian", amp=2 * Ie, shape=(2 * re,)), r, 0.0)
    assert a == pytest.approx(b, rel=1e-12)


@pytest.mark.parametrize("r", [0.0, 0.3, 1.0, 2.2, 5.0, 19.0])
def test_sersic_one_is_exponential(r):
    # n = 1 is an exponential disk: rs = re / nu_1, I0 = Ie e^{nu_1}
    re, Ie = 3.1, 0.4
    nu1 = special.gammaincinv(2.0, 0.5)
    a = val("sersic", comp("sersic", amp=Ie, shape=(re, 1.0)), r, 0.0)
    b = val("expdisk", comp("expdisk", amp=Ie * math.exp(nu1), shape=(re / nu1,)), r, 0.0)
    assert a == pytest.approx(b, rel=1e-12)


def test_de_vaucouleurs_r_quarter_law():
    # n = 4 is the r^{1/4} law: ln I is linear in r^{1/4}
    p = comp("sersic", shape=(5.0, 4.0))
    rs = np.array([0.5, 2.0, 8.0, 30.0])
    y = np.log([val("sersic", p, r, 0.0) for r in rs])
    slope = np.diff(y) / np.diff(rs ** 0.25)
    assert np.allclose(slope, slope[0], rtol=1e-12)


def test_fwhm_half_maximum():
    # P:160 (exact constant, reading F1) and Eq. 14
    for fwhm in (1.2, 3.0, 7.7):
        assert val("gaussian", comp("gaussian", amp=3.0, shape=(fwhm,)), fwhm / 2, 0.0) == pytest.approx(1.5, rel=1e-13)
        for n in (1.0, 2.5, 6.0):
            assert val("moffat", comp("moffat", amp=3.0, shape=(fwhm, n)), 0.0, fwhm / 2) == pytest.approx(1.5, rel=1e-13)
    sigma = 2.0
    assert val("gaussian", comp("gaussian", shape=(CF * sigma,)), sigma, 0.0) == pytest.approx(math.exp(-0.5), rel=1e-13)


def test_moffat_form_and_gaussian_limit():
    fwhm, n, r = 3.5, 3.0, 2.7
    rd = fwhm / (2 * math.sqrt(2 ** (1 / n) - 1))
    assert val("moffat", comp("moffat", shape=(fwhm, n)), r, 0.0) == pytest.approx((1 + (r / rd) ** 2) ** (-n), rel=1e-13)
    # n -> infinity is Gaussian-like (same FWHM)
    g = val("gaussian", comp("gaussian", shape=(fwhm,)), r, 0.0)
    m = val("moffat", comp("moffat", shape=(fwhm, 4000.0)), r, 0.0)
    assert m == pytest.approx(g, rel=2e-3)
    # n = 1 is a Lorentzian: 1 / (1 + (r/rd)^2), rd = FWHM/2
    assert val("moffat", comp("moffat", shape=(fwhm, 1.0)), r, 0.0) == pytest.approx(1 / (1 + (2 * r / fwhm) ** 2), rel=1e-13)


def test_ferrer_shape():
    rout, a, b = 10.0, 1.7, 0.6
    p = comp("ferrer", amp=2.0, shape=(rout, a, b))
    assert val("ferrer", p, 0.0, 0.0) == pytest.approx(2.0)                       # I(0) = I0
    assert val("ferrer", p, rout, 0.0) == 0.0                                     # truncated (S6)
    assert val("ferrer", p, rout * 1.5, 0.0) == 0.0
    assert val("ferrer", p, 4.0, 0.0) == pytest.approx(2.0 * (1 - 0.4 ** (2 - b)) ** a, rel=1e-13)
    I, dI = oracle.component_at("ferrer", p, rout + 1.0, 0.0)
    assert I == 0.0 and not dI.any()
    # "nearly flat core": with b = 0 the slope at the centre vanishes
    p0 = comp("ferrer", shape=(rout, 2.0, 0.0))
    assert val("ferrer", p0, 1e-3, 0.0) == pytest.approx(1.0, abs=1e-7)


def test_king_shape_reading_K1():
    rc, rt = 2.0, 15.0
    for al in (0.7, 2.0, 3.3):
        p = comp("king", amp=1.9, shape=(rc, rt, al))
        assert val("king", p, 0.0, 0.0) == pytest.approx(1.9, rel=1e-13)          # I(0) = I0, finite for any alpha
        assert val("king", p, rt, 0.0) == 0.0
        assert val("king", p, rt - 1e-9, 0.0) == pytest.approx(0.0, abs=1e-6)
        assert val("king", p, 0.5 * rt, 0.0) > 0.0
    # alpha = 2 is King (1962): I ~ [ (1+(r/rc)^2)^{-1/2} - (1+(rt/rc)^2)^{-1/2} ]^2
    p = comp("king", amp=1.0, shape=(rc, rt, 2.0))
    f = lambda r: (1 / math.sqrt(1 + (r / rc) ** 2) - 1 / math.sqrt(1 + (rt / rc) ** 2)) ** 2
    for r in (0.5, 3.0, 9.0):
        assert val("king", p, r, 0.0) == pytest.approx(f(r) / f(0.0), rel=1e-13)


def test_sky_is_flat():
    I, dI = oracle.component_at("sky", comp("sky", amp=0.37), 11.0, -3.0)
    assert I == 0.37 and dI[4] == 1.0 and np.count_nonzero(dI) == 1


# ---- geometry: Eq. 2-4 with readings G1-G3 ------------------------------------
def test_elliptical_radius_definition():
    # r^2 = u^2 + (v/q)^2 with (u,v) the coordinates rotated by theta (reading G2)
    xc, yc, th, q = 1.5, -0.5, 0.7, 0.4
    p = comp("expdisk", xc=xc, yc=yc, theta=th, q=q, shape=(3.0,))
    for x, y in [(4.0, 2.0), (-3.0, 1.0), (0.3, -6.0)]:
        dx, dy = x - xc, y - yc
        u = math.cos(th) * dx + math.sin(th) * dy
        v = -math.sin(th) * dx + math.cos(th) * dy
        r = math.hypot(u, v / q)
        assert val("expdisk", p, x, y) == pytest.approx(math.exp(-r / 3.0), rel=1e-13)


def test_theta_zero_matches_printed_eq3_eq4():
    # at theta = 0 the printed per-term absolute values and reading G2 coincide
    q = 0.5
    p = comp("expdisk", q=q, shape=(2.0,))
    for x, y in [(3.0, 1.0), (-3.0, 1.0), (3.0, -1.0)]:
        r = math.hypot(abs(x), abs(y) / q)
        assert val("expdisk", p, x, y) == pytest.approx(math.exp(-r / 2.0), rel=1e-13)


def test_round_profile_ignores_theta():
    # at q = 1 the light distribution does not depend on theta
    a = val("sersic", comp("sersic", theta=0.0, shape=(3.0, 2.0)), 2.0, 5.0)
    b = val("sersic", comp("sersic", theta=1.1, shape=(3.0, 2.0)), 2.0, 5.0)
    assert a == pytest.approx(b, rel=1e-13)
    # ... and is circular: depends on dx^2 + dy^2 only
    c = val("sersic", comp("sersic", theta=0.6, shape=(3.0, 2.0)), math.hypot(2.0, 5.0), 0.0)
    assert a == pytest.approx(c, rel=1e-13)


def test_theta_distinguishes_sign_and_has_period_pi():
    p_plus = comp("expdisk", theta=0.5, q=0.3, shape=(3.0,))
    p_minus = comp("expdisk", theta=-0.5, q=0.3, shape=(3.0,))
    assert abs(val("expdisk", p_plus, 4.0, 2.0) - val("expdisk", p_minus, 4.0, 2.0)) > 1e-3
    p_pi = comp("expdisk", theta=0.5 + math.pi, q=0.3, shape=(3.0,))
    assert val("expdisk", p_plus, 4.0, 2.0) == pytest.approx(val("expdisk", p_pi, 4.0, 2.0), rel=1e-12)


def _image(theta, H=41, W=41, q=0.3):
    model = {"n_par": 6, "components": [{"kind": "expdisk", "convolve": 1, "slots": {
        "xc": 0, "yc": 1, "theta": 2, "q": 3, "amp": 4, "s0": 5}}]}
    par = np.array([[W / 2, H / 2, theta, q, 1.0, 4.0]])
    return oracle.render(model, par, H, W, np.ones((1, 1)))[0]


def _moments(img):
    H, W = img.shape
    ii, jj = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    t = img.sum()
    ci, cj = (img * ii).sum() / t, (img * jj).sum() / t
    return ((img * (ii - ci) ** 2).sum() / t, (img * (jj - cj) ** 2).sum() / t,
            (img * (ii - ci) * (jj - cj)).sum() / t)


def test_position_angle_convention_G1_G3():
    # theta from +x towards +y on the y-up grid (row index grows downwards)
    vii, vjj, _ = _moments(_image(0.0))
    assert vjj > 3 * vii                      # theta = 0: elongated along a row (x)
    vii, vjj, _ = _moments(_image(math.pi / 2))
    assert vii > 3 * vjj                      # theta = pi/2: along a column (y)
    _, _, vij = _moments(_image(math.pi / 4))
    assert vij < 0                            # bottom-left to top-right: row falls as column grows
    # centred q<1 image is symmetric under the point reflection, and the pi/2
    # rotation equals the transpose of the mirrored image (square cutout)
    a, b = _image(0.3), _image(0.3 + math.pi / 2)
    assert np.allclose(a, a[::-1, ::-1], rtol=1e-12)
    assert np.allclose(b, a.T[::-1, :][:, :], rtol=1e-12) or np.allclose(b, a.T[:, ::-1], rtol=1e-12)


def test_pixel_grid_G1():
    # pixel (i, j) is sampled at x = j + 0.5, y = H - 0.5 - i
    H, W = 6, 9
    model = {"n_par": 6, "components": [{"kind": "gaussian", "convolve": 1, "slots": {
        "xc": 0, "yc": 1, "theta": 2, "q": 3, "amp": 4, "s0": 5}}]}
    i0, j0 = 1, 6
    par = np.array([[j0 + 0.5, H - 0.5 - i0, 0.0, 1.0, 1.0, 2.0]])
    img = oracle.render(model, par, H, W, np.ones((1, 1)))[0]
    assert np.unravel_index(np.argmax(img), img.shape) == (i0, j0)
    assert img[i0, j0] == pytest.approx(1.0, rel=1e-14)
    assert img[i0 + 1, j0] == pytest.approx(img[i0, j0 - 1], rel=1e-13)


def test_boxiness_changes_isophote_shape():
    # Eq. 2: on the axes r is independent of B; on the diagonal B>0 gives smaller r (boxy)
    for B in (-0.5, 0.5):
        p = comp("expdisk", shape=(3.0,), box=B)
        assert val("expdisk", p, 2.0, 0.0) == pytest.approx(math.exp(-2.0 / 3.0), rel=1e-13)
        c = 2 + B
        r = (2 * 1.5 ** c) ** (1 / c)
        assert val("expdisk", p, 1.5, 1.5) == pytest.approx(math.exp(-r / 3.0), rel=1e-13)
