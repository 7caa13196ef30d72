"""Pins for the oracle's special functions and flux relations (not gpu).

Each test checks oracle/gm_oracle.c against something other than itself: a scipy
library routine, a closed form, or numerical quadrature of the oracle's own radial
profile against the paper's total-flux equations (Eq. 5, 8, 10, 15).
"""
import math

import numpy as np
import pytest
from scipy import integrate, special, stats

import oracle

NS = [0.3, 0.5, 0.75, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0, 8.0]


def _golden_nu():
    import pathlib
    rows = {}
    for line in (pathlib.Path(__file__).parent / "golden" / "sersic_nu.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        n, nu, dnu = line.split()
        rows[float(n)] = (float(nu), float(dnu) if dnu != "-" else None)
    return rows


@pytest.mark.parametrize("a,x", [(0.6, 0.2), (1.0, 0.7), (2.0, 1.678), (3.3, 9.0), (12.0, 11.6), (16.0, 40.0)])
def test_gammainc_matches_scipy(a, x):
    assert oracle.gammainc_P(a, x) == pytest.approx(special.gammainc(a, x), rel=1e-13, abs=1e-15)


@pytest.mark.parametrize("n", NS)
def test_nu_is_root_of_half_light(n):
    # r_e encloses half the flux  <=>  gamma(2n, nu) = Gamma(2n)/2
    nu = oracle.sersic_nu(n)
    assert special.gammainc(2 * n, nu) == pytest.approx(0.5, abs=1e-14)
    assert nu == pytest.approx(special.gammaincinv(2 * n, 0.5), rel=1e-13)


def test_nu_closed_forms_and_golden():
    # n = 0.5: P(1,x) = 1 - e^{-x} = 1/2  =>  nu = ln 2 ; n = 1: (1+x) e^{-x} = 1/2
    assert oracle.sersic_nu(0.5) == pytest.approx(math.log(2.0), rel=1e-14)
    nu1 = oracle.sersic_nu(1.0)
    assert (1 + nu1) * math.exp(-nu1) == pytest.approx(0.5, abs=1e-14)
    for n, (nu, dnu) in _golden_nu().items():
        assert oracle.sersic_nu(n) == pytest.approx(nu, rel=2e-10)
        if dnu is not None:
            assert oracle.sersic_dnu_dn(n) == pytest.approx(dnu, rel=2e-8)


@pytest.mark.parametrize("n", NS)
def test_dnu_dn_matches_finite_difference_of_library_inverse(n):
    h = 1e-5 * max(n, 1.0)
    fd = (special.gammaincinv(2 * (n + h), 0.5) - special.gammaincinv(2 * (n - h), 0.5)) / (2 * h)
    assert oracle.sersic_dnu_dn(n) == pytest.approx(fd, rel=1e-7)


def _radial(kind, shape, amp=1.0):
    """I(r) of the oracle for a circular component centred at the origin."""
    p = np.array([0.0, 0.0, 0.0, 1.0, amp, *shape, *([0.0] * (3 - len(shape))), 0.0])
    return lambda r: oracle.component_at(kind, p, r, 0.0)[0]


def _flux_quad(kind, shape, q, rmax=np.inf, amp=1.0, pts=None):
    f = _radial(kind, shape, amp)
    g = lambda r: 2 * math.pi * q * r * f(r)
    edges = [0.0] + sorted(p for p in (pts or []) if p < rmax) + [rmax]
    return sum(integrate.quad(g, a, b, limit=400, epsabs=0, epsrel=1e-12)[0]
               for a, b in zip(edges[:-1], edges[1:]))


@pytest.mark.parametrize("n", [0.5, 1.0, 2.5, 4.0, 6.0])
def test_sersic_total_flux_eq5(n):
    re, q, Ie = 3.7, 0.6, 1.3
    nu = special.gammaincinv(2 * n, 0.5)
    closed = 2 * math.pi * n * Ie * re ** 2 * q * math.exp(nu) * nu ** (-2 * n) * special.gamma(2 * n)
    assert _flux_quad("sersic", [re, n], q, amp=Ie, pts=[re]) == pytest.approx(closed, rel=1e-9)
    # Eq. 5 inverted gives back Ie from that flux
    assert oracle.sersic_Ie_from_flux(closed, re, n, q) == pytest.approx(Ie, rel=1e-12)
    # half of it lies inside r_e
    assert _flux_quad("sersic", [re, n], q, rmax=re, amp=Ie) == pytest.approx(0.5 * closed, rel=1e-9)


def test_expdisk_total_flux_eq8():
    rs, q, I0 = 4.2, 0.35, 2.0
    closed = 2 * math.pi * q * rs ** 2 * I0
    assert _flux_quad("expdisk", [rs], q, amp=I0) == pytest.approx(closed, rel=1e-10)
    assert oracle.expdisk_I0_from_flux(closed, rs, q) == pytest.approx(I0, rel=1e-13)


@pytest.mark.parametrize("a,b", [(1.0, 0.0), (1.7, 0.6), (0.5, 1.5), (3.0, 1.9)])
def test_ferrer_total_flux_eq10(a, b):
    rout, q, I0 = 11.0, 0.8, 0.7
    closed = math.pi * q * rout ** 2 * a * special.beta(a, 1 + 2 / (2 - b)) * I0
    assert _flux_quad("ferrer", [rout, a, b], q, rmax=rout, amp=I0) == pytest.approx(closed, rel=1e-8)
    assert oracle.ferrer_I0_from_flux(closed, rout, a, b, q) == pytest.approx(I0, rel=1e-12)
    if (a, b) == (1.0, 0.0):   # paraboloid: F = pi q r_out^2 I0 / 2
        assert closed == pytest.approx(math.pi * q * rout ** 2 * I0 / 2, rel=1e-14)


@pytest.mark.parametrize("n", [1.5, 3.0, 4.765])
def test_moffat_total_flux_eq15(n):
    fwhm, q, I0 = 3.5, 0.9, 1.1
    rd = fwhm / (2 * math.sqrt(2 ** (1 / n) - 1))
    assert oracle.moffat_rd(fwhm, n) == pytest.approx(rd, rel=1e-14)
    closed = math.pi * q * rd ** 2 * I0 / (n - 1)
    assert _flux_quad("moffat", [fwhm, n], q, amp=I0) == pytest.approx(closed, rel=1e-8)
    assert oracle.moffat_I0_from_flux(closed, fwhm, n, q) == pytest.approx(I0, rel=1e-12)


def test_r_box_eq6():
    assert oracle.r_box(0.0) == pytest.approx(1.0, rel=1e-14)
    # pi (2+B) / (2 beta(1/c,1/c)) is the ratio of the ellipse area pi to the
    # super-ellipse |x|^c + |y|^c <= 1 area 4 Gamma(1+1/c)^2 / Gamma(1+2/c)
    for B in (-0.5, 0.5, 1.0):
        c = 2 + B
        area = 4 * special.gamma(1 + 1 / c) ** 2 / special.gamma(1 + 2 / c)
        assert oracle.r_box(B) == pytest.approx(math.pi / area, rel=1e-13)


def test_boxy_sersic_flux_uses_r_box():
    # 2-D grid sum of a boxy (B != 0) Sersic against Eq. 5 with r_box (Eq. 6)
    n, re, q, B, Ie = 1.0, 6.0, 0.7, 0.6, 1.0
    H = W = 400
    model = {"n_par": 8, "components": [{"kind": "sersic", "convolve": 1, "slots": {
        "xc": 0, "yc": 1, "theta": 2, "q": 3, "amp": 4, "s0": 5, "s1": 6, "box": 7}}]}
    par = np.array([[W / 2, H / 2, 0.4, q, Ie, re, n, B]])
    img = oracle.render(model, par, H, W, np.ones((1, 1)))[0]
    nu = special.gammaincinv(2 * n, 0.5)
    flux = 2 * math.pi * n * Ie * re ** 2 * q * math.exp(nu) * nu ** (-2 * n) * special.gamma(2 * n) / oracle.r_box(B)
    assert img.sum() == pytest.approx(flux, rel=2e-3)
    assert oracle.sersic_Ie_from_flux(flux, re, n, q, B) == pytest.approx(Ie, rel=1e-12)


def test_loglike_eq17_is_chi2_logpdf():
    for chi2, k in [(3.0, 4.0), (4090.0, 4089.0), (12.5, 30.0)]:
        assert oracle.loglike(chi2, k) == pytest.approx(stats.chi2.logpdf(chi2, k), rel=1e-12)
