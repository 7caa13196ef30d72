"""Pins for the oracle's magnitude parameterisation (Eq. 5, 6, 8, 10, 15; P:84-93, P:115,
P:129) and boxiness (Eq. 2) inside the forward model and gradient
(SURVEY 8(f)-2).  Not gpu.

The flux <-> amplitude helpers themselves are pinned to quadrature of the radial laws in
test_oracle_special.py; here: the logarithmic derivatives against finite differences of
those helpers, the rendered total flux against 10^{-0.4 (m - m0)}, equivalence with the
intensity parameterisation, and the chi^2 gradient against central differences."""
import numpy as np
import pytest

import oracle
from gen import models
from gen.psf import asymmetric_psf

# slot order: xc yc theta q amp s0 s1 s2 box m0
CASES = {
    "sersic": [0.0, 0.0, 0.3, 0.7, 18.2, 5.0, 2.5, 0.0, 0.3, 22.5],
    "expdisk": [0.0, 0.0, 0.3, 0.6, 17.5, 4.0, 0.0, 0.0, -0.4, 22.5],
    "ferrer": [0.0, 0.0, 0.3, 0.5, 19.0, 9.0, 1.7, 0.6, 0.2, 22.5],
    "moffat": [0.0, 0.0, 0.3, 0.9, 20.0, 3.0, 2.8, 0.0, 0.1, 22.5],
}


def helper_amp(kind, p):
    """Amplitude through the separately pinned Eq. 5/8/10/15 helpers."""
    q, m, s0, s1, s2, B, m0 = p[3], p[4], p[5], p[6], p[7], p[8], p[9]
    flux = 10.0 ** (-0.4 * (m - m0))
    if kind == "sersic": return oracle.sersic_Ie_from_flux(flux, s0, s1, q, B)
    if kind == "expdisk": return oracle.expdisk_I0_from_flux(flux, s0, q, B)
    if kind == "ferrer": return oracle.ferrer_I0_from_flux(flux, s0, s1, s2, q, B)
    return oracle.moffat_I0_from_flux(flux, s0, s1, q, B)


@pytest.mark.parametrize("kind", list(CASES))
def test_log_amplitude_derivatives_vs_finite_differences_of_the_helpers(kind):
    p = np.array(CASES[kind])
    amp, dla = oracle.amplitude_from_mag(kind, p)
    assert amp == pytest.approx(helper_amp(kind, p), rel=1e-14)
    used = {"sersic": [3, 4, 5, 6, 8, 9], "expdisk": [3, 4, 5, 8, 9],
            "ferrer": [3, 4, 5, 6, 7, 8, 9], "moffat": [3, 4, 5, 6, 8, 9]}[kind]
    for k in range(10):
        if k not in used:
            assert dla[k] == 0.0
            continue
        h = 1e-6 * max(abs(p[k]), 1.0)
        pp, pm = p.copy(), p.copy()
        pp[k] += h; pm[k] -= h
        fd = (np.log(helper_amp(kind, pp)) - np.log(helper_amp(kind, pm))) / (2 * h)
        assert dla[k] == pytest.approx(fd, rel=2e-7, abs=1e-9), (kind, k)


def test_magnitude_is_pogson_scale():
    # 5 magnitudes = a factor 100 in intensity; m = m0 is unit flux (Eq. 5)
    p = np.array(CASES["sersic"])
    a1, _ = oracle.amplitude_from_mag("sersic", p)
    p2 = p.copy(); p2[4] -= 5.0
    a2, _ = oracle.amplitude_from_mag("sersic", p2)
    assert a2 / a1 == pytest.approx(100.0, rel=1e-13)
    p3 = p.copy(); p3[4] = p3[9]
    a3, _ = oracle.amplitude_from_mag("sersic", p3)
    assert a3 == pytest.approx(oracle.sersic_Ie_from_flux(1.0, p[5], p[6], p[3], p[8]), rel=1e-14)


@pytest.mark.parametrize("kind,box", [("expdisk", 0.0), ("expdisk", 0.6), ("moffat", -0.3), ("ferrer", 0.4)])
def test_rendered_total_flux_is_the_magnitude(kind, box):
    # sum of the rendered pixels of a well-resolved, well-contained source = 10^{-0.4 (m - m0)}
    model = models.one_component(kind, convolve=0, box=True, mag=True)
    H = W = 400
    shape = {"expdisk": [9.0], "moffat": [14.0, 4.0], "ferrer": [60.0, 1.6, 0.5]}[kind]
    par = np.array([[W / 2 + 0.13, H / 2 - 0.21, 0.7, 0.65, 16.0, *shape, box, 22.5]])
    img = oracle.render(model, par, H, W, np.ones((1, 1)))
    tol = {"expdisk": 2e-3, "moffat": 2e-3, "ferrer": 1e-3}[kind]
    assert img.sum() == pytest.approx(10.0 ** (-0.4 * (16.0 - 22.5)), rel=tol)


@pytest.mark.parametrize("kind", list(CASES))
def test_magnitude_model_equals_intensity_model(kind):
    mm = models.one_component(kind, box=True, mag=True)
    mi = models.one_component(kind, box=True, mag=False)
    p = np.array(CASES[kind])
    nshape = {"sersic": 2, "expdisk": 1, "ferrer": 3, "moffat": 2}[kind]
    geo = [7.3, 6.1, p[2], p[3]]
    pm = np.array([[*geo, p[4], *p[5:5 + nshape], p[8], p[9]]])
    pi = np.array([[*geo, helper_amp(kind, p), *p[5:5 + nshape], p[8]]])
    psf = asymmetric_psf(5)
    a = oracle.render(mm, pm, 14, 15, psf)
    b = oracle.render(mi, pi, 14, 15, psf)
    assert np.allclose(a, b, rtol=1e-13, atol=0)


def _fd_grad(model, par, data, sigma, mask, psf):
    g = np.zeros_like(par)
    for k in range(par.shape[1]):
        h = 1e-6 * max(abs(par[0, k]), 1.0)
        pp, pm = par.copy(), par.copy()
        pp[0, k] += h; pm[0, k] -= h
        g[0, k] = (oracle.loss_grad(model, pp, data, sigma, mask, psf)[0][0] -
                   oracle.loss_grad(model, pm, data, sigma, mask, psf)[0][0]) / (2 * h)
    return g


@pytest.mark.parametrize("kind", list(CASES))
@pytest.mark.parametrize("convolve", [1, 0])
def test_gradient_in_magnitudes_with_boxiness_vs_central_differences(kind, convolve):
    model = models.one_component(kind, convolve, box=True, mag=True)
    p = np.array(CASES[kind])
    nshape = {"sersic": 2, "expdisk": 1, "ferrer": 3, "moffat": 2}[kind]
    truth = np.array([[6.3, 5.8, p[2], p[3], p[4] - 4.0, *p[5:5 + nshape], p[8], p[9]]])
    truth[0, 5] = min(truth[0, 5], 6.0)
    rng = np.random.default_rng(31 + convolve)
    psf = asymmetric_psf(5)
    M = oracle.render(model, truth, 12, 13, psf)
    sigma = 0.02 * M.max() * (1 + rng.random(M.shape))
    data = M + sigma * rng.normal(size=M.shape)
    mask = (rng.random(M.shape) > 0.1).astype(np.uint8)
    par = truth * (1 + 0.01 * rng.uniform(-1, 1, size=truth.shape))
    _, grad = oracle.loss_grad(model, par, data, sigma, mask, psf)
    fd = _fd_grad(model, par, data, sigma, mask, psf)
    assert np.allclose(grad, fd, rtol=5e-6, atol=2e-6 * np.abs(fd).max())
    k_m, k_m0 = model["names"].index("mag"), model["names"].index("m0")
    assert grad[0, k_m0] == pytest.approx(-grad[0, k_m], rel=1e-12)     # only m - m0 enters


def test_gradient_boxy_bulge_disk_shared_zero_point():
    model = models.boxy_bulge_disk_mag()
    truth = np.array([[7.2, 6.6, 14.5, 2.5, 2.2, 0.7, 0.5, 0.3, 13.8, 4.0, 0.5, 1.9, -0.3, 22.5]])
    rng = np.random.default_rng(4)
    psf = asymmetric_psf(5)
    M = oracle.render(model, truth, 14, 14, psf)
    sigma = 0.03 * M.max() * (1 + rng.random(M.shape))
    data = M + sigma * rng.normal(size=M.shape)
    par = truth * (1 + 0.01 * rng.uniform(-1, 1, size=truth.shape))
    _, grad = oracle.loss_grad(model, par, data, sigma, None, psf)
    fd = _fd_grad(model, par, data, sigma, None, psf)
    assert np.allclose(grad, fd, rtol=5e-6, atol=2e-6 * np.abs(fd).max())
    # the shared zero point collects minus the sum of both magnitude gradients
    assert grad[0, 13] == pytest.approx(-(grad[0, 2] + grad[0, 8]), rel=1e-10)


def test_magnitude_slot_on_a_profile_without_a_relation_is_rejected():
    model = models.one_component("king", mag=True)
    par = np.array([[5.0, 5.0, 0.0, 0.8, 18.0, 2.0, 9.0, 2.0, 22.5]])
    with pytest.raises(AssertionError):
        oracle.render(model, par, 10, 10, np.ones((1, 1)))
