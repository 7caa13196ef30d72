"""Pins for the oracle's chi^2 (Eq. 18) and analytic gradient (not gpu):
brute-force loops, mask/sigma properties (reading X1), central finite differences
on tiny images for every profile, tied parameters, unconvolved components, sky,
and the Gauss-Newton blocks J^T W J / J^T W r."""
import math

import numpy as np
import pytest

import oracle
from gen import models
from gen.psf import asymmetric_psf


def sample_params(model, H, W, rng):
    """A generic in-range parameter vector for any gen.models model."""
    p = np.empty(model["n_par"])
    for k, (role, name) in enumerate(zip(model["roles"], model["names"])):
        if role == "cx": p[k] = W / 2 + rng.uniform(-1.5, 1.5)
        elif role == "cy": p[k] = H / 2 + rng.uniform(-1.5, 1.5)
        elif role == "amp": p[k] = rng.uniform(0.5, 2.0)
        elif role == "radius": p[k] = rng.uniform(2.0, 4.0)
        elif role == "index": p[k] = rng.uniform(0.7, 3.5)
        elif role == "q": p[k] = rng.uniform(0.4, 0.9)
        elif role == "theta": p[k] = rng.uniform(0.1, 3.0)
        elif role == "shape": p[k] = rng.uniform(1.2, 2.5)
        elif role == "sky": p[k] = rng.uniform(-0.1, 0.1)
        elif role == "box": p[k] = rng.uniform(-0.5, 0.8)
        elif role == "mag": p[k] = rng.uniform(16.5, 18.0)
        elif role == "zeropoint": p[k] = 22.5
        if name.endswith("_b") or name == "b": p[k] = rng.uniform(0.2, 1.2)
        if name.endswith("rt"): p[k] = rng.uniform(9.0, 14.0)
        if name.endswith("rout"): p[k] = rng.uniform(7.0, 11.0)
    return p


def make_problem(model, H, W, K, seed, masked=True):
    rng = np.random.default_rng(seed)
    truth = sample_params(model, H, W, rng)[None]
    psf = asymmetric_psf(K)
    M = oracle.render(model, truth, H, W, psf)
    sigma = 0.05 + 0.1 * rng.random((1, H, W))
    data = M + sigma * rng.normal(size=M.shape)
    mask = (rng.random((1, H, W)) > 0.15).astype(np.uint8) if masked else None
    par = truth * (1 + 0.05 * rng.uniform(-1, 1, size=truth.shape))
    return par, data, sigma, mask, psf


def fd_grad(model, par, data, sigma, mask, psf, rel=1e-6):
    g = np.zeros_like(par)
    for k in range(par.shape[1]):
        h = rel * max(abs(par[0, k]), 1.0)
        pp, pm = par.copy(), par.copy()
        pp[0, k] += h; pm[0, k] -= h
        cp, _ = oracle.loss_grad(model, pp, data, sigma, mask, psf)
        cm, _ = oracle.loss_grad(model, pm, data, sigma, mask, psf)
        g[0, k] = (cp[0] - cm[0]) / (2 * h)
    return g


def test_chi2_brute_force_eq18():
    model = models.single_sersic()
    H, W, K = 7, 9, 3
    par, data, sigma, mask, psf = make_problem(model, H, W, K, 1)
    M = oracle.render(model, par, H, W, psf)[0]
    tot = 0.0
    for i in range(H):
        for j in range(W):
            if mask[0, i, j]:
                tot += (data[0, i, j] - M[i, j]) ** 2 / sigma[0, i, j] ** 2
    chi2, _ = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert chi2[0] == pytest.approx(tot, rel=1e-13)


def test_mask_and_sigma_properties_X1():
    model = models.single_sersic()
    par, data, sigma, mask, psf = make_problem(model, 10, 10, 5, 2)
    chi2, grad = oracle.loss_grad(model, par, data, sigma, mask, psf)
    z, gz = oracle.loss_grad(model, par, data, sigma, np.zeros_like(mask), psf)
    assert z[0] == 0.0 and not gz.any()                      # all-zero mask
    c4, g4 = oracle.loss_grad(model, par, data, 0.5 * sigma, mask, psf)
    assert c4[0] == pytest.approx(4 * chi2[0], rel=1e-13)    # halving sigma quadruples chi2
    assert np.allclose(g4, 4 * grad, rtol=1e-12)
    bad = data.copy(); bs = sigma.copy()
    i, j = np.argwhere(mask[0] == 0)[0]
    bad[0, i, j] = np.nan; bs[0, i, j] = 0.0                 # NaN / sigma=0 under the mask
    cn, gn = oracle.loss_grad(model, par, bad, bs, mask, psf)
    assert cn[0] == chi2[0] and np.array_equal(gn, grad)
    cnone, _ = oracle.loss_grad(model, par, data, sigma, None, psf)
    call, _ = oracle.loss_grad(model, par, data, sigma, np.ones_like(mask), psf)
    assert cnone[0] == call[0] and cnone[0] > chi2[0]


def test_model_equals_data_gives_zero():
    model = models.single_sersic()
    par, data, sigma, mask, psf = make_problem(model, 10, 10, 5, 3)
    M = oracle.render(model, par, 10, 10, psf)
    chi2, grad = oracle.loss_grad(model, par, M, sigma, mask, psf)
    assert chi2[0] == 0.0 and not grad.any()


@pytest.mark.parametrize("kind", ["sersic", "expdisk", "ferrer", "king", "gaussian", "moffat"])
@pytest.mark.parametrize("convolve", [1, 0])
def test_gradient_vs_central_differences_each_profile(kind, convolve):
    model = models.one_component(kind, convolve)
    H, W, K = 12, 13, 5
    par, data, sigma, mask, psf = make_problem(model, H, W, K, 10 + len(kind) + convolve)
    _, grad = oracle.loss_grad(model, par, data, sigma, mask, psf)
    fd = fd_grad(model, par, data, sigma, mask, psf)
    assert np.allclose(grad, fd, rtol=2e-6, atol=1e-6 * np.abs(fd).max())


def test_gradient_all_profiles_tied_sky_unconvolved():
    model = models.all_profiles()
    H, W, K = 14, 12, 5
    par, data, sigma, mask, psf = make_problem(model, H, W, K, 77)
    _, grad = oracle.loss_grad(model, par, data, sigma, mask, psf)
    fd = fd_grad(model, par, data, sigma, mask, psf)
    assert np.allclose(grad, fd, rtol=5e-6, atol=1e-6 * np.abs(fd).max())
    assert np.all(np.abs(grad) > 0)          # every parameter matters, incl. sky and tied ones


def test_gradient_bulge_disk_and_boxiness():
    model = models.bulge_disk()
    par, data, sigma, mask, psf = make_problem(model, 12, 12, 5, 5)
    _, grad = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert np.allclose(grad, fd_grad(model, par, data, sigma, mask, psf), rtol=2e-6, atol=1e-7)
    boxy = {"n_par": 8, "components": [{"kind": "sersic", "convolve": 1, "slots": {
        "xc": 0, "yc": 1, "theta": 2, "q": 3, "amp": 4, "s0": 5, "s1": 6, "box": 7}}]}
    rng = np.random.default_rng(9)
    par = np.array([[6.2, 5.7, 0.6, 0.6, 1.0, 3.0, 1.7, 0.4]])
    psf = asymmetric_psf(5)
    M = oracle.render(boxy, par, 12, 12, psf)
    sigma = np.full_like(M, 0.1); data = M + 0.1 * rng.normal(size=M.shape)
    par2 = par * 1.03
    _, grad = oracle.loss_grad(boxy, par2, data, sigma, None, psf)
    assert np.allclose(grad, fd_grad(boxy, par2, data, sigma, None, psf), rtol=5e-6, atol=1e-6)


def test_centre_on_pixel_centre_is_finite_and_smooth_S4():
    model = models.single_sersic()
    H = W = 11
    psf = asymmetric_psf(3)
    for n, tol in ((4.0, None), (1.2, 0.05)):
        par = np.array([[5.5, 5.5, 1.0, 3.0, n, 0.7, 0.3]])   # centre exactly on pixel (5,5)
        M = oracle.render(model, par, H, W, psf)
        assert np.isfinite(M).all()
        sigma = np.full_like(M, 0.1); data = M * 1.1
        chi2, grad = oracle.loss_grad(model, par, data, sigma, None, psf)
        assert np.isfinite(chi2).all() and np.isfinite(grad).all()
        if tol is None:
            continue    # n = 4 point-sampled: the central pixel is a true cusp, only finiteness holds
        par2 = par.copy(); par2[0, 0] += 1e-3
        chi2b, _ = oracle.loss_grad(model, par2, data, sigma, None, psf)
        assert abs(chi2b[0] - chi2[0]) < tol * chi2[0]


def test_sky_adds_constant_everywhere_C3():
    model = {"n_par": 8, "components": models.single_sersic()["components"] + [
        {"kind": "sky", "convolve": 1, "slots": {"amp": 7}}]}          # flag ignored for sky
    par = np.array([[6.0, 6.0, 1.0, 3.0, 1.0, 0.8, 0.2, 0.0]])
    psf = asymmetric_psf(5)
    a = oracle.render(model, par, 12, 12, psf)
    par[0, 7] = 0.25
    b = oracle.render(model, par, 12, 12, psf)
    assert np.allclose(b - a, 0.25, rtol=0, atol=1e-15)       # including edge pixels


def test_gauss_newton_blocks():
    model = models.bulge_disk()
    H, W, K = 10, 11, 5
    par, data, sigma, mask, psf = make_problem(model, H, W, K, 21)
    chi2, grad, jtj, jtr = oracle.loss_grad(model, par, data, sigma, mask, psf, want_jtj=True)
    assert np.allclose(grad, -2 * jtr, rtol=1e-10, atol=1e-12)          # grad = -2 J^T W rho
    # J by central differences of the rendered model
    P = par.shape[1]
    J = np.zeros((P, H * W))
    for k in range(P):
        h = 1e-6 * max(abs(par[0, k]), 1.0)
        pp, pm = par.copy(), par.copy(); pp[0, k] += h; pm[0, k] -= h
        J[k] = ((oracle.render(model, pp, H, W, psf) - oracle.render(model, pm, H, W, psf)) / (2 * h)).ravel()
    w = np.where(mask[0].ravel() != 0, 1 / sigma[0].ravel() ** 2, 0.0)
    ref = (J * w) @ J.T
    assert np.allclose(jtj[0], ref, rtol=1e-5, atol=1e-6 * np.abs(ref).max())
    assert np.allclose(jtj[0], jtj[0].T, rtol=1e-12)
