"""Pins for the oracle's PSF convolution and its adjoint (readings C1, C2; not gpu)."""
import numpy as np
import pytest
from scipy import signal

import oracle
from gen.psf import asymmetric_psf, gaussian_psf, moffat_psf


@pytest.mark.parametrize("H,W,K", [(9, 13, 5), (16, 16, 7), (7, 5, 9), (20, 11, 3), (6, 6, 1)])
def test_conv_is_scipy_convolve2d_same_zero_fill(H, W, K):
    rng = np.random.default_rng(H * 100 + W)
    S = rng.normal(size=(H, W))
    psf = asymmetric_psf(K) if K > 1 else np.array([[0.7]])
    ref = signal.convolve2d(S, psf, mode="same", boundary="fill", fillvalue=0.0)
    assert np.allclose(oracle.conv2d_same(S, psf), ref, rtol=0, atol=1e-14)


@pytest.mark.parametrize("H,W,K", [(9, 13, 5), (16, 16, 7), (7, 5, 9)])
def test_adjoint_is_scipy_correlate2d_and_passes_dot_test(H, W, K):
    rng = np.random.default_rng(K)
    S = rng.normal(size=(H, W)); G = rng.normal(size=(H, W))
    psf = asymmetric_psf(K)
    A = oracle.corr2d_same(G, psf)
    assert np.allclose(A, signal.correlate2d(G, psf, mode="same", boundary="fill"), atol=1e-14)
    # <PSF (*) S, G> = <S, PSF (star) G>
    lhs = (oracle.conv2d_same(S, psf) * G).sum()
    rhs = (S * A).sum()
    assert lhs == pytest.approx(rhs, rel=1e-12)


def test_delta_psf_identity_and_shift():
    rng = np.random.default_rng(3)
    S = rng.normal(size=(8, 10))
    d = np.zeros((5, 5)); d[2, 2] = 1.0
    assert np.array_equal(oracle.conv2d_same(S, d), S)
    d = np.zeros((5, 5)); d[1, 4] = 1.0          # a - h = -1, b - h = +2
    out = oracle.conv2d_same(S, d)               # M[i,j] = S[i+1, j-2]
    assert np.array_equal(out[:-1, 2:], S[1:, :-2])
    assert not out[-1, :].any() and not out[:, :2].any()   # zero fill


def test_linearity_and_flux_conservation():
    psf = moffat_psf(25, 3.5, 3.0)
    assert psf.sum() == pytest.approx(1.0, rel=1e-14)
    S = np.zeros((80, 80)); S[38:43, 37:44] = np.arange(35).reshape(5, 7) + 1.0
    M = oracle.conv2d_same(S, psf)
    # source further than h = 12 px from every edge: a normalised PSF conserves flux
    assert M.sum() == pytest.approx(S.sum(), rel=1e-13)
    S2 = np.random.default_rng(0).normal(size=S.shape)
    assert np.allclose(oracle.conv2d_same(2.0 * S - 3.0 * S2, psf),
                       2.0 * M - 3.0 * oracle.conv2d_same(S2, psf), atol=1e-12)
    # near an edge flux leaks out of the cutout (zero fill, no renormalisation)
    S3 = np.zeros((80, 80)); S3[0, 40] = 1.0
    assert oracle.conv2d_same(S3, psf).sum() < 0.75


def test_rendered_flux_conserved_under_normalised_psf():
    # BASELINE north_star: flux conservation under a normalised PSF
    model = {"n_par": 7, "components": [{"kind": "sersic", "convolve": 1, "slots": {
        "xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}}]}
    par = np.array([[40.3, 39.6, 1.0, 2.0, 0.8, 0.7, 0.5]])
    raw = oracle.render(model, par, 80, 80, np.ones((1, 1)))
    con = oracle.render(model, par, 80, 80, gaussian_psf(15, 3.0))
    assert con.sum() == pytest.approx(raw.sum(), rel=1e-9)
    assert con.max() < raw.max()


def test_shared_and_per_galaxy_psf_agree():
    # reading C4: psf_stride 0 and a replicated [B,K,K] stack give identical results
    model = {"n_par": 7, "components": [{"kind": "sersic", "convolve": 1, "slots": {
        "xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}}]}
    par = np.array([[10.3, 9.6, 1.0, 3.0, 1.5, 0.7, 0.5], [9.0, 11.0, 2.0, 2.0, 3.0, 0.4, 2.0]])
    psf = asymmetric_psf(7)
    a = oracle.render(model, par, 20, 22, psf)
    b = oracle.render(model, par, 20, 22, np.stack([psf, psf]))
    assert np.array_equal(a, b)
    c = oracle.render(model, par, 20, 22, np.stack([psf, psf[::-1].copy()]))
    assert np.array_equal(a[0], c[0]) and not np.allclose(a[1], c[1])
