"""Pins for the oracle's covariance-matrix uncertainties (Sec. 5.2; not gpu):
sigma_p = sqrt(diag[(J^T W J)^-1]) against numpy.linalg.inv, the closed form of a model
that is linear in its free parameters, and the scatter of least-squares refits over
noise realisations (which fixes W = 1/sigma^2 and the absence of stray factors)."""
import numpy as np

import oracle
from gen import models
from gen.psf import asymmetric_psf, gaussian_psf
from test_oracle_lossgrad import make_problem


def test_inverse_matches_numpy_on_random_spd():
    rng = np.random.default_rng(0)
    for P in (1, 2, 5, 11, 32):
        X = rng.normal(size=(3 * P + 2, P)) * 10.0 ** rng.uniform(-3, 3, size=P)   # badly scaled columns
        A = X.T @ X
        sp, st = oracle.covariance_sigma(A)
        assert st == 0
        D = np.sqrt(np.diag(A))
        ref = np.sqrt(np.diag(np.linalg.inv(A / np.outer(D, D)))) / D
        assert np.allclose(sp, ref, rtol=1e-9)


def test_free_mask_drops_rows_and_columns():
    rng = np.random.default_rng(1)
    X = rng.normal(size=(40, 6)); A = X.T @ X
    fm = np.array([1, 0, 1, 1, 0, 1], dtype=np.uint8)
    sp, st = oracle.covariance_sigma(A, fm)
    keep = np.flatnonzero(fm)
    assert st == 0 and sp[1] == 0.0 and sp[4] == 0.0
    assert np.allclose(sp[keep], np.sqrt(np.diag(np.linalg.inv(A[np.ix_(keep, keep)]))), rtol=1e-11)
    # fixing a parameter can only shrink the others' uncertainties
    full, _ = oracle.covariance_sigma(A)
    assert np.all(sp[keep] <= full[keep] * (1 + 1e-12))


def test_singular_matrix_is_flagged():
    A = np.array([[1.0, 2.0], [2.0, 4.0]])
    sp, st = oracle.covariance_sigma(A)
    assert st == 1 and np.isnan(sp).all()
    # a round profile (q = 1) does not depend on theta: zero row/column in J^T W J
    model = models.single_sersic()
    par = np.array([[8.2, 7.9, 1.0, 3.0, 1.5, 1.0, 0.4]])
    sig = np.full((1, 16, 16), 0.1)
    u = oracle.uncertainty(model, par, sig, None, gaussian_psf(5, 2.0))
    # (in floating point the theta column is ~1e-16, not 0: either answer says "unconstrained")
    assert u["status"][0] == 1 or u["sigma_p"][0, 6] > 1e8
    Z = np.diag([1.0, 0.0, 2.0])                                   # an exactly zero row and column
    sp, st = oracle.covariance_sigma(Z)
    assert st == 1 and np.isnan(sp).all()
    fm = np.array([1, 1, 1, 1, 1, 1, 0], dtype=np.uint8)           # hold theta: well posed again
    u = oracle.uncertainty(model, par, sig, None, gaussian_psf(5, 2.0), fm)
    assert u["status"][0] == 0 and np.isfinite(u["sigma_p"][0]).all() and u["sigma_p"][0, 6] == 0.0


def linear_problem():
    # unconvolved Gaussian point source + flat sky: M = I0 U(x,y) + I_sky is linear in (I0, I_sky)
    model = {"n_par": 6, "components": [
        {"kind": "gaussian", "convolve": 0, "slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3}},
        {"kind": "sky", "convolve": 0, "slots": {"amp": 4}}]}
    model["n_par"] = 5
    H, W = 15, 17
    par = np.array([[8.3, 7.6, 2.0, 4.0, 0.3]])
    rng = np.random.default_rng(5)
    sigma = 0.05 + 0.2 * rng.random((1, H, W))
    mask = (rng.random((1, H, W)) > 0.2).astype(np.uint8)
    fm = np.array([0, 0, 1, 0, 1], dtype=np.uint8)
    return model, par, sigma, mask, fm, H, W


def test_linear_model_closed_form():
    model, par, sigma, mask, fm, H, W = linear_problem()
    psf = asymmetric_psf(3)
    unit = par.copy(); unit[0, 2] = 1.0; unit[0, 4] = 0.0
    U = oracle.render(model, unit, H, W, psf)[0]                  # design column of I0
    w = np.where(mask[0] != 0, 1.0 / sigma[0] ** 2, 0.0)
    a, b, c = (w * U * U).sum(), (w * U).sum(), w.sum()
    det = a * c - b * b
    u = oracle.uncertainty(model, par, sigma, mask, psf, fm)
    assert u["status"][0] == 0
    assert np.isclose(u["sigma_p"][0, 2], np.sqrt(c / det), rtol=1e-10)    # 2x2 inverse by hand
    assert np.isclose(u["sigma_p"][0, 4], np.sqrt(a / det), rtol=1e-10)
    assert np.all(u["sigma_p"][0, [0, 1, 3]] == 0.0)
    # amplitude alone: sigma = 1 / sqrt(sum w U^2)
    u1 = oracle.uncertainty(model, par, sigma, mask, psf, np.array([0, 0, 1, 0, 0], dtype=np.uint8))
    assert np.isclose(u1["sigma_p"][0, 2], 1.0 / np.sqrt(a), rtol=1e-10)


def test_sigma_p_is_the_scatter_of_refits():
    model, par, sigma, mask, fm, H, W = linear_problem()
    psf = asymmetric_psf(3)
    unit = par.copy(); unit[0, 2] = 1.0; unit[0, 4] = 0.0
    U = oracle.render(model, unit, H, W, psf)[0].ravel()
    used = mask[0].ravel() != 0
    sg = sigma[0].ravel()[used]
    X = np.stack([U[used], np.ones(used.sum())], axis=1) / sg[:, None]     # whitened design matrix
    truth = np.array([par[0, 2], par[0, 4]])
    rng = np.random.default_rng(11)
    est = np.empty((4000, 2))
    for t in range(4000):
        y = X @ truth + rng.normal(size=used.sum())
        est[t] = np.linalg.lstsq(X, y, rcond=None)[0]
    u = oracle.uncertainty(model, par, sigma, mask, psf, fm)
    assert np.allclose(est.std(axis=0), u["sigma_p"][0, [2, 4]], rtol=0.05)


def test_uncertainty_of_a_real_problem_against_numpy():
    model = models.bulge_disk()
    par, data, sigma, mask, psf = make_problem(model, 14, 13, 5, 33)
    u = oracle.uncertainty(model, par, sigma, mask, psf)
    assert u["status"][0] == 0
    A = u["jtj"][0]
    D = np.sqrt(np.diag(A))
    ref = np.sqrt(np.diag(np.linalg.inv(A / np.outer(D, D)))) / D
    assert np.allclose(u["sigma_p"][0], ref, rtol=1e-7)
    # halving every sigma halves every uncertainty
    u2 = oracle.uncertainty(model, par, sigma / 2, mask, psf)
    assert np.allclose(u2["sigma_p"], u["sigma_p"] / 2, rtol=1e-9)
