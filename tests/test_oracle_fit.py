"""Pins for the oracle's update rule and fit loop (readings O1-O5; not gpu).

The optimiser CHOICE is parity-unpinned against the real galmoss package (the
paper does not name it); the update RULE is pinned here against torch.optim.Adam,
a hand-typed trace, and behaviour on problems with known minimisers.
"""
import math

import numpy as np
import pytest
import torch

import oracle
from gen import configs, models
from gen.psf import gaussian_psf

INF = np.inf


def test_adam_step_matches_torch_optim_adam():
    rng = np.random.default_rng(0)
    P = 6
    u0 = rng.normal(size=P)
    grads = rng.normal(size=(25, P)) * np.array([1e-3, 1.0, 30.0, 1e3, 0.2, 5.0])
    lr = 0.01
    tp = torch.tensor(u0.copy(), dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([tp], lr=lr, betas=(0.9, 0.999), eps=1e-8)
    u = u0.copy(); m = np.zeros(P); s = np.zeros(P)
    lo = np.full(P, -INF); hi = np.full(P, INF)
    for t, g in enumerate(grads, start=1):
        tp.grad = torch.tensor(g.copy())
        opt.step()
        oracle.adam_step(u, g, m, s, t, np.full(P, lr), 1.0, 0.9, 0.999, 1e-8, lo, hi)
        assert np.allclose(u, tp.detach().numpy(), rtol=1e-12, atol=1e-15)


def test_adam_hand_trace_first_steps():
    # one variable, g = 2 each step, lr = 0.1, decay 0.5: typed out from the definition
    u = np.array([1.0]); m = np.zeros(1); s = np.zeros(1)
    b1, b2, eps = 0.9, 0.999, 1e-8
    lo = np.array([-INF]); hi = np.array([INF])
    oracle.adam_step(u, np.array([2.0]), m, s, 1, np.array([0.1]), 0.5, b1, b2, eps, lo, hi)
    # m=0.2, s=0.004; mhat=2, shat=4 -> step = 0.1 * 2 / (2 + 1e-8)
    assert m[0] == pytest.approx(0.2) and s[0] == pytest.approx(0.004)
    assert u[0] == pytest.approx(1.0 - 0.1 * 2 / (2 + 1e-8), rel=1e-15)
    u1 = u[0]
    oracle.adam_step(u, np.array([2.0]), m, s, 2, np.array([0.1]), 0.5, b1, b2, eps, lo, hi)
    m2 = 0.9 * 0.2 + 0.1 * 2; s2 = 0.999 * 0.004 + 0.001 * 4
    step = 0.1 * 0.5 * (m2 / (1 - 0.81)) / (math.sqrt(s2 / (1 - 0.999 ** 2)) + eps)
    assert u[0] == pytest.approx(u1 - step, rel=1e-14)
    # first step is -lr * sign(g) whatever the gradient scale
    for g in (1e-6, 3.0, -1e5):
        u = np.array([0.0]); m = np.zeros(1); s = np.zeros(1)
        oracle.adam_step(u, np.array([g]), m, s, 1, np.array([0.1]), 1.0, b1, b2, 1e-12, lo, hi)
        assert u[0] == pytest.approx(-0.1 * np.sign(g), rel=1e-5)


def test_adam_projection_and_fixed_parameters_O3():
    u = np.array([0.95, 5.0, 1.0]); m = np.zeros(3); s = np.zeros(3)
    lo = np.array([0.0, 0.0, 0.0]); hi = np.array([1.0, 2.0, 10.0])
    oracle.adam_step(u, np.array([-1.0, 1.0, 1.0]), m, s, 1, np.full(3, 0.1), 1.0, 0.9, 0.999, 1e-8,
                     lo, hi, free_mask=np.array([1, 1, 0]))
    assert u[0] == 1.0            # stepped to 1.05, clamped to hi
    assert u[1] == 2.0            # started outside the range: pulled to the edge in one step
    assert u[2] == 1.0 and m[2] == 0.0 and s[2] == 0.0   # held fixed, moments untouched


def _noiseless(model, truth, H, W, psf):
    M = oracle.render(model, truth, H, W, psf)
    sigma = np.full_like(M, 0.01)
    return M, sigma


def test_fit_recovers_truth_on_noiseless_data():
    model = models.single_sersic()
    H = W = 24
    psf = gaussian_psf(7, 2.0)
    truth = np.array([[12.3, 11.6, 1.0, 4.0, 1.5, 0.6, 0.8]])
    data, sigma = _noiseless(model, truth, H, W, psf)
    start = truth * np.array([[1.02, 0.98, 1.15, 0.88, 1.12, 1.1, 1.1]])
    opts = configs.fit_options(model, H, W, 1500)   # Adam is slow along the Ie-re-n valley
    out = oracle.fit(model, start, data, sigma, None, psf, opts, want_trace=True)
    c0, _ = oracle.loss_grad(model, start, data, sigma, None, psf)
    assert out["trace"][0, 0] == pytest.approx(c0[0], rel=1e-14)
    assert out["chi2"][0] < 1e-6 * c0[0]
    assert np.allclose(out["params"], truth, rtol=2e-3)
    assert out["status"][0] == 0 and out["iters_used"][0] == 1500
    # chi2_out is chi^2 AT the returned parameters
    c1, _ = oracle.loss_grad(model, out["params"], data, sigma, None, psf)
    assert out["chi2"][0] == pytest.approx(c1[0], rel=1e-12)


def test_fit_log10_space_chain_rule_O4():
    # one log-space step equals an Adam step driven by g_u = g_p * p * ln 10
    model = models.single_sersic()
    H = W = 16
    psf = gaussian_psf(5, 2.0)
    truth = np.array([[8.2, 7.9, 1.0, 3.0, 1.2, 0.7, 0.4]])
    data, sigma = _noiseless(model, truth, H, W, psf)
    start = truth * 1.1
    opts = configs.fit_options(model, H, W, 1)
    out = oracle.fit(model, start, data, sigma, None, psf, opts)
    _, g = oracle.loss_grad(model, start, data, sigma, None, psf)
    lg = opts["log10_space"].astype(bool)
    u = np.where(lg, np.log10(start[0]), start[0])
    gu = np.where(lg, g[0] * start[0] * math.log(10.0), g[0])
    m = np.zeros(7); s = np.zeros(7)
    lo64 = opts["lo"].astype(np.float64)
    lo = np.where(lg, np.log10(np.maximum(lo64, 1e-300)), lo64)
    hi = np.where(lg, np.log10(opts["hi"]), opts["hi"]).astype(np.float64)
    oracle.adam_step(u, gu, m, s, 1, opts["lr"], opts["lr_decay"], 0.9, 0.999, 1e-8, lo, hi)
    expect = np.where(lg, 10.0 ** u, u)
    assert np.allclose(out["params"][0], expect, rtol=1e-13)
    # finite-difference check of the chain factor in u
    k = 3
    h = 1e-6
    pp, pm = start.copy(), start.copy()
    pp[0, k] = 10 ** (math.log10(start[0, k]) + h); pm[0, k] = 10 ** (math.log10(start[0, k]) - h)
    cp, _ = oracle.loss_grad(model, pp, data, sigma, None, psf)
    cm, _ = oracle.loss_grad(model, pm, data, sigma, None, psf)
    assert gu[k] == pytest.approx((cp[0] - cm[0]) / (2 * h), rel=1e-6)


def test_fit_early_stop_and_fixed_parameter_O5():
    model = models.single_sersic()
    H = W = 20
    psf = gaussian_psf(5, 2.0)
    rng = np.random.default_rng(5)
    truth = np.array([[10.2, 9.7, 1.0, 3.5, 1.0, 0.7, 0.6]])
    M = oracle.render(model, truth, H, W, psf)
    sigma = np.full_like(M, 0.02)
    data = M + 0.02 * rng.normal(size=M.shape)
    start = truth * 1.05
    opts = configs.fit_options(model, H, W, 400, tol=1e-5, patience=5)
    opts["free_mask"] = np.array([1, 1, 1, 1, 0, 1, 1], dtype=np.uint8)   # n held fixed
    out = oracle.fit(model, start, data, sigma, None, psf, opts, want_trace=True)
    assert out["status"][0] == 1 and 5 < out["iters_used"][0] < 400
    assert out["params"][0, 4] == start[0, 4]                            # bit-identical
    t = out["iters_used"][0]
    assert np.isnan(out["trace"][0, t + 1:]).all() and np.isfinite(out["trace"][0, :t + 1]).all()
    assert out["chi2"][0] == out["trace"][0, t]


def test_fit_nonfinite_status():
    model = models.single_sersic()
    H = W = 12
    psf = gaussian_psf(3, 1.5)
    truth = np.array([[6.2, 5.7, 1.0, 2.5, 1.0, 0.7, 0.6]])
    data, sigma = _noiseless(model, truth, H, W, psf)
    data = data.copy(); data[0, 3, 3] = np.nan
    opts = configs.fit_options(model, H, W, 10)
    out = oracle.fit(model, truth * 1.05, data, sigma, None, psf, opts)
    assert out["status"][0] == 2 and out["iters_used"][0] == 0
    assert np.array_equal(out["params"], truth * 1.05) and not np.isfinite(out["chi2"][0])


def test_chi2_per_pixel_near_one_at_truth_X2():
    # at the truth with Gaussian noise chi2/N ~ 1 +- sqrt(2/N)
    def render(model, p, H, W, psf):
        return oracle.render(model, p, H, W, psf)
    b = configs.make_batch(0, range(4), render)
    chi2, _ = oracle.loss_grad(b["model"], b["truth"], b["data"], b["sigma"], b["mask"], b["psf"])
    N = b["H"] * b["W"]
    assert np.all(np.abs(chi2 / N - 1.0) < 6 * math.sqrt(2.0 / N))
