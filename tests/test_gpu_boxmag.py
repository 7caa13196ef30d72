"""-m gpu: boxiness (Eq. 2 with B != 0) and the magnitude parameterisation
(Eq. 5, 6, 8, 10, 15) in the CUDA path, against the fp64
oracle on the same seeded inputs.  Same tolerances as the other parity
tests (gpu_util.py)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2404_07780_b200 as gm
from gen import configs, models
from gpu_util import PAR_RTOL, assert_chi2, assert_grad, assert_pixels, dev
from test_gpu_parity import run_loss_grad, synth
from test_gpu_uncertainty import SIGMA_P_RTOL, assert_jtj, run_unc

pytestmark = pytest.mark.gpu


def check(model, B, H, W, K, seed, per_psf=False):
    par, data, sigma, mask, psf = synth(model, B, H, W, K, seed=seed, per_galaxy_psf=per_psf)
    img = gm.gm_render(model, dev(par), H, W, dev(psf))
    assert_pixels(img.cpu().numpy(), oracle.render(model, par, H, W, psf))
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert_chi2(chi2, oc)
    assert_grad(grad, og)
    scale = np.linalg.norm(og, axis=1, keepdims=True)          # parameter by parameter too
    assert np.all(np.abs(grad - og) <= 1e-3 * scale)
    return grad, og


@pytest.mark.parametrize("kind", ["sersic", "expdisk", "ferrer", "king", "gaussian", "moffat"])
@pytest.mark.parametrize("convolve", [1, 0])
def test_boxiness_each_profile(kind, convolve):
    model = models.one_component(kind, convolve, box=True)
    grad, og = check(model, 4, 33, 30, 9, seed=len(kind) * 3 + convolve)
    k = model["names"].index("box")
    assert np.all(np.abs(og[:, k]) > 0)                         # dchi2/dB really is exercised


@pytest.mark.parametrize("kind", ["sersic", "expdisk", "ferrer", "moffat"])
@pytest.mark.parametrize("convolve,box", [(1, True), (0, True), (1, False)])
def test_magnitudes_each_profile(kind, convolve, box):
    model = models.one_component(kind, convolve, box=box, mag=True)
    grad, og = check(model, 4, 33, 30, 9, seed=len(kind) * 5 + convolve + 2 * box)
    km, k0 = model["names"].index("mag"), model["names"].index("m0")
    assert np.allclose(grad[:, k0], -grad[:, km], rtol=1e-5)    # only m - m0 enters


@pytest.mark.parametrize("H,W,K,per_psf", [(40, 48, 9, False), (128, 128, 25, False), (150, 140, 25, True),
                                           (96, 200, 15, False)])
def test_boxy_bulge_disk_in_magnitudes_fused_and_tiled(H, W, K, per_psf):
    # <= 128 px: the fused kernel; larger: forward / backward tile kernels
    check(models.boxy_bulge_disk_mag(), 3, H, W, K, seed=H + W + K, per_psf=per_psf)


def test_box_zero_equals_plain_ellipse():
    plain, boxy = models.one_component("sersic"), models.one_component("sersic", box=True)
    par = np.array([[20.3, 18.1, 0.7, 0.6, 1.3, 4.0, 2.5]], dtype=np.float32)
    parb = np.concatenate([par, np.zeros((1, 1), np.float32)], axis=1)
    psf = np.ones((1, 1), dtype=np.float32)
    a = gm.gm_render(plain, dev(par), 40, 40, dev(psf)).cpu().numpy()
    b = gm.gm_render(boxy, dev(parb), 40, 40, dev(psf)).cpu().numpy()
    assert np.allclose(a, b, rtol=2e-5, atol=0)      # pow through lg2/ex2 vs sqrt: a few fp32 ulps times nu*t/n


def test_uncertainty_with_boxiness_and_magnitudes():
    model = models.boxy_bulge_disk_mag()
    par, data, sigma, mask, psf = synth(model, 3, 44, 40, 9, seed=12)
    fm = np.array([r != "zeropoint" for r in model["roles"]], dtype=np.uint8)
    u = run_unc(model, par, sigma, mask, psf, fm)
    o = oracle.uncertainty(model, par, sigma, mask, psf, fm)
    assert_jtj(u["jtj"], o["jtj"])
    ok = (u["status"] == 0) & (o["status"] == 0)
    assert ok.all()
    assert np.allclose(u["sigma_p"], o["sigma_p"], rtol=SIGMA_P_RTOL)
    assert np.all(u["sigma_p"][:, model["names"].index("m0")] == 0.0)


def test_fit_in_magnitudes_with_boxiness():
    model = models.one_component("sersic", box=True, mag=True)
    H = W = 48
    rng = np.random.default_rng(8)
    B = 6
    truth = np.stack([[W / 2 + rng.uniform(-1, 1), H / 2 + rng.uniform(-1, 1), rng.uniform(0.2, 2.8),
                       rng.uniform(0.4, 0.9), rng.uniform(15.5, 16.5), rng.uniform(3, 6), rng.uniform(0.8, 3.0),
                       rng.uniform(-0.3, 0.5), 22.5] for _ in range(B)]).astype(np.float32)
    psf = configs.make_batch(0, range(1), lambda m, p, h, w, f: oracle.render(m, p, h, w, f))["psf"]
    M = oracle.render(model, truth, H, W, psf)
    sigma = np.full(M.shape, 0.02 * M.max(), dtype=np.float32)
    data = (M + sigma * rng.normal(size=M.shape)).astype(np.float32)
    start = truth.copy()
    start[:, 4] += rng.uniform(-0.2, 0.2, B); start[:, 5] *= rng.uniform(0.9, 1.1, B)
    start[:, 6] *= rng.uniform(0.9, 1.1, B); start[:, 7] += rng.uniform(-0.1, 0.1, B)
    opts = configs.fit_options(model, H, W, 60)
    assert opts["free_mask"][-1] == 0                           # the zero point is held fixed
    out = gm.gm_fit(model, dev(start), dev(data), dev(sigma), None, dev(psf), opts)
    torch.cuda.synchronize()
    of = oracle.fit(model, start, data, sigma, None, psf, opts)
    p_gpu = out["params"].cpu().numpy().astype(np.float64)
    assert np.array_equal(p_gpu[:, -1], start[:, -1])           # untouched
    assert_chi2(out["chi2"].cpu().numpy(), of["chi2"], rtol=1e-4)
    names = model["names"]
    for k, nm in enumerate(names):
        if nm == "theta":
            d = np.abs((p_gpu[:, k] - of["params"][:, k] + np.pi / 2) % np.pi - np.pi / 2)
            assert np.all(d <= 2e-3), nm
        elif nm == "box":
            assert np.all(np.abs(p_gpu[:, k] - of["params"][:, k]) <= 2e-3), nm     # B crosses 0: absolute
        else:
            assert np.allclose(p_gpu[:, k], of["params"][:, k], rtol=PAR_RTOL, atol=1e-5), nm
    # the fit moved towards the truth
    assert np.abs(of["params"][:, 4] - truth[:, 4]).mean() < np.abs(start[:, 4] - truth[:, 4]).mean()


def test_magnitude_on_a_profile_without_relation_is_einval():
    model = models.one_component("king", mag=True)
    par = np.zeros((1, model["n_par"]), dtype=np.float32)
    with pytest.raises(gm.GmError) as e:
        gm.gm_render(model, dev(par), 16, 16, dev(np.ones((1, 1), np.float32)))
    assert e.value.status == -1
