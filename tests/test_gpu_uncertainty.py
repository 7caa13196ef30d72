"""-m gpu: the covariance row (Sec. 5.2) through the C ABI against
the fp64 oracle: J^T W J and J^T W (D-M) from gm_loss_grad, sigma_p from gm_uncertainty.

Tolerances: J^T W J element (k,l) within 1e-4 of
sqrt(jtj_kk jtj_ll) (the scale of that element); J^T W r like the gradient (1e-3 of its
norm); sigma_p within 1e-2 relative: the relative error of the fp32 Jacobian columns
(~1e-6, partly systematic) is amplified by the condition number of the correlation
matrix, which reaches ~1e3 for the Sersic (Ie, re, n) triple."""
import numpy as np
import pytest
import torch

import oracle
import paper_2404_07780_b200 as gm
from gen import configs, models
from gpu_util import assert_grad, dev, oracle_render
from test_gpu_parity import synth

pytestmark = pytest.mark.gpu

JTJ_RTOL = 1e-4
SIGMA_P_RTOL = 1e-2


def assert_jtj(gpu, orc):
    gpu = np.asarray(gpu, dtype=np.float64)
    d = np.sqrt(np.einsum("bkk->bk", orc))
    scale = d[:, :, None] * d[:, None, :]
    err = np.abs(gpu - orc) / np.maximum(scale, 1e-300)
    assert np.all(err <= JTJ_RTOL), f"jtj worst {err.max():.3e} at {np.unravel_index(err.argmax(), err.shape)}"
    assert np.array_equal(gpu, np.swapaxes(gpu, 1, 2))              # exactly symmetric


def run_unc(model, par, sigma, mask, psf, fm=None):
    out = gm.gm_uncertainty(model, dev(par), dev(sigma), dev(mask), dev(psf), free_mask=fm, want_jtj=True)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items() if not k.startswith("_")}


@pytest.mark.parametrize("H,W,K,per_psf", [(40, 48, 9, False), (37, 45, 7, True), (150, 140, 25, False)])
def test_jtj_jtr_bulge_disk(H, W, K, per_psf):
    model = models.bulge_disk()
    par, data, sigma, mask, psf = synth(model, 3, H, W, K, seed=H + K, per_galaxy_psf=per_psf)
    chi2, grad, jtj, jtr = gm.gm_loss_grad(model, dev(par), dev(data), dev(sigma), dev(mask), dev(psf),
                                           want_jtj=True)
    torch.cuda.synchronize()
    oc, og, oj, ojr = oracle.loss_grad(model, par, data, sigma, mask, psf, want_jtj=True)
    assert_jtj(jtj.cpu().numpy(), oj)
    assert_grad(jtr.cpu().numpy(), ojr)
    assert torch.equal(jtr, -0.5 * grad)


def test_every_profile_tied_unconvolved_sky():
    model = models.all_profiles()                                   # P = 30: 465 pairs
    par, data, sigma, mask, psf = synth(model, 2, 36, 34, 7, seed=9)
    u = run_unc(model, par, sigma, mask, psf)
    o = oracle.uncertainty(model, par, sigma, mask, psf)
    assert_jtj(u["jtj"], o["jtj"])


def test_sigma_p_c0_and_free_mask():
    b = configs.make_batch(0, range(16), oracle_render)
    model = b["model"]
    u = run_unc(model, b["truth"], b["sigma"], b["mask"], b["psf"])
    o = oracle.uncertainty(model, b["truth"], b["sigma"], b["mask"], b["psf"])
    assert (u["status"] == 0).all() and (o["status"] == 0).all()
    assert_jtj(u["jtj"], o["jtj"])
    assert np.allclose(u["sigma_p"], o["sigma_p"], rtol=SIGMA_P_RTOL)
    fm = np.array([1, 1, 1, 1, 0, 1, 1], dtype=np.uint8)            # Sersic n held fixed
    uf = run_unc(model, b["truth"], b["sigma"], b["mask"], b["psf"], fm)
    of = oracle.uncertainty(model, b["truth"], b["sigma"], b["mask"], b["psf"], fm)
    assert np.all(uf["sigma_p"][:, 4] == 0.0)
    assert np.allclose(uf["sigma_p"], of["sigma_p"], rtol=SIGMA_P_RTOL)
    assert np.all(uf["sigma_p"] <= u["sigma_p"] * (1 + 1e-5))


def test_sigma_p_c1_shapes_sampled():
    # C1's shapes (128x128, K = 25, CCD noise model) on 96 galaxies, several chunks of the tile kernels
    b = configs.make_batch(1, range(96), oracle_render)
    u = run_unc(b["model"], b["truth"], b["sigma"], b["mask"], b["psf"])
    o = oracle.uncertainty(b["model"], b["truth"], b["sigma"], b["mask"], b["psf"])
    assert_jtj(u["jtj"], o["jtj"])
    ok = (u["status"] == 0) & (o["status"] == 0)
    assert ok.mean() > 0.95
    rel = np.abs(u["sigma_p"][ok] - o["sigma_p"][ok]) / o["sigma_p"][ok]
    assert np.all(rel <= SIGMA_P_RTOL), f"worst sigma_p rel err {rel.max():.3e}"


def test_round_galaxy_is_flagged_not_garbage():
    # q = 1: the theta column of J is exactly zero in fp32 -> status 1 and NaN, never a number
    model = models.single_sersic()
    par = np.array([[8.2, 7.9, 1.0, 3.0, 1.5, 1.0, 0.4], [8.2, 7.9, 1.0, 3.0, 1.5, 0.7, 0.4]], dtype=np.float32)
    sig = np.full((2, 16, 16), 0.1, dtype=np.float32)
    psf = np.zeros((5, 5), dtype=np.float32); psf[2, 2] = 1.0
    u = run_unc(model, par, sig, None, psf)
    assert u["status"][0] == 1 and np.isnan(u["sigma_p"][0]).all()
    assert u["status"][1] == 0 and np.isfinite(u["sigma_p"][1]).all()


def test_workspace_too_small_is_refused():
    model = models.single_sersic()
    b = configs.make_batch(0, range(2), oracle_render)
    small = torch.empty(gm.gm_workspace_bytes(model, 2, 64, 64, 15) + 256, dtype=torch.uint8, device="cuda")
    with pytest.raises(gm.GmError) as e:
        gm.gm_uncertainty(model, dev(b["truth"]), dev(b["sigma"]), None, dev(b["psf"]), workspace=small)
    assert e.value.status == -4
