"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py
times (whole batch in one call, persistent fused kernel for <= 128 px, tile kernels
above), against the oracle on every galaxy where it finishes in seconds and on a
sample where it does not.  All data images come from the oracle's render (never
from the CUDA path)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2404_07780_b200 as gm
from gen import configs
from gpu_util import assert_chi2, assert_grad, assert_pixels, dev, oracle_render
import fit_parity as fp

pytestmark = pytest.mark.gpu


def _loss_grad(b):
    chi2, grad = gm.gm_loss_grad(b["model"], dev(b["start"]), dev(b["data"]), dev(b["sigma"]),
                                 dev(b["mask"]), dev(b["psf"]))
    torch.cuda.synchronize()
    return chi2.cpu().numpy(), grad.cpu().numpy()


@pytest.fixture(params=["tensor", "ffma2"])
def engine(request):
    """128 x 128 cutouts run both convolutions on the tensor cores by default (gm_tc_fused.cuh);
    gm_set_option(GM_OPT_TENSOR, 0) keeps them on the FP32 FFMA2 path (k_fused).  Both must meet the
    tolerances."""
    gm.gm_set_option(gm.GM_OPT_TENSOR, 1 if request.param == "tensor" else 0)
    yield request.param
    gm.gm_set_option(gm.GM_OPT_TENSOR, 1)


def test_c1_full_batch_loss_grad_every_galaxy(engine):
    # C1 as bench.py runs it: B = 1024, 128x128, K = 25, one gm_loss_grad call
    b = configs.make_batch(1, range(1024), oracle_render)
    chi2, grad = _loss_grad(b)
    oc, og = oracle.loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    assert_chi2(chi2, oc)
    assert_grad(grad, og)
    img = gm.gm_render(b["model"], dev(b["start"][:64]), 128, 128, dev(b["psf"])).cpu().numpy()
    assert_pixels(img, oracle.render(b["model"], b["start"][:64], 128, 128, b["psf"]))


def test_c1_full_batch_fit_sampled():
    # the whole 1,024-galaxy, 200-iteration fit on the GPU; the oracle refits a sample
    b = configs.make_batch(1, range(1024), oracle_render)
    opts = b["opts"]
    p = dev(b["start"]).clone()
    out = gm.gm_fit(b["model"], p, dev(b["data"]), dev(b["sigma"]), None, dev(b["psf"]), opts)
    torch.cuda.synchronize()
    gp = out["params"].cpu().numpy(); gc = out["chi2"].cpu().numpy()
    assert (out["status"].cpu().numpy() == 0).all() and (out["iters_used"].cpu().numpy() == 200).all()
    sample = np.arange(0, 1024, 43)                                # 24 galaxies across the batch
    o = oracle.fit(b["model"], b["start"][sample], b["data"][sample], b["sigma"][sample], None, b["psf"], opts)
    # chi^2 at the fitted point is well conditioned; parameters of faint galaxies sit in flat
    # valleys (SURVEY 8(d) S/N note): whoever misses 1e-3 must be the same fit by the oracle's
    # chi^2 and model image (tests/fit_parity.py)
    assert_chi2(gc[sample], o["chi2"], rtol=1e-4)
    sub = dict(b, start=b["start"][sample], data=b["data"][sample], sigma=b["sigma"][sample],
               galaxies=[b["galaxies"][i] for i in sample])
    g_s = {"params": gp[sample], "chi2": gc[sample], "status": out["status"].cpu().numpy()[sample],
           "iters_used": out["iters_used"].cpu().numpy()[sample]}
    fp.assert_parity("C1 full batch", fp.judge(sub, g_s, o), floor=0.90)
    # the fit must not depend on the batch a galaxy sits in (galaxies are independent)
    p2 = dev(b["start"][sample]).clone()
    out2 = gm.gm_fit(b["model"], p2, dev(b["data"][sample]), dev(b["sigma"][sample]), None, dev(b["psf"]), opts)
    torch.cuda.synchronize()
    assert np.array_equal(out2["params"].cpu().numpy(), gp[sample])


@pytest.mark.parametrize("side", [64, 96, 128, 192, 256])
def test_c2_buckets_masked(side):
    # C2: every cutout side with the 10 % mask; 192 and 256 px run the multi-tile kernels
    gal = range(400)
    b = configs.make_batch(2, gal, oracle_render, side=side)
    assert b["mask"] is not None and 40 <= len(b["galaxies"]) <= 130
    chi2, grad = _loss_grad(b)
    oc, og = oracle.loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    assert_chi2(chi2, oc)
    assert_grad(grad, og)


def test_c3_bulge_disk_full_batch(engine):
    # C3: B = 4096, P = 11; data for all galaxies from the oracle, gradient checked on a sample
    b = configs.make_batch(3, range(4096), oracle_render)
    chi2, grad = _loss_grad(b)
    sample = np.arange(0, 4096, 16)
    oc, og = oracle.loss_grad(b["model"], b["start"][sample], b["data"][sample], b["sigma"][sample], None, b["psf"])
    assert_chi2(chi2[sample], oc)
    assert_grad(grad[sample], og)
    assert np.isfinite(chi2).all() and np.isfinite(grad).all()


def test_c4_shapes_replicated_sample():
    # C4's shapes (256x256, K = 41, Sersic + Ferrer + Moffat, P = 16).  The oracle cannot
    # render 65,536 such cutouts, so 8 distinct galaxies are replicated to a 296-galaxy batch
    # (two per SM): every replica must equal the oracle AND its siblings bit for bit.
    b = configs.make_batch(4, range(8), oracle_render)
    rep = 37
    tile = lambda a: None if a is None else np.ascontiguousarray(np.concatenate([a] * rep))
    bb = dict(b, start=tile(b["start"]), data=tile(b["data"]), sigma=tile(b["sigma"]), mask=tile(b["mask"]))
    chi2, grad = _loss_grad(bb)
    oc, og = oracle.loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    assert_chi2(chi2[:8], oc)
    assert_grad(grad[:8], og)
    assert np.array_equal(chi2.reshape(rep, 8), np.broadcast_to(chi2[:8], (rep, 8)))
    assert np.array_equal(grad.reshape(rep, 8, -1), np.broadcast_to(grad[:8], (rep, 8, grad.shape[1])))
    img = gm.gm_render(b["model"], dev(b["start"]), 256, 256, dev(b["psf"])).cpu().numpy()
    assert_pixels(img, oracle.render(b["model"], b["start"], 256, 256, b["psf"]))
