"""-m gpu: the CUDA path (through the C ABI) against the fp64 oracle, element by
element, on the same seeded inputs.  Shapes span several tiles and ragged tails."""
import math

import numpy as np
import pytest
import torch

import oracle
import paper_2404_07780_b200 as gm
from gen import configs, models
from gen.psf import asymmetric_psf, gaussian_psf, moffat_psf
from gpu_util import (assert_chi2, assert_grad, assert_pixels, dev, oracle_render)
from test_oracle_lossgrad import sample_params

pytestmark = pytest.mark.gpu


def synth(model, B, H, W, K, seed, masked=True, per_galaxy_psf=False):
    rng = np.random.default_rng(seed)
    truth = np.stack([sample_params(model, H, W, rng) for _ in range(B)]).astype(np.float32)
    if per_galaxy_psf:
        psf = np.stack([asymmetric_psf(K, seed=100 + g) for g in range(B)]).astype(np.float32)
    else:
        psf = asymmetric_psf(K).astype(np.float32)
    M = oracle.render(model, truth, H, W, psf)
    sigma = (0.05 + 0.1 * rng.random((B, H, W))).astype(np.float32)
    data = (M + sigma * rng.normal(size=M.shape)).astype(np.float32)
    mask = (rng.random((B, H, W)) > 0.15).astype(np.uint8) if masked else None
    par = (truth * (1 + 0.05 * rng.uniform(-1, 1, size=truth.shape))).astype(np.float32)
    return par, data, sigma, mask, psf


def render_and_engine(model, par, H, W, psf):
    """gm_render with the launch-timing hook on -> (image, families of heavy kernels that ran: 'tensor' / 'ffma2')."""
    gm.gm_profile_enable(1)
    try:
        img = gm.gm_render(model, dev(par), H, W, dev(psf))
        torch.cuda.synchronize()
        kinds = gm.gm_profile_read()
    finally:
        gm.gm_profile_enable(0)
    return img, {"tensor" if name.startswith("tc_") else "ffma2" for name, (_, n) in kinds.items() if n > 0}


def run_loss_grad(model, par, data, sigma, mask, psf):
    chi2, grad = gm.gm_loss_grad(model, dev(par), dev(data), dev(sigma), dev(mask), dev(psf))
    torch.cuda.synchronize()
    return chi2.cpu().numpy(), grad.cpu().numpy()


# ---- config C0 exactly as BASELINE.json states it -------------------------------
def test_c0_render_chi2_gradient():
    b = configs.make_batch(0, range(16), oracle_render)
    model = b["model"]
    img = gm.gm_render(model, dev(b["start"]), b["H"], b["W"], dev(b["psf"]))
    assert_pixels(img.cpu().numpy(), oracle.render(model, b["start"], b["H"], b["W"], b["psf"]))
    chi2, grad = run_loss_grad(model, b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    oc, og = oracle.loss_grad(model, b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    assert_chi2(chi2, oc)
    assert_grad(grad, og)


# ---- every profile, tied parameters, unconvolved point source, sky -------------------
@pytest.mark.parametrize("H,W,K,per_psf", [(40, 48, 9, False), (37, 45, 7, True), (21, 19, 5, False)])
def test_all_profiles_render_and_gradient(H, W, K, per_psf):
    model = models.all_profiles()
    par, data, sigma, mask, psf = synth(model, 3, H, W, K, seed=H * W + K, per_galaxy_psf=per_psf)
    img = gm.gm_render(model, dev(par), H, W, dev(psf))
    assert_pixels(img.cpu().numpy(), oracle.render(model, par, H, W, psf))
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert_chi2(chi2, oc)
    assert_grad(grad, og)
    # parameter by parameter too: each within 1e-3 of the gradient norm
    scale = np.linalg.norm(og, axis=1, keepdims=True)
    assert np.all(np.abs(grad - og) <= 1e-3 * scale)


@pytest.mark.parametrize("kind", ["sersic", "expdisk", "ferrer", "king", "gaussian", "moffat"])
@pytest.mark.parametrize("convolve", [1, 0])
def test_each_profile_alone(kind, convolve):
    model = models.one_component(kind, convolve)
    H, W, K = 33, 30, 9
    par, data, sigma, mask, psf = synth(model, 4, H, W, K, seed=len(kind) * 7 + convolve)
    img = gm.gm_render(model, dev(par), H, W, dev(psf))
    assert_pixels(img.cpu().numpy(), oracle.render(model, par, H, W, psf))
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert_chi2(chi2, oc)
    assert_grad(grad, og)


# ---- several tiles per cutout, ragged tails, every compiled PSF side ------------------
@pytest.mark.parametrize("H,W,K", [(150, 140, 25), (131, 70, 15), (64, 200, 21), (96, 96, 25),
                                   (50, 50, 41), (40, 40, 33), (9, 300, 5), (5, 7, 3), (1, 1, 1),
                                   (130, 129, 11),
                                   # 6 x 12 thread tiles (96 x 192 / 192 x 96 CTA tiles), full and ragged
                                   (192, 192, 25), (180, 96, 9), (96, 190, 15), (200, 380, 5)])
def test_multi_tile_and_ragged(H, W, K):
    model = models.bulge_disk()
    par, data, sigma, mask, psf = synth(model, 2, H, W, K, seed=H + W + K)
    img = gm.gm_render(model, dev(par), H, W, dev(psf))
    assert_pixels(img.cpu().numpy(), oracle.render(model, par, H, W, psf))
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, mask, psf)
    # a handful of pixels gives no averaging: chi^2 inherits 2 eps_pixel M / rho of a
    # single fp32 pixel, so degenerate cutouts get 1e-4
    assert_chi2(chi2, oc, rtol=1e-5 if H * W >= 64 else 1e-4)
    assert_grad(grad, og)


# ---- tensor-core super-tile kernels: several super-tiles per cutout, ragged in both directions, both shapes ----
@pytest.mark.parametrize("H,W,K,per_psf", [(200, 264, 25, False),      # 2 x 3 super-tiles of 128 x 128, ragged
                                           (132, 520, 41, False),      # 64 x 256 super-tiles (3 x 3), ragged
                                           (260, 132, 25, True),       # one PSF per galaxy
                                           (129, 128, 41, False),      # one row beyond a single pass
                                           (100, 100, 25, False),      # one ragged super-tile: shapes up to 128 px that
                                           (128, 96, 15, True),        # are not 64 / 96 / 128 squares
                                           (72, 256, 15, False)])
def test_tensor_super_tiles_ragged(H, W, K, per_psf):
    model = models.bulge_disk()
    B = 3                                                    # fewer items than CTAs, more than one per galaxy
    par, data, sigma, mask, psf = synth(model, B, H, W, K, seed=3 * H + W + K, per_galaxy_psf=per_psf)
    assert gm.gm_get_option(gm.GM_OPT_TENSOR) == 1
    img, fam = render_and_engine(model, par, H, W, psf)
    assert fam == {"tensor"}                                 # this call did take the tensor-core path
    assert_pixels(img.cpu().numpy(), oracle.render(model, par, H, W, psf))
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert_chi2(chi2, oc)
    assert_grad(grad, og)
    # the FFMA2 engine on the same inputs: other kernels, same answers
    gm.gm_set_option(gm.GM_OPT_TENSOR, 0)
    try:
        img2, fam2 = render_and_engine(model, par, H, W, psf)
    finally:
        gm.gm_set_option(gm.GM_OPT_TENSOR, 1)
    assert fam2 == {"ffma2"}
    assert_pixels(img2.cpu().numpy(), oracle.render(model, par, H, W, psf))


# ---- tensor-core kernels with components that do not go through the PSF (point source, sky; R:C3) ----
@pytest.mark.parametrize("H,W,K,per_psf", [(128, 128, 11, False), (96, 96, 15, True), (64, 64, 25, False),
                                           (200, 264, 17, False), (132, 520, 25, True)])
def test_tensor_engine_with_unconvolved_components(H, W, K, per_psf):
    model = models.all_profiles()                            # six laws, tied parameters, an unconvolved source, the sky
    assert any(c["convolve"] == 0 for c in model["components"])
    par, data, sigma, mask, psf = synth(model, 3, H, W, K, seed=7 * H + W + K, per_galaxy_psf=per_psf)
    img, fam = render_and_engine(model, par, H, W, psf)
    assert fam == {"tensor"}
    assert_pixels(img.cpu().numpy(), oracle.render(model, par, H, W, psf))
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, mask, psf)
    assert_chi2(chi2, oc)
    assert_grad(grad, og)
    gm.gm_set_option(gm.GM_OPT_TENSOR, 0)                    # the FFMA2 engine runs other kernels
    try:
        _, fam2 = render_and_engine(model, par, H, W, psf)
    finally:
        gm.gm_set_option(gm.GM_OPT_TENSOR, 1)
    assert fam2 == {"ffma2"}


def test_psf_orientation_not_flipped_or_transposed():
    # a delta PSF off centre must shift the model the way the oracle does
    model = models.single_sersic()
    H = W = 24
    par = np.array([[12.3, 11.6, 1.0, 3.0, 1.5, 0.6, 0.8]], dtype=np.float32)
    psf = np.zeros((5, 5), dtype=np.float32); psf[1, 4] = 1.0
    img = gm.gm_render(model, dev(par), H, W, dev(psf)).cpu().numpy()
    assert_pixels(img, oracle.render(model, par, H, W, psf))


@pytest.mark.parametrize("side,cid", [(64, 0), (128, 1)])
def test_shared_and_per_galaxy_psf_agree_bitwise(side, cid):
    # one PSF for the batch or the same PSF replicated per galaxy (reading C4): identical pixels wherever both run
    # the same engine -- always on the FFMA2 path, and on the tensor-core path where it takes per-galaxy PSFs
    # (128 px; four 64 px cutouts share the lanes of a pass and so one PSF, which sends them to the FFMA2 path)
    b = configs.make_batch(cid, range(4), oracle_render)
    model, K = b["model"], b["psf"].shape[0]
    rep = np.ascontiguousarray(np.broadcast_to(b["psf"], (4, K, K)))
    ref = oracle.render(model, b["start"], side, side, b["psf"])
    for tensor in (1, 0):
        gm.gm_set_option(gm.GM_OPT_TENSOR, tensor)
        try:
            a = gm.gm_render(model, dev(b["start"]), side, side, dev(b["psf"]))
            c = gm.gm_render(model, dev(b["start"]), side, side, dev(rep))
        finally:
            gm.gm_set_option(gm.GM_OPT_TENSOR, 1)
        if tensor == 0 or side == 128:
            assert torch.equal(a, c)
        assert_pixels(a.cpu().numpy(), ref)
        assert_pixels(c.cpu().numpy(), ref)


@pytest.mark.parametrize("H,W,K", [(64, 64, 25), (96, 96, 9), (128, 128, 41), (100, 90, 33), (192, 192, 25),
                                   (256, 256, 41), (140, 200, 15), (37, 45, 7)])
def test_constant_bank_and_shared_memory_taps_agree_bitwise(H, W, K, request):
    # a batch-wide PSF runs the convolution with its taps in the constant bank (FFMA2 with a
    # uniform-register operand), a per-galaxy PSF or gm_set_option(GM_OPT_CONST_TAPS, 0) in shared
    # memory; both add the K^2 products of a pixel in the same order, in k_fused and in the
    # tile kernels, for every compiled PSF side and both thread tiles
    model = models.bulge_disk()
    par, data, sigma, mask, psf = synth(model, 3, H, W, K, seed=7 * H + W + K)
    gm.gm_set_option(gm.GM_OPT_TENSOR, 0)                    # this test is about the FFMA2 engine's two tap homes
    request.addfinalizer(lambda: gm.gm_set_option(gm.GM_OPT_TENSOR, 1))
    def run():
        img = gm.gm_render(model, dev(par), H, W, dev(psf))
        out = gm.gm_loss_grad(model, dev(par), dev(data), dev(sigma), dev(mask), dev(psf))
        torch.cuda.synchronize()
        return [img] + [t for t in out]
    const = run()
    gm.gm_set_option(gm.GM_OPT_CONST_TAPS, 0)
    try:
        shared = run()
    finally:
        gm.gm_set_option(gm.GM_OPT_CONST_TAPS, 1)
    rep = np.ascontiguousarray(np.broadcast_to(psf, (3, K, K)))
    per = [gm.gm_render(model, dev(par), H, W, dev(rep))] + \
        [t for t in gm.gm_loss_grad(model, dev(par), dev(data), dev(sigma), dev(mask), dev(rep))]
    # the pixels must not move at all; where the taps live may change the kernel that runs
    # (k_fused slot geometry, tile kernels) and with it the ORDER of the chi^2 / gradient
    # reductions, so those agree to rounding only
    for other in (shared, per):
        assert torch.equal(const[0], other[0])
        assert_chi2(other[1].cpu().numpy(), const[1].cpu().numpy().astype(np.float64), rtol=2e-6)
        assert_grad(other[2].cpu().numpy(), const[2].cpu().numpy().astype(np.float64), rtol=1e-5)
    assert_chi2(const[1].cpu().numpy(), oracle.loss_grad(model, par, data, sigma, mask, psf)[0])


def test_constant_tap_regions_are_refilled_between_and_across_calls(request):
    # a pool region is reused by the next call with another PSF, and concurrent calls on their own
    # streams hold different PSFs at the same time: nobody may see somebody else's (or stale) taps
    gm.gm_set_option(gm.GM_OPT_TENSOR, 0)                    # the constant-bank taps belong to the FFMA2 engine
    request.addfinalizer(lambda: gm.gm_set_option(gm.GM_OPT_TENSOR, 1))
    model = models.single_sersic()
    H = W = 64; K = 25
    par, data, sigma, mask, _ = synth(model, 4, H, W, K, seed=99)
    psfs = [asymmetric_psf(K, seed=300 + i).astype(np.float32) for i in range(6)]
    gm.gm_set_option(gm.GM_OPT_CONST_TAPS, 0)
    try:
        want = [gm.gm_render(model, dev(par), H, W, dev(p)).clone() for p in psfs]
    finally:
        gm.gm_set_option(gm.GM_OPT_CONST_TAPS, 1)
    for rnd in range(3):                                   # back to back on one stream
        for p, w in zip(psfs, want):
            assert torch.equal(gm.gm_render(model, dev(par), H, W, dev(p)), w)
    streams = [torch.cuda.Stream() for _ in psfs]          # and all at once
    torch.cuda.synchronize()
    outs = []
    for rnd in range(3):
        for p, st in zip(psfs, streams):
            with torch.cuda.stream(st):
                outs.append(gm.gm_render(model, dev(par), H, W, dev(p)))
    torch.cuda.synchronize()
    for i, o in enumerate(outs):
        assert torch.equal(o, want[i % len(psfs)])


# ---- mask / sigma properties on the GPU (reading X1) -------------------------------
def test_mask_properties():
    model = models.single_sersic()
    par, data, sigma, mask, psf = synth(model, 2, 32, 32, 9, seed=3)
    chi2, grad = run_loss_grad(model, par, data, sigma, mask, psf)
    z, gz = run_loss_grad(model, par, data, sigma, np.zeros_like(mask), psf)
    assert not z.any() and not gz.any()
    bad = data.copy(); bs = sigma.copy()
    i, j = np.argwhere(mask[0] == 0)[0]
    bad[0, i, j] = np.nan; bs[0, i, j] = 0.0
    cn, gn = run_loss_grad(model, par, bad, bs, mask, psf)
    assert np.array_equal(cn, chi2) and np.array_equal(gn, grad)
    c_none, _ = run_loss_grad(model, par, data, sigma, None, psf)
    c_ones, _ = run_loss_grad(model, par, data, sigma, np.ones_like(mask), psf)
    assert np.array_equal(c_none, c_ones)
    oc, _ = oracle.loss_grad(model, par, data, sigma, None, psf)
    assert_chi2(c_none, oc)


def test_centre_on_pixel_centre_S4():
    model = models.single_sersic()
    H = W = 16
    psf = asymmetric_psf(5).astype(np.float32)
    par = np.array([[8.5, 7.5, 1.0, 3.0, 4.0, 0.7, 0.3], [8.5, 7.5, 1.0, 3.0, 1.2, 1.0, 0.0]], dtype=np.float32)
    M = oracle.render(model, par, H, W, psf)
    img = gm.gm_render(model, dev(par), H, W, dev(psf)).cpu().numpy()
    assert np.isfinite(img).all()
    assert_pixels(img, M)
    sigma = np.full((2, H, W), 0.1, dtype=np.float32)
    data = (M * 1.1).astype(np.float32)
    chi2, grad = run_loss_grad(model, par, data, sigma, None, psf)
    oc, og = oracle.loss_grad(model, par, data, sigma, None, psf)
    assert np.isfinite(grad).all()
    assert_chi2(chi2, oc)
    assert_grad(grad, og)


def test_results_are_deterministic():
    b = configs.make_batch(0, range(8), oracle_render)
    a1 = run_loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    a2 = run_loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    assert np.array_equal(a1[0], a2[0]) and np.array_equal(a1[1], a2[1])


# ---- host-buffer entry points agree with the device ones ------------------------------
def test_host_entry_points():
    b = configs.make_batch(0, range(5), oracle_render)
    model = b["model"]
    img_h = gm.gm_render_host(model, b["start"], 64, 64, b["psf"])
    img_d = gm.gm_render(model, dev(b["start"]), 64, 64, dev(b["psf"])).cpu().numpy()
    assert np.array_equal(img_h, img_d)
    c_h, g_h = gm.gm_loss_grad_host(model, b["start"], b["data"], b["sigma"], None, b["psf"])
    c_d, g_d = run_loss_grad(model, b["start"], b["data"], b["sigma"], None, b["psf"])
    assert np.array_equal(c_h, c_d) and np.array_equal(g_h, g_d)


# ---- accuracy contract of a rendered pixel (gm_device.cuh) ----------------
@pytest.mark.parametrize("tensor", [1, 0])
def test_render_accuracy_high_n_wings(tensor):
    """Unconvolved Sersic pixels are within 2e-5 relative of the oracle wherever the profile has not underflowed
    (nu t < 30, t = (r / re)^(1/n)): five times tighter than the pixel tolerance, far out in the wings of low-n
    profiles and through the steep cores of high-n ones, where the SFU error of lg2 and the fp32 rounding of the
    exponent are amplified by nu t (worst measured: 1.3e-5 at the nu t -> 30 edge of an n = 0.5 profile)."""
    model = models.one_component("sersic", convolve=0)              # [xc, yc, theta, q, Ie, re, n]
    H = W = 128
    rows = [(n, re, q) for n in (0.5, 1.0, 2.0, 4.0, 6.0, 8.0) for re, q in ((2.0, 0.9), (9.5, 0.35))]
    par = np.array([[64.37, 63.21, 0.3 + 0.2 * k, q, 3.0, re, n] for k, (n, re, q) in enumerate(rows)], dtype=np.float32)
    psf = gaussian_psf(15, 3.0).astype(np.float32)
    gm.gm_set_option(gm.GM_OPT_TENSOR, tensor)
    try:
        img = gm.gm_render(model, dev(par), H, W, dev(psf)).cpu().numpy().astype(np.float64)
    finally:
        gm.gm_set_option(gm.GM_OPT_TENSOR, 1)
    ref = oracle.render(model, par, H, W, psf)
    covered = 0
    for k, (n, re, q) in enumerate(rows):
        nu = oracle.sersic_nu(float(np.float32(n)))
        live = ref[k] > 3.0 * math.exp(nu - 30.0)                  # I = Ie exp(-nu (t - 1)): nu t < 30
        rel = np.abs(img[k] - ref[k])[live] / ref[k][live]
        assert rel.max() < 2e-5, (n, re, q, rel.max())
        covered += int(live.sum())
        if n <= 1.0 and re == 2.0:
            assert not live.all()                                  # the low-n wings do reach the underflow edge
    assert covered > 0.7 * len(rows) * H * W
