"""-m gpu: gm_conv (the PSF convolution on its own, FFMA2 loop or tcgen05 tensor cores) against
oracle.conv2d_same / corr2d_same, which tests/test_oracle_conv.py pins to scipy.signal."""
import numpy as np
import pytest
import torch

import oracle
import paper_2404_07780_b200 as gm
from gen import models
from gen.psf import gaussian_psf, moffat_psf
from gpu_util import assert_pixels, dev

pytestmark = pytest.mark.gpu


def images(B, H, W, seed):
    """Sersic-like cutouts with a steep core and faint wings plus a few negative pixels: the dynamic
    range the fp16 split of the tensor engine has to live with."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:H, 0:W]
    out = np.empty((B, H, W), dtype=np.float32)
    for b in range(B):
        xc, yc = W / 2 + rng.uniform(-3, 3), H / 2 + rng.uniform(-3, 3)
        r = np.hypot(x - xc, (y - yc) / rng.uniform(0.3, 1.0))
        n = rng.uniform(0.5, 6.0)
        img = rng.lognormal(0, 1) * 50.0 * np.exp(-(2 * n - 1 / 3) * ((r / rng.uniform(2, 10)) ** (1 / n) - 1))
        img += rng.normal(0, 1e-3, size=img.shape)
        out[b] = img
    return out


def asymmetric(K, seed):
    rng = np.random.default_rng(seed)
    p = moffat_psf(K, 3.5, 3.0) * (1.0 + 0.3 * rng.uniform(-1, 1, size=(K, K)))
    return (p / p.sum()).astype(np.float32)


@pytest.mark.parametrize("engine", ["ffma2", "tensor"])
@pytest.mark.parametrize("K", [41, 25, 33, 15, 9, 3])
@pytest.mark.parametrize("adjoint", [False, True])
def test_conv_matches_oracle_128(engine, K, adjoint):
    eng = gm.GM_CONV_TENSOR if engine == "tensor" else gm.GM_CONV_FFMA2
    img = images(5, 128, 128, seed=K)
    psf = asymmetric(K, seed=100 + K)
    out = gm.gm_conv(dev(img), dev(psf), engine=eng, adjoint=adjoint).cpu().numpy()
    ref = np.stack([(oracle.corr2d_same if adjoint else oracle.conv2d_same)(img[b], psf) for b in range(5)])
    assert_pixels(out, ref)


@pytest.mark.parametrize("engine", ["ffma2", "tensor"])
def test_conv_many_cutouts_and_per_galaxy_psfs(engine):
    # more cutouts than SMs (the persistent CTAs of the tensor engine take several each), one PSF per cutout
    eng = gm.GM_CONV_TENSOR if engine == "tensor" else gm.GM_CONV_FFMA2
    B, K = 333, 25
    img = images(8, 128, 128, seed=1)
    img = np.ascontiguousarray(np.concatenate([img] * 42)[:B])
    psfs = np.stack([asymmetric(K, seed=500 + (b % 5)) for b in range(B)])
    out = gm.gm_conv(dev(img), dev(psfs), engine=eng).cpu().numpy()
    for b in list(range(0, B, 37)) + [B - 1]:
        assert_pixels(out[b:b + 1], oracle.conv2d_same(img[b], psfs[b])[None])
    shared = gm.gm_conv(dev(img), dev(psfs[0]), engine=eng).cpu().numpy()
    same = [b for b in range(B) if b % 5 == 0]
    assert np.array_equal(shared[same], out[same])       # the same PSF gives the same pixels either way


def test_tensor_engine_precision_and_dynamic_range():
    # fp16 halves after ONE power-of-two scale per cutout: a pixel 2^-k below the brightest keeps about
    # 22 - max(0, k - 18) significant bits, i.e. the ABSOLUTE error stays near 2^-24 of the brightest
    # pixel whatever the dynamic range (the contract of include/gm.h gm_conv).  A delta of 1e4 on a
    # background of 1e-4 (eight decades) and a PSF with five decades between core and wing:
    H = W = 128; K = 41
    img = np.full((1, H, W), 1e-4, dtype=np.float32)
    img[0, 60, 70] = 1e4
    psf = gaussian_psf(K, 6.0).astype(np.float32)
    out = gm.gm_conv(dev(img), dev(psf), engine=gm.GM_CONV_TENSOR).cpu().numpy().astype(np.float64)
    ref = oracle.conv2d_same(img[0], psf)[None]
    assert np.abs(out - ref).max() <= 1e-6 * ref.max()
    near = ref > 1e-3 * ref.max()                       # where the delta dominates: full relative precision
    assert (np.abs(out - ref)[near] / ref[near]).max() < 1e-5
    # galaxy-like cutouts: relative error of the bright pixels (bias of the truncating fp32 accumulation
    # in the tensor core, kept small by visiting the tap rows outside-in) against the FFMA2 engine's
    img = images(8, H, W, seed=5)
    psf = asymmetric(K, seed=7)
    ref = np.stack([oracle.conv2d_same(img[b], psf) for b in range(8)])
    bright = np.abs(ref) > 1e-3 * np.abs(ref).max(axis=(1, 2), keepdims=True)
    for eng, lim in ((gm.GM_CONV_TENSOR, 2e-5), (gm.GM_CONV_FFMA2, 2e-5)):
        out = gm.gm_conv(dev(img), dev(psf), engine=eng).cpu().numpy().astype(np.float64)
        rel = np.abs(out - ref)[bright] / np.abs(ref)[bright]
        assert rel.max() < lim, (eng, rel.max())


def test_tensor_engine_refuses_other_sizes():
    with pytest.raises(gm.GmError):
        gm.gm_conv(torch.zeros(2, 64, 64, device="cuda"), torch.ones(5, 5, device="cuda"), engine=gm.GM_CONV_TENSOR)


def test_tensor_engine_refuses_misaligned_views():
    """gm.h, gm_conv: the tensor engine moves 128-bit rows, so an image or output view that starts 4 bytes off
    a 16-byte boundary is GM_EINVAL before any launch (no fault, no sticky error); the FFMA2 engine takes it."""
    img = images(3, 128, 128, seed=2)
    psf = asymmetric(15, seed=3)
    flat = torch.zeros(3 * 128 * 128 + 1, device="cuda")
    view = flat[1:].view(3, 128, 128)
    view.copy_(dev(img))
    assert view.data_ptr() % 16 == 4
    with pytest.raises(gm.GmError) as e:
        gm.gm_conv(view, dev(psf), engine=gm.GM_CONV_TENSOR)
    assert e.value.status == -1
    oflat = torch.zeros(3 * 128 * 128 + 1, device="cuda")
    with pytest.raises(gm.GmError) as e:
        gm.gm_conv(dev(img), dev(psf), engine=gm.GM_CONV_TENSOR, out=oflat[1:].view(3, 128, 128))
    assert e.value.status == -1
    torch.cuda.synchronize()                                  # the context is still healthy
    ref = np.stack([oracle.conv2d_same(img[b], psf) for b in range(3)])
    assert_pixels(gm.gm_conv(view, dev(psf), engine=gm.GM_CONV_FFMA2).cpu().numpy(), ref)
    assert_pixels(gm.gm_conv(dev(img), dev(psf), engine=gm.GM_CONV_TENSOR).cpu().numpy(), ref)


def test_phase_trace_hook_records_every_phase():
    """gm_trace_set (include/gm.h): CTA 0 of k_tc_fused appends one record per phase boundary; the hook is
    off by default and switches off again with None."""
    import torch
    rng = np.random.default_rng(7)
    model = models.single_sersic()
    B, H, K = 300, 128, 25                                   # three cutouts for CTA 0 of 148
    par = np.tile(np.array([[64.3, 63.1, 1.0, 6.0, 2.0, 0.7, 0.4]], dtype=np.float32), (B, 1))
    psf = np.zeros((K, K), dtype=np.float32); psf[K // 2, K // 2] = 1.0
    data = rng.normal(size=(B, H, H)).astype(np.float32); sigma = np.ones_like(data)
    d = lambda a: torch.from_numpy(a).cuda()
    buf = torch.zeros(gm.binding.TRACE_ROLES * gm.binding.TRACE_CAP, dtype=torch.int64, device="cuda")
    gm.gm_trace_set(buf)
    try:
        gm.gm_loss_grad(model, d(par), d(data), d(sigma), None, d(psf))
        torch.cuda.synchronize()
    finally:
        gm.gm_trace_set(None)
    rec = buf.cpu().numpy().view(np.uint64).reshape(gm.binding.TRACE_ROLES, gm.binding.TRACE_CAP)
    helper = [int(x) for x in rec[0] if x]; mma = [int(x) for x in rec[1] if x]
    tags = [x >> 56 for x in helper]
    # 3 cutouts: produce begin/end, drain wait/begin twice, residual begin/end, gradient begin/end each
    assert tags.count(1) == 3 and tags.count(2) == 3 and tags.count(5) == 3 and tags.count(7) == 3 and tags.count(8) == 3
    assert len(mma) == 2 * 2 * 3                             # job begin / end of two convolutions per cutout
    clk = [x & ((1 << 48) - 1) for x in helper]
    assert all(b >= a for a, b in zip(clk, clk[1:]))         # one thread writes the list in program order
    again = torch.zeros_like(buf)
    gm.gm_loss_grad(model, d(par), d(data), d(sigma), None, d(psf))
    torch.cuda.synchronize()
    assert int(again.abs().sum().item()) == 0
