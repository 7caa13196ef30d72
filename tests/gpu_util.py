"""Helpers shared by the -m gpu parity tests: tolerances from BASELINE.json
north_star and comparison of the CUDA path (through the C ABI binding) with the
fp64 oracle on the same seeded float32 inputs."""
import numpy as np
import torch

import oracle

# BASELINE.json north_star tolerances (restated in DESIGN.md "Parity")
PIX_RTOL = 1e-4          # rendered pixels, relative ...
PIX_FLOOR = 1e-7         # ... plus 1e-7 * max pixel of the oracle image (reading T1)
CHI2_RTOL = 1e-5
GRAD_RTOL = 1e-3         # || g_gpu - g_orc ||_2 <= 1e-3 || g_orc ||_2 per galaxy
PAR_RTOL = 1e-3          # fitted parameters after a fixed iteration count


def dev(a, dtype=None):
    if a is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def oracle_render(model, p, H, W, psf):
    return oracle.render(model, p, H, W, psf)


def assert_pixels(gpu, orc):
    gpu = np.asarray(gpu, dtype=np.float64)
    for g in range(orc.shape[0]):
        tol = PIX_RTOL * np.abs(orc[g]) + PIX_FLOOR * np.abs(orc[g]).max()
        err = np.abs(gpu[g] - orc[g])
        bad = err > tol
        assert not bad.any(), (f"galaxy {g}: {bad.sum()} pixels out of tolerance, worst "
                               f"{(err / np.maximum(tol, 1e-300)).max():.2f}x at "
                               f"{np.unravel_index(np.argmax(err / np.maximum(tol, 1e-300)), err.shape)}")


def assert_chi2(gpu, orc, rtol=CHI2_RTOL):
    gpu = np.asarray(gpu, dtype=np.float64)
    rel = np.abs(gpu - orc) / np.maximum(np.abs(orc), 1e-300)
    assert np.all(rel <= rtol), f"chi2 rel err max {rel.max():.3e} (tol {rtol:g}) at {rel.argmax()}"


def assert_grad(gpu, orc, rtol=GRAD_RTOL):
    gpu = np.asarray(gpu, dtype=np.float64)
    num = np.linalg.norm(gpu - orc, axis=1)
    den = np.linalg.norm(orc, axis=1)
    rel = num / np.maximum(den, 1e-300)
    assert np.all(rel <= rtol), f"grad rel err max {rel.max():.3e} (tol {rtol:g}) at galaxy {rel.argmax()}"
