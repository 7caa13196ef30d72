"""-m gpu: the bootstrap row (Sec. 5.2; reading B1) through the C ABI against the
oracle: multiplicities bit-exact (integer work), refits and error bars within the fit
tolerances."""
import numpy as np
import pytest
import torch

import oracle
import paper_2404_07780_b200 as gm
from gen import configs
from gpu_util import dev, oracle_render

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("shape,masked", [((3, 64, 64), False), ((5, 37, 53), True), ((2, 128, 96), True),
                                          ((1, 1, 1), False), ((2, 33, 40), "empty")])
def test_counts_bit_exact(shape, masked):
    B, H, W = shape
    rng = np.random.default_rng(4)
    mask = None
    if masked == "empty":
        mask = np.zeros(shape, dtype=np.uint8); mask[1, 5, 7] = 1        # galaxy 0 has no used pixel
    elif masked:
        mask = (rng.random(shape) > 0.25).astype(np.uint8)
    for r in (0, 3):
        c = gm.gm_bootstrap_counts(B, H, W, dev(mask), seed=99, r=r, id_offset=1000)
        torch.cuda.synchronize()
        c = c.cpu().numpy()
        for g in range(B):
            ref, n_used = oracle.bootstrap_counts(99, 1000 + g, r, None if mask is None else mask[g], (H, W))
            assert np.array_equal(c[g], ref), (g, r)
            assert c[g].sum() == n_used


def test_counts_full_size_bucket():
    # C2's largest bucket shape at full batch width: sums and zero pattern on every galaxy, a sample of
    # galaxies bit-exact against the oracle
    B, H, W = 1658, 256, 256
    g = torch.Generator(device="cuda"); g.manual_seed(1)
    mask = (torch.rand((B, H, W), device="cuda", generator=g) > 0.1).to(torch.uint8)
    c = gm.gm_bootstrap_counts(B, H, W, mask, seed=7, r=42)
    torch.cuda.synchronize()
    assert torch.equal(c.sum(dim=(1, 2)), mask.sum(dim=(1, 2), dtype=torch.int64).to(c.sum(dim=(1, 2)).dtype))
    assert int((c * (1 - mask.to(torch.int32))).abs().sum()) == 0
    for b in (0, 811, 1657):
        ref, _ = oracle.bootstrap_counts(7, b, 42, mask[b].cpu().numpy(), (H, W))
        assert np.array_equal(c[b].cpu().numpy(), ref)


def test_bootstrap_matches_oracle():
    b = configs.make_batch(0, range(4), oracle_render)
    mask = (np.random.default_rng(3).random(b["data"].shape) > 0.1).astype(np.uint8)
    opts = configs.fit_options(b["model"], 64, 64, 40)
    M = 12
    o = oracle.bootstrap(b["model"], b["start"], b["data"], b["sigma"], mask, b["psf"], opts, M, seed=5, id_offset=10)
    start = dev(b["start"])
    before = start.clone()
    g = gm.gm_bootstrap(b["model"], start, dev(b["data"]), dev(b["sigma"]), dev(mask), dev(b["psf"]), opts,
                        M, seed=5, id_offset=10, want_samples=True)
    torch.cuda.synchronize()
    assert torch.equal(start, before)                              # the start point is not modified
    smp = g["samples"].cpu().numpy().astype(np.float64)
    # every refit follows the oracle's refit (40 iterations: still well conditioned)
    assert np.allclose(smp, o["samples"], rtol=1e-3, atol=1e-5)
    sb = g["sigma_boot"].cpu().numpy().astype(np.float64)
    assert np.allclose(sb, o["sigma_boot"], rtol=2e-2, atol=1e-6), np.abs(sb / o["sigma_boot"] - 1).max()
    assert np.allclose(g["mean"].cpu().numpy(), o["mean"], rtol=1e-3, atol=1e-5)
    # the statistics are those of the returned samples, population variance (1/M)
    assert np.allclose(sb, smp.std(axis=0, ddof=0), rtol=1e-5, atol=1e-7)


def test_bootstrap_fixed_parameter_and_early_stop():
    b = configs.make_batch(0, range(3), oracle_render)
    opts = configs.fit_options(b["model"], 64, 64, 120, tol=1e-5, patience=5)
    opts["free_mask"] = np.array([1, 1, 1, 1, 0, 1, 1], dtype=np.uint8)
    g = gm.gm_bootstrap(b["model"], dev(b["start"]), dev(b["data"]), dev(b["sigma"]), None, dev(b["psf"]), opts,
                        6, seed=1, want_samples=True)
    torch.cuda.synchronize()
    sb = g["sigma_boot"].cpu().numpy()
    assert np.all(sb[:, 4] == 0.0) and np.all(sb[:, [0, 1, 2, 3, 5]] > 0.0)
    assert np.array_equal(g["samples"].cpu().numpy()[:, :, 4], np.broadcast_to(b["start"][:, 4], (6, 3)))
    # a second run gives the same bits
    g2 = gm.gm_bootstrap(b["model"], dev(b["start"]), dev(b["data"]), dev(b["sigma"]), None, dev(b["psf"]), opts,
                         6, seed=1, want_samples=True)
    torch.cuda.synchronize()
    assert torch.equal(g["samples"], g2["samples"]) and torch.equal(g["sigma_boot"], g2["sigma_boot"])


def test_bootstrap_argument_errors():
    b = configs.make_batch(0, range(2), oracle_render)
    opts = configs.fit_options(b["model"], 64, 64, 3)
    args = (b["model"], dev(b["start"]), dev(b["data"]), dev(b["sigma"]), None, dev(b["psf"]), opts)
    with pytest.raises(gm.GmError):
        gm.gm_bootstrap(*args, 0, seed=1)
    with pytest.raises(gm.GmError) as e:
        gm.gm_bootstrap(*args, 4, seed=1, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))
    assert e.value.status == -4
