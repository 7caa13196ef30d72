"""The seeded input generator is reproducible per galaxy and follows BASELINE.json (not gpu)."""
import numpy as np

import oracle
from gen import configs


def _render(model, p, H, W, psf):
    return oracle.render(model, p, H, W, psf)


def test_subset_reproducible_whatever_the_batch():
    a = configs.make_batch(0, range(6), _render)
    b = configs.make_batch(0, [4, 1], _render)
    for key in ("truth", "start", "data", "sigma"):
        assert np.array_equal(a[key][4], b[key][0]) and np.array_equal(a[key][1], b[key][1])
    assert a["data"].dtype == np.float32 and a["psf"].shape == (15, 15)
    assert abs(float(a["psf"].sum()) - 1.0) < 1e-6


def test_c0_recipe_ranges():
    cfg = configs.CONFIGS[0]
    t = configs.truth_params(cfg, range(64), 64, 64)
    assert np.all(np.abs(t[:, 0] - 32) <= 2) and np.all(np.abs(t[:, 1] - 32) <= 2)
    assert np.all((t[:, 3] >= 2) & (t[:, 3] <= 10)) and np.all((t[:, 4] >= 0.5) & (t[:, 4] <= 6))
    assert np.all((t[:, 5] >= 0.2) & (t[:, 5] <= 1)) and np.all((t[:, 6] >= 0) & (t[:, 6] <= np.pi))
    b = configs.make_batch(0, range(3), _render)
    assert np.allclose(b["sigma"][1], 0.05 * b["truth"][1, 2], rtol=1e-6)


def test_c2_buckets_partition_the_sample():
    cfg = configs.CONFIGS[2]
    sides = configs.sides_for(cfg, range(400))
    assert set(np.unique(sides)) == {64, 96, 128, 192, 256}
    b = configs.make_batch(2, range(12), _render, side=64)
    assert b["H"] == 64 and len(b["galaxies"]) == int((sides[:12] == 64).sum())
    if len(b["galaxies"]):
        frac = 1.0 - b["mask"].mean()
        assert 0.07 < frac < 0.13
        assert np.all(b["sigma"] > 0)
