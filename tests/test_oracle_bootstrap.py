"""Pins of the oracle's bootstrap row (Sec. 5.2; reading B1 of DESIGN.md): the
counter-based generator against the published splitmix64 test vectors, the invariants of
a resample with replacement, the weighted chi^2 against the explicit list of drawn
pixels, the population variance against numpy and a hand example, and the size of the
bootstrap error bar against the closed form of a resampled mean."""
import numpy as np

import oracle
from gen import configs, models
from gen.psf import gaussian_psf

M64 = (1 << 64) - 1
GOLDEN = 0x9E3779B97F4A7C15


def test_mix64_is_the_splitmix64_finaliser():
    # splitmix64 (Steele, Lea & Flood 2014; Vigna's reference code): next() = mix(state += golden).
    # Published outputs for seed 0 and for seed 1234567.
    s, out = 0, []
    for _ in range(3):
        s = (s + GOLDEN) & M64
        out.append(oracle.mix64(s))
    assert out == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    s, out = 1234567, []
    for _ in range(3):
        s = (s + GOLDEN) & M64
        out.append(oracle.mix64(s))
    assert out == [6457827717110365317, 3203168211198807973, 9817491932198370423]


def py_counts(seed, gid, r, mask, N):
    """the definition of reading B1, typed again in Python integers"""
    def mix(z):
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
        return z ^ (z >> 31)
    used = [i for i in range(N) if mask is None or mask[i]]
    base = (mix((mix(seed ^ ((gid * GOLDEN) & M64)) + r) & M64))
    c = np.zeros(N, dtype=np.int64)
    for d in range(len(used)):
        z = mix((base + d) & M64)
        c[used[((z >> 32) * len(used)) >> 32]] += 1
    return c


def test_counts_follow_the_definition_and_its_invariants():
    rng = np.random.default_rng(0)
    mask = (rng.random((12, 9)) > 0.3).astype(np.uint8)
    c, n_used = oracle.bootstrap_counts(77, 5, 3, mask, mask.shape)
    assert n_used == mask.sum() and c.sum() == n_used          # n_used draws, all on used pixels
    assert (c[mask == 0] == 0).all() and c.min() >= 0
    assert np.array_equal(c.reshape(-1), py_counts(77, 5, 3, mask.reshape(-1), mask.size))
    # no mask: every pixel can be drawn
    c2, n2 = oracle.bootstrap_counts(77, 5, 3, None, (12, 9))
    assert n2 == 108 and c2.sum() == 108
    assert np.array_equal(c2.reshape(-1), py_counts(77, 5, 3, None, 108))
    # a different resample, galaxy or seed gives different draws; the same key the same draws
    for key in ((77, 5, 4), (77, 6, 3), (78, 5, 3)):
        assert not np.array_equal(oracle.bootstrap_counts(*key, None, (12, 9))[0], c2)
    assert np.array_equal(oracle.bootstrap_counts(77, 5, 3, None, (12, 9))[0], c2)
    # degenerate: nothing used -> nothing drawn
    c0, n0 = oracle.bootstrap_counts(1, 1, 1, np.zeros((4, 4), np.uint8), (4, 4))
    assert n0 == 0 and c0.sum() == 0


def test_multiplicities_have_the_resampling_distribution():
    # N draws from N pixels: c ~ Binomial(N, 1/N): mean 1, variance 1 - 1/N, P(0) = (1-1/N)^N ~ 1/e,
    # P(1) ~ 1/e, P(2) ~ 1/(2e); resamples are uncorrelated
    N = 128 * 128
    cs = np.stack([oracle.bootstrap_counts(2024, 11, r, None, (128, 128))[0].reshape(-1) for r in range(8)])
    assert np.all(cs.sum(axis=1) == N)
    assert abs(cs.var() - (1 - 1 / N)) < 0.02
    for k, p in ((0, np.exp(-1)), (1, np.exp(-1)), (2, np.exp(-1) / 2), (3, np.exp(-1) / 6)):
        assert abs((cs == k).mean() - p) < 4 * np.sqrt(p / cs.size) + 1e-3, k
    cc = np.corrcoef(cs.astype(np.float64))
    assert np.abs(cc - np.eye(8)).max() < 0.04
    # uniform over the image: the four quadrants get a quarter of the draws each
    q = cs.reshape(8, 2, 64, 2, 64).sum(axis=(0, 2, 4)) / cs.sum()
    assert np.abs(q - 0.25).max() < 0.01


def test_weighted_chi2_is_the_sum_over_the_drawn_pixels():
    # a pixel drawn twice counts twice: chi^2 with sigma / sqrt(c) and mask c > 0 equals the
    # plain sum over the explicit list of draws
    b = configs.make_batch(0, range(2), lambda m, p, H, W, psf: oracle.render(m, p, H, W, psf))
    M = oracle.render(b["model"], b["start"], 64, 64, b["psf"])
    for g in range(2):
        c, _ = oracle.bootstrap_counts(9, g, 0, None, (64, 64))
        sig = np.where(c > 0, b["sigma"][g] / np.sqrt(np.maximum(c, 1)), b["sigma"][g])
        chi2, _ = oracle.loss_grad(b["model"], b["start"][g:g + 1], b["data"][g:g + 1], sig[None],
                                   (c > 0).astype(np.uint8)[None], b["psf"])
        draws = np.repeat(np.arange(c.size), c.reshape(-1))
        assert draws.size == 4096
        r = (b["data"][g].astype(np.float64) - M[g]).reshape(-1)[draws] / b["sigma"][g].astype(np.float64).reshape(-1)[draws]
        assert abs(chi2[0] - np.sum(r * r)) <= 1e-10 * chi2[0]


def _flat_model():
    # a sky-only model: the fit of a constant is the weighted mean of the data
    return {"n_par": 1, "roles": ["sky"], "components": [{"kind": "sky", "convolve": 0, "slots": {"amp": 0}}]}


def test_bootstrap_of_a_mean_matches_the_closed_form():
    # D = mu + N(0, s^2) on N pixels, model = constant: every refit returns the mean of its
    # resample, whose scatter over resamples is s_D sqrt((N-1)/N) / sqrt(N) in expectation
    # (the textbook bootstrap standard error of a mean).  Pins the scale of sigma_boot (1/M, not
    # 1/(M-1); no missing or extra sqrt; weights c, not c^2) to a few percent.
    rng = np.random.default_rng(5)
    H = W = 24
    N = H * W
    data = (3.0 + 0.5 * rng.normal(size=(2, H, W))).astype(np.float32)
    sigma = np.full((2, H, W), 0.5, dtype=np.float32)
    psf = gaussian_psf(5, 2.0).astype(np.float32)
    opts = {"n_iter": 400, "lr": np.array([0.05]), "lo": np.array([-np.inf]), "hi": np.array([np.inf]),
            "lr_decay": 0.01 ** (1 / 399)}
    out = oracle.bootstrap(_flat_model(), np.array([[2.5], [3.5]]), data, sigma, None, psf, opts, 200, seed=3)
    # each sample is the weighted mean of its resample (the refit converged)
    for r in (0, 57, 199):
        for g in range(2):
            c, _ = oracle.bootstrap_counts(3, g, r, None, (H, W))
            assert abs(out["samples"][r, g, 0] - (c * data[g]).sum() / c.sum()) < 2e-4
    expect = data.reshape(2, -1).std(axis=1) / np.sqrt(N)
    assert np.all(np.abs(out["sigma_boot"][:, 0] / expect - 1.0) < 0.15), out["sigma_boot"][:, 0] / expect
    # population variance (1/M), as the paper's formula; numpy.std is the library routine
    assert np.allclose(out["sigma_boot"], out["samples"].std(axis=0, ddof=0), rtol=1e-12)
    assert np.allclose(out["mean"], out["samples"].mean(axis=0), rtol=1e-12)
    # hand example of the formula: samples 1, 2, 3, 6 -> mean 3, sigma^2 = (4+1+0+9)/4 = 3.5
    x = np.array([1.0, 2.0, 3.0, 6.0])
    assert np.isclose(np.sqrt(((x - x.mean()) ** 2).sum() / 4), np.sqrt(3.5))


def test_bootstrap_and_covariance_error_bars_agree_for_gaussian_noise():
    # Fig. 4 / P:210: both estimate the same 1-sigma interval when the noise model is right;
    # on a bright galaxy with Gaussian noise they agree within the bootstrap's own scatter
    model = models.single_sersic()
    H = W = 40
    psf = gaussian_psf(9, 2.5).astype(np.float32)
    truth = np.array([[20.3, 19.6, 2.0, 5.0, 1.5, 0.6, 0.7]], dtype=np.float32)
    M = oracle.render(model, truth, H, W, psf)
    rng = np.random.default_rng(2)
    sigma = np.full(M.shape, 0.05, dtype=np.float32)
    data = (M + 0.05 * rng.normal(size=M.shape)).astype(np.float32)
    opts = configs.fit_options(model, H, W, 250)
    best = oracle.fit(model, truth, data, sigma, None, psf, opts)["params"]
    cov = oracle.uncertainty(model, best, sigma, None, psf)["sigma_p"][0]
    boot = oracle.bootstrap(model, best, data, sigma, None, psf, opts, 40, seed=8)["sigma_boot"][0]
    ratio = boot / cov
    assert np.all((ratio > 0.6) & (ratio < 1.6)), ratio
