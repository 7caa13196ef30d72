"""Seeded synthetic SDSS-like inputs for BASELINE.json configs C0..C4.

These inputs STAND IN for the paper's SDSS g-band sample (8,289 cutouts of
128x128 px with 41x41 PSFs), which is not available; shapes, sizes and
value ranges follow BASELINE.json ``configs`` (recipe restated in DESIGN.md).

This module holds no arithmetic of the method: the noiseless truth image is
produced by a ``render(model, params_f32, H, W, psf_f32) -> [B,H,W]`` callable
supplied by the caller (the oracle in tests, the CUDA ``gm_render`` in bench).

RNG: ``numpy.random.Generator(PCG64)`` seeded from
``SeedSequence(20240407, spawn_key=(config, galaxy, stream))`` with stream
0 = truth, 1 = start point, 2 = noise, 3 = cutout side, 4 = mask, so any subset
of galaxies is reproducible whatever the batch size.  Everything is drawn in
float64 and cast to float32 once; the same float32 arrays go to both sides.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import models, psf as psfmod

SEED = 20240407
GAIN = 4.7          # e-/ADU
SKY_E = 100.0       # e-/px
READ_E = 5.0        # e- rms


@dataclass(frozen=True)
class Config:
    cid: int
    name: str
    B: int
    sides: tuple
    K: int
    psf_kind: str
    model_name: str
    noise: str           # "gauss" (C0) | "ccd" (C1-C4)
    start: str           # "c0" | "c1"
    n_iter: int
    mask_frac: float = 0.0
    tol: float = 0.0
    patience: int = 10
    extra: dict = field(default_factory=dict)


CONFIGS = {
    0: Config(0, "C0", 16, (64,), 15, "gauss3", "single_sersic", "gauss", "c0", 0),
    1: Config(1, "C1", 1024, (128,), 25, "moffat3.5", "single_sersic", "ccd", "c1", 200),
    2: Config(2, "C2", 8289, (64, 96, 128, 192, 256), 25, "moffat3.5", "single_sersic", "ccd", "c1",
              500, mask_frac=0.10, tol=1e-6, patience=10),
    3: Config(3, "C3", 4096, (128,), 25, "moffat3.5", "bulge_disk", "ccd", "c1", 300),
    4: Config(4, "C4", 65536, (256,), 41, "moffat3.5", "sersic_bar_nucleus", "ccd", "c1", 200),
    # not a BASELINE.json entry: the SHAPES of the paper's own SDSS run (8,289 cutouts of 128x128
    # with 41x41 PSFs), single Sersic, otherwise as C1
    5: Config(5, "P1", 8289, (128,), 41, "moffat3.5", "single_sersic", "ccd", "c1", 200),
}


def get_model(cfg: Config) -> dict:
    return getattr(models, cfg.model_name)()


def make_psf(cfg: Config) -> np.ndarray:
    if cfg.psf_kind == "gauss3":
        p = psfmod.gaussian_psf(cfg.K, 3.0)
    else:
        p = psfmod.moffat_psf(cfg.K, 3.5, 3.0)
    return p.astype(np.float32)


def _rng(cid: int, g: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence(SEED, spawn_key=(cid, int(g), stream))))


def sides_for(cfg: Config, galaxies) -> np.ndarray:
    """Cutout side of each galaxy (C2: uniform over the five sides)."""
    if len(cfg.sides) == 1:
        return np.full(len(galaxies), cfg.sides[0], dtype=np.int64)
    return np.array([cfg.sides[_rng(cfg.cid, g, 3).integers(len(cfg.sides))] for g in galaxies],
                    dtype=np.int64)


# ---- truth parameters -------------------------------------------------------
def _truth_one(model_name: str, r: np.random.Generator, H: int, W: int) -> np.ndarray:
    U = r.uniform
    xc = W / 2 + U(-2, 2); yc = H / 2 + U(-2, 2)

    def sersic(re_lo=2.0, re_hi=10.0, n_lo=0.5, n_hi=6.0):
        return [r.lognormal(0.0, 1.0), U(re_lo, re_hi), U(n_lo, n_hi), U(0.2, 1.0), U(0.0, np.pi)]

    if model_name == "single_sersic":
        return np.array([xc, yc] + sersic())
    if model_name == "bulge_disk":
        bulge = sersic(1.0, 6.0, 2.0, 6.0)
        disk = [r.lognormal(0.0, 1.0), U(4.0, 20.0), U(0.2, 1.0), U(0.0, np.pi)]
        return np.array([xc, yc] + bulge + disk)
    if model_name == "sersic_bar_nucleus":
        ser = sersic()
        bar = [r.lognormal(0.0, 1.0), U(5.0, 30.0), U(0.5, 3.0), U(0.0, 2.0), U(0.2, 1.0), U(0.0, np.pi)]
        nuc = [r.lognormal(0.0, 1.0), U(1.5, 4.0), U(1.5, 5.0)]
        return np.array([xc, yc] + ser + bar + nuc)
    raise KeyError(model_name)


def truth_params(cfg: Config, galaxies, H: int, W: int) -> np.ndarray:
    return np.stack([_truth_one(cfg.model_name, _rng(cfg.cid, g, 0), H, W) for g in galaxies])


# ---- fit options (readings O2-O4) -------------------------------------------
_ROLE = {  # role: (lr, log10_space, lo, hi)   lo/hi None = set from the cutout size
    "cx": (0.05, 0, None, None), "cy": (0.05, 0, None, None),
    "amp": (0.01, 1, 1e-6, 1e6), "radius": (0.01, 1, 0.3, None),
    "index": (0.01, 1, 0.3, 8.0), "q": (0.01, 0, 0.05, 1.0),
    "theta": (0.02, 0, -np.inf, np.inf), "shape": (0.01, 0, 0.05, 10.0),
    "sky": (0.01, 0, -np.inf, np.inf),
    # boxiness B of Eq. 2 (c = B + 2 stays well above 0), magnitude m with
    # its zero point m0 (Eq. 5; 0.025 mag = 0.01 dex in flux, the step of an "amp")
    "box": (0.01, 0, -1.0, 2.0), "mag": (0.025, 0, -np.inf, np.inf),
    "zeropoint": (0.0, 0, -np.inf, np.inf),
}


def bounds(model: dict, H: int, W: int):
    lo = np.empty(model["n_par"]); hi = np.empty(model["n_par"])
    for k, (role, name) in enumerate(zip(model["roles"], model["names"])):
        _, _, l, h = _ROLE[role]
        if role == "cx":
            l, h = W / 2 - W / 4, W / 2 + W / 4
        elif role == "cy":
            l, h = H / 2 - H / 4, H / 2 + H / 4
        elif role == "radius":
            h = H / 2
        if name.endswith("f_b") or name.endswith("fe_b"):
            l, h = 0.0, 1.95           # Ferrer b: exponent 2-b must stay positive (Eq. 9)
        if name.endswith("m_n"):
            l, h = 1.05, 10.0          # Moffat total flux needs n > 1 (Eq. 15)
        lo[k], hi[k] = l, h
    return lo, hi


def fit_options(model: dict, H: int, W: int, n_iter: int, tol: float = 0.0, patience: int = 10) -> dict:
    P = model["n_par"]
    lo, hi = bounds(model, H, W)
    lr = np.array([_ROLE[r][0] for r in model["roles"]])
    lg = np.array([_ROLE[r][1] for r in model["roles"]], dtype=np.uint8)
    decay = 0.01 ** (1.0 / max(n_iter - 1, 1))      # last step ~1 % of the first (O2)
    return {"n_iter": int(n_iter), "beta1": 0.9, "beta2": 0.999, "eps": 1e-8, "lr_decay": decay,
            "lr": lr.astype(np.float32), "lo": lo.astype(np.float32), "hi": hi.astype(np.float32),
            "log10_space": lg,
            "free_mask": np.array([r != "zeropoint" for r in model["roles"]], dtype=np.uint8),   # m0 is given
            "tol": float(tol),
            "patience": int(patience)}


# ---- start point ------------------------------------------------------------
def start_params(cfg: Config, model: dict, truth: np.ndarray, galaxies, H: int, W: int) -> np.ndarray:
    lo, hi = bounds(model, H, W)
    out = np.empty_like(truth)
    wide = cfg.start == "c1"
    fs = (0.8, 1.2) if wide else (0.9, 1.1)
    dc = 1.0 if wide else 0.5
    for row, g in enumerate(galaxies):
        r = _rng(cfg.cid, g, 1)
        for k, role in enumerate(model["roles"]):
            t = truth[row, k]
            if role in ("cx", "cy"):
                v = t + r.uniform(-dc, dc)
            elif role == "theta":
                v = t * r.uniform(*fs) if wide else t + r.uniform(-0.1, 0.1)
            else:
                v = t * r.uniform(*fs)
            out[row, k] = min(max(v, lo[k]), hi[k])
    return out


# ---- noise ------------------------------------------------------------------
def _noise_one(cfg: Config, g: int, M: np.ndarray, Ie: float):
    r = _rng(cfg.cid, g, 2)
    if cfg.noise == "gauss":
        s = 0.05 * Ie
        D = M + r.normal(0.0, s, size=M.shape)
        sigma = np.full(M.shape, s)
    else:
        lam = GAIN * np.clip(M, 0.0, None) + SKY_E
        Ne = r.poisson(lam).astype(np.float64) + r.normal(0.0, READ_E, size=M.shape)
        D = Ne / GAIN - SKY_E / GAIN
        sigma = np.sqrt(lam + READ_E ** 2) / GAIN
    if cfg.mask_frac > 0.0:
        mask = (_rng(cfg.cid, g, 4).random(M.shape) >= cfg.mask_frac).astype(np.uint8)
    else:
        mask = np.ones(M.shape, dtype=np.uint8)
    return D, sigma, mask


def make_batch(cid: int, galaxies, render, side: int | None = None, workers: int = 1, **overrides) -> dict:
    """Inputs for the given galaxy indices of config ``cid`` (one cutout side).

    ``overrides`` replace fields of the config (``K=41``, ``psf_kind="moffat3.5"`` ...): the same
    recipe on another shape, e.g. C0's constant-sigma noise on 128 px cutouts under a 41 x 41 PSF.

    ``render(model, params_f32[B,P], H, W, psf_f32) -> ndarray[B,H,W]`` supplies the
    noiseless model.  For C2, ``side`` selects the size bucket; galaxies whose
    drawn side differs are dropped.  ``workers`` > 1 draws the noise of different galaxies in
    threads (every galaxy has its own generator, so the result does not depend on it).
    """
    cfg = CONFIGS[cid]
    if overrides:
        from dataclasses import replace
        cfg = replace(cfg, **overrides)
    galaxies = list(galaxies)
    if len(cfg.sides) > 1:
        assert side is not None
        sd = sides_for(cfg, galaxies)
        galaxies = [g for g, s in zip(galaxies, sd) if s == side]
    else:
        side = cfg.sides[0] if side is None else side
    H = W = int(side)
    model = get_model(cfg)
    psf = make_psf(cfg)
    truth = truth_params(cfg, galaxies, H, W).astype(np.float32)
    M = np.asarray(render(model, truth, H, W, psf), dtype=np.float64)
    B = len(galaxies)
    data = np.empty((B, H, W), dtype=np.float32)
    sigma = np.empty((B, H, W), dtype=np.float32)
    mask = np.empty((B, H, W), dtype=np.uint8)
    amp_idx = model["roles"].index("amp")
    def noise(row):
        D, s, m = _noise_one(cfg, galaxies[row], M[row], float(truth[row, amp_idx]))
        data[row] = D; sigma[row] = s; mask[row] = m

    if workers > 1 and B > 1:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=workers) as ex:
            list(ex.map(noise, range(B)))
    else:
        for row in range(B):
            noise(row)
    start = start_params(cfg, model, truth.astype(np.float64), galaxies, H, W).astype(np.float32)
    return {"cfg": cfg, "model": model, "galaxies": galaxies, "H": H, "W": W, "K": cfg.K,
            "psf": psf, "truth": truth, "start": start, "data": data, "sigma": sigma,
            "mask": mask if cfg.mask_frac > 0.0 else None,
            "opts": fit_options(model, H, W, cfg.n_iter, cfg.tol, cfg.patience)}
