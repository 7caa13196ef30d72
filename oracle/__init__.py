"""ctypes loader for the fp64 CPU oracle (``oracle/gm_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2404_07780_b200`` and shares no code with the CUDA path.

Models are described by plain data (see ``gen.models``): a dict
``{"n_par": P, "components": [{"kind": str, "convolve": 0|1, "slots": {...}}]}``
where ``slots`` maps the names ``xc yc theta q amp s0 s1 s2 box m0`` to indices in
the per-galaxy parameter vector (missing = unused; a used ``m0`` slot means the
``amp`` slot holds a magnitude, Eq. 5/8/10/15).  Cites: P:35 (inputs),
P:61/P:322-327 (summed components, shared parameters), P:598 (psf flag).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gm_oracle.c"
_LIB = _HERE / "libgm_oracle.so"

KINDS = {"sersic": 0, "expdisk": 1, "ferrer": 2, "king": 3, "gaussian": 4, "moffat": 5, "sky": 6}
SLOT_NAMES = ("xc", "yc", "theta", "q", "amp", "s0", "s1", "s2", "box", "m0")

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2 -fopenmp).  Building is not using."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        d = C.c_double
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        bp = C.POINTER(C.c_uint8)
        i = C.c_int
        L.gmo_gammainc_P.restype = d; L.gmo_gammainc_P.argtypes = [d, d]
        L.gmo_sersic_nu.restype = d; L.gmo_sersic_nu.argtypes = [d]
        L.gmo_sersic_dnu_dn.restype = d; L.gmo_sersic_dnu_dn.argtypes = [d]
        L.gmo_r_box.restype = d; L.gmo_r_box.argtypes = [d]
        L.gmo_sersic_Ie_from_flux.restype = d; L.gmo_sersic_Ie_from_flux.argtypes = [d] * 5
        L.gmo_expdisk_I0_from_flux.restype = d; L.gmo_expdisk_I0_from_flux.argtypes = [d] * 4
        L.gmo_ferrer_I0_from_flux.restype = d; L.gmo_ferrer_I0_from_flux.argtypes = [d] * 6
        L.gmo_moffat_rd.restype = d; L.gmo_moffat_rd.argtypes = [d, d]
        L.gmo_moffat_I0_from_flux.restype = d; L.gmo_moffat_I0_from_flux.argtypes = [d] * 5
        L.gmo_loglike.restype = d; L.gmo_loglike.argtypes = [d, d]
        L.gmo_component_at.restype = None; L.gmo_component_at.argtypes = [i, i, dp, d, d, dp, dp]
        L.gmo_amplitude_from_mag.restype = i; L.gmo_amplitude_from_mag.argtypes = [i, dp, dp, dp]
        L.gmo_conv2d_same.restype = None; L.gmo_conv2d_same.argtypes = [dp, i, i, dp, i, dp]
        L.gmo_corr2d_same.restype = None; L.gmo_corr2d_same.argtypes = [dp, i, i, dp, i, dp]
        L.gmo_render.restype = i
        L.gmo_render.argtypes = [i, ip, i, i, i, i, i, dp, C.c_int64, dp, dp]
        L.gmo_loss_grad.restype = i
        L.gmo_loss_grad.argtypes = [i, ip, i, i, i, i, i, dp, C.c_int64, dp, dp, bp, dp, dp, dp, dp, dp]
        L.gmo_covariance_sigma.restype = i; L.gmo_covariance_sigma.argtypes = [i, dp, bp, dp]
        L.gmo_adam_step.restype = None
        L.gmo_adam_step.argtypes = [i, dp, dp, dp, dp, i, dp, d, d, d, d, dp, dp, bp]
        L.gmo_fit.restype = i
        L.gmo_fit.argtypes = [i, ip, i, i, i, i, i, dp, C.c_int64, dp, dp, bp, dp, i, d, d, d, d,
                              dp, dp, dp, bp, bp, d, i, dp, ip, ip, dp]
        L.gmo_mix64.restype = C.c_uint64; L.gmo_mix64.argtypes = [C.c_uint64]
        L.gmo_bootstrap_counts.restype = C.c_int64
        L.gmo_bootstrap_counts.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, bp, C.c_int64, ip]
        L.gmo_num_threads.restype = i; L.gmo_num_threads.argtypes = []
        L.gmo_set_num_threads.restype = None; L.gmo_set_num_threads.argtypes = [i]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _bp(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint8)) if a is not None else None


def _f64(a):
    return None if a is None else np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _u8(a):
    return None if a is None else np.ascontiguousarray(np.asarray(a).astype(np.uint8))


def descriptor(model: dict) -> np.ndarray:
    comps = model["components"]
    d = np.full((len(comps), 2 + len(SLOT_NAMES)), -1, dtype=np.int32)
    for c, comp in enumerate(comps):
        d[c, 0] = KINDS[comp["kind"]]
        d[c, 1] = int(comp.get("convolve", 1))
        for name, idx in comp["slots"].items():
            d[c, 2 + SLOT_NAMES.index(name)] = int(idx)
    return d


def _psf_args(psf, B):
    psf = _f64(psf)
    if psf.ndim == 2:
        return psf, 0, psf.shape[0]
    assert psf.ndim == 3 and psf.shape[0] == B
    return psf, psf.shape[1] * psf.shape[2], psf.shape[1]


# ---- scalar helpers -------------------------------------------------------
def gammainc_P(a, x):
    return lib().gmo_gammainc_P(float(a), float(x))


def sersic_nu(n):
    return lib().gmo_sersic_nu(float(n))


def sersic_dnu_dn(n):
    return lib().gmo_sersic_dnu_dn(float(n))


def r_box(B):
    return lib().gmo_r_box(float(B))


def sersic_Ie_from_flux(flux, re, n, q, B=0.0):
    return lib().gmo_sersic_Ie_from_flux(float(flux), float(re), float(n), float(q), float(B))


def expdisk_I0_from_flux(flux, rs, q, B=0.0):
    return lib().gmo_expdisk_I0_from_flux(float(flux), float(rs), float(q), float(B))


def ferrer_I0_from_flux(flux, rout, a, b, q, B=0.0):
    return lib().gmo_ferrer_I0_from_flux(float(flux), float(rout), float(a), float(b), float(q), float(B))


def moffat_rd(fwhm, n):
    return lib().gmo_moffat_rd(float(fwhm), float(n))


def moffat_I0_from_flux(flux, fwhm, n, q, B=0.0):
    return lib().gmo_moffat_I0_from_flux(float(flux), float(fwhm), float(n), float(q), float(B))


def loglike(chi2, k):
    return lib().gmo_loglike(float(chi2), float(k))


def component_at(kind: str, p, x, y, mag=False):
    """Value and d/d(xc,yc,theta,q,amp,s0,s1,s2,box[,m0]) of one component at (x,y).
    p has 9 entries (intensity amplitude) or 10 (mag=True: amp slot = magnitude m,
    last entry = zero point m0); the derivative vector has as many."""
    p = _f64(p)
    n = p.shape[0]
    assert n in (9, 10) and (n == 10 or not mag)
    p10 = np.zeros(10); p10[:n] = p
    I = C.c_double(0.0)
    dI = np.zeros(10)
    lib().gmo_component_at(KINDS[kind], int(bool(mag)), _dp(p10), float(x), float(y), C.byref(I), _dp(dI))
    return I.value, dI[:n]


def amplitude_from_mag(kind: str, p10):
    """Eq. 5 / 8 / 10 / 15: (amplitude, d ln amp / d slot [10]) for slot values p10."""
    p = _f64(p10)
    assert p.shape == (10,)
    amp = C.c_double(0.0)
    dla = np.zeros(10)
    rc = lib().gmo_amplitude_from_mag(KINDS[kind], _dp(p), C.byref(amp), _dp(dla))
    assert rc == 0, rc
    return amp.value, dla


def conv2d_same(S, psf):
    S = _f64(S); psf = _f64(psf)
    out = np.empty_like(S)
    lib().gmo_conv2d_same(_dp(S), S.shape[0], S.shape[1], _dp(psf), psf.shape[0], _dp(out))
    return out


def corr2d_same(G, psf):
    G = _f64(G); psf = _f64(psf)
    out = np.empty_like(G)
    lib().gmo_corr2d_same(_dp(G), G.shape[0], G.shape[1], _dp(psf), psf.shape[0], _dp(out))
    return out


# ---- batched calls --------------------------------------------------------
def render(model, params, H, W, psf):
    params = _f64(params)
    B, P = params.shape
    assert P == model["n_par"]
    d = descriptor(model)
    psf, stride, K = _psf_args(psf, B)
    out = np.empty((B, H, W))
    rc = lib().gmo_render(len(d), d.ctypes.data_as(C.POINTER(C.c_int32)), P, B, H, W, K,
                          _dp(psf), stride, _dp(params), _dp(out))
    assert rc == 0, rc
    return out


def loss_grad(model, params, data, sigma, mask, psf, want_jtj=False):
    params = _f64(params); data = _f64(data); sigma = _f64(sigma); mask = _u8(mask)
    B, P = params.shape
    _, H, W = data.shape
    d = descriptor(model)
    psf, stride, K = _psf_args(psf, B)
    chi2 = np.empty(B); grad = np.empty((B, P))
    jtj = np.empty((B, P, P)) if want_jtj else None
    jtr = np.empty((B, P)) if want_jtj else None
    rc = lib().gmo_loss_grad(len(d), d.ctypes.data_as(C.POINTER(C.c_int32)), P, B, H, W, K,
                             _dp(psf), stride, _dp(data), _dp(sigma), _bp(mask), _dp(params),
                             _dp(chi2), _dp(grad), _dp(jtj), _dp(jtr))
    assert rc == 0, rc
    if want_jtj:
        return chi2, grad, jtj, jtr
    return chi2, grad


def covariance_sigma(jtj, free_mask=None):
    """sigma_p = sqrt(diag[(J^T W J)^-1]) over the free parameters.
    jtj [P,P] -> (sigma_p [P], status)."""
    jtj = _f64(jtj)
    P = jtj.shape[0]
    out = np.empty(P)
    fm = _u8(free_mask)
    rc = lib().gmo_covariance_sigma(P, _dp(jtj), _bp(fm), _dp(out))
    return out, rc


def uncertainty(model, params, sigma, mask, psf, free_mask=None):
    """Covariance-matrix uncertainties of every galaxy (Sec. 5.2).
    -> {"sigma_p" [B,P], "status" [B], "jtj" [B,P,P]}"""
    params = _f64(params)
    B, P = params.shape
    zeros = np.zeros_like(_f64(sigma))                    # J = dM/dp does not depend on the data
    _, _, jtj, _ = loss_grad(model, params, zeros, sigma, mask, psf, want_jtj=True)
    sp = np.empty((B, P)); st = np.zeros(B, dtype=np.int32)
    for g in range(B):
        sp[g], st[g] = covariance_sigma(jtj[g], free_mask)
    return {"sigma_p": sp, "status": st, "jtj": jtj}


def adam_step(u, g_u, m, s, t, lr, lr_decay, beta1, beta2, eps, ulo, uhi, free_mask=None):
    """In-place Adam step on float64 arrays u, m, s."""
    P = u.shape[0]
    fm = _u8(free_mask)
    lib().gmo_adam_step(P, _dp(u), _dp(_f64(g_u)), _dp(m), _dp(s), int(t), _dp(_f64(lr)),
                        float(lr_decay), float(beta1), float(beta2), float(eps),
                        _dp(_f64(ulo)), _dp(_f64(uhi)), _bp(fm))


def fit(model, params, data, sigma, mask, psf, opts: dict, want_trace=False):
    """opts: n_iter, beta1, beta2, eps, lr_decay, lr[P], lo[P], hi[P],
    log10_space[P], free_mask[P], tol, patience (same meaning as gm_fit_opts)."""
    params = _f64(params).copy(); data = _f64(data); sigma = _f64(sigma); mask = _u8(mask)
    B, P = params.shape
    _, H, W = data.shape
    d = descriptor(model)
    psf, stride, K = _psf_args(psf, B)
    n_iter = int(opts["n_iter"])
    lr = _f64(opts["lr"]); lo = _f64(opts["lo"]); hi = _f64(opts["hi"])
    lg = _u8(opts.get("log10_space", np.zeros(P)))
    fm = _u8(opts.get("free_mask", np.ones(P)))
    chi2 = np.empty(B); iters = np.zeros(B, dtype=np.int32); status = np.zeros(B, dtype=np.int32)
    trace = np.full((B, n_iter), np.nan) if want_trace else None
    i32p = C.POINTER(C.c_int32)
    rc = lib().gmo_fit(len(d), d.ctypes.data_as(i32p), P, B, H, W, K, _dp(psf), stride,
                       _dp(data), _dp(sigma), _bp(mask), _dp(params), n_iter,
                       float(opts.get("beta1", 0.9)), float(opts.get("beta2", 0.999)),
                       float(opts.get("eps", 1e-8)), float(opts.get("lr_decay", 1.0)),
                       _dp(lr), _dp(lo), _dp(hi), _bp(lg), _bp(fm),
                       float(opts.get("tol", 0.0)), int(opts.get("patience", 10)),
                       _dp(chi2), iters.ctypes.data_as(i32p), status.ctypes.data_as(i32p), _dp(trace))
    assert rc == 0, rc
    out = {"params": params, "chi2": chi2, "iters_used": iters, "status": status}
    if want_trace:
        out["trace"] = trace
    return out


def mix64(z: int) -> int:
    return int(lib().gmo_mix64(C.c_uint64(z & 0xFFFFFFFFFFFFFFFF)))


def bootstrap_counts(seed: int, gid: int, r: int, mask, shape):
    """Multiplicities c[H,W] of resample r of galaxy gid (reading B1)."""
    N = int(np.prod(shape))
    m = None if mask is None else _u8(mask).reshape(-1)
    counts = np.zeros(N, dtype=np.int32)
    n_used = lib().gmo_bootstrap_counts(C.c_uint64(seed), C.c_uint64(gid), C.c_uint64(r), _bp(m), N,
                                        counts.ctypes.data_as(C.POINTER(C.c_int32)))
    return counts.reshape(shape), int(n_used)


def bootstrap(model, params, data, sigma, mask, psf, opts: dict, n_resample: int, seed: int, id_offset: int = 0):
    """Bootstrap uncertainties (Sec. 5.2): n_resample refits from `params`, each on
    pixels resampled with replacement (weights c / sigma^2, pixels with c = 0 ignored);
    sigma_boot^2 = (1/M) sum (m_i - mean)^2.
    -> {"sigma_boot" [B,P], "mean" [B,P], "samples" [M,B,P], "counts" [B,H,W] of the last resample}"""
    params = _f64(params); data = _f64(data); sigma = _f64(sigma)
    B, P = params.shape
    _, H, W = data.shape
    samples = np.empty((n_resample, B, P))
    counts = np.zeros((B, H, W), dtype=np.int32)
    for r in range(n_resample):
        for g in range(B):
            counts[g], _ = bootstrap_counts(seed, id_offset + g, r, None if mask is None else mask[g], (H, W))
        used = counts > 0
        sig_r = np.where(used, sigma / np.sqrt(np.maximum(counts, 1)), sigma)     # w = c / sigma^2
        samples[r] = fit(model, params, data, sig_r, used.astype(np.uint8), psf, opts)["params"]
    mean = samples.mean(axis=0)
    return {"sigma_boot": np.sqrt(((samples - mean) ** 2).sum(axis=0) / n_resample), "mean": mean,
            "samples": samples, "counts": counts}


def num_threads() -> int:
    return lib().gmo_num_threads()


def set_num_threads(n: int) -> None:
    lib().gmo_set_num_threads(int(n))
