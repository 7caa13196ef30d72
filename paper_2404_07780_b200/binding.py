"""ctypes binding of libgm.so: same names as the C entry points of include/gm.h.

Only marshals arguments (torch tensors -> device pointers, dict model ->
gm_component array).  There is NO fallback: a missing library, a missing CUDA
device or a non-zero status raises.

A model is plain data (see gen.models / include/gm.h gm_component):
``{"n_par": P, "components": [{"kind": "sersic", "convolve": 1,
"slots": {"xc": 0, "yc": 1, "amp": 2, "s0": 3, "s1": 4, "q": 5, "theta": 6}}]}``.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libgm.so"

GM_MAX_COMP, GM_MAX_PAR, GM_MAX_K, GM_NSLOT = 8, 32, 41, 10
GM_OPT_FUSED, GM_OPT_CONST_TAPS, GM_OPT_TENSOR = 0, 1, 2
GM_CONV_FFMA2, GM_CONV_TENSOR = 0, 1
_KINDS = {"sersic": 0, "expdisk": 1, "ferrer": 2, "king": 3, "gaussian": 4, "moffat": 5, "sky": 6}
_SLOTS = ("xc", "yc", "theta", "q", "amp", "s0", "s1", "s2", "box", "m0")


class GmError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = _lib().gm_strerror(status).decode()
        if status == -3:
            msg += ": " + _lib().gm_last_cuda_error_string().decode()
        super().__init__(f"{where} failed with status {status} ({msg})")


class _Component(C.Structure):
    _fields_ = [("kind", C.c_int32), ("convolve", C.c_int32), ("slot", C.c_int32 * GM_NSLOT)]


class _Model(C.Structure):
    _fields_ = [("n_comp", C.c_int32), ("n_par", C.c_int32), ("comp", C.POINTER(_Component))]


class _Batch(C.Structure):
    _fields_ = [("B", C.c_int32), ("H", C.c_int32), ("W", C.c_int32), ("K", C.c_int32),
                ("data", C.c_void_p), ("sigma", C.c_void_p), ("mask", C.c_void_p),
                ("psf", C.c_void_p), ("psf_stride", C.c_int64)]


class _BootOpts(C.Structure):
    _fields_ = [("n_resample", C.c_int32), ("seed", C.c_uint64), ("id_offset", C.c_uint64)]


class _FitOpts(C.Structure):
    _fields_ = [("n_iter", C.c_int32), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float),
                ("lr_decay", C.c_float), ("lr", C.c_void_p), ("lo", C.c_void_p), ("hi", C.c_void_p),
                ("log10_space", C.c_void_p), ("free_mask", C.c_void_p), ("tol", C.c_float),
                ("patience", C.c_int32)]


_handle = None


def library_path() -> Path:
    return _LIB_PATH


def _lib():
    global _handle
    if _handle is None:
        if not _LIB_PATH.exists():
            raise ImportError(
                f"{_LIB_PATH} is missing: build the CUDA extension first "
                "(python -m paper_2404_07780_b200.build, or __graft_entry__.build()); "
                "there is no CPU fallback")
        L = C.CDLL(str(_LIB_PATH))
        vp, sz, i = C.c_void_p, C.c_size_t, C.c_int
        mp, bp, op = C.POINTER(_Model), C.POINTER(_Batch), C.POINTER(_FitOpts)
        L.gm_workspace_bytes.restype = sz; L.gm_workspace_bytes.argtypes = [mp, bp]
        L.gm_render.restype = i; L.gm_render.argtypes = [mp, bp, vp, vp, vp, sz, vp]
        L.gm_loss_grad.restype = i; L.gm_loss_grad.argtypes = [mp, bp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.gm_fit.restype = i; L.gm_fit.argtypes = [mp, bp, vp, op, vp, vp, vp, vp, sz, vp]
        pp = C.POINTER(C.c_void_p)
        L.gm_fit_multi.restype = i
        L.gm_fit_multi.argtypes = [mp, C.c_int32, bp, pp, op, pp, pp, pp, pp, C.POINTER(sz), pp]
        L.gm_fit_multi_host.restype = i
        L.gm_fit_multi_host.argtypes = [mp, C.c_int32, bp, pp, op, pp, pp, pp]
        bo = C.POINTER(_BootOpts)
        L.gm_bootstrap_workspace_bytes.restype = sz; L.gm_bootstrap_workspace_bytes.argtypes = [mp, bp, C.c_int32]
        L.gm_bootstrap_counts.restype = i; L.gm_bootstrap_counts.argtypes = [bp, bo, C.c_int32, vp, vp, sz, vp]
        L.gm_bootstrap_counts_static.restype = i
        L.gm_bootstrap_counts_static.argtypes = [bp, bo, C.c_int32, vp, vp]
        L.gm_bootstrap.restype = i; L.gm_bootstrap.argtypes = [mp, bp, vp, op, bo, vp, vp, vp, vp, sz, vp]
        L.gm_uncertainty_workspace_bytes.restype = sz; L.gm_uncertainty_workspace_bytes.argtypes = [mp, bp]
        L.gm_uncertainty.restype = i; L.gm_uncertainty.argtypes = [mp, bp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.gm_render_host.restype = i; L.gm_render_host.argtypes = [mp, bp, vp, vp]
        L.gm_loss_grad_host.restype = i; L.gm_loss_grad_host.argtypes = [mp, bp, vp, vp, vp]
        L.gm_fit_host.restype = i; L.gm_fit_host.argtypes = [mp, bp, vp, op, vp, vp, vp]
        L.gm_loglike.restype = i; L.gm_loglike.argtypes = [C.c_int32, vp, vp, C.c_int32, vp]
        L.gm_strerror.restype = C.c_char_p; L.gm_strerror.argtypes = [i]
        L.gm_version.restype = i; L.gm_version.argtypes = []
        L.gm_last_cuda_error.restype = i; L.gm_last_cuda_error.argtypes = []
        L.gm_last_cuda_error_string.restype = C.c_char_p; L.gm_last_cuda_error_string.argtypes = []
        L.gm_last_launch_count.restype = C.c_int64; L.gm_last_launch_count.argtypes = []
        L.gm_conv_workspace_bytes.restype = sz; L.gm_conv_workspace_bytes.argtypes = [i, bp]
        L.gm_conv.restype = i; L.gm_conv.argtypes = [i, i, bp, vp, vp, sz, vp]
        L.gm_init.restype = i; L.gm_init.argtypes = [vp]
        L.gm_set_option.restype = i; L.gm_set_option.argtypes = [i, i]
        L.gm_get_option.restype = i; L.gm_get_option.argtypes = [i]
        L.gm_measure_fp32_peak.restype = i
        L.gm_trace_set.restype = i; L.gm_trace_set.argtypes = [vp]
        L.gm_measure_fp32_peak.argtypes = [i, C.POINTER(C.c_double), vp]
        L.gm_profile_enable.restype = i; L.gm_profile_enable.argtypes = [i]
        L.gm_profile_read.restype = i
        L.gm_profile_read.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        _handle = L
    return _handle


# ---- marshalling ---------------------------------------------------------------
def _model_struct(model: dict):
    comps = model["components"]
    arr = (_Component * len(comps))()
    for c, comp in enumerate(comps):
        arr[c].kind = _KINDS[comp["kind"]]
        arr[c].convolve = int(comp.get("convolve", 1))
        for k in range(GM_NSLOT):
            arr[c].slot[k] = -1
        for name, idx in comp["slots"].items():
            arr[c].slot[_SLOTS.index(name)] = int(idx)
    m = _Model(len(comps), int(model["n_par"]), arr)
    m._keep = arr
    return m


def _dev(t, dtype, name):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}")
    return t.data_ptr()


def _batch_struct(B, H, W, psf, data=None, sigma=None, mask=None, host=False):
    if host:
        ptr = lambda a: None if a is None else a.ctypes.data
        K = psf.shape[-1]
        shared = psf.ndim == 2
        return _Batch(B, H, W, K, ptr(data), ptr(sigma), ptr(mask), ptr(psf), 0 if shared else K * K)
    K = psf.shape[-1]
    if psf.ndim == 2:
        stride = 0
    else:
        if psf.ndim != 3 or psf.shape[0] != B:
            raise ValueError("per-galaxy psf must be [B,K,K]")
        stride = K * K
    if psf.shape[-2] != K:
        raise ValueError("psf must be square")
    for name, t in (("data", data), ("sigma", sigma), ("mask", mask)):
        if t is not None and tuple(t.shape) != (B, H, W):
            raise ValueError(f"{name} must have shape [B,H,W] = {(B, H, W)}, got {tuple(t.shape)}")
    devs = {t.device for t in (psf, data, sigma, mask) if isinstance(t, torch.Tensor)}
    if len(devs) > 1:
        raise ValueError(f"all tensors of a batch must live on one device, got {sorted(map(str, devs))}")
    return _Batch(B, H, W, K, _dev(data, torch.float32, "data"), _dev(sigma, torch.float32, "sigma"),
                  _dev(mask, torch.uint8, "mask"), _dev(psf, torch.float32, "psf"), stride)


def _on_stream(fn):
    """Run the entry point with `stream` as torch's current stream, so that the tensors it
    allocates (results, a temporary workspace) belong to the stream the kernels run on."""
    import functools

    @functools.wraps(fn)
    def wrapper(*args, **kw):
        stream = kw.get("stream")
        if stream is None:
            return fn(*args, **kw)
        with torch.cuda.stream(stream):
            return fn(*args, **kw)
    return wrapper


def _stream_ptr(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _workspace(m, b, workspace, uncertainty=False):
    fn = _lib().gm_uncertainty_workspace_bytes if uncertainty else _lib().gm_workspace_bytes
    need = fn(C.byref(m), C.byref(b))
    if need == 0:
        raise GmError(-1, "gm_workspace_bytes")
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    off = (-workspace.data_ptr()) % 256
    return workspace, workspace.data_ptr() + off, workspace.numel() - off


def _check(rc, where):
    if rc != 0:
        raise GmError(rc, where)


def _opts_struct(opts: dict, P: int):
    lr = np.ascontiguousarray(opts["lr"], dtype=np.float32)
    lo = np.ascontiguousarray(opts["lo"], dtype=np.float32)
    hi = np.ascontiguousarray(opts["hi"], dtype=np.float32)
    lg = np.ascontiguousarray(opts.get("log10_space", np.zeros(P)), dtype=np.uint8)
    fm = np.ascontiguousarray(opts.get("free_mask", np.ones(P)), dtype=np.uint8)
    for a in (lr, lo, hi, lg, fm):
        if a.shape != (P,):
            raise ValueError("fit option arrays must have n_par entries")
    o = _FitOpts(int(opts["n_iter"]), float(opts.get("beta1", 0.9)), float(opts.get("beta2", 0.999)),
                 float(opts.get("eps", 1e-8)), float(opts.get("lr_decay", 1.0)), lr.ctypes.data,
                 lo.ctypes.data, hi.ctypes.data, lg.ctypes.data, fm.ctypes.data,
                 float(opts.get("tol", 0.0)), int(opts.get("patience", 10)))
    o._keep = (lr, lo, hi, lg, fm)
    return o


# ---- entry points (same names as include/gm.h) ---------------------------------
def gm_version() -> int:
    return _lib().gm_version()


def gm_loglike(chi2, n_used, n_free: int):
    """ln L of Eq. 17 per galaxy, k = n_used - n_free.  Host helper: chi2 [B] (numpy or a
    tensor, copied to the host), n_used [B] int; returns float64 numpy [B] (NaN where k < 1 or chi2 <= 0)."""
    c = np.ascontiguousarray(chi2.detach().cpu().numpy() if isinstance(chi2, torch.Tensor) else chi2, dtype=np.float32)
    n = np.ascontiguousarray(n_used.detach().cpu().numpy() if isinstance(n_used, torch.Tensor) else n_used, dtype=np.int32)
    if c.ndim != 1 or n.shape != c.shape:
        raise ValueError("chi2 and n_used: one entry per galaxy")
    out = np.empty(c.shape[0], dtype=np.float64)
    _check(_lib().gm_loglike(c.shape[0], c.ctypes.data, n.ctypes.data, int(n_free), out.ctypes.data), "gm_loglike")
    return out


def gm_strerror(status: int) -> str:
    return _lib().gm_strerror(int(status)).decode()


def gm_last_launch_count() -> int:
    return int(_lib().gm_last_launch_count())


def gm_init(stream=None) -> None:
    """Build the per-device tables now (asynchronous on the stream); optional."""
    _check(_lib().gm_init(_stream_ptr(stream)), "gm_init")


def gm_set_option(option: int, value: int) -> None:
    _check(_lib().gm_set_option(int(option), int(value)), "gm_set_option")


def gm_get_option(option: int) -> int:
    return int(_lib().gm_get_option(int(option)))


TRACE_ROLES, TRACE_CAP = 3, 2048                      # GM_TRACE_ROLES, GM_TRACE_CAP


def gm_trace_set(buf) -> None:
    """Phase trace of k_tc_fused into `buf` (int64 CUDA tensor of TRACE_ROLES * TRACE_CAP zeros), or None: off."""
    if buf is not None and (not buf.is_cuda or buf.dtype != torch.int64 or buf.numel() < TRACE_ROLES * TRACE_CAP):
        raise ValueError("gm_trace_set: int64 CUDA tensor of TRACE_ROLES * TRACE_CAP elements")
    _check(_lib().gm_trace_set(None if buf is None else C.c_void_p(buf.data_ptr())), "gm_trace_set")


def gm_measure_fp32_peak(repeats: int = 20, stream=None) -> float:
    """Measured FP32 peak in TFLOP/s (a pure fma.rn.f32x2 kernel, CUDA events)."""
    v = C.c_double()
    _check(_lib().gm_measure_fp32_peak(int(repeats), C.byref(v), _stream_ptr(stream)), "gm_measure_fp32_peak")
    return float(v.value)


def gm_profile_enable(on: bool) -> None:
    _check(_lib().gm_profile_enable(1 if on else 0), "gm_profile_enable")


PROF_KINDS = ("forward", "backward", "fused", "tc_forward", "tc_backward", "tc_fused")   # GM_PROF_*


def gm_profile_read():
    """-> {kind: (ms, launches)} since the last read; kinds as GM_PROF_* of include/gm.h."""
    ms = (C.c_double * len(PROF_KINDS))(); n = (C.c_int64 * len(PROF_KINDS))()
    _check(_lib().gm_profile_read(ms, n), "gm_profile_read")
    return {name: (ms[i], int(n[i])) for i, name in enumerate(PROF_KINDS)}


def gm_workspace_bytes(model: dict, B: int, H: int, W: int, K: int, per_galaxy_psf: bool = False) -> int:
    m = _model_struct(model)
    b = _Batch(B, H, W, K, None, None, None, None, K * K if per_galaxy_psf else 0)
    return int(_lib().gm_workspace_bytes(C.byref(m), C.byref(b)))


@_on_stream
def gm_render(model, params, H, W, psf, out=None, workspace=None, stream=None):
    """M[B,H,W] for params[B,P].  Asynchronous on the stream."""
    B = params.shape[0]
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf)
    if out is None:
        out = torch.empty((B, H, W), dtype=torch.float32, device=params.device)
    ws, wp, wn = _workspace(m, b, workspace)
    rc = _lib().gm_render(C.byref(m), C.byref(b), _dev(params, torch.float32, "params"),
                          _dev(out, torch.float32, "out"), wp, wn, _stream_ptr(stream))
    _check(rc, "gm_render")
    out._gm_ws = ws
    return out


@_on_stream
def gm_conv(image, psf, engine=GM_CONV_FFMA2, adjoint=False, out=None, workspace=None, stream=None):
    """out[B,H,W] = psf (*) image (true convolution, zero fill, same size; adjoint: correlation) with the
    FFMA2 loop or on the tensor cores (include/gm.h gm_conv).  Asynchronous on the stream."""
    B, H, W = image.shape
    b = _batch_struct(B, H, W, psf, data=image)
    need = _lib().gm_conv_workspace_bytes(int(engine), C.byref(b))
    if need == 0:
        raise GmError(-2, "gm_conv_workspace_bytes")
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=image.device)
    off = (-workspace.data_ptr()) % 256
    if out is None:
        out = torch.empty_like(image)
    rc = _lib().gm_conv(int(engine), int(bool(adjoint)), C.byref(b), _dev(out, torch.float32, "out"),
                        workspace.data_ptr() + off, workspace.numel() - off, _stream_ptr(stream))
    _check(rc, "gm_conv")
    out._gm_ws = workspace
    return out


@_on_stream
def gm_loss_grad(model, params, data, sigma, mask, psf, want_grad=True, chi2=None, grad=None,
                 workspace=None, stream=None, want_jtj=False):
    """chi^2[B] (Eq. 18) and d chi^2 / d p [B,P].  Asynchronous on the stream.
    want_jtj: also J^T W J [B,P,P] and J^T W (D-M) [B,P]; returns 4 tensors."""
    B, P = params.shape
    _, H, W = data.shape
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, data, sigma, mask)
    if chi2 is None:
        chi2 = torch.empty(B, dtype=torch.float32, device=params.device)
    if want_grad and grad is None:
        grad = torch.empty((B, P), dtype=torch.float32, device=params.device)
    jtj = torch.empty((B, P, P), dtype=torch.float32, device=params.device) if want_jtj else None
    jtr = torch.empty((B, P), dtype=torch.float32, device=params.device) if want_jtj else None
    ws, wp, wn = _workspace(m, b, workspace, uncertainty=want_jtj)
    rc = _lib().gm_loss_grad(C.byref(m), C.byref(b), _dev(params, torch.float32, "params"),
                             _dev(chi2, torch.float32, "chi2"),
                             _dev(grad, torch.float32, "grad") if want_grad else None,
                             _dev(jtj, torch.float32, "jtj"), _dev(jtr, torch.float32, "jtr"),
                             wp, wn, _stream_ptr(stream))
    _check(rc, "gm_loss_grad")
    chi2._gm_ws = ws
    if want_jtj:
        return chi2, grad, jtj, jtr
    return (chi2, grad) if want_grad else chi2


def gm_uncertainty_workspace_bytes(model: dict, B: int, H: int, W: int, K: int) -> int:
    m = _model_struct(model)
    b = _Batch(B, H, W, K, None, None, None, None, 0)
    return int(_lib().gm_uncertainty_workspace_bytes(C.byref(m), C.byref(b)))


@_on_stream
def gm_uncertainty(model, params, sigma, mask, psf, free_mask=None, want_jtj=False, workspace=None,
                   stream=None):
    """sigma_p[B,P] = sqrt(diag[(J^T W J)^-1]) at params (Sec. 5.2).  Asynchronous.
    -> {"sigma_p", "status", ["jtj"]}"""
    B, P = params.shape
    _, H, W = sigma.shape
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, None, sigma, mask)
    fm = None
    if free_mask is not None:
        fm = np.ascontiguousarray(free_mask, dtype=np.uint8)
        if fm.shape != (P,):
            raise ValueError("free_mask must have n_par entries")
    sp = torch.empty((B, P), dtype=torch.float32, device=params.device)
    status = torch.empty(B, dtype=torch.int32, device=params.device)
    jtj = torch.empty((B, P, P), dtype=torch.float32, device=params.device) if want_jtj else None
    ws, wp, wn = _workspace(m, b, workspace, uncertainty=True)
    rc = _lib().gm_uncertainty(C.byref(m), C.byref(b), _dev(params, torch.float32, "params"),
                               None if fm is None else fm.ctypes.data, sp.data_ptr(),
                               _dev(jtj, torch.float32, "jtj"), status.data_ptr(), wp, wn, _stream_ptr(stream))
    _check(rc, "gm_uncertainty")
    out = {"sigma_p": sp, "status": status, "_ws": ws}
    if want_jtj:
        out["jtj"] = jtj
    return out


@_on_stream
def gm_fit(model, params, data, sigma, mask, psf, opts, workspace=None, stream=None):
    """Batched fixed-iteration fit; params[B,P] is updated IN PLACE.  Asynchronous."""
    B, P = params.shape
    _, H, W = data.shape
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, data, sigma, mask)
    o = _opts_struct(opts, P)
    chi2 = torch.empty(B, dtype=torch.float32, device=params.device)
    iters = torch.empty(B, dtype=torch.int32, device=params.device)
    status = torch.empty(B, dtype=torch.int32, device=params.device)
    ws, wp, wn = _workspace(m, b, workspace)
    rc = _lib().gm_fit(C.byref(m), C.byref(b), _dev(params, torch.float32, "params"), C.byref(o),
                       chi2.data_ptr(), iters.data_ptr(), status.data_ptr(), wp, wn, _stream_ptr(stream))
    _check(rc, "gm_fit")
    return {"params": params, "chi2": chi2, "iters_used": iters, "status": status, "_ws": ws}


@_on_stream
def gm_bootstrap_counts(B, H, W, mask, seed, r, id_offset=0, stream=None):
    """int32 multiplicities [B,H,W] of bootstrap resample r (reading B1).  Asynchronous."""
    dev = mask.device if mask is not None else torch.device("cuda")
    b = _Batch(B, H, W, 1, None, None, _dev(mask, torch.uint8, "mask"), None, 0)
    o = _BootOpts(1, int(seed), int(id_offset))
    counts = torch.empty((B, H, W), dtype=torch.int32, device=dev)
    ws = torch.empty(4 * B * (H * W + 1) + 1024, dtype=torch.uint8, device=dev)
    off = (-ws.data_ptr()) % 256
    rc = _lib().gm_bootstrap_counts(C.byref(b), C.byref(o), int(r), counts.data_ptr(), ws.data_ptr() + off,
                                    ws.numel() - off, _stream_ptr(stream))
    _check(rc, "gm_bootstrap_counts")
    counts._gm_ws = ws
    return counts


STATIC_MAX_PIXELS, STATIC_MAX_B = 1 << 20, 4096       # GM_STATIC_MAX_PIXELS, GM_STATIC_MAX_B


@_on_stream
def gm_bootstrap_counts_static(B, H, W, mask, seed, r, id_offset=0, out=None, stream=None):
    """gm_bootstrap_counts without a workspace, for callers that may not allocate device memory
    (plug-ins given fixed buffers, services with a memory plan fixed at start-up, threads where an
    allocation could deadlock).  The scratch is an array built into libgm.so, so B <= STATIC_MAX_B and
    B*H*W <= STATIC_MAX_PIXELS, else GmError(GM_ETOOLARGE).  Pass `out` (int32 CUDA tensor [B,H,W]) and
    this wrapper allocates nothing either; without it the result tensor comes from torch.  Calls share
    the one array: keep them on one stream (or ordered by events), never overlapping.  Make the first
    call on a device during set-up, before any stream capture.  Asynchronous."""
    dev = mask.device if mask is not None else (out.device if out is not None else torch.device("cuda"))
    b = _Batch(B, H, W, 1, None, None, _dev(mask, torch.uint8, "mask"), None, 0)
    o = _BootOpts(1, int(seed), int(id_offset))
    if out is None:
        out = torch.empty((B, H, W), dtype=torch.int32, device=dev)
    elif (not out.is_cuda or out.dtype != torch.int32 or not out.is_contiguous()
          or tuple(out.shape) != (B, H, W)):
        raise ValueError("out: contiguous int32 CUDA tensor [B,H,W]")
    rc = _lib().gm_bootstrap_counts_static(C.byref(b), C.byref(o), int(r), out.data_ptr(), _stream_ptr(stream))
    _check(rc, "gm_bootstrap_counts_static")
    return out


@_on_stream
def gm_bootstrap(model, params, data, sigma, mask, psf, opts, n_resample, seed, id_offset=0,
                 want_samples=False, workspace=None, stream=None):
    """Bootstrap uncertainties (Sec. 5.2): n_resample refits from params[B,P] (not
    modified).  Asynchronous.  -> {"sigma_boot" [B,P], "mean" [B,P], ["samples" [M,B,P]]}"""
    B, P = params.shape
    _, H, W = data.shape
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, data, sigma, mask)
    o = _opts_struct(opts, P)
    bo = _BootOpts(int(n_resample), int(seed), int(id_offset))
    need = _lib().gm_bootstrap_workspace_bytes(C.byref(m), C.byref(b), int(n_resample))
    if need == 0:
        raise GmError(-1, "gm_bootstrap_workspace_bytes")
    if workspace is None:
        workspace = torch.empty(need + 256, dtype=torch.uint8, device=params.device)
    off = (-workspace.data_ptr()) % 256
    sb = torch.empty((B, P), dtype=torch.float32, device=params.device)
    mean = torch.empty((B, P), dtype=torch.float32, device=params.device)
    smp = torch.empty((n_resample, B, P), dtype=torch.float32, device=params.device) if want_samples else None
    rc = _lib().gm_bootstrap(C.byref(m), C.byref(b), _dev(params, torch.float32, "params"), C.byref(o),
                             C.byref(bo), sb.data_ptr(), mean.data_ptr(), None if smp is None else smp.data_ptr(),
                             workspace.data_ptr() + off, workspace.numel() - off, _stream_ptr(stream))
    _check(rc, "gm_bootstrap")
    out = {"sigma_boot": sb, "mean": mean, "_ws": workspace}
    if want_samples:
        out["samples"] = smp
    return out


def gm_fit_multi(model, batches, streams=None):
    """gm_fit of several size buckets at once, batch i on streams[i] (mixed cutout
    sizes).  batches: list of dicts {"params", "data", "sigma", "mask", "psf", "opts",
    ["workspace"]}; params are updated IN PLACE.  streams: list of torch.cuda.Stream
    (default: one new stream per batch, each made to wait for the current stream; the
    current stream then waits for all of them, so the call orders like gm_fit).
    Asynchronous.  -> list of result dicts like gm_fit's."""
    n = len(batches)
    m = _model_struct(model)
    own = streams is None
    cur = torch.cuda.current_stream()
    if own:
        streams = [torch.cuda.Stream() for _ in range(n)]
        ev = torch.cuda.Event(); ev.record(cur)
        for s in streams:
            s.wait_event(ev)
    if len(streams) != n:
        raise ValueError("one stream per batch")
    barr = (_Batch * n)(); oarr = (_FitOpts * n)()
    vpa = lambda: (C.c_void_p * n)()
    par, chi, its, sts, wsp, stp = vpa(), vpa(), vpa(), vpa(), vpa(), vpa()
    wsn = (C.c_size_t * n)()
    keep, outs = [], []
    for k, bt in enumerate(batches):
        params = bt["params"]
        B, P = params.shape
        _, H, W = bt["data"].shape
        barr[k] = _batch_struct(B, H, W, bt["psf"], bt["data"], bt["sigma"], bt.get("mask"))
        o = _opts_struct(bt["opts"], P)
        oarr[k] = o
        chi2 = torch.empty(B, dtype=torch.float32, device=params.device)
        iters = torch.empty(B, dtype=torch.int32, device=params.device)
        status = torch.empty(B, dtype=torch.int32, device=params.device)
        ws, wp, wn = _workspace(m, barr[k], bt.get("workspace"))
        par[k] = _dev(params, torch.float32, "params"); chi[k] = chi2.data_ptr()
        its[k] = iters.data_ptr(); sts[k] = status.data_ptr(); wsp[k] = wp; wsn[k] = wn
        stp[k] = streams[k].cuda_stream
        keep.append(o)
        outs.append({"params": params, "chi2": chi2, "iters_used": iters, "status": status, "_ws": ws})
    rc = _lib().gm_fit_multi(C.byref(m), n, barr, par, oarr, chi, its, sts, wsp, wsn, stp)
    _check(rc, "gm_fit_multi")
    if own:
        for s, o in zip(streams, outs):
            e = torch.cuda.Event(); e.record(s)
            cur.wait_event(e)
            for t in (o["params"], o["chi2"], o["iters_used"], o["status"], o["_ws"]):
                t.record_stream(s)
    return outs


# ---- host-buffer entry points (numpy in, numpy out; copies inside the call) ------
def _np(a, dtype, name):
    if a is None:
        return None
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous:
        raise TypeError(f"{name} must be a C-contiguous numpy array of {dtype}")
    return a


def gm_render_host(model, params, H, W, psf):
    params = _np(params, np.float32, "params"); psf = _np(psf, np.float32, "psf")
    B = params.shape[0]
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, host=True)
    out = np.empty((B, H, W), dtype=np.float32)
    _check(_lib().gm_render_host(C.byref(m), C.byref(b), params.ctypes.data, out.ctypes.data), "gm_render_host")
    return out


def gm_loss_grad_host(model, params, data, sigma, mask, psf):
    params = _np(params, np.float32, "params"); psf = _np(psf, np.float32, "psf")
    data = _np(data, np.float32, "data"); sigma = _np(sigma, np.float32, "sigma")
    mask = _np(mask, np.uint8, "mask")
    B, P = params.shape
    _, H, W = data.shape
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, data, sigma, mask, host=True)
    chi2 = np.empty(B, dtype=np.float32); grad = np.empty((B, P), dtype=np.float32)
    _check(_lib().gm_loss_grad_host(C.byref(m), C.byref(b), params.ctypes.data, chi2.ctypes.data,
                                    grad.ctypes.data), "gm_loss_grad_host")
    return chi2, grad


def gm_fit_host(model, params, data, sigma, mask, psf, opts):
    """params (numpy [B,P]) is updated in place; returns dict of numpy arrays."""
    params = _np(params, np.float32, "params"); psf = _np(psf, np.float32, "psf")
    data = _np(data, np.float32, "data"); sigma = _np(sigma, np.float32, "sigma")
    mask = _np(mask, np.uint8, "mask")
    B, P = params.shape
    _, H, W = data.shape
    m = _model_struct(model)
    b = _batch_struct(B, H, W, psf, data, sigma, mask, host=True)
    o = _opts_struct(opts, P)
    chi2 = np.empty(B, dtype=np.float32)
    iters = np.empty(B, dtype=np.int32); status = np.empty(B, dtype=np.int32)
    _check(_lib().gm_fit_host(C.byref(m), C.byref(b), params.ctypes.data, C.byref(o), chi2.ctypes.data,
                              iters.ctypes.data, status.ctypes.data), "gm_fit_host")
    return {"params": params, "chi2": chi2, "iters_used": iters, "status": status}


def gm_fit_multi_host(model, batches):
    """gm_fit_multi with numpy buffers (copies inside the call, every bucket on its own
    stream).  batches: list of dicts {"params", "data", "sigma", "mask", "psf", "opts"};
    params updated in place.  -> list of dicts of numpy arrays."""
    n = len(batches)
    m = _model_struct(model)
    barr = (_Batch * n)(); oarr = (_FitOpts * n)()
    vpa = lambda: (C.c_void_p * n)()
    par, chi, its, sts = vpa(), vpa(), vpa(), vpa()
    keep, outs = [], []
    for k, bt in enumerate(batches):
        params = _np(bt["params"], np.float32, "params"); psf = _np(bt["psf"], np.float32, "psf")
        data = _np(bt["data"], np.float32, "data"); sigma = _np(bt["sigma"], np.float32, "sigma")
        mask = _np(bt.get("mask"), np.uint8, "mask")
        B, P = params.shape
        _, H, W = data.shape
        barr[k] = _batch_struct(B, H, W, psf, data, sigma, mask, host=True)
        o = _opts_struct(bt["opts"], P)
        oarr[k] = o
        chi2 = np.empty(B, dtype=np.float32)
        iters = np.empty(B, dtype=np.int32); status = np.empty(B, dtype=np.int32)
        par[k] = params.ctypes.data; chi[k] = chi2.ctypes.data
        its[k] = iters.ctypes.data; sts[k] = status.ctypes.data
        keep.append(o)
        outs.append({"params": params, "chi2": chi2, "iters_used": iters, "status": status})
    _check(_lib().gm_fit_multi_host(C.byref(m), n, barr, par, oarr, chi, its, sts), "gm_fit_multi_host")
    return outs
