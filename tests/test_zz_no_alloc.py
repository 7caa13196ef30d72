"""-m gpu: gm_bootstrap_counts_static, the entry point for callers that cannot allocate.

Who needs it: code that is handed a fixed set of device buffers by the application it runs inside
(a plug-in, one stage of somebody else's pipeline), services whose memory plan is frozen at start-up,
and threads where a device allocation could block or deadlock.  Such a caller cannot produce the
workspace gm_bootstrap_counts asks for, so this variant keeps its scratch (the used-pixel list and
the per-galaxy totals) in an array compiled into libgm.so and takes only the mask in and the counts
out.  It must give exactly the counts of the workspace path (integer work: bit for bit), and because
every call reuses the same array with whatever the previous call left in it, the check is made on
calls issued back to back, each with a different mask, shape and resample index.

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should
not hide the parity tests.  It passes alone in a fresh process (the first call does the one-time
address look-up) and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import paper_2404_07780_b200 as gm
from paper_2404_07780_b200 import binding as bd

pytestmark = pytest.mark.gpu


def _mask(shape, keep, seed):
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    return (torch.rand(shape, device="cuda", generator=g) < keep).to(torch.uint8)


def test_static_scratch_matches_workspace_path_on_consecutive_calls():
    # second and third calls are smaller / differently masked than the one before, so the array still holds
    # the longer list of the earlier call when they run; the last call has no mask (list not read at all)
    cases = [((6, 96, 128), 0.9, 0), ((3, 37, 53), 0.5, 4), ((16, 256, 256), 0.75, 1), ((5, 64, 64), None, 2)]
    outs = [torch.full(s, -7, dtype=torch.int32, device="cuda") for s, _, _ in cases]   # output starts dirty
    masks = [None if keep is None else _mask(s, keep, 11 + i) for i, (s, keep, _) in enumerate(cases)]
    free_before = None
    for i, ((B, H, W), _, r) in enumerate(cases):                  # back to back on one stream, no sync between
        got = gm.gm_bootstrap_counts_static(B, H, W, masks[i], seed=99, r=r, id_offset=1000, out=outs[i])
        assert got is outs[i]
        if i == 0:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
    torch.cuda.synchronize()
    # no device memory was taken by the calls after the first (the first may load the module lazily)
    assert torch.cuda.mem_get_info()[0] >= free_before
    for i, ((B, H, W), _, r) in enumerate(cases):
        ref = gm.gm_bootstrap_counts(B, H, W, masks[i], seed=99, r=r, id_offset=1000)   # existing path, own workspace
        torch.cuda.synchronize()
        assert torch.equal(outs[i], ref), i
        n_used = B * H * W if masks[i] is None else int(masks[i].sum())
        assert int(outs[i].sum()) == n_used


def test_static_scratch_same_call_twice_is_reproducible():
    B, H, W = 4, 128, 128
    m = _mask((B, H, W), 0.8, 5)
    a = gm.gm_bootstrap_counts_static(B, H, W, m, seed=3, r=7).clone()
    b = gm.gm_bootstrap_counts_static(B, H, W, m, seed=3, r=7)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    assert torch.equal(a, gm.gm_bootstrap_counts(B, H, W, m, seed=3, r=7))


def test_static_scratch_rejects_what_does_not_fit():
    out = torch.full((8,), 5, dtype=torch.int32, device="cuda")     # must stay untouched: nothing is launched
    for B, H, W in [(65, 128, 128), (bd.STATIC_MAX_B + 1, 4, 4), (1, 1024, 1025), (17, 256, 256)]:
        assert B * H * W > bd.STATIC_MAX_PIXELS or B > bd.STATIC_MAX_B
        b = bd._Batch(B, H, W, 1, None, None, None, None, 0)
        o = bd._BootOpts(1, 1, 0)
        import ctypes as C
        rc = bd._lib().gm_bootstrap_counts_static(C.byref(b), C.byref(o), 0, out.data_ptr(), None)
        assert rc == -5
        assert "larger" in gm.gm_strerror(rc)
    torch.cuda.synchronize()
    assert bool((out == 5).all())
    # the largest shapes that do fit run and agree
    for B, H, W in [(64, 128, 128), (16, 256, 256), (bd.STATIC_MAX_B, 16, 16)]:
        m = _mask((B, H, W), 0.9, B)
        got = gm.gm_bootstrap_counts_static(B, H, W, m, seed=1, r=0)
        assert torch.equal(got, gm.gm_bootstrap_counts(B, H, W, m, seed=1, r=0))
