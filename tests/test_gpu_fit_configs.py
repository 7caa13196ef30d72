"""-m gpu: gm_fit / gm_fit_multi against the oracle's fit on the configurations bench.py
times (BASELINE.json C0 ... C4; SURVEY section 4 tier 3).  The criterion is the complete one
of tests/fit_parity.py: every galaxy meets 1e-3 on every parameter, or is shown by the oracle
to be the same fit (chi^2 within 1e-5, model image within 0.05 sigma per pixel); the floors
on the per-parameter pass rate are what profiles/r02_parity.md records, rounded down."""
import numpy as np
import pytest

import fit_parity as fp

pytestmark = pytest.mark.gpu


def _chi2_at_oracle_params_close(j, rtol):
    assert np.all(j["chi2_rel"] <= rtol), f"chi2 of the fit: rel diff max {j['chi2_rel'].max():.3e}"


def test_c0_fixed_150_iterations():
    b, opts = fp.case_c0()
    j = fp.judge(b, fp.gpu_fit(b, opts), fp.oracle_fit(b, opts))
    fp.assert_parity("C0", j, floor=0.99)
    _chi2_at_oracle_params_close(j, 1e-4)


def test_c1_200_iterations_sample():
    sample = list(range(0, 1024, 43))
    b, opts = fp.case_c1(sample)
    j = fp.judge(b, fp.gpu_fit(b, opts), fp.oracle_fit(b, opts))
    fp.assert_parity("C1", j, floor=0.95)
    _chi2_at_oracle_params_close(j, 1e-4)


def test_c2_every_bucket_through_fit_multi_early_stop_masked():
    # mask on, tol 1e-6 / patience 10, cap 500, all five sides in ONE gm_fit_multi call: the
    # 64 / 96 / 128 px buckets run k_fused with the live list, 192 / 256 px the tile kernels.
    # The iteration at which the stop rule fires is not unique at tol = 1e-6 (fit_parity.py), so
    # (1) wherever the GPU stopped earlier than the oracle's own run, the oracle's chi^2 was already flat,
    # (2) the oracle's trajectory read at the GPU's iteration count must be the GPU's parameters.
    buckets = fp.case_c2(range(60))
    assert sorted(b["H"] for b, _ in buckets) == [64, 96, 128, 192, 256]
    outs = fp.gpu_fit_multi(buckets)
    stopped = 0
    for (b, opts), g in zip(buckets, outs):
        assert b["mask"] is not None and opts["tol"] > 0 and opts["n_iter"] == 500
        own = fp.oracle_fit(b, opts, want_trace=True)
        ok, dt = fp.stop_decision_ok(g, own, opts)
        assert ok, f"C2/{b['H']}px: the GPU stopped a galaxy while the oracle's chi^2 still moved; |d iterations| = {dt}"
        # (3) against the oracle's own stop: iteration counts within MAX_STOP_SHIFT, end points the same fit within
        # the looser bounds of fit_parity.py (the two runs legitimately end tens of iterations apart)
        fp.assert_close_to_own_stop(f"C2/{b['H']}px", b, g, own, dt)
        o = fp.oracle_fit_at_iters(b, opts, g["iters_used"])
        j = fp.judge(b, g, o)
        # profiles/r02_parity.md (120-galaxy sample): 0.966 .. 1.000 per bucket; the 8 .. 19 galaxies per bucket of
        # this smaller sample leave 0.91 in the worst one
        fp.assert_parity(f"C2/{b['H']}px", j, floor=0.90)
        _chi2_at_oracle_params_close(j, 1e-4)
        stopped += int((g["status"] == 1).sum())
    assert stopped > 0, "early stop never triggered: the test would not cover the live list"


def test_c3_bulge_disk_128px_k25():
    b, opts = fp.case_c3(16, 100)
    assert b["model"]["n_par"] == 11 and b["H"] == 128 and b["K"] == 25
    j = fp.judge(b, fp.gpu_fit(b, opts), fp.oracle_fit(b, opts))
    fp.assert_parity("C3", j, floor=0.99)
    _chi2_at_oracle_params_close(j, 1e-4)


def test_c4_three_components_256px_k41():
    b, opts = fp.case_c4(4, 30)
    assert b["model"]["n_par"] == 16 and b["H"] == 256 and b["K"] == 41
    j = fp.judge(b, fp.gpu_fit(b, opts), fp.oracle_fit(b, opts))
    fp.assert_parity("C4", j, floor=0.99)
    _chi2_at_oracle_params_close(j, 1e-4)
