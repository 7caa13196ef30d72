#!/usr/bin/env python
"""Writes the fit-parity table of the round (profiles/r02_parity.md) to stdout.

    python tests/parity_report.py > gpurun_out/r02_parity.md      (on a B200, through gpurun)

Test-side script: it calls only ``oracle/`` (the fp64 fits) and the binding (gm_fit,
gm_fit_multi), on the seeded inputs of gen/configs.py, with the judging functions of
tests/fit_parity.py -- the same ones the -m gpu tests assert with."""
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT)); sys.path.insert(0, str(ROOT / "tests"))

import fit_parity as fp  # noqa: E402


def rows_for(name, b, opts, g, o, dt):
    j = fp.judge(b, g, o)
    model = b["model"]
    lines = []
    B = len(b["galaxies"])
    hdr = (f"### {name}: {B} galaxies, {b['H']}x{b['W']}, K = {b['K']}, P = {model['n_par']}, "
           f"n_iter = {opts['n_iter']}" + (f", tol = {opts['tol']:g}, patience = {opts['patience']}" if opts["tol"] > 0 else "") +
           (", 10 % masked" if b["mask"] is not None else ""))
    lines.append(hdr)
    lines.append("")
    lines.append("| parameter | pass rate at 1e-3 | median rel. deviation | max rel. deviation |")
    lines.append("|---|---|---|---|")
    for k, nm in enumerate(model["names"]):
        lines.append(f"| {nm} | {j['ok'][:, k].mean():.3f} | {np.median(j['dev'][:, k]):.2e} | {j['dev'][:, k].max():.2e} |")
    lines.append(f"| **all** | **{j['ok'].mean():.4f}** | {np.median(j['dev']):.2e} | {j['dev'].max():.2e} |")
    lines.append("")
    nm = len(j["miss"])
    lines.append(f"Galaxies with every parameter inside 1e-3: {B - nm} of {B}.  chi^2 of the fit, GPU against oracle: "
                 f"max relative difference {j['chi2_rel'].max():.2e}.  Status equal: {j['status_equal']}; "
                 f"iterations GPU {j['iters_gpu'].min()}..{j['iters_gpu'].max()} (mean {j['iters_gpu'].mean():.1f}), "
                 f"oracle {j['iters_orc'].min()}..{j['iters_orc'].max()} (mean {j['iters_orc'].mean():.1f}); "
                 f"max |difference| {np.abs(j['iters_gpu'] - j['iters_orc']).max()}.  Oracle fit took {dt:.1f} s.")
    if nm:
        lines.append("")
        lines.append(f"The {nm} galaxies that miss 1e-3 somewhere, judged by the oracle at both end points "
                     f"(same fit = chi^2 within {fp.CHI2_RTOL:g} and image within {fp.IMG_SIGMA_TOL:g} sigma per pixel): "
                     f"**{int(j['miss_valid'].sum())} of {nm} are the same fit**; worst d chi^2 / chi^2 = "
                     f"{j['miss_dchi2'].max():.2e}, worst max-pixel |dM| / sigma = {j['miss_dimg_sigma'].max():.2e}.")
    lines.append("")
    return lines, j


def main():
    out = ["# Round 2 -- fit parity, gm_fit / gm_fit_multi against oracle.fit (fp64), per configuration",
           "",
           "Written by `python tests/parity_report.py` on a B200 (through `gpurun`); the same judging code as",
           "`tests/test_gpu_fit_configs.py`.  Criterion: fitted parameters within 1e-3 relative of the oracle's",
           "(theta modulo pi, skipped where q > 0.95, reading M1).  Galaxies that miss it are re-evaluated BY THE",
           "ORACLE at both end points: chi^2 must agree to 1e-5 and the model images to 0.05 sigma on every used pixel.",
           ""]
    t0 = time.time()
    b, opts = fp.case_c0()
    g = fp.gpu_fit(b, opts); o = fp.oracle_fit(b, opts); dt = time.time() - t0
    out += rows_for("C0 shapes, 150 iterations", b, opts, g, o, dt)[0]

    t0 = time.time()
    b, opts = fp.case_c1(list(range(0, 1024, 16)))
    g = fp.gpu_fit(b, opts); o = fp.oracle_fit(b, opts); dt = time.time() - t0
    out += rows_for("C1 (64-galaxy sample of the 1,024)", b, opts, g, o, dt)[0]

    out += ["## C2: early stop (tol 1e-6, patience 10, cap 500), 10 % masked, all five buckets in one gm_fit_multi call",
            "",
            "The stop rule compares |chi2_t - chi2_(t-1)| with 1e-6 chi2_t, the resolution of an fp32 chi^2, so the iteration",
            "at which it fires is not unique between the fp32 and the fp64 evaluation (reading O5) while the parameters still",
            "drift along the flat valley.  Each bucket is therefore compared twice: (a) with the oracle's trajectory read at the",
            "iteration where the GPU stopped each galaxy (equal update counts: this is the parameter parity), and (b) with the",
            "oracle's own early-stop run (status, iteration counts, and how far apart the two end points are).",
            ""]
    buckets = fp.case_c2(range(120))
    gs = fp.gpu_fit_multi(buckets)
    for (b, opts), g in zip(buckets, gs):
        t0 = time.time()
        o = fp.oracle_fit_at_iters(b, opts, g["iters_used"]); dt = time.time() - t0
        out += rows_for(f"C2, {b['H']} px bucket (a) oracle at the GPU's iteration counts", b, opts, g, o, dt)[0]
        t0 = time.time()
        o = fp.oracle_fit(b, opts, want_trace=True); dt = time.time() - t0
        ok, dtv = fp.stop_decision_ok(g, o, opts)
        out += rows_for(f"C2, {b['H']} px bucket (b) oracle with its own early stop", b, opts, g, o, dt)[0]
        out += [f"Every GPU stop that came before the oracle's happened where the oracle's chi^2 moved by less than "
                f"{fp.STOP_SLACK:g} tol per iteration over the patience window: {ok} (largest difference of the stopping "
                f"iteration {int(dtv.max())}).", ""]

    t0 = time.time()
    b, opts = fp.case_c3(32, 300)
    g = fp.gpu_fit(b, opts); o = fp.oracle_fit(b, opts); dt = time.time() - t0
    out += rows_for("C3 (first 32 galaxies, the full 300 iterations)", b, opts, g, o, dt)[0]

    t0 = time.time()
    b, opts = fp.case_c4(8, 60)
    g = fp.gpu_fit(b, opts); o = fp.oracle_fit(b, opts); dt = time.time() - t0
    out += rows_for("C4 model and shapes (first 8 galaxies, 60 iterations)", b, opts, g, o, dt)[0]
    print("\n".join(out))


if __name__ == "__main__":
    main()
