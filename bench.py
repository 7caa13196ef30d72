#!/usr/bin/env python
"""bench.py -- throughput of the batched galaxy-fit hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 1|3|...] [--sweep]

One "step" = one pass of the whole hot path over one batch: a full ``gm_fit`` of the
workload (render -> PSF convolution -> chi^2 -> adjoint convolution -> gradient ->
Adam update, n_iter times, plus the closing chi^2 evaluation).  The N=1 workload is
BASELINE.json ``configs[1]`` (C1: 1,024 single-Sersic galaxies, 128x128, 25x25 Moffat
PSF, 200 iterations).  With N>1 every rank fits its own 1,024 galaxies (weak scaling,
no data-path collective: galaxies are independent).

Prints ONE JSON line (rank 0).  metric = galaxy-pixel chi^2+gradient evaluations per
second = B*H*W*n_iter / step time, whole job.  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "galaxy_pixel_chi2_grad_evals_per_s"
UNIT = "pixel-evals/s"
SM_COUNT = 148
FP32_LANES = 128


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        return json.loads(p.read_text()), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *exc):
        self.out = ""
        if self.proc is not None:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.out, _ = self.proc.communicate(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
                self.out, _ = self.proc.communicate()

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in getattr(self, "out", "").splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        busy = [c for c, p in zip(sm, pw) if p > 0.5 * max(pw)] or sm
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": len(sm)}


def workload_name(cfg, B, H, W, K, n_iter):
    return (f"{cfg.name}: {B} galaxies, {cfg.model_name}, {H}x{W} fp32 cutouts, {K}x{K} "
            f"{'Moffat' if cfg.psf_kind.startswith('moffat') else 'Gaussian'} PSF, "
            f"{n_iter}-iteration gm_fit")


# ---------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (the other
    place bench.py may execute oracle/).  Each step is a bounded sample of the same
    workload: `cores` galaxies x a few iterations of C1's shapes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from gen import configs
    cfg = configs.CONFIGS[args.config]
    cores = oracle.num_threads()
    n_gal, n_iter = cores, 3
    side = cfg.sides[len(cfg.sides) // 2]
    cand = list(range(40 * cores))
    gal = [g for g, s in zip(cand, configs.sides_for(cfg, cand)) if s == side][:n_gal]
    b = configs.make_batch(cfg.cid, gal, lambda m, p, H, W, psf: oracle.render(m, p, H, W, psf), side=side)
    n_gal = len(b["galaxies"])
    opts = configs.fit_options(b["model"], b["H"], b["W"], n_iter)

    def step():
        oracle.fit(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"], opts)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    value = n_gal * b["H"] * b["W"] * n_iter / dt
    sample = f"{n_gal} galaxies x {n_iter} iterations of {cfg.name} ({b['H']}x{b['W']}, K={b['K']}) per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg, cfg.B, b["H"], b["W"], b["K"], cfg.n_iter),
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def streamed(k, model, n_batches):
    """BASELINE config C4 is "streamed in batches": n_batches batches through the device-pointer
    C ABI on two streams with two sets of device buffers, so that the host-to-device copy of batch
    i + 1 (from pinned host memory) and the read-back of batch i - 1 overlap the fit of batch i.
    The same synthetic batch is re-sent every time (its bytes cross the bus every time); wall
    clock with a device synchronise on both sides."""
    import torch

    import paper_2404_07780_b200 as gm
    hd, hs, hm, _, hp = k["host"]
    psf = k["dev"][3]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    sets = [{"data": torch.empty_like(k["dev"][0]), "sigma": torch.empty_like(k["dev"][1]),
             "mask": None if hm is None else torch.empty_like(k["dev"][2]),
             "params": torch.empty_like(k["dev"][4]), "ws": torch.empty_like(k["ws"]),
             "back": torch.empty_like(hp).pin_memory()} for _ in streams]

    def run(n):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for i in range(n):
            st, b = streams[i % 2], sets[i % 2]
            with torch.cuda.stream(st):
                b["data"].copy_(hd, non_blocking=True)
                b["sigma"].copy_(hs, non_blocking=True)
                if hm is not None:
                    b["mask"].copy_(hm, non_blocking=True)
                b["params"].copy_(hp, non_blocking=True)
                gm.gm_fit(model, b["params"], b["data"], b["sigma"], b["mask"], psf, k["opts"],
                          workspace=b["ws"], stream=st)
                b["back"].copy_(b["params"], non_blocking=True)
        torch.cuda.synchronize()
        return time.perf_counter() - t0

    run(2)                                                              # warm-up
    sec = run(n_batches)
    B, H, W = k["B"], k["H"], k["W"]
    h2d = hd.numel() * 4 + hs.numel() * 4 + (0 if hm is None else hm.numel()) + hp.numel() * 4
    return {"batches": n_batches, "galaxies": n_batches * B, "seconds": sec,
            "galaxies_fitted_per_s": n_batches * B / sec,
            "value": n_batches * B * H * W * k["opts"]["n_iter"] / sec, "unit": UNIT,
            "h2d_bytes_per_batch": int(h2d), "d2h_bytes_per_batch": int(hp.numel() * 4),
            "how": "two streams, two device buffer sets, H2D / fit / D2H of consecutive batches overlap; "
                   "gm_fit through the device-pointer C ABI; fixed iteration count assumed"}


def cpu_baseline(cfg, side):
    """The oracle timed on the box's host cores on a bounded sample (~10-30 s)."""
    import oracle
    from gen import configs
    cores = oracle.num_threads()
    n_gal = 2 * cores
    cand = list(range(40 * cores))
    gal = [g for g, s in zip(cand, configs.sides_for(cfg, cand)) if s == side][:n_gal]
    b = configs.make_batch(cfg.cid, gal, lambda m, p, H, W, psf: oracle.render(m, p, H, W, psf), side=side)
    n_gal = len(b["galaxies"])
    # size the iteration count from one timed evaluation so the sample takes ~15 s
    t0 = time.perf_counter()
    oracle.loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    t_eval = time.perf_counter() - t0
    n_iter = int(min(max(15.0 / max(t_eval, 1e-3), 2), cfg.n_iter or 200))
    opts = configs.fit_options(b["model"], b["H"], b["W"], n_iter)
    t0 = time.perf_counter()
    oracle.fit(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"], opts)
    dt = time.perf_counter() - t0
    return {"value": n_gal * b["H"] * b["W"] * n_iter / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "galaxies_per_s_at_full_iters": n_gal / (dt * (cfg.n_iter or n_iter) / n_iter),
            "sample": f"{n_gal} galaxies x {n_iter} iterations of {cfg.name} ({b['H']}x{b['W']}, K={b['K']}), "
                      f"{dt:.1f} s, OpenMP over galaxies"}


# ---------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_2404_07780_b200 as gm
    from gen import configs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = configs.CONFIGS[args.config]
    Btot = args.batch or min(cfg.B, 8289)
    n_iter = args.iters or cfg.n_iter or 200
    gal = range(rank * Btot, rank * Btot + Btot)   # weak scaling: every rank its own galaxies

    def render(model, p, H, W, psf):               # truth images from the CUDA path itself
        out = gm.gm_render(model, torch.from_numpy(p).cuda(), H, W, torch.from_numpy(psf).cuda())
        torch.cuda.synchronize()
        return out.cpu().numpy()

    # one bucket per cutout side (C2: five; every other config: one), each its own gm_batch
    pin = lambda a: None if a is None else torch.from_numpy(a).pin_memory()
    d = lambda t: None if t is None else t.cuda(non_blocking=True)
    sides = [args.side] if args.side else list(cfg.sides)
    buckets = []
    for side in sides:
        b = configs.make_batch(cfg.cid, gal, render, side=side)
        if not b["galaxies"]:
            continue
        if args.per_galaxy_psf:                     # the paper's data: one PSF image per galaxy
            b["psf"] = np.ascontiguousarray(np.broadcast_to(b["psf"], (len(b["galaxies"]),) + b["psf"].shape))
        opts = dict(b["opts"]); opts["n_iter"] = n_iter
        opts["lr_decay"] = 0.01 ** (1.0 / max(n_iter - 1, 1))
        if args.no_early_stop:
            opts["tol"] = 0.0
        host = tuple(map(pin, (b["data"], b["sigma"], b["mask"], b["psf"], b["start"])))
        devt = tuple(map(d, host))
        B, H, W, K = len(b["galaxies"]), b["H"], b["W"], b["K"]
        buckets.append({"b": b, "B": B, "H": H, "W": W, "K": K, "opts": opts, "host": host, "dev": devt,
                        "params": devt[4].clone(),
                        "ws": torch.empty(gm.gm_workspace_bytes(b["model"], B, H, W, K, args.per_galaxy_psf) + 256,
                                          dtype=torch.uint8, device="cuda")})
    model = buckets[0]["b"]["model"]
    K = buckets[0]["K"]
    B = sum(k["B"] for k in buckets)
    early = any(k["opts"]["tol"] > 0.0 for k in buckets)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    multi = len(buckets) > 1 and not args.serial_buckets
    side_streams = [torch.cuda.Stream() for _ in buckets] if multi else None

    def step():
        outs, n = [], 0
        for k in buckets:
            k["params"].copy_(k["dev"][4])
        if multi:
            # every size bucket on its own stream, iterations interleaved (gm_fit_multi): the SMs a
            # bucket leaves idle once most of its galaxies stopped early take another bucket's work
            ev0 = torch.cuda.Event(); ev0.record(stream)
            for s in side_streams:
                s.wait_event(ev0)
            outs = gm.gm_fit_multi(model, [{"params": k["params"], "data": k["dev"][0], "sigma": k["dev"][1],
                                            "mask": k["dev"][2], "psf": k["dev"][3], "opts": k["opts"],
                                            "workspace": k["ws"]} for k in buckets], streams=side_streams)
            n = gm.gm_last_launch_count()
            for s in side_streams:
                e = torch.cuda.Event(); e.record(s)
                stream.wait_event(e)
            return outs, n
        for k in buckets:
            data, sigma, mask, psf, start = k["dev"]
            outs.append(gm.gm_fit(model, k["params"], data, sigma, mask, psf, k["opts"], workspace=k["ws"],
                                  stream=stream))
            n += gm.gm_last_launch_count()
        return outs, n

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        outs, _ = step()
    barrier()

    # ---- timed region: K steps, device time by CUDA events on the launching stream
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches = 0
    gm.gm_profile_enable(True)
    with ClockSampler(local) as clk:
        barrier()
        for s in range(args.steps):
            flush.zero_()                           # L2 flushed between steps (not timed)
            ev[s][0].record(stream)
            outs, n = step()
            ev[s][1].record(stream)
            launches += n
        barrier()
    prof = gm.gm_profile_read()
    gm.gm_profile_enable(False)
    t_ms = sum(a.elapsed_time(z) for a, z in ev)
    t = torch.tensor([t_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    t_ms = float(t.item())
    ms_per_step = t_ms / args.steps

    # chi^2+gradient evaluations actually made: iters_used per galaxy (= n_iter without early stop)
    status = np.concatenate([o["status"].cpu().numpy() for o in outs])
    iters = np.concatenate([o["iters_used"].cpu().numpy() for o in outs])
    red = np.concatenate([o["chi2"].cpu().numpy() /
                          np.maximum(k["H"] * k["W"] if k["b"]["mask"] is None
                                     else k["b"]["mask"].reshape(k["B"], -1).sum(1), 1)
                          for o, k in zip(outs, buckets)])
    evals = float(sum(o["iters_used"].sum().item() * k["H"] * k["W"] for o, k in zip(outs, buckets)))
    # algorithmic convolution flops of one step: 2 convolutions per evaluation + the closing forward
    # (status 0: n_iter evaluations + closing forward; stopped early or non-finite: the evaluation
    # that triggered the stop ran both convolutions but applied no update)
    def n_convs(o):
        it = o["iters_used"].cpu().numpy().astype(np.float64); st = o["status"].cpu().numpy()
        return float(np.where(st == 0, 2.0 * it + 1.0, 2.0 * (it + 1.0)).sum())
    conv_flops = float(sum(n_convs(o) * 2.0 * k["H"] * k["W"] * k["K"] ** 2 for o, k in zip(outs, buckets)))
    value = world * evals / (ms_per_step * 1e-3)

    # ---- e2e: the same step through the host-buffer C-ABI call (copies inside)
    e2e = None
    if rank == 0 or world > 1:
        hps = [k["host"][4].numpy().copy() for k in buckets]
        hargs = [tuple(None if t is None else t.numpy() for t in k["host"][:4]) for k in buckets]

        def host_step():
            for k, hp in zip(buckets, hps):
                hp[...] = k["b"]["start"]
            if multi:
                gm.gm_fit_multi_host(model, [{"params": hp, "data": ha[0], "sigma": ha[1], "mask": ha[2],
                                              "psf": ha[3], "opts": k["opts"]}
                                             for k, hp, ha in zip(buckets, hps, hargs)])
                return
            for k, hp, ha in zip(buckets, hps, hargs):
                gm.gm_fit_host(model, hp, *ha, k["opts"])

        host_step()                                                   # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            host_step()
        te = torch.tensor([(time.perf_counter() - t0) / args.steps], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        h2d = sum(a.nbytes for ha in hargs for a in ha if a is not None) + sum(hp.nbytes for hp in hps)
        d2h = sum(hp.nbytes for hp in hps) + 3 * B * 4
        e2e = {"value": world * evals / float(te.item()), "unit": UNIT, "ms_per_step": float(te.item()) * 1e3,
               "galaxies_fitted_per_s": world * B / float(te.item()),
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "api": ("gm_fit_multi_host" if multi else "gm_fit_host") +
                      " (host buffers; cudaMalloc + H2D + fit + D2H inside the call)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the heavy kernels (all run the same K^2-tap FFMA2 loop)
    pk, pk_src = peaks()
    clocks = clk.summary()
    f_mhz = pk.get("sm_max_mhz", 1965.0)
    peak_tflops = SM_COUNT * FP32_LANES * 2 * f_mhz * 1e6 / 1e12
    kern = {name: {"launches": n, "avg_ms": ms / n, "share_of_step": ms / t_ms if world == 1 else None}
            for name, (ms, n) in prof.items() if n}
    heavy_ms = sum(ms for ms, n in prof.values() if n)
    dom = max(kern, key=lambda k: kern[k]["avg_ms"] * kern[k]["launches"]) if kern else None
    roofline = None
    if dom:
        # buckets on concurrent streams: per-launch event times overlap one another, so the
        # kernels' time is the step's own device time, not the sum over launches
        achieved = (conv_flops / (ms_per_step * 1e-3) if multi else
                    args.steps * conv_flops / (heavy_ms * 1e-3)) / 1e12
        n_dom = kern[dom]["launches"]
        big = max(buckets, key=lambda k: k["B"] * k["H"] * k["W"])
        traffic = None
        # dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
        # ncu --set full capture summarised in profiles/r01_fused_ncu.md (kernel,bytes per line)
        tf = ROOT / "profiles" / "r01_traffic.csv"
        if tf.exists() and len(buckets) == 1:
            key = f"{dom}_K{K}_{big['H']}x{big['W']}_B{big['B']}"
            for line in tf.read_text().splitlines()[1:]:
                name, _, nbytes = line.partition(",")
                if name.strip() == key:
                    traffic = int(nbytes)
        px_bytes = 9 if big["b"]["mask"] is not None else 8
        roofline = {"bound": "alu", "kernel": f"k_{dom}<K={K}>", "achieved": achieved,
                    "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                    "traffic": traffic,
                    "peak_source": f"{SM_COUNT} SMs x {FP32_LANES} FP32 lanes x 2 flop x {f_mhz:.0f} MHz "
                                   f"(sm_max_mhz of {pk_src} MEASURED_PEAKS.json; an FFMA2 loop measured "
                                   "36.8 TFMA/s = 73.7 TFLOP/s on this pool, DESIGN.md)",
                    "algorithmic_flops_per_launch": args.steps * conv_flops / max(n_dom, 1)
                    if len(kern) == 1 else None,
                    "how": "2*K^2 flops per pixel per convolution x convolutions actually run "
                           "(2 per chi^2+gradient evaluation + the closing forward) / summed CUDA-event time of the "
                           "heavy kernels (forward, backward, fused) inside the timed region" +
                           ("; size buckets run concurrently on one stream each, so the divisor is the step's "
                            "device time and the per-kernel averages include time shared between streams"
                            if multi else ""),
                    "hbm_gbs_algorithmic": (evals * args.steps * px_bytes) / (heavy_ms * 1e-3) / 1e9,
                    "hbm_peak_gbs": pk.get("hbm_gbs"), "kernels": kern}
        # whole-step view: the same flops against the step time (small kernels and gaps included)
        roofline["step_frac"] = (conv_flops / (ms_per_step * 1e-3) / 1e12) / peak_tflops

    wl = (workload_name(cfg, B, buckets[0]["H"], buckets[0]["W"], K, n_iter) if len(buckets) == 1 else
          f"{cfg.name}: {B} galaxies, {cfg.model_name}, sides " +
          ", ".join(f"{k['H']}px x{k['B']}" for k in buckets) +
          f", {K}x{K} Moffat PSF, {'10% masked, ' if cfg.mask_frac else ''}gm_fit capped at {n_iter} iterations"
          + (" with early stop" if early else ""))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl + (", one PSF per galaxy [B,K,K]" if args.per_galaxy_psf else ""),
                       "global_batch": B * world,
                       "buckets": ("gm_fit_multi, one stream per cutout side" if multi else
                                   "gm_fit per cutout side, one after the other") if len(buckets) > 1 else None,
                       "parallelism": f"dp{world} (independent galaxies, no collective)",
                       "l2": "flushed between steps (256 MiB write)",
                       "inputs": "seeded synthetic SDSS-like (gen/configs.py), resident in HBM"},
            "galaxies_fitted_per_s": world * B / (ms_per_step * 1e-3),
            "fit_summary": {"status_counts": {str(k): int((status == k).sum()) for k in np.unique(status)},
                            "mean_iters": float(iters.mean()),
                            "median_reduced_chi2": float(np.median(red))},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline}
    if len(buckets) == 1 and rank == 0:
        # BASELINE metric (i) as SURVEY 8(d) words it: B*H*W*reps / t(gm_loss_grad), 3 warm-ups, 20 timed
        # calls at the start parameters, CUDA events on the launching stream, L2 flushed before each call
        k = buckets[0]
        data, sigma, mask, psf, start = k["dev"]
        chi2 = torch.empty(k["B"], dtype=torch.float32, device="cuda"); grad = torch.empty_like(start)
        lg = lambda: gm.gm_loss_grad(model, start, data, sigma, mask, psf, chi2=chi2, grad=grad,
                                     workspace=k["ws"], stream=stream)
        for _ in range(3):
            lg()
        tt = []
        for _ in range(20):
            flush.zero_()
            a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); lg(); z.record(stream)
            tt.append((a, z))
        torch.cuda.synchronize()
        ms = statistics.median(a.elapsed_time(z) for a, z in tt)
        line["loss_grad"] = {"value": k["B"] * k["H"] * k["W"] / (ms * 1e-3), "unit": UNIT, "ms_per_call": ms,
                             "calls": 20, "stat": "median",
                             "frac": 2 * 2.0 * k["B"] * k["H"] * k["W"] * k["K"] ** 2 / (ms * 1e-3) / 1e12 / peak_tflops,
                             "api": "gm_loss_grad (prologue, taps, chi^2 + gradient, finalize: the whole call)"}
    if args.stream_batches > 1 and len(buckets) == 1 and rank == 0:
        line["streamed"] = streamed(buckets[0], model, args.stream_batches)
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(cfg, buckets[len(buckets) // 2]["H"])
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1 = C1)")
    ap.add_argument("--batch", type=int, default=0, help="galaxies per GPU (default: the config's)")
    ap.add_argument("--side", type=int, default=0, help="cutout side for the mixed-size config C2")
    ap.add_argument("--iters", type=int, default=0, help="override the iteration count")
    ap.add_argument("--no-early-stop", action="store_true")
    ap.add_argument("--serial-buckets", action="store_true",
                    help="C2: one gm_fit per size bucket, one after the other, instead of gm_fit_multi")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--per-galaxy-psf", action="store_true",
                    help="pass the PSF as [B,K,K] (taps in shared memory instead of the constant bank)")
    ap.add_argument("--stream-batches", type=int, default=0,
                    help="also stream this many batches through two streams (C4: 65,536 galaxies = 32 x 2048)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
