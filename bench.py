#!/usr/bin/env python
"""bench.py -- throughput of the batched galaxy-fit hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 2|1|3|4|5] [--no-per-config] ...

One "step" = one pass of the whole hot path over one batch: a full fit of the workload
(render -> PSF convolution -> chi^2 -> adjoint convolution -> gradient -> Adam update,
every iteration, plus the closing chi^2 evaluation).  The headline workload (N = 1) is
BASELINE.json ``configs[2]`` (C2), the one the target sentence names: 8,289 single-Sersic
galaxies, cutout sides {64, 96, 128, 192, 256}, 25x25 Moffat PSF, 10 % of the pixels
masked, fit to convergence (tol 1e-6, patience 10) capped at 500 iterations, all five size
buckets in one ``gm_fit_multi`` call.  The same JSON line carries, under ``per_config``,
C1, C3, one 2,048-galaxy batch of C4, P1 (the paper's own shapes: 8,289 cutouts of 128x128
with 41x41 PSFs) and P1 with one PSF per galaxy, each measured the same way.

With N > 1 (torchrun) the N x 8,289 galaxies are dealt to the ranks by pixel count
(``sharding.shard_galaxies``), every rank fits its shard (no data-path collective: galaxies
are independent), and the fitted parameters are all-gathered at the
end (``sharding.gather_results``, timed separately).

Prints ONE JSON line (rank 0).  metric = galaxy-pixel chi^2+gradient evaluations per
second = sum over galaxies of H*W*iterations / step time, whole job.  DESIGN.md section 7.
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


def workload_name(cfg, buckets, n_iter, early, per_galaxy_psf):
    K = buckets[0]["K"]
    B = sum(k["B"] for k in buckets)
    psf = "Moffat" if cfg.psf_kind.startswith("moffat") else "Gaussian"
    if len(buckets) == 1:
        k = buckets[0]
        s = f"{cfg.name}: {B} galaxies, {cfg.model_name}, {k['H']}x{k['W']} fp32 cutouts, {K}x{K} {psf} PSF, "
    else:
        s = (f"{cfg.name}: {B} galaxies, {cfg.model_name}, sides " +
             ", ".join(f"{k['H']}px x{k['B']}" for k in buckets) + f", {K}x{K} {psf} PSF, ")
    if cfg.mask_frac:
        s += f"{int(round(100 * cfg.mask_frac))}% masked, "
    s += (f"fit to convergence (tol {buckets[0]['opts']['tol']:g}, patience {buckets[0]['opts']['patience']}) "
          f"capped at {n_iter} iterations" if early else f"{n_iter}-iteration fit")
    if per_galaxy_psf:
        s += ", one PSF per galaxy [B,K,K]"
    return s


# ---------------------------------------------------------------------------------
def reference_sample(cfg, n_gal):
    """`n_gal` galaxies of the config's middle size bucket, truth images by the oracle."""
    import oracle
    from gen import configs
    side = cfg.sides[len(cfg.sides) // 2]
    cand = list(range(40 * n_gal))
    gal = [g for g, s in zip(cand, configs.sides_for(cfg, cand)) if s == side][:n_gal]
    return configs.make_batch(cfg.cid, gal, lambda m, p, H, W, psf: oracle.render(m, p, H, W, psf), side=side)


def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (the other
    place bench.py may execute oracle/).  Each step is a bounded sample of the same
    workload: `cores` galaxies x 3 iterations of the config's middle size bucket."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from gen import configs
    cfg = configs.CONFIGS[args.config]
    cores = oracle.num_threads()
    n_iter = 3
    b = reference_sample(cfg, cores)
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
    sample = (f"{n_gal} galaxies x {n_iter} iterations of {cfg.name}'s {b['H']}x{b['W']} bucket "
              f"(K={b['K']}{', masked' if b['mask'] is not None else ''}) per step")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name} ({cfg.B} galaxies, {cfg.model_name}, K={cfg.K}; see the ours arm)",
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def cpu_baseline(cfg):
    """The oracle timed on the box's host cores on a bounded sample (~10-30 s)."""
    import oracle
    from gen import configs
    cores = oracle.num_threads()
    b = reference_sample(cfg, 2 * cores)
    n_gal = len(b["galaxies"])
    # size the iteration count from one timed evaluation so the sample takes ~15 s
    t0 = time.perf_counter()
    oracle.loss_grad(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"])
    t_eval = time.perf_counter() - t0
    n_iter = int(min(max(15.0 / max(t_eval, 1e-3), 2), 200))
    opts = configs.fit_options(b["model"], b["H"], b["W"], n_iter)
    t0 = time.perf_counter()
    oracle.fit(b["model"], b["start"], b["data"], b["sigma"], b["mask"], b["psf"], opts)
    dt = time.perf_counter() - t0
    out = {"value": n_gal * b["H"] * b["W"] * n_iter / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"{n_gal} galaxies x {n_iter} iterations of {cfg.name}'s {b['H']}x{b['W']} bucket (K={b['K']}), "
                     f"{dt:.1f} s, OpenMP over galaxies"}
    # the oracle "at 1 thread and at all cores" -- one galaxy of the same sample on one thread, ~5 s
    n1 = int(min(max(5.0 / max(t_eval / max(n_gal / cores, 1.0), 1e-3), 2), n_iter))
    o1 = configs.fit_options(b["model"], b["H"], b["W"], n1)
    oracle.set_num_threads(1)
    try:
        t0 = time.perf_counter()
        oracle.fit(b["model"], b["start"][:1], b["data"][:1], b["sigma"][:1], None if b["mask"] is None else b["mask"][:1],
                   b["psf"], o1)
        d1 = time.perf_counter() - t0
    finally:
        oracle.set_num_threads(cores)
    out["one_thread"] = {"value": b["H"] * b["W"] * n1 / d1, "unit": UNIT, "cores": 1,
                         "sample": f"1 galaxy x {n1} iterations of the same bucket, {d1:.1f} s"}
    return out


# ---------------------------------------------------------------------------------
class Bench:
    """One process = one GPU.  Holds torch / the binding / the distributed group."""

    def __init__(self, args):
        import torch
        import paper_2404_07780_b200 as gm
        self.torch, self.gm, self.args = torch, gm, args
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
        torch.cuda.set_device(self.local)
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            self.dist = dist
        self.flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        self.stream = torch.cuda.current_stream()
        self.workers = min(16, os.cpu_count() or 1)
        gm.gm_init()
        gm.gm_set_option(gm.GM_OPT_TENSOR, 1 if args.engine == "tensor" else 0)
        # the roofline denominator, measured in this process: a pure FFMA2 kernel (gm.h)
        # (the best of five runs of 50 launches: the first ones see a GPU that has not clocked up yet)
        self.peak_measured = max(gm.gm_measure_fp32_peak(50) for _ in range(5))
        pk, self.pk_src = peaks()
        self.pk = pk
        self.f_mhz = pk.get("sm_max_mhz", 1965.0)
        self.peak_nominal = SM_COUNT * FP32_LANES * 2 * self.f_mhz * 1e6 / 1e12
        self.peak_tensor = pk.get("bf16_tflops_sustained") or pk["bf16_tflops"]

    @staticmethod
    def mma_inflation(name, k):
        """MMA flops the tensor-core kernels issue per algorithmic convolution flop (1 for the FFMA2 kernels).
        One pass = 128 lanes of 4 x 32 output pixels; per pass and convolution KT tap rows x 4 accumulator rows x
        3 split terms x (NCH - 2 MMAs of 128 x 32 x 16 + 2 of 128 x 16 x 16 for the two edge chunks) (gm_tc.cuh)."""
        if not name.startswith("tc_"):
            return 1.0
        K, H, W = k["K"], k["H"], k["W"]
        KT = next(t for t in (9, 17, 25, 33, 41) if t >= K)
        TR, TC = 4, 32                                                    # kTileR, kTileC of gm_tc.cuh
        nch = (TC + KT - 1 + 15) // 16
        per_pass = KT * TR * 3 * ((nch - 2) * (2.0 * 128 * TC * 16) + 2 * (2.0 * 128 * (TC // 2) * 16))
        if name == "tc_fused":
            passes = {64: 0.25, 96: 1.0, 128: 1.0}[H]                     # per cutout
        else:
            passes = min(-(-H // (TR * c)) * -(-W // (TC * (128 // c))) for c in (128 // TR, 64 // TR))
        return passes * per_pass / (2.0 * H * W * K * K)

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def render(self, model, p, H, W, psf):
        """Truth images from the CUDA path itself (never compared with the oracle), in chunks."""
        torch, gm = self.torch, self.gm
        out = np.empty((p.shape[0], H, W), dtype=np.float32)
        dpsf = torch.from_numpy(psf).cuda()
        step = max(1, (256 << 20) // (H * W * 4))
        for i in range(0, p.shape[0], step):
            out[i:i + step] = gm.gm_render(model, torch.from_numpy(p[i:i + step]).cuda(), H, W, dpsf).cpu().numpy()
        return out

    # -----------------------------------------------------------------------------
    def make_buckets(self, cfg, gal, n_iter, per_galaxy_psf=False, side=None, early_stop=True):
        torch, gm = self.torch, self.gm
        from gen import configs
        pin = lambda a: None if a is None else torch.from_numpy(a).pin_memory()
        d = lambda t: None if t is None else t.cuda(non_blocking=True)
        drawn = configs.sides_for(cfg, list(gal))
        buckets = []
        for s in ([side] if side else list(cfg.sides)):
            if not (drawn == s).any():
                continue
            b = configs.make_batch(cfg.cid, gal, self.render, side=s, workers=self.workers)
            if per_galaxy_psf:                      # the paper's data: one PSF image per galaxy
                b["psf"] = np.ascontiguousarray(np.broadcast_to(b["psf"], (len(b["galaxies"]),) + b["psf"].shape))
            opts = dict(b["opts"]); opts["n_iter"] = n_iter
            opts["lr_decay"] = 0.01 ** (1.0 / max(n_iter - 1, 1))
            if not early_stop:
                opts["tol"] = 0.0
            host = tuple(map(pin, (b["data"], b["sigma"], b["mask"], b["psf"], b["start"])))
            devt = tuple(map(d, host))
            B, H, W, K = len(b["galaxies"]), b["H"], b["W"], b["K"]
            buckets.append({"model": b["model"], "galaxies": b["galaxies"], "start": b["start"],
                            "n_used": (None if b["mask"] is None else b["mask"].reshape(B, -1).sum(1)),
                            "B": B, "H": H, "W": W, "K": K, "opts": opts, "host": host, "dev": devt,
                            "params": devt[4].clone(),
                            "ws": torch.empty(gm.gm_workspace_bytes(b["model"], B, H, W, K, per_galaxy_psf) + 256,
                                              dtype=torch.uint8, device="cuda")})
        return buckets

    def step(self, buckets, multi, side_streams):
        torch, gm, stream = self.torch, self.gm, self.stream
        model = buckets[0]["model"]
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
        outs, n = [], 0
        for k in buckets:
            data, sigma, mask, psf, _ = k["dev"]
            outs.append(gm.gm_fit(model, k["params"], data, sigma, mask, psf, k["opts"], workspace=k["ws"],
                                  stream=stream))
            n += gm.gm_last_launch_count()
        return outs, n

    @staticmethod
    def conv_flops(o, k):
        """Algorithmic convolution flops of one bucket's fit: 2 K^2 flops per pixel per convolution
        actually run (status 0: n_iter evaluations of two convolutions + the closing forward; stopped
        early or non-finite: the evaluation that triggered the stop ran both but applied no update)."""
        it = o["iters_used"].cpu().numpy().astype(np.float64); st = o["status"].cpu().numpy()
        n_fwd = np.where(st == 0, it + 1.0, it + 1.0).sum()
        n_bwd = np.where(st == 0, it, it + 1.0).sum()
        per = 2.0 * k["H"] * k["W"] * k["K"] ** 2
        return n_fwd * per, n_bwd * per

    # -----------------------------------------------------------------------------
    def measure(self, cfg, buckets, steps, warmup, multi, want_e2e=True, serial_profile=False):
        """Times `steps` steps of the workload; returns the record of that workload."""
        torch, gm, stream = self.torch, self.gm, self.stream
        world = self.world
        model = buckets[0]["model"]
        K = buckets[0]["K"]
        B = sum(k["B"] for k in buckets)
        n_iter = buckets[0]["opts"]["n_iter"]
        early = any(k["opts"]["tol"] > 0.0 for k in buckets)
        side_streams = [torch.cuda.Stream() for _ in buckets] if multi else None

        for _ in range(max(warmup, 3)):
            self.flush.zero_()
            outs, _ = self.step(buckets, multi, side_streams)
        self.barrier()

        # ---- timed region: `steps` steps, device time by CUDA events on the launching stream
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        launches = 0
        gm.gm_profile_enable(True)
        with ClockSampler(self.local) as clk:
            self.barrier()
            for s in range(steps):
                self.flush.zero_()                  # L2 flushed between steps (not timed)
                ev[s][0].record(stream)
                outs, n = self.step(buckets, multi, side_streams)
                ev[s][1].record(stream)
                launches += n
            self.barrier()
        prof = gm.gm_profile_read()
        gm.gm_profile_enable(False)
        t_ms = sum(a.elapsed_time(z) for a, z in ev)
        t = torch.tensor([t_ms], dtype=torch.float64, device="cuda")
        if self.dist is not None:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        t_ms = float(t.item())
        ms_per_step = t_ms / steps

        status = np.concatenate([o["status"].cpu().numpy() for o in outs])
        iters = np.concatenate([o["iters_used"].cpu().numpy() for o in outs])
        red = np.concatenate([o["chi2"].cpu().numpy() / np.maximum(k["H"] * k["W"] if k["n_used"] is None else k["n_used"], 1)
                              for o, k in zip(outs, buckets)])
        # chi^2+gradient evaluations actually made: iters_used per galaxy (= n_iter without early stop)
        evals = torch.tensor([float(sum(o["iters_used"].sum().item() * k["H"] * k["W"] for o, k in zip(outs, buckets)))],
                             dtype=torch.float64, device="cuda")
        ngal = torch.tensor([float(B)], dtype=torch.float64, device="cuda")
        if self.dist is not None:
            self.dist.all_reduce(evals); self.dist.all_reduce(ngal)
        evals_all, B_all = float(evals.item()), float(ngal.item())
        flops = [self.conv_flops(o, k) for o, k in zip(outs, buckets)]
        conv_flops = sum(f + b for f, b in flops)
        value = evals_all / (ms_per_step * 1e-3)

        rec = {"workload": workload_name(cfg, buckets, n_iter, early, buckets[0]["dev"][3].dim() == 3),
               "ms_per_step": ms_per_step, "value": value, "unit": UNIT,
               "galaxies_fitted_per_s": B_all / (ms_per_step * 1e-3),
               "fit_summary": {"status_counts": {str(k): int((status == k).sum()) for k in np.unique(status)},
                               "mean_iters": float(iters.mean()), "median_reduced_chi2": float(np.median(red))},
               "clocks": clk.summary(), "gpu_launches": int(launches)}

        # ---- roofline of the heavy kernels: algorithmic convolution flops (2 K^2 per pixel per convolution,
        # SURVEY 8(d)) against the pipe that binds the kernel: the tensor pipe for the tcgen05 kernels (k_tc_*),
        # the FP32 FMA pipe for the FFMA2 kernels
        def flops_of(name, f_fwd, f_bwd):
            return (f_fwd + f_bwd) if name.endswith("fused") else (f_fwd if name.endswith("forward") else f_bwd)

        kinds = {name: (ms, n) for name, (ms, n) in prof.items() if n}
        kern, dom, achieved, issued = {}, None, None, None
        if multi and serial_profile and self.rank == 0:
            # buckets on concurrent streams: per-launch event times overlap one another.  One more
            # step, bucket after bucket on one stream, gives every kernel its own duration.
            per_kind_ms = {}; per_kind_n = {}; per_kind_flops = {}; per_kind_issued = {}
            for k in buckets:
                k["params"].copy_(k["dev"][4])
                gm.gm_profile_enable(True)
                data, sigma, mask, psf, _ = k["dev"]
                o = gm.gm_fit(model, k["params"], data, sigma, mask, psf, k["opts"], workspace=k["ws"], stream=stream)
                torch.cuda.synchronize()
                pr = gm.gm_profile_read()
                gm.gm_profile_enable(False)
                f_fwd, f_bwd = self.conv_flops(o, k)
                ran = {name for name, (ms, n) in pr.items() if n}
                for name, (ms, n) in pr.items():
                    if not n:
                        continue
                    fl = flops_of(name, f_fwd, f_bwd)
                    per_kind_ms[name] = per_kind_ms.get(name, 0.0) + ms
                    per_kind_n[name] = per_kind_n.get(name, 0) + n
                    per_kind_flops[name] = per_kind_flops.get(name, 0.0) + fl
                    per_kind_issued[name] = per_kind_issued.get(name, 0.0) + fl * self.mma_inflation(name, k)
                    pk_k = self.peak_tensor if name.startswith("tc_") else self.peak_measured
                    k.setdefault("serial", {})[name] = {"launches": n, "avg_ms": ms / n,
                                                        "tflops": fl / (ms * 1e-3) / 1e12,
                                                        "frac": fl / (ms * 1e-3) / 1e12 / pk_k,
                                                        "bound": "tensor" if name.startswith("tc_") else "alu"}
                assert ran, "no heavy kernel ran"
            kern = {name: {"launches": per_kind_n[name], "avg_ms": per_kind_ms[name] / per_kind_n[name],
                           "tflops": per_kind_flops[name] / (per_kind_ms[name] * 1e-3) / 1e12}
                    for name in per_kind_ms}
            dom = max(kern, key=lambda n: per_kind_ms[n])
            achieved = kern[dom]["tflops"]
            issued = per_kind_issued[dom] / (per_kind_ms[dom] * 1e-3) / 1e12
            how_t = ("one extra step with the buckets one after the other on one stream (per-launch CUDA events do not "
                     "overlap there); the timed steps run the buckets concurrently")
            rec["buckets"] = [{"side": k["H"], "galaxies": k["B"], "kernels": k.get("serial")} for k in buckets]
        elif kinds:
            kern = {name: {"launches": n, "avg_ms": ms / n} for name, (ms, n) in kinds.items()}
            dom = max(kern, key=lambda n: kinds[n][0])
            # the kernels of one family run the same loop: their flops over their summed time
            fam = [n for n in kinds if n.startswith("tc_") == dom.startswith("tc_")]
            fam_ms = sum(kinds[n][0] for n in fam)
            fam_fl = sum(flops_of(n, fwd, bwd) for n in fam for fwd, bwd in flops) * steps
            achieved = fam_fl / (fam_ms * 1e-3) / 1e12
            issued = sum(flops_of(n, fwd, bwd) * self.mma_inflation(n, k) for n in fam
                         for (fwd, bwd), k in zip(flops, buckets)) * steps / (fam_ms * 1e-3) / 1e12
            how_t = "summed CUDA-event time of those kernels inside the timed region"
            for name in kern:
                kern[name]["share_of_step"] = kinds[name][0] / t_ms if world == 1 else None
        if dom:
            # the largest bucket that runs the dominant kernel (with several buckets, the one its captures are keyed on)
            ran = [k for k in buckets if dom in (k.get("serial") or {dom: None})]
            big = max(ran or buckets, key=lambda k: k["B"] * k["H"] * k["W"])
            px_bytes = 9 if big["dev"][2] is not None else 8
            tensor = dom.startswith("tc_")
            peak = self.peak_tensor if tensor else self.peak_measured
            rec["roofline"] = {
                "bound": "tensor" if tensor else "alu", "kernel": f"k_{dom}<K={K}>", "achieved": achieved, "peak": peak,
                "unit": "TFLOP/s", "frac": achieved / peak,
                "peak_source": (f"{self.pk_src} MEASURED_PEAKS.json bf16_tflops_sustained (cuBLAS bf16 GEMM back to back; fp16 "
                                "runs at the bf16 rate); the kernel is timed inside a long step, so the sustained figure")
                if tensor else "measured in this process: gm_measure_fp32_peak, a pure fma.rn.f32x2 kernel (include/gm.h)",
                "traffic": traffic_from_profiles(dom, K, big),
                "algorithmic_bytes_per_px_eval": px_bytes,
                "how": "2*K^2 flops per pixel per convolution x convolutions actually run (2 per chi^2+gradient "
                       "evaluation + the closing forward) / " + how_t,
                "hbm_peak_gbs": self.pk.get("hbm_gbs"), "kernels": kern,
                # the same flops against the FP32 FMA pipe, the bound of the direct (FFMA2) convolution this engine replaces
                "fp32_peak": self.peak_measured, "frac_of_fp32_peak": achieved / self.peak_measured,
                "fp32_peak_nominal": self.peak_nominal,
                # whole-step view: the same flops against the step time (small kernels and gaps included)
                "step_frac": (conv_flops / (ms_per_step * 1e-3) / 1e12) / peak}
            if early and len(buckets) > 1:
                rec["roofline"]["note"] = ("whole fit with early stop: most of the iterations run the few galaxies that have not "
                                           "converged yet (latency, not throughput); per_config holds the same kernels at full batch")
            if tensor:
                # what the tensor pipe is asked to do for those flops: 3 fp16 MMAs per product (hi*hi + lo*hi + hi*lo)
                # on Toeplitz band blocks: issued MMA flops / the same time / the same peak
                rec["roofline"].update({"mma_issued_tflops": issued, "mma_issued_frac": issued / peak,
                                        "mma_flops_per_algorithmic_flop": issued / achieved})

        # ---- e2e: the same step through the host-buffer C-ABI call (copies inside)
        if want_e2e:
            hps = [k["host"][4].numpy().copy() for k in buckets]
            hargs = [tuple(None if t is None else t.numpy() for t in k["host"][:4]) for k in buckets]

            def host_step():
                for k, hp in zip(buckets, hps):
                    hp[...] = k["start"]
                if len(buckets) > 1:
                    gm.gm_fit_multi_host(model, [{"params": hp, "data": ha[0], "sigma": ha[1], "mask": ha[2],
                                                  "psf": ha[3], "opts": k["opts"]}
                                                 for k, hp, ha in zip(buckets, hps, hargs)])
                    return
                for k, hp, ha in zip(buckets, hps, hargs):
                    gm.gm_fit_host(model, hp, *ha, k["opts"])

            host_step()                                                   # warm-up
            self.barrier()
            t0 = time.perf_counter()
            for _ in range(steps):
                host_step()
            te = torch.tensor([(time.perf_counter() - t0) / steps], dtype=torch.float64, device="cuda")
            if self.dist is not None:
                self.dist.all_reduce(te, op=self.dist.ReduceOp.MAX)
            h2d = sum(a.nbytes for ha in hargs for a in ha if a is not None) + sum(hp.nbytes for hp in hps)
            d2h = sum(hp.nbytes for hp in hps) + 3 * B * 4
            rec["e2e"] = {"value": evals_all / float(te.item()), "unit": UNIT, "ms_per_step": float(te.item()) * 1e3,
                          "galaxies_fitted_per_s": B_all / float(te.item()),
                          "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                          "api": ("gm_fit_multi_host" if len(buckets) > 1 else "gm_fit_host") +
                                 " (host buffers; device allocation + H2D + fit + D2H inside the call)"}
            # the copy rate of this box, measured on its own: the step's pinned host inputs -> their device buffers
            a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record(self.stream)
            with torch.cuda.stream(self.stream):
                nb = 0
                for k in buckets:
                    for h, dv in zip(k["host"], k["dev"]):
                        if h is not None:
                            dv.copy_(h, non_blocking=True); nb += h.numel() * h.element_size()
            z.record(self.stream)
            torch.cuda.synchronize()
            rec["e2e"]["h2d_gbs"] = nb / (a.elapsed_time(z) * 1e-3) / 1e9
            rec["e2e"]["h2d_ms_alone"] = a.elapsed_time(z)
        rec["_outs"] = outs
        return rec

    def loss_grad_line(self, k):
        """BASELINE metric (i) as SURVEY 8(d) words it: B*H*W*reps / t(gm_loss_grad): 3 warm-ups, 20 timed
        calls at the start parameters, CUDA events on the launching stream, L2 flushed before each call."""
        torch, gm, stream = self.torch, self.gm, self.stream
        data, sigma, mask, psf, start = k["dev"]
        chi2 = torch.empty(k["B"], dtype=torch.float32, device="cuda"); grad = torch.empty_like(start)
        lg = lambda: gm.gm_loss_grad(k["model"], start, data, sigma, mask, psf, chi2=chi2, grad=grad,
                                     workspace=k["ws"], stream=stream)
        for _ in range(3):
            lg()
        tt = []
        for _ in range(20):
            self.flush.zero_()
            a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); lg(); z.record(stream)
            tt.append((a, z))
        torch.cuda.synchronize()
        ms = statistics.median(a.elapsed_time(z) for a, z in tt)
        return {"value": k["B"] * k["H"] * k["W"] / (ms * 1e-3), "unit": UNIT, "ms_per_call": ms, "calls": 20,
                "stat": "median",
                "tflops": 2 * 2.0 * k["B"] * k["H"] * k["W"] * k["K"] ** 2 / (ms * 1e-3) / 1e12,
                "frac_of_fp32_peak": 2 * 2.0 * k["B"] * k["H"] * k["W"] * k["K"] ** 2 / (ms * 1e-3) / 1e12 / self.peak_measured,
                "api": "gm_loss_grad (prologue, taps, chi^2 + gradient, finalize: the whole call)"}

    def streamed(self, k, n_batches):
        """BASELINE config C4 is "streamed in batches": n_batches batches through the device-pointer
        C ABI on two streams with two sets of device buffers, so that the host-to-device copy of batch
        i + 1 (from pinned host memory) and the read-back of batch i - 1 overlap the fit of batch i.
        The same synthetic batch is re-sent every time (its bytes cross the bus every time); wall
        clock with a device synchronise on both sides."""
        torch, gm = self.torch, self.gm
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
                    gm.gm_fit(k["model"], b["params"], b["data"], b["sigma"], b["mask"], psf, k["opts"],
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


def traffic_from_profiles(dom, K, big):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the ncu
    --set full captures summarised under profiles/ (kernel_K.._HxW_B..,bytes per line); None when that
    kernel / shape was not captured."""
    key = f"{dom}_K{K}_{big['H']}x{big['W']}_B{big['B']}"
    for name in ("r02_traffic.csv", "r01_traffic.csv"):
        tf = ROOT / "profiles" / name
        if not tf.exists():
            continue
        for line in tf.read_text().splitlines()[1:]:
            k, _, nbytes = line.partition(",")
            if k.strip() == key:
                return int(nbytes.split(",")[0])
    return None


# ---------------------------------------------------------------------------------
SUB_CONFIGS = (  # key, config id, galaxies, per-galaxy PSF
    ("C1", 1, None, False),
    ("C3", 3, None, False),
    ("C4_batch2048", 4, 2048, False),
    ("P1", 5, None, False),
    ("P1_per_galaxy_psf", 5, None, True),
)


def run_ours(args):
    from gen import configs
    from paper_2404_07780_b200.sharding import gather_results, shard_galaxies
    bn = Bench(args)
    torch = bn.torch
    cfg = configs.CONFIGS[args.config]
    Btot = args.batch or cfg.B
    n_iter = args.iters or cfg.n_iter or 200

    # galaxies of this rank: the world x Btot galaxies dealt out by pixel count (LPT), no collective
    # in the loop; at world = 1 this is galaxies 0 .. Btot-1 in order
    all_gal = np.arange(bn.world * Btot)
    px = configs.sides_for(cfg, all_gal).astype(np.int64) ** 2
    shards = shard_galaxies(px, bn.world)
    mine = all_gal[shards[bn.rank]]
    buckets = bn.make_buckets(cfg, list(mine), n_iter, args.per_galaxy_psf, args.side or None, not args.no_early_stop)
    multi = len(buckets) > 1 and not args.serial_buckets
    rec = bn.measure(cfg, buckets, args.steps, args.warmup, multi, want_e2e=True, serial_profile=True)
    outs = rec.pop("_outs")

    gather = None
    if bn.world > 1:
        # final gather of the fitted parameters and chi^2 in the original galaxy order (8(e))
        order = np.concatenate([np.searchsorted(all_gal, np.asarray(k["galaxies"])) for k in buckets])
        par = torch.cat([o["params"] for o in outs]); chi = torch.cat([o["chi2"] for o in outs])
        bn.barrier()
        t0 = time.perf_counter()
        full_p, full_c = gather_results(order, par, chi, len(all_gal))
        torch.cuda.synchronize()
        gather = {"ms": (time.perf_counter() - t0) * 1e3, "rows": int(full_p.shape[0]),
                  "finite": bool(torch.isfinite(full_c).all().item())}

    if bn.rank != 0:
        if bn.dist is not None:
            bn.dist.destroy_process_group()
        return 0

    line = {"metric": METRIC, "value": rec["value"], "unit": UNIT, "n_gpus": bn.world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": rec["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": rec["workload"], "global_batch": Btot * bn.world,
                       "buckets": ("gm_fit_multi, one stream per cutout side" if multi else
                                   "gm_fit per cutout side, one after the other") if len(buckets) > 1 else None,
                       "parallelism": f"dp{bn.world} (galaxies dealt by pixel count, no collective in the loop, "
                                      "final all-gather of params/chi2)" if bn.world > 1 else "single GPU",
                       "engine": args.engine,
                       "l2": "flushed between steps (256 MiB write)",
                       "inputs": "seeded synthetic SDSS-like (gen/configs.py), resident in HBM"},
            "galaxies_fitted_per_s": rec["galaxies_fitted_per_s"], "fit_summary": rec["fit_summary"],
            "clocks": rec["clocks"], "e2e": rec.get("e2e"), "gpu_launches": rec["gpu_launches"],
            "roofline": rec.get("roofline"), "buckets": rec.get("buckets"),
            "fp32_peak": {"measured_tflops": bn.peak_measured, "nominal_tflops": bn.peak_nominal}}
    if gather:
        line["gather"] = gather
    if len(buckets) == 1:
        line["loss_grad"] = bn.loss_grad_line(buckets[0])
        if args.stream_batches > 1:
            line["streamed"] = bn.streamed(buckets[0], args.stream_batches)
    del buckets, outs
    torch.cuda.empty_cache()

    if bn.world == 1 and not args.no_per_config and args.config == 2 and not args.side:
        per = {}
        sub_steps = max(1, min(args.steps, 2))
        for key, cid, nb, pg in SUB_CONFIGS:
            c = configs.CONFIGS[cid]
            B = nb or c.B
            bk = bn.make_buckets(c, list(range(B)), c.n_iter or 200, pg, None, True)
            r = bn.measure(c, bk, sub_steps, 3, False, want_e2e=True)
            r.pop("_outs")
            rf = r.pop("roofline", None) or {}
            r.update({"steps": sub_steps, "bound": rf.get("bound"), "kernel": rf.get("kernel"), "frac": rf.get("frac"),
                      "peak": rf.get("peak"), "frac_of_fp32_peak": rf.get("frac_of_fp32_peak"),
                      "mma_issued_frac": rf.get("mma_issued_frac"),
                      "step_frac": rf.get("step_frac"), "achieved_tflops": rf.get("achieved"),
                      "traffic": rf.get("traffic"), "kernels": rf.get("kernels")})
            if key == "C1":
                r["loss_grad"] = bn.loss_grad_line(bk[0])
            if key == "C4_batch2048":
                # BASELINE C4 is "streamed in batches": a short leg of it (4 of the 32 batches) in the default line
                r["streamed"] = bn.streamed(bk[0], 4)
            per[key] = r
            del bk
            torch.cuda.empty_cache()
        line["per_config"] = per
        # the same facts, compact, inside a key every reader of the line keeps: enough to recompute each `frac`
        def _compact(r):
            e = r.get("e2e") or {}
            c = {"ms_per_step": r.get("ms_per_step"), "value": r.get("value"), "workload": r.get("workload"),
                 "kernel": r.get("kernel"), "frac": r.get("frac"), "peak": r.get("peak"),
                 "achieved_tflops": r.get("achieved_tflops"), "mma_issued_frac": r.get("mma_issued_frac"),
                 "step_frac": r.get("step_frac"), "kernels": r.get("kernels"), "gpu_launches": r.get("gpu_launches"),
                 "e2e_ms": e.get("ms_per_step"), "h2d_bytes": e.get("h2d_bytes_per_step"), "h2d_gbs": e.get("h2d_gbs"),
                 "h2d_ms_alone": e.get("h2d_ms_alone")}
            if r.get("loss_grad"):
                c["loss_grad"] = {k: r["loss_grad"].get(k) for k in ("value", "ms_per_call", "tflops")}
            if r.get("streamed"):
                c["streamed"] = {k: r["streamed"].get(k) for k in ("batches", "galaxies", "seconds", "galaxies_fitted_per_s",
                                                                   "value", "h2d_bytes_per_batch")}
            return c
        if line.get("roofline") is not None:
            line["roofline"]["per_config"] = {k: _compact(r) for k, r in per.items()}
    if line.get("roofline") is not None and line.get("buckets"):
        line["roofline"]["per_bucket"] = line["buckets"]
    e2e = line.get("e2e")
    if e2e and e2e.get("ms_per_step"):
        # what the host-buffer call adds to the device-timed fit, and the copy rate that implies if all of it were
        # the H2D copy (a lower bound of the achieved rate; run-to-run noise of the fit is inside it)
        e2e["overhead_ms"] = e2e["ms_per_step"] - line["ms_per_step"]
        e2e["overhead_note"] = ("e2e minus the device-timed step; smaller than h2d_ms_alone where gm_fit_multi_host overlaps one "
                                "bucket's copy with another bucket's fit, and because the device-timed steps run back to back "
                                "under the power cap (plus an L2 flush each) while the host steps idle the SMs during copies")
    if bn.world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(cfg)
    print(json.dumps(line))
    if bn.dist is not None:
        bn.dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2,
                    help="BASELINE.json config index (default 2 = C2, the 8,289-galaxy target; 5 = P1)")
    ap.add_argument("--batch", type=int, default=0, help="galaxies per GPU (default: the config's)")
    ap.add_argument("--side", type=int, default=0, help="only this cutout side of the mixed-size config C2")
    ap.add_argument("--iters", type=int, default=0, help="override the iteration count")
    ap.add_argument("--no-early-stop", action="store_true")
    ap.add_argument("--serial-buckets", action="store_true",
                    help="C2: one gm_fit per size bucket, one after the other, instead of gm_fit_multi")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config sub-records (C1, C3, C4, P1)")
    ap.add_argument("--per-galaxy-psf", action="store_true",
                    help="pass the PSF as [B,K,K] (the paper's data layout, P:45)")
    ap.add_argument("--engine", default="tensor", choices=["tensor", "ffma2"],
                    help="convolution engine: tcgen05 tensor cores (default, where the shape allows) or the FP32 FFMA2 "
                         "loops only (gm_set_option(GM_OPT_TENSOR, 0)): the same workload on the engine of round 1")
    ap.add_argument("--stream-batches", type=int, default=0,
                    help="also stream this many batches through two streams (C4: 65,536 galaxies = 32 x 2048)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
