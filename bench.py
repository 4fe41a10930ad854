#!/usr/bin/env python
"""bench.py -- headline benchmark of the SPS hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c4_hmc|c3_approx|c2_exact|c5_nuts] [--protocol config|paper]

Default workload = BASELINE.json configs[3] ("c4_hmc"): full HMC on the approximate path, 10,000 synthetic galaxies x 4
chains x (500 warmup + 500 samples) x 16 leapfrog steps; metric = galaxy posteriors per GPU-minute.  One "step" = one
complete sps_hmc_run over the batch.  `--protocol paper` replaces the transition counts by the paper's own protocol
(100 adaptation + 3000 kept steps) so that the figure beside the paper's ~1,000 posteriors / GPU-minute is
like for like.  With N > 1 every rank runs the same number of galaxies (weak scaling; galaxies are independent, no
data-path collective) and the value is the job aggregate; `--gpus N` without torchrun's environment re-launches itself
under torchrun.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from paper_2506_19919_b200.sharding import aggregate_throughput, max_over_ranks, rank_seed  # noqa: E402


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def n(self):
        return len(self.rows)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
# workload construction (synthetic, seeded)
# ------------------------------------------------------------------------------------------------
def make_hmc_inputs(sps, W, table, ph, prior, n_gal, seed, rank=0, exact_mask=None, exact_seed=0):
    """True parameters drawn from the prior; observed fluxes = the library's own photometry of the truth with 5-10 %
    Gaussian noise (bench.py may not touch oracle/ outside the cpu_baseline leg).  Every galaxy's data come from the path
    it is fitted with: the approximate path, or the exact path where exact_mask is set (BASELINE.json configs[4])."""
    import torch
    thu = W.draw_theta_unbounded(prior, n_gal, rank_seed(seed, rank)).astype(np.float32)
    f = sps.sps_photometry(table, ph, sps.PATH_APPROX, torch.tensor(thu, device="cuda")).cpu().numpy().astype(np.float64)
    d, s = W.noisy_observations(f, rank_seed(seed, rank) + 7, 0.05, 0.10)
    if exact_mask is not None and exact_mask.any():
        fx = sps.sps_photometry(table, ph, sps.PATH_EXACT, torch.tensor(thu[exact_mask], device="cuda")).cpu().numpy().astype(np.float64)
        dx, sx = W.noisy_observations(fx, exact_seed + 11, 0.05, 0.10)
        d[exact_mask] = dx; s[exact_mask] = sx
    return d.astype(np.float32), s.astype(np.float32)


def run_ours(args):
    import torch
    import paper_2506_19919_b200 as sps
    from paper_2506_19919_b200 import workloads as W

    rank = int(os.environ.get("RANK", 0)); world = int(os.environ.get("WORLD_SIZE", 1)); local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = dict(W.CONFIGS[args.workload])
    grid = W.make_grid(cfg["grid"]); prior = W.make_prior(); ph = sps.PriorHandle(prior.as_array())
    table = sps.sps_create_table(grid)
    peaks, peaks_src = _peaks()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")        # > 126 MB L2
    hmc = args.workload in ("c4_hmc", "c5_nuts")
    profile_step = None

    if hmc:
        n_gal = args.n_gal or cfg["n_gal"]
        if args.protocol == "paper":
            cfg["n_warmup"], cfg["n_sample"] = 100, 3000
        n_warmup, n_sample = args.n_warmup or cfg["n_warmup"], args.n_sample or cfg["n_sample"]
        mask = None
        if args.workload == "c5_nuts":
            # BASELINE.json configs[4]: NUTS, tree depth <= 8, exact path on a seeded 10 % of the galaxies
            mask = np.random.default_rng(cfg["seed"]).random(n_gal) < cfg["exact_fraction"]                   # True = exact
        d, s = make_hmc_inputs(sps, W, table, ph, prior, n_gal, cfg["seed"], rank, mask, cfg["seed"])
        d_host = torch.from_numpy(d).pin_memory(); s_host = torch.from_numpy(s).pin_memory()                   # (complete before pinning)
        d_dev = d_host.cuda(); s_dev = s_host.cuda()
        kw = dict(sampler=sps.SAMPLER_HMC, path=sps.PATH_APPROX, n_chain=cfg["n_chain"], n_warmup=n_warmup, n_sample=n_sample,
                  n_leapfrog=cfg.get("n_leapfrog", 0), eps0=0.01, seed=cfg["seed"])
        evals_per_step = n_gal * cfg["n_chain"] * (n_warmup + n_sample) * cfg.get("n_leapfrog", 0)
        if args.workload == "c5_nuts":
            kw.update(sampler=sps.SAMPLER_NUTS, max_depth=cfg["max_depth"], path_of_gal=torch.tensor((~mask).astype(np.int32), device="cuda"))
            kw.pop("n_leapfrog")
        units_per_step = n_gal                                                   # galaxy posteriors
        last = {}

        def step():
            last["out"] = sps.sps_hmc_run(table, ph, d_dev, s_dev, **kw)

        def step_e2e():
            dd = d_host.cuda(non_blocking=True); ss = s_host.cuda(non_blocking=True)
            out = sps.sps_hmc_run(table, ph, dd, ss, **kw)
            return out["mean"].cpu(), out["sd"].cpu(), out["rhat"].cpu()

        def profile_step():                                                      # a short run of the same launch shape, for kernel times
            sps.sps_hmc_run(table, ph, d_dev, s_dev, **{**kw, "n_warmup": min(n_warmup, 12), "n_sample": min(n_sample, 12)})
        h2d = d_host.numel() * 4 * 2
        d2h = n_gal * cfg["n_chain"] * 13 * 4 * 2 + n_gal * 13 * 4
        metric, unit, to_value = "galaxy posteriors/GPU-minute", "posteriors/min", lambda units, sec: 60.0 * units / sec
        rows_per_launch = n_gal * cfg["n_chain"]
    else:
        n = args.n_rows or cfg["batch"]
        path = sps.PATH_APPROX if args.workload == "c3_approx" else sps.PATH_EXACT
        thu = W.draw_theta_unbounded(prior, n, rank_seed(cfg["seed"], rank), z_uniform=(0.1, 3.0)).astype(np.float32)
        fb = np.random.default_rng(cfg["seed"]).normal(size=(n, grid.n_band)).astype(np.float32)
        th_host = torch.from_numpy(thu).pin_memory(); fb_host = torch.from_numpy(fb).pin_memory()
        th_dev = th_host.cuda(); fb_dev = fb_host.cuda()
        evals_per_step = n; units_per_step = n
        step = lambda: sps.sps_photometry(table, ph, path, th_dev, True, fb_dev)
        profile_step = step

        def step_e2e():
            a = th_host.cuda(non_blocking=True); b = fb_host.cuda(non_blocking=True)
            fl, tb = sps.sps_photometry(table, ph, path, a, True, b)
            return fl.cpu(), tb.cpu()
        h2d = n * (13 + grid.n_band) * 4; d2h = n * (13 + grid.n_band) * 4
        metric, unit, to_value = "flux+gradient evaluations/s", "evals/s", lambda units, sec: units / sec
        rows_per_launch = n

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    # ---- timed region 1: inputs resident in HBM, the code path users get (no per-kernel profiling, CUDA graphs on) -----
    launches0 = sps.sps_launch_count()
    clocks = ClockSampler(local); clocks.start()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_region = time.perf_counter()
    for a, b in ev:
        flush.fill_(1)                                                          # L2 flush between timed iterations
        a.record(); step(); b.record()
    barrier()
    launches = sps.sps_launch_count() - launches0
    # short workloads: keep the device under the same load (untimed) until the sampler has seen >= 1 s of it
    while time.perf_counter() - t_region < 1.2 and not hmc:
        for _ in range(20):
            step()
        torch.cuda.synchronize()
    clk = clocks.stop()
    dev_s = sum(a.elapsed_time(b) for a, b in ev) / 1e3
    # ---- timed region 2: end to end through the public API with host buffers -----------------------
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps if not args.no_e2e else 0):
        step_e2e()
    barrier()
    e2e_s = (time.perf_counter() - t0) if not args.no_e2e else float("inf")
    dev_s, e2e_s = max_over_ranks([dev_s, e2e_s], dist, device="cuda")
    # ---- untimed: per-kernel event timing of the same launch shape, and the pipe peaks of this run -----------------------
    sps.sps_profile(True, 4)
    profile_step()
    torch.cuda.synchronize()
    prof = {k: sps.sps_profile_read(k) for k in ("prologue", "approx_contract", "epilogue", "exact_fwd", "exact_bwd")}
    sps.sps_profile(False, 1)
    pipe = {"mufu_per_s": sps.sps_measure_peak("mufu"), "ffma_per_s": sps.sps_measure_peak("ffma")}
    extra = {}
    if hmc:
        o = last["out"]
        conv = float((o["rhat"].max(1).values < 1.2).float().mean().item())
        extra = {"rhat_below_1p2": conv, "median_ess": float(o["ess"][:, :13].min(1).values.median().item())}
        if args.workload == "c5_nuts":
            evals_per_step = int(o["n_leapfrog"].sum().item())
            hist = o["depth_hist"].cpu().numpy().tolist()
            extra.update({"mean_leapfrogs_per_transition": evals_per_step / (n_gal * cfg["n_chain"] * (n_warmup + n_sample)),
                          "divergences": int(o["divergences"].sum().item()), "tree_depth_hist": hist})
    pairs = sps.sps_exact_last_work(table) if args.workload == "c2_exact" else 0
    if rank != 0:
        return
    value = to_value(aggregate_throughput(units_per_step * args.steps, world, dev_s), 1.0)
    out = {"metric": metric, "value": value, "unit": unit}
    if hmc:
        # a fit counts as converged at R-hat < 1.2; beside the raw figure, the converged ones
        out["rhat_below_1p2"] = extra.pop("rhat_below_1p2")
        out["converged_posteriors_per_min"] = value * out["rhat_below_1p2"]
    out.update({"n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * dev_s / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic (seeded stand-in SSP spectra, Gaussian filters, prior-drawn galaxies)",
                "config": {"workload": args.workload, "protocol": args.protocol, **{k: v for k, v in cfg.items() if k != "seed"},
                           "n_gal_per_gpu": args.n_gal or cfg.get("n_gal"), "l2": "flushed between timed steps (256 MB write)"},
                "loglike_grad_evals_per_s": evals_per_step * args.steps * world / dev_s,
                "e2e": {"value": to_value(aggregate_throughput(units_per_step * args.steps, world, e2e_s), 1.0), "unit": unit, "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h},
                "gpu_launches": int(launches), "clocks": clk, "impl": "ours", **extra})
    kernel_ms = {k: {"avg_ms": v[0] / v[1], "launches_profiled": v[2]} for k, v in prof.items() if v[1]}
    share = {k: v["avg_ms"] * v["launches_profiled"] for k, v in kernel_ms.items()}
    tot = sum(share.values())
    for k in kernel_ms:
        kernel_ms[k]["share_of_profiled_kernels"] = share[k] / tot
    dom = max(share, key=share.get)                                              # the dominant kernel of THIS run
    out["kernel_ms"] = kernel_ms
    roofs = {k: kernel_roofline(k, kernel_ms[k]["avg_ms"] * 1e-3, rows_per_launch, grid, peaks, peaks_src, pipe, hmc, pairs) for k in kernel_ms}
    out["roofline"] = roofs[dom]
    out["roofline_step"] = [roofs[k] for k in kernel_ms if k != dom]
    out["evaluation"] = evaluation_roofline(args.workload, kernel_ms, dev_s / args.steps, evals_per_step, rows_per_launch, grid, peaks, peaks_src, pipe, pairs)
    out["pipe_peaks"] = {**pipe, "how": "sps_measure_peak: 64 warps/SM of 8 independent ex2.approx / fma chains, CUDA events, this run"}
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, args.protocol, budget_s=args.cpu_budget)
    print(json.dumps(out))
