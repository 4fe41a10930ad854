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
            last["prof"] = sps.sps_hmc_run(table, ph, d_dev, s_dev, **{**kw, "n_warmup": min(n_warmup, 12), "n_sample": min(n_sample, 12)})
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
    step_ms = [a.elapsed_time(b) for a, b in ev]                                # (this rank's; an occasional step on a shared box runs ~15 % long)
    dev_s = sum(step_ms) / 1e3
    # ---- timed region 2: end to end through the public API with host buffers -----------------------
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps if not args.no_e2e else 0):
        step_e2e()
    barrier()
    e2e_s = (time.perf_counter() - t0) if not args.no_e2e else float("inf")
    dev_s, e2e_s = max_over_ranks([dev_s, e2e_s], dist, device="cuda")
    # ---- untimed: per-kernel event timing of the same launch shape, and the pipe peaks of this run -----------------------
    # every 4th launch of a kernel is timed (NUTS alternates the approximate and the exact rows' launches of the row kernels:
    # an odd stride samples both)
    sps.sps_profile(True, 3 if args.workload == "c5_nuts" else 4)
    sps.sps_exact_work_since(table)                                              # (reset)
    profile_step()
    torch.cuda.synchronize()
    pair_sum, pair_calls = sps.sps_exact_work_since(table)
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
    pairs = pair_sum // max(1, pair_calls)                                       # average exact-path work per launch of the profiled pass
    if rank != 0:
        return
    value = to_value(aggregate_throughput(units_per_step * args.steps, world, dev_s), 1.0)
    out = {"metric": metric, "value": value, "unit": unit}
    if hmc:
        # a fit counts as converged at R-hat < 1.2; beside the raw figure, the converged ones
        out["rhat_below_1p2"] = extra.pop("rhat_below_1p2")
        out["converged_posteriors_per_min"] = value * out["rhat_below_1p2"]
    out.update({"n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * dev_s / args.steps, "step_ms": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
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
    # rows per launch: the batch, except under NUTS, whose launches shrink as trees finish and are split by path: there the
    # average over the profiled pass = its row evaluations (sum of the chains' leapfrog counts) x the path's share / launches
    rows_k = {k: rows_per_launch for k in kernel_ms}
    if args.workload == "c5_nuts":
        prof_evals = float(last["prof"]["n_leapfrog"].sum().item())
        fx = cfg["exact_fraction"]
        share_k = {"prologue": 1.0, "epilogue": 1.0, "approx_contract": 1.0 - fx, "exact_fwd": fx, "exact_bwd": fx}
        rows_k = {k: max(1, int(round(prof_evals * share_k[k] / max(1, prof[k][2])))) for k in kernel_ms}
    roofs = {k: kernel_roofline(k, kernel_ms[k]["avg_ms"] * 1e-3, rows_k[k], grid, peaks, peaks_src, pipe, hmc, pairs) for k in kernel_ms}
    for k in kernel_ms:
        roofs[k]["rows_per_launch"] = rows_k[k]
    out["roofline"] = roofs[dom]
    out["roofline_step"] = [roofs[k] for k in kernel_ms if k != dom]
    out["evaluation"] = evaluation_roofline(args.workload, kernel_ms, dev_s / args.steps, evals_per_step, rows_per_launch, grid, peaks, peaks_src, pipe, pairs)
    out["pipe_peaks"] = {**pipe, "how": "sps_measure_peak: 64 warps/SM of 8 independent ex2.approx / fma chains, CUDA events, this run"}
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, args.protocol, budget_s=args.cpu_budget)
    print(json.dumps(out))


# ------------------------------------------------------------------------------------------------
# rooflines (DESIGN.md sections 5 and 6 derive every count used here)
# ------------------------------------------------------------------------------------------------
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures (profiles/), at the
# launch sizes named there; None where no capture of that launch size exists.
NCU_TRAFFIC = {
    ("prologue", 40000): 85.8e6, ("approx_contract", 40000): 59.0e6, ("epilogue", 40000): 140.1e6,   # profiles/r02_hmc_kernels_full.md
    ("exact_fwd", 8192): 96.4e6, ("exact_bwd", 8192): 252.1e6,                                        # profiles/r02_exact_gemm_full.md
}


# lts__t_sectors.sum x 32 B per launch from the same captures (every L2 access: SM loads, stores, TMA, atomics and the fills)
NCU_L2 = {("prologue", 40000): 384.1e6, ("approx_contract", 40000): 264.3e6, ("epilogue", 40000): 229.8e6}      # profiles/r02_hmc_kernels_full.md


def algorithmic_counts(grid):
    """Operations the METHOD needs per parameter row (13-parameter model), independent of this implementation
    (DESIGN.md 5.1 derives them from the quadrature that the 1e-5 weights tolerance requires)."""
    n_age, n_Z, n_band = grid.n_age, grid.n_Z, grid.n_band
    nodes = 2 * n_age + 64                                   # two Gauss points per age bin + the panels of the bins that reach t ~ 0
    c = {"quadrature_nodes": nodes}
    c["prologue_mufu"] = 5 * nodes + 2 * 13 + 3 * (n_Z - 1) + 4          # lg2, 2 ex2, rcp, 1/t per node; C1; MDF edges; z -> t_obs
    c["prologue_fma"] = 16 * nodes + 14 * n_age + 40
    c["epilogue_mufu"] = 2 * 13 + 3 * (n_Z - 1) + 5 * 13                   # C1 slopes, MDF densities, skew-normal prior
    c["epilogue_fma"] = (2 * 5 + 14) * n_age + 100
    c["contract_mufu"] = 7 * n_band                                       # dust at lambda_eff / (1+z)
    c["contract_fma"] = 6 * n_Z * n_band + 2 * 2 * n_Z * n_band + 200     # the sums over metallicity of P, m_bar, V
    c["contract_flop_fp32"] = 2 * 2 * (2 * n_age * n_Z * n_band)          # Eq. (6) forward + reverse over the two c_SSP arrays of the z cell
    c["hbm_bytes"] = 4 * (13 + n_band) * 2                                # theta + observations in, logP + gradient out (184 B)
    return c


def kernel_roofline(kernel, avg_s, rows, grid, peaks, peaks_src, pipe, hmc, pairs=0):
    base = {"kernel": kernel, "avg_launch_ms": 1e3 * avg_s, "traffic": NCU_TRAFFIC.get((kernel, rows))}
    if base["traffic"] is not None:                                               # achieved HBM and L2 rates of this kernel (north_star asks for both)
        base["achieved_hbm_gbs"] = base["traffic"] / avg_s / 1e9
    if NCU_L2.get((kernel, rows)) is not None:
        base["achieved_l2_gbs"] = NCU_L2[(kernel, rows)] / avg_s / 1e9
    C = algorithmic_counts(grid)
    tensor_peak = float(peaks["bf16_tflops_sustained" if hmc else "bf16_tflops"])
    tensor_note = ("sustained bf16 peak: the kernel runs inside a seconds-long step" if hmc else "burst bf16 peak: the kernel is timed in a short step") + f" ({peaks_src})"
    if kernel == "prologue":
        ach = C["prologue_mufu"] * rows / avg_s / 1e9
        peak = pipe["mufu_per_s"] / 1e9
        return {**base, "bound": "alu", "achieved": ach, "peak": peak, "unit": "G MUFU/s", "frac": ach / peak,
                "peak_note": f"special-function pipe, measured in this run (sps_measure_peak); achieved = {C['prologue_mufu']} algorithmic MUFU operations "
                             f"per row ({C['quadrature_nodes']} quadrature nodes x 5 + C1 + MDF edges: DESIGN.md 5.1), not this implementation's instruction count"}
    if kernel == "epilogue":
        bytes_row = 4 * (6 * grid.n_age + grid.n_Z + 16 + 13 + 13 + 1 + ((3 * 13 + 1) + 2 * 13 if hmc else 0))
        ach = bytes_row * rows / avg_s / 1e9
        peak = float(peaks["hbm_gbs"])
        return {**base, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "peak_note": f"HBM copy bandwidth ({peaks_src}); achieved = {bytes_row} bytes per row that this kernel must move as long as the per-bin "
                             "partials travel through HBM (DESIGN.md 5.1); the method itself needs 184 B per row"}
    if kernel == "approx_contract":
        flop = 3.0 * C["contract_flop_fp32"] * rows
        ach = flop / avg_s / 1e12
        return {**base, "bound": "tensor", "achieved": ach, "peak": tensor_peak, "unit": "TFLOP/s", "frac": ach / tensor_peak,
                "peak_note": f"{tensor_note}; achieved = 3 FP16 split products x {C['contract_flop_fp32']} fp32-equivalent flop per row (Eq. 6 forward + reverse)"}
    K = grid.n_age * grid.n_Z
    flop = 3.0 * 2.0 * K * float(pairs)
    ach = flop / avg_s / 1e12
    return {**base, "bound": "tensor", "achieved": ach, "peak": tensor_peak, "unit": "TFLOP/s", "frac": ach / tensor_peak,
            "peak_note": f"{tensor_note}; achieved = 3 BF16 split products x 2 x {K} flop x {pairs} (row, wavelength) pairs under a filter's support "
                         f"= {pairs / max(1, rows):.0f} of {grid.n_wave} wavelengths per row (skipped and padded columns never count)"}


def evaluation_roofline(workload, kernel_ms, step_s, evals_per_step, rows, grid, peaks, peaks_src, pipe, pairs):
    """One whole log-likelihood + gradient evaluation of `rows` rows: measured time against the bound
    max(t_MUFU, t_FMA, t_tensor, t_HBM) of the METHOD's operation counts at this run's measured peaks."""
    C = algorithmic_counts(grid)
    launches_per_step = max(1.0, evals_per_step / rows)
    measured_s = step_s / launches_per_step
    kernels_s = sum(v["avg_ms"] for v in kernel_ms.values()) * 1e-3
    mufu = (C["prologue_mufu"] + C["epilogue_mufu"] + (C["contract_mufu"] if workload != "c2_exact" else 0)) * rows / pipe["mufu_per_s"]
    fma = (C["prologue_fma"] + C["epilogue_fma"] + (C["contract_fma"] if workload != "c2_exact" else 0)) * rows / pipe["ffma_per_s"]
    if workload == "c2_exact":
        tensor = 2 * 3.0 * 2.0 * grid.n_age * grid.n_Z * float(pairs) / (float(peaks["bf16_tflops"]) * 1e12)      # forward + reverse GEMM
    else:
        tensor = 3.0 * C["contract_flop_fp32"] * rows / (float(peaks["bf16_tflops_sustained"]) * 1e12)
    hbm = C["hbm_bytes"] * rows / (float(peaks["hbm_gbs"]) * 1e9)
    terms = {"mufu": mufu, "fma": fma, "tensor": tensor, "hbm": hbm}
    binding = max(terms, key=terms.get)
    tr = [NCU_TRAFFIC.get((k, rows)) for k in kernel_ms]
    l2 = [NCU_L2.get((k, rows)) for k in kernel_ms]
    rates = {}
    if all(t is not None for t in tr):
        rates["achieved_hbm_gbs"] = sum(tr) / measured_s / 1e9
    if all(t is not None for t in l2):
        rates["achieved_l2_gbs"] = sum(l2) / measured_s / 1e9
    return {**rates, "rows": rows, "measured_us": 1e6 * measured_s, "sum_of_kernel_times_us": 1e6 * kernels_s, "bound_us": 1e6 * terms[binding], "binding": binding,
            "frac": terms[binding] / measured_s, "terms_us": {k: 1e6 * v for k, v in terms.items()},
            "algorithmic_hbm_bytes": C["hbm_bytes"] * rows, "dram_bytes_ncu": (sum(tr) if all(t is not None for t in tr) else None),
            "note": "bound = max over pipes of (algorithmic operations per row x rows / peak measured in this run); the pipes overlap, so the terms are not added"}


# ------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------------
_WK = {}


def _worker_init(workload, seed):
    from threadpoolctl import threadpool_limits
    from oracle import sps_model as M
    from paper_2506_19919_b200 import workloads as W
    threadpool_limits(limits=1)
    cfg = dict(W.CONFIGS[workload])
    grid = W.make_grid(cfg["grid"]); prior = W.make_prior()
    _WK.update(cfg=cfg, grid=grid, prior=prior, P=prior.as_array(), cssp=M.cssp_table(grid) if workload != "c2_exact" else None)


def _worker_galaxy(task):
    """One galaxy of the HMC workloads: n_chain chains x n_tr transitions of the oracle's sampler on the approximate path."""
    from oracle import sampler as S
    from oracle import sps_model as M
    from paper_2506_19919_b200 import workloads as W
    g, n_tr = task
    cfg, grid, prior, P, cssp = (_WK[k] for k in ("cfg", "grid", "prior", "P", "cssp"))
    n_chain, L = cfg["n_chain"], cfg.get("n_leapfrog", 16)
    thu = W.draw_theta_unbounded(prior, 1, cfg["seed"] + 1000 + g)
    f = M.photometry_approx(M.bound(thu, P)[0], grid, cssp)[0]
    d, s = W.noisy_observations(f, cfg["seed"] + 7 + g, 0.05, 0.10)
    gal = np.zeros(n_chain, int)
    fn = lambda th: M.logp_and_grad(th, grid, P, d[gal], s[gal], "approx", cssp)[:2]
    ids = np.arange(g * n_chain, (g + 1) * n_chain)
    S.run_chains(S.init_chains(P, cfg["seed"], ids, 13), fn, cfg["seed"], 0, n_tr, 0.01, "hmc", n_leapfrog=L, chain_ids=ids)
    return n_chain * n_tr * L


def _worker_rows(task):
    """A block of rows of the kernel-only workloads through the oracle (flux + full Jacobian)."""
    from oracle import sps_model as M
    from paper_2506_19919_b200 import workloads as W
    block, n, workload = task
    cfg, grid, prior, P, cssp = (_WK[k] for k in ("cfg", "grid", "prior", "P", "cssp"))
    th = M.bound(W.draw_theta_unbounded(prior, n, cfg["seed"] + block, z_uniform=(0.1, 3.0)), P)[0]
    (M.photometry_approx(th, grid, cssp) if workload == "c3_approx" else M.photometry_exact(th, grid))
    return n


def cpu_worker(workload, protocol, budget_s):
    """Runs in a process of its own (no CUDA context): the float64 oracle, as it stands, over all host cores."""
    import multiprocessing as mp
    from paper_2506_19919_b200 import workloads as W
    cores = os.cpu_count() or 1
    cfg = dict(W.CONFIGS[workload])
    if protocol == "paper":
        cfg["n_warmup"], cfg["n_sample"] = 100, 3000
    with mp.get_context("fork").Pool(cores, initializer=_worker_init, initargs=(workload, cfg["seed"])) as pool:
        pool.map(abs, range(cores))                                    # workers up, tables built (setup, untimed as for the GPU)
        if workload in ("c4_hmc", "c5_nuts"):
            n_gal = max(64, 4 * cores)
            t0 = time.perf_counter()
            pool.map(_worker_galaxy, [(g, 1) for g in range(cores)])   # calibration: one transition per galaxy on every core
            per_tr = (time.perf_counter() - t0)
            n_tr = int(max(2, min(200, budget_s / max(per_tr, 1e-3) / (n_gal / cores))))
            t0 = time.perf_counter()
            evals = sum(pool.map(_worker_galaxy, [(g, n_tr) for g in range(n_gal)]))
            sec = time.perf_counter() - t0
            L = cfg.get("n_leapfrog", 16)
            per_post = cfg["n_chain"] * (cfg["n_warmup"] + cfg["n_sample"]) * L
            return {"value": 60.0 * (evals / sec) / per_post, "unit": "posteriors/min", "cores": cores, "kind": "oracle",
                    "sample": f"{n_gal} galaxies x {cfg['n_chain']} chains x {n_tr} HMC transitions x {L} leapfrogs of the float64 numpy oracle over {cores} "
                              f"processes ({evals} loglike+grad evals in {sec:.1f} s), scaled linearly in galaxies and transitions to {per_post} evals per posterior",
                    "loglike_grad_evals_per_s": evals / sec}
        n = 2 if workload == "c2_exact" else 64
        t0 = time.perf_counter()
        pool.map(_worker_rows, [(b, n, workload) for b in range(cores)])
        per_block = time.perf_counter() - t0
        blocks = int(max(cores, min(4096, cores * budget_s / max(per_block, 1e-3))))
        t0 = time.perf_counter()
        done = sum(pool.map(_worker_rows, [(1000 + b, n, workload) for b in range(blocks)]))
        sec = time.perf_counter() - t0
        return {"value": done / sec, "unit": "evals/s", "cores": cores, "kind": "oracle",
                "sample": f"{done} rows of the workload's parameter draws through the float64 numpy oracle (flux + full Jacobian) over {cores} processes in {sec:.1f} s"}


def cpu_baseline(workload, protocol, budget_s=20.0):
    r = subprocess.run([sys.executable, os.path.abspath(__file__), "--cpu-worker", "--workload", workload, "--protocol", protocol,
                        "--cpu-budget", str(budget_s)], capture_output=True, text=True, timeout=600)
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    if r.returncode != 0 or not lines:
        return {"value": None, "unit": "", "cores": os.cpu_count(), "kind": "oracle", "sample": "failed: " + r.stderr[-300:]}
    return json.loads(lines[-1])


def run_reference(args):
    """--impl reference: there is no reference implementation (the paper ships no code); for this tier the reference arm
    is the oracle timed on the host cores.  Rank 0 alone runs it."""
    if int(os.environ.get("RANK", 0)) != 0:
        return
    from paper_2506_19919_b200 import workloads as W
    cfg = dict(W.CONFIGS[args.workload])
    if args.protocol == "paper":
        cfg["n_warmup"], cfg["n_sample"] = 100, 3000
    per_step = max(4.0, min(25.0, 100.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        cpu_baseline(args.workload, args.protocol, budget_s=2.0)
    t0 = time.perf_counter()
    res = [cpu_baseline(args.workload, args.protocol, budget_s=per_step) for _ in range(args.steps)]
    sec = time.perf_counter() - t0
    v = float(np.mean([r["value"] for r in res]))
    hmc = args.workload in ("c4_hmc", "c5_nuts")
    out = {"impl": "reference", "metric": "galaxy posteriors/GPU-minute" if hmc else "flux+gradient evaluations/s", "value": v,
           "unit": res[0]["unit"], "n_gpus": int(os.environ.get("WORLD_SIZE", 1)), "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * sec / max(1, args.steps), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic (seeded stand-in SSP spectra, Gaussian filters, prior-drawn galaxies)",
           "config": {"workload": args.workload, "protocol": args.protocol, **{k: v2 for k, v2 in cfg.items() if k != "seed"},
                      "n_gal_per_gpu": args.n_gal or cfg.get("n_gal"), "l2": "flushed between timed steps (256 MB write)"},
           "cpu_baseline": {**res[0], "value": v}, "e2e": {"value": v, "unit": res[0]["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4_hmc", choices=["c4_hmc", "c3_approx", "c2_exact", "c5_nuts"])
    ap.add_argument("--protocol", default="config", choices=["config", "paper"],
                    help="config: BASELINE.json's transition counts; paper: 100 adaptation + 3000 kept steps (PAPER.md:105)")
    ap.add_argument("--n-gal", type=int, default=0)
    ap.add_argument("--n-rows", type=int, default=0)
    ap.add_argument("--n-warmup", type=int, default=0)
    ap.add_argument("--n-sample", type=int, default=0)
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end leg (side workloads only; the e2e value is then 0)")
    ap.add_argument("--cpu-worker", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.cpu_worker:
        print(json.dumps(cpu_worker(args.workload, args.protocol, args.cpu_budget)))
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` on its own: one rank per GPU under torchrun (the driver launches torchrun itself)
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        sys.exit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
