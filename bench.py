#!/usr/bin/env python
"""bench.py -- headline benchmark of the SPS hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4_hmc|c3_approx|c2_exact|c5_nuts]

Default workload = BASELINE.json configs[3] ("c4_hmc"): full HMC on the approximate path, 10,000 synthetic
galaxies x 4 chains x (500 warmup + 500 samples) x 16 leapfrog steps; metric = galaxy posteriors per GPU-minute.
One "step" = one complete sps_hmc_run over the batch.  With N > 1 (torchrun) every rank runs the same number of
galaxies (weak scaling; galaxies are independent, no data-path collective) and the value is the job aggregate.
Prints ONE JSON line on rank 0.
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
                                          "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
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
def make_hmc_inputs(sps, W, table, ph, prior, n_gal, seed, rank=0):
    """True parameters drawn from the prior; observed fluxes = the library's own approximate-path photometry of the
    truth with 5-10 % Gaussian noise (bench.py may not touch oracle/ outside the cpu_baseline leg)."""
    import torch
    thu = W.draw_theta_unbounded(prior, n_gal, rank_seed(seed, rank)).astype(np.float32)
    f = sps.sps_photometry(table, ph, sps.PATH_APPROX, torch.tensor(thu, device="cuda")).cpu().numpy().astype(np.float64)
    d, s = W.noisy_observations(f, rank_seed(seed, rank) + 7, 0.05, 0.10)
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

    if args.workload in ("c4_hmc", "c5_nuts"):
        n_gal = args.n_gal or cfg["n_gal"]
        d, s = make_hmc_inputs(sps, W, table, ph, prior, n_gal, cfg["seed"], rank)
        d_host = torch.from_numpy(d).pin_memory(); s_host = torch.from_numpy(s).pin_memory()
        d_dev = d_host.cuda(); s_dev = s_host.cuda()
        kw = dict(sampler=sps.SAMPLER_HMC, path=sps.PATH_APPROX, n_chain=cfg["n_chain"], n_warmup=args.n_warmup or cfg["n_warmup"],
                  n_sample=args.n_sample or cfg["n_sample"], n_leapfrog=cfg.get("n_leapfrog", 0), eps0=0.01, seed=cfg["seed"])
        evals_per_step = n_gal * cfg["n_chain"] * (kw["n_warmup"] + kw["n_sample"]) * cfg.get("n_leapfrog", 0)
        if args.workload == "c5_nuts":
            # BASELINE.json configs[4]: NUTS, tree depth <= 8, exact path on a seeded 10 % of the galaxies (their data come
            # from the exact path), approximate path on the rest; evaluations are counted from the chains' leapfrog totals
            mask = (np.random.default_rng(cfg["seed"]).random(n_gal) >= cfg["exact_fraction"]).astype(np.int32)      # 1 = approximate
            thu_x = W.draw_theta_unbounded(prior, n_gal, rank_seed(cfg["seed"], rank)).astype(np.float32)[mask == 0]
            fx = sps.sps_photometry(table, ph, sps.PATH_EXACT, torch.tensor(thu_x, device="cuda")).cpu().numpy().astype(np.float64)
            dx, sx = W.noisy_observations(fx, cfg["seed"] + 11, 0.05, 0.10)
            d[mask == 0] = dx; s[mask == 0] = sx
            kw.update(sampler=sps.SAMPLER_NUTS, max_depth=cfg["max_depth"], path_of_gal=torch.tensor(mask, device="cuda"))
            kw.pop("n_leapfrog")
        units_per_step = n_gal                                                   # galaxy posteriors
        last = {}

        def step():
            last["out"] = sps.sps_hmc_run(table, ph, d_dev, s_dev, **kw)

        def step_e2e():
            dd = d_host.cuda(non_blocking=True); ss = s_host.cuda(non_blocking=True)
            out = sps.sps_hmc_run(table, ph, dd, ss, **kw)
            return out["mean"].cpu(), out["sd"].cpu(), out["rhat"].cpu()
        h2d = d_host.numel() * 4 * 2
        d2h = n_gal * cfg["n_chain"] * 13 * 4 * 2 + n_gal * 13 * 4
        metric, unit, to_value = "galaxy posteriors/GPU-minute", "posteriors/min", lambda units, sec: 60.0 * units / sec
        dom_kernel, rows_per_launch = "approx_contract", n_gal * cfg["n_chain"]
    else:
        n = args.n_rows or cfg["batch"]
        path = sps.PATH_APPROX if args.workload == "c3_approx" else sps.PATH_EXACT
        thu = W.draw_theta_unbounded(prior, n, rank_seed(cfg["seed"], rank), z_uniform=(0.1, 3.0)).astype(np.float32)
        fb = np.random.default_rng(cfg["seed"]).normal(size=(n, grid.n_band)).astype(np.float32)
        th_host = torch.from_numpy(thu).pin_memory(); fb_host = torch.from_numpy(fb).pin_memory()
        th_dev = th_host.cuda(); fb_dev = fb_host.cuda()
        evals_per_step = n; units_per_step = n
        step = lambda: sps.sps_photometry(table, ph, path, th_dev, True, fb_dev)

        def step_e2e():
            a = th_host.cuda(non_blocking=True); b = fb_host.cuda(non_blocking=True)
            fl, tb = sps.sps_photometry(table, ph, path, a, True, b)
            return fl.cpu(), tb.cpu()
        h2d = n * (13 + grid.n_band) * 4; d2h = n * (13 + grid.n_band) * 4
        metric, unit, to_value = "flux+gradient evaluations/s", "evals/s", lambda units, sec: units / sec
        dom_kernel, rows_per_launch = ("approx_contract" if path == sps.PATH_APPROX else "exact_fwd"), n

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    # ---- timed region 1: inputs resident in HBM ---------------------------------------------------
    sps.sps_profile(True, 8)
    launches0 = sps.sps_launch_count()
    clocks = ClockSampler(local); clocks.start()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.fill_(1)                                                          # L2 flush between timed iterations
        a.record(); step(); b.record()
    barrier()
    clk = clocks.stop()
    dev_s = sum(a.elapsed_time(b) for a, b in ev) / 1e3
    launches = sps.sps_launch_count() - launches0
    prof = {k: sps.sps_profile_read(k) for k in ("prologue", "approx_contract", "epilogue", "exact_fwd", "exact_bwd")}
    sps.sps_profile(False, 1)
    # ---- timed region 2: end to end through the public API with host buffers -----------------------
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps if not args.no_e2e else 0):
        step_e2e()
    barrier()
    e2e_s = (time.perf_counter() - t0) if not args.no_e2e else float("inf")
    dev_s, e2e_s = max_over_ranks([dev_s, e2e_s], dist, device="cuda")
    extra = {}
    if args.workload == "c5_nuts":
        o = last["out"]
        evals_per_step = int(o["n_leapfrog"].sum().item())
        extra = {"mean_leapfrogs_per_transition": evals_per_step / (n_gal * cfg["n_chain"] * (kw["n_warmup"] + kw["n_sample"])),
                 "rhat_below_1p2": float((o["rhat"].max(1).values < 1.2).float().mean().item()), "divergences": int(o["divergences"].sum().item())}
    elif args.workload == "c4_hmc":
        extra = {"rhat_below_1p2": float((last["out"]["rhat"].max(1).values < 1.2).float().mean().item())}
    pairs = sps.sps_exact_last_work(table) if args.workload == "c2_exact" else 0
    if rank != 0:
        return
    value = to_value(aggregate_throughput(units_per_step * args.steps, world, dev_s), 1.0)
    out = {"metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * dev_s / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic (seeded stand-in SSP spectra, Gaussian filters, prior-drawn galaxies)",
           "config": {"workload": args.workload, **{k: v for k, v in cfg.items() if k != "seed"},
                      "n_gal_per_gpu": args.n_gal or cfg.get("n_gal"), "l2": "flushed between timed steps (256 MB write)"},
           "loglike_grad_evals_per_s": evals_per_step * args.steps * world / dev_s,
           "e2e": {"value": to_value(aggregate_throughput(units_per_step * args.steps, world, e2e_s), 1.0), "unit": unit, "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": d2h},
           "gpu_launches": int(launches), "clocks": clk, "impl": "ours", **extra}
    out["roofline"] = roofline(prof, dom_kernel, rows_per_launch, grid, peaks, peaks_src, pairs)
    out["roofline_step"] = [r for r in (row_kernel_roofline(prof, k, rows_per_launch, grid, peaks, peaks_src, args.workload in ("c4_hmc", "c5_nuts")) for k in ("prologue", "epilogue")) if r]
    out["kernel_ms"] = {k: {"avg_ms": (v[0] / v[1] if v[1] else None), "launches": v[2]} for k, v in prof.items() if v[2]}
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, cfg, budget_s=args.cpu_budget)
    print(json.dumps(out))


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed ncu --set full
# captures (profiles/), taken at the launch sizes named there; None where no capture of that launch size exists.
NCU_TRAFFIC = {
    ("approx_contract", 40000): 84.8e6,   # profiles/r01_hmc_kernels_full.md: 79.78 MB read + 5.00 MB written (40,000 rows per launch)
    ("exact_fwd", 8192): 74.2e6,          # profiles/r01_exact_gemm_full.md: 72.18 MB read + 2.02 MB written (8,192 rows per launch)
}


# warp instructions per row of the two row kernels, from the committed ncu --set full capture (smsp__inst_executed.sum over
# 40,000 rows, profiles/r01_hmc_kernels_full.md): the prologue's work is transcendental-heavy quadrature, not a byte stream.
NCU_WARP_INST_PER_ROW = {"prologue": 62160578 / 40000.0, "epilogue": 29196415 / 40000.0}
NCU_TRAFFIC_ROW_KERNELS = {("prologue", 40000): 71.1e6, ("epilogue", 40000): 139.9e6}   # same capture: dram read + written per launch


def row_kernel_roofline(prof, kernel, rows_per_launch, grid, peaks, peaks_src, fused_leapfrog):
    """The other kernels of an evaluation, reported beside the contraction's roofline.
    prologue (a0-a5): instruction-issue bound ("alu"): achieved = ncu's warp instructions per row x rows per launch / the live
    launch time, against 148 SMs x 4 schedulers x the maximum SM clock (one warp instruction per scheduler per clock).  The
    instruction count is this implementation's, not an algorithmic minimum: the fraction says how busy the issue slots are.
    epilogue (a10 reverse of a0-a5 + the fused leapfrog update): an HBM stream: algorithmic bytes per row = the five stored
    per-bin vectors and a_bar (n_age words each), m_bar (n_Z), the 64-byte row scalars, theta, the leapfrog operands
    (p, theta, inverse mass, eps; sampler workloads only) in; grad, logp, p, theta out; against the measured HBM copy bandwidth."""
    ms, timed, allc = prof[kernel]
    if not timed:
        return None
    avg_s = ms / timed / 1e3
    base = {"kernel": kernel, "avg_launch_ms": 1e3 * avg_s, "timed_launches": timed, "launches": allc,
            "traffic": NCU_TRAFFIC_ROW_KERNELS.get((kernel, rows_per_launch))}
    if kernel == "prologue":
        clock_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        peak = 148 * 4 * clock_hz / 1e9
        ach = NCU_WARP_INST_PER_ROW[kernel] * rows_per_launch / avg_s / 1e9
        return {**base, "bound": "alu", "achieved": ach, "peak": peak, "unit": "G warp-inst/s", "frac": ach / peak,
                "peak_note": f"issue-slot peak = 148 SM x 4 schedulers x {clock_hz / 1e6:.0f} MHz ({peaks_src} clock); achieved = "
                             f"{NCU_WARP_INST_PER_ROW[kernel]:.0f} warp instructions per row (ncu, profiles/r01_hmc_kernels_full.md)"}
    bytes_row = 4 * (6 * grid.n_age + grid.n_Z + 16 + 13 + 13 + 1 + ((3 * 13 + 1) + 2 * 13 if fused_leapfrog else 0))
    ach = bytes_row * rows_per_launch / avg_s / 1e9
    peak = float(peaks["hbm_gbs"])
    return {**base, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
            "peak_note": f"HBM copy bandwidth ({peaks_src}); achieved = {bytes_row} algorithmic bytes per row; the kernel also issues "
                         f"{NCU_WARP_INST_PER_ROW[kernel]:.0f} warp instructions per row (issue slots 76 % busy in the ncu capture)"}


def roofline(prof, kernel, rows_per_launch, grid, peaks, peaks_src, pairs=0):
    """Roofline of the dominant kernel.
    approx_contract: tensor bound (tcgen05 kernel, FP16 two-term split): per row the forward + reverse pass over the two
    c_SSP arrays of its z cell is 2 MAC per table word = 4 * 2 n_age*n_Z*n_band flop, times the 3 split products, against the
    measured bf16 burst peak (FP16 runs at the same rate); the table operands are L2 resident, so there is no HBM stream.
    (The fp32 SIMT kernel that serves other table shapes is FMA-pipe bound: DESIGN.md 5.2.)
    exact_fwd: tensor bound: 3 split products x 2 x n_age*n_Z flop per (row, wavelength) pair under some filter's support
    (sps_exact_last_work: skipped and padded columns never count), against the measured bf16 burst peak (BF16X3)."""
    ms, timed, allc = prof[kernel]
    if not timed:
        return {"bound": "alu", "achieved": None, "peak": None, "unit": "TFLOP/s", "frac": None, "traffic": None}
    avg_s = ms / timed / 1e3
    if kernel == "approx_contract":
        words = 2 * grid.n_age * grid.n_Z * grid.n_band
        flop = 3.0 * 2.0 * 2.0 * words * rows_per_launch
        peak = float(peaks["bf16_tflops"])
        bound, note = "tensor", (f"bf16 burst peak ({peaks_src}; FP16 operands, same rate); achieved = 3 FP16 split products x 2 passes x 2 x "
                                 f"{words} table words per row; the kernel is bound by its per-row staging / band step, not by the tensor pipe (DESIGN.md 5.2)")
    else:
        K = grid.n_age * grid.n_Z
        flop = 3.0 * 2.0 * K * float(pairs)
        peak = float(peaks["bf16_tflops"])
        bound, note = "tensor", (f"bf16 burst peak ({peaks_src}); achieved = 3 BF16 split products x 2 x {K} flop x {pairs} (row, wavelength) "
                                 f"pairs under a filter's support = {pairs / max(1, rows_per_launch):.0f} of {grid.n_wave} wavelengths per row")
    ach = flop / avg_s / 1e12
    return {"bound": bound, "kernel": kernel, "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
            "traffic": NCU_TRAFFIC.get((kernel, rows_per_launch)), "avg_launch_ms": 1e3 * avg_s, "timed_launches": timed, "launches": allc,
            "peak_note": note}


def cpu_baseline(workload, cfg, budget_s=20.0):
    """The float64 oracle, as it stands, timed on this box's host cores on a bounded sample of the same workload."""
    from threadpoolctl import threadpool_limits
    from oracle import sampler as S
    from oracle import sps_model as M
    from paper_2506_19919_b200 import workloads as W
    grid = W.make_grid(cfg["grid"]); prior = W.make_prior(); P = prior.as_array()
    with threadpool_limits(limits=1):
        if workload in ("c4_hmc", "c5_nuts"):
            cssp = M.cssp_table(grid, M.z_grid(grid))          # setup, untimed (as for the GPU)
            n_gal, n_chain, L = 2, cfg["n_chain"], cfg.get("n_leapfrog", 16)
            thu = W.draw_theta_unbounded(prior, n_gal, cfg["seed"])
            f = M.photometry_approx(M.bound(thu, P)[0], grid, cssp)[0]
            d, s = W.noisy_observations(f, cfg["seed"] + 7, 0.05, 0.10)
            gal = np.repeat(np.arange(n_gal), n_chain)
            fn = lambda th: M.logp_and_grad(th, grid, P, d[gal], s[gal], "approx", cssp)[:2]
            th0 = S.init_chains(P, cfg["seed"], np.arange(n_gal * n_chain), 13)
            n_tr, t0 = 0, time.perf_counter()
            while time.perf_counter() - t0 < budget_s:
                S.run_chains(th0, fn, cfg["seed"], 0, 2, 0.01, "hmc", n_leapfrog=L)
                n_tr += 2
            sec = time.perf_counter() - t0
            evals = n_gal * n_chain * n_tr * L
            per_post = n_chain * (cfg["n_warmup"] + cfg["n_sample"]) * L
            return {"value": 60.0 * (evals / sec) / per_post, "unit": "posteriors/min", "cores": 1, "kind": "oracle",
                    "sample": f"{n_gal} galaxies x {n_chain} chains x {n_tr} HMC transitions x {L} leapfrogs of the float64 numpy oracle "
                              f"({evals} loglike+grad evals in {sec:.1f} s), scaled linearly to {per_post} evals per posterior",
                    "loglike_grad_evals_per_s": evals / sec}
        n = 8 if workload == "c2_exact" else 256
        thu = W.draw_theta_unbounded(prior, n, cfg["seed"], z_uniform=(0.1, 3.0))
        th = M.bound(thu, P)[0]
        cssp = M.cssp_table(grid) if workload == "c3_approx" else None
        done, t0 = 0, time.perf_counter()
        while time.perf_counter() - t0 < budget_s:
            (M.photometry_approx(th, grid, cssp) if workload == "c3_approx" else M.photometry_exact(th, grid))
            done += n
        sec = time.perf_counter() - t0
        return {"value": done / sec, "unit": "evals/s", "cores": 1, "kind": "oracle",
                "sample": f"{done} rows of the workload's parameter draws through the float64 numpy oracle (flux + full Jacobian)"}


def run_reference(args):
    """--impl reference: there is no reference implementation (the paper ships no code); for this tier the reference arm
    is the oracle timed on the host cores."""
    if int(os.environ.get("RANK", 0)) != 0:
        return
    from paper_2506_19919_b200 import workloads as W
    cfg = dict(W.CONFIGS[args.workload])
    per_step = max(5.0, min(30.0, 90.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        cpu_baseline(args.workload, cfg, budget_s=2.0)
    t0 = time.perf_counter()
    res = [cpu_baseline(args.workload, cfg, budget_s=per_step) for _ in range(args.steps)]
    sec = time.perf_counter() - t0
    v = float(np.mean([r["value"] for r in res]))
    hmc = args.workload in ("c4_hmc", "c5_nuts")
    out = {"impl": "reference", "metric": "galaxy posteriors/GPU-minute" if hmc else "flux+gradient evaluations/s", "value": v,
           "unit": res[0]["unit"], "n_gpus": int(os.environ.get("WORLD_SIZE", 1)), "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * sec / max(1, args.steps), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic", "config": {"workload": args.workload, **{k: v2 for k, v2 in cfg.items() if k != "seed"}},
           "cpu_baseline": {**res[0], "value": v}, "e2e": {"value": v, "unit": res[0]["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4_hmc", choices=["c4_hmc", "c3_approx", "c2_exact", "c5_nuts"])
    ap.add_argument("--n-gal", type=int, default=0)
    ap.add_argument("--n-rows", type=int, default=0)
    ap.add_argument("--n-warmup", type=int, default=0)
    ap.add_argument("--n-sample", type=int, default=0)
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end leg (side workloads only; the e2e value is then 0)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
