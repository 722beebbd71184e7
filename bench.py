#!/usr/bin/env python
"""bench.py — throughput of the Pulscan boxcar-search hot path on B200 (one JSON line on stdout, rank 0).

A "step" is one pass of the whole path (normalise + power, boxcar sweep over every width 1..zmax, exact evaluation of
marked blocks, significance, threshold, compaction) over one batch of synthetic spectra through `pulscan_search`.
Workload: BASELINE.json configs[2], the batched 2^22-bin DM-trial config the north_star quotes its target on
(256 × 4,194,305 complex64 bins = 8.59 GB: larger than L2, so consecutive steps cannot be served from cache).
`--config k` (1-5) selects another BASELINE config.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

N > 1: one process per GPU under torchrun; every rank searches its own full-size batch (weak scaling, no data-path
collective: spectra are independent); time = max over ranks, value = all ranks' bins / time.
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "fourier_bins_searched_per_sec_at_zmax"
UNIT = "bins/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config, 1-based (default 3 = configs[2])")
    ap.add_argument("--batch", type=int, default=0, help="override the config's batch (debugging only)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--log10-p-flag", type=float, default=0.0)
    ap.add_argument("--numharm", type=int, default=1, help="also search the harmonic-summed spectra Y_2..Y_numharm "
                    "(PAPER.md:L201-220; pulscan_search_harmonics; not the headline)")
    ap.add_argument("--fast-norm", action="store_true", help="the paper's approximate median-of-medians normalisation "
                    "(Alg. 1, PAPER.md:L624-650) instead of the exact one (not the headline: results differ)")
    ap.add_argument("--z-step", type=int, default=1, help="search every z_step-th drift only (PAPER.md:L152; not the headline)")
    ap.add_argument("--log-sampling", action="store_true", help="search z = 0, 1, 2, 4, ... only (PAPER.md:L411; not the headline)")
    return ap.parse_args()


def workload(args):
    from paper_2406_15186_b200 import synth
    wl = synth.CONFIGS[args.config]
    if args.batch:
        wl = wl.scaled(batch=args.batch)
    return wl


def config_dict(wl, n_gpus, args=None):
    sampling = "every width 1..zmax"
    norm = "median of medians, Alg. 1 (approximate)" if (args is not None and args.fast_norm) else "exact median/MAD"
    if args is not None and args.log_sampling:
        sampling = "drifts z = 0, 1, 2, 4, ... (PAPER.md:L411)"
    elif args is not None and args.z_step != 1:
        sampling = f"every {args.z_step}-th drift (PAPER.md:L152)"
    return {
        "widths_searched": sampling, "normalisation": norm,
        "workload": f"BASELINE.json configs[{int(wl.name[3]) - 1}] ({wl.name}): {wl.batch} spectra x {wl.n_bins} complex64 bins "
                    f"per GPU, zmax={wl.zmax}, norm_block={wl.norm_block}, block_width={wl.block_width}, "
                    f"sigma_threshold={wl.sigma_threshold}",
        "n_bins": wl.n_bins, "batch_per_gpu": wl.batch, "zmax": wl.zmax, "norm_block": wl.norm_block,
        "block_width": wl.block_width, "sigma_threshold": wl.sigma_threshold,
        "input_bytes_per_gpu": wl.batch * wl.n_bins * 8,
        "cache": cache_policy(wl)[1],
        "parallelism": f"dp{n_gpus} over spectra, no collective on the data path",
    }


L2_BYTES = 126e6


def cache_policy(wl):
    """(number of distinct input copies the steps rotate over, what the JSON line says about the cache).  An input larger than
    twice the L2 cannot be served from cache between steps; a smaller one (configs 1-2) is replicated until the copies
    together exceed 2.5 x L2 and step i reads copy i mod R, so that no step finds its input in L2."""
    nbytes = wl.batch * wl.n_bins * 8
    if nbytes > 2 * L2_BYTES:
        return 1, "inputs larger than L2 (no flush needed)"
    r = max(8, int(2.5 * L2_BYTES // nbytes) + 1)
    return r, f"input rotated over {r} distinct copies ({r * nbytes / 1e6:.0f} MB > 2 x L2): no step finds its input in L2"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            p = [x.strip() for x in l.split(",")]
            if len(p) < 6:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for nm, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def measured_hbm_peak():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            return float(json.loads(f.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except (ValueError, KeyError):
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(kernel: str, cfg: int):
    """dram bytes per launch of `kernel` from the committed ncu summary (profiles/traffic.json), scaled per bin."""
    f = ROOT / "profiles" / "traffic.json"
    if not f.exists():
        return None
    try:
        t = json.loads(f.read_text())
        return t.get(f"cfg{cfg}", {}).get(kernel)
    except ValueError:
        return None


def cpu_baseline(wl, X_host_rows, budget_s=15.0, z_step=1, log_sampling=False):
    """The oracle, as it stands, on a bounded sample of the same spectra (host rows already in memory)."""
    import oracle
    import numpy as np
    oracle.build()
    t0 = time.perf_counter()
    oracle.search(X_host_rows[0], wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold, z_step=z_step, log_sampling=log_sampling)
    t1 = time.perf_counter() - t0
    extra = int(max(0, min(len(X_host_rows) - 1, round(budget_s / max(t1, 1e-3)) - 1)))
    t_all, n_sp = t1, 1
    if extra:
        t0 = time.perf_counter()
        oracle.search(np.ascontiguousarray(X_host_rows[1:1 + extra]), wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold,
                      z_step=z_step, log_sampling=log_sampling)
        t_all += time.perf_counter() - t0
        n_sp += extra
    return {"value": n_sp * wl.n_bins / t_all, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{n_sp} of {wl.batch} spectra of the workload ({n_sp * wl.n_bins} bins, all {wl.zmax} widths), "
                      f"{t_all:.1f} s wall"}


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores; each step is one spectrum of the workload."""
    from paper_2406_15186_b200 import dist as pdist, synth
    rank, _, world = pdist.env_rank_world()
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    wl = workload(args)
    X, _ = synth.make_spectra(wl, device="cpu", spectra=range(min(wl.batch, 2)))
    rows = X.numpy()
    per_step = 1
    for _ in range(args.warmup):
        oracle.search(rows[0], wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold, z_step=args.z_step, log_sampling=args.log_sampling)
    t0 = time.perf_counter()
    for i in range(args.steps):
        oracle.search(rows[i % len(rows)], wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold, z_step=args.z_step,
                      log_sampling=args.log_sampling)
    dt = time.perf_counter() - t0
    value = args.steps * per_step * wl.n_bins / dt
    sample = f"{per_step} spectrum of the workload per step ({wl.n_bins} bins x {wl.zmax} widths)"
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_dict(wl, args.gpus, args),
        "bin_widths_per_sec": value * wl.zmax,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)
    return 0


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as tdist
    from paper_2406_15186_b200 import binding, dist as pdist, synth

    rank, local_rank, world = pdist.env_rank_world()
    if world > 1:
        torch.cuda.set_device(local_rank)
        tdist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", torch.cuda.current_device())
    wl = workload(args).scaled(seed=workload(args).seed + 1000 * rank)  # every rank its own spectra
    X, _ = synth.make_spectra(wl, device=dev)
    bins = wl.batch * wl.n_bins
    steps, warm = args.steps, max(args.warmup, 3)
    n_copies = cache_policy(wl)[0]
    copies = [X] + [X.clone() for _ in range(n_copies - 1)]      # small inputs: rotate so that L2 never holds the next one

    plan = binding.Plan(wl.n_bins, wl.batch, wl.zmax, wl.block_width, wl.sigma_threshold, norm_block=wl.norm_block,
                        tile=args.tile, log10_p_flag=args.log10_p_flag, z_step=args.z_step, log_sampling=args.log_sampling,
                        numharm=args.numharm, median_of_medians=args.fast_norm)
    plan.attach(dev)
    run_search = plan.search_harmonics if args.numharm > 1 else plan.search
    plan.set_profiling(warm + steps)
    stream = torch.cuda.current_stream()
    for i in range(warm):
        run_search(copies[i % n_copies], stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(); pdist.barrier(); torch.cuda.synchronize()
    with ClockSampler(torch.cuda.current_device()) as clk:
        e0.record(stream)
        for i in range(steps):
            run_search(copies[(warm + i) % n_copies], stream)
        e1.record(stream)
        torch.cuda.synchronize(); pdist.barrier(); torch.cuda.synchronize()
    ms_total = pdist.max_over_ranks(e0.elapsed_time(e1))
    total_bins = pdist.sum_over_ranks(bins)
    ms_step = ms_total / steps
    value = total_bins / (ms_step * 1e-3)
    n_cand = int(plan.d_count.item())
    stats = plan.stats()
    flagged = int(stats[0])

    # per-kernel device times of the timed steps (CUDA events recorded by the library on the launching stream)
    if args.numharm > 1:   # the per-stage events belong to pulscan_search: the whole step is held against the roofline
        peak, peak_src = measured_hbm_peak()
        gbs = lambda nbytes, t_ms: nbytes / (t_ms * 1e-3) / 1e9
        H = args.numharm
        # least own traffic of the harmonic path, per input bin: 8 read + 4 (P written) + 4 (P read by the sweep of Y_1) + the
        # decimation pass (P read at least once: 4; each Y_H written: 4/H) + each Y_H read by its sweep (4/H).  A lower bound:
        # the decimation pass re-reads P from DRAM where a row's reuse distance exceeds the L2
        own = 8 + 4 + 4 + 4 + sum(8.0 / h for h in range(2, H + 1))
        roofline = {"bound": "hbm", "kernel": "whole step (pulscan_search_harmonics: kernel (a), harmonic_sum_kernel, sweep + refine "
                    "+ exact per Y_H)", "achieved": gbs(8 * bins, ms_step), "peak": peak, "unit": "GB/s",
                    "frac": gbs(8 * bins, ms_step) / peak, "algorithmic_bytes_per_bin": 8, "algorithmic_bytes_per_launch": 8 * bins,
                    "own_bytes_per_bin": own, "frac_own_traffic": gbs(own * bins, ms_step) / peak, "traffic": None,
                    "peak_source": peak_src, "path_frac": gbs(8 * bins, ms_step) / peak if world == 1 else None}
        e2e = None
        if not args.no_e2e:   # host buffer -> H2D -> pulscan_search_harmonics -> D2H of count and records, wall clock
            Xh = torch.empty(X.shape, dtype=X.dtype, pin_memory=True)
            Xh.copy_(X)
            Xd = torch.empty_like(X)
            def one():
                Xd.copy_(Xh, non_blocking=True)
                plan.search_harmonics(Xd, stream)
                return plan.hcandidates()
            rec = one()
            torch.cuda.synchronize(); pdist.barrier()
            t0 = time.perf_counter()
            for _ in range(args.e2e_steps):
                rec = one()
            dt = pdist.max_over_ranks(time.perf_counter() - t0)
            assert len(rec) == n_cand, "host-buffer search disagrees with device-buffer search"
            e2e = {"value": total_bins * args.e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(Xh.numel() * 8),
                   "d2h_bytes_per_step": int(4 + 24 * len(rec)), "steps": args.e2e_steps, "ms_per_step": 1e3 * dt / args.e2e_steps}
            del Xd
        cpu = None
        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            import oracle
            oracle.build()
            rows = X[: min(wl.batch, 16)].cpu().numpy()
            t0 = time.perf_counter()
            oracle.search_harmonics(rows[:1], wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold, H, z_step=args.z_step,
                                    log_sampling=args.log_sampling, median_of_medians=args.fast_norm)
            t1 = time.perf_counter() - t0
            extra = int(max(0, min(len(rows) - 1, round(15.0 / max(t1, 1e-3)) - 1)))
            if extra:
                t0 = time.perf_counter()
                oracle.search_harmonics(rows[1:1 + extra], wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold, H,
                                        z_step=args.z_step, log_sampling=args.log_sampling, median_of_medians=args.fast_norm)
                t1 += time.perf_counter() - t0
            cpu = {"value": (1 + extra) * wl.n_bins / t1, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                   "sample": f"{1 + extra} of {wl.batch} spectra of the workload, harmonic sums up to {H}, {t1:.1f} s wall"}
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
                              "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                              "dtype": "f32", "data": "synthetic", "config": dict(config_dict(wl, world, args), numharm=args.numharm),
                              "bin_widths_per_sec": value * wl.zmax, "candidates_per_step": n_cand, "clocks": clk.summary(),
                              "e2e": e2e, "gpu_launches": (plan.launches_per_search + 1 + 3 * (args.numharm - 1)) * steps,
                              "roofline": roofline, "cpu_baseline": cpu}), flush=True)
        plan.destroy()
        if world > 1:
            tdist.destroy_process_group()
        return 0
    prof = np.array([plan.profile(s) for s in range(warm, warm + steps)], dtype=np.float64).mean(axis=0)
    # Bytes per bin.  ALGORITHMIC: the path reads every complex64 bin once = 8 B/bin, and that is what the
    # dominant kernel and the whole path are held against (any intermediate is the design's own cost).  OWN TRAFFIC: what a
    # kernel really moves — kernel (a) 8 read + 1 written as sums of 4-bin groups (4 when the plan keeps the per-bin power
    # array), the boxcar stage 1 (4) read.  Which of the two the plan keeps is read from the plan itself.
    keeps_p = "intermediate in HBM: float32 power" in plan.describe()
    own = {"norm_power_kernel": 12 if keeps_p else 9, "boxcar_sweep_kernel": 4 if keeps_p else 1}
    ms = {"norm_power_kernel": prof[1], "boxcar_sweep_kernel": prof[2], "block_exact_kernel": prof[3]}
    dom = max(("norm_power_kernel", "boxcar_sweep_kernel"), key=lambda k: ms[k])
    peak, peak_src = measured_hbm_peak()
    dom_ms = ms[dom]
    gbs = lambda nbytes, t_ms: nbytes / (t_ms * 1e-3) / 1e9
    achieved = gbs(8 * bins, dom_ms)
    traffic_per_bin = recorded_traffic(dom, args.config)
    # The boxcar stage (sweep + refine, prof[2]) on its OWN traffic: the ncu-measured DRAM bytes per bin of the two kernels where
    # the committed capture has them and the plan streams the group sums as in that capture, else the bytes it must read.
    # §8's "fraction of HBM" for kernel (b) is this quantity; the stage is bound by instruction issue, so it also gets an issue
    # roofline: warp-instructions per bin from the same capture (smsp__inst_executed.sum) against 4 schedulers x 1 instruction
    # per clock x SMs at the SM clock sampled during the timed region.
    sweep_ncu = None if keeps_p else recorded_traffic("boxcar_sweep_kernel", args.config)
    if sweep_ncu is not None:
        sweep_ncu += recorded_traffic("sweep_refine_kernel", args.config) or 0.0
    sweep_bytes = sweep_ncu if sweep_ncu is not None else own["boxcar_sweep_kernel"]
    default_sweep = not (keeps_p or args.log_sampling or args.z_step != 1 or args.tile or args.log10_p_flag)   # as captured
    sweep_instr = recorded_traffic("boxcar_stage_warp_instr_per_bin", args.config) if default_sweep else None
    clocks = clk.summary()
    sm_hz = 1e6 * (clocks.get("sm_mhz") or 1965.0)
    issue_peak = 4.0 * torch.cuda.get_device_properties(dev).multi_processor_count * sm_hz
    sweep_issue = None
    if sweep_instr is not None:
        rate = sweep_instr * bins / (prof[2] * 1e-3)
        sweep_issue = {"bound": "alu", "achieved": rate, "peak": issue_peak, "unit": "warp-instr/s", "frac": rate / issue_peak,
                       "warp_instr_per_bin": sweep_instr, "peak_source": "4 warp schedulers x SMs x sampled SM clock",
                       "instr_source": "profiles/traffic.json (ncu smsp__inst_executed.sum of sweep + refine per bin)"}
    roofline = {
        "bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "algorithmic_bytes_per_bin": 8, "algorithmic_bytes_per_launch": 8 * bins,
        "frac_own_traffic": gbs(own[dom] * bins, dom_ms) / peak, "own_bytes_per_bin": own[dom],
        "traffic": (traffic_per_bin * bins) if traffic_per_bin else None, "peak_source": peak_src,
        "traffic_source": "profiles/traffic.json (ncu dram__bytes_read+write per bin x bins of this launch)" if traffic_per_bin else None,
        "kernel_ms": dom_ms,
        "kernel_ms_all": {"memsets": prof[0], "norm_power_kernel": prof[1], "boxcar_sweep_kernel": prof[2],
                          "block_exact_kernel": prof[3]},
        "path_algorithmic_GBps": gbs(8 * bins, ms_step) if world == 1 else None,
        "path_frac": gbs(8 * bins, ms_step) / peak if world == 1 else None,
        "sweep_achieved": gbs(sweep_bytes * bins, prof[2]), "sweep_frac": gbs(sweep_bytes * bins, prof[2]) / peak,
        "sweep_bytes_per_bin": sweep_bytes,
        "sweep_bytes_source": "profiles/traffic.json (ncu, sweep + refine)" if sweep_ncu is not None else "bytes the stage must read",
        "sweep_algorithmic_frac": gbs(4 * bins, prof[2]) / peak, "sweep_algorithmic_bytes_per_bin": 4,
        "sweep_issue": sweep_issue,
    }
    launches = plan.launches_per_search * steps

    # end to end through the C ABI with host buffers (H2D of the spectra + D2H of count and records inside the timed region)
    e2e = None
    if not args.no_e2e:
        plan_h = binding.Plan(wl.n_bins, wl.batch, wl.zmax, wl.block_width, wl.sigma_threshold, norm_block=wl.norm_block,
                              tile=args.tile, log10_p_flag=args.log10_p_flag, host_staging=True, z_step=args.z_step,
                              log_sampling=args.log_sampling)
        plan_h.attach(dev)
        Xh = torch.empty(X.shape, dtype=X.dtype, pin_memory=True)
        Xh.copy_(X)
        hc = np.empty(plan_h.max_candidates, dtype=binding.CANDIDATE_DTYPE)
        rec = plan_h.search_host(Xh, hc)  # warm-up
        torch.cuda.synchronize(); pdist.barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            rec = plan_h.search_host(Xh, hc)
        dt = pdist.max_over_ranks(time.perf_counter() - t0)
        assert len(rec) == n_cand, "host-buffer search disagrees with device-buffer search"
        e2e = {"value": total_bins * args.e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(Xh.numel() * 8),
               "d2h_bytes_per_step": int(4 + 20 * len(rec)), "steps": args.e2e_steps, "ms_per_step": 1e3 * dt / args.e2e_steps}
        plan_h.destroy()
        del plan_h

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(wl, X[: min(wl.batch, 96)].cpu().numpy(), z_step=args.z_step, log_sampling=args.log_sampling)

    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": config_dict(wl, world, args), "bin_widths_per_sec": value * wl.zmax,
            "latency_us_per_search": ms_step * 1e3 if n_copies > 1 else None,
            "candidates_per_step": n_cand, "blocks_flagged_by_sweep": flagged,
            "sweep_cells_refined": int(stats[2]), "sweep_cells_flagged": int(stats[9]), "norm_blocks_redone": int(stats[1]), "clocks": clocks,
            "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
        }
        print(json.dumps(out), flush=True)
    plan.destroy()
    if world > 1:
        tdist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and world == 1 and args.impl == "ours":
        # not under torchrun: launch one process per GPU ourselves
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 2000), str(Path(__file__).resolve())] + sys.argv[1:]
        return subprocess.call(cmd)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
