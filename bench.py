#!/usr/bin/env python
"""bench.py -- template x SFT Hough accumulations per second of the BinarySkyHough hot path on one B200.

One STEP = one pass of the whole hot path over one sky patch, normalised powers already resident in HBM:
    bsh_build_peakgram -> bsh_stage1_hough (number count of every template + top-1000) -> bsh_stage2_power (re-score, sort)

    --config 3 (default)  BASELINE.json configs[2], the full-size search patch: 8000 SFTs (two detectors x 4000, 30 % gaps),
                          8x8 pixels, 40 x 60 x 120 binary templates, 90 f0 bins = 1.659e9 templates, 1.327e13 accumulations;
                          WEIGHTED FP32 number count (Eq. 22) -- the headline `value`.
    --config 2            configs[1]: 2000 SFTs, 1.3824e8 templates; unweighted count is the headline of that line.
    --config 5            configs[4]: sweep over sky patches of the 256-patch hemisphere tiling on two CUDA streams.

The default line also carries, as named sub-objects, the unweighted count on the same patch, config 2 (both counts), a
config-5 sweep over 32 patches, the fraction-N_C toplist and the front end (NEXT-2) timings.
`e2e` = the same patch through bsh_search_patch_host() with HOST buffers (H2D of rho and w, D2H of the toplist inside the
timed region).  `roofline` describes the dominant kernel (the stage-1 accumulation of the headline mode) against on-chip
peaks MEASURED in the same run (bsh_measure_peaks).  `cpu_baseline` is the plain oracle (oracle/, Eq. 15 with one cos per
accumulation) timed on this box's host cores on a bounded sub-grid, all cores and single-threaded.

    python bench.py [--config 3|2|5] [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
For N > 1 launch under torchrun (one rank per GPU); ranks process different seeded patches, no data-path collective
(weak scaling, DESIGN.md section "Multi-GPU").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "template*SFT Hough accumulations/sec"
UNIT = "accumulations/s"

# --- roofline models of the stage-1 accumulation kernels ----------------------------------------
# Weighted count ("the weighted sum of 1s and 0s"): the method's work is ONE FP32 add per accumulation
# (template x SFT); everything else (track, predicates, staging) is overhead of the formulation.  Bound: the FP32-add
# pipe, peak = measured predicated-FADD lanes/clk/SM x SMs x clock.
# Unweighted count: unit of work = one (pixel, binary template, SFT) TRIPLE = n_f0 (90) accumulations sharing one
# track evaluation and one 96-bit window; bound by plain instruction issue.  Algorithmic lane-instructions per triple:
#   FP64  g = D - B (1), y at both band ends (2), round by magic add (2), equal-shift test (1)                      6
#   count 3 window words x full adder (2 LOP3) + ripple into the 6 high planes once per 32 SFTs (36 / 32)           7.125
#   INT   position select on a break (1), break mask (1), shared-memory address (1)                                 3
#   LSU   window read (LDS.64 + LDS.32) 2, binary terms of 2 templates per load 0.5, Doppler terms of 2 SFTs
#         per load shared by 2 templates 0.25                                                                       2.75
ALGO_OPS_PER_TRIPLE = 6.0 + 7.125 + 3.0 + 2.75
SMEM_BYTES_PER_TRIPLE = 12.0 + 4.0 + 4.0      # 96-bit window + D (8 B per 2 templates) + B (one wavefront per 32 triples)
ALU_OPS_PER_TRIPLE = 6.0 + 1.125 + 3.0         # the integer-ALU pipe's share of the above
GATHER_LANES_PER_SM_CLK = 32                   # north_star bound (b) read literally: one 4-byte lane-gather per accumulation
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures (profiles/)
NCU_DRAM_BYTES = {(3, "weighted"): 117.2e6, (2, "weighted"): 9.26e6, (2, "unweighted"): 13.14e6}
NCU_DRAM_SOURCE = ("profiles/r02_stage1_wpix_full.md, r02_stage1_pix_full.md (config-2 launches, ncu --set full) and "
                   "profiles/r02_dram_config3.md (config-3 weighted launch, dram metrics only)")


def measured_peaks_file():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (nvidia-ml-py)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.02)

    def result(self):
        self.stop_flag = True
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "nvml unavailable"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


def workload_for(config: int, rank: int = 0):
    if config == 2:
        return synth.config2(seed=2 + rank), "config2 (BASELINE.json configs[1])"
    if config == 3:
        return synth.config3(seed=3 + 100 * rank), "config3 (BASELINE.json configs[2])"
    c5 = synth.config5(seed=5 + 100 * rank)
    return c5, "config5 (BASELINE.json configs[4])"


# ---------------------------------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the plain oracle on a bounded sample of the same workload
# ---------------------------------------------------------------------------------------------------------------------
def oracle_subgrid(wl, seconds: float, n_threads: int = 0):
    """A sub-grid of the workload (all f0 bins and all SFTs, a few pixels x binary templates) that the oracle's DIRECT
    mode (Eq. 15 with one libm cos per accumulation) finishes in ~`seconds` on n_threads (0 = all cores)."""
    import oracle
    pk = oracle.peakgram(wl.rho)
    n_it, rate = 2, 0.0
    while True:                                             # probe until the run is long enough to time (>= 0.3 s)
        probe = wl.subgrid(ia=[0], ip=[0], it=list(range(min(n_it, len(wl.tasc_frac)))), pix=list(range(min(8, wl.n_pix))))
        t0 = time.perf_counter()
        oracle.stage1(probe, pk, wl.w, mode=oracle.DIRECT, n_threads=n_threads)
        dt = time.perf_counter() - t0
        rate = probe.n_accumulations / max(dt, 1e-6)
        if dt >= 0.3 or n_it >= len(wl.tasc_frac):
            break
        n_it *= 4
    n_b = int(max(2, min(wl.n_binary * wl.n_pix, rate * seconds / (wl.n_f0 * wl.n_sft))))
    n_it = min(len(wl.tasc_frac), max(1, n_b // 8))
    n_pix = min(wl.n_pix, max(1, n_b // n_it))
    return wl.subgrid(ia=[0], ip=[0], it=list(range(n_it)), pix=list(range(n_pix))), pk


def run_oracle_steps(wl, label, steps: int, warmup: int, seconds_per_step: float, n_threads: int = 0):
    """`steps` passes of the oracle's whole path (stage 1 of every template of the sub-grid, toplist by full sort, stage 2)."""
    import oracle
    sub, pk = oracle_subgrid(wl, seconds_per_step, n_threads)
    for _ in range(min(warmup, 1)):
        oracle.stage1(sub, pk, wl.w, mode=oracle.DIRECT, n_threads=n_threads)
    t0 = time.perf_counter()
    for _ in range(steps):
        cnt, wc = oracle.stage1(sub, pk, wl.w, mode=oracle.DIRECT, n_threads=n_threads)
        top = oracle.toplist(wc, min(wl.topk, cnt.size))
        oracle.stage2(sub, top, wl.rho, wl.w, mode=oracle.DIRECT, n_threads=n_threads)
    dt = time.perf_counter() - t0
    cores = n_threads if n_threads > 0 else oracle.max_threads()
    sample = (f"oracle DIRECT mode on a sub-grid of {label}: {sub.n_pix} pixels x {sub.n_binary} binary templates x "
              f"{sub.n_f0} f0 x {sub.n_sft} SFTs = {sub.n_accumulations:.3e} accumulations per step")
    return steps * sub.n_accumulations / dt, dt / steps, cores, sample


def cpu_baseline(wl, label):
    """All host cores (~12 s) and one thread (~6 s), same oracle, same inputs; extrapolation flagged as such."""
    import oracle
    all_threads = oracle.max_threads()                  # read BEFORE the single-thread leg: that leg's omp_set_num_threads(1)
    value, _, cores, sample = run_oracle_steps(wl, label, 1, 0, seconds_per_step=12.0)   # is process-wide and would otherwise
    v1, _, _, sample1 = run_oracle_steps(wl, label, 1, 0, seconds_per_step=6.0, n_threads=1)   # leave the tier-2 leg on 1 thread
    pk = oracle.peakgram(wl.rho)
    sub2 = wl.subgrid(ia=[0], ip=list(range(min(6, len(wl.P)))))
    t0 = time.perf_counter()
    oracle.tier2_stage1(sub2, pk, n_threads=all_threads)
    dt2 = time.perf_counter() - t0
    assert oracle.max_threads() == all_threads
    tier2 = {"value": sub2.n_accumulations / dt2, "unit": UNIT, "cores": all_threads,
             "kind": "tier-2 CPU reference (oracle/bsh_tier2.c): the same track-sharing math as the GPU path -- one track "
                     "evaluation per (pixel, binary template, SFT), bytes of the band added by a vector loop",
             "sample": f"{sub2.n_pix} pixels x {sub2.n_binary} binary templates x {sub2.n_f0} f0 x {sub2.n_sft} SFTs = "
                       f"{sub2.n_accumulations:.3e} accumulations"}
    return {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "tier2": tier2,
            "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": sample1},
            "extrapolated_full_config_seconds": {"all_cores": wl.n_accumulations / value,
                                                 "single_thread": wl.n_accumulations / v1,
                                                 "note": "EXTRAPOLATED linearly from the sub-grid rate to the full config"}}


def main_reference(args, rank, world):
    if rank != 0:
        return
    wl, label = workload_for(args.config)
    if args.config == 5:
        wl = wl.patch_workload(0)
    value, s_per_step, cores, sample = run_oracle_steps(wl, label, args.steps, args.warmup, seconds_per_step=5.0)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": s_per_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": f"{label}, bounded sub-grid", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------------
class Patch:
    """One sky patch resident on the device + the step of the hot path over it."""

    def __init__(self, torch, bsh, ctx, wl):
        self.torch, self.bsh, self.ctx, self.wl = torch, bsh, ctx, wl
        self.d_rho = torch.from_numpy(wl.rho).cuda()
        self.d_w = torch.from_numpy(wl.w).cuda()

    def step(self, mode, topk=None):
        ctx, wl = self.ctx, self.wl
        d_peak = ctx.build_peakgram(self.d_rho, 1.6)
        d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=mode, topk=topk or wl.topk, d_w=self.d_w)
        ctx.stage2_power(self.d_rho, wl, d_top, n_top, d_w=self.d_w, sort_by_power=True)
        return d_top, n_top


def main_ours(args, rank, local_rank, world):
    import torch
    import paper_1904_04873_b200 as bsh
    from paper_1904_04873_b200 import sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    ctx = bsh.Context(local_rank)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def timed(fn, steps, warmup, stat_key="stage1_kernel_ms"):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        kern_ms = []
        l0 = ctx.stats()["launches"]
        t0 = time.perf_counter()
        for a, b in ev:
            flush.fill_(1)                                  # L2 flush between timed iterations (not timed)
            a.record()
            fn()
            b.record()
            b.synchronize()
            kern_ms.append(ctx.stats()[stat_key])
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        if dist:
            dist.barrier()
        total_ms = sum(a.elapsed_time(b) for a, b in ev)
        launches = ctx.stats()["launches"] - l0
        total_ms = sharding.max_over_ranks(total_ms, dist)
        return total_ms, float(np.mean(kern_ms)), launches, wall

    peaks = ctx.measure_peaks() if rank == 0 else None

    if args.config == 5:
        return main_config5(args, rank, world, torch, bsh, ctx, dist, peaks)

    wl, label = workload_for(args.config, rank)              # each rank owns a different seeded patch (weak scaling)
    patch = Patch(torch, bsh, ctx, wl)
    head_mode = bsh.BSH_WEIGHTED if args.config == 3 else bsh.BSH_UNWEIGHTED
    other_mode = bsh.BSH_UNWEIGHTED if args.config == 3 else bsh.BSH_WEIGHTED
    names = {bsh.BSH_WEIGHTED: "weighted", bsh.BSH_UNWEIGHTED: "unweighted"}

    if args.profile:                                         # the command ncu wraps: only the chosen accumulation mode
        mode = bsh.BSH_WEIGHTED if args.profile == "weighted" else bsh.BSH_UNWEIGHTED
        _, k_ms, _, _ = timed(lambda: patch.step(mode), args.steps, args.warmup)
        print(json.dumps({"profile_run": True, "config": args.config, "mode": args.profile, "kernel_ms": k_ms}), flush=True)
        return

    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    total_ms, k_ms, launches, wall = timed(lambda: patch.step(head_mode), args.steps, args.warmup)
    clocks = sampler.result()
    st = ctx.stats()
    acc_per_step = wl.n_accumulations
    value = world * args.steps * acc_per_step / (total_ms * 1e-3)

    # the other number count on the same patch
    o_steps = max(1, min(args.steps, 5))
    o_total_ms, ok_ms, _, _ = timed(lambda: patch.step(other_mode), o_steps, 1)
    st_o = ctx.stats()

    # end to end through the host-buffer entry point
    h_rho = torch.from_numpy(wl.rho).pin_memory()
    h_w = torch.from_numpy(wl.w).pin_memory()
    h_out = torch.zeros(wl.topk * bsh.CAND_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    h_out_np = h_out.numpy().view(bsh.CAND_DTYPE)

    def e2e_step():
        ctx.search_patch_host(h_rho.numpy(), h_w.numpy(), wl, mode=head_mode, topk=wl.topk, out=h_out_np)
    e_steps = max(1, min(args.steps, 10))
    e_total_ms, _, _, _ = timed(e2e_step, e_steps, max(1, min(args.warmup, 2)))
    e2e_value = world * e_steps * acc_per_step / (max(e_total_ms, 1e-9) * 1e-3)

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    extras = {}
    if args.config == 3 and not args.lean:
        extras["config2"] = sub_config2(torch, bsh, ctx, timed, peaks)
        extras["config5_sweep"] = sweep_config5(torch, bsh, n_patches=32)
        extras["nc_fraction"] = sub_nc_fraction(torch, bsh, ctx)
        extras["frontend"] = sub_frontend(torch, bsh, ctx, wl, flush)
        extras["eccentric"] = sub_eccentric(torch, bsh, ctx, timed)
        extras["postprocessing"] = sub_post(torch, bsh, ctx)

    kinds = {names[head_mode]: (k_ms, total_ms / args.steps, st), names[other_mode]: (ok_ms, o_total_ms / o_steps, st_o)}
    roof = {m: roofline(m, wl, kinds[m][0], kinds[m][2], peaks) for m in kinds}
    head = names[head_mode]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ("f64 track / f32 weighted count / f32 power" if head == "weighted"
                  else "f64 track / u32 bit-sliced count / f32 power"),
        "data": "synthetic",
        "config": {"workload": f"{label}: 1 sky patch, {wl.n_sft} SFTs, {wl.n_pix} pixels, {len(wl.ap)}x{len(wl.P)}x"
                               f"{len(wl.tasc_frac)} binary templates, {wl.n_f0} f0 bins; {head} number count -> top-"
                               f"{wl.topk} -> stage-2 power",
                   "templates_per_patch": wl.n_templates, "accumulations_per_patch": acc_per_step,
                   "l2": "256 MiB buffer written between timed iterations", "ms_per_sky_patch": total_ms / args.steps,
                   "patches_per_rank": 1},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(wl.rho.nbytes + wl.w.nbytes),
                "d2h_bytes_per_step": int(h_out.numel()), "ms_per_step": e_total_ms / e_steps, "steps": e_steps,
                "call": "bsh_search_patch_host (pinned host buffers)"},
        "gpu_launches": int(launches),
        "roofline": roof[head],
        names[other_mode]: {"value": world * o_steps * acc_per_step / (o_total_ms * 1e-3), "unit": UNIT,
                            "ms_per_step": o_total_ms / o_steps, "steps": o_steps, "roofline": roof[names[other_mode]],
                            "n_passes": st_o["n_passes"]},
        "stage_ms": {"peakgram": st["peakgram_ms"], "stage1_setup": st["stage1_setup_ms"], "stage1_kernel": k_ms,
                     "stage1_select": st["stage1_select_ms"], "stage2": st["stage2_ms"]},
        "stage1": {"n_candidates": st["n_candidates"], "threshold": st["threshold"], "n_passes": st["n_passes"],
                   "kernel_variant": st["kernel_variant"], "threads_per_block": st["threads_per_block"],
                   "grid_blocks": st["grid_blocks"]},
        "measured_peaks": peaks,
        "cpu_baseline": cpu_baseline(wl, label),
        "wall_s_timed_region": wall,
    }
    line.update(extras)
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


def kernel_name(variant: int, weighted: bool) -> str:
    fam = variant // 1000
    if weighted:
        return {3: "stage1_weighted_pix_kernel", 1: "stage1_weighted_pos_kernel"}.get(fam, "stage1_weighted_kernel")
    return {2: "stage1_unweighted_pix_kernel", 1: "stage1_unweighted_pos_kernel"}.get(fam, "stage1_unweighted_kernel")


def roofline(mode: str, wl, k_ms: float, st: dict, pk: dict) -> dict:
    """Roofline object of the stage-1 accumulation kernel of `mode` against the peaks measured in this run."""
    n_sm, mhz = pk["n_sm"], pk["sm_clock_mhz"]
    per_s = n_sm * mhz * 1e6                                          # SM-clocks per second, whole chip
    triples = wl.n_pix * wl.n_binary * wl.n_sft
    acc = wl.n_accumulations
    secs = k_ms * 1e-3
    common = {"kernel": kernel_name(st["kernel_variant"], mode == "weighted"), "kernel_ms": k_ms,
              "traffic": NCU_DRAM_BYTES.get((2 if wl.n_sft < 4000 else 3, mode)), "traffic_source": NCU_DRAM_SOURCE,
              "gather_bound": {"note": "north_star bound (b) read literally: one 4-byte shared-memory lane-gather per "
                                       "accumulation at 32 lanes/clk/SM; the 90 f0 bins of a band share each gathered window",
                               "frac": acc / secs / (GATHER_LANES_PER_SM_CLK * per_s)},
              "hbm_bound": {"note": "tables of a patch are a few MB, read once from DRAM then served by L2: never the bound",
                            "hbm_gbs_measured": measured_peaks_file().get("hbm_gbs")}}
    if mode == "weighted":
        peak = pk["fadd_lanes_per_clk_sm"] * per_s / 1e12
        achieved = acc / secs / 1e12
        return {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFADD/s (one FP32 add per accumulation)",
                "frac": achieved / peak, "ops_per_accumulation": 1.0, "accumulations_per_launch_set": acc,
                "peak_source": f"measured in this run (bsh_measure_peaks): predicated FADD {pk['fadd_lanes_per_clk_sm']:.1f} "
                               f"lanes/clk/SM x {n_sm} SMs x {mhz:.0f} MHz", **common}
    issue_lanes = 128.0 * pk["issue_warp_inst_per_clk_smsp"]
    peak = issue_lanes * per_s / 1e12
    achieved = triples * ALGO_OPS_PER_TRIPLE / secs / 1e12
    lds_peak = pk["lds64_bytes_per_clk_sm"] * per_s / 1e9
    lds_ach = triples * SMEM_BYTES_PER_TRIPLE / secs / 1e9
    alu_peak = pk["lop3_lanes_per_clk_sm"] * per_s / 1e12
    alu_ach = triples * ALU_OPS_PER_TRIPLE / secs / 1e12
    fp64_peak = min(pk["dadd_lanes_per_clk_sm"], pk["dmul_lanes_per_clk_sm"]) * per_s / 1e12
    return {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tlaneop/s", "frac": achieved / peak,
            "ops_per_triple": ALGO_OPS_PER_TRIPLE, "triples_per_launch": triples,
            "peak_source": f"measured in this run (bsh_measure_peaks): warp-issue rate {pk['issue_warp_inst_per_clk_smsp']:.3f} "
                           f"warp-instructions/clk/scheduler x 4 x 32 lanes x {n_sm} SMs x {mhz:.0f} MHz",
            "smem_view": {"bytes_per_triple": SMEM_BYTES_PER_TRIPLE, "achieved_gbs": lds_ach, "peak_gbs": lds_peak,
                          "frac": lds_ach / lds_peak, "peak_source": "measured conflict-free LDS.64"},
            "alu_pipe_view": {"ops_per_triple": ALU_OPS_PER_TRIPLE, "achieved_tlaneops": alu_ach, "peak_tlaneops": alu_peak,
                              "frac": alu_ach / alu_peak, "peak_source": "measured LOP3"},
            "fp64_pipe_view": {"ops_per_triple": 6.0, "achieved_tlaneops": triples * 6.0 / secs / 1e12,
                               "peak_tlaneops": fp64_peak, "frac": triples * 6.0 / secs / 1e12 / fp64_peak,
                               "peak_source": "measured DADD / DMUL (no FMA)"},
            **common}


def sub_config2(torch, bsh, ctx, timed, peaks):
    wl = synth.config2()
    patch = Patch(torch, bsh, ctx, wl)
    out = {"workload": "config2 (BASELINE.json configs[1]): 2000 SFTs, 1.3824e8 templates", "accumulations_per_patch": wl.n_accumulations}
    for mode, name, steps in ((bsh.BSH_UNWEIGHTED, "unweighted", 10), (bsh.BSH_WEIGHTED, "weighted", 5)):
        total_ms, k_ms, _, _ = timed(lambda: patch.step(mode), steps, 3)
        st = ctx.stats()
        out[name] = {"value": steps * wl.n_accumulations / (total_ms * 1e-3), "unit": UNIT, "ms_per_step": total_ms / steps,
                     "steps": steps, "roofline": roofline(name, wl, k_ms, st, peaks)}
    return out


def sweep_config5(torch, bsh, n_patches=32, c5=None):
    """Config 5: patches of the hemisphere tiling streamed over two CUDA streams (two contexts), one shared peakgram;
    the launch/collect split lets patch n + 1 accumulate while patch n is selected and re-scored.  Device-timed: events
    on both streams, max of the two."""
    c5 = c5 or synth.config5()
    stride = max(1, c5.n_patches // n_patches)
    ids = [i * stride for i in range(n_patches)]              # spread over the whole hemisphere (all declinations)
    wls = [c5.patch_workload(i) for i in ids]
    d_rho = torch.from_numpy(c5.base.rho).cuda()
    out = {"workload": f"config5 (BASELINE.json configs[4]): {n_patches} of the 256 patches (every {stride}th), 8000 SFTs, "
                       "1.3824e8 templates per patch, unweighted count -> top-1000 -> stage 2 per patch",
           "patches": n_patches}
    for n_streams in (1, 2):
        streams = [torch.cuda.Stream() for _ in range(n_streams)]
        ctxs = [bsh.Context(0, stream=s) for s in streams]
        with torch.cuda.stream(streams[0]):
            d_peak = ctxs[0].build_peakgram(d_rho)
        torch.cuda.synchronize()
        keep = [torch.from_numpy(w.w).cuda() for w in wls]
        for rep in range(2):                                  # first pass warms tables and allocations
            torch.cuda.synchronize()
            start = [torch.cuda.Event(enable_timing=True) for _ in streams]
            stop = [torch.cuda.Event(enable_timing=True) for _ in streams]
            for s, e in zip(streams, start):
                e.record(s)
            t0 = time.perf_counter()
            pending = [None] * n_streams
            for n, ip in enumerate(list(range(n_patches)) + [None] * n_streams):
                s = n % n_streams
                if pending[s] is not None:
                    jp = pending[s]
                    with torch.cuda.stream(streams[s]):
                        d_top, n_top = ctxs[s].stage1_collect()
                        ctxs[s].stage2_power(d_rho, wls[jp], d_top, n_top, d_w=keep[jp], sort_by_power=True)
                    pending[s] = None
                if ip is not None:
                    with torch.cuda.stream(streams[s]):
                        ctxs[s].stage1_launch(d_peak, wls[ip], mode=bsh.BSH_UNWEIGHTED, topk=1000, d_w=keep[ip])
                    pending[s] = ip
            for s, e in zip(streams, stop):
                e.record(s)
            torch.cuda.synchronize()
            wall = time.perf_counter() - t0
            dev_ms = max(a.elapsed_time(b) for a in start for b in stop)
        acc = sum(w.n_accumulations for w in wls)
        out[f"streams_{n_streams}"] = {"ms_per_patch": dev_ms / n_patches, "value": acc / (dev_ms * 1e-3), "unit": UNIT,
                                      "wall_ms_per_patch": wall / n_patches * 1e3}
        for c in ctxs:
            c.close()
    return out


def sub_nc_fraction(torch, bsh, ctx):
    """toplist = fraction N_C = 5 % of config 2's templates, stage 2 on the
    half-overlapped SFT set (2 N rows)."""
    wl = synth.config2()
    wl2 = synth.overlapped_stage2_set(wl, seed=12)
    k = int(0.05 * wl.n_templates)
    d_rho, d_w = torch.from_numpy(wl.rho).cuda(), torch.from_numpy(wl.w).cuda()
    d_rho2, d_w2 = torch.from_numpy(wl2.rho).cuda(), torch.from_numpy(wl2.w).cuda()
    res = {}
    for rep in range(2):
        torch.cuda.synchronize()
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        d_peak = ctx.build_peakgram(d_rho, 1.6)
        d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=bsh.BSH_UNWEIGHTED, topk=k, d_w=d_w)
        e[1].record()
        ctx.stage2_power(d_rho2, wl2, d_top, n_top, d_w=d_w2, sort_by_power=True)
        e[2].record()
        torch.cuda.synchronize()
        st = ctx.stats()
        res = {"workload": "config 2, N_C = 5 % of 1.3824e8 templates -> stage 2 on 4000 half-overlapped SFTs",
               "candidates": n_top, "stage1_ms": e[0].elapsed_time(e[1]), "selection_ms": st["stage1_select_ms"],
               "stage2_ms": e[1].elapsed_time(e[2]), "total_ms": e[0].elapsed_time(e[2]),
               "stage2_gathers_per_s": n_top * wl2.n_sft / (e[1].elapsed_time(e[2]) * 1e-3),
               "n_passes": st["n_passes"]}
        del d_top
    return res


def sub_frontend(torch, bsh, ctx, wl, flush):
    """SURVEY NEXT-2 (Eq. 20-21): complex SFT bins -> 101-bin running-median normalised power ->
    peakgram, one fused kernel, at the size of the headline patch.  HBM-bound by its algorithmic bytes (8 B per raw bin in,
    4 B per power + 1 bit per peak out); reported against the measured HBM copy bandwidth."""
    window = 101
    raw = synth.raw_sft_bins(31, wl.n_sft, wl.n_bins + window - 1)
    d_raw = torch.from_numpy(raw).cuda()
    ms = []
    for _ in range(6):
        flush.fill_(1)
        ctx.normalise_peakgram(d_raw, window=window)
        ms.append(ctx.stats()["frontend_ms"])
    t = float(np.median(ms[1:]))
    n, n_raw, k = wl.n_sft, raw.shape[1], wl.n_bins
    algo_bytes = 8 * n * n_raw + 4 * n * k + 4 * n * ((k + 31) // 32)
    hbm = measured_peaks_file().get("hbm_gbs")
    return {"workload": f"{n} SFTs x {n_raw} raw complex bins -> {k} slab columns, running median over {window} bins",
            "kernel": "normalise_peakgram_kernel", "kernel_ms": t, "algorithmic_bytes": algo_bytes,
            "roofline": {"bound": "hbm", "achieved": algo_bytes / (t * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                         "frac": (algo_bytes / (t * 1e-3) / 1e9 / hbm) if hbm else None,
                         "note": "the per-row sort and median scan are on-chip work above the HBM floor; the kernel runs once "
                                 "per band, in front of ~50 sky patches (L451)"}}


def sub_eccentric(torch, bsh, ctx, timed):
    """SURVEY NEXT-3 (Eq. 14): config 2 with every template on an eccentric orbit (one pair e cos w, e sin w != 0,
    so the template count is unchanged): the accumulation kernel's time against the circular search."""
    import dataclasses
    wl = synth.widened(synth.config2(), 2)                   # 2 more margin bins: a_p Omega e f T < 1.2 bins at e = 0.03
    wle = dataclasses.replace(wl, ecosw=np.array([0.03 * math.cos(0.7)]), esinw=np.array([0.03 * math.sin(0.7)]))
    out = {"workload": "config 2 on a slab with 2 more margin bins per side, every template with (e cos w, e sin w) = "
                       "0.03 (cos 0.7, sin 0.7); same template count as the circular search"}
    for name, w in (("circular", wl), ("eccentric", wle)):
        patch = Patch(torch, bsh, ctx, w)
        for mode, mname in ((bsh.BSH_UNWEIGHTED, "unweighted"), (bsh.BSH_WEIGHTED, "weighted")):
            _, k_ms, _, _ = timed(lambda: patch.step(mode), 5, 2)
            out[f"{name}_{mname}_kernel_ms"] = k_ms
    return out


def sub_post(torch, bsh, ctx):
    """SURVEY NEXT-4 (section V.E, Eq. 44): 5000 candidates (L496) -> clusters + centroids; two lists -> coincidences."""
    a, b = synth.candidate_list(41, n_background=4900, chain=40), synth.candidate_list(42, n_background=4900)
    da = tuple(torch.from_numpy(x).cuda() for x in (a.param, a.res, a.sig))
    db = tuple(torch.from_numpy(x).cuda() for x in (b.param, b.res, b.sig))
    out = {"workload": f"{a.n} candidates: clustering window sqrt(14) bins; {a.n} x {b.n} coincidences, window 3 bins (L511)"}
    for rep in range(2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        c = ctx.post_cluster(da, math.sqrt(14.0))
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        pa, _, _, _ = ctx.post_coincidences(da, db, 3.0)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        out.update({"cluster_ms": (t1 - t0) * 1e3, "n_clusters": int(c["root"].numel()), "coincidences_ms": (t2 - t1) * 1e3,
                    "n_pairs": int(pa.numel()), "pair_distances_per_s": (a.n * a.n) / max(t1 - t0, 1e-9)})
    return out


def main_config5(args, rank, world, torch, bsh, ctx, dist, peaks):
    c5, label = workload_for(5, rank)
    n_patches = max(2, args.steps)
    sampler = ClockSampler(physical_gpu_index(int(os.environ.get("LOCAL_RANK", "0"))))
    sampler.start()
    sw = sweep_config5(torch, bsh, n_patches=n_patches, c5=c5)
    clocks = sampler.result()
    if dist:
        dist.barrier()
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return
    two = sw["streams_2"]
    wl0 = c5.patch_workload(0)
    line = {"metric": METRIC, "value": world * two["value"], "unit": UNIT, "n_gpus": world, "steps": n_patches,
            "warmup": n_patches, "ms_per_step": two["ms_per_patch"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 track / u32 bit-sliced count / f32 power", "data": "synthetic",
            "config": {"workload": sw["workload"], "ms_per_sky_patch": two["ms_per_patch"],
                       "l2": "per-patch tables exceed nothing; patches differ, 8 MB power slab re-read per patch",
                       "templates_per_patch": wl0.n_templates, "accumulations_per_patch": wl0.n_accumulations},
            "clocks": clocks, "sweep": sw, "measured_peaks": peaks, "gpu_launches": None,
            "note": "a step is one sky patch; the first sweep over the patches is the warm-up"}
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[2, 3, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lean", action="store_true", help="skip the config-2 / config-5 / N_C sub-objects of the default line")
    ap.add_argument("--profile", default=None, choices=["weighted", "unweighted"],
                    help="only the timed steps of one accumulation mode (no e2e, no oracle): the command ncu wraps")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        main_reference(args, rank, world)
    else:
        main_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
