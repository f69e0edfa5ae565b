#!/usr/bin/env python
"""bench.py -- template x SFT Hough accumulations per second on the BASELINE.json config-2 sky patch.

One STEP = one pass of the whole hot path over one sky patch (BASELINE.json configs[1]: 2000 SFTs, 8x8 pixels,
20 x 30 x 40 binary templates, 90 f0 bins = 1.3824e8 templates, 2.7648e11 accumulations):
    bsh_build_peakgram -> bsh_stage1_hough (unweighted number count + top-1000) -> bsh_stage2_power (re-score + sort)
with the normalised powers already resident in HBM.  `value` = accumulations of all ranks / device time (max over ranks).
`e2e` = the same patch through bsh_search_patch_host() with HOST buffers (H2D of rho and w, D2H of the toplist inside the
timed region).  `roofline` describes the dominant kernel (stage-1 accumulation); `cpu_baseline` is the plain oracle
(oracle/, Eq. 15 with one cos per accumulation) timed on this box's host cores on a bounded sub-grid.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
For N > 1 launch under torchrun (one rank per GPU); ranks process different seeded patches, no data-path collective
(weak scaling, DESIGN.md section "Multi-GPU").
"""
from __future__ import annotations

import argparse
import json
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

# --- roofline model of the stage-1 accumulation kernel -----------------------------------------
# Unit of work: one (pixel, binary template, SFT) TRIPLE = n_f0 (90) accumulations.  The kernel is bound on chip by plain
# instruction throughput: every pipe it uses (integer ALU, FP64, LSU/shared memory) is 40-60 % busy and the warp
# schedulers issue 63 % of their slots (ncu, profiles/r01d_stage1_pix_full.md); HBM is idle.  Roofline = warp-issue peak.
N_SM = 148
LANES_PER_SM_CLK = 128            # 4 SMSPs x 32 lanes: one warp instruction per scheduler per clock
# algorithmic lane-instructions per triple -- what this formulation must execute whatever the schedule:
#   FP64  g = D - B (1), y at both band ends (2), round by magic add (2), equal-shift test (1)                      6
#   count 3 window words x full adder (2 LOP3) + ripple into the 6 high planes once per 32 SFTs (36 / 32)           7.125
#   INT   position select on a break (1), break mask (1), shared-memory address (1)                                 3
#   LSU   window read (LDS.64 + LDS.32) 2, binary terms of 2 templates per load 0.5, Doppler terms of 2 SFTs
#         per load shared by 2 templates 0.25                                                                       2.75
ALGO_OPS_PER_TRIPLE = 6.0 + 7.125 + 3.0 + 2.75
# secondary views: the shared-memory data pipe (one 128-byte wavefront per clock per SM) and the integer-ALU pipe alone
SMEM_BYTES_PER_CLK_SM = 128
SMEM_BYTES_PER_TRIPLE = 12.0 + 4.0 + 4.0      # 96-bit window + D (8 B per 2 templates) + B (one wavefront per 32 triples)
ALU_LANES_PER_SM_CLK = 64                      # 16 lanes/clk/SMSP (B300_MICROARCH.md: alu-pipe rt_SMSP = 2)
ALU_OPS_PER_TRIPLE = 6.0 + 1.125 + 3.0
# weighted kernel: one predicated FP32 add + one predicate-generating op per accumulation, plus the track per triple
OPS_PER_TRIPLE_WEIGHTED_FIXED = 19.0
OPS_PER_ACC_WEIGHTED = 2.0
GATHER_LANES_PER_SM_CLK = 32      # north_star bound (b) read literally: one 4-byte lane-gather per accumulation
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the kernel (ncu --set full, profiles/r01d_stage1_pix_full.md)
NCU_DRAM_BYTES_PER_LAUNCH = 13085184 + 598784


def measured_peaks():
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


# ---------------------------------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the plain oracle on a bounded sample of the same workload
# ---------------------------------------------------------------------------------------------------------------------
def oracle_sample(wl, target_seconds: float):
    """Times oracle.stage1 (DIRECT: Eq. 15 with one libm cos per accumulation, OpenMP over templates) on a sub-grid of the
    workload: all 90 f0 bins and all SFTs, a few pixels x binary templates, sized to ~target_seconds."""
    import oracle
    pk = oracle.peakgram(wl.rho)
    probe = wl.subgrid(ia=[0], ip=[0], it=[0, 1], pix=[0, 1])
    t0 = time.perf_counter()
    oracle.stage1(probe, pk, wl.w, mode=oracle.DIRECT)
    rate = probe.n_accumulations / max(time.perf_counter() - t0, 1e-6)
    n_b = int(max(2, min(wl.n_binary * wl.n_pix, rate * target_seconds / (wl.n_f0 * wl.n_sft))))
    n_it = min(len(wl.tasc_frac), max(1, n_b // 8))
    n_pix = min(wl.n_pix, max(1, n_b // n_it))
    sub = wl.subgrid(ia=[0], ip=[0], it=list(range(n_it)), pix=list(range(n_pix)))
    return sub, pk


def run_oracle_steps(wl, steps: int, warmup: int, seconds_per_step: float):
    import oracle
    sub, pk = oracle_sample(wl, seconds_per_step)
    for _ in range(min(warmup, 1)):
        oracle.stage1(sub, pk, wl.w, mode=oracle.DIRECT)
    t0 = time.perf_counter()
    for _ in range(steps):
        cnt, _ = oracle.stage1(sub, pk, wl.w, mode=oracle.DIRECT)
        top = oracle.toplist(cnt.astype(np.float64), min(wl.topk, cnt.size))
        oracle.stage2(sub, top, wl.rho, wl.w, mode=oracle.DIRECT)
    dt = time.perf_counter() - t0
    sample = (f"oracle DIRECT mode on a sub-grid of config 2: {sub.n_pix} pixels x {sub.n_binary} binary templates x "
              f"{sub.n_f0} f0 x {sub.n_sft} SFTs = {sub.n_accumulations:.3e} accumulations per step")
    return steps * sub.n_accumulations / dt, dt / steps, oracle.max_threads(), sample


def main_reference(args, rank, world):
    if rank != 0:
        return
    wl = synth.config2()
    value, s_per_step, cores, sample = run_oracle_steps(wl, args.steps, args.warmup, seconds_per_step=8.0)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": s_per_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": {"workload": "config2 (BASELINE.json configs[1]), bounded sub-grid", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------------
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

    wl = synth.config2(seed=2 + rank)                      # each rank owns a different seeded patch (weak scaling)
    ctx = bsh.Context(local_rank)
    d_rho = torch.from_numpy(wl.rho).cuda()
    d_w = torch.from_numpy(wl.w).cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    h_rho = torch.from_numpy(wl.rho).pin_memory()
    h_w = torch.from_numpy(wl.w).pin_memory()
    h_out = torch.zeros(wl.topk * bsh.CAND_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    h_out_np = h_out.numpy().view(bsh.CAND_DTYPE)

    def step(mode):
        d_peak = ctx.build_peakgram(d_rho, 1.6)
        d_top, n_top = ctx.stage1_hough(d_peak, wl, mode=mode, topk=wl.topk, d_w=d_w)
        ctx.stage2_power(d_rho, wl, d_top, n_top, d_w=d_w, sort_by_power=True)
        return d_top, n_top

    def timed(fn, steps, warmup):
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
            kern_ms.append(ctx.stats()["stage1_kernel_ms"])
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        if dist:
            dist.barrier()
        total_ms = sum(a.elapsed_time(b) for a, b in ev)
        launches = ctx.stats()["launches"] - l0
        total_ms = sharding.max_over_ranks(total_ms, dist)
        return total_ms, kern_ms, launches, wall

    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    total_ms, kern_ms, launches, wall = timed(lambda: step(bsh.BSH_UNWEIGHTED), args.steps, args.warmup)
    clocks = sampler.result()
    st = ctx.stats()
    acc_per_step = wl.n_accumulations
    value = world * args.steps * acc_per_step / (total_ms * 1e-3)

    # secondary: the weighted number count (FP32 weighted sum) on the same patch
    w_steps = max(1, min(args.steps, 5))
    if args.no_weighted:
        print(json.dumps({"profile_run": True, "unweighted_kernel_ms": float(np.mean(kern_ms))}), flush=True)
        return
    w_total_ms, w_kern_ms, _, _ = timed(lambda: step(bsh.BSH_WEIGHTED), w_steps, 1)
    st_w = ctx.stats()

    if args.profile:
        print(json.dumps({"profile_run": True, "unweighted_kernel_ms": float(np.mean(kern_ms)),
                          "weighted_kernel_ms": float(np.mean(w_kern_ms))}), flush=True)
        return

    # end to end through the host-buffer entry point
    def e2e_step():
        ctx.search_patch_host(h_rho.numpy(), h_w.numpy(), wl, mode=bsh.BSH_UNWEIGHTED, topk=wl.topk, out=h_out_np)
    e_total_ms, _, _, e_wall = timed(e2e_step, args.steps, max(1, min(args.warmup, 2)))
    e2e_value = world * args.steps * acc_per_step / (total_ms_safe(e_total_ms))

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    k_ms = float(np.mean(kern_ms))
    triples = wl.n_pix * wl.n_binary * wl.n_sft
    issue_peak = N_SM * LANES_PER_SM_CLK * sm_max * 1e6 / 1e12                    # Tlaneop/s
    smem_peak = N_SM * SMEM_BYTES_PER_CLK_SM * sm_max * 1e6 / 1e9                 # GB/s
    smem_achieved = triples * SMEM_BYTES_PER_TRIPLE / (k_ms * 1e-3) / 1e9
    alu_peak = N_SM * ALU_LANES_PER_SM_CLK * sm_max * 1e6 / 1e12
    alu_achieved = triples * ALU_OPS_PER_TRIPLE / (k_ms * 1e-3) / 1e12
    algo_achieved = triples * ALGO_OPS_PER_TRIPLE / (k_ms * 1e-3) / 1e12
    gather_peak = N_SM * GATHER_LANES_PER_SM_CLK * sm_max * 1e6
    wk_ms = float(np.mean(w_kern_ms))
    w_ops = triples * OPS_PER_TRIPLE_WEIGHTED_FIXED + wl.n_accumulations * OPS_PER_ACC_WEIGHTED
    cpu_value, _, cores, sample = run_oracle_steps(wl, 1, 0, seconds_per_step=15.0)
    kname = {2: "stage1_unweighted_pix_kernel", 1: "stage1_unweighted_pos_kernel"}.get(st["kernel_variant"] // 1000,
                                                                                       "stage1_unweighted_kernel")

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64 track / u32 bit-sliced count / f32 power", "data": "synthetic",
        "config": {"workload": "config2 (BASELINE.json configs[1]): 1 sky patch, 2000 SFTs, 8x8 pixels, 20x30x40 binary "
                               "templates, 90 f0 bins; unweighted number count -> top-1000 -> stage-2 power",
                   "templates_per_patch": wl.n_templates, "accumulations_per_patch": acc_per_step,
                   "l2": "256 MiB buffer written between timed iterations", "ms_per_sky_patch": total_ms / args.steps,
                   "patches_per_rank": 1},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(wl.rho.nbytes + wl.w.nbytes),
                "d2h_bytes_per_step": int(h_out.numel()), "ms_per_step": e_total_ms / args.steps,
                "call": "bsh_search_patch_host (pinned host buffers)"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "kernel": kname, "achieved": algo_achieved, "peak": issue_peak, "unit": "Tlaneop/s",
                     "frac": algo_achieved / issue_peak, "traffic": NCU_DRAM_BYTES_PER_LAUNCH,
                     "kernel_ms": k_ms, "kernel_share_of_step": k_ms / (total_ms / args.steps),
                     "ops_per_triple": ALGO_OPS_PER_TRIPLE, "triples_per_launch": triples,
                     "peak_source": f"warp-issue peak: 148 SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz (guide unit counts "
                                    "and clock; MEASURED_PEAKS.json holds only HBM and bf16 peaks, and HBM is idle here: "
                                    "13.5 MB of DRAM traffic per launch)",
                     "smem_view": {"bytes_per_triple": SMEM_BYTES_PER_TRIPLE, "achieved_gbs": smem_achieved,
                                   "peak_gbs": smem_peak, "frac": smem_achieved / smem_peak},
                     "alu_pipe_view": {"ops_per_triple": ALU_OPS_PER_TRIPLE, "achieved_tlaneops": alu_achieved,
                                       "peak_tlaneops": alu_peak, "frac": alu_achieved / alu_peak},
                     "gather_bound": {"note": "north_star bound (b) read literally: one 4-byte shared-memory lane-gather "
                                              "per accumulation at 32 lanes/clk/SM; > 1 because the 90 f0 bins of a band "
                                              "share each gathered window",
                                      "achieved_gathers_per_s": acc_per_step / (k_ms * 1e-3), "peak": gather_peak,
                                      "frac": acc_per_step / (k_ms * 1e-3) / gather_peak},
                     "hbm_bound": {"note": "position table + (cos, sin) + D tables are ~3 MB per patch, read once from "
                                           "DRAM then served by L2: ~0.5 us at the measured HBM rate, never the bound",
                                   "hbm_gbs_measured": peaks.get("hbm_gbs")}},
        "weighted": {"value": world * w_steps * acc_per_step / (w_total_ms * 1e-3), "unit": UNIT,
                     "ms_per_step": w_total_ms / w_steps, "kernel_ms": wk_ms, "kernel": "stage1_weighted_kernel",
                     "roofline_frac_issue": w_ops / (wk_ms * 1e-3) / 1e12 / issue_peak, "n_passes": st_w["n_passes"]},
        "stage_ms": {"peakgram": st["peakgram_ms"], "stage1_setup": st["stage1_setup_ms"], "stage1_kernel": k_ms,
                     "stage1_select": st["stage1_select_ms"], "stage2": st["stage2_ms"]},
        "stage1": {"n_candidates": st["n_candidates"], "threshold": st["threshold"], "n_passes": st["n_passes"],
                   "kernel_variant": st["kernel_variant"], "threads_per_block": st["threads_per_block"],
                   "grid_blocks": st["grid_blocks"]},
        "cpu_baseline": {"value": cpu_value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "wall_s_timed_region": wall,
    }
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


def total_ms_safe(ms):
    return max(ms, 1e-9) * 1e-3


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--profile", action="store_true",
                    help="only the timed unweighted + weighted steps (no e2e, no oracle): the command ncu wraps")
    ap.add_argument("--no-weighted", action="store_true", help="with --profile: skip the weighted-count pass")
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
