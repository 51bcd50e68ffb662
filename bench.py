#!/usr/bin/env python
"""bench.py - throughput of the fringe-search hot path on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config ID] [--impl reference]

One "step" = one volks_fringe_search over the whole synthetic workload (all baselines, IFs, widths
and windows of the config; candidates compacted).  Prints ONE JSON line on rank 0.
  value      windows/s with the visibility slab already resident in HBM (device-timed, CUDA events)
  e2e        the same metric through the public API with HOST buffers: pinned host -> device copy of
             the slab and device -> host read of the candidate list inside the timed region
  roofline   dominant kernel: EXECUTED flops per launch / live CUDA-event duration vs the FP32 FMA peak
             measured in the same run (volks_measure_fp32_peak; bound "alu"; DESIGN.md section 6 states the
             per-unit flops); the SURVEY 8(d) algorithmic count is printed beside it, labelled
  other_configs  configs[3] and configs[4] timed the same way (default run only), so that north_star's
             "configs[2-4]" are all driver-visible
  cpu_baseline  the float64 oracle, as it stands, on the host cores, on a bounded sample
With --impl reference the oracle itself is the timed program (rank 0 only).
"""
import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

import workloads

SM_COUNT, FP32_LANES_PER_SM = 148, 128      # B200 (guide: 148 SMs, 4 SMSP x 32 FP32 lanes)
METRIC = "fringe-search windows/s (and visibilities/s) at 1 B200; % of FP32 roofline"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2,
                    help="BASELINE.json configs[ID] (default 2); 5 = the paper's EL060-shaped 4 s segment (use with --allif)")
    ap.add_argument("--impl", default="volks", choices=["volks", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="default run only: skip the extra timing of configs[3] and configs[4]")
    ap.add_argument("--peaks", action="store_true", help="also write the dense per-window peak array")
    ap.add_argument("--allif", action="store_true",
                    help="time f2 instead: VOLKS2's all-IF one-delay search (Eq. 1) on the config's slab, band padded x2")
    ap.add_argument("--dm", type=float, default=0.0,
                    help="dedisperse (f1, fused into the slab load) with this DM [pc cm^-3]; 0 = plain search")
    return ap.parse_args()


class ClockSampler(threading.Thread):
    """Samples SM clock / throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.1):
        super().__init__(daemon=True)
        self.index, self.period, self.stop_flag = index, period, False
        self.sm, self.reasons, self.max_mhz, self.power = [], set(), None, []

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                nv.nvmlClocksEventReasonSwPowerCap if hasattr(nv, "nvmlClocksEventReasonSwPowerCap") else 0x4: "sw_power_cap",
                0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                0x80: "hw_power_brake_slowdown",
            }
            while not self.stop_flag:
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = 0
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(self.period)
        except Exception as e:  # NVML missing: report that, never fail the bench
            self.reasons.add("nvml_unavailable:%s" % type(e).__name__)

    def summary(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm),
                "power_w_max": max(self.power) if self.power else None}


def algorithmic_flops(c):
    """SURVEY.md 8(d) per-unit figures: delay FFT once per AP (5 Nf log2 Nf) + per window
    Nf*(5 Nt log2 Nt) column FFTs + ~5 Nt Nf for |.|^2/max/sum.  Returns (total, per-width list)."""
    npair, nap, nf = c["nbl"] * c["nif"], c["nap"], c["nf"]
    row = npair * nap * 5.0 * nf * math.log2(nf) if nf > 1 else 0.0
    per_w = []
    for w, s, nt in zip(c["widths"], c["strides"], c["nts"]):
        nw = workloads.gen.nwin(nap, w, s) * npair
        per_w.append(nw * (nf * 5.0 * nt * math.log2(nt) + 5.0 * nt * nf))
    return row + sum(per_w), row, per_w


def nominal_flops(c):
    """north_star's accounting: 5 N log2 N per padded plane, N = Nt*Nf."""
    npair, nap, nf = c["nbl"] * c["nif"], c["nap"], c["nf"]
    tot = 0.0
    for w, s, nt in zip(c["widths"], c["strides"], c["nts"]):
        n = nt * nf
        tot += workloads.gen.nwin(nap, w, s) * npair * 5.0 * n * math.log2(n)
    return tot


def oracle_sample(c, budget_s=20.0):
    """Bounded sample of config `c` for the oracle: ONE (bl, ifq) pair, the first `nap_s` APs, all
    widths (cached-rows mode).  nap_s is sized from a small calibration run so that the sample costs
    about `budget_s` of CPU work.  Returns (vis_sample numpy, nap_s)."""
    from oracle import volks_oracle
    wmax = max(c["widths"])
    nap_cal = min(c["nap"], max(2 * wmax, 96))
    vis, cc, _ = workloads.generate(c["id"], nbl=1, nif=1, nap=nap_cal, npulses=0)
    t = time.perf_counter()
    volks_oracle.search(vis.numpy(), c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    dt = max(time.perf_counter() - t, 1e-4)
    nwin_cal = sum(workloads.gen.nwin(nap_cal, w, s) for w, s in zip(c["widths"], c["strides"]))
    rate = max(nwin_cal, 1) / dt
    per_ap = sum(1.0 / s for s in c["strides"])
    nap_s = int(min(c["nap"], max(nap_cal, budget_s * rate / per_ap)))
    return nap_s


def time_oracle(c, nap_s):
    """Run the oracle (as it stands) on one pair x nap_s APs; returns (windows, seconds, cores)."""
    from oracle import volks_oracle
    vis, cc, _ = workloads.generate(c["id"], nbl=1, nif=1, nap=nap_s, npulses=min(c["npulses"], 2))
    v = vis.numpy()
    t = time.perf_counter()
    pk, used = volks_oracle.search(v, c["widths"], c["strides"], c["nts"], c["nf"], mode="cached")
    dt = time.perf_counter() - t
    return len(pk), dt, used


def workload_name(c):
    return ("configs[%d]: %d bl x %d IF x %d ch x %d AP cf32, widths %s stride %s, plane Nt %s x Nf %d"
            % (c["id"], c["nbl"], c["nif"], c["nchan"], c["nap"], c["widths"], c["strides"], c["nts"], c["nf"]))


def run_reference(args):
    """--impl reference: the oracle is the timed program; each step one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import volks_oracle
    volks_oracle.build()
    c = workloads.config(args.config)
    total = max(args.steps + args.warmup, 1)
    nap_s = oracle_sample(c, budget_s=min(20.0, 150.0 / total))
    for _ in range(args.warmup):
        time_oracle(c, nap_s)
    nwin, secs, used = 0, 0.0, 1
    for _ in range(args.steps):
        n, dt, used = time_oracle(c, nap_s)
        nwin += n
        secs += dt
    val = nwin / secs if secs > 0 else 0.0
    sample = "1 (bl,IF) pair x first %d APs of %s, all widths, cached-rows mode, per step" % (nap_s, workload_name(c))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "windows/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(c), "sample": sample},
        "cpu_baseline": {"value": val, "unit": "windows/s", "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "windows/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "visibilities_per_s": nap_s * c["nchan"] * args.steps / secs if secs > 0 else 0.0,
        "gpu_launches": 0,
    }))


def ncu_traffic_table():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the rate kernels, parsed from the committed
    ncu summary profiles/dram_traffic.csv (columns: config,kernel,width,dram_bytes_per_launch,source; the
    commands that made it are in profiles/dram_traffic.md).  Missing file or row -> traffic null."""
    tab = {}
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if os.path.exists(path):
        for line in open(path).read().splitlines()[1:]:
            f = line.split(",")
            if len(f) >= 4:
                tab[(int(f[0]), f[1], int(f[2]))] = (float(f[3]), f[4] if len(f) > 4 else "")
    return tab


def max_over_ranks(dist, ms, device):
    """Replicas only: the one cross-rank step is the MAX of the device-timed
    milliseconds; `dist` is torch.distributed or None (single process)."""
    if dist is None:
        return float(ms)
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, units_per_rank, ms_step):
    """Whole-job throughput of `world` independent replicas, each doing `units_per_rank` per step."""
    return world * units_per_rank / (ms_step * 1e-3)


KIND_NAMES = {1: "row_fft", 2: "col", 3: "finalize", 4: "scan", 5: "scatter", 6: "slide", 7: "colfft", 8: "allif", 9: "fixup",
              10: "winthr", 11: "bound", 12: "recover", 13: "coleval", 14: "sfold", 15: "sfold_eval"}


# Executed flops per unit, pinned by ncu (profiles/r02_counters.md: sm__sass_thread_inst_executed_op_fp32_pred_on counts a
# packed FFMA2 / FMUL2 / FADD2 once per thread; the FFMA2 : (FMUL2 + FADD2) mix comes from the kernel's SASS):
#   k_slide, w >= 16: 4.96e11 flops per w = 64 launch of config 2 / 6.29e10 bin-steps = 7.9 flops per bin per window (a complex
#     multiply-add is 8 flops only for the non-trivial half of the twiddles; the others are two adds; + 3 for |.|^2)
#   k_colfft2, Nt = 512: 5553 / 6359 / 7089 packed instructions per (window, delay column) for w <= 64 / 128 / 256 (pass 1
#     pruned to the non-zero inputs) at 2.47 / 2.45 / 2.42 flops each: 13700 / 15600 / 17200 against the SURVEY count 25600
SLIDE_FLOPS_PER_BIN = 7.9
# ... and the same counters as FP32 lane-OPERATIONS (an add, a multiply and an FMA each count once per lane; a packed
# instruction is two lanes): k_slide 1.625e11 thread-instructions x 2 / 6.288e10 bin-steps = 5.17 per bin per window;
# k_colfft2 2 x (5553 / 6359 / 7089) per (window, column).  Against the peak OPERATION rate (measured FMA peak / 2 flops per
# FMA) this is the share of the FP32 pipe's issue slots the kernel fills - what ncu reports as FMA-pipe cycles active.
SLIDE_OPS_PER_BIN = 5.17
COLFFT2_OPS_PER_COLUMN = {4: 11106.0, 8: 12718.0, 16: 14178.0}
# k_colfft2 SKIP (the default candidates-only mode: pass 2 only where a candidate is possible; profiles/r02_counters.md,
# configs[4]'s data): 2071 / 2884 / 3617 packed instructions per (window, column): pass 1 + the 32 FFMA2 of the bound
# (w <= 64 / 128 now run k_colfft2e, which adds the energies of the pass-1 sums: 2328 / 3140 packed instructions per (window,
# column), 257 / 256 of them the FMUL2 + FFMA2 of |S|^2 at 3 flops on average)
COLFFT2_SKIP_FLOPS_PER_COLUMN = {4: 6670.0, 8: 8620.0, 16: 9560.0}
COLFFT2_SKIP_OPS_PER_COLUMN = {4: 4656.0, 8: 6280.0, 16: 7234.0}
COLFFT2_FLOPS_PER_COLUMN = {4: 13700.0, 8: 15600.0, 16: 17200.0}
# k_slide<FOLD> (kind 14, the folded sliding sum of the candidates-only mode; profiles/r02_counters.md, configs[2] w = 64):
# 5.111e10 FP32 thread-instructions per launch, 8.87e9 of them scalar (the FFMAs of the octagonal bound); the rest is half
# packed arithmetic (per step 4 FFMA2 : 2 FMUL2 : 4 FADD2 = 2.8 flops each) and half FMNMX / FSETP (comparisons: no flops)
# = 7.69e10 flops per launch / 6.288e10 bin-steps = 1.22 flops per bin per window (the 16 bins of a (residue, column) share
# ONE complex update); lane-operations 2 x 2.11e10 + 8.87e9 = 5.11e10 -> 0.81 per bin per window
SFOLD_FLOPS_PER_BIN = 1.22
SFOLD_OPS_PER_BIN = 0.81
# warp instructions per bin per window (smsp__inst_executed.sum / bin-steps): against the issue rate of 148 SMs x 4
# schedulers x the SM clock this is the share of issue slots filled
WARP_INST_PER_BIN = {6: 8.715e9 / 6.288e10, 14: 2.828e9 / 6.288e10}
SM_COUNT_ISSUE = 148 * 4


def executed_flops_per_launch(c, kind, wid, nlaunch, npair, nap, alg_flops, cand_only=False):
    """Flops the kernel really executes per launch, counter-pinned where a capture exists; a
    kernel without one is charged the SURVEY 8(d) algorithmic count (an upper bound: pruned inputs execute fewer)."""
    if wid < 0:
        return alg_flops
    w_, s_, nt_ = c["widths"][wid], c["strides"][wid], c["nts"][wid]
    nwin = workloads.gen.nwin(nap, w_, s_) * npair
    if kind == 6:
        return nwin * nt_ * c["nf"] * SLIDE_FLOPS_PER_BIN / nlaunch
    if kind == 14:
        return nwin * nt_ * c["nf"] * SFOLD_FLOPS_PER_BIN / nlaunch
    nz = 1
    while nz * 16 < w_:
        nz *= 2
    if kind == 7 and nt_ == 512 and nz in COLFFT2_FLOPS_PER_COLUMN:
        return nwin * c["nf"] * (COLFFT2_SKIP_FLOPS_PER_COLUMN if cand_only else COLFFT2_FLOPS_PER_COLUMN)[nz] / nlaunch
    return alg_flops


def executed_ops_per_launch(c, kind, wid, nlaunch, npair, nap, cand_only=False):
    """FP32 lane-operations per launch (see SLIDE_OPS_PER_BIN), or None for kernels without a counter capture."""
    if wid < 0:
        return None
    w_, s_, nt_ = c["widths"][wid], c["strides"][wid], c["nts"][wid]
    nwin = workloads.gen.nwin(nap, w_, s_) * npair
    if kind == 6:
        return nwin * nt_ * c["nf"] * SLIDE_OPS_PER_BIN / nlaunch
    if kind == 14:
        return nwin * nt_ * c["nf"] * SFOLD_OPS_PER_BIN / nlaunch
    nz = 1
    while nz * 16 < w_:
        nz *= 2
    if kind == 7 and nt_ == 512 and nz in COLFFT2_OPS_PER_COLUMN:
        return nwin * c["nf"] * (COLFFT2_SKIP_OPS_PER_COLUMN if cand_only else COLFFT2_OPS_PER_COLUMN)[nz] / nlaunch
    return None


def executed_warp_inst_per_launch(c, kind, wid, nlaunch, npair, nap):
    """Warp instructions per launch of the sliding kernels (ncu-pinned), or None."""
    if wid < 0 or kind not in WARP_INST_PER_BIN or c["nts"][wid] < 32:
        return None
    nwin = workloads.gen.nwin(nap, c["widths"][wid], c["strides"][wid]) * npair
    return nwin * c["nts"][wid] * c["nf"] * WARP_INST_PER_BIN[kind] / nlaunch


def measure_fp32_peak(vk, local, stream):
    """The FP32 FMA peak measured in this run (volks_measure_fp32_peak: dependent-free FFMA chains, CUDA
    events, best of 5 launches of ~20 ms), with the SM clock sampled while it runs."""
    smp = ClockSampler(local, period=0.02)
    smp.start()
    best, mean, ms = vk.measure_fp32_peak(5, stream)
    smp.stop_flag = True
    smp.join()
    ck = smp.summary()
    derived = SM_COUNT * FP32_LANES_PER_SM * 2 * (ck["sm_max_mhz"] or 1965) * 1e6 / 1e12
    return {"tflops": best, "tflops_mean": mean, "launch_ms": ms, "sm_mhz": ck["sm_mhz"], "reasons": ck["reasons"],
            "derived_tflops": derived,
            "kind": "measured: volks_measure_fp32_peak (FFMA chains, 64 warps/SM, best of 5 launches; SM clock median "
                    "%s MHz during the probe); derived 148 SM x 128 lanes x 2 x sm_max_mhz = %.2f" % (ck["sm_mhz"], derived)}


def measure(vk, args, cfg_id, dev, local, rank, dist, steps, warmup, peak, traffic, also_full_index=False):
    """Device-timed throughput + per-launch roofline of one config.  Returns a dict (tensors included, for
    the e2e leg of the main config)."""
    vis, c, _ = workloads.generate(cfg_id, device=dev, seed=workloads.config(cfg_id)["seed"] + 17 * rank)
    nbl, nif, nap, nchan = vis.shape
    if args.allif:
        # band padded x2, or x4 = the paper's padding factor for the EL060-shaped config 5
        nfa = workloads.gen.next_pow2((4 if cfg_id == 5 else 2) * nif * nchan)
        plan = vk.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], None, nfa, c["snr_thresh"], allif=True)
    else:
        plan = vk.Plan(nbl, nif, nap, nchan, c["widths"], c["strides"], c["nts"], c["nf"], c["snr_thresh"])
    stream = torch.cuda.current_stream(dev)
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device=dev)
    ncand = torch.zeros(1, dtype=torch.int32, device=dev)
    peaks = torch.empty(plan.nwin_total * vk.PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev) if args.peaks else None
    shift = None
    if args.dm:
        # IFs of 16 MHz above 1400 MHz (L band, like EL060: PAPER.md:172-173), referenced to the top frequency
        f = 1400.0 + 16.0 * np.arange(nif)[:, None] + (16.0 / nchan) * np.arange(nchan)[None, :]
        shift = torch.as_tensor(vk.dm_shifts(args.dm, f, f.max(), c["t_ap"]), device=dev)

    # candidate capacity from the plan's own count: one sizing run (the count is the true total even when the
    # list overflows), then a buffer that holds the whole list
    cap = 1 << 16
    cands = torch.empty(cap * vk.CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    plan.fringe_search(vis, ws, cands, ncand, peaks, stream, shift=shift)
    torch.cuda.synchronize(dev)
    n0 = int(ncand.item()) & 0xFFFFFFFF
    if n0 > cap:
        cap = (n0 + (1 << 16)) & ~((1 << 16) - 1)
        cands = torch.empty(cap * vk.CAND_DTYPE.itemsize, dtype=torch.uint8, device=dev)

    def step():
        plan.fringe_search(vis, ws, cands, ncand, peaks, stream, shift=shift)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(max(warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    sampler.stop_flag = True
    sampler.join()
    ms_total = max_over_ranks(dist, ms_total, dev)
    ms_step = ms_total / steps
    nwin = plan.nwin_total
    nvis = nbl * nif * nap * nchan
    world = int(os.environ.get("WORLD_SIZE", "1"))
    value = aggregate_value(world, nwin, ms_step)
    n_found = int(ncand.item()) & 0xFFFFFFFF

    # ---- the other index mode: every window's peak written (dense peak array), nothing pruned ----
    full_ms = None
    if also_full_index and peaks is None and not args.allif:
        pk_all = torch.empty(plan.nwin_total * vk.PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev)
        for _ in range(2):
            plan.fringe_search(vis, ws, cands, ncand, pk_all, stream, shift=shift)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        f0.record(stream)
        for _ in range(3):
            plan.fringe_search(vis, ws, cands, ncand, pk_all, stream, shift=shift)
        f1.record(stream)
        torch.cuda.synchronize(dev)
        full_ms = max_over_ranks(dist, f0.elapsed_time(f1), dev) / 3
        del pk_all

    # ---- roofline leg: per-launch CUDA-event durations on the launching stream ----
    plan.profile(True)
    per = {}
    reps = 2
    for _ in range(reps):
        step()
        torch.cuda.synchronize(dev)
        for kind, wid, ms in plan.profile_read():
            per.setdefault((kind, wid), []).append(ms)
    plan.profile(False)
    tot_alg, row_alg, per_w_alg = algorithmic_flops(c)
    nlaunch = {k: len(v) / reps for k, v in per.items()}
    share = {k: sum(v) / reps for k, v in per.items()}
    step_sum = sum(share.values())
    dom = max(share, key=share.get)
    dom_ms_avg = float(np.mean(per[dom]))
    kname = "%s[w=%s]" % (KIND_NAMES.get(dom[0], str(dom[0])), c["widths"][dom[1]] if dom[1] >= 0 else "all")
    kernel_ms = {"%s[%d]" % (KIND_NAMES.get(k[0], str(k[0])), k[1]): round(v, 4) for k, v in sorted(share.items())}
    clocks = sampler.summary()
    base = dict(vk=vk, plan=plan, vis=vis, c=c, ws=ws, cands=cands, ncand=ncand, peaks=peaks, stream=stream, dev=dev,
                rank=rank, world=world, dist=dist, ms_step=ms_step, value=value, nwin=nwin, nvis=nvis, n_found=n_found,
                clocks=clocks, cap=cap, shift=shift, full_ms=full_ms)
    if args.allif:
        # f2 is bandwidth work: the row pass reads the slab once and writes the all-IF delay spectra, every
        # width's k_allif reads them once.  Roofline of the dominant kernel against measured HBM bandwidth.
        peaks_json = os.path.join(ROOT, "MEASURED_PEAKS.json")
        hbm = json.load(open(peaks_json))["hbm_gbs"] if os.path.exists(peaks_json) else 6650.0
        ybytes = nbl * nap * plan.nf * 8.0                        # the band's delay spectra (row padding is never touched)
        dom_bytes = (ybytes + nvis * 8.0 if dom[0] == 1 else ybytes) / nlaunch[dom]
        gbs = dom_bytes / (dom_ms_avg * 1e-3) / 1e9
        base["roofline"] = {
            "bound": "hbm", "kernel": kname, "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
            "traffic": None, "launch_ms": dom_ms_avg, "share_of_step": share[dom] / step_sum,
            "peak_kind": "measured (MEASURED_PEAKS.json hbm_gbs)" if os.path.exists(peaks_json) else "fallback 6650 GB/s",
            "bytes_kind": "algorithmic: the chunk's all-IF delay spectra read once (row pass: + the slab read once)",
            "kernel_ms": kernel_ms}
        return base
    if dom[0] in (1, 11):
        # the row pass (slab read once, delay spectra written once) and the pruning pass (delay spectra read once)
        # are bandwidth work: roofline against the measured HBM copy bandwidth
        peaks_json = os.path.join(ROOT, "MEASURED_PEAKS.json")
        hbm = json.load(open(peaks_json))["hbm_gbs"] if os.path.exists(peaks_json) else 6650.0
        ybytes = nbl * nif * nap * c["nf"] * 8.0                          # the Nf columns of a row (its padding is never touched)
        dom_bytes = (ybytes + nvis * 8.0 + nbl * nif * nap * 4.0 if dom[0] == 1 else ybytes) / nlaunch[dom]
        gbs = dom_bytes / (dom_ms_avg * 1e-3) / 1e9
        tr = traffic.get((c["id"], KIND_NAMES.get(dom[0], ""), -1))
        base["roofline"] = {
            "bound": "hbm", "kernel": kname, "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
            "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None,
            "launch_ms": dom_ms_avg, "share_of_step": share[dom] / step_sum,
            "peak_kind": "measured (MEASURED_PEAKS.json hbm_gbs)" if os.path.exists(peaks_json) else "fallback 6650 GB/s",
            "bytes_kind": "algorithmic: the chunk's delay spectra %s" % ("written once + the slab read once + per-AP energies"
                                                                          if dom[0] == 1 else "read once"),
            "hbm_gbs_algorithmic": nvis * 8 / (ms_step * 1e-3) / 1e9, "kernel_ms": kernel_ms}
        return base
    if dom[1] >= 0:
        dom_alg = per_w_alg[dom[1]] / nlaunch[dom]
    else:
        dom_alg = 0.0
    cand_only = peaks is None              # default options: no dense peak array = the candidates-only index mode
    exec_flops = executed_flops_per_launch(c, dom[0], dom[1], nlaunch[dom], nbl * nif, nap, dom_alg, cand_only)
    peak_tf = peak["tflops"]
    exec_tf = exec_flops / (dom_ms_avg * 1e-3) / 1e12
    alg_tf = dom_alg / (dom_ms_avg * 1e-3) / 1e12
    tr = traffic.get((c["id"], KIND_NAMES.get(dom[0], ""), c["widths"][dom[1]] if dom[1] >= 0 else -1))
    ops = executed_ops_per_launch(c, dom[0], dom[1], nlaunch[dom], nbl * nif, nap, cand_only)
    winst = executed_warp_inst_per_launch(c, dom[0], dom[1], nlaunch[dom], nbl * nif, nap)
    roofline = {
        "bound": "alu", "kernel": kname, "achieved": exec_tf, "peak": peak_tf, "unit": "TFLOP/s",
        "frac": exec_tf / peak_tf, "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None,
        "launch_ms": dom_ms_avg, "share_of_step": share[dom] / step_sum,
        "flops_kind": "executed, pinned by ncu's instruction counters (profiles/r02_counters.md): k_slide 7.9 flops per bin "
                      "per window (its folded form, sfold, 1.22: one complex update serves the 16 bins of a (residue, column)), k_colfft2 (Nt 512) 13700 / 15600 / 17200 flops per (window, column) for w <= 64 / 128 / 256; "
                      "other kernels the SURVEY 8(d) count",
        "fma_pipe_note": "packed FP32 adds and multiplies occupy the FMA pipe like FMAs but count half the flops, so the "
                         "flop fraction understates the pipe: ncu reads the FMA pipe 68 % busy for k_slide w = 64 and k_colfft2 w = 64 (profiles/r02_counters.md)",
        "peak_kind": peak["kind"], "peak_derived_tflops": peak["derived_tflops"],
        "fp32_op_frac": None if ops is None else ops / (dom_ms_avg * 1e-3) / (peak_tf * 1e12 / 2.0),
        "fp32_op_kind": "executed FP32 lane-operations (add, multiply and FMA each one; ncu-pinned) / time / peak operation rate "
                        "(measured FMA peak / 2): the share of FP32 issue slots filled; `frac` counts flops, which halves every add",
        "issue_frac": None if winst is None or not clocks.get("sm_mhz") else
                      winst / (dom_ms_avg * 1e-3) / (SM_COUNT_ISSUE * clocks["sm_mhz"] * 1e6),
        "issue_kind": "executed warp instructions (ncu-pinned per bin per window) / time / (148 SMs x 4 schedulers x the median "
                      "SM clock of this run): the kernel mixes FMA-pipe, ALU-pipe (min / max / compare) and shared-memory "
                      "instructions, so the issue rate bounds it before any one pipe does",
        "algorithmic_tflops": alg_tf, "algorithmic_frac": alg_tf / peak_tf,
        "algorithmic_kind": "SURVEY 8(d) FFT-equivalent flops / time: exceeds 1 by construction for the sliding path "
                            "(an algorithmic speed-up, not a fraction of the machine)",
        "whole_step_algorithmic_tflops": tot_alg / (ms_step * 1e-3) / 1e12,
        "whole_step_nominal_tflops": nominal_flops(c) / (ms_step * 1e-3) / 1e12,
        "hbm_gbs_algorithmic": nvis * 8 / (ms_step * 1e-3) / 1e9,
        "kernel_ms": kernel_ms,
    }
    if roofline["frac"] > 1.0:
        roofline["error"] = "executed flops above the measured peak: the per-bin accounting is wrong"
    base["roofline"] = roofline
    return base


def run_e2e(R, steps):
    """Same metric through the public API with HOST buffers: every step copies the slab from pinned
    host memory to the device, runs the search and reads the WHOLE candidate list back."""
    vk, plan, dev, stream = R["vk"], R["plan"], R["dev"], R["stream"]
    h_vis = torch.empty(R["vis"].shape, dtype=torch.complex64, pin_memory=True)
    h_vis.copy_(R["vis"])
    h_n = torch.zeros(1, dtype=torch.int32, pin_memory=True)
    h_c = torch.empty(R["cap"] * vk.CAND_DTYPE.itemsize, dtype=torch.uint8, pin_memory=True)
    d2h, overflow = 0, False

    stage = torch.empty(2 * plan.stage_bytes, dtype=torch.uint8, device=dev)

    def step():
        nonlocal d2h, overflow
        # the public host-slab call: chunked pinned-host -> device copies overlapped with the kernels
        plan.search_host(h_vis, stage, R["ws"], R["cands"], R["ncand"], R["peaks"], stream, shift=R["shift"])
        h_n.copy_(R["ncand"], non_blocking=True)
        stream.synchronize()
        nf_ = int(h_n.item()) & 0xFFFFFFFF
        overflow = overflow or nf_ > R["cap"]
        n = min(nf_, R["cap"]) * vk.CAND_DTYPE.itemsize
        if n:
            h_c[:n].copy_(R["cands"][:n], non_blocking=True)
            stream.synchronize()
        d2h = 4 + n

    step()
    if R["dist"] is not None:
        R["dist"].barrier()
    torch.cuda.synchronize(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(R["dist"], ms, dev) / steps
    return {"value": R["world"] * R["nwin"] / (ms * 1e-3), "unit": "windows/s", "ms_per_step": ms,
            "h2d_bytes_per_step": int(h_vis.numel() * 8), "d2h_bytes_per_step": int(d2h),
            "candidates_read_back": int((d2h - 4) // vk.CAND_DTYPE.itemsize), "overflow": bool(overflow)}


def brief(R):
    """The part of a measurement that goes under other_configs."""
    rf = R["roofline"]
    return {"workload": workload_name(R["c"]), "ms_per_step": R["ms_step"], "windows_per_s": R["value"],
            "visibilities_per_s": R["world"] * R["nvis"] / (R["ms_step"] * 1e-3), "windows": R["nwin"],
            "candidates": R["n_found"], "clocks": R["clocks"],
            "roofline": {k: rf[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "launch_ms",
                                            "share_of_step", "fp32_op_frac", "issue_frac", "algorithmic_frac", "bytes_kind", "kernel_ms") if k in rf}}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import paper_2108_05602_b200 as vk
    vk.lib()                                   # fails loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    traffic = ncu_traffic_table()
    # N independent replicas (the path needs no exchange; north_star fixes one
    # GPU, so --gpus N runs N replicas, each the full config with its own seed)
    peak = measure_fp32_peak(vk, local, torch.cuda.current_stream(dev))
    R = measure(vk, args, args.config, dev, local, rank, dist, args.steps, args.warmup, peak, traffic, also_full_index=True)
    c = R["c"]
    e2e = None if args.no_e2e else run_e2e(R, max(1, min(args.steps, 3)))
    launches = R["plan"].launches * args.steps
    plan_nf = R["plan"].nf
    others = {}
    if args.config == 2 and not args.allif and not args.dm and not args.no_other_configs:
        main_line = {k: R[k] for k in ("value", "ms_step", "nwin", "nvis", "n_found", "clocks", "roofline", "world", "rank", "full_ms")}
        R["plan"].close()
        R = None
        torch.cuda.empty_cache()
        for other in (3, 4):
            Ro = measure(vk, args, other, dev, local, rank, dist, max(1, min(args.steps, 3)), 3, peak, traffic)
            others[str(other)] = brief(Ro)
            Ro["plan"].close()
            Ro = None
            torch.cuda.empty_cache()
        R = main_line
    cpu = None
    if R["rank"] == 0 and R["world"] == 1 and not args.no_cpu_baseline:
        from oracle import volks_oracle
        volks_oracle.build()
        nap_s = oracle_sample(c, budget_s=15.0)
        n, dt, used = time_oracle(c, nap_s)
        cpu = {"value": n / dt, "unit": "windows/s", "cores": used, "kind": "oracle",
               "sample": "1 (bl,IF) pair x first %d APs, all widths, float64 cached-rows mode: %d windows in %.1f s"
                         % (nap_s, n, dt)}
    if R["rank"] == 0:
        out = {
            "metric": METRIC, "value": R["value"], "unit": "windows/s", "n_gpus": R["world"],
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": R["ms_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": workload_name(c), "snr_thresh": c["snr_thresh"],
                       "l2": "input slab (%.2f GB) larger than L2, no flush needed" % (R["nvis"] * 8 / 1e9)
                       if R["nvis"] * 8 > 126e6 else "input smaller than L2 (latency-bound config, report only)",
                       "replicas": R["world"], "dense_peaks": bool(args.peaks), "dm": args.dm,
                       "index_mode": "full (dense peak array: every window's peak bin)" if args.peaks else
                                     "candidates-only (default volks_options): candidates complete and bit-identical to the full "
                                     "mode; peak bins found for possible candidates only, segments of narrow windows whose "
                                     "amplitude-sum bound excludes a candidate are not transformed",
                       "search": "f2 all-IF one-delay search (Eq. 1), nfa %d" % plan_nf if args.allif else "2-D per-IF fringe search"},
            "visibilities_per_s": R["world"] * R["nvis"] / (R["ms_step"] * 1e-3),
            "windows": R["nwin"], "candidates": R["n_found"],
            "clocks": R["clocks"], "e2e": e2e, "gpu_launches": launches,
            "full_index": None if R.get("full_ms") is None else
                          {"ms_per_step": R["full_ms"], "windows_per_s": R["world"] * R["nwin"] / (R["full_ms"] * 1e-3),
                           "what": "the same search with the dense per-window peak array (every window transformed and indexed)"},
            "roofline": R["roofline"], "cpu_baseline": cpu, "fp32_peak_probe": {k: peak[k] for k in ("tflops", "tflops_mean", "launch_ms", "sm_mhz", "reasons", "derived_tflops")},
        }
        if others:
            out["other_configs"] = others
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
