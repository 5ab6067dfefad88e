#!/usr/bin/env python
"""bench.py — throughput of the w-projection gridding hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--workload config4[:n_dump[:random]]|config1|config2|config3:N:S|config5] [--nvis n] [--prec f32|f64]

One "step" = one pass of the whole hot path over one batch of synthetic
visibilities that is already resident in HBM: grid zero-fill -> binning (a1) -> gridder (a2) ->
dirty image (a3).  a0 (wkernel_build) is setup and untimed.  The metric is grid-point updates/s
(sum of S_p^2 over the gridded visibilities / time).

Default workload: BASELINE config 4 at full size — the largest single-GPU configuration (512 stations,
130 816 baselines x 360 dumps x 8 channels = 376 750 080 visibilities, N = 8192, 128 w-planes, ragged
support 8..32, 2.8e10 updates per step); BASELINE.json's metric names no config, so the rule "largest
single-GPU configuration" applies.  Inputs (5.6 GB) are far larger than the 126 MB L2, so no explicit L2
flush is needed between iterations (stated in `config`).  The other configs stay reachable by flag.

Multi-GPU: the path does not shard (north_star: "no sharding and no collectives"), so --gpus N
under torchrun runs N independent replicas ("replicas only") and reports their sum.

`--impl reference` times the oracle (oracle/, plain fp64 C loops) on the host cores on a bounded
prefix of the same workload; rank 0 only.
"""
import argparse
import ctypes
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "grid-point updates/sec (vis x support^2)"
UNIT = "updates/s"
# FP32 FMA peak used for the "alu" roofline: 148 SMs x 128 FP32 lanes x 2 flop x
# 1.965 GHz (max SM clock, MEASURED_PEAKS.json / B200_PROFILING.md); FP64 is half of that.
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
FLOP_PER_UPDATE = 8          # one complex multiply-add = 4 real FMA


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=48)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--nvis", type=int, default=0, help="override the visibility count (0 = the config's)")
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--option", action="append", default=[], help="library option name=value (tuning)")
    ap.add_argument("--order", default="position", choices=["position", "baseline"],
                    help="position: wpg_grid (sort by window start); baseline: the paper's Eq. (1)-(2) order, "
                         "wpg_grid_baseline_order (track-based workloads, uniform stacks)")
    ap.add_argument("--op", default="grid", choices=["grid", "degrid"],
                    help="grid: the headline step; degrid: wpg_degrid of a random grid for all visibilities (a4+ extra)")
    ap.add_argument("--npol", type=int, default=1, choices=[1, 2, 4],
                    help="2 | 4: wpg_grid_pol with N(0,1) visibilities of that many correlations (not the headline config)")
    ap.add_argument("--no-row-block", action="store_true",
                    help="do not pass the rows-per-time-step hint of track-based workloads to the library")
    return ap.parse_args()


def make_workload(spec, nvis, device, prefix_rows=None):
    """prefix_rows (config 4 only): generate just the first rows of the workload (the CPU legs time a bounded prefix;
    cell, w_max and the values are those of the full workload)."""
    from paper_1905_03213_b200 import synth
    kw = {"nvis": nvis} if nvis else {}
    parts = spec.split(":")
    if parts[0] == "config1":
        return synth.config1(**kw)
    if parts[0] == "config2":
        return synth.config2(device=device, **kw)
    if parts[0] == "config3":
        N = int(parts[1]) if len(parts) > 1 else 2048
        S = int(parts[2]) if len(parts) > 2 else 8
        return synth.config3(N=N, S=S, **kw)
    if parts[0] == "config4":          # config4[:n_dump[:random]]; the config's 50 sources + noise unless ":random" (N(0,1) values)
        n_dump = int(parts[1]) if len(parts) > 1 and parts[1] else 360
        values = "random" if len(parts) > 2 and parts[2] == "random" else "model"
        return synth.config4(n_dump=n_dump, values=values, device=device, prefix_rows=prefix_rows)
    if parts[0] == "config5":
        return synth.config5(device=device, **kw)
    raise SystemExit("unknown workload %r" % spec)


def workload_config(wl, prec, order="position"):
    """Names the workload (the FULL one, also when a CPU leg holds only a prefix of its rows)."""
    nchan = int(wl.freq.size)
    rows = int(wl.notes.get("full_rows", wl.uvw.shape[0]))
    in_bytes = rows * 24 + rows * nchan * 12
    return {"workload": wl.name, "grid_N": wl.grid_N, "nvis": rows * nchan, "nchan": nchan,
            "Nw": wl.Nw, "support": wl.support if np.isscalar(wl.support) else list(wl.support),
            "oversample": wl.oversample, "precision": prec,
            "step": "grid zero-fill + binning (a1) + gridder (a2) + dirty_image (a3); wkernel_build (a0) untimed",
            "row_block": int(wl.notes.get("row_block", 0)), "order": order,
            "l2": "inputs (%.0f MB) larger than the 126 MB L2; no explicit flush" % (in_bytes / 1e6)}


# --------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._halt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:          # NVML missing: report that, do not fake numbers
            self.nv, self.err = None, repr(e)

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._halt.wait(0.005)

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + self.err]}
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# --------------------------------------------------------------------------- oracle legs
def oracle_stack(wl):
    from oracle import wkernel as owk
    sup = wl.support
    if not np.isscalar(sup):
        sup = owk.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, sup[1], sup[2])
    return owk.build_stack(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell)


def oracle_threads(wl):
    """All host cores; a private grid per thread (the paper's CPU method) costs N^2 x 16 B each, so
    the count is capped at a quarter of the available host memory (stated in `cpu_baseline.sample` when it binds)."""
    from oracle import gridder as ogrid
    cores = os.cpu_count() or 1
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 32e9
    cap = max(1, int(0.25 * avail // (wl.grid_N * wl.grid_N * 16)))
    return max(1, min(cores, ogrid.max_threads(), cap, 64))


def time_oracle(wl, st, rows, threads):
    from oracle import gridder as ogrid
    t0 = time.perf_counter()
    _, stats = ogrid.grid(wl.uvw[:rows], wl.vis[:rows], wl.weight[:rows], wl.freq, st, threads=threads)
    return time.perf_counter() - t0, stats["n_updates"]


def rows_for(wl, st, threads, target_s):
    """Rows of the workload's prefix that the oracle passes over in about `target_s` seconds.  Two probes, because a
    call has a fixed cost that a single probe would mistake for work: with OpenMP every thread allocates, zeroes and
    finally adds up its private N x N grid (1 GB each at N = 8192)."""
    nrow = wl.uvw.shape[0]
    p1 = min(nrow, 200_000 if threads > 1 else 20_000)
    p2 = min(nrow, 4 * p1)
    t1, _ = time_oracle(wl, st, p1, threads)
    if p2 == p1:
        return nrow
    t2, _ = time_oracle(wl, st, p2, threads)
    per_row = max((t2 - t1) / (p2 - p1), 1e-12)
    fixed = max(t1 - p1 * per_row, 0.0)
    return int(min(nrow, max(p2, (target_s - fixed) / per_row)))


def sized_oracle_run(wl, st, threads, target_s, max_passes=50):
    """The oracle on a prefix of the workload sized for about `target_s` seconds (a workload it finishes sooner is
    passed over several times).  Returns (updates/s, description)."""
    nrow = wl.uvw.shape[0]
    rows = rows_for(wl, st, threads, target_s)
    t_sum, upd_sum, passes = 0.0, 0, 0
    while passes == 0 or (rows == nrow and t_sum < target_s and passes < max_passes):
        dt, upd = time_oracle(wl, st, rows, threads)
        t_sum += dt; upd_sum += upd; passes += 1
    return upd_sum / t_sum, ("%d pass(es) over the first %d of %d rows (%d updates per pass) of %s, fp64, %s, %.1f s in total"
                             % (passes, rows, nrow, upd_sum // passes, wl.name,
                                "OpenMP private grids (%d threads)" % threads if threads > 1 else "1 thread", t_sum))


def cpu_baseline(wl, target_s=12.0):
    """The oracle as it stands on the host cores: all cores (OpenMP, private grid per thread — the paper's CPU
    method) and one thread (the paper's own comparison, 1 vs 56 threads), each on a bounded prefix of
    the same workload (throughput per update makes a prefix legitimate)."""
    st = oracle_stack(wl)
    threads = oracle_threads(wl)
    v_all, sample_all = sized_oracle_run(wl, st, threads, target_s)
    v_one, sample_one = sized_oracle_run(wl, st, 1, 6.0, max_passes=5)
    return {"value": v_all, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample_all,
            "host_cores": os.cpu_count(),
            "one_thread": {"value": v_one, "unit": UNIT, "cores": 1, "sample": sample_one}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # input generation (not timed) may use the GPU if there is one; the oracle itself runs on the host cores only.
    # Config 4: only a prefix of the 3.77e8 visibilities is generated — the oracle could not pass over more anyway.
    try:
        import torch
        gen_dev = "cuda" if torch.cuda.is_available() else None
    except ImportError:
        gen_dev = None
    prefix = (6_000_000 if gen_dev else 300_000) if args.workload.split(":")[0] == "config4" else None
    wl = make_workload(args.workload, args.nvis, gen_dev, prefix_rows=prefix)
    st = oracle_stack(wl)
    threads = oracle_threads(wl)
    nrow = wl.uvw.shape[0]
    total = max(1, args.steps + args.warmup)
    budget_s = min(20.0, 120.0 / total)                      # whole run within a few minutes
    rows = rows_for(wl, st, threads, budget_s)
    for _ in range(args.warmup):
        time_oracle(wl, st, rows, threads)
    t_sum, upd_sum = 0.0, 0
    for _ in range(args.steps):
        dt, upd = time_oracle(wl, st, rows, threads)
        t_sum += dt; upd_sum += upd
    value = upd_sum / t_sum
    sample = "each step = first %d of %d rows of %s, fp64 oracle, OpenMP private grids (%d threads of %d host cores)" % (
        rows, int(wl.notes.get("full_rows", nrow)), wl.name, threads, os.cpu_count() or 1)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_sum / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, "f64"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# --------------------------------------------------------------------------- multi-rank plumbing
def max_over_ranks(value, dist, device):
    """Max of a per-rank scalar over the process group (None = single process)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(n_updates_per_rank, world, ms_step_max):
    """Whole-job throughput of `world` replicas that each process n_updates per step (weak scaling)."""
    return world * n_updates_per_rank / (ms_step_max * 1e-3)


# --------------------------------------------------------------------------- the CUDA arm
def measured_peaks(ctx, f32):
    """(ALU TFLOP/s, L1 GB/s, HBM GB/s, HBM source): the first two measured in this run through wpg_microbench
    (fma.rn.f32x2 | fma.rn.f64 issue rate; L1-resident 16-byte loads), HBM from the driver's MEASURED_PEAKS.json."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            hbm_gbs = float(json.load(f)["hbm_gbs"]); hbm_src = "measured (MEASURED_PEAKS.json)"
    except (OSError, ValueError, KeyError):
        hbm_gbs, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
    fma_per_s, _ = ctx.microbench(3 if f32 else 4, 20000 if f32 else 10000)          # packed f32x2 FMAs (2 FMA) | f64 FMAs
    alu_tflops = fma_per_s * (4.0 if f32 else 2.0) / 1e12
    l1_loads_per_s, _ = ctx.microbench(2, 4000)                                       # L1-resident 16-byte loads
    return alu_tflops, l1_loads_per_s * 16 / 1e9, hbm_gbs, hbm_src


def l2_feed_gbs(ctx):
    """GB/s of 16-byte loads of whole 512-byte slices from an L2-resident region that does not stay in L1
    (wpg_microbench 9): the coefficient feed when the slices miss L1, bounded by the L2 -> L1 fill path."""
    loads_per_s, _ = ctx.microbench(9, 2000)
    return loads_per_s * 16 / 1e9


def traffic_from_profiles(workload, prec):
    """dram bytes per gridder launch from the committed ncu --set full capture, if there is one."""
    path = os.path.join(ROOT, "profiles", "gridder_traffic.json")
    try:
        with open(path) as f:
            return json.load(f).get("%s/%s" % (workload, prec), {}).get("dram_bytes_per_launch")
    except (OSError, ValueError):
        return None


def run_b200(args):
    import torch
    from paper_1905_03213_b200 import synth, wpgrid

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus > 1 and world != args.gpus:
        raise SystemExit("--gpus %d needs torchrun with %d ranks (WORLD_SIZE=%d)" % (args.gpus, args.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libwpgrid has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    dev = torch.device("cuda", local)
    prec = wpgrid.F32 if args.prec == "f32" else wpgrid.F64
    wl = make_workload(args.workload, args.nvis, dev)
    ctx = wpgrid.Context(local)
    row_block = 0 if args.no_row_block else int(wl.notes.get("row_block", 0))
    ctx.set_option("row_block", row_block)     # rows are time-major, baseline-minor (Measurement Set order)
    for o in args.option:
        k, v = o.split("=")
        ctx.set_option(k, int(v))
    ctx.set_option("timing", 1)
    sup = wl.support
    if not np.isscalar(sup):
        sup, _ = wpgrid.ragged_support(wl.Nw, wl.w_max, wl.grid_N, wl.cell, wl.oversample, sup[1], sup[2])
    stack = ctx.wkernel_build(wl.Nw, wl.w_max, sup, wl.oversample, wl.grid_N, wl.cell, prec)      # a0, untimed

    # inputs resident in HBM before the timed region
    d_vis = torch.from_numpy(wl.vis).to(dev); d_uvw = torch.from_numpy(wl.uvw).to(dev)
    d_wt = torch.from_numpy(wl.weight).to(dev); d_freq = torch.from_numpy(wl.freq).to(dev)
    nrow, nchan = wl.uvw.shape[0], wl.freq.size
    wsum = float(wl.weight.sum())
    grid = ctx.new_grid(stack)
    ws = torch.empty(ctx.grid_workspace_bytes(nrow, nchan, stack), dtype=torch.uint8, device=dev)
    iws = torch.empty(int(ctx.lib.wpg_dirty_image_workspace_bytes(wl.grid_N, prec)), dtype=torch.uint8, device=dev)

    if args.npol > 1:
        return run_pol(args, ctx, wl, stack, d_uvw, d_wt, d_freq, dev, world, rank, dist)
    if args.op == "degrid":
        return run_degrid(args, ctx, wl, stack, d_uvw, d_freq, prec, dev, world, rank, dist)
    if args.order == "baseline":
        n_ant = int(wl.notes["n_ant"])
        a1, a2 = synth.track_antennas(n_ant, nrow)
        d_a1, d_a2 = torch.from_numpy(a1).to(dev), torch.from_numpy(a2).to(dev)
        ws = torch.empty(int(ctx.lib.wpg_baseline_workspace_bytes(nrow, nchan, n_ant, prec)), dtype=torch.uint8, device=dev)

        def grid_call(g, stats=False):
            return ctx.grid_baseline_order(d_vis, d_uvw, d_wt, d_freq, d_a1, d_a2, n_ant, stack, grid=g, workspace=ws, stats=stats)
    else:
        def grid_call(g, stats=False):
            return ctx.grid(d_vis, d_uvw, d_wt, d_freq, stack, grid=g, workspace=ws, stats=stats)

    def step():
        grid.zero_()
        grid_call(grid)
        return ctx.dirty_image(grid, stack, wsum, workspace=iws)

    _, stats = grid_call(ctx.new_grid(stack), stats=True)
    n_updates = stats["n_updates"]
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    ctx.phase_ms()                                     # drop the warm-up phase timings

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = ctx.launch_count()
    barrier()
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = ctx.launch_count() - launches0
    ms_total = e0.elapsed_time(e1)
    bin_ms, grid_ms = ctx.phase_ms()
    ms_total = max_over_ranks(ms_total, dist, dev)
    ms_step = ms_total / args.steps
    value = aggregate_value(n_updates, world, ms_step)

    # ---- e2e: host buffers through wpg_grid_host, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        h = [torch.from_numpy(x).pin_memory() for x in (wl.vis, wl.uvw, wl.weight, wl.freq)]
        N = wl.grid_N
        h_grid = torch.empty((N, N), dtype=torch.complex64 if prec == wpgrid.F32 else torch.complex128).pin_memory()
        h_img = torch.empty((N, N), dtype=torch.float32 if prec == wpgrid.F32 else torch.float64).pin_memory()
        for _ in range(2):
            ctx.grid_host(*h, stack, out=h_grid, image_out=h_img, weight_sum=wsum)
        ksteps = max(3, min(args.steps, 10))
        barrier()
        t0 = time.perf_counter()
        for _ in range(ksteps):
            ctx.grid_host(*h, stack, out=h_grid, image_out=h_img, weight_sum=wsum)   # synchronises
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, dist, dev)
        e2e = {"value": aggregate_value(n_updates, world, 1e3 * dt / ksteps), "unit": UNIT,
               "h2d_bytes_per_step": int(sum(x.numel() * x.element_size() for x in h)),
               "d2h_bytes_per_step": int(h_grid.numel() * h_grid.element_size() + h_img.numel() * h_img.element_size()),
               "ms_per_step": 1e3 * dt / ksteps, "steps": ksteps,
               "call": "wpg_grid_host (pinned host buffers -> host grid + image)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, the gridder.  Per update the method needs 4 real FMA
    # (8 flop) and one coefficient (8 B c64 / 16 B c128) that no other update of the visibility shares, read through
    # L1; per visibility 16 / 24 B of sorted record from HBM.  The binding bound is min(ALU, L1 coefficient feed,
    # HBM) in updates/s; all three peaks are MEASURED in this run (wpg_microbench) or by the driver
    # (MEASURED_PEAKS.json hbm_gbs), never derived.
    f32 = prec == wpgrid.F32
    coef_bytes, rec_bytes = (8, 16) if f32 else (16, 24)
    alu_tflops, l1_gbs, hbm_gbs, hbm_src = measured_peaks(ctx, f32)
    upd_per_s = n_updates / (grid_ms * 1e-3)
    bounds = {"alu": alu_tflops * 1e12 / FLOP_PER_UPDATE,
              "l1": l1_gbs * 1e9 / coef_bytes,
              "hbm": hbm_gbs * 1e9 / rec_bytes * (n_updates / max(stats["n_gridded"], 1))}
    binding = min(bounds, key=bounds.get)
    if binding == "l1":
        ach, peak, unit = upd_per_s * coef_bytes / 1e9, l1_gbs, "GB/s"
        per_unit = "%d B of coefficient per update through L1" % coef_bytes
    elif binding == "alu":
        ach, peak, unit = upd_per_s * FLOP_PER_UPDATE / 1e12, alu_tflops, "TFLOP/s"
        per_unit = "8 flop per update"
    else:
        ach, peak, unit = stats["n_gridded"] * rec_bytes / (grid_ms * 1e-3) / 1e9, hbm_gbs, "GB/s"
        per_unit = "%d B of record per visibility" % rec_bytes
    traffic = traffic_from_profiles(wl.name, args.prec)
    roofline = {"bound": binding, "kernel": "gridder (a2)", "achieved": ach, "peak": peak, "unit": unit,
                "frac": ach / peak, "traffic": traffic,
                "traffic_note": None if traffic is not None else "no ncu --set full capture of this workload/precision under profiles/",
                "peak_source": "measured in this run (wpg_microbench: L1-resident LDG.128, fma.rn.%s)" % ("f32x2" if f32 else "f64")
                               if binding != "hbm" else hbm_src,
                "algorithmic": per_unit, "updates_per_launch": n_updates,
                "gridder_ms": grid_ms, "binning_ms": bin_ms, "gridder_updates_per_s": upd_per_s,
                "bounds_updates_per_s": bounds,
                "alu": {"achieved": upd_per_s * FLOP_PER_UPDATE / 1e12, "peak": alu_tflops, "unit": "TFLOP/s",
                        "frac": upd_per_s * FLOP_PER_UPDATE / 1e12 / alu_tflops, "peak_source": "measured in this run"},
                "l1": {"achieved": upd_per_s * coef_bytes / 1e9, "peak": l1_gbs, "unit": "GB/s",
                       "frac": upd_per_s * coef_bytes / 1e9 / l1_gbs, "peak_source": "measured in this run"}}
    # beside it: the same feed when the slices do NOT stay in L1 (ncu finds 61-98 % of the gridder's
    # coefficient sectors missing L1 — the stack is 1-30 MB — and then the L2 -> L1 fill path, 64 B/clk/SM, is the limit)
    l2_gbs = l2_feed_gbs(ctx)
    roofline["l2_feed"] = {"achieved": upd_per_s * coef_bytes / 1e9, "peak": l2_gbs, "unit": "GB/s",
                           "frac": upd_per_s * coef_bytes / 1e9 / l2_gbs,
                           "peak_source": "measured in this run (wpg_microbench 9: LDG.128 of 512-byte slices, L2-resident, L1-missing)",
                           "note": "achieved counts %d B per update; merged records (compression) and L1 hits load less, "
                                   "so this fraction can exceed 1" % coef_bytes}
    # second entry: the binning pass (a1), HBM-bound.  Algorithmic bytes per visibility: the raw
    # inputs read once (24 / nchan + 12), the sorted record written (16 | 24), 8 B of key / offset traffic.
    bin_bytes_per_vis = 24.0 / nchan + 12 + rec_bytes + 8
    bin_gbs = bin_bytes_per_vis * nrow * nchan / (bin_ms * 1e-3) / 1e9
    roofline["binning"] = {"bound": "hbm", "kernel": "binning (a1): count + scan + scatter", "achieved": bin_gbs,
                           "peak": hbm_gbs, "unit": "GB/s", "frac": bin_gbs / hbm_gbs, "peak_source": hbm_src,
                           "algorithmic": "%.1f B per visibility" % bin_bytes_per_vis, "ms": bin_ms}
    # atomic roofline (BASELINE metric: "% of HBM/atomic roofline"): the measured reduction rate into a buffer of
    # the grid's size is the ceiling of a one-atomic-per-update design; the naive gridder is that design
    red_per_s, _ = ctx.microbench(0, 1000, max(1 << 25, wl.grid_N * wl.grid_N * 8))
    n_naive = min(nrow, max(1, 20_000_000 // nchan))              # a prefix: the naive design is 10-20x slower
    g_naive = ctx.new_grid(stack)
    nv = (d_vis[:n_naive], d_uvw[:n_naive], d_wt[:n_naive], d_freq)
    _, s_naive = ctx.grid_naive(*nv, stack, grid=g_naive, stats=True)
    n0, n1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0.record()
    for _ in range(3):
        ctx.grid_naive(*nv, stack, grid=g_naive)
    n1.record(); torch.cuda.synchronize()
    naive_ms = n0.elapsed_time(n1) / 3
    del g_naive
    roofline["atomic"] = {"red_v2_f32_per_s": red_per_s, "naive_gridder_updates_per_s": s_naive["n_updates"] / (naive_ms * 1e-3),
                          "naive_sample": "first %d rows" % n_naive,
                          "gridder_over_red_ceiling": upd_per_s / red_per_s,
                          "note": "measured after the timed region; fp32 reduction rate also quoted for fp64 runs"}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": args.prec, "data": "synthetic", "config": workload_config(wl, args.prec, args.order),
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
           "stats": stats, "timed_region_ms": ms_total, "multi_gpu": "replicas only" if world > 1 else "single GPU"}
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(wl)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def timed_loop(step, args, dist, dev, local):
    """Warm-up, then K timed steps bracketed by barrier + synchronize, CUDA events, max over ranks, clocks sampled."""
    import torch
    for _ in range(max(args.warmup, 3)):
        step()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); sampler.start(); e0.record()
    for _ in range(args.steps):
        step()
    e1.record(); barrier()
    clocks = sampler.stop()
    return max_over_ranks(e0.elapsed_time(e1), dist, dev) / args.steps, clocks


def run_pol(args, ctx, wl, stack, d_uvw, d_wt, d_freq, dev, world, rank, dist):
    """Polarised gridding, not the headline metric: a step = zero-fill of the npol grids +
    binning + polarised gridder + one dirty image per correlation."""
    import torch
    from paper_1905_03213_b200 import wpgrid
    npol = args.npol
    f32 = stack.prec == wpgrid.F32
    nrow, nchan, N = d_uvw.shape[0], d_freq.shape[0], wl.grid_N
    gen = torch.Generator(device=dev).manual_seed(3)
    vis = torch.view_as_complex(torch.randn((nrow, nchan, npol, 2), dtype=torch.float32, device=dev, generator=gen))
    need = int(ctx.lib.wpg_grid_pol_workspace_bytes(ctx.h, nrow, nchan, npol, ctypes.byref(stack.desc), stack.prec))
    ws = torch.empty(need, dtype=torch.uint8, device=dev)
    grid = torch.zeros((npol, N, N), dtype=torch.complex64 if f32 else torch.complex128, device=dev)
    iws = torch.empty(int(ctx.lib.wpg_dirty_image_workspace_bytes(N, stack.prec)), dtype=torch.uint8, device=dev)
    wsum = float(wl.weight.sum())
    _, stats = ctx.grid_pol(vis, d_uvw, d_wt, d_freq, stack, grid=torch.zeros_like(grid), workspace=ws, stats=True)
    n_updates = stats["n_updates"] * npol

    def step():
        grid.zero_()
        ctx.grid_pol(vis, d_uvw, d_wt, d_freq, stack, grid=grid, workspace=ws)
        for p in range(npol):
            ctx.dirty_image(grid[p], stack, wsum, workspace=iws)

    step(); torch.cuda.synchronize(); ctx.phase_ms()
    launches0 = ctx.launch_count()
    ms, clocks = timed_loop(step, args, dist, dev, dev.index or 0)
    launches = (ctx.launch_count() - launches0) * args.steps // (args.steps + max(args.warmup, 3))
    bin_ms, grid_ms = ctx.phase_ms()
    if rank == 0:
        # one coefficient (8 | 16 B) feeds npol updates: L1 bytes per update shrink by npol, the ALU work does not
        alu_tflops, l1_gbs, hbm_gbs, hbm_src = measured_peaks(ctx, f32)
        ups = n_updates / (grid_ms * 1e-3)
        coef = (8 if f32 else 16) / npol
        bounds = {"alu": alu_tflops * 1e12 / FLOP_PER_UPDATE, "l1": l1_gbs * 1e9 / coef}
        binding = min(bounds, key=bounds.get)
        ach, peak, unit = ((ups * FLOP_PER_UPDATE / 1e12, alu_tflops, "TFLOP/s") if binding == "alu"
                           else (ups * coef / 1e9, l1_gbs, "GB/s"))
        out = {"metric": METRIC + ", %d correlations" % npol, "unit": UNIT, "value": aggregate_value(n_updates, world, ms),
               "ms_per_step": ms, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": args.prec, "data": "synthetic (positions of the workload, N(0,1) visibilities per correlation)",
               "config": dict(workload_config(wl, args.prec), npol=npol), "stats": stats, "clocks": clocks,
               "gpu_launches": int(launches),
               "roofline": {"bound": binding, "kernel": "polarised gridder", "achieved": ach, "peak": peak, "unit": unit,
                            "frac": ach / peak, "traffic": None, "peak_source": "measured in this run (wpg_microbench)",
                            "binning_ms": bin_ms, "gridder_ms": grid_ms, "gridder_updates_per_s": ups,
                            "bounds_updates_per_s": bounds}}
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def run_degrid(args, ctx, wl, stack, d_uvw, d_freq, prec, dev, world, rank, dist):
    """Degridding throughput (not the headline metric): a step = one wpg_degrid of a random grid
    for all visibilities of the workload.  A gather: per update one grid value and one coefficient (16 | 32 B) come
    through L1 — that feed is the bound, half the gridder's."""
    import torch
    from paper_1905_03213_b200 import wpgrid
    f32 = prec == wpgrid.F32
    N = wl.grid_N
    gen = torch.Generator(device=dev).manual_seed(1)
    g = torch.randn((N, N), dtype=torch.complex64 if f32 else torch.complex128, device=dev, generator=gen)
    out, cnt = ctx.degrid(g, d_uvw, d_freq, stack, counts=True)
    sup = stack.support.astype(np.int64)
    # updates = sum S_p^2 over predicted visibilities: exact for uniform stacks
    n_updates = cnt["n_predicted"] * int(sup[0]) ** 2 if stack.uniform else None

    def step():
        ctx.degrid(g, d_uvw, d_freq, stack, out=out)

    launches0 = ctx.launch_count()
    ms, clocks = timed_loop(step, args, dist, dev, dev.index or 0)
    launches = (ctx.launch_count() - launches0) * args.steps // (args.steps + max(args.warmup, 3))
    if rank == 0:
        line = {"metric": "grid-point updates/sec (degridding, vis x support^2)", "unit": UNIT,
                "value": None if n_updates is None else aggregate_value(n_updates, world, ms),
                "ms_per_step": ms, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.prec,
                "data": "synthetic (positions of the workload, N(0,1) grid)", "config": workload_config(wl, args.prec),
                "counts": cnt, "op": "degrid", "clocks": clocks, "gpu_launches": int(launches)}
        if n_updates is not None:
            alu_tflops, l1_gbs, hbm_gbs, hbm_src = measured_peaks(ctx, f32)
            ups = n_updates / (ms * 1e-3)
            per_upd = 16 if f32 else 32
            line["roofline"] = {"bound": "l1", "kernel": "degrid_kernel", "achieved": ups * per_upd / 1e9, "peak": l1_gbs,
                                "unit": "GB/s", "frac": ups * per_upd / 1e9 / l1_gbs, "traffic": None,
                                "algorithmic": "%d B per update through L1 (grid value + coefficient)" % per_upd,
                                "peak_source": "measured in this run (wpg_microbench: L1-resident LDG.128)",
                                "alu_frac": ups * FLOP_PER_UPDATE / 1e12 / alu_tflops}
            if not args.no_cpu_baseline and world == 1:
                from oracle import gridder as ogrid
                st = oracle_stack(wl)
                rows = min(wl.uvw.shape[0], 400_000)
                gh = g.cpu().numpy().astype(np.complex128)
                t0 = time.perf_counter()
                _, c = ogrid.degrid(wl.uvw[:rows], wl.freq, st, gh)
                dt = time.perf_counter() - t0
                line["cpu_baseline"] = {"value": c["n_predicted"] * int(sup[0]) ** 2 / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                        "sample": "oracle_degrid (plain C, fp64, 1 thread) on the first %d rows, %.1f s" % (rows, dt)}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
