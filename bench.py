#!/usr/bin/env python
"""bench.py — fp64 grid-point-steps/s of the MHD step (BASELINE.json metric) on B200, one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--size 512] [--impl ours|reference]

A "step" is one explicit time step (one pass of the whole hot path: sweeps S1-S5) of the 512^3 ABC-dynamo
config of BASELINE.json (config 5; `--size 256` gives config 4).  Inputs are seeded and synthetic.
  value        N^3 * K * n_gpus / (max over ranks of the device time of mhd_step(K)), state resident in HBM
  e2e          same metric through the C ABI with HOST (pinned) buffers: set_fields + step(K) + get_fields
  roofline     the dominant kernel family, SURVEY.md 8(d) style: algorithmic bytes per launch / CUDA-event time per launch
               against the measured HBM copy peak (MEASURED_PEAKS.json); `alu` = the same kernel on FLOPS (8(d) count)
               against twice the DFMA rate measured in this run; every family and the whole step beside it
  size_256     the other size the metric is quoted on (config 4, 256^3), measured in the same run
  cpu_baseline the CPU oracle, as it stands, on a bounded sample (128^3 grid of the same config), all cores and one thread
Multi-GPU: the path does not shard without an all-to-all: `--gpus N` runs N independent
replicas (weak scaling), one process per GPU under torchrun, timed as the max over ranks.
`--impl reference` times the oracle (the reference arm of this tier) on the host cores of rank 0.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 grid-point-steps/s"
UNIT = "grid-point-steps/s"
TRAFFIC_FILE = os.path.join("profiles", "traffic_r02.json")   # ncu DRAM bytes per launch of the committed capture
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


# ----------------------------------------------------------------------------------------------------------------
# clocks during the timed region (profiling recipe)
# ----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
        return self

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            p = [x.strip() for x in line.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for nm, val in zip(names, p[3:7]):
                if val.lower() == "active":
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------------------
# distributed plumbing (one process per GPU; replicas only)
# ----------------------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def aggregate(ms_local: float, units_local: float, dist=None):
    """max-over-ranks time and summed work: (ms_max, units_total).  `dist` = torch.distributed or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms_local, units_local
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    u = torch.tensor([units_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ----------------------------------------------------------------------------------------------------------------
# algorithmic bytes per launch; one field-sweep = 8 B per grid point
# ----------------------------------------------------------------------------------------------------------------
def fused_flops_per_line(N: int) -> float:
    """SURVEY.md 8(d) flop count of the fused x sweep per (y,z) line: 27 real line transforms at 2.5 N log2 N each
    plus ~90 flop per grid point of point-wise products."""
    return 27 * 2.5 * N * math.log2(N) + 90.0 * N


def sweep_bytes(N: int, prune: bool, fuse_current: bool = True, fuse_s5: bool = False):
    """Per-family algorithmic bytes of ONE right-hand side: what the kernels must read + write."""
    kc = N // 3
    H = N // 2
    a = (2 * kc + 1) / N if prune else 1.0          # kept fraction of a full axis
    ah = (kc + 1) / H if prune else 1.0             # kept fraction of the stored half axis
    f = 8.0 * N ** 3                                # bytes of one full field sweep
    b = {}
    if fuse_current:     # S1 reads the 8 state fields and builds J^ on load; writes 11
        b["strided_inverse"] = f * ah * (8 * a * a + 11 * a) + 11 * f * ah * (a + 1.0)   # z pass, y pass (read + write)
    else:
        b["build_current"] = (3 + 3) * f * ah * a * a
        b["strided_inverse"] = 11 * f * ah * (a * a + a) + 11 * f * ah * (a + 1.0)
    b["x_fused"] = (11 + 16) * f * ah
    if fuse_s5:          # sweep S5 in one launch: reads 16 z-full products + U^ + R^old, writes U^ + R^old
        b["strided_forward"] = 16 * f * ah * (1.0 + a)                                # y pass
        b["forward_z_assemble"] = 16 * f * ah * a + (8 + 8 + 8 + 8) * f * ah * a * a
    else:
        b["strided_forward"] = 16 * f * ah * (1.0 + a) + 16 * f * ah * (a + a * a)    # y pass, z pass
        b["assemble"] = (16 + 8 + 8 + 8 + 8) * f * ah * a * a
    return b


def unpruned_reference_bytes(N: int) -> float:
    """148 field-sweeps x 8 B = 1184 B per grid-point-step (fused, unpruned three-pass design)."""
    return 1184.0 * N ** 3


# ----------------------------------------------------------------------------------------------------------------
def run_reference(args):
    """Reference arm of this tier = the CPU oracle, as it stands, on a bounded sample of the workload."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import oracle
    from paper_1810_12707_b200 import inputs
    n = 128
    cfg = inputs.config45(n)
    o = oracle.Oracle(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
    o.set_fields(cfg.prim, "primitive")
    for _ in range(args.warmup):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(1)
    dt = time.perf_counter() - t0
    value = n ** 3 * args.steps / dt
    cores = oracle.get_threads()
    sample = "config 4/5 initial condition on a %d^3 grid, %d AB2 steps (bounded sample of the %d^3 workload)" % (n, args.steps, args.size)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config5_abc_dynamo_%d" % args.size, "reference_grid": n, "integrator": "AB2"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def cpu_baseline(size):
    """The oracle as it stands on a bounded sample: 128^3 grid of the same initial condition, all host cores (the headline
    `value`) and one thread (single-thread and all-cores)."""
    import oracle
    from paper_1810_12707_b200 import inputs
    all_cores = oracle.get_threads()
    res = {}
    for label, threads, n, steps in (("all_cores", all_cores, 128, 10), ("single_thread", 1, 64, 3)):
        cfg = inputs.config45(n)
        oracle.set_threads(threads)
        o = oracle.Oracle(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
        o.set_fields(cfg.prim, "primitive")
        o.step(1)
        t0 = time.perf_counter()
        o.step(steps)
        dt = time.perf_counter() - t0
        res[label] = {"value": n ** 3 * steps / dt, "cores": threads, "steps": steps, "seconds": dt, "n": n}
        o.close()
    oracle.set_threads(all_cores)
    a = res["all_cores"]
    return {"value": a["value"], "unit": UNIT, "cores": a["cores"], "kind": "oracle",
            "sample": "config 4/5 initial condition on a %d^3 grid, %d AB2 steps, %.1f s (bounded sample of the %d^3 workload)"
                      % (a["n"], a["steps"], a["seconds"], size),
            "single_thread": {"value": res["single_thread"]["value"], "cores": 1,
                              "sample": "%d^3 grid, %d AB2 steps, %.1f s" % (res["single_thread"]["n"], res["single_thread"]["steps"],
                                                                             res["single_thread"]["seconds"])}}


def time_steps(g, torch, nsteps, dist):
    """Device time of mhd_step(nsteps) on the solver's stream, barrier + synchronize on both sides."""
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    g.step(nsteps)
    e1.record(g.stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return e0.elapsed_time(e1)


def fft_metric(g, torch, N, peak, nf=8, reps=5):
    """Stand-alone batched 3-D R2C + C2R (BASELINE.json: '3D FFT achieved HBM GB/s vs peak')."""
    H = N // 2
    real = [torch.randn((N, N, N), dtype=torch.float64, device=g.device) for _ in range(nf)]
    spec = [torch.empty((N, N, H, 2), dtype=torch.float64, device=g.device) for _ in range(nf)]
    out = {}
    for prune in (False, True):
        for name, fn in (("r2c", lambda: g.fft3d_r2c(real, spec, None, prune)), ("c2r", lambda: g.fft3d_c2r(spec, real, prune))):
            fn(); fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(g.stream)
            for _ in range(reps):
                fn()
            e1.record(g.stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            gbs = 48.0 * N ** 3 * nf / ms / 1e6
            out[name + ("_pruned" if prune else "")] = {"ms_per_field": ms / nf, "gbs_3pass_48B_per_pt": gbs,
                                                         "frac_of_peak_3pass": gbs / peak,
                                                         "gbs_1r1w_16B_per_pt": 16.0 * N ** 3 * nf / ms / 1e6}
    # cuFFT (via torch.fft) as a timing reference only — never on the product path
    x = real[0]
    del spec, real                                       # cuFFT needs its own work area: give the memory back first
    y = torch.empty((N, N, H + 1), dtype=torch.complex128, device=g.device)
    for _ in range(3):
        torch.fft.rfftn(x, out=y)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(4 * reps):
        torch.fft.rfftn(x, out=y)
    e1.record()
    torch.cuda.synchronize()
    out["cufft_d2z_reference_ms_per_field"] = e0.elapsed_time(e1) / (4 * reps)
    out["accounting"] = "SURVEY.md 8(d): 3 passes x (8 B read + 8 B written) = 48 B per point and transform; peak = %.0f GB/s measured copy" % peak
    del y, x
    return out


def tracer_metric(g, torch, N, L, np_, K, ms_step_plain):
    """Tracer particles (Sec. VI): particle-pushes/s of the gather + Boris kernel in a frozen field (two
    launches of different length, so that the 3-field inverse transform of mhd_tracers_push cancels), and the cost of
    carrying the tracers through mhd_step (B taken from the fused x sweep)."""
    gen = torch.Generator(device=g.device).manual_seed(7)
    pos = [torch.rand(np_, dtype=torch.float64, device=g.device, generator=gen) * L for _ in range(3)]
    g.tracers_set(pos)                      # v0 = CIC of u

    def timed(fn):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(g.stream); fn(); e1.record(g.stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    g.tracers_push(1)
    n1, n2 = 2, 22
    t1 = min(timed(lambda: g.tracers_push(n1)) for _ in range(3))
    t2 = min(timed(lambda: g.tracers_push(n2)) for _ in range(3))
    per_push_ms = (t2 - t1) / (n2 - n1)
    g.step(2)
    ms_with = timed(lambda: g.step(K)) / K
    # bytes that must move per push: 6 x 8 B of particle state read + written; the grid rows come from L1 / L2 once the
    # storage is sorted by grid row (MHD_OPT_TRACER_SORT), from DRAM at sector granularity (~670 B per push) if it is not
    return {"particles": np_, "pushes_per_s_frozen_field": np_ / (per_push_ms * 1e-3), "ms_per_push_launch": per_push_ms,
            "particle_state_bytes_per_push": 96, "particle_state_gbs": 96.0 * np_ / per_push_ms / 1e6,
            "ms_per_step_with_tracers": ms_with, "ms_per_step_without": ms_step_plain,
            "step_overhead_frac": ms_with / ms_step_plain - 1.0,
            "positions": "uniform random (seeded) in the box; v0 = CIC of u"}


def pcie_peaks(torch, device, nbytes=1 << 30, reps=4):
    """Measured pinned-memory copy bandwidth of this box (GB/s): host->device alone, device->host alone, and both
    directions at once on two streams — the ceiling of the chunked pipeline when arrays live on the host."""
    h_in = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    h_out = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d_in = torch.empty(nbytes, dtype=torch.uint8, device=device)
    d_out = torch.empty(nbytes, dtype=torch.uint8, device=device)
    s1, s2 = torch.cuda.Stream(device), torch.cuda.Stream(device)

    def run(do_in, do_out):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(reps):
            if do_in:
                with torch.cuda.stream(s1):
                    d_in.copy_(h_in, non_blocking=True)
            if do_out:
                with torch.cuda.stream(s2):
                    h_out.copy_(d_out, non_blocking=True)
        torch.cuda.synchronize()
        return nbytes * reps / (time.perf_counter() - t0) / 1e9

    run(True, True)
    return {"h2d_alone_gbs": run(True, False), "d2h_alone_gbs": run(False, True), "each_direction_when_both_gbs": run(True, True)}


def hbm_peak():
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        return float(json.load(open(peaks_path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def build_roofline(g, N, K, step_ms, prof, peak, peak_src, fuse_current=True, fuse_s5=False, in_core=True, rhs_per_step=1):
    """per kernel family, algorithmic bytes per launch / CUDA-event time per launch against the HBM copy
    peak; the dominant family (largest share of the step) is the top-level object."""
    sb = sweep_bytes(N, prune=True, fuse_current=fuse_current, fuse_s5=fuse_s5)
    fam = {}
    for name, b in sb.items():
        p = prof.get(name, {"ms": 0.0, "launches": 0})
        if p["launches"] == 0:
            continue
        per_launch_bytes = b * rhs_per_step * K / p["launches"]
        avg_ms = p["ms"] / p["launches"]
        fam[name] = {"ms_per_step": p["ms"] / K, "launches_per_step": p["launches"] / K,
                     "alg_bytes_per_launch": per_launch_bytes, "avg_launch_ms": avg_ms,
                     "gbs": per_launch_bytes / avg_ms / 1e6, "frac_of_peak": per_launch_bytes / avg_ms / 1e6 / peak}
    if not fam:
        return None
    dom = max(fam, key=lambda k: fam[k]["ms_per_step"])
    alg_pruned = sum(sb.values()) * rhs_per_step
    roofline = {"bound": "hbm", "kernel": dom, "achieved": fam[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": fam[dom]["frac_of_peak"], "traffic": None, "peak_source": peak_src,
                "share_of_step": fam[dom]["ms_per_step"] / step_ms,
                "whole_step": {"alg_bytes_pruned": alg_pruned, "gbs_pruned": alg_pruned / step_ms / 1e6,
                               "frac_pruned": alg_pruned / step_ms / 1e6 / peak,
                               "alg_bytes_unpruned_1184B": unpruned_reference_bytes(N),
                               "gbs_vs_1184B": unpruned_reference_bytes(N) / step_ms / 1e6,
                               "frac_vs_1184B": unpruned_reference_bytes(N) / step_ms / 1e6 / peak,
                               "frac_vs_1184B_nominal_8TBs": unpruned_reference_bytes(N) / step_ms / 1e6 / 8000.0},
                "families": fam}
    tpath = os.path.join(ROOT, TRAFFIC_FILE)
    if os.path.exists(tpath):   # DRAM bytes per launch from the committed ncu capture: NOT measured in this run
        try:
            tj = json.load(open(tpath))
            tr = tj.get(str(N), {})
            roofline["traffic"] = tr.get(dom)
            roofline["traffic_source"] = "%s (ncu dram__bytes_read + dram__bytes_write per launch, capture of commit %s; not measured in this run)" % (
                TRAFFIC_FILE, tj.get("commit", "?"))
            if in_core and all(k in tr for k in fam):
                roofline["whole_step"]["dram_bytes_measured_ncu"] = sum(tr[k] * fam[k]["launches_per_step"] for k in fam)
        except Exception:
            pass
    if "x_fused" in fam and in_core:
        # the fused x sweep on FLOPS: SURVEY.md 8(d) count (27 x 2.5 N log2 N + 90 N per line) against twice the DFMA
        # instruction rate of the fp64 pipe, measured in this run by a register-only FMA kernel (mhd_probe_fp64)
        flops = fused_flops_per_line(N) * N * N
        peak_f = 2.0 * g.probe_fp64()
        ach = flops / (fam["x_fused"]["avg_launch_ms"] * 1e-3)
        roofline["alu"] = {"bound": "alu", "kernel": "x_fused", "achieved": ach / 1e12, "peak": peak_f / 1e12, "unit": "TFLOP/s (fp64)",
                           "frac": ach / peak_f, "flops_per_line": fused_flops_per_line(N),
                           "flop_count": "SURVEY.md 8(d): 27 real line transforms x 2.5 N log2 N + 90 N point-wise, per (y,z) line",
                           "peak_source": "2 x the DFMA rate of a register-only kernel measured in this run (mhd_probe_fp64); "
                                          "64 lanes/clk/SM x 148 SMs x 1.965 GHz x 2 = %.1f TFLOP/s" % (148 * 64 * 1.965e9 * 2 / 1e12)}
    return roofline


def measure_other_size(MHD, inputs, torch, N, device, peak, peak_src, steps=50, warm=5):
    """The second size the metric is quoted on, measured in the same run: value, ms per step, family fractions."""
    cfg = inputs.config45(N)
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, device=device)
    g.set_fields([torch.from_numpy(p).to(device) for p in cfg.prim], "primitive")
    g.step(warm)
    g.profile_enable(True)
    ms = time_steps(g, torch, steps, None)
    prof = g.profile_get()
    g.profile_enable(False)
    r = build_roofline(g, N, steps, ms / steps, prof, peak, peak_src)
    out = {"workload": "config4_abc_dynamo_%d^3" % N, "value": float(N) ** 3 * steps / (ms * 1e-3), "unit": UNIT,
           "ms_per_step": ms / steps, "steps": steps, "warmup": warm,
           "roofline": {k: r[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "share_of_step", "traffic")},
           "families": {k: {"ms_per_step": v["ms_per_step"], "frac_of_peak": v["frac_of_peak"]} for k, v in r["families"].items()},
           "whole_step": r["whole_step"]}
    if "alu" in r:
        out["alu"] = {k: r["alu"][k] for k in ("achieved", "peak", "unit", "frac")}
    del g
    torch.cuda.empty_cache()
    return out


def measure_1024(MHD, inputs, torch, device, peak, peak_src, steps=3, warm=1):
    """BASELINE config 6 (1024^3) where the driver sees it: the chunked pipeline with every array in HBM
    (compact storage, 106 GB, no PCIe traffic in the step), a few steps timed with CUDA events.  Skips with a stated reason
    when the GPU or the host lacks the memory: 8 x 8.6 GB of inputs are synthesised in (pageable) host memory and handed to
    mhd_set_fields as host pointers."""
    from paper_1810_12707_b200 import binding as B
    N = 1024
    need_dev = B.lib().mhd_workspace_bytes(N, B.MHD_FLAG_OUT_OF_CORE) + (20 << 30)     # + input synthesis / staging headroom
    free_dev = torch.cuda.mem_get_info(device)[0]
    if free_dev < need_dev:
        return {"skipped": "needs %.0f GB of free HBM, %.0f GB free" % (need_dev / 1e9, free_dev / 1e9)}
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = None
    if avail is not None and avail < 90e9:
        return {"skipped": "needs ~75 GB of host memory for the synthetic inputs, %.0f GB available" % (avail / 1e9)}
    t0 = time.perf_counter()
    cfg = inputs.config6(N)
    t_inputs = time.perf_counter() - t0
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, device=device, flags=B.MHD_FLAG_OUT_OF_CORE)
    t0 = time.perf_counter()
    g.set_fields(cfg.prim, "primitive")
    t_set = time.perf_counter() - t0
    cfg.prim = None
    g.step(warm)
    g.profile_enable(True)
    l0 = g.launch_count()
    ms = time_steps(g, torch, steps, None)
    launches = g.launch_count() - l0
    prof = g.profile_get()
    g.profile_enable(False)
    d = g.diagnostics()
    out = {"workload": "config6_turbulence_out_of_core_1024^3", "placement": "device (compact storage, everything in HBM)",
           "value": float(N) ** 3 * steps / (ms * 1e-3), "unit": UNIT, "s_per_step": ms / steps / 1e3, "steps": steps, "warmup": warm,
           "device_workspace_gb": g.workspace_bytes / 1e9, "gpu_launches": launches,
           "inputs_s": t_inputs, "set_fields_from_pageable_host_s": t_set,
           "sanity": {"rho_min": d["rho_min"], "p_min": d["p_min"], "max_divb": d["max_divb"], "mass": d["mass"]},
           "paper_context": "PAPER.md Table III L368-375: 512^3 out-of-core 80.97 s/step (P100); no 1024^3 in the paper"}
    try:
        r = build_roofline(g, N, steps, ms / steps, prof, peak, peak_src, in_core=False)
        if r:
            out["families"] = {k: {"ms_per_step": v["ms_per_step"], "frac_of_peak": v["frac_of_peak"]} for k, v in r["families"].items()}
            out["whole_step"] = {k: r["whole_step"][k] for k in ("alg_bytes_pruned", "gbs_pruned", "frac_pruned")}
    except Exception as e:          # the family accounting is a by-product; the timing above stands without it
        out["families_error"] = repr(e)
    del g
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    rank, local_rank, world = dist_env()
    import torch
    if not torch.cuda.is_available():
        print(json.dumps({"error": "no CUDA device; the product path has no CPU fallback"}))
        return 2
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        backend = os.environ.get("MHD_BENCH_BACKEND", "nccl")      # "gloo": several ranks on ONE GPU in the tests
        if backend == "nccl":
            dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        else:
            dist_mod.init_process_group(backend)
        dist = dist_mod
    from paper_1810_12707_b200 import build as mhd_build
    if rank == 0:
        mhd_build.build()
    if dist is not None:
        dist.barrier()
    from paper_1810_12707_b200 import MHD, inputs

    N = args.size
    from paper_1810_12707_b200 import binding as B
    flags = {"incore": 0, "device": B.MHD_FLAG_OUT_OF_CORE, "state_host": B.MHD_FLAG_OUT_OF_CORE | B.MHD_FLAG_STATE_ON_HOST,
             "all_host": B.MHD_FLAG_OUT_OF_CORE | B.MHD_FLAG_STATE_ON_HOST | B.MHD_FLAG_WORK_ON_HOST}[args.placement]
    if args.budget_mib:
        flags |= B.MHD_FLAG_BUDGET_MIB(args.budget_mib)
    if N == 1024 and not flags:
        print(json.dumps({"error": "1024^3 does not fit in core (48 full fields = 412 GB): use --placement device|state_host|all_host"}))
        return 2
    cfg = inputs.config6(N) if N == 1024 else inputs.config45(N)     # config 6 = the out-of-core workload of BASELINE.json
    if args.decompose:
        # slab decomposition: ONE problem over all ranks, two all-to-alls per step (strong scaling)
        from paper_1810_12707_b200.dist import DistMHD
        flags = B.MHD_FLAG_OUT_OF_CORE
        g = DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, rank=rank, world=world, device="cuda:%d" % local_rank,
                    per_rank_storage=True)
        if world > 1 and not args.packed_exchange:
            g.connect_peers_ipc()        # rows go straight into the owners' workspaces (P2P stores); barriers instead of all-to-alls
        args.no_e2e = args.no_fft = True
    else:
        g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, device="cuda:%d" % local_rank, flags=flags)
    pin_inputs = N < 1024        # 8 x 8.6 GB of inputs stay pageable at 1024^3 (the pinned budget goes to the solver's arrays)
    host = [torch.from_numpy(p).pin_memory() if pin_inputs else torch.from_numpy(p) for p in cfg.prim]
    cfg.prim = None
    opts = {}
    integ = {"ab2": 0, "rk4": 1, "pc": 2}[args.integrator]
    if integ:
        g.set_option(3, integ)      # MHD_OPT_INTEGRATOR
    for kv in args.option:
        k, v = kv.split("=")
        opts[int(k)] = int(v)
        g.set_option(int(k), int(v))
    g.set_fields(host, "primitive")
    if args.no_e2e:
        host = None          # frees the input copies (matters at 1024^3: 69 GB)
    K, W = args.steps, max(args.warmup, 3)

    # ---- device-resident timing -----------------------------------------------------------------------------
    g.step(W)
    sampler = ClockSampler(local_rank).start()
    g.profile_enable(True)
    l0 = g.launch_count()
    ms = time_steps(g, torch, K, dist)
    launches = g.launch_count() - l0
    prof = g.profile_get()
    ooc = None
    if flags:
        g.profile_enable(False)
        x0 = g.transfer_bytes()
        e0 = getattr(g, "exchanged_bytes", 0)
        ms_np = time_steps(g, torch, K, dist)
        e1 = getattr(g, "exchanged_bytes", 0)          # without the per-family events (they serialise nothing, but to be sure)
        x1 = g.transfer_bytes()
        ms = ms_np
        ooc = {"placement": args.placement, "budget_mib": args.budget_mib, "device_workspace_gb": g.workspace_bytes / 1e9,
               "pinned_host_gb": g.pinned_bytes / 1e9, "in_core_workspace_gb": 48 * 8.0 * N ** 3 / 1e9,
               "h2d_bytes_per_step": (x1[0] - x0[0]) / K, "d2h_bytes_per_step": (x1[1] - x0[1]) / K,
               "h2d_gbs": (x1[0] - x0[0]) / ms_np / 1e6, "d2h_gbs": (x1[1] - x0[1]) / ms_np / 1e6,
               "s_per_step": ms_np / K / 1e3}
        if g.pinned_bytes:
            ooc["pcie_measured"] = pcie_peaks(torch, g.device)
            ooc["bound"] = "pcie"
            ooc["frac_of_duplex_pcie"] = max(ooc["h2d_gbs"], ooc["d2h_gbs"]) / ooc["pcie_measured"]["each_direction_when_both_gbs"]
    g.profile_enable(False)
    clocks = sampler.stop()
    if args.decompose:
        ooc["decomposed"] = {"world": world, "sent_to_peers_bytes_per_step_per_rank": (e1 - e0) / K,
                             "exchange": "direct P2P stores from the z-pass / forward-y kernels + 2 barriers per step" if g.direct else
                                         "packed: torch.distributed.all_to_all_single (NCCL), 2 per step: 11 and 16 work fields"}
    ms_max, units = aggregate(ms, float(N) ** 3 * K / (world if args.decompose else 1), dist)
    value = units / (ms_max * 1e-3)

    # ---- roofline of the dominant kernel family ---------------------------------------------------------------
    peak, peak_src = hbm_peak()
    fuse_s5 = opts.get(14, 0) != 0      # MHD_OPT_FUSE_ASSEMBLE (include/mhd_bench.h)
    roofline = build_roofline(g, N, K, ms / K, prof, peak, peak_src, fuse_current=opts.get(4, 1) != 0, fuse_s5=fuse_s5,
                              in_core=not flags, rhs_per_step={"ab2": 1, "rk4": 4, "pc": 2}[args.integrator])
    alg_pruned = sum(sweep_bytes(N, True, opts.get(4, 1) != 0, fuse_s5).values()) * {"ab2": 1, "rk4": 4, "pc": 2}[args.integrator]

    # ---- end to end through the C ABI with host buffers ----------------------------------------------------------
    e2e = None
    if not args.no_e2e:
        outh = host   # results land in the same pinned buffers
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        g.set_fields(host, "primitive")        # host pointers: returns after the stream has drained
        t1 = time.perf_counter()
        g.step(K)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        g.get_fields("primitive", "host", out=outh)
        torch.cuda.synchronize()
        t3 = time.perf_counter()
        t_e2e = (t3 - t0) * 1e3
        ms_e, units_e = aggregate(t_e2e, float(N) ** 3 * K, dist)
        fb = 8.0 * N ** 3 * 8
        e2e = {"value": units_e / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": fb / K, "d2h_bytes_per_step": fb / K,
               "what": "mhd_set_fields(%s host) + mhd_step(%d) + mhd_get_fields(%s host), wall clock"
                       % ("pinned" if pin_inputs else "pageable", K, "pinned" if pin_inputs else "pageable"),
               # where the end-to-end time goes on this rank: the two calls that cross PCIe (copy + 8 transforms each) and the steps
               "copy_s": {"set_fields": t1 - t0, "get_fields": t3 - t2, "steps": t2 - t1,
                          "pcie_gbs_if_all_copy": 2 * fb / 1e9 / max((t1 - t0) + (t3 - t2), 1e-9)}}

    extra = {}
    if rank == 0 and not args.no_fft and not flags:
        host = None
        extra["fft3d"] = fft_metric(g, torch, N, peak)
    if rank == 0 and args.tracers > 0 and not flags:
        extra["tracers"] = tracer_metric(g, torch, N, cfg.L, args.tracers, K, ms / K)
    if rank == 0 and world == 1 and not flags and N == 512 and not args.no_256 and not opts and not integ:
        g = None
        torch.cuda.empty_cache()
        extra["size_256"] = measure_other_size(MHD, inputs, torch, 256, "cuda:%d" % local_rank, peak, peak_src)
        if not args.no_1024:
            try:
                extra["size_1024"] = measure_1024(MHD, inputs, torch, "cuda:%d" % local_rank, peak, peak_src)
            except Exception as e:      # never lose the headline line to the optional largest size
                extra["size_1024"] = {"skipped": "failed: %r" % (e,)}
                torch.cuda.empty_cache()
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(N)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "strong" if args.decompose else "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": ("config6_turbulence_out_of_core_%d^3" % N) if N == 1024 else
                           "config%d_abc_dynamo_%d^3" % (5 if N == 512 else 4, N), "N": N, "dt": cfg.dt, "placement": args.placement,
                           "mu": cfg.mu, "eta": cfg.eta, "integrator": args.integrator.upper(), "rhs_per_step": {"ab2": 1, "rk4": 4, "pc": 2}[args.integrator],
                           "options": opts, "pruned": 1,
                           "parallelism": ("slab decomposition x%d" if args.decompose else "replicas x%d") % world,
                           "l2": "no flush: one step streams %.1f GB, far beyond the 126 MB L2" % (alg_pruned / 1e9)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu, "out_of_core": ooc,
                "paper_context": {"256^3 s/step P100/V100": [0.32, 0.22], "512^3 s/step P100/V100 (out-of-core)": [80.97, 92.81],
                                  "source": "PAPER.md Table III L368-375; other hardware, context only"}}
        line.update(extra)
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--size", type=int, default=512, choices=[64, 128, 256, 512, 1024])
    ap.add_argument("--placement", default="incore", choices=["incore", "device", "state_host", "all_host"],
                    help="incore: the tuned in-core path; others: the chunked pipeline (include/mhd.h MHD_FLAG_OUT_OF_CORE) with "
                         "everything in HBM / U^ and R^old in pinned host memory / the work fields there too")
    ap.add_argument("--budget-mib", type=int, default=0, help="cap on the device workspace of the chunked pipeline")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-fft", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-256", action="store_true", help="skip the 256^3 measurement that the default 512^3 run adds")
    ap.add_argument("--no-1024", action="store_true", help="skip the 1024^3 (config 6, everything in HBM) measurement of the default run")
    ap.add_argument("--decompose", action="store_true",
                    help="with --gpus N under torchrun: ONE problem decomposed over the N GPUs (ky bricks / z slabs, two NCCL "
                         "all-to-alls per step) instead of N replicas; with N = 1 it measures the pack / unpack overhead")
    ap.add_argument("--packed-exchange", action="store_true",
                    help="--decompose: pack -> NCCL all_to_all_single -> unpack instead of direct peer stores")
    ap.add_argument("--integrator", default="ab2", choices=["ab2", "rk4", "pc"],
                    help="time integrator (PAPER.md L25, Table I): Adams-Bashforth 2 (the metric's), RK4, predictor-corrector")
    ap.add_argument("--tracers", type=int, default=0, metavar="NP",
                    help="also measure NP tracer particles (PAPER.md Sec. VI): frozen-field pushes/s and the step overhead")
    ap.add_argument("--option", action="append", default=[], metavar="ID=VALUE",
                    help="mhd_set_option(ID, VALUE) before the run (include/mhd.h MHD_OPT_*), for A/B measurements")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
