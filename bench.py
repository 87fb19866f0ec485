#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the SMAUG+ hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one full MHD time step (dt reduction + 4 x {ghost fill, fused RHS/hyperdiffusion/RK stage
kernel}) over the whole grid.  Default workload at N=1: Orszag-Tang 8000 x 8000, fp64, periodic, CFL 0.3,
hyperdiffusion on, RK4 -- the configuration BASELINE.json's north_star quotes the target on; its state
(3.1 GB per buffer) is far larger than L2, so no L2 flush is needed between timed iterations.

Prints ONE JSON line (rank 0).  `value` = cell-updates/s with the state resident in HBM; `e2e` = the same
through the C ABI with HOST buffers (set_state H2D + steps + get_state D2H inside the timed region);
`roofline` = algorithmic bytes of the fused stage kernel / its CUDA-event duration vs the measured HBM peak;
`cpu_baseline` = the oracle, as it stands, timed on one host core on a bounded sample of the same workload.
The default invocation (one GPU, no workload flags) also carries `rows`: compact entries (ms_per_step, roofline.frac,
kernel, clocks; each timed for >= 0.5 s) for 8000 x 8000 without hyperdiffusion, BASELINE configs 1-4, 8000 x 8000 on a
uniform background, the 256^3 three-dimensional form and the 2 x 2 decomposition group; `--no-rows` leaves them out.
N > 1: the path does not shard ("replicas only") -- every rank runs an independent replica.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import smaug_inputs as si  # noqa: E402

WORKLOADS = {
    # name: (nx, ny, generator, default steps)
    "orszag_tang_8000": (8000, 8000, "ot"),
    "orszag_tang_4000": (4000, 4000, "ot"),
    "orszag_tang_2044": (2044, 2044, "ot"),
    "orszag_tang_1000": (1000, 1000, "ot"),
    "brio_wu_800": (800, 1, "bw"),
    # SURVEY 8(f) NEXT-2 (not a BASELINE config): stratified magnetised atmosphere with a pulse, non-uniform
    # background + gravity, periodic in x, open in y -- split_kernel<128, .., BG>
    "stratified_4000": (4000, 4000, "strat"),
    # SURVEY 8(d) extra row: the 8000^2 Orszag-Tang state as a perturbation on a uniform non-zero background
    # (exercises the background loads and the energy source) -- split_kernel<128, .., BG>
    "orszag_tang_8000_bg": (8000, 8000, "otbg"),
    # the three-dimensional form (include/smaug3d.h): a 3-D Orszag-Tang-like vortex, eight fields,
    # periodic, hyperdiffusion on, RK4 (smaug_inputs.orszag_tang_3d; the paper prints no 3-D configuration)
    "orszag_tang_3d_128": (128, 128, "ot3d"),
    "orszag_tang_3d_256": (256, 256, "ot3d"),
    "orszag_tang_3d_384": (384, 384, "ot3d"),
}
# Algorithmic HBM bytes per cell-update of the fused step as built: per stage the
# kernel reads the 6 input planes once and writes 6; stages 2-3 also read w^n; stage 2 also writes the
# accumulator; stage 4 reads it:  96 + 192 + 144 + 144 = 576 B (SURVEY 8(d) counts 624 for its variant).
BYTES_PER_CELL_UPDATE = 576.0
STAGES_PER_STEP = 4
# Second ceiling, reported beside the HBM roofline: fp64-pipe thread-instructions the stage
# kernel executes per cell and launch (DFMA + DADD + DMUL + DSETP), taken from the committed ncu capture
# (sm__inst_executed_pipe_fp64.sum x 32 / cells; profiles/stage_kernel_ncu.json), against 64 fp64 lanes per SM and clock.
FP64_LANES_PER_SM = 64
N_SM = 148
METRIC = "fp64 MHD cell-updates/s"
UNIT = "cell-updates/s"


def make_state(name):
    """(w, bc, gamma, bg, (gx, gy)) of a workload."""
    nx, ny, kind = WORKLOADS[name]
    if kind == "strat":
        return si.stratified_atmosphere(nx, ny)
    if kind == "otbg":
        w, bc, gamma = si.orszag_tang(nx, ny)
        rho_b, e_b, bx_b, by_b = 0.1, 0.2, 0.05, 0.03
        w[0] -= rho_b; w[3] -= e_b; w[4] -= bx_b; w[5] -= by_b
        return w, bc, gamma, si.uniform_background(nx, ny, rho_b, e_b, bx_b, by_b), (0.0, 0.0)
    w, bc, gamma = si.orszag_tang(nx, ny) if kind == "ot" else si.brio_wu(nx, ny)
    return w, bc, gamma, None, (0.0, 0.0)


def bytes_per_cell_update(has_bg, rk_order=4):
    """Algorithmic HBM bytes per cell-update: RK4 576 (see above); RK2 (midpoint) 96 + 144 = 240 (stage 2 reads w1 with
    its halo and w^n pointwise, writes w^{n+1}); Euler 96; + the four background planes read once per stage."""
    stages = {4: 4, 2: 2, 1: 1}[rk_order]
    return {4: BYTES_PER_CELL_UPDATE, 2: 240.0, 1: 96.0}[rk_order] + (stages * 4 * 8 if has_bg else 0)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:  # noqa: BLE001
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_capture(key):
    """Per-launch counters of the stage kernel from the committed `ncu --set full` capture of this workload key
    (profiles/stage_kernel_ncu.json, written from the capture named there), or {}: `dram_bytes` = dram__bytes_read.sum +
    dram__bytes_write.sum, `fp64_thread_inst_per_cell` = 32 x sm__inst_executed_pipe_fp64.sum / cells (mean of the RK
    stages).  These are constants of a committed capture, not measurements of this run: `capture` says which."""
    p = os.path.join(ROOT, "profiles", "stage_kernel_ncu.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get(key) or {}
        except Exception:  # noqa: BLE001
            return {}
    return {}


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:  # noqa: BLE001
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:  # noqa: BLE001
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx = float(parts[1])
            except ValueError:
                continue
            for nm, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(values, device, world):
    """MAX over ranks of a list of floats (replica timing: the job is as slow as its slowest rank)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def replica_value(cells, steps, world, ms):
    """Whole-job cell-updates/s of `world` independent replicas that all finished within `ms`."""
    return world * float(cells) * steps / (ms * 1e-3)


def oracle_rate(sample_n, steps, warmup=0, threads=1, kind="ot"):
    """cell-updates/s of the oracle (as it stands) on a sample_n^2 grid of the workload's kind."""
    import oracle
    if kind == "strat":
        w, bc, gamma, bg, (gx, gy) = si.stratified_atmosphere(sample_n, sample_n)
        o = oracle.Oracle(sample_n, sample_n, gamma, bc, bg=bg, threads=threads, gx=gx, gy=gy)
    elif kind == "otbg":
        w, bc, gamma = si.orszag_tang(sample_n)
        w[0] -= 0.1; w[3] -= 0.2; w[4] -= 0.05; w[5] -= 0.03
        o = oracle.Oracle(sample_n, sample_n, gamma, bc, bg=si.uniform_background(sample_n, sample_n, 0.1, 0.2, 0.05, 0.03),
                          threads=threads)
    else:
        w, bc, gamma = si.orszag_tang(sample_n)
        o = oracle.Oracle(sample_n, sample_n, gamma, bc, threads=threads)
    o.set_state(w)
    if warmup:
        o.step(warmup, 0.3)
    t0 = time.perf_counter()
    o.step(steps, 0.3)
    el = time.perf_counter() - t0
    o.close()
    return sample_n * sample_n * steps / el, el


# Rows the default invocation adds beside the headline (BASELINE.json lists five configs, SURVEY 8(d):
# "additionally report each OT size with HD_ON=0"): (workload, hyperdiffusion on, decomposition or None)
ROWS = [("orszag_tang_8000", False, None), ("brio_wu_800", True, None), ("orszag_tang_1000", True, None),
        ("orszag_tang_2044", True, None), ("orszag_tang_4000", True, None), ("orszag_tang_8000_bg", True, None),
        ("orszag_tang_3d_256", True, None), ("orszag_tang_8000", True, (2, 2))]


def compact_row(pkg, name, hd=True, decomp=None, min_ms=500.0, device=0, state=None):
    """One entry of `rows`: the workload timed on the device for at least `min_ms` (step count calibrated from a short
    untimed run that also serves as warm-up), once as the product runs it (CUDA-graph replay where the library uses
    it) for ms_per_step, and -- for a single 2-D context -- once more with CUDA events around the stage kernels for
    the roofline fraction of the fused stage kernel.  Clocks are sampled from before the calibration run to the end."""
    import torch
    nx, ny, kind = WORKLOADS[name]
    sampler = ClockSampler(device)
    three_d = kind == "ot3d"
    if three_d:
        w_np, bc, gamma = si.orszag_tang_3d(nx)
        sim = pkg.Smaug3D(nx, nx, nx, gamma, bc, hd_on=1 if hd else 0)
        cells, has_bg = float(nx) ** 3, False
        sim.set_state(torch.from_numpy(w_np))
    else:
        w_np, bc, gamma, bg_np, (gx, gy) = state if state is not None else make_state(name)
        bg = None if bg_np is None else torch.from_numpy(bg_np).cuda(device)
        has_bg = bg_np is not None
        params = dict(hd_on=1 if hd else 0, gx=gx, gy=gy)
        sim = (pkg.SmaugGroup(decomp[0], decomp[1], nx, ny, gamma, bc, bg=bg, **params) if decomp
               else pkg.Smaug(nx, ny, gamma, bc, bg=bg, device=torch.device("cuda", device), **params))
        cells = float(nx) * ny
        sim.set_state(w_np if torch.is_tensor(w_np) else torch.from_numpy(w_np))
    del w_np

    def timed(k):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        sim.step(k, 0.3)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    k0 = 200 if cells < 1e4 else (20 if cells < 2e6 else 4)
    timed(k0)                                                   # warm-up (graph capture, smem attributes)
    per = timed(k0) / k0
    K = int(min(max(8, math.ceil(min_ms / per)), 200000))
    ms = timed(K)
    row = {"workload": name, "hd": hd, "steps": K, "ms_per_step": ms / K, "value": cells * K / (ms * 1e-3), "unit": UNIT,
           "launch_path": "as smaug_step runs it (CUDA-graph replay where the library uses it)"}
    peak, _ = peaks()
    if decomp:
        row["decomposition"] = f"{decomp[0]}x{decomp[1]} members on one device (smaug_group_*)"
        row["kernel"] = "smaug::split_kernel per member + group_pull_kernel"
        row["roofline"] = {"frac": cells * BYTES_PER_CELL_UPDATE / (ms / K * 1e-3) / 1e9 / peak,
                           "basis": "whole step: 576 B per cell-update / ms_per_step (exchange and barriers included)"}
    elif three_d:
        row["kernel"] = "smaug3 RK stage (ghost3, kappa3, stage3)"
        cap = ncu_capture(name)
        row["roofline"] = {"frac": cells * 768.0 / (ms / K * 1e-3) / 1e9 / peak,
                           "basis": "whole step: 768 B per cell-update of a fully fused stage / ms_per_step; the kernels as "
                                    "built move more than that (kappa / Phi volumes go through HBM): see traffic",
                           "algorithmic_bytes_per_stage": 192.0 * cells, "traffic": cap.get("dram_bytes"),
                           "traffic_over_algorithmic": (cap["dram_bytes"] / (192.0 * cells)) if cap.get("dram_bytes") else None,
                           "traffic_source": cap.get("capture")}
    else:
        row["kernel"] = "smaug::" + sim.kernel_name()
        bpcu = bytes_per_cell_update(has_bg, 4)
        if sim.kernel_name().startswith("line_step_kernel"):
            row["roofline"] = {"frac": None, "basis": "whole steps in one persistent cluster launch, state in distributed "
                                                      "shared memory: no HBM traffic per step to set against a roofline"}
        else:
            sim.set_kernel_timing(True)
            k2 = max(8, K // 4)
            ms2 = timed(k2)
            stage_ms, stage_n = sim.kernel_timing()
            sim.set_kernel_timing(False)
            avg = stage_ms / max(stage_n, 1)
            ach = bpcu / 4 * cells / (avg * 1e-3) / 1e9
            row["roofline"] = {"frac": ach / peak, "achieved": ach, "unit": "GB/s", "avg_launch_ms": avg, "launches_timed": stage_n,
                               "bytes_per_launch": bpcu / 4 * cells, "ms_per_step_with_events": ms2 / k2,
                               "basis": "fused stage kernel alone: algorithmic bytes per launch / CUDA-event duration"}
            if cells * 48 * 4 < 4e8:
                row["roofline"]["l2"] = "working set comparable to L2 (126 MB): DRAM traffic is below algorithmic"
    t_sim, dt_last = sim.time()
    row["sim"] = {"t": t_sim, "last_dt": dt_last}
    row["clocks"] = sampler.stop()
    sim.close()
    return row


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/unit/config keys (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    n = 512
    rate, el = oracle_rate(n, args.steps, warmup=args.warmup, threads=1)
    sample = (f"oracle (oracle/smaug_oracle.cpp, -O2, 1 thread) on Orszag-Tang {n}x{n}, same IC/params as the "
              f"workload, {args.steps} timed steps after {args.warmup} warm-up")
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "sample": f"orszag_tang_{n}", "cfl": 0.3, "hd": True, "rk_order": 4},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    import paper_1710_06423_b200 as pkg
    pkg.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    name = args.workload
    nx, ny, _ = WORKLOADS[name]
    w_np, bc, gamma, bg_np, (gx, gy) = make_state(name)
    w_host = torch.from_numpy(w_np).pin_memory()
    out_host = torch.empty_like(w_host).pin_memory()
    bg_dev = None if bg_np is None else torch.from_numpy(bg_np).to(dev)
    has_bg = bg_np is not None
    del w_np, bg_np
    sim = pkg.Smaug(nx, ny, gamma, bc, bg=bg_dev, device=dev, hd_on=0 if args.no_hd else 1, gx=gx, gy=gy,
                    rk_order=args.rk_order)
    del bg_dev
    sim.set_state(w_host)

    K, W = args.steps, args.warmup
    # ---- device-resident timing: W warm-up steps, then exactly K steps between CUDA events
    sim.step(W, 0.3)
    sim.set_kernel_timing(not args.no_kernel_timing)
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    sim.step(K, 0.3)
    e1.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - launches0
    stage_ms, stage_n = sim.kernel_timing()
    sim.set_kernel_timing(False)
    t_sim, dt_last = sim.time()

    # ---- end to end through the C ABI with HOST buffers: H2D set_state + K steps + D2H get_state
    barrier()
    t0 = time.perf_counter()
    sim.set_state(w_host)
    sim.step(K, 0.3)
    sim.get_state(out_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    finite = bool(torch.isfinite(out_host[:, ::97, ::89]).all())

    ms, e2e_ms = max_over_ranks([ms, e2e_s * 1e3], dev, world)

    if rank == 0:
        cells = float(nx) * ny
        value = replica_value(cells, K, world, ms)
        e2e = replica_value(cells, K, world, e2e_ms)
        peak, peak_src = peaks()
        info = sim.kernel_info()
        stages = {4: 4, 2: 2, 1: 1}[args.rk_order]
        bpcu = bytes_per_cell_update(has_bg, args.rk_order)
        per_launch_bytes = bpcu / stages * cells
        cap = ncu_capture(name + ("_nohd" if args.no_hd else "") + ("_rk%d" % args.rk_order if args.rk_order != 4 else ""))
        fp64_per_cell = cap.get("fp64_thread_inst_per_cell")
        avg_launch_ms = stage_ms / max(stage_n, 1)
        achieved = per_launch_bytes / (avg_launch_ms * 1e-3) / 1e9 if stage_n and avg_launch_ms > 0 else None
        state_bytes = 6 * 8 * cells
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "nx": nx, "ny": ny, "cfl": 0.3, "hd": not args.no_hd, "rk_order": args.rk_order,
                       "background": ("stratified, g = (%g, %g)" % (gx, gy) if gy or gx else "uniform") if has_bg else "zero", "parallelism": "replicas only" if world > 1 else "1 gpu",
                       "l2": "working set >> L2, no flush needed" if cells * 48 > 4e8 else
                             "working set comparable to L2 (126 MB): DRAM traffic is below algorithmic"},
            "hbm_gbs_algorithmic": value / world * bpcu / 1e9,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": (achieved / peak) if achieved else None,
                         "frac_of_nominal_8TBs": (achieved / 8000.0) if achieved else None, "traffic": cap.get("dram_bytes"),
                         "traffic_source": cap.get("capture"),
                         "traffic_bytes_per_cell_update": (cap["dram_bytes"] * stages / cells) if cap.get("dram_bytes") else None,
                         "algorithmic_bytes_per_cell_update": bpcu,
                         "peak_source": peak_src, "kernel": f"smaug::{sim.kernel_name()} (fused RK stage)",
                         "bytes_per_launch": per_launch_bytes, "avg_launch_ms": avg_launch_ms,
                         "launches_timed": stage_n, "stage_kernel_share_of_step": stage_ms / ms,
                         "note": None if stage_n else "--no-kernel-timing: steps replayed as CUDA graphs, no per-kernel events",
                         "launch": info},
            "fp64_pipe": ({"achieved": fp64_per_cell * cells / (avg_launch_ms * 1e-3) / 1e12,
                           "peak": N_SM * FP64_LANES_PER_SM * ((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6 / 1e12,
                           "unit": "T fp64-instr/s", "instr_per_cell_stage": fp64_per_cell,
                           "note": "secondary ceiling: fp64-pipe thread-instructions per cell and launch from the "
                                   "committed ncu capture (sm__inst_executed_pipe_fp64), x cells / measured duration"}
                          if stage_n and avg_launch_ms > 0 and fp64_per_cell else None),
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": state_bytes / K,
                    "d2h_bytes_per_step": state_bytes / K,
                    "note": "smaug_set_state(host) + smaug_step(K) + smaug_get_state(host), pinned host memory"},
            "gpu_launches": launches,
            "clocks": clocks,
            "sim": {"t": t_sim, "last_dt": dt_last, "finite": finite},
        }
        if line["fp64_pipe"]:
            fp = line["fp64_pipe"]
            fp["frac"] = fp["achieved"] / fp["peak"]
            # the two floors of one launch: the kernel can be no faster than the higher one
            rf = line["roofline"]
            rf["hbm_floor_ms"] = per_launch_bytes / (peak * 1e9) * 1e3
            rf["fp64_floor_ms"] = fp64_per_cell * cells / (fp["peak"] * 1e12) * 1e3
            if rf["fp64_floor_ms"] > rf["hbm_floor_ms"]:
                rf["bound"] = "alu"
                rf["bound_note"] = ("the fp64 pipe sets the higher floor of this kernel (fp64_floor_ms > hbm_floor_ms), so it "
                                    "is ALU-bound in principle; achieved / peak / frac stay the HBM figures north_star asks "
                                    "for, the ALU figures are in `fp64_pipe`; frac can reach at most hbm_floor_ms / fp64_floor_ms")
                rf["max_hbm_frac_at_full_fp64_pipe"] = rf["hbm_floor_ms"] / rf["fp64_floor_ms"]
        if not args.no_cpu_baseline and world == 1:
            n_s, steps_s = 1000, 6
            kind = WORKLOADS[name][2] if has_bg else "ot"
            rate, el = oracle_rate(n_s, steps_s, threads=1, kind=kind)
            line["cpu_baseline"] = {
                "value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                "sample": f"{ {'strat': 'stratified atmosphere', 'otbg': 'Orszag-Tang on a uniform background'}.get(kind, 'Orszag-Tang')} {n_s}x{n_s} (same IC and "
                          f"parameters), {steps_s} steps, {el:.1f} s, "
                          f"1 of {os.cpu_count()} host cores"}
        if args.rows and world == 1:
            sim.close()
            rows = []
            for wl, hd, decomp in ROWS:
                try:
                    st = (w_host, bc, gamma, None, (0.0, 0.0)) if wl == name and not has_bg else None
                    rows.append(compact_row(pkg, wl, hd=hd, decomp=decomp, device=local, state=st))
                except Exception as e:  # noqa: BLE001
                    rows.append({"workload": wl, "hd": hd, "error": repr(e)})
            line["rows"] = rows
        print(json.dumps(line), flush=True)
    sim.close()
    if world > 1:
        dist.destroy_process_group()


def run_3d(args):
    """A 3-D workload: same JSON line; a step = dt + 4 x {ghost fill, derived quantities, kappa /
    interface fluxes, cell-centred fluxes, assembly + RK combine + reduction}.  The roofline
    entry is taken over the whole stage (its kernels together) against what a fully fused stage must move:
    8 fields x 8 B x (4 reads with halo + 4 writes + 2 x w^n + accumulator written once and read once) = 768 B per
    cell-update, 192 B per cell and stage."""
    import torch
    import paper_1710_06423_b200 as pkg
    pkg.lib()
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("bench.py: the 3-D rows are single-GPU rows")
    torch.cuda.set_device(0)
    name = args.workload
    n = WORKLOADS[name][0]
    w_np, bc, gamma = si.orszag_tang_3d(n)
    w_host = torch.from_numpy(w_np).pin_memory()
    out_host = torch.empty_like(w_host).pin_memory()
    del w_np
    sim = pkg.Smaug3D(n, n, n, gamma, bc, hd_on=0 if args.no_hd else 1, rk_order=args.rk_order)
    sim.set_state(w_host)
    K, W = args.steps, args.warmup
    sim.step(W, 0.3)
    sim.set_kernel_timing(True)
    sampler = ClockSampler(0)
    launches0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    sim.step(K, 0.3)
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - launches0
    kinds = sim.kernel_timing()
    sim.set_kernel_timing(False)
    t_sim, dt_last = sim.time()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    sim.set_state(w_host)
    sim.step(K, 0.3)
    sim.get_state(out_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    finite = bool(torch.isfinite(out_host[:, ::7, ::5, ::3]).all())
    cells = float(n) ** 3
    stages = {4: 4, 2: 2}[args.rk_order]
    bpcu = {4: 768.0, 2: 320.0}[args.rk_order]
    peak, peak_src = peaks()
    stage_ms = sum(v[0] for v in kinds.values()) / (K * stages)
    achieved = bpcu / stages * cells / (stage_ms * 1e-3) / 1e9
    top = max(kinds, key=lambda k: kinds[k][0])
    cap = ncu_capture(name + ("_nohd" if args.no_hd else "") + ("_rk%d" % args.rk_order if args.rk_order != 4 else ""))
    line = {
        "metric": METRIC, "value": cells * K / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": name, "nx": n, "ny": n, "nz": n, "fields": 8, "cfl": 0.3, "hd": not args.no_hd,
                   "rk_order": args.rk_order, "background": "zero", "parallelism": "1 gpu",
                   "l2": "working set >> L2, no flush needed" if cells * 64 > 4e8 else "working set comparable to L2 (126 MB)"},
        "hbm_gbs_algorithmic": cells * K / (ms * 1e-3) * bpcu / 1e9,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "frac_of_nominal_8TBs": achieved / 8000.0, "traffic": cap.get("dram_bytes"),
                     "traffic_source": cap.get("capture"), "peak_source": peak_src,
                     "traffic_over_algorithmic": (cap["dram_bytes"] / (bpcu / stages * cells)) if cap.get("dram_bytes") else None,
                     "achieved_note": "`achieved` divides the bytes a fully fused stage must move by the measured time; the "
                                      "kernels as built move `traffic` (ncu, per stage), several times more",
                     "kernel": "smaug3 RK stage (ghost3, kappa3, stage3); "
                               f"largest share: {top}",
                     "bytes_per_launch": bpcu / stages * cells, "avg_launch_ms": stage_ms,
                     "launches_timed": int(sum(v[1] for v in kinds.values())),
                     "stage_kernel_share_of_step": sum(v[0] for v in kinds.values()) / ms,
                     "ms_per_stage_by_kind": {k: v[0] / (K * stages) for k, v in kinds.items()}},
        "e2e": {"value": cells * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 64 * cells / K, "d2h_bytes_per_step": 64 * cells / K,
                "note": "smaug3_set_state(host) + smaug3_step(K) + smaug3_get_state(host), pinned host memory"},
        "gpu_launches": launches, "clocks": clocks, "sim": {"t": t_sim, "last_dt": dt_last, "finite": finite},
    }
    if not args.no_cpu_baseline:
        import oracle
        ns, steps_s = 64, 3
        w, bc, gamma = si.orszag_tang_3d(ns)
        o = oracle.Oracle3D(ns, ns, ns, gamma, bc, hd_on=0 if args.no_hd else 1, rk_order=args.rk_order)
        o.set_state(w)
        t0 = time.perf_counter()
        o.step(steps_s, 0.3)
        el = time.perf_counter() - t0
        o.close()
        line["cpu_baseline"] = {"value": ns ** 3 * steps_s / el, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"3-D oracle on the same vortex at {ns}^3, {steps_s} steps, {el:.1f} s, 1 of {os.cpu_count()} host cores"}
    print(json.dumps(line), flush=True)
    sim.close()


def run_decomp(args):
    """--decomp PXxPY: the decomposed run of the workload on one device beside the unsplit run of the same steps
    (the decomposition's own cost: exchange kernels, barriers between the members' streams, smaller launches)."""
    import torch
    import paper_1710_06423_b200 as pkg
    pkg.lib()
    px, py = (int(v) for v in args.decomp.lower().split("x"))
    name = args.workload
    nx, ny, _ = WORKLOADS[name]
    w_np, bc, gamma, bg_np, (gx, gy) = make_state(name)
    w_host = torch.from_numpy(w_np).pin_memory()
    bg = None if bg_np is None else torch.from_numpy(bg_np).cuda()
    params = dict(hd_on=0 if args.no_hd else 1, gx=gx, gy=gy, rk_order=args.rk_order)
    K, W = args.steps, args.warmup

    def timed(sim):
        sim.set_state(w_host)
        sim.step(W, 0.3)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        sim.step(K, 0.3)                      # synchronises before returning
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) * 1e3

    one = pkg.Smaug(nx, ny, gamma, bc, bg=bg, **params)
    ms_one = timed(one)
    t_one = one.time()
    one.close()
    devices = [int(v) for v in args.devices.split(",")] if args.devices else None
    if devices is not None and len(devices) != px * py:
        raise SystemExit(f"bench.py: --devices needs {px * py} entries (member b * px + a runs on devices[b * px + a])")
    grp = pkg.SmaugGroup(px, py, nx, ny, gamma, bc, bg=bg, devices=devices, **params)
    ms_grp = timed(grp)
    t_grp = grp.time()
    n_stage, n_exch = grp.launch_count()
    # the paper's three terms and tau, from CUDA events on the members' streams over K more steps
    grp.set_timing(True)
    t0 = time.perf_counter()
    grp.step(K, 0.3)
    ms_tau = (time.perf_counter() - t0) * 1e3
    tau = grp.tau()
    grp.set_timing(False)
    grp.close()
    cells = float(nx) * ny
    line = {
        "metric": METRIC, "value": cells * K / (ms_grp * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W,
        "ms_per_step": ms_grp / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": name, "nx": nx, "ny": ny, "cfl": 0.3, "hd": not args.no_hd, "rk_order": args.rk_order,
                   "decomposition": f"{px}x{py} members on " + ("one device" if devices is None or len(set(devices)) == 1
                                                                 else f"devices {devices} (one process, peer access; EXPERIMENTAL path)")
                                    + " (smaug_group_*)",
                   "timing": "host wall clock around the synchronising step call, after a device synchronise"},
        "unsplit": {"value": cells * K / (ms_one * 1e-3), "ms_per_step": ms_one / K},
        "decomposition_cost": ms_grp / ms_one - 1.0,
        "bit_identical_time": list(t_grp) == list(t_one),
        "gpu_launches": n_stage + n_exch, "exchange_launches": n_exch,
        "tau": {"T_comp_ms_per_step": tau["t_comp"] / K, "T_comm_ms_per_step": tau["t_comm"] / K,
                "T_idle_ms_per_step": tau["t_idle"] / K, "tau": tau["tau"], "ms_per_step_while_timed": ms_tau / K,
                "definition": "PAPER.md:138-144: T = T_comp + T_comm + T_idle, tau = ln(T_comp / (T_comm + T_idle)); mean over "
                              "the members; T_comm = halo-pull kernels, T_comp = stage kernels, T_idle = a member's wait "
                              "in the inter-member barriers after its own work",
                "caveat": "all members share ONE device here: a member's intervals include the time its kernels wait for "
                          "or share the SMs with the other members' kernels, so tau describes the lockstep schedule on "
                          "one GPU, not a link; across GPUs the same call measures the paper's quantity"},
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="orszag_tang_8000", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-timing", action="store_true",
                    help="no CUDA events around the stage kernels (roofline = null); smaug_step then replays CUDA "
                         "graphs of whole steps, which is what a user gets -- matters on launch-bound small grids")
    ap.add_argument("--rk-order", type=int, default=4, choices=[4, 2],
                    help="4: classical RK4 (PAPER.md:45, the default); 2: midpoint rule (SURVEY 8(f) NEXT-4 extra row)")
    ap.add_argument("--decomp", default=None, metavar="PXxPY",
                    help="extra row (SURVEY 8(f) NEXT-1): run the workload as a PX x PY decomposition group on ONE device "
                         "(halo pull through peer pointers, shared reduction, lockstep stages) and report its rate")
    ap.add_argument("--devices", default=None, metavar="D0,D1,...",
                    help="with --decomp: run ONE group across these visible devices in this single process (member "
                         "b * PX + a on the (b * PX + a)-th entry; the devices need peer access).  Default: all members on "
                         "the current device.  The several-GPU path is experimental: it has not run on hardware yet")
    ap.add_argument("--no-rows", action="store_true",
                    help="leave out the `rows` list (the other BASELINE configs, HD off, background, 3-D and 2x2-group "
                         "rows, each timed for >= 0.5 s) that the default single-GPU invocation adds to its line")
    ap.add_argument("--no-hd", action="store_true",
                    help="hyperdiffusion off (the 'Without HD' column of the paper's Table 1); extra row, not the default")
    args = ap.parse_args()
    # the extra rows ride on the default headline invocation only (one GPU, default workload and scheme)
    args.rows = (not args.no_rows and args.impl == "ours" and args.gpus == 1 and args.workload == "orszag_tang_8000"
                 and not args.no_hd and args.rk_order == 4 and not args.decomp and not args.no_kernel_timing)
    if args.impl == "reference":
        run_reference(args)
    elif WORKLOADS[args.workload][2] == "ot3d":
        run_3d(args)
    elif args.decomp:
        run_decomp(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
