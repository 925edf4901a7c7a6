#!/usr/bin/env python
"""bench.py — grind time of the MFC hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4|5|3|2|1] [--impl ours|reference] [--no-also]
    python bench.py --probe-fp64        (the FP64 DFMA probe alone, with its clock record: profiles/fp64_probe.json)

A "step" is one pass of the whole hot path over the whole grid: the CFL reduction (mfc_cfl_dt) followed by
one SSP-RK3 step = 3 x (x/y/z sweeps: cons->prim, WENO5-JS, HLLC, flux divergence, alpha div(u) source)
+ 3 x (RK stage + clamp), through the C ABI (mfc_advance).  Metric: grind time = time / (RHS evaluations x
cells x equations) in ns, RHS evaluations = 3 per step.

Default workload: BASELINE.json configs[3] (3D periodic two-fluid mixing, 256^3, 8 equations — the shape of
the paper's Table-1 benchmark case), seeded synthetic input (mfc_workloads).  The state arrays
(1.07 GB each, 4 of them touched per step) are far larger than the 126 MB L2, so no L2 flush is needed.

With no --config (config 4, N = 1) the line also carries, under "also", configs 5 (512^3, 10 equations, 5 steps) and 3
(1024^2, 50 steps) and config 4 with the paper's default mapped weights (10 steps), each with its own roofline and clock record.  "roofline" names the dominant kernel and the roof that
binds it (north_star: "the slower of the two"): the floor times of that launch for the FP64 ALUs (algorithmic
flops / derived peak) and for HBM (ALGORITHMIC bytes of the RK stage / measured copy bandwidth) are both printed, `frac` is
against the larger; `design_hbm_frac` is the separate statement about the three-sweep design (its compulsory bytes over the
copy bandwidth); `traffic` / `traffic_ratio` come from the committed ncu capture (stale captures are refused);
`frac_whole_step` is the larger of the two algorithmic floors of the whole step over the step time.  `also_summary`, near the
front of the line, has one compact entry for configs 5, 3, 1, 2 and config 4 with mapped weights.

N > 1 (torchrun): the path runs on one GPU (north_star); ranks are independent replicas ("replicas only",
DESIGN.md §9) — no data-path collective; time is the max over ranks, value the whole-job aggregate.

--impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a bounded replica of the
same workload; rank 0 only.
"""
import argparse
import dataclasses
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "rhs_grind_time"
UNIT = "ns/cell/eqn/rhs_eval"

# Algorithmic flops per cell per RHS evaluation of the plain definition (add/sub, mul, div, sqrt = 1 flop
# each), counted by the operation-counting instantiation of the oracle and extrapolated to n -> infinity
# (tests/test_host_logic.py re-derives them).  Key: BASELINE.json config index.
ALG_FLOPS_PER_CELL_RHS = {1: 538.0, 2: 779.0, 3: 1798.0, 4: 3057.0, 5: 3780.0}
# the same count with the other nonlinear weights (--weno m: mapped; --weno z: WENO-Z)
ALG_FLOPS_PER_CELL_RHS_BY_WENO = {"js": ALG_FLOPS_PER_CELL_RHS,
                                  "m": {1: 914.0, 2: 1343.0, 3: 3114.0, 4: 5313.0, 5: 6600.0},
                                  "z": {1: 547.0, 2: 797.0, 3: 1844.6, 4: 3128.9, 5: 3867.6}}
# FP64 peak "derived from unit counts and clocks": 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz.
FP64_PEAK_TFLOPS_DERIVED = 148 * 64 * 2 * 1.965e9 / 1e12
# The measured counterpart is taken live in every run by mfc_measure_fp64 (DFMA chains, all SMs); a capture with its clock
# record is kept in profiles/fp64_probe.json (made by `python bench.py --probe-fp64`).
# One replica size per configuration for BOTH oracle timings (cpu_baseline and --impl reference); None = the configuration itself
ORACLE_REPLICA_N = {1: None, 2: None, 3: 512, 4: 128, 5: 96}


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device):
        self.device = device
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.device), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm_sorted = sorted(sm)
        return {"sm_mhz": sm_sorted[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def reduce_max_ms(ms, world):
    """max over ranks of a device-timed duration (every multi-GPU number is the slowest rank's)."""
    if world == 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device="cuda" if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def grind_ns(ms, steps, cells, neq, replicas=1):
    """ns per cell per equation per RHS evaluation; 3 RHS evaluations per RK3 step; whole job = all replicas."""
    return ms * 1e6 / (3.0 * steps * cells * neq * replicas)


def sweep_alg_bytes_per_cell(kernel, neq, ndim):
    """compulsory HBM bytes per cell of one launch of a sweep kernel inside an RK3 step of the three-sweep design
    (DESIGN.md §6, §8): the first sweep (x) reads q and writes the partial L; a middle sweep reads q and L and writes L; the
    last sweep of a stage (y in 2-D, z in 3-D; x in 1-D) also applies the RK stage: it reads q, L and — in stages 2 and 3,
    where q^n is not the swept state — q^n, and writes the new stage state: (24 + 32 + 32)/3 per equation on average."""
    last = {1: "sweep_x", 2: "sweep_y", 3: "sweep_z"}[ndim]
    if kernel == last:
        return ((16 if ndim == 1 else 24) + 8 * 2.0 / 3.0) * neq
    return (16 if kernel == "sweep_x" else 24) * neq


def stage_alg_bytes_per_cell(neq):
    """ALGORITHMIC bytes per cell of one RK stage whatever the kernel design — read the swept state once,
    read q^n too where it is another array (stages 2, 3), write the new stage state once: (16 + 24 + 24)/3 per equation on
    the average of the three stages.  A launch of the dominant sweep kernel (one per stage) is charged ALL of it: the HBM
    floor this gives is the one a fully fused stage kernel would have, the most any design could ask of that launch."""
    return (16 + 24 + 24) / 3.0 * neq


def kernel_sources_sha256():
    """hash of the CUDA sources: profiles/traffic.json records the one its ncu capture was made with"""
    import hashlib
    h = hashlib.sha256()
    for fn in ("mfc_b200.cu", "mfc_device.cuh"):
        with open(os.path.join(ROOT, "paper_2503_07953_b200", "csrc", fn), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def run_reference(args, rank):
    """The oracle, as it stands, on the host cores: each step = one RK3 step (no CFL reduction: the oracle's
    cfl_dt is serial) on a bounded replica of the workload."""
    if rank != 0:
        return
    import mfc_workloads as W
    from oracle import oracle as O
    n_ref = ORACLE_REPLICA_N[args.config]
    case = dataclasses.replace(W.config(args.config, n=n_ref), weno=args.weno, model=args.model, eta=args.eta)
    q = W.initial_state(case)
    orc = O.Oracle(case)
    dt = orc.cfl_dt(q, case.cfl)
    for _ in range(args.warmup):
        orc.rk3_step(q, dt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.rk3_step(q, dt)
    sec = time.perf_counter() - t0
    val = grind_ns(sec * 1e3, args.steps, case.cells, case.neq)
    cores = O.num_threads()
    sample = f"{args.steps} RK3 steps on a {'x'.join(str(v) for v in case.n[:case.ndim])} replica of config {args.config}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3 / max(args.steps, 1), "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": case.name, "cells": case.cells, "neq": case.neq, "note": "CPU oracle on a bounded replica"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def cpu_baseline(config_index, weno="js", model="allaire", eta=0.0, budget_s=20.0):
    import mfc_workloads as W
    from oracle import oracle as O
    n_ref = ORACLE_REPLICA_N[config_index]
    case = dataclasses.replace(W.config(config_index, n=n_ref), weno=weno, model=model, eta=eta)
    q = W.initial_state(case)
    orc = O.Oracle(case)
    dt = orc.cfl_dt(q, case.cfl)
    t0 = time.perf_counter()
    steps = 0
    while steps < 2 or (time.perf_counter() - t0 < budget_s / 2 and steps < 50):  # about 10 s of host work
        orc.rk3_step(q, dt)
        steps += 1
        if time.perf_counter() - t0 > budget_s:
            break
    sec = time.perf_counter() - t0
    return {"value": grind_ns(sec * 1e3, steps, case.cells, case.neq), "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{steps} RK3 steps ({3 * steps} RHS evaluations) on a {'x'.join(str(v) for v in case.n[:case.ndim])} "
                      f"replica of config {config_index} ({sec:.1f} s of host time)"}


def median(xs):
    xs = sorted(xs)
    return xs[len(xs) // 2] if len(xs) % 2 else 0.5 * (xs[len(xs) // 2 - 1] + xs[len(xs) // 2])


def probe_fp64(M, local_rank):
    """live DFMA probe with the clock record of the probe itself"""
    sampler = ClockSampler(local_rank)
    sampler.start()
    try:
        best = (0.0, 0.0)
        for _ in range(3):  # ~60 ms of FP64 load per call: three calls so that nvidia-smi (100 ms period) sees the load
            r = M.measure_fp64(local_rank)
            best = (max(best[0], r[0]), max(best[1], r[1]))
    except Exception as exc:  # a library without the probe
        sampler.stop()
        return None, None, {"error": str(exc)}
    return best[0], best[1], sampler.stop()


def measure(args, config_index, steps, rank, local_rank, world, with_e2e):
    """Times `steps` steps of one configuration (device-resident), the per-kernel profile and the roofline figures.
    Returns the dict of that configuration (value, ms_per_step, clocks, roofline, ...)."""
    import torch
    import mfc_workloads as W
    import paper_2503_07953_b200 as M

    case = dataclasses.replace(W.config(config_index, n=args.n if config_index == args.config else None),
                               weno=args.weno, model=args.model, eta=args.eta)
    q0 = W.initial_state(case)
    slab = None
    if args.decomp == "slab":
        from paper_2503_07953_b200 import slab as S
        d = case.ndim - 1
        if case.ndim < 2 or case.bc_lo[d] != W.BC_PERIODIC:
            raise SystemExit("bench.py --decomp slab: needs a 2-D/3-D configuration periodic in its last direction (config 4)")
        n_glob = list(case.n)
        n_glob[d] *= world                      # the rank's block repeated `world` times along the last direction
        slab = S.Slab(dataclasses.replace(case, n=tuple(n_glob)), rank, world, local_rank,
                      torch.distributed if world > 1 else None)
        g = slab.grid
        advance = lambda q, cfl, n: slab.advance(q, cfl, n)
    else:
        g = M.Grid.from_case(case, device=local_rank)
        advance = lambda q, cfl, n: g.advance(q, cfl, n)
    qd = torch.from_numpy(q0).cuda()
    cells, neq = case.cells, case.neq

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            torch.distributed.barrier()
            torch.cuda.synchronize()

    # ---- device-resident timing: the headline value
    for _ in range(args.warmup):
        advance(qd, case.cfl, 1)
    g.check()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    bad_reasons = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    for attempt in (1, 2):  # a run that saw a thermal / hardware slowdown is re-measured once (sw_power_cap is kept and noted)
        sampler = ClockSampler(local_rank)
        l0 = g.launch_count()
        barrier()
        sampler.start()
        ev0.record()
        advance(qd, case.cfl, steps)
        ev1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        barrier()
        launches = g.launch_count() - l0
        ms = reduce_max_ms(ev0.elapsed_time(ev1), world)
        g.check()
        clocks["attempt"] = attempt
        if not (bad_reasons & set(clocks.get("reasons") or [])):
            break
    value = grind_ns(ms, steps, cells, neq, world)

    # ---- SURVEY 8(d) "median of >= 10 repetitions": (b) single steps, each bracketed by its own events
    reps = []
    for _ in range(10):
        ev0.record()
        advance(qd, case.cfl, 1)
        ev1.record()
        torch.cuda.synchronize()
        reps.append(ev0.elapsed_time(ev1))
    step_median_ms = reduce_max_ms(median(reps), world)

    # ---- (a) mfc_rhs alone (SURVEY 8(d) metric (i)): x, y, z sweeps without the RK stage, rhs written to its own array
    rhs_only = None
    if slab is None:
        rd = torch.empty_like(qd)
        for _ in range(3):
            g.rhs(qd, rd)
        torch.cuda.synchronize()
        rr = []
        for _ in range(11):
            ev0.record()
            g.rhs(qd, rd)
            ev1.record()
            torch.cuda.synchronize()
            rr.append(ev0.elapsed_time(ev1))
        r_ms = reduce_max_ms(median(rr), world)
        rhs_only = {"value": r_ms * 1e6 / (cells * neq), "unit": "ns/cell/eqn/rhs_eval", "ms_per_rhs": r_ms, "evals": len(rr),
                    "statistic": "median", "call": "mfc_rhs"}
        del rd

    # ---- per-kernel device times (CUDA events around every launch, on the launching stream) for the roofline
    g.set_profiling(True)
    advance(qd, case.cfl, steps)
    prof = g.get_profile()
    g.set_profiling(False)
    tot_ms = sum(v[0] for v in prof.values())
    kern = {k: {"ms_per_launch": v[0] / v[1], "launches_per_step": v[1] / steps, "share_of_step": v[0] / tot_ms}
            for k, v in prof.items() if v[1]}
    sweeps = [k for k in ("sweep_x", "sweep_y", "sweep_z") if k in kern]
    dom = max(sweeps, key=lambda k: kern[k]["ms_per_launch"] * kern[k]["launches_per_step"])
    dur_s = kern[dom]["ms_per_launch"] * 1e-3
    flops_rhs = ALG_FLOPS_PER_CELL_RHS_BY_WENO[args.weno][config_index] * cells
    flops_launch = flops_rhs / case.ndim
    bytes_launch = sweep_alg_bytes_per_cell(dom, neq, case.ndim) * cells
    hbm_peak, hbm_src = measured_peaks()
    # dram bytes per launch: NOT measured in this run (the counters need ncu) but read from the committed ncu --set full
    # capture; the file records the hash of the CUDA sources it was captured with, and a capture of other sources is
    # reported as stale instead of being passed off as this build's
    traffic, traffic_all, traffic_note = None, {}, "no profiles/traffic.json"
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            tj = json.load(f)
        fresh = tj.get("kernel_sources_sha256") == kernel_sources_sha256()
        traffic_note = ("committed ncu --set full capture, " + str(tj.get("source")) +
                        ("; captured with the CUDA sources of this build" if fresh else
                         "; STALE: captured with other CUDA sources than this build's (kernel_sources_sha256 differs)"))
        if fresh:
            traffic_all = tj.get(f"config{config_index}", {})
            traffic = traffic_all.get(dom)
    dfma_tf, dfma3_tf, probe_clocks = probe_fp64(M, local_rank)
    alu = {"achieved": flops_launch / dur_s / 1e12, "peak": FP64_PEAK_TFLOPS_DERIVED, "unit": "TFLOP/s",
           "frac": flops_launch / dur_s / 1e12 / FP64_PEAK_TFLOPS_DERIVED,
           "peak_source": "derived: 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md §8)",
           "measured_dfma_tflops": dfma_tf, "measured_dfma_three_register_operands_tflops": dfma3_tf,
           "frac_of_measured_dfma_peak": (flops_launch / dur_s / 1e12 / dfma_tf) if dfma_tf else None,
           "probe_clocks": probe_clocks, "alg_flops_per_launch": flops_launch}
    hbm = {"achieved": bytes_launch / dur_s / 1e9, "peak": hbm_peak, "unit": "GB/s", "frac": bytes_launch / dur_s / 1e9 / hbm_peak,
           "peak_source": hbm_src + " (MEASURED_PEAKS.json hbm_gbs)" if hbm_src == "measured" else "fallback of B200_PROFILING.md",
           "alg_bytes_per_launch": bytes_launch,
           "bytes_are": "compulsory bytes of this kernel in the three-sweep design (q, partial L, q^n read; new state written)"}
    # SURVEY.md §8(d) / north_star "the roofline taken as the slower of the two": both floors from ALGORITHMIC work — the flops
    # of this launch, and the bytes any design must move for the stage (stage_alg_bytes_per_cell) — the larger floor binds.
    # The compulsory bytes of the three-sweep DESIGN (hbm above) are a statement about this design, kept as design_hbm_frac.
    alg_bytes_launch = stage_alg_bytes_per_cell(neq) * cells
    hbm_alg = {"achieved": alg_bytes_launch / dur_s / 1e9, "peak": hbm_peak, "unit": "GB/s",
               "frac": alg_bytes_launch / dur_s / 1e9 / hbm_peak, "alg_bytes_per_launch": alg_bytes_launch,
               "bytes_are": "algorithmic bytes of one RK stage (SURVEY 8(d)): (16 + 24 + 24)/3 x neq per cell"}
    t_alu, t_hbm = flops_launch / (FP64_PEAK_TFLOPS_DERIVED * 1e12), alg_bytes_launch / (hbm_peak * 1e9)
    t_hbm_design = bytes_launch / (hbm_peak * 1e9)
    bound = "alu" if t_alu >= t_hbm else "hbm"
    sel = alu if bound == "alu" else hbm_alg
    step_s = ms * 1e-3 / steps
    # whole step: algorithmic flops of 3 RHS evaluations / algorithmic bytes of SURVEY 8(d) (RHS: 16 neq per cell; an RK stage
    # re-reads q^n in stages 2, 3 and the CFL reduction reads q once: (3*16 + 2*8 + 8) neq per cell per step) over the step time
    step_bytes = (3 * 16 + 2 * 8 + 8) * neq * cells
    whole = {"alu_frac": 3 * flops_rhs / step_s / 1e12 / FP64_PEAK_TFLOPS_DERIVED, "alu_tflops": 3 * flops_rhs / step_s / 1e12,
             "hbm_frac_algorithmic_bytes": step_bytes / step_s / 1e9 / hbm_peak, "alg_bytes_per_step": step_bytes,
             "ms_per_step": step_s * 1e3}
    # measured DRAM bytes of a whole step over its algorithmic bytes (wasted traffic), when the capture covers every sweep
    if all(k in traffic_all for k in sweeps):
        step_traffic = sum(traffic_all[k] * kern[k]["launches_per_step"] for k in sweeps) + traffic_all.get("cfl", 8.0 * neq * cells)
        whole["traffic_bytes_per_step"] = step_traffic
        whole["traffic_ratio"] = step_traffic / step_bytes
    whole["frac"] = max(whole["alu_frac"], whole["hbm_frac_algorithmic_bytes"])
    roofline = {"kernel": dom, "bound": bound, "achieved": sel["achieved"], "peak": sel["peak"], "unit": sel["unit"],
                "frac": sel["frac"], "traffic": traffic,
                "traffic_ratio": (traffic / alg_bytes_launch) if traffic else None, "traffic_source": traffic_note,
                "ms_per_launch": dur_s * 1e3,
                "denominator": ("alu: derived FP64 peak 37.2 TFLOP/s" if bound == "alu" else "hbm: measured copy bandwidth") +
                               "; floor times of this launch from algorithmic work: alu %.3f ms, hbm %.3f ms (three-sweep design's "
                               "compulsory bytes: %.3f ms)" % (t_alu * 1e3, t_hbm * 1e3, t_hbm_design * 1e3),
                "design_hbm_frac": hbm["frac"], "alu": alu, "hbm_algorithmic": hbm_alg, "hbm_design": hbm,
                "frac_whole_step": whole["frac"], "whole_step": whole, "kernels": kern}

    # ---- end to end through the C ABI with HOST buffers: H2D of the state, the step, D2H of the state, every step
    e2e = None
    if with_e2e:
        qh = torch.from_numpy(q0.copy()).pin_memory()
        if slab is None:
            step_host = lambda: g.advance_host(qh, case.cfl, 1)  # syncs inside
            call = "mfc_advance_host(q_host pinned, cfl, 1) per step"
        else:
            def step_host():  # the slab path has no host-buffer entry point: the copies are made here
                qd.copy_(qh, non_blocking=True)
                slab.advance(qd, case.cfl, 1)
                qh.copy_(qd, non_blocking=True)
                torch.cuda.synchronize()
            call = "pinned H2D copy + Slab.advance(q, cfl, 1) + D2H copy per step"
        for _ in range(2):
            step_host()
        n_e2e = max(2, min(steps, 10))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            step_host()
        sec = time.perf_counter() - t0
        e_ms = reduce_max_ms(sec * 1e3, world)
        e2e = {"value": grind_ns(e_ms, n_e2e, cells, neq, world), "unit": UNIT, "h2d_bytes_per_step": 8 * neq * cells,
               "d2h_bytes_per_step": 8 * neq * cells, "steps": n_e2e, "ms_per_step": e_ms / n_e2e,
               "call": call}
        del qh
    g.close()
    del qd
    torch.cuda.empty_cache()
    return {
        "value": value, "ms_per_step": ms / steps, "ms_per_step_median_of_10_single_steps": step_median_ms, "steps": steps,
        "config": {"workload": case.name, "grid": list(case.n[:case.ndim]), "cells": cells, "neq": neq, "nfluids": case.nfluids,
                   "weno": {"js": "WENO5-JS", "m": "WENO5-M (mapped)", "z": "WENO5-Z"}[args.weno], "model": args.model, "eta": args.eta,
                   "rhs_evals_per_step": 3,
                   "parallelism": ("slabs along the last direction, %d x 3-layer halo exchanges per step" % (3 * 2) if slab is not None
                                   else "replicas only" if world > 1 else "single GPU"),
                   "l2": "inputs larger than L2 (state array %.0f MB vs 126 MB L2)" % (8e-6 * neq * cells) if 8 * neq * cells > 3e8
                   else "working set fits L2: latency/L2-bound configuration, roofline target does not apply"},
        "cell_updates_per_s": cells * world * steps / (ms * 1e-3),
        "clocks": clocks, "gpu_launches": launches, "e2e": e2e, "rhs_only": rhs_only, "roofline": roofline,
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)  # BASELINE.json config 4: "50 RK3 steps"
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--n", type=int, default=None, help="override cells per direction (tests only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--weno", default="js", choices=["js", "m", "z"],
                    help="nonlinear weights: js = BASELINE.json's WENO5-JS (default), m = mapped (the paper's default), z = WENO-Z")
    ap.add_argument("--model", default="allaire", choices=["allaire", "kapila"], help="volume-fraction equation (kapila: two fluids)")
    ap.add_argument("--eta", type=float, default=0.0, help="uniform shear viscosity (0: inviscid, BASELINE.json)")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default, DESIGN.md §9) or one periodic domain of N stacked slabs "
                         "exchanging 3-layer halos over NCCL (weak scaling: every rank owns one configuration-sized slab)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="headline configuration only (default: config 4 plus, at N = 1, "
                    "configs 5 and 3 under \"also\")")
    ap.add_argument("--probe-fp64", action="store_true", help="only the FP64 DFMA probe with its clock record (profiles/fp64_probe.json)")
    args = ap.parse_args()
    rank, local_rank, world = env_int("RANK", 0), env_int("LOCAL_RANK", 0), env_int("WORLD_SIZE", 1)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: at least 3 warm-up steps

    if args.impl == "reference":
        run_reference(args, rank)
        return 0

    import torch
    import paper_2503_07953_b200 as M

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if args.probe_fp64:
        out = []
        for _ in range(3):
            dfma, dfma3, clocks = probe_fp64(M, local_rank)
            out.append({"dfma_tflops": dfma, "dfma_three_register_operands_tflops": dfma3, "clocks_during_probe": clocks})
        print(json.dumps({"command": "python bench.py --probe-fp64", "gpu": torch.cuda.get_device_name(local_rank),
                          "derived_peak_tflops": FP64_PEAK_TFLOPS_DERIVED,
                          "what": "mfc_measure_fp64: register-resident DFMA chains on all SMs, 8 chains per thread, 16 warps per SM; "
                                  "x = fma(x, a, b) with loop-invariant a, b / fma of three distinct changing registers",
                          "runs": out}, indent=1))
        return 0
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    head = measure(args, args.config, args.steps, rank, local_rank, world, with_e2e=not args.no_e2e)
    out = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": head["ms_per_step"], "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
    }
    out["also_summary"] = None   # filled below; sits near the front of the line so that a truncated tail does not lose it
    for k in ("config", "cell_updates_per_s", "clocks", "gpu_launches", "e2e", "rhs_only", "roofline",
              "ms_per_step_median_of_10_single_steps"):
        out[k] = head[k]

    def summary(r):
        return {"workload": r["config"]["workload"], "weno": r["config"]["weno"], "steps": r["steps"], "ms_per_step": r["ms_per_step"],
                "value": r["value"], "kernel": r["roofline"]["kernel"], "bound": r["roofline"]["bound"], "frac": r["roofline"]["frac"],
                "frac_whole_step": r["roofline"]["frac_whole_step"], "sm_mhz": r["clocks"].get("sm_mhz"),
                "reasons": r["clocks"].get("reasons"), "gpu_launches": r["gpu_launches"]}
    out["paper_context"] = "PAPER.md:720-726 Table 1 (other hardware, whole step): GH200 0.32, H100 SXM 0.38, A100 0.62 ns"
    # the other two configurations the target names ("the 3D configs") and the full-size 2-D one, each with its own roofline
    # and clock record: config 5 (512^3, 10 equations, the largest single-GPU workload) and config 3 (1024^2)
    if args.config == 4 and world == 1 and not args.no_also and args.n is None and args.decomp == "replicas":
        also, summ = {}, []
        for idx, st in ((5, 5), (3, 50), (1, 200), (2, 200)):
            try:
                r = measure(args, idx, st, rank, local_rank, world, with_e2e=False)
                summ.append(summary(r))
                also[r["config"]["workload"]] = {k: r[k] for k in (
                    "value", "ms_per_step", "ms_per_step_median_of_10_single_steps", "steps", "config", "cell_updates_per_s",
                    "clocks", "gpu_launches", "rhs_only", "roofline")}
            except Exception as exc:  # e.g. not enough host or device memory for 512^3
                also[str(idx)] = {"error": repr(exc)}
        if args.weno == "js":  # the headline configuration with the paper's own default weights (mapped)
            try:
                import copy
                am = copy.copy(args)
                am.weno = "m"
                r = measure(am, 4, 10, rank, local_rank, world, with_e2e=False)
                summ.append(summary(r))
                also[r["config"]["workload"] + " with WENO5-M"] = {k: r[k] for k in (
                    "value", "ms_per_step", "ms_per_step_median_of_10_single_steps", "steps", "config", "cell_updates_per_s",
                    "clocks", "gpu_launches", "rhs_only", "roofline")}
            except Exception as exc:
                also["4 with WENO5-M"] = {"error": repr(exc)}
        out["also"] = also
        out["also_summary"] = summ
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.config, args.weno, args.model, args.eta)
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        torch.distributed.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
