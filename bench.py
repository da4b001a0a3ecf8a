#!/usr/bin/env python
"""bench.py -- throughput of the fused fp64 Godunov hydro step on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A "step" is one pass of the whole hot path: hx_compute_dt (CFL reduction, fused into the previous
update) + hx_step (ghost fill + fused unsplit MUSCL-Hancock/HLLC update with sources).  `value` is
Mcell-updates/s with the state resident in HBM (perf = n_x n_y n_z n_itr / t_elaps);
`e2e` is the same metric with the step driven through HOST buffers (hx_set_state from pinned memory
+ step + hx_get_state to pinned memory inside the timed region).  `roofline` is for the step kernel
alone, timed with CUDA events inside the library (HX_OPT_TIMING).  `cpu_baseline` is the CPU oracle
timed on this box's host cores on a reduced copy of the same workload.

N > 1 (torchrun): the path does not shard in this build: every rank runs an
independent replica of the workload on its own GPU, no data-path collective; time = max over ranks.
`--impl reference` times the CPU oracle (the only reference there is) on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2503_04428_b200 import workloads as wl  # noqa: E402

METRIC = "fp64 Mcell-updates/s per step (3D) on 1 B200; achieved HBM GB/s vs roofline"
UNIT = "Mcell-updates/s"

# full-size workloads (BASELINE.json configs) and the reduced copy the CPU oracle is timed on
WORKLOADS = {
    "rt_3d": (lambda: wl.rt_3d(512), lambda: wl.rt_3d((96, 96, 96))),
    "sedov_3d": (lambda: wl.sedov_3d(256), lambda: wl.sedov_3d((96, 96, 96))),
    "wedge_3d": (lambda: wl.wedge_3d((1024, 256, 256)), lambda: wl.wedge_3d((192, 48, 48))),
    "sedov_wedge_3d": (lambda: wl.sedov_wedge_3d(256), lambda: wl.sedov_wedge_3d(64)),   # PAPER.md Sect. 4.3
    "wedge_3d_rad": (lambda: wl.wedge_3d_rad((1024, 256, 256)), lambda: wl.wedge_3d_rad((96, 24, 24))),   # Eq. 6-7
    "wedge_3d_ns5": (lambda: wl.wedge_3d((1024, 256, 256), n_scalars=5), lambda: wl.wedge_3d((192, 48, 48), n_scalars=5)),   # nvar 10, ideal gas
    "wedge_3d_sn": (lambda: wl.wedge_3d_sn((1024, 256, 256)), lambda: wl.wedge_3d_sn((96, 24, 24))),   # rad EOS + 5 scalars + point mass
    "wedge_3d_selfgrav": (lambda: wl.wedge_3d_selfgrav((1024, 256, 256)), lambda: wl.wedge_3d_selfgrav((192, 48, 48))),   # Eq. 4
    "wedge_3d_emon": (lambda: wl.wedge_3d_emon((1024, 256, 256)), lambda: wl.wedge_3d_emon((192, 48, 48))),   # SURVEY 8(f) rank 2 on the spherical wedge
    "wedge_3d_sn_emon": (lambda: wl.wedge_3d_sn_emon((1024, 256, 256)), lambda: wl.wedge_3d_sn_emon((96, 24, 24))),   # rad EOS + 5 scalars + point mass + monitoring
    "cold_stream_3d": (lambda: wl.cold_stream_3d(256), lambda: wl.cold_stream_3d(64)),   # Eq. 10-12
    "kh_2d": (lambda: wl.kh_2d(1024), lambda: wl.kh_2d(512)),
    "sod_1d": (lambda: wl.sod_1d(1000), lambda: wl.sod_1d(1000)),
    # small case for quick checks of this script
    "rt_3d_small": (lambda: wl.rt_3d((128, 128, 128)), lambda: wl.rt_3d((48, 48, 48))),
    "wedge_3d_small": (lambda: wl.wedge_3d((256, 64, 64)), lambda: wl.wedge_3d((96, 24, 24))),
}
DEFAULT_WORKLOAD = "rt_3d"


def alg_flops_per_cell(spec):
    """Algorithmic fp64 flops per cell-update (hand count from O1-O7 with every predictor and
    face flux computed once; + and x count 1 each, so an FMA is 2; div and sqrt 1 each).
    3-D: 629 for nvar = 5, HLLC/HLL + minmod; +4 per slope for MC / van Leer, +6 van Albada; +84 per passive
    scalar; +31 gravity; +65 spherical sources; +1025 for the gas + radiation EOS (Newton solves for T).
    2-D (Cartesian): 380 for nvar = 4 (cons->prim 9, slopes 40, face states 32, cons + analytic flux of 4 face states
    80, 4 predicted states 68, U^n 8, 2 HLLC 94, update 32, CFL rate 17); +50 per passive scalar; +20 gravity."""
    ns = spec["nvar"] - 2 - spec["ndim"]
    nvar = spec["nvar"]
    lim_extra = {wl.LIM_NONE: -1, wl.LIM_MINMOD: 0, wl.LIM_VANLEER: 4, wl.LIM_VANALBADA: 6, wl.LIM_MC: 4}[spec["limiter"]]
    if spec["ndim"] == 2:
        return 380 + 50 * ns + 2 * nvar * lim_extra + (20 if spec["gravity"] != wl.GRAV_NONE else 0)
    f = 629 + 84 * ns + 3 * nvar * lim_extra
    if spec["gravity"] != wl.GRAV_NONE:
        f += 31
    if spec["coords"] == wl.SPHERICAL:
        f += 65
    if spec.get("eos", 0) == wl.EOS_GAS_RADIATION:
        # Eq. 6-7: 15 Newton-Raphson solves for T per cell-update (cons->prim, 6 face states P->e, 6 predicted states
        # e->P, U^n, CFL rate), about 7 iterations of 9 flop (+, x, one division) each; Eq. 7 adds ~10 per sound speed
        f += 15 * 7 * 9 + 8 * 10
    return f


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
                power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(make_reduced, budget_s=12.0, max_steps=None):
    """The CPU oracle as it stands on a reduced copy of the workload; returns (Mcell/s, description, cores)."""
    from oracle import ox
    spec, W = make_reduced()
    o = ox.Oracle(spec)
    o.set_state(W, ox.PRIMITIVE)
    ncell = int(np.prod(spec["n"]))
    o.step(o.compute_dt(spec["cfl"]))      # warm-up (page faults, thread pool)
    steps, t0 = 0, time.perf_counter()
    while True:
        o.step(o.compute_dt(spec["cfl"]))
        steps += 1
        el = time.perf_counter() - t0
        if el > budget_s or (max_steps and steps >= max_steps):
            break
    return ncell * steps / el / 1e6, f"{spec['name']} reduced to {spec['n'][:spec['ndim']]}, {steps} steps, {el:.1f} s", ox.num_threads(), el / steps


def run_reference(args):
    """--impl reference: there is no reference code for this paper; the arm times the CPU oracle."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    make_full, make_reduced = WORKLOADS[args.workload]
    from oracle import ox
    spec, W = make_reduced()
    o = ox.Oracle(spec)
    o.set_state(W, ox.PRIMITIVE)
    ncell = int(np.prod(spec["n"]))
    for _ in range(args.warmup):
        o.step(o.compute_dt(spec["cfl"]))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(o.compute_dt(spec["cfl"]))
    el = time.perf_counter() - t0
    val = ncell * args.steps / el / 1e6
    sample = f"{spec['name']} reduced to {spec['n'][:spec['ndim']]} cells, {args.steps} steps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "note": "CPU oracle (no reference code exists for this paper), bounded sample of the workload"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": ox.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def aggregate_max_ms(local_ms, world, backend_device=None):
    """Max over ranks of the timed region (device time).  Single rank: identity."""
    if world == 1:
        return local_ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


LIMITERS = {"none": wl.LIM_NONE, "minmod": wl.LIM_MINMOD, "vanleer": wl.LIM_VANLEER, "vanalbada": wl.LIM_VANALBADA, "mc": wl.LIM_MC}
SOLVERS = {"hll": wl.RIEMANN_HLL, "hllc": wl.RIEMANN_HLLC}


def override(problem, args):
    spec, W = problem
    spec = dict(spec)
    if args.limiter:
        spec["limiter"] = LIMITERS[args.limiter]
    if args.riemann:
        spec["riemann"] = SOLVERS[args.riemann]
    return spec, W


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2503_04428_b200 import hx

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    make_full, make_reduced = WORKLOADS[args.workload]
    if args.limiter or args.riemann:       # measured variants of a workload: other limiter / solver
        mf, mr = make_full, make_reduced
        make_full, make_reduced = (lambda: override(mf(), args)), (lambda: override(mr(), args))
    spec, W = make_full()          # N > 1: every rank runs the same workload (independent replicas, same seed, same overrides)
    ncell = int(np.prod(spec["n"]))
    nvar = spec["nvar"]
    cfl = spec["cfl"]
    K = args.steps if args.steps > 0 else (spec["steps"] or 300)
    stream = torch.cuda.current_stream()
    sim = hx.Hydro(spec, stream=stream)
    if args.kernel != "auto":
        sim.set_option(hx.OPT_KERNEL, {"generic": hx.KERNEL_GENERIC, "tile2": hx.KERNEL_TILED}[args.kernel])
    W = np.ascontiguousarray(W)
    sim.set_state(W, hx.PRIMITIVE)
    U0 = sim.get_state()                      # conserved initial state (host) for the e2e leg
    del W

    # ---- device-resident timing -------------------------------------------------------------
    for _ in range(args.warmup):
        sim.step(sim.compute_dt(cfl))
    sim.compute_dt(cfl)
    sim.set_option(hx.OPT_TIMING, 1)
    ms0, cnt0 = sim.kernel_time()
    launches0 = sim.launch_count
    clocks = ClockSampler(local_rank)
    clocks.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    for _ in range(K):
        sim.step(sim.compute_dt(cfl))
    ev1.record(stream)
    barrier()
    local_ms = ev0.elapsed_time(ev1)
    clk = clocks.stop()
    sim.compute_dt(cfl)                       # collects the last event pair
    ms1, cnt1 = sim.kernel_time()
    launches = sim.launch_count - launches0
    sim.set_option(hx.OPT_TIMING, 0)
    total_ms = aggregate_max_ms(local_ms, world, dev)
    value = world * ncell * K / (total_ms * 1e-3) / 1e6
    kernel_ms = (ms1 - ms0) / max(1, cnt1 - cnt0)

    # ---- end to end through host buffers ----------------------------------------------------
    # Every step copies its input state from pinned host memory to the GPU (hx_set_state), advances it (hx_compute_dt +
    # hx_step) and copies the result back to pinned host memory (hx_get_state).  Two handles on two streams work on
    # independent inputs in turn (HX_OPT_ASYNC_HOST), so that the upload of one step overlaps the download of the
    # previous one on the full-duplex link; each handle's own H2D -> step -> D2H chain stays ordered on its stream.
    e2e_steps = max(2, min(2 * K, args.e2e_steps))
    nbytes = ncell * nvar * 8
    h_in = torch.from_numpy(U0).pin_memory()
    del U0
    s2 = torch.cuda.Stream()
    sims = [sim, hx.Hydro(spec, stream=s2)]
    if args.kernel != "auto":
        sims[1].set_option(hx.OPT_KERNEL, {"generic": hx.KERNEL_GENERIC, "tile2": hx.KERNEL_TILED}[args.kernel])
    h_out = [torch.empty_like(h_in).pin_memory() for _ in sims]
    for sm, ho in zip(sims, h_out):
        sm.set_option(hx.OPT_ASYNC_HOST, 1)
        sm.set_state(h_in.numpy(), hx.CONSERVED)
        sm.step(sm.compute_dt(cfl))
        sm.get_state(ho.numpy(), hx.CONSERVED)          # warm-up of the host path
        sm.sync()
    barrier()
    ev0.record(stream)
    for s in range(e2e_steps):
        sm, ho = sims[s % 2], h_out[s % 2]
        sm.set_state(h_in.numpy(), hx.CONSERVED)         # enqueued behind this handle's previous download
        sm.step(sm.compute_dt(cfl))                      # waits for this handle's upload only
        sm.get_state(ho.numpy(), hx.CONSERVED)
    stream.wait_stream(s2)
    ev1.record(stream)
    for sm in sims:
        sm.sync()
    barrier()
    e2e_ms = aggregate_max_ms(ev0.elapsed_time(ev1), world, dev)
    e2e_value = world * ncell * e2e_steps / (e2e_ms * 1e-3) / 1e6
    assert torch.equal(h_out[0][:, :2], h_out[1][:, :2]), "the two pipelined handles disagree on the same input"
    kernel_name = sim.step_kernel
    sims[1].close()
    del h_in, h_out, sims

    if rank != 0:
        return
    peak, peak_src = measured_peaks()
    alg_bytes = 16 * nvar * ncell                        # read U^n once + write U^{n+1} once
    achieved = alg_bytes / (kernel_ms * 1e-3) / 1e9
    traffic, traffic_source = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")   # dram bytes per launch from the committed ncu captures
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            traffic = tj.get(args.workload, {}).get(kernel_name)
            if traffic is not None:
                traffic_source = "profiles/traffic.json (%s)" % tj.get("_source", "ncu --set full capture, see profiles/README.md")
        except Exception:
            traffic = None
    fp64_peak, dfma_lat = hx.probe_fp64()              # measured FP64 FMA rate of this GPU (TFLOP/s) and DFMA latency
    alg_flops = alg_flops_per_cell(spec) * ncell
    alu_achieved = alg_flops / (kernel_ms * 1e-3) / 1e12
    cpu_val, cpu_sample, cores, _ = time_oracle(make_reduced, budget_s=args.cpu_budget)
    state_gb = 2 * nvar * ncell * 8 / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "grid": spec["n"][:spec["ndim"]], "nvar": nvar, "cells": ncell,
                   "scheme": "unsplit MUSCL-Hancock + %s + %s, fp64" % ({v: k for k, v in SOLVERS.items()}[spec["riemann"]], {v: k for k, v in LIMITERS.items()}[spec["limiter"]]), "cfl": cfl, "step_kernel": kernel_name,
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (no sharding, SURVEY 8(e))",
                   "l2": f"inputs larger than L2 (two state buffers = {state_gb:.1f} GB vs 126 MB L2)" if state_gb > 0.5
                         else "state fits in L2: HBM fraction not meaningful for this workload"},
        # the path is FP64-pipe bound on B200: the binding roof is "alu"; the HBM figures stay beside it
        "roofline": {"bound": "alu", "achieved": alu_achieved, "peak": fp64_peak, "unit": "TFLOP/s", "frac": alu_achieved / fp64_peak,
                     "traffic": traffic, "traffic_source": traffic_source, "kernel": kernel_name, "kernel_ms": kernel_ms,
                     "algorithmic_flops_per_cell": alg_flops_per_cell(spec), "algorithmic_flops_per_launch": alg_flops,
                     "peak_source": "measured on this GPU by hx_probe_fp64 (independent DFMA chains on all SMs; nominal 148 SM x 64 lanes x 2 x 1.965 GHz = 37.2)",
                     "dfma_dependent_latency_cycles": dfma_lat, "kernel_share_of_step": kernel_ms / (total_ms / K)},
        "roofline_hbm": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src},
        "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": cpu_sample},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                "pipeline": "2 handles on 2 streams, independent inputs, async pinned-host copies (HX_OPT_ASYNC_HOST)"},
        "gpu_launches": launches,
        "clocks": clk,
    }
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="timed steps (default: the workload's own step count)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=12)
    ap.add_argument("--limiter", default=None, choices=sorted(LIMITERS), help="override the workload's slope limiter")
    ap.add_argument("--riemann", default=None, choices=sorted(SOLVERS), help="override the workload's Riemann solver")
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "tile2"], help="step kernel (A/B runs)")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of CPU oracle timing")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        if args.steps <= 0:
            args.steps = 5
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
