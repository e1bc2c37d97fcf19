#!/usr/bin/env python
"""bench.py -- pixel-lens FP64 gradient+Hessian evaluations per second on B200.

A "step" is one pass of the whole hot path (rows a1-a5: pack the lens
list, hand the records to the launches, superpose first and second derivatives over all lenses at every
pixel, fused kappa/gamma/mu epilogue, stores) over BASELINE.json config 3:
4096 x 4096 pixels x 1000 dPIE potentials, outputs ax ay kappa gamma1 gamma2 mu, the
Hessian never written.  One process per GPU; at N > 1 every rank evaluates its own lens
model (an MCMC-style independent sample) on the same grid -- the path shards by
independent problems with no exchange step, so there is no collective on the data path
and `scaling` is "weak".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on the
host cores on a bounded sample of the same workload.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import lens_inputs as li  # noqa: E402

METRIC = "pixel-lens FP64 gradient+Hessian evals/sec"
UNIT = "evals/s"

# Executed FP64 flops per (pixel, lens) dPIE evaluation of each kernel variant (2*DFMA + DMUL + DADD
# thread-instructions / evaluations).  grad+hess: ncu counters, profiles/r01_cfg3_ncu.md (81.0 FP64
# instructions, 120.0 flop); grad / hess: the same count read from the SASS inner loop (56.75 and 46
# instructions).  DESIGN.md sec. 7.  This is what the hardware did -- `roofline.achieved` never claims more.
FLOPS_PER_EVAL = {"grad+hess": 120.0, "grad": 84.75, "hess": 69.0}
FP64_INSTR_PER_EVAL = {"grad+hess": 81.0, "grad": 56.75, "hess": 46.0}
# SURVEY.md sec. 8(d) canonical count for the cheapest exact formulation it knew (context: this kernel's
# formulation is cheaper, so evals/s x canonical flops can exceed the FLOP/s peak and is NOT a roofline fraction)
CANONICAL_FLOPS_PER_EVAL = {"grad+hess": 278.0, "grad": 205.0, "hess": 105.0}
# FP64 CUDA-core peak: 148 SMs x 64 FP64 FMA lanes x 2 flop x SM clock (B200_PROFILING.md:
# 148 SMs, clocks.max.sm 1965 MHz).  The live DFMA probe (lh_fp64_peak_probe) is the
# measured counterpart and is what `roofline.peak` reports.
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# dram bytes (read+write) per launch of the timed kernel from `ncu --set full` (profiles/r01_cfg3_ncu.md:
# a middle lens chunk of cfg 3 reads and writes the five carried accumulators)
NCU_TRAFFIC_BYTES = {3: 1.289e9}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (bench line: 3)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--delens", action="store_true",
                    help="NEXT row f1 alone (not the default bench line): lh_delens_grid on the deflection planes of "
                         "--config (default 3) for 80 synthetic sources (M1149 has 80, PAPER.md:208)")
    ap.add_argument("--chi2", action="store_true",
                    help="NEXT row f3 alone (not the default bench line): lh_chi2 on --config (default 3) with 80 "
                         "sources / 227 image constraints (the shape of M1149, PAPER.md:208) at seeded random positions")
    ap.add_argument("--stats", action="store_true",
                    help="NEXT row f2 on a batch config (use --config 4): per-pixel mean and variance of ax ay kappa "
                         "gamma1 gamma2 over the models through lh_grid_stats_batch (not the default bench line)")
    return ap.parse_args()


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------- CPU oracle leg
def oracle_sample(cfg, seconds: float):
    """Time the oracle as it stands on a bounded sample: whole rows of the configured grid,
    all lenses, all host cores (threads over disjoint row ranges)."""
    import oracle

    cores = os.cpu_count() or 1
    g, L = cfg.grid, cfg.lenses[: cfg.nlens]
    t0 = time.perf_counter()
    oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=cfg.outputs, threads=cores, rows=(0, cores))
    rate = cores * g.nx * cfg.nlens / (time.perf_counter() - t0)  # evals/s, all cores, rough
    rows = int(max(cores, min(g.ny, seconds * rate / (g.nx * cfg.nlens))))
    rows = max(cores, rows // cores * cores)
    t0 = time.perf_counter()
    oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=cfg.outputs, threads=cores, rows=(0, rows))
    dt = time.perf_counter() - t0
    evals = rows * g.nx * cfg.nlens
    return {"value": evals / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"rows 0..{rows - 1} of the {g.nx}x{g.ny} grid x {cfg.nlens} lenses "
                      f"({evals:.3g} evals, {dt:.1f} s; oracle/lens_oracle.c single-threaded per row slab, "
                      f"{cores} slabs in parallel)"}, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = li.config(args.config)
    per_step = max(1.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(min(args.warmup, 1)):
        oracle_sample(cfg, per_step / 4)
    vals, times = [], []
    base = None
    for _ in range(args.steps):
        base, dt = oracle_sample(cfg, per_step)
        vals.append(base["value"]); times.append(dt)
    v = float(np.mean(vals))
    base["value"] = v
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args), "cpu_baseline": base,
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workload_config(cfg, args):
    g = cfg.grid
    return {"workload": f"BASELINE.json configs[{args.config}] {cfg.name}: {g.nx}x{g.ny} px, {cfg.nlens} lenses"
                        + (f" x {cfg.nmodel} models" if cfg.nmodel > 1 else ""),
            "outputs": (["mean+variance over models of"] if getattr(args, "stats", False) else []) + list(cfg.outputs),
            "evals_per_step_per_gpu": cfg.evals,
            "l2": "L2 flushed between timed steps by rewriting a 256 MiB buffer (outside the timed events); output "
                  "planes %d MiB/step; the lens records (%d KiB) travel in the kernel parameters"
                  % (len(cfg.outputs) * cfg.nmodel * g.npix * 8 >> 20, cfg.nmodel * cfg.nlens * 192 >> 10),
            "parallelism": f"independent lens models per GPU x{args.gpus}, no collective"}


# ----------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2004_06352_b200 as lh

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    # LH_BENCH_BACKEND=gloo lets the N > 1 path be exercised where there are fewer GPUs than ranks (ranks then
    # share devices and only the timing reduction goes through the process group); the driver uses NCCL.
    backend = os.environ.get("LH_BENCH_BACKEND", "nccl")
    local = local % max(1, torch.cuda.device_count()) if backend != "nccl" else local
    torch.cuda.set_device(local)
    red_dev = "cuda" if backend == "nccl" else "cpu"
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)

    cfg = li.config(args.config)
    g = cfg.grid
    lenses = cfg.lenses
    if world > 1 and rank > 0 and cfg.nmodel == 1:
        # another independent sample of the same model family for this rank (same shape, other seed)
        lenses = li.cluster(1000 * args.config + rank, {1: 2, 2: 3, 3: 4}.get(args.config, 0), cfg.nlens
                            - {1: 2, 2: 3, 3: 4}.get(args.config, 0), {0: 40.0, 3: 150.0}.get(args.config, 100.0))
    shape = (cfg.nmodel, g.ny, g.nx)
    if args.stats:
        import dataclasses
        cfg = dataclasses.replace(cfg, outputs=("ax", "ay", "kappa", "gamma1", "gamma2"))
        shape = (g.ny, g.nx)
        var = {n: torch.empty(shape, dtype=torch.float64, device="cuda") for n in cfg.outputs}
    out = {n: torch.empty(shape, dtype=torch.float64, device="cuda") for n in cfg.outputs}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    lh.lh_set_stream(stream)

    def step():
        if args.stats:
            lh.lh_grid_stats_batch(lenses, cfg.nmodel, cfg.nlens, g, out, var)
        else:
            lh.lh_grid_eval_batch(lenses, cfg.nmodel, cfg.nlens, g, **out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches0 = lh.lh_launch_count()
    with ClockSampler(local) as clk:
        barrier()
        for a, b in ev:
            flush.zero_()  # L2 flush, outside the timed events
            a.record(stream)
            step()
            b.record(stream)
        barrier()
    launches = lh.lh_launch_count() - launches0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=red_dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = world * cfg.evals / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned), H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        host = {n: torch.empty(shape, dtype=torch.float64).pin_memory() for n in cfg.outputs}
        hvar = {n: torch.empty(shape, dtype=torch.float64).pin_memory() for n in cfg.outputs} if args.stats else None
        def step_host():
            if args.stats:  # host lens list in; mean and variance planes copied to pinned host memory
                step()
                for n in host:
                    host[n].copy_(out[n], non_blocking=True)
                    hvar[n].copy_(var[n], non_blocking=True)
                torch.cuda.synchronize()
            else:
                lh.lh_grid_eval_host(lenses, cfg.nmodel, cfg.nlens, g, **host)
        step_host()
        barrier()
        t0 = time.perf_counter()
        k_e2e = max(1, min(args.steps, 3))
        for _ in range(k_e2e):
            step_host()  # synchronises its stream before returning
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device=red_dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * cfg.evals * k_e2e / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(cfg.nmodel * cfg.nlens * 192 + cfg.nmodel * 8),
               "d2h_bytes_per_step": int(len(cfg.outputs) * g.npix * 16 if args.stats else
                                         len(cfg.outputs) * cfg.nmodel * g.npix * 8),
               "ms_per_step": 1e3 * dt / k_e2e, "steps": k_e2e,
               "note": "lh_grid_eval_host: host lens list in, pinned host planes out, packing + copies + sync timed; "
                       "the D2H copy of each of 8 row slabs overlaps the computation of the next"}
        del host

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel: FP64 CUDA-core ALU bound
    peak_flops, _ = lh.lh_fp64_peak_probe(1 << 15)
    mode = "grad+hess" if (set(cfg.outputs) & {"ax", "ay"}) and (set(cfg.outputs) - {"ax", "ay"}) else (
        "grad" if set(cfg.outputs) <= {"ax", "ay"} else "hess")
    fpe = FLOPS_PER_EVAL[mode]
    step_s = float(np.mean(step_ms)) * 1e-3
    per_step = launches / args.steps
    launch_s = step_s / per_step          # average duration of one superpose_kernel launch (CUDA events)
    launch_evals = cfg.evals / per_step   # units one launch processes
    achieved = fpe * launch_evals / launch_s / 1e12
    instr_rate = FP64_INSTR_PER_EVAL[mode] * launch_evals / launch_s  # FP64 thread-instructions / s
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_flops / 1e12, "unit": "TFLOP/s",
                "frac": achieved / (peak_flops / 1e12), "traffic": NCU_TRAFFIC_BYTES.get(args.config),
                "peak_source": "measured live: lh_fp64_peak_probe (DFMA chains, all SMs); nominal "
                               f"{NOMINAL_FP64_TFLOPS:.1f} TFLOP/s = 148 SM x 64 lanes x 2 x 1.965 GHz "
                               "(MEASURED_PEAKS.json has no FP64 entry)",
                "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                "flops_per_eval": fpe, "flops_per_eval_source": "executed FP64 flops (ncu / SASS), dPIE, " + mode,
                "fp64_issue_frac": instr_rate / (148 * 64 * 1.965e9),
                "fp64_issue_note": "FP64 thread-instructions/s over 148 x 64 lanes x 1.965 GHz; only "
                                   f"{100 * (fpe / FP64_INSTR_PER_EVAL[mode] - 1):.0f} % of them are FMAs, and every non-FP64 "
                                   "instruction costs a dispatch cycle of the same port (DESIGN.md sec. 7)",
                "canonical_flops_per_eval": CANONICAL_FLOPS_PER_EVAL[mode],
                "achieved_canonical": CANONICAL_FLOPS_PER_EVAL[mode] * cfg.evals / step_s / 1e12,
                "kernel": "lh::superpose_kernel<%s>" % mode, "launches_per_step": per_step,
                "kernel_ms": launch_s * 1e3, "units_per_launch": launch_evals,
                "store_gbs": len(cfg.outputs) * cfg.nmodel * g.npix * 8 / step_s / 1e9}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, args),
            "clocks": clk.summary(), "gpu_launches": int(launches), "roofline": roofline}
    if e2e:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world >= 1:
        line["cpu_baseline"], _ = oracle_sample(cfg, args.cpu_seconds)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_chi2(args):
    """f3 measured alone: one step = one chi^2 evaluation (all four stages of PAPER.md:192-194 on the device)."""
    import torch

    import paper_2004_06352_b200 as lh

    torch.cuda.set_device(0)
    cfg = li.config(args.config)
    g, L = cfg.grid, cfg.lenses[: cfg.nlens]
    rng = np.random.default_rng(1)
    ns, K = 80, 227
    half = 0.3 * g.nx * g.dx / 2
    cons = li.make_constraints((k if k < ns else int(rng.integers(0, ns)), rng.uniform(-half, half),
                                rng.uniform(-half, half), 0.3) for k in range(K))
    chi = torch.zeros(1, dtype=torch.float64, device="cuda")
    nim = torch.zeros(1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()
    lh.lh_set_stream(stream)
    for _ in range(max(args.warmup, 3)):
        lh.lh_chi2(L, g, cons, ns, chi, None, None, nim)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    n0 = lh.lh_launch_count()
    with ClockSampler(0) as clk:
        for a, b in ev:
            a.record(stream)
            lh.lh_chi2(L, g, cons, ns, chi, None, None, nim)
            b.record(stream)
        torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    evals = g.npix * cfg.nlens + K * cfg.nlens
    line = {"metric": "chi^2 evaluations/sec (eq. 6, four stages)", "value": 1e3 / ms, "unit": "chi2/s", "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "chi2": float(chi.item()), "images_found": int(nim.item()),
            "gradient_evals_per_s": evals / (ms * 1e-3),
            "config": {"workload": f"NEXT row f3: configs[{args.config}] {g.nx}x{g.ny} px x {cfg.nlens} lenses, "
                                   f"{ns} sources, {K} image constraints"},
            "clocks": clk.summary(), "gpu_launches": int(lh.lh_launch_count() - n0)}
    print(json.dumps(line), flush=True)


def run_delens(args):
    """f1 measured alone: one step = lh_delens_grid over the whole grid for 80 sources (deflection planes resident)."""
    import torch

    import paper_2004_06352_b200 as lh

    torch.cuda.set_device(0)
    cfg = li.config(args.config)
    g = cfg.grid
    ax = torch.empty((g.ny, g.nx), dtype=torch.float64, device="cuda")
    ay = torch.empty_like(ax)
    stream = torch.cuda.current_stream()
    lh.lh_set_stream(stream)
    lh.lh_grid_gradient(cfg.lenses[: cfg.nlens], g, ax, ay)
    ns = 80
    rng = np.random.default_rng(1234)
    half = 0.3 * g.nx * g.dx / 2
    src = np.column_stack([rng.uniform(-half, half, ns), rng.uniform(-half, half, ns)])
    cap = 1 << 16
    images = torch.zeros(32 * cap, dtype=torch.uint8, device="cuda")
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(max(args.warmup, 3)):
        lh.lh_delens_grid(ax, ay, g, src, images, cap, count)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    n0 = lh.lh_launch_count()
    with ClockSampler(0) as clk:
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            lh.lh_delens_grid(ax, ay, g, src, images, cap, count)
            b.record(stream)
        torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    cells = (g.nx - 1) * (g.ny - 1)
    t0 = time.perf_counter()
    import oracle
    rows = 256  # bounded oracle sample: the first 256 rows of cells
    hax, hay = ax[: rows + 1].cpu().numpy(), ay[: rows + 1].cpu().numpy()
    t0 = time.perf_counter()
    oracle.delens(hax, hay, g.x0, g.y0, g.dx, src)
    dt = time.perf_counter() - t0
    line = {"metric": "triangulated-grid delensing, cell-source tests/sec", "value": cells * ns / (ms * 1e-3),
            "unit": "cell-source tests/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "images_found": int(count.item()),
            "config": {"workload": f"NEXT row f1: {g.nx}x{g.ny} vertices of configs[{args.config}], {ns} sources"},
            "clocks": clk.summary(), "gpu_launches": int(lh.lh_launch_count() - n0),
            "roofline": {"bound": "alu", "achieved": cells * ns / (ms * 1e-3) / 1e12, "peak": 148 * 64 * 1.965e9 / 4 / 1e12,
                         "unit": "T cell-source tests/s", "frac": cells * ns / (ms * 1e-3) / (148 * 64 * 1.965e9 / 4),
                         "traffic": None,
                         "note": "the common path of a (cell, source) pair is the exact bounding-box reject = 4 FP64 "
                                 "compares; peak = 148 SM x 64 FP64 lanes x 1.965 GHz / 4.  HBM side: the two "
                                 "deflection planes are read once (16 B per vertex) = %.0f GB/s of the measured 6545"
                                 % (16.0 * g.npix / (ms * 1e-3) / 1e9)},
            "cpu_baseline": {"value": rows * (g.nx - 1) * ns / dt, "unit": "cell-source tests/s", "cores": 1,
                             "kind": "oracle", "sample": f"first {rows} cell rows, {ns} sources, {dt:.1f} s"}}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse()
    if a.chi2 and a.impl != "reference":
        run_chi2(a)
        raise SystemExit(0)
    if a.delens and a.impl != "reference":
        run_delens(a)
        raise SystemExit(0)
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
