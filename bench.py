#!/usr/bin/env python
"""bench.py -- pixel-lens FP64 gradient+Hessian evaluations per second on B200.

A "step" is one pass of the whole hot path (rows a1-a5: pack the lens list, hand the records to
the launches, superpose first and second derivatives over all lenses at every pixel, fused kappa/gamma/mu epilogue,
stores) over BASELINE.json config 3: 4096 x 4096 pixels x 1000 dPIE potentials, outputs ax ay kappa gamma1 gamma2
mu, the Hessian never written.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--scaling auto|strong|weak] [--impl reference]

One process per GPU.  The path shards with no exchange step (pixels are independent):
  * N > 1, --scaling strong (the default for N > 1, "the grid is split among the
    GPUs", Fig. 7, Table A.4): rank r evaluates rows lens_inputs.row_slab(r, N) of the ONE map with lh_grid_eval_rows
    on its own device, the whole lens list replicated; `value` = evals of the one map / the slowest rank's time.
    Assembling the map on rank 0 (one gather of the slabs) is timed separately (`assemble`), it is not part of the
    computation.  For a BATCH config (--config 4) the same arm shards the other way SURVEY.md sec. 8(e) names, "for the
    batch path, models per GPU" (one map per tested parameter set): rank r evaluates models
    lens_inputs.model_slab(nmodel, r, N) of the ONE batch with lh_grid_gradient_batch (a pointer offset into the lens
    array) into its slice of [nmodel][ny][nx] -- in peer mode straight into rank 0's planes; `value` = evals of the
    whole batch / the slowest rank's time; rank 0 checks the assembled batch bitwise against its own single-device batch.
  * --scaling weak: every rank evaluates its own lens model on the full grid (independent MCMC samples).
Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded
sample of the same workload.
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
for _p in (ROOT, os.path.join(ROOT, "tests")):
    if _p not in sys.path:
        sys.path.insert(0, _p)

import lens_inputs as li  # noqa: E402

METRIC = "pixel-lens FP64 gradient+Hessian evals/sec"
UNIT = "evals/s"

# Executed FP64 thread-instructions per (pixel, lens) dPIE evaluation of each kernel variant, (DFMA, DMUL, DADD), read
# from the SASS of the lens loop of the built library: tests/test_sass_cpu.py RECOUNTS them with cuobjdump and fails
# when these constants and the kernel drift apart (the loop holds 4 evaluations, 8 in the gradient-only and the Hessian-only
# variants, whose per-row subexpressions are therefore shared by 8).  flop = 2 DFMA + DMUL + DADD.
# This is what the hardware did -- `roofline.achieved` never claims more.  DESIGN.md sec. 7.
FP64_OPS_PER_EVAL = {"grad+hess": (40.0, 28.75, 10.25), "grad": (30.0, 16.25, 9.125), "hess": (22.0, 16.375, 6.125)}
FP64_INSTR_PER_EVAL = {k: sum(v) for k, v in FP64_OPS_PER_EVAL.items()}
FLOPS_PER_EVAL = {k: 2 * v[0] + v[1] + v[2] for k, v in FP64_OPS_PER_EVAL.items()}
# SURVEY.md sec. 8(d) canonical count for the cheapest exact formulation it knew (context: this kernel's
# formulation is cheaper, so evals/s x canonical flops can exceed the FLOP/s peak and is NOT a roofline fraction)
CANONICAL_FLOPS_PER_EVAL = {"grad+hess": 278.0, "grad": 205.0, "hess": 105.0}
# FP64 CUDA-core peak: 148 SMs x 64 FP64 FMA lanes x 2 flop x SM clock (B200_PROFILING.md: 148 SMs, clocks.max.sm
# 1965 MHz).  The live DFMA probe (lh_fp64_peak_probe) is the measured counterpart and is what `roofline.peak` reports.
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
FP64_LANES_PER_S = 148 * 64 * 1.965e9
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the timed kernel, from one `ncu --set full` capture per
# config (profiles/r02_all_configs_ncu.md, profiles/r02_cfg3_ncu.md: a middle lens chunk where the model is chunked;
# launches whose output fits the 126 MB L2 show almost no DRAM traffic inside the launch -- write-back caching)
NCU_TRAFFIC_BYTES = {0: 1.04e5, 1: 1.02e5, 2: 5.44e7, 3: 6.191e8, 4: 1.688e7}
# the NEXT-row kernels (profiles/r03_next_rows_ncu.md): delens_kernel on 4096^2 vertices x 80 sources; the statistics
# epilogue launch (last lens chunk of a model of cfg 4 with --stats).  tests/test_profiles_cpu.py compares all of these
# constants with the figures in the profile notes they cite.
NCU_TRAFFIC_DELENS_BYTES = 2.725e8
NCU_TRAFFIC_STATS_BYTES = 1.568e8


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (bench line: 3)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="auto", choices=["auto", "strong", "weak"],
                    help="N > 1: strong (default) = ONE job over the GPUs: row slabs of the one map, or for a batch config "
                         "(--config 4) the models of the one batch; weak = an independent job per rank")
    ap.add_argument("--assemble", default="auto", choices=["auto", "peer", "gather"],
                    help="strong scaling: how the one map reaches rank 0 -- peer: every rank's kernel stores its rows straight "
                         "into rank 0's planes (CUDA IPC + NVLink peer access, no second pass); gather: one dist.gather "
                         "after the computation; auto: peer when the mapping succeeds on every rank, else gather")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="target CPU time of the all-cores oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config block (cfg 0, 1, 2, 4)")
    ap.add_argument("--delens", action="store_true",
                    help="NEXT row f1 alone (not the default bench line): lh_delens_grid on the deflection planes of "
                         "--config (default 3) for 80 synthetic sources (M1149 has 80, PAPER.md:208)")
    ap.add_argument("--chi2", action="store_true",
                    help="NEXT row f3 alone (not the default bench line): lh_chi2 on --config (default 3) with 80 "
                         "sources / 227 image constraints (the shape of M1149, PAPER.md:208) at seeded random positions")
    ap.add_argument("--shared", action="store_true",
                    help="NEXT row f4 on config 4 (not the default bench line): the 298 galaxies the 64 models have in common "
                         "are evaluated once (lh_grid_eval_batch_shared), each model adds its 2 halos")
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


# ----------------------------------------------------------------------------- CPU oracle legs
def oracle_sample(cfg, seconds: float, threads: int | None = None, min_rows: int = 0):
    """Time the oracle as it stands on a bounded sample: whole rows of the configured grid (first model of a
    batch), all lenses, `threads` host threads over disjoint row ranges (default: all cores)."""
    import oracle

    cores = threads or os.cpu_count() or 1
    g, L = cfg.grid, cfg.lenses[: cfg.nlens]
    probe = max(cores, 2)
    t0 = time.perf_counter()
    oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=cfg.outputs, threads=cores, rows=(0, min(probe, g.ny)))
    rate = min(probe, g.ny) * g.nx * cfg.nlens / (time.perf_counter() - t0)  # evals/s, rough
    rows = int(max(cores, min_rows, min(g.ny, seconds * rate / (g.nx * cfg.nlens))))
    rows = min(g.ny, max(cores, rows // cores * cores))
    t0 = time.perf_counter()
    oracle.grid(L, g.x0, g.y0, g.dx, g.nx, g.ny, planes=cfg.outputs, threads=cores, rows=(0, rows))
    dt = time.perf_counter() - t0
    evals = rows * g.nx * cfg.nlens
    whole = " (the whole map)" if rows == g.ny and cfg.nmodel == 1 else " (a slab: the work is exactly linear in rows)"
    return {"value": evals / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"rows 0..{rows - 1} of the {g.nx}x{g.ny} grid x {cfg.nlens} lenses{whole} "
                      f"({evals:.3g} evals, {dt:.1f} s; oracle/lens_oracle.c single-threaded per row range, "
                      f"{cores} range(s) in parallel)"}, dt


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
            "config": workload_config(cfg, args, 1, "weak"), "cpu_baseline": base,
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workload_config(cfg, args, world, scaling):
    g = cfg.grid
    if world == 1:
        par = "one GPU"
    elif scaling == "strong" and cfg.nmodel > 1:
        par = (f"the {cfg.nmodel} models of the ONE batch over {world} GPUs (lens_inputs.model_slab, lh_grid_gradient_batch on "
               "each rank's models), no collective in the computation; peer stores or one gather assemble the batch")
    elif scaling == "strong":
        par = (f"row slabs of the ONE map over {world} GPUs (lens_inputs.row_slab, lh_grid_eval_rows), lens list "
               "replicated, no collective in the computation; one gather assembles the map (timed apart)")
    else:
        par = f"an independent lens model per GPU x{world} (MCMC-style samples), no collective"
    return {"workload": f"BASELINE.json configs[{args.config}] {cfg.name}: {g.nx}x{g.ny} px, {cfg.nlens} lenses"
                        + (f" x {cfg.nmodel} models" if cfg.nmodel > 1 else ""),
            "outputs": (["mean+variance over models of"] if getattr(args, "stats", False) else []) + list(cfg.outputs),
            "evals_per_step": cfg.evals * (world if scaling == "weak" else 1),
            "l2": "L2 flushed between timed steps by rewriting a 256 MiB buffer (outside the timed events); output "
                  "planes %d MiB/step; the lens records (%d KiB) travel in the kernel parameters"
                  % (len(cfg.outputs) * cfg.nmodel * g.npix * 8 >> 20, cfg.nmodel * cfg.nlens * 192 >> 10),
            "parallelism": par}


def variant_of(outputs):
    o = set(outputs)
    return "grad+hess" if (o & {"ax", "ay"}) and (o - {"ax", "ay"}) else ("grad" if o <= {"ax", "ay"} else "hess")


def stats_of(ms):
    ms = [float(x) for x in ms]
    return {"ms_mean": float(np.mean(ms)), "ms_median": float(np.median(ms)), "ms_best": float(np.min(ms)), "n": len(ms)}


# ----------------------------------------------------------------------------- our arm: helpers
def time_device_steps(torch, lh, step, steps, warmup, stream, flush):
    """W untimed steps, then K steps each bracketed by CUDA events on the launching stream (L2 flushed before each,
    outside the events).  Returns (per-step ms, launches in the timed region)."""
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    n0 = lh.lh_launch_count()
    for a, b in ev:
        flush.zero_()
        a.record(stream)
        step()
        b.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in ev], lh.lh_launch_count() - n0


def sampled_parity(torch, cfg, out, model=0, n=1000, seed=2026):
    """Parity of the planes the LAST timed step left on the device: `n` seeded pixels (plus the corners) against the
    oracle evaluated pixel by pixel, by the rules of tests/parity.py.  Returns the worst |d|/allowed (<= 1 passes)."""
    import oracle
    from parity import report_planes

    g = cfg.grid
    ii, jj = li.random_points(seed, g, n)
    ii = np.concatenate([ii, [0, g.nx - 1, 0, g.nx - 1]])
    jj = np.concatenate([jj, [0, 0, g.ny - 1, g.ny - 1]])
    need = set(cfg.outputs)
    if "mu" in need:
        need |= {"kappa", "gamma1", "gamma2"}
    L = cfg.lenses[model * cfg.nlens:(model + 1) * cfg.nlens]
    ref = oracle.points(L, g.x0 + ii * g.dx, g.y0 + jj * g.dx, planes=tuple(sorted(need)))
    it, jt = torch.as_tensor(ii, device="cuda"), torch.as_tensor(jj, device="cuda")
    got = {}
    for name in cfg.outputs:
        t = out[name]
        t = t[model] if t.dim() == 3 else t
        got[name] = t[jt, it].cpu().numpy()
    rep = report_planes(got, ref)
    worst = max(r["worst"] for r in rep.values())
    return {"pixels": int(len(ii)), "worst_ratio": float(worst), "ok": bool(worst <= 1.0),
            "planes": {k: float(v["worst"]) for k, v in rep.items()},
            "rule": "tests/parity.py: |d| <= max(1e-11 |P|, 1e-13 max|P|) per plane, mu conditioned (R13); "
                    "the planes of the last timed step vs oracle.points"}


# FP64 thread-instructions per evaluation of the other lens classes (same source: SASS lens loops, recounted by
# tests/test_sass_cpu.py) -- only used for the FP64 issue fraction of the mixed config 2
FP64_INSTR_PER_EVAL_CLASS = {"grad+hess": {"dpie": 79.0, "nsie": 57.0, "sis": 17.75},
                             "grad": {"dpie": 55.375, "nsie": 41.375, "sis": 10.25},
                             "hess": {"dpie": 44.5, "nsie": 29.5, "sis": 15.375}}


def fp64_instr_of(cfg, mode):
    """FP64 thread-instructions one pass over `cfg` executes per pixel and model (sum over its lenses by class)."""
    t = cfg.lenses["type"][: cfg.nlens]
    k = FP64_INSTR_PER_EVAL_CLASS[mode]
    return float(np.sum(t == li.DPIE) * k["dpie"] + np.sum(t == li.NSIE) * k["nsie"] + np.sum(t == li.SIS) * k["sis"])


def config_block(torch, lh, stream, flush, which=(0, 1, 2, 4), steps=5, oracle_too=True):
    """ms/step, evals/s and FP64 issue fraction of the other BASELINE configs (device-resident, CUDA events), and the
    single-thread oracle rate beside each (the whole map for cfg 0-1, a 64-row slab for cfg 2, 4)."""
    block = {}
    for idx in which:
        c = li.config(idx)
        g = c.grid
        out = {n: torch.empty((c.nmodel, g.ny, g.nx), dtype=torch.float64, device="cuda") for n in c.outputs}

        def step():
            lh.lh_grid_eval_batch(c.lenses, c.nmodel, c.nlens, g, **out)

        ms, launches = time_device_steps(torch, lh, step, steps, 3, stream, flush)
        mode = variant_of(c.outputs)
        st = stats_of(ms)
        sec = st["ms_median"] * 1e-3
        # what a sampler that needs each result before its next proposal sees: host lens list in,
        # device planes out, a synchronize after every call -- wall clock, no L2 flush (the sampler would not flush
        # either).  Beside it the host-only share: validation + packing of all the call's lenses (lh_pack_model).
        torch.cuda.synchronize()
        k_sync = max(steps, 20 if c.evals < 2e9 else steps)
        walls = []
        for _ in range(k_sync):
            t0 = time.perf_counter()
            step()
            torch.cuda.synchronize()
            walls.append((time.perf_counter() - t0) * 1e3)
        L = c.lenses.reshape(c.nmodel, c.nlens)
        packs = []
        for _ in range(5):
            t0 = time.perf_counter()
            for m in range(c.nmodel):
                lh.lh_pack_model(L[m])
            packs.append((time.perf_counter() - t0) * 1e3)
        per_call = {"ms_median": float(np.median(walls)), "ms_best": float(np.min(walls)), "calls": k_sync,
                    "overhead_ms": float(np.median(walls)) - st["ms_median"],
                    "overhead_frac_of_kernel_time": float(np.median(walls)) / st["ms_median"] - 1.0,
                    "host_pack_ms": float(np.median(packs)),
                    "note": "one call + torch.cuda.synchronize(), wall clock (validation, packing, ctypes, launches, "
                            "kernels, sync); overhead = that minus the device-timed median; host_pack_ms = lh_pack_model "
                            f"over the call's {c.nmodel * c.nlens} lenses from Python, one call per model (includes "
                            "ctypes and the table allocation: an upper bound of the packing inside the call)"}
        block[f"cfg{idx}"] = {
            "workload": f"{c.name}: {g.nx}x{g.ny} px x {c.nlens} lenses" + (f" x {c.nmodel} models" if c.nmodel > 1 else ""),
            "outputs": list(c.outputs), "kernel": f"superpose_kernel<{mode}>", "steps": steps, **st,
            "evals_per_s": c.evals / sec, "launches_per_step": launches / steps,
            "fp64_issue_frac": fp64_instr_of(c, mode) * g.npix * c.nmodel / sec / FP64_LANES_PER_S,
            "traffic": NCU_TRAFFIC_BYTES.get(idx), "per_call_synchronised": per_call,
            "parity_last_step": sampled_parity(torch, c, out, model=c.nmodel - 1, n=300)}
        del out
        if oracle_too:
            one, _ = oracle_sample(c, 0.0, threads=1, min_rows=g.ny if idx <= 1 else 64)
            block[f"cfg{idx}"]["oracle_single_thread"] = {k: one[k] for k in ("value", "unit", "cores", "sample")}
    return block


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
    # share devices and the reductions / the gather go through host memory); the driver uses NCCL.
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

    def reduce_max(x):
        if world == 1:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=red_dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = li.config(args.config)
    g = cfg.grid
    scaling = args.scaling
    if scaling == "auto":
        scaling = "strong" if (world > 1 and not args.stats) else "weak"
    if scaling == "strong" and args.stats:
        raise SystemExit("--scaling strong: the statistics mode folds every model on one device (use --scaling weak)")
    # split (i) rows of the ONE map, split (ii) "for the batch path, models per GPU"
    by_model = scaling == "strong" and cfg.nmodel > 1
    by_rows = scaling == "strong" and not by_model
    m0, m1 = li.model_slab(cfg.nmodel, rank, world) if by_model else (0, cfg.nmodel)
    nmine = m1 - m0
    lenses = cfg.lenses
    lenses_mine = cfg.lenses[m0 * cfg.nlens:m1 * cfg.nlens]  # by_model: this rank's models (a pointer offset at the C ABI)
    if scaling == "weak" and world > 1 and rank > 0 and cfg.nmodel == 1:
        # another independent sample of the same model family for this rank (same shape, other seed)
        nh = {1: 2, 2: 3, 3: 4}.get(args.config, 0)
        lenses = li.cluster(1000 * args.config + rank, nh, cfg.nlens - nh, {0: 40.0, 3: 150.0}.get(args.config, 100.0))
    j0, nrows = li.row_slab(g, rank, world) if by_rows else (0, g.ny)
    shape = (nrows, g.nx) if by_rows else (nmine, g.ny, g.nx)
    whole = (g.ny, g.nx) if by_rows else (cfg.nmodel, g.ny, g.nx)  # the assembled result on rank 0
    first = j0 * g.nx if by_rows else m0 * g.npix                   # element offset of this rank's part inside it
    if args.stats:
        import dataclasses
        cfg = dataclasses.replace(cfg, outputs=("ax", "ay", "kappa", "gamma1", "gamma2"))
        shape = (g.ny, g.nx)
        var = {n: torch.empty(shape, dtype=torch.float64, device="cuda") for n in cfg.outputs}
    out = {n: torch.empty(shape, dtype=torch.float64, device="cuda") for n in cfg.outputs}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    lh.lh_set_stream(stream)

    # ---- strong scaling, peer mode: rank 0 owns the one map; every other rank maps it (CUDA IPC) and its kernel
    # stores its rows straight into it -- the assembly rides on the epilogue stores, no gather, no second pass
    peer, peer_ptrs, owner_map = None, {}, None
    if scaling == "strong" and world > 1 and args.assemble in ("auto", "peer"):
        ok, err = 1, ""
        handles = [None]
        if rank == 0:
            try:
                owner_map = {n: torch.empty(whole, dtype=torch.float64, device="cuda") for n in cfg.outputs}
                handles = [{n: lh.lh_ipc_export(t) for n, t in owner_map.items()}]
            except Exception as e:  # e.g. an allocator whose memory cannot be exported
                ok, err, handles = 0, repr(e), [None]
        dist.broadcast_object_list(handles, src=0)  # every rank takes part, whatever happened on rank 0
        if handles[0] is None:
            ok = 0
        elif rank == 0:
            peer = {n: (owner_map[n][j0:j0 + nrows] if by_rows else owner_map[n][m0:m1]) for n in cfg.outputs}
        else:
            try:
                for n in cfg.outputs:
                    peer_ptrs[n] = lh.lh_ipc_open(*handles[0][n])
                peer = {n: peer_ptrs[n] + first * 8 for n in cfg.outputs}  # address of this rank's first row / model
            except Exception as e:  # no peer access between the two devices: fall back to the gather
                ok, err = 0, repr(e)
        t = torch.tensor([float(ok)], dtype=torch.float64, device=red_dev)
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        if float(t.item()) < 1.0:
            if args.assemble == "peer":
                raise SystemExit(f"--assemble peer: the owner's map could not be mapped on every rank ({err})")
            for ptr in peer_ptrs.values():
                lh.lh_ipc_close(ptr)
            peer, peer_ptrs, owner_map = None, {}, None

    def run_part(target):
        """this rank's part of the strong-scaling job into `target` (its own planes, or its place in rank 0's)"""
        if by_rows and nrows > 0:
            lh.lh_grid_eval_rows(lenses, g, j0, nrows, **target)
        elif by_model and nmine > 0:
            if tuple(cfg.outputs) == ("ax", "ay"):  # the north-star call of the batch path
                lh.lh_grid_gradient_batch(lenses_mine, nmine, cfg.nlens, g, target["ax"], target["ay"])
            else:
                lh.lh_grid_eval_batch(lenses_mine, nmine, cfg.nlens, g, **target)

    def run_whole(target):
        """the whole job on this device (rank 0's bitwise reference of the assembled result)"""
        if by_rows:
            lh.lh_grid_eval(lenses, g, **target)
        else:
            lh.lh_grid_eval_batch(cfg.lenses, cfg.nmodel, cfg.nlens, g, **target)

    def step():
        if args.stats:
            lh.lh_grid_stats_batch(lenses, cfg.nmodel, cfg.nlens, g, out, var)
        elif scaling == "strong":
            run_part(peer if peer is not None else out)
        else:
            lh.lh_grid_eval_batch(lenses, cfg.nmodel, cfg.nlens, g, **out)

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
    launches = lh.lh_launch_count() - launches0  # this rank's
    launches_all = launches
    if world > 1:
        t = torch.tensor([float(launches)], dtype=torch.float64, device=red_dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        launches_all = int(t.item())
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = reduce_max(sum(step_ms))  # MAX over ranks of the device time of the K steps
    ms_per_step = total_ms / args.steps
    job_evals = cfg.evals * (world if scaling == "weak" else 1)  # units ALL ranks processed per step
    value = job_evals / (ms_per_step * 1e-3)

    # ---- strong scaling, peer mode: the timed steps already left the whole map in rank 0's planes
    assemble = None
    if peer is not None:
        run_part(out)  # this rank's own copy (parity sample, e2e comparison)
        barrier()  # every writer synchronised: the owner may read
        assemble = {"ms": 0.0, "bytes": int(len(cfg.outputs) * int(np.prod(whole)) * 8), "mode": "peer",
                    "how": ("every rank's kernels store its " + ("rows" if by_rows else "models") + " straight into rank 0's planes "
                            "(CUDA IPC mapping, peer access over NVLink): the assembly is inside the timed steps, no gather, "
                            "no second pass"),
                    "bitwise_check": None}
        if rank == 0:
            ref = {n: torch.empty(whole, dtype=torch.float64, device="cuda") for n in cfg.outputs}
            run_whole(ref)
            torch.cuda.synchronize()
            assemble["bitwise_check"] = all(bool((owner_map[n].view(torch.int64) == ref[n].view(torch.int64)).all())
                                            for n in cfg.outputs)
            del ref
        barrier()
        for ptr in peer_ptrs.values():
            lh.lh_ipc_close(ptr)
    # ---- strong scaling, gather mode: the time to assemble the one map on rank 0 (not part of the computation)
    if scaling == "strong" and world > 1 and peer is None:
        if by_rows:
            rows_of = [li.row_slab(g, r, world)[1] for r in range(world)]
            unit = (g.nx,)
        else:  # units are whole models
            rows_of = [b - a for a, b in (li.model_slab(cfg.nmodel, r, world) for r in range(world))]
            unit = (g.ny, g.nx)
        pad = max(rows_of)
        full = {n: torch.empty((world, pad) + unit, dtype=torch.float64, device="cuda") for n in cfg.outputs} if rank == 0 else None
        mine = {n: torch.zeros((pad,) + unit, dtype=torch.float64, device="cuda") for n in cfg.outputs}
        for n in cfg.outputs:
            mine[n][:rows_of[rank]].copy_(out[n])

        def gather():
            for n in cfg.outputs:
                if backend == "nccl":
                    dist.gather(mine[n], list(full[n].unbind(0)) if rank == 0 else None, dst=0)
                else:  # gloo stand-in: through host memory
                    parts = [torch.empty((pad,) + unit, dtype=torch.float64) for _ in range(world)] if rank == 0 else None
                    dist.gather(mine[n].cpu(), parts, dst=0)
                    if rank == 0:
                        full[n].copy_(torch.stack(parts))

        gather()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(3):
            gather()
        e1.record(stream)
        torch.cuda.synchronize()
        dev_ms = reduce_max(e0.elapsed_time(e1) / 3)
        wall_ms = reduce_max((time.perf_counter() - t0) * 1e3 / 3)
        assemble = {"ms": dev_ms if backend == "nccl" else wall_ms, "bytes": int(len(cfg.outputs) * int(np.prod(whole)) * 8),
                    "mode": "gather", "how": ("one dist.gather (NCCL) of every rank's slab of each plane into rank 0's map, CUDA events, "
                            "max over ranks" if backend == "nccl" else "gloo stand-in through host memory, wall clock"),
                    "bitwise_check": None}
        if rank == 0:  # the assembled map is the single-device map, bit for bit (checked on rank 0's own device)
            ref = {n: torch.empty(whole, dtype=torch.float64, device="cuda") for n in cfg.outputs}
            run_whole(ref)
            torch.cuda.synchronize()
            ok = True
            for n in cfg.outputs:
                asm = torch.cat([full[n][r, :rows_of[r]] for r in range(world)])
                ok = ok and bool((asm.view(torch.int64) == ref[n].view(torch.int64)).all())
            assemble["bitwise_check"] = ok
            del ref
        del mine, full

    # ---- end to end through the C ABI with HOST buffers: H2D of the lens list + D2H of the planes inside the timed region
    e2e = None
    if not args.no_e2e:
        k_e2e = max(5, min(args.steps, 10))

        def e2e_run(pinned: bool):
            def alloc():
                t = torch.empty(shape, dtype=torch.float64)
                return t.pin_memory() if pinned else t
            host = {n: alloc() for n in cfg.outputs}
            hvar = {n: alloc() for n in cfg.outputs} if args.stats else None

            def step_host():
                if args.stats:  # host lens list in; mean and variance planes copied to host memory
                    step()
                    for n in host:
                        host[n].copy_(out[n], non_blocking=pinned)
                        hvar[n].copy_(var[n], non_blocking=pinned)
                    torch.cuda.synchronize()
                elif by_rows:
                    if nrows > 0:
                        lh.lh_grid_eval_rows_host(lenses, g, j0, nrows, **host)
                elif by_model:
                    if nmine > 0:
                        lh.lh_grid_eval_host(lenses_mine, nmine, cfg.nlens, g, **host)
                else:
                    lh.lh_grid_eval_host(lenses, cfg.nmodel, cfg.nlens, g, **host)

            step_host()
            barrier()
            times = []
            for _ in range(k_e2e):
                t0 = time.perf_counter()
                step_host()  # synchronises its stream before returning
                torch.cuda.synchronize()
                times.append((time.perf_counter() - t0) * 1e3)
            total = reduce_max(sum(times))
            bitwise = all(bool((host[n].view(torch.int64) == out[n].cpu().view(torch.int64)).all()) for n in cfg.outputs) \
                if not args.stats else None
            return total / k_e2e, times, bitwise

        ms_pin, t_pin, bit_pin = e2e_run(True)
        ms_page, t_page, bit_page = e2e_run(False)
        nl = nmine * cfg.nlens
        e2e = {"value": job_evals / (ms_pin * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(nl * 192 + nmine * 8),
               "d2h_bytes_per_step": int(len(cfg.outputs) * g.npix * 16 if args.stats else
                                         len(cfg.outputs) * int(np.prod(shape)) * 8),
               "ms_per_step": ms_pin, "steps": k_e2e, **{k: v for k, v in stats_of(t_pin).items() if k != "n"},
               "host_memory": "pinned", "same_bits_as_device_planes": bit_pin,
               "pageable": {"value": job_evals / (ms_page * 1e-3), "ms_per_step": ms_page, "steps": k_e2e,
                            **{k: v for k, v in stats_of(t_page).items() if k != "n"},
                            "same_bits_as_device_planes": bit_page},
               "note": ("lh_grid_eval_rows_host" if by_rows else "lh_grid_eval_host")
                       + ": host lens list in, host planes out, validation + packing + copies + sync timed (wall clock "
                         "around the call, max over ranks); the D2H copy of each of up to 8 pieces overlaps the computation "
                         "of the next; bytes are per rank"}

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel: FP64 CUDA-core ALU bound
    peak_flops, _ = lh.lh_fp64_peak_probe(1 << 15)
    mode = variant_of(cfg.outputs)
    fpe = FLOPS_PER_EVAL[mode]
    step_s = float(np.mean(step_ms)) * 1e-3      # rank 0's own steps
    per_step = launches / args.steps
    rank_evals = cfg.evals * (nrows / g.ny if by_rows else (nmine / cfg.nmodel if by_model else 1.0))
    launch_s = step_s / max(per_step, 1e-9)       # average duration of one superpose_kernel launch (CUDA events)
    launch_evals = rank_evals / max(per_step, 1e-9)  # units one launch processes
    achieved = fpe * launch_evals / launch_s / 1e12
    instr_rate = FP64_INSTR_PER_EVAL[mode] * launch_evals / launch_s  # FP64 thread-instructions / s
    d, m, a = FP64_OPS_PER_EVAL[mode]
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_flops / 1e12, "unit": "TFLOP/s",
                "frac": achieved / (peak_flops / 1e12),
                "traffic": NCU_TRAFFIC_STATS_BYTES if (args.stats and args.config == 4) else NCU_TRAFFIC_BYTES.get(args.config),
                "peak_source": "measured live: lh_fp64_peak_probe (DFMA chains, all SMs); nominal "
                               f"{NOMINAL_FP64_TFLOPS:.1f} TFLOP/s = 148 SM x 64 lanes x 2 x 1.965 GHz "
                               "(MEASURED_PEAKS.json has no FP64 entry)",
                "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                "flops_per_eval": fpe, "fp64_instr_per_eval": {"dfma": d, "dmul": m, "dadd": a},
                "flops_per_eval_source": "executed FP64 flops of the dPIE lens loop, " + mode
                                         + " (SASS; recounted by tests/test_sass_cpu.py)",
                "fp64_issue_frac": instr_rate / FP64_LANES_PER_S,
                "fp64_issue_note": "FP64 thread-instructions/s over 148 x 64 lanes x 1.965 GHz; only "
                                   f"{100 * d / (d + m + a):.0f} % of them are FMAs, and every non-FP64 "
                                   "instruction costs a dispatch cycle of the same port (DESIGN.md sec. 7)",
                "canonical_flops_per_eval": CANONICAL_FLOPS_PER_EVAL[mode],
                "achieved_canonical": CANONICAL_FLOPS_PER_EVAL[mode] * rank_evals / step_s / 1e12,
                "kernel": "lh::superpose_kernel<%s>" % mode, "launches_per_step": per_step,
                "kernel_ms": launch_s * 1e3, "units_per_launch": launch_evals,
                "store_gbs": len(cfg.outputs) * int(np.prod(shape)) * 8 / step_s / 1e9}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, **{k: v for k, v in stats_of(step_ms).items() if k != "n"},
            "higher_is_better": True, "scaling": scaling if world > 1 else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(cfg, args, world, scaling),
            "clocks": clk.summary(), "gpu_launches": int(launches_all), "roofline": roofline}
    if world > 1:
        line["gpu_launches_rank0"] = int(launches)
    if not args.stats:
        sub = cfg if not by_rows else None
        if sub is not None:  # rank 0 holds models [0, nmine): local and global model index agree
            line["parity_last_step"] = sampled_parity(torch, cfg, out, model=nmine - 1)
        else:  # rank 0's slab: rows [0, nrows) of the same grid
            import dataclasses
            slab = dataclasses.replace(cfg, grid=li.Grid(g.x0, g.y0, g.dx, g.nx, nrows))
            line["parity_last_step"] = sampled_parity(torch, slab, out)
    if assemble:
        line["assemble"] = assemble
    if e2e:
        line["e2e"] = e2e
    if world == 1 and not args.no_configs and args.config == 3 and not args.stats:
        line["configs"] = config_block(torch, lh, stream, flush, oracle_too=not args.no_cpu_baseline)
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"], _ = oracle_sample(cfg, args.cpu_seconds)
        one, _ = oracle_sample(cfg, 0.0, threads=1, min_rows=64 if cfg.evals > 2e9 else g.ny)
        line["cpu_baseline"]["single_thread"] = {k: one[k] for k in ("value", "unit", "cores", "sample")}
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


def run_shared(args):
    """f4 measured alone: one step = lh_grid_eval_batch_shared on config 4 (shared galaxies once + 2 halos per model),
    reported apart from the headline as SURVEY.md sec. 8(a6) asks: it is NOT the 2.0e10-evaluation workload of cfg 4."""
    import torch

    import paper_2004_06352_b200 as lh

    torch.cuda.set_device(0)
    c = li.config(4)
    g = c.grid
    L = c.lenses.reshape(c.nmodel, c.nlens)
    shared, varying = L[0, 2:].copy(), np.ascontiguousarray(L[:, :2]).reshape(-1)
    assert all(np.array_equal(L[m, 2:], shared) for m in range(c.nmodel))
    out = {n: torch.empty((c.nmodel, g.ny, g.nx), dtype=torch.float64, device="cuda") for n in c.outputs}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    lh.lh_set_stream(stream)

    def step():
        lh.lh_grid_eval_batch_shared(shared, varying, c.nmodel, 2, g, **out)

    with ClockSampler(0) as clk:
        ms, launches = time_device_steps(torch, lh, step, args.steps, max(args.warmup, 3), stream, flush)
    st = stats_of(ms)
    done = g.npix * (len(shared) + 2 * c.nmodel)  # evaluations actually executed
    line = {"metric": "shared-lens batch, maps/sec (64 models of 300 lenses, 298 shared)", "value": c.nmodel / (st["ms_mean"] * 1e-3),
            "unit": "model maps/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": st["ms_mean"],
            **{k: v for k, v in st.items() if k != "n"}, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"NEXT row f4: configs[4] {g.nx}x{g.ny} px, {c.nmodel} models = {len(shared)} shared + 2 own lenses"},
            "evals_executed_per_step": int(done), "evals_of_the_plain_batch": int(c.evals),
            "executed_evals_per_s": done / (st["ms_mean"] * 1e-3), "clocks": clk.summary(), "gpu_launches": int(launches),
            "parity_last_step": sampled_parity(torch, c, out, model=c.nmodel - 1, n=300)}
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
            "roofline": {"bound": "hbm", "achieved": 16.0 * g.npix / (ms * 1e-3) / 1e9, "peak": 6545.0, "unit": "GB/s",
                         "frac": 16.0 * g.npix / (ms * 1e-3) / 1e9 / 6545.0,
                         "traffic": NCU_TRAFFIC_DELENS_BYTES if (args.config == 3 and ns == 80) else None,
                         "note": "algorithmic bytes = the two deflection planes read once (16 B per vertex); the found "
                                 "images are a few KB.  A warp owns a tile of 32 x 8 cells, fetches each of its 33 x 9 vertices "
                                 "once and keeps only the sources inside the box of their source-plane images (usually none; "
                                 "32-bit monotone keys, redux.sync), so what is left is streaming the planes: ncu reads 268.5 MB "
                                 "of DRAM for 268.4 MB algorithmic (profiles/r03_next_rows_ncu.md); "
                                 "peak = MEASURED_PEAKS.json hbm_gbs (copy bandwidth, of measured)"},
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
    if a.shared and a.impl != "reference":
        run_shared(a)
        raise SystemExit(0)
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
