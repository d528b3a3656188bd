#!/usr/bin/env python
"""bench.py -- MSM energy+forces+potentials+virial particles/s on B200 (BASELINE.json metric).

A "step" is one msm_evaluate over one batch of synthetic input: the whole hot path (sort, pair,
anterpolation, restriction, per-level convolution, top level, prolongation, interpolation,
reductions), all outputs requested. Default workload: BASELINE config 4 at N = 999 999 (fp32), the
largest single-GPU configuration; `--workload` selects another (see workloads.WORKLOAD_NAMES).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

N > 1 (under torchrun): the path does not shard (replicas only), so every
rank evaluates its own replica of the workload; value = N * particles / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
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

METRIC = "msm_energy_forces_particles_per_s"
UNIT = "particles/s"
FLOP_PER_PAIR = 30.0          # r^2, rsqrt, Horner g and g', 4 accumulations
FLOP_PER_CANDIDATE = 9.0      # distance test of a cell-list candidate (pair row)
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965


def derived_alu_peak_tflops(dtype: str) -> float:
    """FP32: 148 SMs x 128 FMA lanes x 2 flop x 1.965 GHz (guide's unit counts and max clock);
    FP64: half the lanes (64 per SM on B200; the DFMA microbenchmark measures ~0.47 of FFMA)."""
    lanes = FP32_LANES if dtype == "f32" else FP32_LANES // 2
    return SM_COUNT * lanes * 2 * SM_MAX_GHZ * 1e-3


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (the recipe's clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def mark(self):
        time.sleep(0.25)              # let nvidia-smi deliver at least one sample under load
        self.first = len(self.rows)

    def start(self):
        self.first = 0
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()

    def snapshot(self):
        """Clocks and throttle reasons of the samples since the last mark()."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        sm, mx, reasons = [], [], set()
        for r in self.rows[min(self.first, max(len(self.rows) - 1, 0)):]:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def count_pairs(w) -> float:
    """Directed in-cutoff pairs of the workload (the pair kernel's algorithmic unit)."""
    import numpy as np
    try:
        from scipy.spatial import cKDTree
        bs = [b if p else 0.0 for b, p in zip(w.box, w.periodic)]
        pos = np.array(w.positions, copy=True)
        for ax in range(3):
            if w.periodic[ax]:
                pos[:, ax] -= w.box[ax] * np.floor(pos[:, ax] / w.box[ax])
                pos[pos[:, ax] >= w.box[ax], ax] = 0.0
        tree = cKDTree(pos, boxsize=bs if any(w.periodic) else None)
        return float(tree.count_neighbors(tree, w.a) - w.n)
    except Exception:
        vol = w.box[0] * w.box[1] * w.box[2]
        return w.n * (w.n - 1) / vol * 4.0 / 3.0 * math.pi * w.a ** 3


def stage_work(stage: str, w, plan, esz: int, pairs: float):
    """Algorithmic work of one stage per evaluation -> (kind, amount): kind 'flop' (ALU-bound
    stages) or 'byte' (HBM-bound stages). Per-unit figures: DESIGN.md "Algorithmic work"."""
    info = plan.info
    n = w.n

    def G(l):
        d = info.grid_dims[l - 1]
        return d[0] * d[1] * d[2]
    nt = info.n_tiled
    if stage == "pair":
        # 30 flop per in-cutoff directed pair + 9 flop per candidate of the a/2 cell
        # scheme (the other particles of the 5^3 cells around a particle's cell)
        nc = info.pair_cells
        cells = 1
        reach = 1
        for ax in range(3):
            cells *= nc[ax]
            reach *= min(5, nc[ax])
        candidates = n * max(reach * n / cells - 1.0, 0.0)
        return "flop", FLOP_PER_PAIR * pairs + FLOP_PER_CANDIDATE * candidates
    if stage == "conv":                                       # 2 T_s flop per grid point and level
        return "flop", sum(2.0 * info.stencil_taps[l - 1] * G(l) for l in range(1, nt))
    if stage == "conv_virial":                                # correlation over the half space of taps
        return "flop", sum(1.0 * info.stencil_taps[l - 1] * G(l) for l in range(1, nt))
    if stage == "filter":
        return "byte", sum(2.0 * esz * G(l) for l in range(1, nt))   # read Q^l, write the filtered copy
    if stage == "sort":
        return "byte", n * (4 * esz) * 2 + n * 4 * 2         # read pos,q; write sorted records; perm
    if stage == "anterpolate":
        return "flop", n * (3 * w.p * 2 * w.p + 2.0 * w.p ** 3)
    if stage == "interpolate":
        return "flop", n * (6 * w.p * 2 * w.p + 8.0 * w.p ** 3)
    if stage == "restrict":
        return "byte", sum(esz * (G(l) + G(l + 1)) for l in range(1, nt))
    if stage == "prolongate":
        return "byte", sum(esz * (G(l + 1) + 2 * G(l)) for l in range(1, nt))
    if stage == "top":
        return "flop", 2.0 * info.top_points ** 2
    return "byte", n * esz * 2.0                              # reduce


def max_over_ranks(ms_total: float, ms_e2e: float, world: int, dev):
    """Device-timed step sums of this rank -> the maximum over all ranks (MAX all-reduce)."""
    import torch
    t = torch.tensor([ms_total, ms_e2e], dtype=torch.float64, device=dev)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0]), float(t[1])


def whole_job_value(world: int, particles: int, steps: int, ms_total: float) -> float:
    """Replicas: every rank evaluated `particles` particles `steps` times in `ms_total` (max over ranks)."""
    return world * particles * steps / (ms_total * 1e-3)


def stored_traffic(kernel: str, workload: str, dtype: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full`
    capture) of the stage's kernel on this workload, from profiles/r2b_dram_traffic.csv; None if
    that kernel / workload pair was not captured."""
    try:
        with open(os.path.join(ROOT, "profiles", "r2b_dram_traffic.csv")) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 4 and c[0] == kernel and c[1] == workload and c[2] == dtype:
                    return float(c[3])
    except Exception:
        pass
    return None


def measure(w, prec, local, dev, steps, warmup, world, flush, sampler=None, full=True):
    """One workload in one precision -> dict(value, ms_per_step, stages, roofline, e2e, ...).

    Three timed regions of `steps` evaluations each, all bracketed the same way (L2 flush outside
    the per-step CUDA-event pair, synchronize on both sides): (1) per-stage event records on (one
    stream, serial) -> `stages` / `roofline`; (2) records off: the library replays its CUDA graph
    with the pair and virial kernels beside the grid pipeline -> `value`; (3) host buffers through
    msm_evaluate_host -> `e2e`. full=False runs (2) only (the sweep points)."""
    import torch
    from paper_2510_05961_b200 import msm
    esz = 4 if prec == "fp32" else 8
    plan = msm.Plan.for_workload(w, prec, device=local)
    dt = plan.torch_dtype
    pos = torch.tensor(w.positions, dtype=dt, device=dev).contiguous()
    q = torch.tensor(w.charges, dtype=dt, device=dev).contiguous()
    F = torch.zeros((w.n, 3), dtype=dt, device=dev)
    V = torch.zeros(w.n, dtype=dt, device=dev)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, per_step=None):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        for s in range(steps):
            flush.fill_(s & 0xFF)                               # L2 flush, outside the event pair
            ev[s][0].record()
            fn()
            ev[s][1].record()
            torch.cuda.synchronize()
            if per_step:
                per_step()
        barrier()
        return sum(a.elapsed_time(b) for a, b in ev)

    res = {"particles": w.n, "dtype": "f32" if prec == "fp32" else "f64"}
    stage_sum, launches, energy = {}, [0], [0.0]
    if full:
        plan.set_profiling(True)          # one cudaEventRecord between stages: per-stage times, live
        for _ in range(warmup):
            plan.evaluate(pos, q, F, V)
        if sampler:
            sampler.mark()                # only samples taken from here on (the timed regions) count

        def collect():
            for k, v in plan.stage_times().items():
                stage_sum[k] = stage_sum.get(k, 0.0) + v
            launches[0] += plan.launch_count()

        def step():
            energy[0], _ = plan.evaluate(pos, q, F, V)          # energy + forces + potentials + virial
        ms_prof = timed(step, collect)
    plan.set_profiling(False)
    for _ in range(warmup):
        plan.evaluate(pos, q, F, V)
    if sampler and not full:
        sampler.mark()
    ms_fast = timed(lambda: plan.evaluate(pos, q, F, V))
    if not full:
        ms_fast, _ = max_over_ranks(ms_fast, 0.0, world, dev)
        res.update({"value": whole_job_value(world, w.n, steps, ms_fast), "ms_per_step": ms_fast / steps,
                    "grids": [list(plan.info.grid_dims[i]) for i in range(plan.info.n_tiled)],
                    "h": float(plan.info.grid_h[0][0]),
                    "grid_points_per_particle": float(np_prod(plan.info.grid_dims[0])) / w.n})
        plan.close()
        return res
    clocks = sampler.snapshot() if sampler else None

    # ---- end-to-end arm: host buffers through msm_evaluate_host, copies inside the timed region
    hpos = torch.tensor(w.positions, dtype=dt).pin_memory()
    hq = torch.tensor(w.charges, dtype=dt).pin_memory()
    hF = torch.zeros((w.n, 3), dtype=dt).pin_memory()
    hV = torch.zeros(w.n, dtype=dt).pin_memory()
    for _ in range(max(1, min(warmup, 3))):
        plan.evaluate_host(hpos, hq, hF, hV)
    ms_e2e = timed(lambda: plan.evaluate_host(hpos, hq, hF, hV))

    # ---- context: the same step without the virial (energy + forces + potentials only)
    for _ in range(3):
        plan.evaluate(pos, q, F, V, True, False)
    ms_nov = timed(lambda: plan.evaluate(pos, q, F, V, True, False))

    ms_prof, ms_e2e = max_over_ranks(ms_prof, ms_e2e, world, dev)
    ms_fast, _ = max_over_ranks(ms_fast, 0.0, world, dev)

    peaks, peak_src = load_peaks()
    dtype = res["dtype"]
    alu_peak = derived_alu_peak_tflops(dtype)
    fma_meas = msm.measure_fma_peak(prec, local)
    pairs = count_pairs(w)
    stages = {}
    for k, v in stage_sum.items():
        ms = v / steps
        kind, amount = stage_work(k, w, plan, esz, pairs)
        if kind == "flop":
            ach = amount / (ms * 1e-3) * 1e-12 if ms > 0 else 0.0
            stages[k] = {"ms": round(ms, 5), "bound": "alu", "achieved": round(ach, 4), "unit": "TFLOP/s",
                         "frac": round(ach / alu_peak, 5)}
        else:
            ach = amount / (ms * 1e-3) * 1e-9 if ms > 0 else 0.0
            stages[k] = {"ms": round(ms, 5), "bound": "hbm", "achieved": round(ach, 2), "unit": "GB/s",
                         "frac": round(ach / peaks["hbm_gbs"], 5)}
    dom = max(stages, key=lambda k: stages[k]["ms"])
    d = stages[dom]
    res.update({
        "value": whole_job_value(world, w.n, steps, ms_fast), "ms_per_step": ms_fast / steps,
        "e2e": {"value": whole_job_value(world, w.n, steps, ms_e2e), "unit": UNIT,
                "h2d_bytes_per_step": w.n * 4 * esz, "d2h_bytes_per_step": w.n * 4 * esz + 64,
                "ms_per_step": ms_e2e / steps},
        "profiled": {"value": whole_job_value(world, w.n, steps, ms_prof), "unit": UNIT,
                     "ms_per_step": ms_prof / steps,
                     "note": "the same K steps with per-stage CUDA-event records, timed the same way just before the "
                             "`value` steps; the library then keeps every kernel on one stream (no pair/virial "
                             "overlap); `stages` and `roofline` come from these steps"},
        "without_virial": {"value": w.n * steps / (ms_nov * 1e-3), "unit": UNIT, "ms_per_step": ms_nov / steps,
                           "note": "rank 0, energy+forces+potentials only; context, not the metric"},
        "roofline": {"kernel": dom, "bound": d["bound"], "achieved": d["achieved"],
                     "peak": round(alu_peak, 2) if d["bound"] == "alu" else peaks["hbm_gbs"], "unit": d["unit"],
                     "frac": d["frac"], "traffic": stored_traffic(dom, w.name, dtype),
                     "traffic_unit": "DRAM bytes per launch, ncu --set full (profiles/r2b_dram_traffic.csv)",
                     "algorithmic": stage_work(dom, w, plan, esz, pairs)[1],
                     "algorithmic_unit": "flop per launch" if d["bound"] == "alu" else "bytes per launch",
                     "peak_source": ("derived: 148 SM x %d lanes x 2 x 1.965 GHz" % (128 if dtype == "f32" else 64))
                     if d["bound"] == "alu" else f"{peak_src} MEASURED_PEAKS.json hbm_gbs",
                     "measured_fma_tflops": round(fma_meas, 2),
                     "share_of_step": round(d["ms"] / (ms_prof / steps), 4),
                     "timed_in": "the profiled K steps (serial, one stream); see `profiled`"},
        "stages": stages, "gpu_launches": launches[0], "energy": energy[0], "clocks": clocks,
        "grids": [list(plan.info.grid_dims[i]) for i in range(plan.info.n_tiled)], "mu": int(plan.info.mu),
    })
    plan.close()
    return res


def batch_bench(local, dev, B=64, steps=10, warmup=3):
    """Section 8(f) rank 2: B systems of config 1's shape (512 charges, open 20 A cube, fp64, p = 4,
    h = 2, a = 6, 3 levels) evaluated one at a time (msm_evaluate, graph replay) and as one batch
    (msm_evaluate_batch): particles/s of both and their ratio; energy + forces + potentials + virial."""
    import numpy as np
    import torch
    from paper_2510_05961_b200 import msm
    cap = 512
    rng = np.random.default_rng(7)
    pos = rng.random((B, cap, 3)) * 20.0
    q = np.tile(np.where(np.arange(cap) % 2 == 0, 1.0, -1.0), (B, 1))
    tp = torch.tensor(pos, device=dev); tq = torch.tensor(q, device=dev)
    F = torch.zeros((B, cap, 3), dtype=torch.float64, device=dev); V = torch.zeros((B, cap), dtype=torch.float64, device=dev)
    n = [cap] * B

    def timed(fn):
        for _ in range(warmup):
            fn()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for s in range(steps):
            ev[s][0].record(); fn(); ev[s][1].record()
            torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev) / steps

    plan = msm.Plan((20.0,) * 3, (0, 0, 0), 2.0, 6.0, 4, 3, "fp64", max_particles=cap, device=local)
    p0, q0, F0, V0 = tp[0].contiguous(), tq[0].contiguous(), F[0], V[0]
    ms_one = timed(lambda: plan.evaluate(p0, q0, F0, V0))
    plan.close()
    batch = msm.Batch(B, (20.0,) * 3, (0, 0, 0), 2.0, 6.0, 4, 3, "fp64", max_particles=cap, device=local)
    ms_batch = timed(lambda: batch.evaluate(n, tp, tq, F, V))
    batch.close()
    return {"systems": B, "particles_per_system": cap, "dtype": "f64", "workload": "cfg1_open512 shape",
            "one_at_a_time": {"ms_per_system": ms_one, "value": cap / (ms_one * 1e-3), "unit": UNIT},
            "batched": {"ms_per_batch": ms_batch, "value": B * cap / (ms_batch * 1e-3), "unit": UNIT},
            "speedup": ms_one * B / ms_batch}


def np_prod(v):
    r = 1
    for x in v:
        r *= int(x)
    return r


def run_ours(args, rank: int, world: int):
    import torch
    from paper_2510_05961_b200.workloads import BASELINE_SWEEP, COMMENSURATE_SERIES, make_workload

    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    w = make_workload(args.workload)
    m = measure(w, w.precision, local, dev, args.steps, args.warmup, world, flush, sampler)
    extras = world == 1 and not args.main_only and args.workload == "cfg4_water1m"
    fp64, sweep = None, None
    if extras:
        # the other half of the metric ("fp64, fp32"): the fp64 config 5 and the timed workload in fp64
        k = max(5, args.steps // 2)
        fp64 = {}
        w5 = make_workload("cfg5_slab100k")
        fp64["cfg5_slab100k"] = measure(w5, "fp64", local, dev, k, args.warmup, world, flush, sampler)
        fp64["cfg4_water1m"] = measure(w, "fp64", local, dev, k, args.warmup, world, flush, sampler)
        # time per evaluation vs N: the four BASELINE points and the commensurate h = 2.09 series
        sweep = {"note": "ms per evaluation (fp32, all outputs, graph replay), L2 flushed between steps; "
                         "BASELINE points have h = 1.94 / 2.09 / 2.25 / 1.68 (power-of-two grids, reading G1), "
                         "the commensurate series has h = 2.09 at every N",
                 "baseline_points": [], "commensurate_h2.09": []}
        for key, names in (("baseline_points", BASELINE_SWEEP), ("commensurate_h2.09", COMMENSURATE_SERIES)):
            for name in names:
                ws = w if name == args.workload else make_workload(name)
                r = measure(ws, "fp32", local, dev, k, args.warmup, world, flush, None, full=False)
                r["workload"] = name
                sweep[key].append(r)
                del ws
    batch = batch_bench(local, dev) if extras else None
    if sampler:
        sampler.stop()
    if rank != 0:
        return None
    out = {
        "metric": METRIC, "value": m["value"], "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": m["ms_per_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": m["dtype"], "data": "synthetic",
        "config": {"workload": args.workload, "particles": w.n, "box": list(w.box), "periodic": list(w.periodic),
                   "p": w.p, "h_target": w.h, "a": w.a, "levels": w.levels, "mu": m["mu"], "grids": m["grids"],
                   "outputs": "energy+forces+potentials+virial", "parallelism": "replicas" if world > 1 else "1gpu",
                   "l2": "256 MiB fill between steps (outside the per-step event pairs)"},
        "e2e": m["e2e"], "profiled": m["profiled"], "without_virial": m["without_virial"],
        "gpu_launches": m["gpu_launches"], "clocks": m["clocks"], "roofline": m["roofline"], "stages": m["stages"],
        "energy": m["energy"],
    }
    if fp64:
        out["fp64"] = fp64
    if sweep:
        out["sweep"] = sweep
    if batch:
        out["batch"] = batch
    if world == 1 and args.grid_microbench > 0:
        peaks, _ = load_peaks()
        out["grid_microbench"] = grid_microbench(args.grid_microbench, local, peaks["hbm_gbs"])
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, 1, 0)[0]
    return out


def grid_microbench(M: int, local: int, hbm_gbs: float):
    """S4/S7 (and the omega' filter of S5) on a grid that does not fit the L2: the same library
    call on a periodic M^3 finest grid (fp32, p = 4, h = 2, a = 9, top grid 8^3) with a few
    particles, per-stage CUDA-event times, against the algorithmic bytes of SURVEY.md 8(d):
    restriction reads G_l and writes G_l / 8, prolongation reads G_l / 8 + G_l and writes G_l, the
    filter reads and writes G_l, summed over the levels."""
    import numpy as np
    import torch
    from paper_2510_05961_b200 import msm
    dev = torch.device("cuda", local)
    L = 2.0 * M
    rng = np.random.default_rng(1)
    n = 20000
    pos = rng.random((n, 3)) * L
    q = rng.uniform(-1, 1, n)
    q -= q.mean()
    levels = int(np.log2(M)) - 2
    plan = msm.Plan((L,) * 3, (1, 1, 1), 2.0, 9.0, 4, levels, "fp32", max_particles=n, device=local)
    tp = torch.tensor(pos, dtype=torch.float32, device=dev)
    tq = torch.tensor(q, dtype=torch.float32, device=dev)
    F = torch.zeros((n, 3), dtype=torch.float32, device=dev)
    V = torch.zeros(n, dtype=torch.float32, device=dev)
    plan.set_profiling(True)
    acc = {}
    reps = 3
    for i in range(2 + reps):
        plan.evaluate(tp, tq, F, V, True, False)
        if i >= 2:
            for k, v in plan.stage_times().items():
                acc[k] = acc.get(k, 0.0) + v / reps
    sum_g = float(sum((M >> l) ** 3 for l in range(levels - 1)))      # points of the levels that have a coarser one
    byts = {"restrict": 4 * sum_g * (1 + 1 / 8), "prolongate": 4 * sum_g * (2 + 1 / 8), "filter": 4 * sum_g * 2}
    out = {"grid": [M, M, M], "dtype": "f32", "p": 4, "levels": levels, "device_mb": round(plan.info.device_bytes / 1e6, 1),
           "peak_gbs": hbm_gbs}
    for k, b in byts.items():
        gbs = b / (acc[k] * 1e-3) / 1e9
        out[k] = {"ms": round(acc[k], 4), "algorithmic_mb": round(b / 1e6, 1), "achieved_gbs": round(gbs, 1),
                  "frac": round(gbs / hbm_gbs, 4)}
    plan.close()
    return out


# The oracle's bounded sample of each workload: same recipe, density and plan parameters, fewer
# particles where the full case would take minutes on the host (the whole 10^6 case is one to two
# minutes per evaluation; every other workload is timed whole).
CPU_SAMPLE = {"cfg4_water1m": "cfg4_water300k", "cfg4_water1m_fp64": "cfg4_water300k",
              "cfg4c_water1920k": "cfg4c_water240k"}


def cpu_baseline(workload: str, steps: int, warmup: int):
    """Time the oracle as it stands (gcc -O2 -fopenmp, fp64) on the host cores."""
    import oracle
    from paper_2510_05961_b200.workloads import make_workload
    sample = CPU_SAMPLE.get(workload, workload)
    w = make_workload(sample)
    orc = oracle.Oracle(w.box, w.periodic, w.h, w.a, w.p, w.levels, mu=4)
    for _ in range(warmup):
        orc.evaluate(w.positions, w.charges, want_virial=True)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        orc.evaluate(w.positions, w.charges, want_virial=True)
        times.append(time.perf_counter() - t0)
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    total = sum(times)
    note = "whole workload" if sample == workload else \
        f"{sample}: {w.n} particles of the same recipe, density and plan parameters"
    return {"value": w.n * steps / total, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{note}; one full oracle evaluation (fp64, all outputs) per step",
            "sample_particles": w.n, "seconds_per_step": total / steps}, w


def run_reference(args, rank: int):
    if rank != 0:
        return None
    cb, w = cpu_baseline(args.workload, args.steps, min(args.warmup, 1))
    return {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": cb["seconds_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "sample": cb["sample"]},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4_water1m")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--main-only", action="store_true",
                    help="skip the fp64 objects and the N sweep of the default run")
    ap.add_argument("--grid-microbench", type=int, default=512,
                    help="finest grid size M (power of two) of the HBM-bound grid-stage measurement; 0 skips it")
    ap.add_argument("--only-grid-microbench", action="store_true", help="print the grid_microbench object alone")
    ap.add_argument("--only-batch", action="store_true", help="print the batch object alone")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.only_grid_microbench:
        print(json.dumps({"grid_microbench": grid_microbench(args.grid_microbench, 0, load_peaks()[0]["hbm_gbs"])}), flush=True)
        return
    if args.only_batch:
        import torch
        torch.cuda.set_device(0)
        print(json.dumps({"batch": batch_bench(0, torch.device("cuda", 0))}), flush=True)
        return
    if args.impl == "reference":
        args.steps = args.steps if args.steps is not None else 2
        args.warmup = args.warmup if args.warmup is not None else 1
        out = run_reference(args, rank)
    else:
        args.steps = args.steps if args.steps is not None else 20
        args.warmup = max(3, args.warmup if args.warmup is not None else 5)
        out = run_ours(args, rank, world)
    if out is not None:
        print(json.dumps(out), flush=True)
    if world > 1 and args.impl == "ours":
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
