#!/usr/bin/env python
"""bench.py -- one JSON line for the per-cell thermochemistry update (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch of synthetic cells:
df_thermo_T_from_h -> df_thermo_properties -> df_chem_ann_source (bf16 21-1600-800-400-19 MLP)
on BASELINE.json configs[2] (the headline: 2,097,152 cells, K = 19), through the C ABI.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cells n] [--impl reference]

N > 1: launched by torchrun, one rank per GPU, every rank runs the same per-GPU workload on its
own cells (weak scaling; the path has no exchange step, so there is no collective in the data
path), timing = max over ranks of the CUDA-event time between two barriers.
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
sys.path.insert(0, ROOT)

METRIC = "cells/sec for full thermo+transport+ANN-chemistry update"
UNIT = "cells/s"
CFG = 3                      # BASELINE.json configs[2] (1-based numbering in synth.CONFIGS)
FLOPS_PER_CELL_MLP = 3282400  # 2 * (21*1600 + 1600*800 + 800*400 + 400*19)
HIDDEN = [1600, 800, 400]


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm=p["hbm_gbs"], bf16=p["bf16_tflops"], bf16_sust=p["bf16_tflops_sustained"], src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sust=1400.0, src="fallback")  # B200_PROFILING.md


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (profiling recipe)."""
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
    # asked for as well when this driver's nvidia-smi knows them (probed once): they explain a clock below max
    EXTRA = ("hw_power_brake_slowdown", "sync_boost", "applications_clocks_setting")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index
        self.names = self.NAMES

    def _query(self, names):
        return "clocks.sm,clocks.max.sm," + ",".join("clocks_event_reasons." + n for n in names)

    def __enter__(self):
        try:
            probe = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self._query(self.NAMES + self.EXTRA)}",
                                    "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=20)
            if probe.returncode == 0 and probe.stdout.count(",") >= 1 + len(self.NAMES + self.EXTRA):
                self.names = self.NAMES + self.EXTRA
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self._query(self.names)}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except (OSError, subprocess.SubprocessError):
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def __exit__(self, *exc):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except subprocess.TimeoutExpired:
                self.proc.kill()
            self.thr.join(timeout=2)

    def summary(self, t0=0.0, t1=float("inf")):
        """Median SM clock and active throttle reasons over the samples read in [t0, t1] (perf_counter)."""
        sm, mx, reasons = [], 0.0, set()
        for ts, r in self.rows:
            if not (t0 <= ts <= t1 + 0.15):
                continue
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(self.names, r[2:2 + len(self.names)]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def make_inputs(n: int, rank: int):
    """Seeded synthetic cfg3 fields (DESIGN.md input recipe); rank shifts the cell seed only."""
    from paper_2312_05800_b200 import synth
    seed = synth.config_seed(CFG)
    mech = synth.make_mechanism(19, seed)
    ann = synth.make_ann(19, HIDDEN, 1, seed)
    cells = synth.cells_stratified(19, n, seed + 1000 * rank)
    return mech, ann, cells


def run_reference(args):
    """The oracle (as it stands) timed on the host cores on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle
    # bounded sample per step: about 2e6 cell-updates in total (~2 minutes on 16 cores), never above --ref-cells
    ns = max(4096, min(args.ref_cells, int(2.0e6 / max(1, args.steps + args.warmup))))
    mech, ann, cells = make_inputs(ns, 0)
    om, oa = oracle.Mech(mech), oracle.Ann(ann)
    _, h = om.mixture_cp_h(cells.T, cells.Y)
    h32 = h.astype(np.float32)

    def step():
        T = om.T_from_h(h32, cells.Y, cells.T_guess)
        T32 = T.astype(np.float32)
        om.properties(T32, cells.p, cells.Y)
        oa.source(om, T32, cells.p, cells.Y)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    val = ns / dt
    cores = oracle.get_threads()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[2] sample: {ns} of 2097152 cells, K=19, T_from_h+properties+MLP 21-1600-800-400-19"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{ns} cells per step (the full config is 2097152)"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def max_over_ranks(dist, x: float, device="cpu") -> float:
    """Timing rule for N > 1: the slowest rank defines the step (no-op without a process group)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world: int, cells_per_gpu: int, ms_per_step: float) -> float:
    """Whole-job cells/s of `world` replicas that each process cells_per_gpu cells per step (weak scaling)."""
    return world * cells_per_gpu / (ms_per_step * 1e-3)


def cpu_baseline(ns: int):
    """cpu_baseline leg: the fp64 oracle on a bounded sample, all host cores (rank 0, N = 1 only)."""
    from oracle import oracle
    mech, ann, cells = make_inputs(ns, 0)
    om, oa = oracle.Mech(mech), oracle.Ann(ann)
    _, h = om.mixture_cp_h(cells.T, cells.Y)
    h32 = h.astype(np.float32)
    t0 = time.perf_counter()
    T32 = om.T_from_h(h32, cells.Y, cells.T_guess).astype(np.float32)
    om.properties(T32, cells.p, cells.Y)
    oa.source(om, T32, cells.p, cells.Y)
    dt = time.perf_counter() - t0
    return {"value": ns / dt, "unit": UNIT, "cores": oracle.get_threads(), "kind": "oracle",
            "sample": f"first {ns} cells of the workload, one pass, {dt:.1f} s"}


def run_gpu(args):
    import torch
    from paper_2312_05800_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    n, K = args.cells, 19
    mech, ann, cells = make_inputs(n, rank)
    gm, ga = B.Mech(mech), B.Ann(ann)
    # enthalpy field: computed once on the device by the product path itself (setup, untimed)
    dT0, dp, dY = (torch.from_numpy(x).cuda() for x in (cells.T, cells.p, cells.Y))
    dh = torch.empty(n, device="cuda")
    B.df_thermo_properties(gm, dT0, dp, dY, h=dh)
    dTg = torch.from_numpy(cells.T_guess).cuda()
    dT = torch.empty(n, device="cuda")
    cp, mu, lam = (torch.empty(n, device="cuda") for _ in range(3))
    D = torch.empty(K, n, device="cuda")
    om = torch.empty(K, n, device="cuda")
    ws = B.alloc_workspace(ga, n)
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    marks = []

    def step(record: bool):
        dT.copy_(dTg)                      # the previous time step's T as Newton guess (A4)
        e = [ev() for _ in range(4)] if record else None
        if record: e[0].record(stream)
        B.df_thermo_T_from_h(gm, dh, dY, dT)
        if record: e[1].record(stream)
        B.df_thermo_properties(gm, dT, dp, dY, cp=cp, mu=mu, lam=lam, D=D)
        if record: e[2].record(stream)
        B.df_chem_ann_source(ga, gm, dT, dp, dY, omega=om, workspace=ws)
        if record:
            e[3].record(stream)
            marks.append(e)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    t_start, t_end = ev(), ev()
    with ClockSampler(local) as clk:          # started before the warm-up so it is sampling by the timed region
        for _ in range(max(args.warmup, 3)):
            step(False)
        barrier()
        w0 = time.perf_counter()
        t_start.record(stream)
        for _ in range(args.steps):
            step(True)
        t_end.record(stream)
        barrier()
        w1 = time.perf_counter()
    ms = t_start.elapsed_time(t_end)
    ms = max_over_ranks(dist, ms, "cuda")
    ms_step = ms / args.steps
    value = aggregate_value(world, n, ms_step)
    k_ms = [float(np.mean([e[i].elapsed_time(e[i + 1]) for e in marks])) for i in range(3)]

    # ---- optional: each kernel timed alone (its own launches back to back, the board not power-limited by the MLP) ----
    alone_ms = None
    if args.kernels_alone:
        def alone(launch, reps=12):
            ts = []
            for _ in range(reps):
                dT.copy_(dTg)
                a, b = ev(), ev()
                a.record(stream); launch(); b.record(stream)
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            return float(np.median(ts[2:]))
        time.sleep(2.0)
        alone_ms = {"T_from_h": alone(lambda: B.df_thermo_T_from_h(gm, dh, dY, dT))}
        B.df_thermo_T_from_h(gm, dh, dY, dT)
        alone_ms["properties"] = alone(lambda: B.df_thermo_properties(gm, dT0, dp, dY, cp=cp, mu=mu, lam=lam, D=D))
        alone_ms["ann_bf16"] = alone(lambda: B.df_chem_ann_source(ga, gm, dT0, dp, dY, omega=om, workspace=ws), reps=5)

    # ---- e2e: the same step through df_step_host with pinned HOST buffers ----
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hh, hp, hg, hY = pin(dh.cpu().numpy()), pin(cells.p), pin(cells.T_guess), pin(cells.Y)
    oT, ocp, omu, olam = (torch.empty(n).pin_memory() for _ in range(4))
    oD, oom = torch.empty(K, n).pin_memory(), torch.empty(K, n).pin_memory()
    ctx = B.HostCtx(gm, ga, n)
    e2e_steps = max(2, min(args.steps, 5))
    for _ in range(2):
        ctx.step(n, n, hh, hp, hg, hY, T=oT, cp=ocp, mu=omu, lam=olam, D=oD, omega=oom)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.step(n, n, hh, hp, hg, hY, T=oT, cp=ocp, mu=omu, lam=olam, D=oD, omega=oom)   # synchronises inside
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_s = max_over_ranks(dist, e2e_s, "cuda")
    h2d = 4 * n * (3 + K)
    d2h = 4 * n * (4 + 2 * K)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    pk = peaks()
    achieved = FLOPS_PER_CELL_MLP * n / (k_ms[2] * 1e-3) / 1e12
    clocks = clk.summary(w0, w1)
    # B200_PROFILING.md: burst peak for a kernel timed alone, sustained peak for one timed inside a long step; the
    # step loop counts as "long" when the power cap was seen active during the timed region
    low = bool(clocks["sm_mhz"] and clocks["sm_max_mhz"] and clocks["sm_mhz"] < 0.95 * clocks["sm_max_mhz"])
    capped = bool({"sw_power_cap", "hw_power_brake_slowdown"} & set(clocks["reasons"])) or low
    peak = pk["bf16_sust"] if capped else pk["bf16"]
    why = "power-limited clocks in the timed region: " + (", ".join(clocks["reasons"]) or "SM clock below 95 % of max")
    peak_src = f"{pk['src']} bf16 {'sustained (' + why + ')' if capped else 'burst'}"
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f16 operands (bf16-valued weights) / f32 accumulate; f32 thermo+transport", "data": "synthetic",
        "config": {"workload": f"configs[2]: {n} cells/GPU, K=19, T_from_h -> properties -> bf16 MLP 21-1600-800-400-19",
                   "cells_per_gpu": n, "l2": "inputs (176 MB/step at the full size) exceed the 126 MB L2; no explicit flush",
                   "parallelism": f"replicas x{world} (no collective in the data path)"},
        "kernel_ms": {"T_from_h": k_ms[0], "properties": k_ms[1], "ann_bf16": k_ms[2]},
        **({"kernel_alone_ms": alone_ms} if alone_ms else {}),
        "roofline": {"bound": "tensor", "kernel": "ann_bf16_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak,
                     # dram__bytes_read.sum + dram__bytes_write.sum of one launch at the full size (profiles/r1_summary.md)
                     "traffic": 325.7e6 if n == 2097152 else None,
                     "peak_source": peak_src, "frac_vs_burst": achieved / pk["bf16"],
                     "frac_vs_sustained": achieved / pk["bf16_sust"],
                     "algorithmic": f"{FLOPS_PER_CELL_MLP} flop/cell x {n} cells/launch"},
        "e2e": {"value": world * n / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": 3 * args.steps,
        "clocks": clocks,
    }
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.ref_cells)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cells", type=int, default=2097152, help="cells per GPU (default: configs[2])")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-cells", type=int, default=262144, help="cells per oracle pass (cpu_baseline / reference arm)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernels-alone", action="store_true",
                    help="also time each kernel alone (median of its own launches), reported as kernel_alone_ms")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

