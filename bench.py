#!/usr/bin/env python
"""bench.py -- one JSON line for the per-cell thermochemistry update (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch of synthetic cells:
df_thermo_T_from_h -> df_thermo_properties -> df_chem_ann_source (bf16 21-1600-800-400-19 MLP)
on BASELINE.json configs[2] (the headline: 2,097,152 cells, K = 19), through the C ABI.  The same line carries
  kernels   one roofline entry per kernel of that step (T_from_h: hbm, properties: alu, ann_bf16: tensor),
  fp32_peak the FFMA-chain peak measured in this run (df_probe_fp32_peak), next to the nominal figure,
  configs   short timed runs of the other BASELINE configs (1, 2, 4, 5) with their own roofline fractions,
  e2e       the step through df_step_host with pinned HOST buffers,
  cpu_baseline  the fp64 oracle on the host cores (bounded sample).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cells n] [--impl reference] [--no-configs]

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
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x FP32 lanes x 2 (FMA) x clocks.max.sm = 74.45


def props_flops(K: int) -> float:
    """minimum-formulation flops per cell of the property pass, F(K) = 12.5 K^2 + 51.5 K + 10."""
    return 12.5 * K * K + 51.5 * K + 10.0



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




# ---- DRAM traffic per launch from the committed ncu export -------------------------------------
NCU_RAW = os.path.join(ROOT, "profiles", "r2_ncu_raw.csv")   # `ncu -i ... --page raw --csv`, see profiles/r2_summary.md
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def ncu_traffic(kernel_substr: str, grid_x=None):
    """dram__bytes_read.sum + dram__bytes_write.sum of the captured launch of `kernel_substr` whose grid is grid_x
    blocks (None: its largest captured grid), read from the committed ncu raw-page export (wide CSV: a header row, a
    units row, one row per launch).  None when the export or the launch is not there."""
    import csv
    if not os.path.exists(NCU_RAW):
        return None
    with open(NCU_RAW, newline="") as f:
        rows = [r for r in csv.reader(f) if r]
    best, cols, units, skip = None, None, None, False
    for r in rows:          # the file is several exports one after the other: every header row resets the columns
        if "Kernel Name" in r:
            try:
                cols = (r.index("Kernel Name"), r.index("Grid Size"), r.index("dram__bytes_read.sum"), r.index("dram__bytes_write.sum"))
            except ValueError:
                cols = None
            skip = True     # the row after a header holds the units
            continue
        if skip:
            units, skip = r, False
            continue
        if cols is None or units is None:
            continue
        ck, cg, cr, cw = cols
        if len(r) <= max(cols) or kernel_substr not in r[ck]:
            continue
        try:
            gx = int(r[cg].strip("() ").split(",")[0])
            val = (float(r[cr].replace(",", "")) * _UNIT.get(units[cr], 1.0)
                   + float(r[cw].replace(",", "")) * _UNIT.get(units[cw], 1.0))
        except ValueError:
            continue
        if grid_x is not None and gx == grid_x:
            return val
        if grid_x is None and (best is None or gx > best[0]):
            best = (gx, val)
    return best[1] if best else None


def make_inputs(n: int, rank: int):
    """Seeded synthetic cfg3 fields (DESIGN.md input recipe); rank shifts the cell seed only."""
    from paper_2312_05800_b200 import synth
    seed = synth.config_seed(CFG)
    mech = synth.make_mechanism(19, seed)
    ann = synth.make_ann(19, HIDDEN, 1, seed)
    cells = synth.cells_stratified(19, n, seed + 1000 * rank)
    return mech, ann, cells


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _oracle_step(om, oa, cells, h32):
    T32 = om.T_from_h(h32, cells.Y, cells.T_guess).astype(np.float32)
    om.properties(T32, cells.p, cells.Y)
    oa.source(om, T32, cells.p, cells.Y)


def _oracle_setup(ns):
    """The oracle as it stands (oracle/oracle.cpp, never tuned), compiled for THIS host: g++ -O3 -march=native
    -ffp-contract=off (the tests use the portable -O2 build of the same source)."""
    from oracle import oracle
    oracle.use_native_build()
    mech, ann, cells = make_inputs(ns, 0)
    om, oa = oracle.Mech(mech), oracle.Ann(ann)
    _, h = om.mixture_cp_h(cells.T, cells.Y)
    return oracle, om, oa, cells, h.astype(np.float32)


def run_reference(args):
    """The oracle timed on the host cores on a bounded sample of the same workload (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # bounded sample per step: about 2e6 cell-updates in total (~2 minutes on 16 cores), never above --ref-cells
    ns = max(4096, min(args.ref_cells, int(2.0e6 / max(1, args.steps + args.warmup))))
    oracle, om, oa, cells, h32 = _oracle_setup(ns)
    for _ in range(args.warmup):
        _oracle_step(om, oa, cells, h32)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_step(om, oa, cells, h32)
    dt = (time.perf_counter() - t0) / args.steps
    val = ns / dt
    cores = oracle.get_threads()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"configs[2] sample: {ns} of 2097152 cells, K=19, T_from_h+properties+MLP 21-1600-800-400-19"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{ns} cells per step (the full config is 2097152)",
                         "build": oracle.build_flags(), "cpu": cpu_model()},
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
    """cpu_baseline leg: the fp64 oracle on a bounded sample of the workload, all host cores, plus the same on one
    thread over 1/64 of the sample (rank 0, N = 1 only)."""
    oracle, om, oa, cells, h32 = _oracle_setup(ns)
    cores = oracle.get_threads()
    t0 = time.perf_counter()
    _oracle_step(om, oa, cells, h32)
    dt = time.perf_counter() - t0
    n1 = max(1024, ns // 64)
    from paper_2312_05800_b200 import synth
    sub = synth.Cells(n1, cells.T[:n1], cells.p[:n1], np.ascontiguousarray(cells.Y[:, :n1]), cells.T_guess[:n1])
    oracle.set_threads(1)
    t0 = time.perf_counter()
    _oracle_step(om, oa, sub, h32[:n1])
    dt1 = time.perf_counter() - t0
    oracle.set_threads(cores)
    return {"value": ns / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {ns} cells of the workload, one pass, {dt:.1f} s",
            "one_thread": {"value": n1 / dt1, "unit": UNIT, "sample": f"first {n1} cells, one pass, {dt1:.1f} s"},
            "build": oracle.build_flags(), "cpu": cpu_model()}


# ---- GPU legs ---------------------------------------------------------------------------------------
def _median_launch_ms(torch, stream, launch, reps, before=None, warm=3):
    """Median and minimum CUDA-event time of `launch`, each launch bracketed by its own pair of events on the
    launching stream; `before` (untimed) restores in/out arguments, e.g. the Newton guess."""
    ts = []
    for i in range(warm + reps):
        if before is not None:
            before(i)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        launch(i)
        b.record(stream)
        torch.cuda.synchronize()
        if i >= warm:
            ts.append(a.elapsed_time(b))
    return float(np.median(ts)), float(np.min(ts))


def measure_fp32_peak(torch, B, stream):
    """FFMA-chain peak of this board, now: scalar FFMA and packed FFMA2 variants."""
    out = {}
    blocks, iters = 148 * 16, 1024     # ~2.5 ms per launch: a burst, like the kernels it is the denominator of
    for name, variant in (("ffma", 0), ("ffma2", 1)):
        flops = [0.0]

        def launch(_i):
            flops[0] = B.df_probe_fp32_peak(variant, blocks, iters)
        med, mn = _median_launch_ms(torch, stream, launch, reps=10, warm=2)
        out[name] = flops[0] / (mn * 1e-3) / 1e12
        out[name + "_median"] = flops[0] / (med * 1e-3) / 1e12
    out["measured"] = max(out["ffma"], out["ffma2"])
    # issue rates behind the property kernels' pair loops: time per warp-iteration and SMSP of eight
    # MUFU.RCP, and of the pair loop's mix (2 MUFU.RCP + 6 FFMA2), in units of one FFMA2 of the same run and in clocks under
    # the architectural figure MUFU.RCP = 8 clocks per warp and SMSP (4 lanes per clock)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    iblocks, iiters = sms * 4, 20000          # 16 warps per SM: 4 per SMSP
    per = {}
    for name, variant in (("mufu8", 2), ("pair_mix", 3)):
        wi = [0.0]

        def launch_i(_i):
            wi[0] = B.df_probe_fp32_peak(variant, iblocks, iiters)
        _med, mn = _median_launch_ms(torch, stream, launch_i, reps=5, warm=1)
        per[name] = mn * 1e-3 / (wi[0] / (sms * 4))          # seconds per warp-iteration on one SMSP
    t_ffma2 = 128.0 / (out["ffma2"] * 1e12 / (sms * 4))       # seconds per warp-wide FFMA2 (64 FMA = 128 flop) on one SMSP
    t_mufu = per["mufu8"] / 8.0
    out["issue"] = {"mufu_rcp_per_ffma2": t_mufu / t_ffma2, "pair_mix_per_ffma2": per["pair_mix"] / t_ffma2,
                    "clk_if_mufu_is_8": {"ffma2": 8.0 * t_ffma2 / t_mufu, "pair_mix_2mufu_6ffma2": 8.0 * per["pair_mix"] / t_mufu},
                    "how": "df_probe_fp32_peak variants 2, 3: 4 warps per SMSP, 20000 iterations, best of 5"}
    out["nominal"] = FP32_NOMINAL_TFLOPS
    out["unit"] = "TFLOP/s"
    out["how"] = ("df_probe_fp32_peak: 148 x 16 blocks x 256 threads, 16 register-only dependent FMA chains per thread "
                  "x 1024 iterations (~2.5 ms bursts), best of 10 (CUDA events); nominal = 148 SM x 128 lanes x 2 x 1.965 GHz")
    return out


def alu_entry(kernel, flops_per_cell, n, ms, fp32, extra=None):
    ach = flops_per_cell * n / (ms * 1e-3) / 1e12
    e = {"kernel": kernel, "bound": "alu", "achieved": ach, "peak": fp32["measured"], "unit": "TFLOP/s",
         "frac": ach / fp32["measured"], "frac_vs_nominal": ach / fp32["nominal"], "ms": ms,
         "peak_source": "FP32 FMA peak measured in this run (fp32_peak.measured)",
         "algorithmic": f"{flops_per_cell:.0f} flop/cell x {n} cells/launch"}
    e.update(extra or {})
    return e


def hbm_entry(kernel, bytes_per_cell, n, ms, pk, extra=None):
    ach = bytes_per_cell * n / (ms * 1e-3) / 1e9
    e = {"kernel": kernel, "bound": "hbm", "achieved": ach, "peak": pk["hbm"], "unit": "GB/s", "frac": ach / pk["hbm"],
         "ms": ms, "peak_source": f"{pk['src']} HBM copy bandwidth",
         "algorithmic": f"{bytes_per_cell} B/cell x {n} cells/launch"}
    e.update(extra or {})
    return e


def bench_configs(torch, B, stream, pk, fp32, quick=False):
    """Short timed runs of BASELINE configs 1, 2, 4, 5 (the headline is configs[2] = cfg3)."""
    from paper_2312_05800_b200 import synth
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = {}

    # ---- cfg1: 4096 cells, K = 9, fp32 MLP 11-64-64-9: launch-latency bound, reported in microseconds per call ----
    mech, ann, cells = synth.make_config(1)
    gm, ga = B.Mech(mech), B.Ann(ann)
    n, K = cells.n, mech.K
    T0, p, Y, Tg = dev(cells.T), dev(cells.p), dev(cells.Y), dev(cells.T_guess)
    h = torch.empty(n, device="cuda")
    B.df_thermo_properties(gm, T0, p, Y, h=h)
    T, cp, mu, lam = (torch.empty(n, device="cuda") for _ in range(4))
    D, om = torch.empty(K, n, device="cuda"), torch.empty(K, n, device="cuda")
    t1, _ = _median_launch_ms(torch, stream, lambda i: B.df_thermo_T_from_h(gm, h, Y, T), 20, before=lambda i: T.copy_(Tg))
    t2, _ = _median_launch_ms(torch, stream, lambda i: B.df_thermo_properties(gm, T, p, Y, cp=cp, mu=mu, lam=lam, D=D), 20)
    t3, _ = _median_launch_ms(torch, stream, lambda i: B.df_chem_ann_source(ga, gm, T, p, Y, omega=om), 20)
    # the same step as ONE CUDA-graph launch (df_step_plan / df_thermochem_step, NEXT-2), and as three calls back to back
    plan = B.StepPlan(gm, ga, h, p, Y, T, T_guess=Tg, cp=cp, mu=mu, lam=lam, D=D, omega=om)
    tg_, _ = _median_launch_ms(torch, stream, lambda i: plan.launch(), 20)

    def three(i):
        T.copy_(Tg)
        B.df_thermo_T_from_h(gm, h, Y, T)
        B.df_thermo_properties(gm, T, p, Y, cp=cp, mu=mu, lam=lam, D=D)
        B.df_chem_ann_source(ga, gm, T, p, Y, omega=om)
    t3c, _ = _median_launch_ms(torch, stream, three, 20)
    plan.close()
    out["cfg1"] = {"workload": "configs[0]: 4096 cells, K=9, T_from_h + properties + fp32 MLP 11-64-64-9",
                   "us_per_call": {"T_from_h": 1e3 * t1, "properties": 1e3 * t2, "ann_fp32": 1e3 * t3},
                   "us_per_step": {"three_calls": 1e3 * t3c, "one_graph_launch": 1e3 * tg_},
                   "cells_per_s": n / (tg_ * 1e-3), "note": "launch-latency bound (problem < 1 MB): no roofline fraction"}
    del gm, ga

    # ---- cfg2: 262,144 cells, K = 19, the tensor-path MLP alone; 6 rotating buffer sets (the 42 MB of one set would
    # sit in the 126 MB L2) ----
    mech, ann, cells = synth.make_config(2)
    gm, ga = B.Mech(mech), B.Ann(ann)
    n, K = cells.n, mech.K
    sets = []
    for s_ in range(6):
        sets.append((dev(np.roll(cells.T, 4096 * s_)), dev(cells.p), dev(np.roll(cells.Y, 4096 * s_, axis=1)),
                     torch.empty(K, n, device="cuda")))
    ws = B.alloc_workspace(ga, n)

    def ann_launch(i):
        T_, p_, Y_, o_ = sets[i % len(sets)]
        B.df_chem_ann_source(ga, gm, T_, p_, Y_, omega=o_, workspace=ws)
    med, mn = _median_launch_ms(torch, stream, ann_launch, 12)
    ach = FLOPS_PER_CELL_MLP * n / (med * 1e-3) / 1e12
    out["cfg2"] = {"workload": "configs[1]: 262144 cells, K=19, bf16 MLP 21-1600-800-400-19 alone, 6 rotating buffer sets",
                   "ms": med, "ms_min": mn, "cells_per_s": n / (med * 1e-3),
                   "roofline": {"kernel": "ann_bf16_kernel", "bound": "tensor", "achieved": ach, "peak": pk["bf16"], "unit": "TFLOP/s",
                                "frac": ach / pk["bf16"], "peak_source": f"{pk['src']} bf16 burst (kernel timed alone)",
                                "algorithmic": f"{FLOPS_PER_CELL_MLP} flop/cell x {n} cells/launch",
                                "note": "2048 tiles over 148 CTAs = 13.8 waves: 1 - 13.84/14 = 1.1 % tail"}}
    # ---- NEXT-1: one MLP per species, 19 networks 21-1600-800-400-1 on the same field ----
    nets = synth.make_mmlp(K, HIDDEN, 1, synth.config_seed(2))
    gn = B.AnnMmlp(nets)
    wsm = B.alloc_workspace_mmlp(gn, n, n)

    def mmlp_launch(i):
        T_, p_, Y_, o_ = sets[i % len(sets)]
        B.df_chem_ann_source_mmlp(gn, gm, T_, p_, Y_, omega=o_, workspace=wsm)
    med, mn = _median_launch_ms(torch, stream, mmlp_launch, 4, warm=1)
    fl = K * 2 * (21 * 1600 + 1600 * 800 + 800 * 400 + 400 * 1)
    ach = fl * n / (med * 1e-3) / 1e12
    out["mmlp"] = {"workload": "NEXT-1 (P:79): 19 per-species MLPs 21-1600-800-400-1 on configs[1]'s 262144 cells "
                               "(19 tensor-chain launches + 1 epilogue launch per call)",
                   "ms": med, "ms_min": mn, "cells_per_s": n / (med * 1e-3),
                   "roofline": {"kernel": "ann_bf16_kernel x19", "bound": "tensor", "achieved": ach, "peak": pk["bf16_sust"], "unit": "TFLOP/s",
                                "frac": ach / pk["bf16_sust"], "frac_vs_burst": ach / pk["bf16"],
                                "peak_source": f"{pk['src']} bf16 sustained (a 15 ms back-to-back tensor load)",
                                "algorithmic": f"{fl} flop/cell x {n} cells/call"}}
    del gm, ga, sets, ws, gn, wsm, nets
    torch.cuda.empty_cache()

    # ---- the two pointwise passes of SURVEY 8(f) NEXT-3 / NEXT-4 on the headline field (2,097,152 cells, K = 19) ----
    mech, _, cells = synth.make_config(3)
    gm = B.Mech(mech)
    n, K = cells.n, mech.K
    T0, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    cp, lam, mu = (torch.empty(n, device="cuda") for _ in range(3))
    D = torch.empty(K, n, device="cuda")
    B.df_thermo_properties(gm, T0, p, Y, cp=cp, mu=mu, lam=lam, D=D)
    rho, psi, alpha, s_ = (torch.empty(n, device="cuda") for _ in range(4))
    rhoD, hk = torch.empty(K, n, device="cuda"), torch.empty(K, n, device="cuda")
    med, mn = _median_launch_ms(torch, stream, lambda i: B.df_thermo_extras(gm, T0, p, Y, cp=cp, lam=lam, D=D, rho=rho, psi=psi,
                                                                              alpha=alpha, rhoD=rhoD, hk=hk, s=s_), 8)
    out["extras"] = {"workload": f"df_thermo_extras, {n} cells, K=19: rho, psi, alpha, rhoD[19], hk[19], s",
                     "roofline": hbm_entry("extras_kernel", 8 * (2 * K + 4), n, med, pk, {"ms_min": mn})}
    gen = torch.Generator(device="cuda").manual_seed(5)
    ks = torch.rand(n, device="cuda", generator=gen) * 10 + 0.01
    ep = torch.rand(n, device="cuda", generator=gen) * 1e4 + 0.1
    om0 = torch.randn(K, n, device="cuda", generator=gen) * 50
    om = torch.empty_like(om0)
    kap = torch.empty(n, device="cuda")
    med, mn = _median_launch_ms(torch, stream, lambda i: B.df_chem_pasr_scale(gm, T0, p, Y, mu, ks, ep, 500.0, om, kappa=kap), 8,
                                before=lambda i: om.copy_(om0))
    out["pasr"] = {"workload": f"df_chem_pasr_scale, {n} cells, K=19 (omega scaled in place, kappa written)",
                   "roofline": hbm_entry("pasr_kernel", 4 * (3 * K + 6), n, med, pk, {"ms_min": mn})}
    del gm, T0, p, Y, cp, lam, mu, D, rho, psi, alpha, s_, rhoD, hk, ks, ep, om0, om, kap
    torch.cuda.empty_cache()

    # ---- cfg4: 2,097,152 cells, K = 53, property pass only ----
    mech, _, cells = synth.make_config(4)
    gm = B.Mech(mech)
    n, K = cells.n, mech.K
    T0, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    cp, hh, mu, lam = (torch.empty(n, device="cuda") for _ in range(4))
    D = torch.empty(K, n, device="cuda")
    med, mn = _median_launch_ms(torch, stream, lambda i: B.df_thermo_properties(gm, T0, p, Y, cp=cp, h=hh, mu=mu, lam=lam, D=D),
                                3 if quick else 8)
    out["cfg4"] = {"workload": "configs[3]: 2097152 cells, K=53, properties (cp, h, mu, lambda, D[53])", "ms": med, "ms_min": mn,
                   "cells_per_s": n / (med * 1e-3),
                   "roofline": alu_entry("props_kernel (K=53)", props_flops(K), n, med, fp32,
                                         {"hbm_bytes_per_cell": 4 * (2 * K + 6), "traffic": ncu_traffic("props_group_kernel")})}
    del gm, T0, p, Y, cp, hh, mu, lam, D
    torch.cuda.empty_cache()

    # ---- cfg5: 16,777,216 cells, K = 19, T_from_h (+ cp at the root) on the robustness field, warm and cold guess ----
    mech, _, cells = synth.make_config(5, n=(1 << 21) if quick else None)
    gm = B.Mech(mech)
    n, K = cells.n, mech.K
    Y = dev(cells.Y)
    h = torch.empty(n, device="cuda")
    B.df_thermo_properties(gm, dev(cells.T), None, Y, h=h)
    warm, cold = dev(cells.T_guess), torch.full((n,), 1000.0, device="cuda")
    T, cp = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    res = {}
    for name, g in (("warm", warm), ("cold", cold)):
        med, mn = _median_launch_ms(torch, stream, lambda i: B.df_thermo_T_from_h(gm, h, Y, T, cp=cp, n_unconverged=cnt), 8,
                                    before=lambda i, g=g: T.copy_(g))
        res[name] = hbm_entry("t_from_h kernel (K=19)", 4 * (K + 2) + 8, n, med, pk,
                              {"ms_min": mn, "cells_per_s": n / (med * 1e-3),
                               "max_abs_T_error_vs_drawn_K": float((T - dev(cells.T)).abs().max())})
    out["cfg5"] = {"workload": f"configs[4]: {n} cells, K=19, robustness field (T 250-3500 K, near-pure and 1e-20-trace cells), "
                               "df_thermo_T_from_h with cp written: 4(K+2) B in + T + cp out = 92 B/cell",
                   "unconverged": int(cnt.item()), "warm": res["warm"], "cold": res["cold"]}
    return out


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

    # ---- each kernel of the step timed alone (its own launches back to back, the board not power-limited by the MLP) ----
    time.sleep(1.0)
    alone_ms = {}
    alone_ms["T_from_h"], _ = _median_launch_ms(torch, stream, lambda i: B.df_thermo_T_from_h(gm, dh, dY, dT), 10,
                                                before=lambda i: dT.copy_(dTg))
    alone_ms["properties"], _ = _median_launch_ms(torch, stream,
                                                  lambda i: B.df_thermo_properties(gm, dT, dp, dY, cp=cp, mu=mu, lam=lam, D=D), 10)
    alone_ms["ann_bf16"], _ = _median_launch_ms(torch, stream,
                                                lambda i: B.df_chem_ann_source(ga, gm, dT, dp, dY, omega=om, workspace=ws), 4, warm=1)

    pk = peaks()
    fp32 = measure_fp32_peak(torch, B, stream) if rank == 0 else None

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
    ctx.close()
    del ctx, hh, hp, hg, hY, oT, ocp, omu, olam, oD, oom
    achieved = FLOPS_PER_CELL_MLP * n / (k_ms[2] * 1e-3) / 1e12
    clocks = clk.summary(w0, w1)
    # B200_PROFILING.md: burst peak for a kernel timed alone, sustained peak for one timed inside a long step; the
    # step loop counts as "long" when the power cap was seen active during the timed region
    low = bool(clocks["sm_mhz"] and clocks["sm_max_mhz"] and clocks["sm_mhz"] < 0.95 * clocks["sm_max_mhz"])
    capped = bool({"sw_power_cap", "hw_power_brake_slowdown"} & set(clocks["reasons"])) or low
    peak = pk["bf16_sust"] if capped else pk["bf16"]
    why = "power-limited clocks in the timed region: " + (", ".join(clocks["reasons"]) or "SM clock below 95 % of max")
    peak_src = f"{pk['src']} bf16 {'sustained (' + why + ')' if capped else 'burst'}"
    blocks256 = (n + 255) // 256
    ann_roof = {"bound": "tensor", "kernel": "ann_bf16_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak,
                # dram__bytes_read.sum + dram__bytes_write.sum of one launch at this size, from the committed ncu export
                "traffic": ncu_traffic("ann_bf16_kernel", min(148, (n + 127) // 128)) if n == 2097152 else None,
                "peak_source": peak_src, "frac_vs_burst": achieved / pk["bf16"],
                "frac_vs_sustained": achieved / pk["bf16_sust"],
                "algorithmic": f"{FLOPS_PER_CELL_MLP} flop/cell x {n} cells/launch"}
    a_alone = FLOPS_PER_CELL_MLP * n / (alone_ms["ann_bf16"] * 1e-3) / 1e12
    kernels = {
        # bytes the timed call really moves: h, T guess, Y[19] in; T out (no cp requested in the step)
        "t_from_h": hbm_entry("t_from_h kernel (K=19)", 4 * (K + 2) + 4, n, k_ms[0], pk,
                              {"ms_alone": alone_ms["T_from_h"],
                               "frac_alone": (4 * (K + 2) + 4) * n / (alone_ms["T_from_h"] * 1e-3) / 1e9 / pk["hbm"],
                               "traffic": ncu_traffic("t_from_h", blocks256) if n == 2097152 else None,
                               "note": "2.1 M cells: 184.5 MB per launch; configs.cfg5 has the 16.8 M-cell figure"}),
        "properties": alu_entry("props kernel (K=19)", props_flops(K), n, k_ms[1], fp32,
                                {"ms_alone": alone_ms["properties"],
                                 "frac_alone": props_flops(K) * n / (alone_ms["properties"] * 1e-3) / 1e12 / fp32["measured"],
                                 "frac_alone_vs_nominal": props_flops(K) * n / (alone_ms["properties"] * 1e-3) / 1e12 / fp32["nominal"],
                                 # in the loop the kernel runs at the clock the MLP's power draw leaves (clocks.sm_mhz); the
                                 # measured peak is a full-clock burst: the same fraction with the peak scaled to that clock
                                 "frac_at_loop_clock": (props_flops(K) * n / (k_ms[1] * 1e-3) / 1e12 / fp32["measured"]
                                                        * clocks["sm_max_mhz"] / clocks["sm_mhz"])
                                 if clocks.get("sm_mhz") and clocks.get("sm_max_mhz") else None,
                                 "hbm_bytes_per_cell": 4 * (2 * K + 6),
                                 "traffic": ncu_traffic("props_fixed", None) if n == 2097152 else None}),
        "ann_bf16": dict(ann_roof, ms=k_ms[2], ms_alone=alone_ms["ann_bf16"], frac_alone_vs_burst=a_alone / pk["bf16"]),
    }
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f16 operands (bf16-valued weights) / f32 accumulate; f32 thermo+transport", "data": "synthetic",
        "config": {"workload": f"configs[2]: {n} cells/GPU, K=19, T_from_h -> properties -> bf16 MLP 21-1600-800-400-19",
                   "cells_per_gpu": n, "l2": "inputs (176 MB/step at the full size) exceed the 126 MB L2; no explicit flush",
                   "parallelism": f"replicas x{world} (no collective in the data path)"},
        "kernel_ms": {"T_from_h": k_ms[0], "properties": k_ms[1], "ann_bf16": k_ms[2]},
        "kernel_alone_ms": alone_ms,
        "roofline": ann_roof,
        "kernels": kernels,
        "fp32_peak": fp32,
        "e2e": {"value": world * n / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": 3 * args.steps,
        "clocks": clocks,
    }
    if world == 1 and not args.no_configs:
        del dT0, dp, dY, dh, dTg, dT, cp, mu, lam, D, om, ws
        torch.cuda.empty_cache()
        out["configs"] = bench_configs(torch, B, stream, pk, fp32, quick=args.quick_configs)
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
    ap.add_argument("--no-configs", action="store_true", help="skip the configs block (BASELINE configs 1, 2, 4, 5)")
    ap.add_argument("--quick-configs", action="store_true", help="configs block at reduced repetitions / cfg5 at 2 M cells")
    ap.add_argument("--kernels-alone", action="store_true", help="accepted for compatibility: kernel_alone_ms is always reported")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
