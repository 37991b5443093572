#!/usr/bin/env python
"""bench.py -- cells advanced through dt_cfd per second (BASELINE.json's metric) on N B200s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--cells n] [--impl reference]

A "step" is one pass of the whole hot path (rows a1-a7) over one batch of synthetic cells:
one `stev_integrate` call that takes every cell from t = 0 to t = dt_cfd.  The default workload is BASELINE.json's
config 3 (1,048,576 cells, 53 species / 325 reactions, MLP cp/h), the configuration the north star's target is stated
on.  State is resident in HBM when the timed region starts and is restored from a pristine device copy between steps
(outside the CUDA-event pairs).  Under torchrun every rank integrates its own interleaved shard of an N-times larger
field (weak scaling; cells are independent, so there is no data-path collective); the time is the max
over ranks.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "cells advanced through dt_cfd per second"
UNIT = "cells/s"


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index 0..4 (default 3: the target config)")
    ap.add_argument("--cells", type=int, default=None, help="cells per GPU (default: the config's full size)")
    ap.add_argument("--impl", default="stev", choices=["stev", "reference"])
    ap.add_argument("--chunk-steps", type=int, default=0)
    ap.add_argument("--max-steps", type=int, default=None,
                    help="override the per-cell step cap (profiling runs only: cuts the 200000-step tail cells short; the "
                         "line then reports finished_fraction < 1)")
    ap.add_argument("--lanes", type=int, default=0)
    ap.add_argument("--order", type=int, default=1, help="stev_params.order_cells (include/stev.h): 1 default, 0 index order, "
                                                          "2 hottest first cell by cell, 3 hottest first in groups of four")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--ref-cells", type=int, default=None, help="cells per step of the --impl reference arm")
    ap.add_argument("--state-precision", default="f64", choices=["f64", "f32"],
                    help="f32: stev_params.state_precision = STEV_STATE_FP32 (PAPER.md:428); reported with dtype f32, beside the f64 headline")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config object (the other BASELINE.json configs at full size)")
    ap.add_argument("--per-config-budget", type=float, default=330.0,
                    help="seconds since start after which config 4 at full size (one call of about two minutes) is skipped")
    ap.add_argument("--what", default="integrate", choices=["integrate", "estimator"],
                    help="estimator: time the standalone MLP forward pass (row a7) of config 3/4 on the fp32, TF32 and BF16 paths")
    return ap.parse_args()


# ----------------------------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region (B200_PROFILING.md "clocks line")
# ----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        self.path = f"/tmp/stev_clocks_{os.getpid()}.csv"
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                parts = [x.strip() for x in line.split(",")]
                if len(parts) < 7:
                    continue
                try:
                    sm.append(float(parts[0]))
                    smax.append(float(parts[1]))
                    power.append(float(parts[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, parts[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=float(max(power)))
        return out


# ----------------------------------------------------------------------------------------------------------------
def oracle_time(w, n_cells: int, n_threads: int | None = None):
    """Times the CPU oracle, as it stands, on the first n_cells of workload w.  Returns (cells/s, seconds, cell_steps, threads)."""
    from oracle import stev_oracle
    n = min(n_cells, w.n_cells)
    t0 = time.perf_counter()
    r = stev_oracle.integrate(w.mech, w.estimator, w.params, w.T[:n], w.p[:n], np.ascontiguousarray(w.Y[:, :n]), w.dt_cfd,
                              n_threads=n_threads)
    dt = time.perf_counter() - t0
    return n / dt, dt, int(r["steps"].sum()), r["n_threads"]


def run_reference(args):
    """The reference arm of this tier IS the oracle: plain CPU fp64 STEV on the box's host cores, bounded sample."""
    rank = _env_int("RANK", 0)
    if rank != 0:
        return 0
    from stev_inputs.configs import make_workload, FULL_CELLS
    from oracle import stev_oracle
    stev_oracle.build()
    cores = os.cpu_count() or 1
    per_step = args.ref_cells or {0: 4096, 1: 256, 2: 256, 3: 32 * cores, 4: 128}[args.config]
    w = make_workload(args.config, per_step * (args.steps + args.warmup))
    times, steps_total = [], 0
    for s in range(args.warmup + args.steps):
        lo = s * per_step
        sub = type(w)(config=w.config, name=w.name, mech=w.mech, estimator=w.estimator, params=w.params, dt_cfd=w.dt_cfd,
                      T=w.T[lo:lo + per_step], p=w.p[lo:lo + per_step], Y=np.ascontiguousarray(w.Y[:, lo:lo + per_step]),
                      blocks=w.blocks)
        cps, dt, cs, thr = oracle_time(sub, per_step, cores)
        if s >= args.warmup:
            times.append(dt)
            steps_total += cs
    total = sum(times)
    value = per_step * args.steps / total
    sample = f"{per_step} cells per step (consecutive seeded cells of {w.name}), {args.steps} steps"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "cells_full": FULL_CELLS[args.config], "cells_per_step": per_step,
                       "species": w.mech.n_species, "reactions": w.mech.n_reactions, "dt_cfd": w.dt_cfd},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample,
                             "cell_steps_per_s": steps_total / total},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------------------------
def run_estimator(args):
    """Row a7 on its own (BASELINE.json config 4: 'run on the tensor-core (TF32/BF16) path vs the fp32 CUDA-core path'):
    one step = one stev_estimator_eval call over all cells of the config; inputs and outputs resident in HBM."""
    import torch
    import paper_1905_09395_b200 as stev
    from stev_inputs.configs import make_workload, FULL_CELLS
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device")
    stev.load()
    config = args.config if args.config in (3, 4) else 4
    n = FULL_CELLS[config] if args.cells is None else args.cells
    w = make_workload(config, n)
    e = w.estimator
    est = stev.Estimator(None, e)
    dev = torch.device("cuda:0")
    X = torch.empty((n, e.n_in), dtype=torch.float32, device=dev)
    X[:, 0] = torch.tensor(w.T, dtype=torch.float32, device=dev)
    if e.n_in > 1:
        X[:, 1] = torch.tensor(w.p, dtype=torch.float32, device=dev)
        X[:, 2:] = torch.tensor(w.Y.T, dtype=torch.float32, device=dev)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    bytes_per_call = 4 * n * (e.n_in + e.n_out)
    flop_per_call = 2.0 * n * (e.n_in * e.n_hidden + e.n_hidden * e.n_out)
    stream = torch.cuda.current_stream()
    res = {}
    for name in ("FP32", "TF32", "BF16"):
        prec = getattr(stev, "STEV_PREC_" + name)
        for _ in range(max(args.warmup, 3)):
            out = stev.stev_estimator_eval(est, X, prec)
        ms = []
        for _ in range(max(args.steps, 3)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            out = stev.stev_estimator_eval(est, X, prec)
            e1.record(stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        t = float(np.mean(ms)) * 1e-3
        res[name] = {"ms": 1e3 * t, "cells_per_s": n / t, "hbm_gbs": bytes_per_call / t / 1e9,
                     "hbm_frac_of_measured": bytes_per_call / t / 1e9 / hbm_peak, "tflops": flop_per_call / t / 1e12}
        del out
    best = max(("TF32", "BF16"), key=lambda k: res[k]["cells_per_s"])
    line = {"metric": "cells evaluated per second by the standalone MLP estimator (row a7)", "value": res[best]["cells_per_s"],
            "unit": "cells/s", "n_gpus": 1, "steps": max(args.steps, 3), "warmup": max(args.warmup, 3),
            "ms_per_step": res[best]["ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": best.lower(), "data": "synthetic",
            "config": {"workload": f"{w.name}: estimator {e.n_in}-{e.n_hidden}-{e.n_out}", "cells": n,
                       "l2": f"inputs + outputs {bytes_per_call >> 20} MiB, larger than L2"},
            "paths": res, "gpu_launches": max(args.steps, 3),
            "roofline": {"bound": "hbm", "kernel": "estimator_tc_kernel", "achieved": res[best]["hbm_gbs"], "peak": hbm_peak,
                         "unit": "GB/s", "frac": res[best]["hbm_frac_of_measured"], "traffic": None,
                         "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "fallback 6650 GB/s (of fallback)",
                         "bytes_per_cell": 4 * (e.n_in + e.n_out)}}
    print(json.dumps(line), flush=True)
    return 0


def measure_config(stev, workmodel, config: int, n: int, dev, sm_max: float, warmup: int = 1, state_precision: int = 0,
                   max_steps=None) -> dict:
    """One BASELINE.json config at n cells with the default kernel selection: `warmup` untimed calls, one timed call
    (CUDA events on the launching stream, state restored from a pristine copy outside the events)."""
    import torch
    from stev_inputs.configs import make_workload
    w = make_workload(config, n)
    mech = stev.Mechanism(w.mech)
    est = stev.Estimator(mech, w.estimator) if w.estimator is not None else None
    params = dict(w.params)
    if max_steps is not None:
        params["max_steps"] = max_steps
    prm = stev.stev_params_default(state_precision=state_precision, **params)
    T0 = torch.tensor(w.T, dtype=torch.float64, device=dev)
    p = torch.tensor(w.p, dtype=torch.float64, device=dev)
    Y0 = torch.tensor(w.Y, dtype=torch.float64, device=dev)
    T, Y = torch.empty_like(T0), torch.empty_like(Y0)
    steps = torch.zeros(n, dtype=torch.int32, device=dev)
    status = torch.zeros(n, dtype=torch.uint8, device=dev)
    ws = torch.empty(max(stev.stev_workspace_bytes(mech, est, prm, n), 256), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    ms = 0.0
    for k in range(warmup + 1):
        T.copy_(T0)
        Y.copy_(Y0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        rc = stev.stev_integrate(mech, est, prm, T, p, Y, w.dt_cfd, steps, status, workspace=ws, stream=stream)
        e1.record(stream)
        e1.synchronize()
        ms = e0.elapsed_time(e1)
    st = stev.stev_last_stats()
    cell_steps = int(steps.cpu().numpy().astype(np.int64).sum())
    work = workmodel.cell_step_work(w.mech, w.estimator, dft_enable=bool(w.params["dft_enable"]),
                                    first_high_bin=w.params["dft_first_high_bin"], alpha_on=w.params["alpha"] > 0,
                                    adiabatic=w.params["energy_mode"] == 0)
    peak = 2.0 * workmodel.fp64_peak_instr_per_s(sm_max) * (2.0 if state_precision else 1.0)
    return {"workload": w.name, "cells": n, "ms_per_call": ms, "cells_per_s": n / (ms * 1e-3),
            "cell_steps_per_s": cell_steps / (ms * 1e-3), "mean_steps_per_cell": cell_steps / n,
            "finished_fraction": float((status == 0).float().mean().item()), "return_code": rc,
            "kernel_lanes_per_cell": st["lanes_per_cell"], "specialised": st["specialised"],
            "dtype": "f32" if state_precision else "f64", "warmup_calls": warmup,
            "frac": work.fp64_flop * cell_steps / (ms * 1e-3) / peak,
            "frac_of": "fp32 FMA peak (2 x the fp64 rate)" if state_precision else "derived fp64 peak"}


def measure_estimator_paths(stev, dev, hbm_peak: float) -> dict:
    """Row a7 on its own (config 4's estimator over all 4,194,304 cells): fp32 CUDA cores, TF32 and BF16 tcgen05."""
    import torch
    from stev_inputs.configs import make_workload, FULL_CELLS
    n = FULL_CELLS[4]
    w = make_workload(4, 4096)
    e = w.estimator
    est = stev.Estimator(None, e)
    g = torch.Generator(device=dev).manual_seed(4)
    X = torch.rand((n, e.n_in), dtype=torch.float32, device=dev, generator=g)
    X[:, 0] = 1000.0 + 1500.0 * X[:, 0]
    X[:, 1] = 1.0e6 * (1.0 + 4.0 * X[:, 1])
    bytes_per_call = 4 * n * (e.n_in + e.n_out)
    stream = torch.cuda.current_stream()
    out = {}
    for name in ("FP32", "TF32", "BF16"):
        prec = getattr(stev, "STEV_PREC_" + name)
        for _ in range(3):
            stev.stev_estimator_eval(est, X, prec)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(3):
            stev.stev_estimator_eval(est, X, prec)
        e1.record(stream)
        e1.synchronize()
        t = e0.elapsed_time(e1) / 3 * 1e-3
        out[name.lower()] = {"ms": 1e3 * t, "cells_per_s": n / t, "hbm_gbs": bytes_per_call / t / 1e9,
                             "hbm_frac": bytes_per_call / t / 1e9 / hbm_peak}
    out["cells"] = n
    out["shape"] = f"{e.n_in}-{e.n_hidden}-{e.n_out}"
    return out


def main():
    t_start = time.perf_counter()
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.what == "estimator":
        return run_estimator(args)

    import torch
    import paper_1905_09395_b200 as stev
    from paper_1905_09395_b200 import multi, workmodel
    from stev_inputs.configs import make_workload, FULL_CELLS

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle arm)")
    ctx = multi.init(args.gpus)
    rank, world, dev = ctx.rank, ctx.world, ctx.device
    stev.load()

    n = FULL_CELLS[args.config] if args.cells is None else args.cells
    w = make_workload(args.config, n, rank=rank, world=world, weak=True)
    S = w.mech.n_species
    mech = stev.Mechanism(w.mech)
    est = stev.Estimator(mech, w.estimator) if w.estimator is not None else None
    params = dict(w.params)
    if args.max_steps is not None:
        params["max_steps"] = args.max_steps
    f32 = args.state_precision == "f32"
    prm = stev.stev_params_default(chunk_steps=args.chunk_steps, lanes_per_cell=args.lanes, order_cells=args.order,
                                   state_precision=1 if f32 else 0, **params)

    T0 = torch.tensor(w.T, dtype=torch.float64, device=dev)
    p = torch.tensor(w.p, dtype=torch.float64, device=dev)
    Y0 = torch.tensor(w.Y, dtype=torch.float64, device=dev)
    T, Y = torch.empty_like(T0), torch.empty_like(Y0)
    steps = torch.zeros(n, dtype=torch.int32, device=dev)
    status = torch.zeros(n, dtype=torch.uint8, device=dev)
    ws = torch.empty(max(stev.stev_workspace_bytes(mech, est, prm, n), 256), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def one_step(timed: bool):
        T.copy_(T0)
        Y.copy_(Y0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        rc = stev.stev_integrate(mech, est, prm, T, p, Y, w.dt_cfd, steps, status, workspace=ws, stream=stream)
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), rc, stev.stev_last_stats()

    for _ in range(max(args.warmup, 0)):
        one_step(False)

    # fp64 throughput probes for the roofline denominator (outside the timed region)
    dfma_per_s = stev.stev_microbench(0, 4096)
    cexp_per_s = stev.stev_microbench(1, 512)

    multi.barrier(ctx)
    torch.cuda.synchronize()
    sampler = ClockSampler(ctx.local_rank) if rank == 0 else None
    t_wall0 = time.perf_counter()
    ms, launches, rc = [], 0, 0
    for _ in range(args.steps):
        m, rc, st = one_step(True)
        ms.append(m)
        launches += st["kernel_launches"]
    torch.cuda.synchronize()
    multi.barrier(ctx)
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop() if sampler else None

    total_ms = multi.max_over_ranks(ctx, float(sum(ms)))
    steps_h = steps.cpu().numpy().astype(np.int64)
    status_h = status.cpu().numpy()
    cell_steps_rank = int(steps_h.sum())
    finished_rank = int((status_h == 0).sum())
    cell_steps_all = multi.sum_over_ranks(ctx, cell_steps_rank)
    finished_all = multi.sum_over_ranks(ctx, finished_rank)
    ms_per_step = total_ms / args.steps
    value = world * n / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        Th0 = torch.tensor(w.T, dtype=torch.float64).pin_memory()
        ph = torch.tensor(w.p, dtype=torch.float64).pin_memory()
        Yh0 = torch.tensor(w.Y, dtype=torch.float64).pin_memory()
        Th, Yh = torch.empty_like(Th0).pin_memory(), torch.empty_like(Yh0).pin_memory()
        sh = torch.zeros(n, dtype=torch.int32).pin_memory()
        sth = torch.zeros(n, dtype=torch.uint8).pin_memory()
        reps = max(1, min(args.steps, 2))
        tt = []
        for k in range(1 + reps):
            Th.copy_(Th0)
            Yh.copy_(Yh0)
            multi.barrier(ctx)
            t0 = time.perf_counter()
            stev.stev_integrate_host(mech, est, prm, Th, ph, Yh, w.dt_cfd, sh, sth)
            dt = time.perf_counter() - t0
            if k > 0:
                tt.append(dt)
        e2e_s = multi.max_over_ranks(ctx, float(sum(tt))) / reps
        same = bool(np.array_equal(sh.numpy(), steps_h) and np.array_equal(Yh.numpy(), Y.cpu().numpy()))
        e2e = {"value": world * n / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 8 * n * (2 + S),
               "d2h_bytes_per_step": 8 * n * (1 + S) + 5 * n, "steps": reps, "ms_per_step": 1e3 * e2e_s,
               "matches_device_path_bitwise": same, "api": "stev_integrate_host (pinned host buffers)"}

    if rank != 0:
        multi.finish(ctx)
        return 0

    # ---- roofline of the dominant kernel (the integrator: one launch per step when chunk_steps = 0)
    work = workmodel.cell_step_work(w.mech, w.estimator, dft_enable=bool(w.params["dft_enable"]),
                                    first_high_bin=w.params["dft_first_high_bin"], alpha_on=w.params["alpha"] > 0,
                                    adiabatic=w.params["energy_mode"] == 0)
    kernel_s = (sum(ms) / args.steps) * 1e-3  # CUDA events on the launching stream around the launch(es) of one step
    flop = work.fp64_flop * cell_steps_rank
    instr = work.fp64_instr * cell_steps_rank
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_instr = workmodel.fp64_peak_instr_per_s(sm_max)
    peak_tflops = 2.0 * peak_instr / 1e12
    kernel_name = {512: "stev_ls_kernel (lock-step block, DFT history in tensor memory)",
                   513: "stev_ls_kernel<LsDyn> (lock-step block, run-time dimensions)"}.get(st["lanes_per_cell"],
                                                                             f"stev_integrate_kernel<{st['lanes_per_cell']}>")
    # DRAM bytes of one launch from ncu (dram__bytes_read.sum + dram__bytes_write.sum), known only for the captured
    # workloads: profiles/r1_groups_cfg3.md (config 3 at full size, default kernel, by launch order)
    # not measured by this run (ncu is not running): the DRAM bytes of the dominant kernel are in profiles/ per capture
    traffic = None
    roofline = {"bound": "alu", "kernel": kernel_name,
                "achieved": flop / kernel_s / 1e12, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": flop / kernel_s / 1e12 / peak_tflops, "traffic": traffic,
                "traffic_source": "null here; ncu captures of this kernel and workload: profiles/r2_traffic_cfg3.md",
                "peak_source": f"derived: 148 SM x 64 DFMA/clk x 2 x {sm_max:.0f} MHz (DESIGN.md section 8); not in MEASURED_PEAKS.json",
                "fp64_instr": {"achieved_per_s": instr / kernel_s, "peak_per_s": peak_instr,
                               "frac": instr / kernel_s / peak_instr, "measured_dfma_per_s": dfma_per_s,
                               "frac_of_measured_dfma": instr / kernel_s / dfma_per_s,
                               "measured_contract_exp_per_s": cexp_per_s},
                "per_cell_step": {"fp64_fma": work.fma, "fp64_other": work.other, "fp32_fma": work.fp32_fma,
                                  "hbm_bytes": 0},
                "cell_steps_per_launch": cell_steps_rank / max(1, st["passes"]),
                "hbm_bytes_per_launch": n * (8 * (2 + S) + 8 * (1 + S) + 5)}

    cpu_baseline = None
    if not args.no_cpu_baseline and not f32:
        cores = os.cpu_count() or 1
        n_s = {0: 4096, 1: 4096, 2: 2048, 3: 768 * cores, 4: 1024}[args.config]   # about 10-30 s of oracle time
        n_s = min(n_s, n)
        cps, dt, cs, thr = oracle_time(w, n_s, cores)
        cpu_baseline = {"value": cps, "unit": UNIT, "cores": thr, "kind": "oracle",
                        "sample": f"first {n_s} cells of this rank's field, {dt:.1f} s", "cell_steps_per_s": cs / dt}

    per_config = None
    if world == 1 and not args.no_per_config and args.config == 3 and args.cells is None and args.lanes == 0 and args.max_steps is None and not f32:
        # the other BASELINE.json configs at full size (1 warm-up + 1 timed call each; config 4 -- one call takes about two
        # minutes -- last, without warm-up, and only inside the wall-clock budget), and row a7 on its own
        per_config = {}
        from stev_inputs.configs import FULL_CELLS as _FULL
        for c in (0, 1, 2):
            per_config[str(c)] = measure_config(stev, workmodel, c, _FULL[c], dev, sm_max)
        per_config["3"] = {"workload": w.name, "cells": n, "ms_per_call": ms_per_step, "cells_per_s": value,
                           "cell_steps_per_s": cell_steps_all / (ms_per_step * 1e-3), "finished_fraction": finished_all / (world * n),
                           "frac": roofline["frac"], "dtype": "f64", "kernel_lanes_per_cell": st["lanes_per_cell"]}
        try:
            per_config["3_f32"] = measure_config(stev, workmodel, 3, 262144, dev, sm_max, state_precision=1)
        except Exception as ex:   # the binary32 state path may refuse a mechanism
            per_config["3_f32"] = {"unavailable": str(ex)[:200]}
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        per_config["estimator_a7"] = measure_estimator_paths(stev, dev, float(peaks.get("hbm_gbs", 6650.0)))
        if time.perf_counter() - t_start < args.per_config_budget:
            per_config["4"] = measure_config(stev, workmodel, 4, _FULL[4], dev, sm_max, warmup=0)
        else:
            per_config["4"] = {"skipped": f"wall-clock budget of {args.per_config_budget:.0f} s used up before config 4"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32" if f32 else "f64",
            "data": "synthetic",
            "config": {"workload": w.name, "cells_per_gpu": n, "species": S, "reactions": w.mech.n_reactions,
                       "reversible": w.mech.n_reversible, "dt_cfd": w.dt_cfd,
                       "estimator": None if w.estimator is None else f"mlp {w.estimator.n_in}-{w.estimator.n_hidden}-{w.estimator.n_out} fp32",
                       "parallelism": f"cells sharded over {world} GPU(s), no collective",
                       "l2": f"inputs larger than L2 ({(8 * n * (2 + S)) >> 20} MiB of state per GPU, restored between steps)",
                       "chunk_steps": args.chunk_steps, "max_steps": params["max_steps"], "lanes_per_cell": st["lanes_per_cell"],
                       "threads_per_block": st["threads_per_block"], "blocks": st["blocks"], "smem_bytes": st["smem_bytes"]},
            "cell_steps_per_s": cell_steps_all / (ms_per_step * 1e-3), "mean_steps_per_cell": cell_steps_all / (world * n),
            "finished_fraction": finished_all / (world * n), "return_code": rc,
            "wall_s_timed_region": t_wall, "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "per_config": per_config}
    print(json.dumps(line), flush=True)
    multi.finish(ctx)
    return 0


if __name__ == "__main__":
    sys.exit(main())
