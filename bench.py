#!/usr/bin/env python
"""bench.py — DG+HABC node-updates/s on B200 (BASELINE.json metric), with roofline and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--precision 64|32] [--impl reference]

One "step" = one full time step (5 LSRK stages, every kernel of SURVEY §8(a)) over the whole synthetic mesh.
N>1 (torchrun): independent replicas, one per GPU ("replicas only") — weak scaling, no collective
on the data path.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import CONFIGS, make_workload  # noqa: E402

METRIC = "DG+HABC node-updates/sec"
UNIT = "node-updates/s"
# measured on this pool's B200 with a DFMA / DMMA / FFMA microbenchmark (profiles/r01_peaks.md; the probe's source is a
# working file, no longer tracked): DFMA 36.98,
# DMMA 37.19 TFLOP/s (the same fp64 unit; the mixed DMMA+DFMA loop of that probe reaches 33.5), FFMA 71.2
FP64_TFLOPS_MEASURED = 37.0
FP32_TFLOPS_MEASURED = 71.2
HBM_FALLBACK_GBS = 6650.0


def algorithmic_bytes_per_element(N: int, precision: int) -> float:
    """per element and LSRK stage the 3D kernel must move q,res in and out (16 Np values), the
    neighbours' face traces (4 fields x 4 Nfp values), 24 geometric/material values, and 20 B of connectivity."""
    Np, Nfp = (N + 1) * (N + 2) * (N + 3) // 6, (N + 1) * (N + 2) // 2
    return (precision // 8) * (16 * Np + 16 * Nfp + 24) + 20


def algorithmic_flops_per_element(N: int) -> float:
    """DESIGN.md §7 (minimal operation count): 6 matvec rows per node (12 Np flop), 24 flop to form the
    contravariant velocity and combine the gradient, LIFT on one flux scalar per face node (8 Nfp per node),
    ~14 flop per face node for the flux, 40 per node for the face combination + update."""
    Np, Nfp = (N + 1) * (N + 2) * (N + 3) // 6, (N + 1) * (N + 2) // 2
    return Np * (12 * Np + 24 + 8 * Nfp + 40) + 4 * Nfp * 14


def habc_work_per_launch(N: int, J: int, T: int, E: int, C: int, precision: int) -> dict:
    """DESIGN.md §7, HABC levels: algorithmic (bytes, flops) of ONE launch (one LSRK stage) of each auxiliary kernel.
    Counts follow the arrays each kernel must touch: state and residual in and out, the closure sums, the neighbour /
    parent traces, the per-cell records and tables; the small inverse matrices are counted once per launch."""
    sz, Nfp, N1 = precision // 8, (N + 1) * (N + 2) // 2, N + 1
    return {
        "face2d": (T * (J * (12 * Nfp + 9 * N1) * sz + (Nfp + 3 * N1 + 23) * sz + 4 * (3 + 3 * N1)),
                   T * J * (Nfp * (8 * Nfp + 6 * N1 + 30) + 3 * N1 * 14)),
        "edge1d": (E * (J * J * (8 * N1 + 6) * sz + (2 * J * N1 + 8) * sz + 8),
                   E * J * J * (N1 * (4 * N1 + 16) + 28)),
        "close_face": (T * (Nfp * (J + 10) * sz + 16), T * Nfp * (2 * J + 12)),
        "close_edge": (E * N1 * (J * J + 10 * J) * sz + 8 * J * J * sz, E * N1 * (14 * J * J + 12 * J)),
        "close_corner": (C * 9 * J * J * sz + 9 * J ** 4 * sz, C * (18 * J ** 4 + 12 * J * J)),
    }


def sweep(local: int, hbm_peak: float) -> dict:
    """BASELINE.json configs[3]: the 82,944-tet mesh at J = 4, N = 1..8, both precisions, per kernel: device time per
    launch, algorithmic GB/s and TFLOP/s, fraction of the slower roof.  The 3D kernel is timed inside a replayed step
    (dg_options.time_kernels), the auxiliary kernels by dg_profile_step (a host sync per launch, outside any timed
    region)."""
    import torch
    from paper_1610_05023_b200 import Solver
    cells = []
    sampler = ClockSampler(local)
    sampler.start()
    for N in range(1, 9):
        w = make_workload("cfg4", N=N, J=4)
        for prec in (64, 32):
            s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, precision=prec, device=local, time_kernels=True)
            x, y, z = s.get_nodes()
            cn = np.repeat(w.c[:, None], s.Np, axis=1)
            s.set_initial(*w.fields(x, y, z, cn, 1.0))
            s.step(3)
            nst = 5
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(s.stream):
                e0.record(s.stream)
                s.step(nst)
                e1.record(s.stream)
            s.synchronize()
            ms_step = e0.elapsed_time(e1) / nst
            k3 = float(np.mean(s.last_step_kernel_ms()))
            prof = s.profile_step()
            alu_peak = FP64_TFLOPS_MEASURED if prec == 64 else FP32_TFLOPS_MEASURED

            def row(name, ms, nbytes, nflops):
                t_roof = max(nbytes / (hbm_peak * 1e9), nflops / (alu_peak * 1e12))
                return {"kernel": name, "us": 1e3 * ms, "GBs": nbytes / (ms * 1e-3) / 1e9,
                        "TFLOPs": nflops / (ms * 1e-3) / 1e12, "frac": t_roof / (ms * 1e-3)}
            rows = [row(s.info["kernel_name"], k3, algorithmic_bytes_per_element(N, prec) * s.K,
                        algorithmic_flops_per_element(N) * s.K)]
            names = {"face2d": "k_face2d_mma" if prec == 64 and N <= 5 else "k_face2d", "edge1d": "k_edge1d",
                     "close_face": "k_close_face", "close_edge": "k_close_edge", "close_corner": "k_close_corner"}
            for key, (nbytes, nflops) in habc_work_per_launch(N, w.J, s.T, s.E, s.C, prec).items():
                rows.append(row(names[key], prof[key] / 5.0, nbytes, nflops))
            cells.append({"N": N, "J": w.J, "dtype": f"f{prec}", "K": s.K, "ms_per_step": ms_step,
                          "node_updates_per_s": s.K * s.Np / (ms_step * 1e-3), "kernels": rows})
            s.close()
            del s
    sampler.stop_flag = True
    return {"workload": "cfg4 (82,944 tets), J = 4, N = 1..8", "steps_per_cell": 5, "warmup_per_cell": 3,
            "units": {"us": "per launch", "GBs": "algorithmic bytes / time", "TFLOPs": "algorithmic flops / time",
                      "frac": "slower-roof time / time (HBM peak below; ALU 37.0 / 71.2 TFLOP/s)"},
            "hbm_peak_GBs": hbm_peak, "clocks": sampler.summary(), "cells": cells}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.01)

    def summary(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def oracle_sample(workload: str, precision: int, budget_s: float = 20.0):
    """Time the oracle (as it stands) on a bounded sample of the workload: same N, J, materials rule, pulse, on a
    coarser hex grid (n=8), for as many steps as fit the budget.  Returns (node-updates/s, description, cores)."""
    from oracle.solver import OracleSolver
    d = CONFIGS[workload]
    n = min(d["n"], 8)
    w = make_workload(workload, n=n)
    o = OracleSolver(w.verts, w.tets, w.N, w.J, w.c, w.rho, face_bc=w.face_bc)
    x = o.nodes()
    cn = np.repeat(w.c[:, None], x.shape[1], axis=1)
    o.set_initial(np.stack(w.fields(x[..., 0], x[..., 1], x[..., 2], cn, 1.0)))
    o.step(1)
    steps, t0, cpu0 = 0, time.perf_counter(), time.process_time()
    while True:
        o.step(1)
        steps += 1
        el = time.perf_counter() - t0
        if el > budget_s or steps >= 50:
            break
    nodes = o.H.tet.K * o.H.tet.ref.Np
    # threads the numpy oracle really kept busy: process CPU time over wall time of the timed loop
    cpu = time.process_time() - cpu0
    cores = max(1, int(round(cpu / el)))
    avail = len(os.sched_getaffinity(0))
    desc = (f"{workload} rule on a {'x'.join(str(m) for m in w.shape)} hex grid ({o.H.tet.K} tets, N={w.N}, J={w.J}), "
            f"{steps} steps, fp64 numpy; cores = CPU time / wall time = {cpu / el:.2f} of {avail} available")
    return nodes * steps / el, desc, cores, el / steps, avail


def workload_config(name: str, w) -> dict:
    """The part of `config` that names the workload as it is really run: the GPU arm at full size, the --impl reference arm
    on the bounded sample the oracle times (with `sample_of` naming the full configuration)."""
    Np = (w.N + 1) * (w.N + 2) * (w.N + 3) // 6
    return {"workload": name, "n_hex": w.n, "hex_grid": list(w.shape), "N": w.N, "J": w.J, "K": w.K, "nodes": w.K * Np}


def roofline(s, w, prec: int, prof: dict, workload: str, kernel_ms) -> dict:
    """Roofline object of the dominant kernel (the fused 3D stage): algorithmic bytes / flops per launch
    over its launch time INSIDE the timed region -- CUDA events recorded on the solver's stream before and after the
    kernel of each of the five stages of the last timed step, inside the replayed graph (dg_options.time_kernels) --
    against the measured peaks.  `prof` (dg_profile_step, outside the timed region, a host sync after every launch)
    gives the per-kernel split of a step."""
    vol_ms = float(np.mean(kernel_ms))                            # per launch
    bytes_launch = algorithmic_bytes_per_element(w.N, prec) * s.K
    flops_launch = algorithmic_flops_per_element(w.N) * s.K
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", HBM_FALLBACK_GBS))
    alu_peak = FP64_TFLOPS_MEASURED if prec == 64 else FP32_TFLOPS_MEASURED
    hbm = {"bound": "hbm", "achieved": bytes_launch / (vol_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
           "peak_source": "MEASURED_PEAKS.json" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md)"}
    hbm["frac"] = hbm["achieved"] / hbm["peak"]
    alu = {"bound": "alu", "achieved": flops_launch / (vol_ms * 1e-3) / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
           "peak_source": "profiles/r01_peaks.md (DFMA / DMMA / FFMA microbenchmark on this pool: 37.0 / 37.2 / 71.2)"}
    alu["frac"] = alu["achieved"] / alu["peak"]
    t_mem, t_alu = bytes_launch / (hbm_peak * 1e9), flops_launch / (alu_peak * 1e12)
    roof = dict(hbm if t_mem >= t_alu else alu)
    roof.update({"kernel": s.info["kernel_name"], "ms_per_launch": vol_ms,
                 "ms_per_launch_source": "CUDA events around the kernel in the 5 stages of a step, recorded in the replayed graph on the solver's stream, in a short second timed run right after the headline one (which runs without the event nodes)",
                 "ms_per_launch_stages": [float(x) for x in kernel_ms], "ms_per_launch_profiled": prof["vol3d"] / 5.0,
                 "traffic": None, "traffic_source": None,
                 "roof_ms": 1e3 * max(t_mem, t_alu), "frac_of_slower_roof": max(t_mem, t_alu) / (vol_ms * 1e-3),
                 "hbm": hbm, "alu": alu, "kernel_share_of_step": prof["vol3d"] / max(sum(prof.values()), 1e-12),
                 "per_kernel_ms_per_step": prof})
    traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")     # from the ncu --set full captures under profiles/
    if os.path.exists(traffic_file):
        for ln in open(traffic_file).read().splitlines()[1:]:
            cols = ln.split(",", 3)
            if len(cols) == 4 and cols[0] == f"{workload}_f{prec}" and cols[2] == s.info["kernel_name"]:
                roof["traffic"] = float(cols[1])
                roof["traffic_source"] = f"static: ncu --set full capture of {cols[2]} recorded in profiles/traffic.csv ({cols[3]}); not measured in this run"
    return roof


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    per_step_budget = 6.0
    vals = []
    for _ in range(args.warmup + args.steps):
        v, desc, cores, step_s, avail = oracle_sample(args.workload, 64, budget_s=per_step_budget)
        vals.append((v, step_s))
    vals = vals[args.warmup:]
    value = float(np.mean([v for v, _ in vals]))
    n_sample = min(CONFIGS[args.workload]["n"], 8)                    # what oracle_sample really times
    w = make_workload(args.workload, n=n_sample)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean([s for _, s in vals])),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload_config(args.workload, w), sample_of=args.workload,
                           note="the numpy oracle times a bounded sample: this config's rule on the smaller grid named here, not the full-size mesh of the GPU arm",
                           parallelism="host CPU, rank 0 only"),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "cores_available": avail, "kind": "oracle",
                             "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def measure(args, w, prec: int, rep, local: int) -> dict:
    """One precision: set the problem up, time `steps` steps device-resident, the per-kernel times and roofline, and
    the end-to-end run through the C ABI with host buffers."""
    import torch
    from paper_1610_05023_b200 import Solver

    world = rep.world
    t_setup = time.perf_counter()
    s = Solver(w.verts, w.tets, w.N, w.J, w.c, w.rho, precision=prec, device=local, kernel=args.kernel, face_bc=w.face_bc)
    x, y, z = s.get_nodes()
    cn = np.repeat(w.c[:, None], s.Np, axis=1)
    fields = [np.ascontiguousarray(f) for f in w.fields(x, y, z, cn, 1.0)]
    del x, y, z
    s.set_initial(*fields)
    t_setup = time.perf_counter() - t_setup
    nodes = s.K * s.Np
    barrier = rep.barrier

    # ---- device-resident throughput
    s.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(s.stream):
        ev0.record(s.stream)
        s.step(args.steps)
        ev1.record(s.stream)
    barrier()
    sampler.stop_flag = True
    ms = rep.max_over_ranks(ev0.elapsed_time(ev1))
    value = world * nodes * args.steps / (ms * 1e-3)

    # ---- the dominant kernel inside a step: a second, short timed run with dg_options.time_kernels on (10 event-record
    #      nodes per step in the replayed graph).  The headline above runs without them; both step times are reported.
    s.set_time_kernels(True)
    s.step(1)                                                      # capture + one untimed replay
    nk = max(3, min(args.steps, 5))
    evk0, evk1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(s.stream):
        evk0.record(s.stream)
        s.step(nk)
        evk1.record(s.stream)
    s.synchronize()
    ms_step_events = evk0.elapsed_time(evk1) / nk
    kernel_ms = s.last_step_kernel_ms()                            # the 3D kernel inside the last of those steps
    s.set_time_kernels(False)

    # ---- per-kernel device time (outside the timed region): the dominant kernel's roofline
    prof = {k: 0.0 for k in ("vol3d", "face2d", "edge1d", "close_face", "close_edge", "close_corner")}
    nprof = 3
    for _ in range(nprof):
        for k, v in s.profile_step().items():
            prof[k] += v / nprof
    roof = roofline(s, w, prec, prof, args.workload, kernel_ms)
    roof["ms_per_step_with_kernel_events"] = ms_step_events
    roof["kernel_share_of_step"] = 5.0 * float(np.mean(kernel_ms)) / ms_step_events      # from the in-step events
    roof["kernel_share_of_step_profiled"] = prof["vol3d"] / max(sum(prof.values()), 1e-12)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of the four fp64 fields, the steps, D2H of
    #      the four fields, all inside the timed region
    pin_in = torch.empty((4, s.K, s.Np), dtype=torch.float64, pin_memory=True)
    pin_out = torch.empty((4, s.K, s.Np), dtype=torch.float64, pin_memory=True)
    host_in, host_out = pin_in.numpy(), pin_out.numpy()
    for i in range(4):
        host_in[i] = fields[i]
    del fields
    barrier()
    t0 = time.perf_counter()
    s.set_initial(host_in[0], host_in[1], host_in[2], host_in[3])
    s.step(args.steps)
    q, _, _ = s.get_fields(aux=False, out=host_out)
    e2e_s = rep.max_over_ranks(time.perf_counter() - t0)
    h2d = 4 * nodes * 8                                            # the C ABI takes and returns fp64 arrays
    e2e = {"value": world * nodes * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d / args.steps,
           "d2h_bytes_per_step": h2d / args.steps, "seconds": e2e_s,
           "what": "dg_set_initial(pinned host fp64) + dg_step(steps) + dg_get_fields(pinned host fp64), wall clock"}
    finite = bool(np.isfinite(q).all())
    launches = s.launches_per_step * args.steps
    info = dict(s.info)
    s.close()
    del s, pin_in, pin_out, host_in, host_out, q
    torch.cuda.empty_cache()
    return {"value": value, "ms_per_step": ms / args.steps, "roofline": roof, "e2e": e2e, "gpu_launches": launches,
            "clocks": sampler.summary(),
            "run": {"T": info["T"], "E": info["E"], "corners": info["C"], "dt": info["dt"], "setup_s": t_setup,
                    "finite": finite, "kernel": info["kernel_name"], "launches_per_step": info["launches_per_step"]}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--precision", type=int, default=64)
    ap.add_argument("--n", type=int, default=None, help="override hexes per side (debug only; invalidates the metric)")
    ap.add_argument("--N", type=int, default=None, help="override the polynomial degree (degree sweep of configs[3])")
    ap.add_argument("--J", type=int, default=None, help="override the HABC order (degree sweep of configs[3])")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--kernel", type=int, default=0, help="dg_options.kernel (0 = the library's choice)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the run in the other precision")
    ap.add_argument("--no-sweep", action="store_true", help="skip the per-kernel degree sweep of configs[3]")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_1610_05023_b200.replicas import Replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    rep = Replicas.from_env("nccl")
    rank, world, local = rep.rank, rep.world, rep.local
    torch.cuda.set_device(local)

    w = make_workload(args.workload, n=args.n, N=args.N, J=args.J)
    prec = args.precision
    first = measure(args, w, prec, rep, local)
    line = {"metric": METRIC, "value": first["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": first["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": f"f{prec}", "data": "synthetic",
            "config": dict(workload_config(args.workload, w), parallelism="replicas only" if world > 1 else "single GPU",
                           l2="state (q,res) exceeds L2 many times over; no flush needed"),
            "run": first["run"], "node_stages_per_s": 5 * first["value"], "roofline": first["roofline"],
            "e2e": first["e2e"], "gpu_launches": first["gpu_launches"], "clocks": first["clocks"]}
    if not args.no_secondary:
        # BASELINE.json's metric is quoted "(fp64/fp32)": the same workload, steps and warm-up in the other precision
        other = 32 if prec == 64 else 64
        sec = measure(args, w, other, rep, local)
        line["secondary"] = {"dtype": f"f{other}", "value": sec["value"], "unit": UNIT, "ms_per_step": sec["ms_per_step"],
                             "roofline": sec["roofline"], "e2e": sec["e2e"], "gpu_launches": sec["gpu_launches"],
                             "clocks": sec["clocks"], "run": sec["run"]}
    if world == 1 and args.workload == "cfg5" and not args.no_sweep:
        line["sweep"] = sweep(local, first["roofline"]["hbm"]["peak"])
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, desc, cores, _, avail = oracle_sample(args.workload, prec)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "cores_available": avail, "kind": "oracle",
                                "sample": desc}
    if rank == 0:
        print(json.dumps(line))
    rep.close()


if __name__ == "__main__":
    main()
