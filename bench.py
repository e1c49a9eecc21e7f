#!/usr/bin/env python
"""bench.py -- throughput of the residual + RK3 hot path on the 256^3 Taylor-Green vortex
(BASELINE.json config 3): fp64 grid-point RK-stage updates per second, with the roofline of the
dominant kernel and the CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n 256]

A "step" is one full low-storage RK3 step (3 x {halo fill, residual, stage update} + final halo
fill) of one replica; N > 1 runs N independent replicas ("replicas only": north_star rules out
sharding), one process per GPU under torchrun, timed as the max over ranks.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "fp64 grid-point RK-stage updates/s at 256^3 TGV"
UNIT = "updates/s"
# Algorithmic flop per grid point (restated in DESIGN.md "Roofline"): every add /
# mul / compare / max / div / sqrt = 1 flop, counted on a CSE'd scalar statement of the method.
FLOP_SWEEP = {0: 1256 + 15 + 19, 1: 1356 + 15 + 19,      # WENO-Z5, TENO5: interface + difference + primitives
              2: 1856 + 15 + 19,                          # TENO6: + ~50 per reconstruction (hand count)
              3: 1206 + 15 + 19,                          # WENO-JS5: WENO-Z5 minus tau and the (1 + (.)^2) factors
              4: 90,                                      # central4: 4 stencil points x ~17 flop + combination, per direction
              5: 900}                                     # WENO-Z3: projections as for the 5-point schemes, ~25 per reconstruction
FLOP_VISCOUS = 300
FLOP_RK = 20


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, uuid):
        self.rows = []
        self.proc = None
        self.uuid = uuid

    def start(self):
        try:
            cmd = ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"]
            if self.uuid:
                cmd += ["-i", self.uuid]
            self.proc = subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text()), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0}, "fallback (B200_PROFILING.md)"


def ncu_traffic_bytes(kernel):
    """dram read+write bytes per launch of `kernel` (sweep_x / sweep_y / sweep_z) from the committed
    ncu capture (profiles/dominant_kernel_traffic.txt), if it has one."""
    p = ROOT / "profiles" / "dominant_kernel_traffic.txt"
    try:
        for line in p.read_text().splitlines():
            if line.startswith(f"traffic_bytes_per_launch[{kernel}]="):
                return float(line.split("=", 1)[1])
    except Exception:
        pass
    return None


def cpu_oracle_rate(n, nsteps=1, scheme=1):
    """One RK3 step of the n^3 TGV with the oracle as it stands, all host cores."""
    from oracle import oracle as O
    from paper_2007_14933_b200 import workloads as W
    case = W.tgv(n, scheme=scheme)
    if scheme == W.WENOJS5:
        case.eps = 1e-6
    orc = O.Oracle(**case.physics())
    Q = case.Q0.copy()
    import numpy as np
    dU, R = np.zeros_like(Q), np.zeros_like(Q)
    t0 = time.perf_counter()
    for _ in range(nsteps):
        orc.rk3_step(Q, dU, R, case.dt)
    dt = time.perf_counter() - t0
    assert np.isfinite(Q).all()
    return case.npoints * 3 * nsteps / dt, orc.nthreads, dt


def run_reference(args):
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    n = 64
    for _ in range(args.warmup if args.warmup < 2 else 1):      # the oracle has no warm-up effects worth 3 steps
        cpu_oracle_rate(n)
    times = []
    cores = 1
    for _ in range(args.steps):
        rate, cores, dt = cpu_oracle_rate(n)
        times.append(dt)
    total = sum(times)
    value = n ** 3 * 3 * args.steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "TGV 256^3 TENO5 + central-4 viscous, RK3 (BASELINE.json config 3)",
                   "sample": f"each step = one RK3 step of the same TGV field on {n}^3 points (1/64 of the workload)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{args.steps} RK3 steps of the {n}^3 TGV, OpenMP over grid lines"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def max_over_ranks(ms, device=None):
    """Device time of the slowest rank (replicas only: no data-path collective)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return ms
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_updates_per_s(npoints, steps, world, ms):
    """Whole-job throughput: every replica advanced npoints x 3 stages x steps in the slowest rank's time."""
    return world * npoints * 3 * steps / (ms * 1e-3)


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the osbli hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    from paper_2007_14933_b200 import build as b
    if rank == 0:
        b.build()
    if world > 1:
        dist.barrier()
    from paper_2007_14933_b200 import osbli
    from paper_2007_14933_b200 import workloads as W

    n = args.n
    scheme = {"wenoz5": W.WENOZ5, "teno5": W.TENO5, "teno6": W.TENO6, "wenojs5": W.WENOJS5,
              "central4": W.CENTRAL4, "wenoz3": W.WENOZ3}[args.scheme]
    case = W.tgv(n, scheme=scheme)
    if scheme == W.WENOJS5:
        case.eps = 1e-6                                   # eq. (21)
    sol = osbli.Solver(device=dev, **case.physics())
    hQ = sol.to_padded(case.Q0, pinned_host=True)
    Q = hQ.to(dev)
    Qtmp = sol.empty_state()
    stream = torch.cuda.current_stream(dev)
    state_bytes = int(sol.layout.total_doubles) * 8

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    peak_tflops = sol.measure_fp64_peak() if rank == 0 else 0.0

    for _ in range(max(args.warmup, 3)):
        sol.rk3_step(Q, Qtmp, case.dt)
    barrier()

    # ---- timed region: K steps, inputs resident in HBM (state 0.79 GB >> 126 MB L2) ----------
    props = torch.cuda.get_device_properties(dev)
    uuid = getattr(props, "uuid", None)
    sampler = ClockSampler(f"GPU-{uuid}" if uuid and not str(uuid).startswith("GPU-") else (str(uuid) if uuid else None))
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    l0 = sol.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        sol.rk3_step(Q, Qtmp, case.dt)
    e1.record(stream)
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), dev)
    launches = sol.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    assert bool(torch.isfinite(Q).all()), "state blew up"

    # ---- same K steps again with per-launch events: device time per kernel class ----------------
    sol.profile_begin()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    for _ in range(args.steps):
        sol.rk3_step(Q, Qtmp, case.dt)
    p1.record(stream)
    prof = sol.profile_end()
    ms_prof = p0.elapsed_time(p1)

    # ---- end to end through the C ABI with HOST buffers: H2D + step + D2H every step ------------
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_steps = args.steps
    t0.record(stream)
    for _ in range(e2e_steps):
        sol.advance_host(hQ, Q, Qtmp, case.dt, 1)
    t1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(t0.elapsed_time(t1), dev)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    npts = case.npoints
    value = aggregate_updates_per_s(npts, args.steps, world, ms)
    e2e_value = aggregate_updates_per_s(npts, e2e_steps, world, ms_e2e)

    # dominant kernel = the sweep direction with the largest device time
    dom = max(("sweep_x", "sweep_y", "sweep_z"), key=lambda k: prof[k][0])
    dom_ms, dom_cnt = prof[dom]
    dom_avg_s = dom_ms * 1e-3 / max(dom_cnt, 1)
    # the stage update is fused into the last sweep (z) when no separate update kernel ran
    fused = prof["rk_update"][1] == 0
    flop_point = FLOP_SWEEP[case.scheme] + (FLOP_RK if (fused and dom == "sweep_z") else 0)
    flop_launch = flop_point * npts
    achieved = flop_launch / dom_avg_s * 1e-12
    peaks, peak_src = measured_peaks()
    total_prof_ms = sum(v[0] for v in prof.values())
    step_flop = (3 * FLOP_SWEEP[case.scheme] + FLOP_VISCOUS + FLOP_RK)
    roofline = {
        "bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops if peak_tflops > 0 else None,
        "traffic": ncu_traffic_bytes(dom),
        "peak_source": "fp64 DFMA micro-benchmark run in this process (osbli_measure_fp64_peak); nominal 148 SM x 64 lanes x 2 x 1.965 GHz = 37.2",
        "algorithmic_flop_per_point": flop_point,
        "fused_stage_update": fused,
        "avg_launch_ms": dom_avg_s * 1e3,
        "whole_step_useful_flop_frac": step_flop * value / world * 1e-12 / peak_tflops if peak_tflops > 0 else None,
        "kernel_share_of_step": {k: (v[0] / total_prof_ms if total_prof_ms > 0 else None) for k, v in prof.items()},
        "kernel_ms_per_launch": {k: (v[0] / v[1] if v[1] else None) for k, v in prof.items()},
        "profiled_ms_per_step": ms_prof / args.steps,
        "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src,
    }

    cpu_n = 256 if n >= 256 else n          # one RK3 step of the same field: about 10 s on 16 cores at 256^3
    cpu_rate, cpu_cores, cpu_dt = cpu_oracle_rate(cpu_n, scheme=scheme)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"TGV {n}^3 periodic, {args.scheme.upper()} + central-4 viscous, low-storage RK3, dt={case.dt} "
                               f"(BASELINE.json config {3 if (n == 256 and args.scheme == 'teno5') else ('5' if (n == 512 and args.scheme == 'teno5') else '?')})",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"state {state_bytes / 1e9:.2f} GB per array >> 126 MB L2 (inputs larger than L2)"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 5 * npts * 8, "d2h_bytes_per_step": 5 * npts * 8,
                "ms_per_step": ms_e2e / e2e_steps,
                "api": "osbli_advance_host (interior nodes of the pinned host state -> device, 1 RK3 step, device -> host), every step"},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": cpu_cores, "kind": "oracle",
                         "sample": f"1 RK3 step (3 stage evaluations) of the same TGV on {cpu_n}^3 points, {cpu_dt:.1f} s"},
    }
    print(json.dumps(line))
    sol.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=256, help="grid points per side (256 = BASELINE.json config 3)")
    ap.add_argument("--scheme", default="teno5", choices=["wenoz5", "teno5", "teno6", "wenojs5", "central4", "wenoz3"],
                    help="reconstruction (teno5 = BASELINE.json config 3; the others are side measurements)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
