#!/usr/bin/env python
"""bench.py -- throughput of the residual + RK3 hot path on the 256^3 Taylor-Green vortex
(BASELINE.json config 3): fp64 grid-point RK-stage updates per second, with the roofline of the
dominant kernel and the CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3|4|5]
                  [--n 256 --scheme teno5 --perturb 0.0   (side measurements on the TGV path)]

--config 3 (default) is the headline: BASELINE.json config 3, 256^3 TGV, TENO5 + viscous.  --config 5 is the same
at 512^3, --config 4 the curvilinear shock / boundary-layer slab (WENO-Z5, Sutherland, walls); same JSON schema.
`--gpus N` does not spawn ranks: for N > 1 launch under torchrun (`python -m torch.distributed.run --nnodes=1
--nproc-per-node N --master-addr 127.0.0.1 ... bench.py --gpus N`), one replica per GPU.

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
              5: 900,                                     # WENO-Z3: projections as for the 5-point schemes, ~25 per reconstruction
              6: 2300}                                    # WENO-Z7: 8-point projections, ~110 per reconstruction (hand count)
FLOP_VISCOUS = 300
FLOP_RK = 20
# Curvilinear grids (config 4): SURVEY.md 8(d) estimates "metric products add ~25 %" and 5500 flop per point-stage
# in total: sweep = 1.25 x the Cartesian count, viscous (chain rule, Sutherland, closures) = the remainder.
CURV_FACTOR = 1.25
FLOP_VISCOUS_CURV = 5500 - 3 * round(CURV_FACTOR * (1256 + 15 + 19)) - FLOP_RK
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 * 1e-12          # SMs x fp64 lanes x 2 x max SM clock


def make_case(args):
    """The workload: (case, metrics or None, label, BASELINE.json config number or None)."""
    from paper_2007_14933_b200 import workloads as W
    schemes = {"wenoz5": W.WENOZ5, "teno5": W.TENO5, "teno6": W.TENO6, "wenojs5": W.WENOJS5,
               "central4": W.CENTRAL4, "wenoz3": W.WENOZ3, "wenoz7": W.WENOZ7}
    if args.config == 4:
        case = W.sbli_slab()
        label = ("SBLI slab 500x250x8 curvilinear, WENO-Z5 + central-4 viscous (Sutherland), isothermal wall / Dirichlet / "
                 f"extrapolation / periodic, low-storage RK3, dt={case.dt} (BASELINE.json config 4)")
        return case, W.approximate_metrics(case), label, 4
    n = 512 if args.config == 5 else args.n
    scheme = schemes[args.scheme]
    case = W.tgv(n, scheme=scheme)
    if scheme == W.WENOJS5:
        case.eps = 1e-6                                   # eq. (21)
    if args.perturb > 0.0:
        case.Q0 = W.perturb(case, seed=5, amp=args.perturb)
    cfg = 3 if (n == 256 and args.scheme == "teno5" and args.perturb == 0.0) else (5 if (n == 512 and args.scheme == "teno5" and args.perturb == 0.0) else None)
    label = (f"TGV {n}^3 periodic, {args.scheme.upper()} + central-4 viscous, low-storage RK3, dt={case.dt}"
             + (f", state perturbed by {args.perturb} (side measurement: non-smooth data)" if args.perturb > 0.0 else "")
             + (f" (BASELINE.json config {cfg})" if cfg else " (side measurement, not a BASELINE.json config)"))
    return case, None, label, cfg


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


def executed_fp64_from_profiles(kernel):
    """Executed fp64 instructions per point of `kernel` from the committed ncu capture (profiles/r2_measured_ai.txt:
    smsp__sass_thread_inst_executed_op_dadd/dmul/dfma_pred_on per launch), static like `traffic`."""
    p = ROOT / "profiles" / "r2_measured_ai.txt"
    out = {}
    try:
        for line in p.read_text().splitlines():
            if line.startswith(f"{kernel}."):
                k, v = line.split("=", 1)
                out[k.split(".", 1)[1]] = float(v)
    except Exception:
        return None
    return out or None


def cpu_oracle_rate(case, nsteps=1, nthreads=None):
    """nsteps RK3 steps of `case` with the oracle as it stands (all host cores unless nthreads is given)."""
    import numpy as np
    from oracle import oracle as O
    metrics = None
    if case.coords is not None:
        metrics = O.metrics_from_coords(case.coords, case.n, case.periodic, delta=case.delta)
    orc = O.Oracle(metrics=metrics, nthreads=nthreads, **case.physics())
    Q = case.Q0.copy()
    dU, R = np.zeros_like(Q), np.zeros_like(Q)
    t0 = time.perf_counter()
    for _ in range(nsteps):
        orc.rk3_step(Q, dU, R, case.dt)
    dt = time.perf_counter() - t0
    assert np.isfinite(Q).all()
    return case.npoints * 3 * nsteps / dt, orc.nthreads, dt


def cpu_sample_case(args, full=False):
    """The bounded sample of the workload the oracle is timed on: (case, description)."""
    from paper_2007_14933_b200 import workloads as W
    if args.config == 4:
        n = (500, 250, 8) if full else (250, 125, 8)
        return W.sbli_slab(n=n), f"the same slab (grid, flow, boundaries) on {n[0]}x{n[1]}x{n[2]} points"
    big = 512 if args.config == 5 else args.n
    n = min(big, 256) if full else 64
    schemes = {"wenoz5": W.WENOZ5, "teno5": W.TENO5, "teno6": W.TENO6, "wenojs5": W.WENOJS5, "central4": W.CENTRAL4, "wenoz3": W.WENOZ3, "wenoz7": W.WENOZ7}
    case = W.tgv(n, scheme=schemes[args.scheme])
    if case.scheme == W.WENOJS5:
        case.eps = 1e-6
    return case, f"the same TGV field on {n}^3 points"


def run_reference(args):
    rank = env_int("RANK", 0)
    if rank != 0:
        return 0
    _, _, label, _ = make_case_label_only(args)
    case, what = cpu_sample_case(args)
    for _ in range(args.warmup if args.warmup < 2 else 1):      # the oracle has no warm-up effects worth 3 steps
        cpu_oracle_rate(case)
    times = []
    cores = 1
    for _ in range(args.steps):
        rate, cores, dt = cpu_oracle_rate(case)
        times.append(dt)
    total = sum(times)
    value = case.npoints * 3 * args.steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": label, "sample": f"each step = one RK3 step of {what}"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{args.steps} RK3 steps of {what}, OpenMP over grid lines"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def make_case_label_only(args):
    """Workload label without building the (possibly 6 GB) state."""
    if args.config == 4:
        return None, None, ("SBLI slab 500x250x8 curvilinear, WENO-Z5 + central-4 viscous (Sutherland), low-storage RK3 "
                            "(BASELINE.json config 4)"), 4
    n = 512 if args.config == 5 else args.n
    cfg = 3 if (n == 256 and args.scheme == "teno5") else (5 if (n == 512 and args.scheme == "teno5") else None)
    return None, None, (f"TGV {n}^3 periodic, {args.scheme.upper()} + central-4 viscous, low-storage RK3"
                        + (f" (BASELINE.json config {cfg})" if cfg else "")), cfg


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

    case, metrics, label, cfg = make_case(args)
    sol = osbli.Solver(device=dev, metrics=metrics, **case.physics())
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
    # Every step is one independent batch item: a pinned host state goes to the device, is advanced by one RK3
    # step and comes back.  osbli_advance_host_batch pipelines the items over three device states (copy in /
    # compute / copy out on three streams); the serial figure (osbli_advance_host, one item at a time) is kept.
    barrier()
    e2e_steps = args.steps
    hQs = [hQ, sol.to_padded(case.Q0, pinned_host=True), sol.to_padded(case.Q0, pinned_host=True)]
    Qs = [Q, sol.empty_state(), sol.empty_state()]
    sol.advance_host_batch([hQs[b % 3] for b in range(3)], Qs, Qtmp, case.dt, 1)        # warm-up (streams, events, pages)
    barrier()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    sol.advance_host_batch([hQs[b % 3] for b in range(e2e_steps)], Qs, Qtmp, case.dt, 1)
    t1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(t0.elapsed_time(t1), dev)
    t0.record(stream)
    for _ in range(min(e2e_steps, 5)):
        sol.advance_host(hQ, Q, Qtmp, case.dt, 1)
    t1.record(stream)
    barrier()
    ms_e2e_serial = max_over_ranks(t0.elapsed_time(t1), dev) / min(e2e_steps, 5)
    assert all(bool(torch.isfinite(t).all()) for t in hQs), "e2e state blew up"

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    npts = case.npoints
    value = aggregate_updates_per_s(npts, args.steps, world, ms)
    e2e_value = aggregate_updates_per_s(npts, e2e_steps, world, ms_e2e)

    # dominant kernel = the kernel class with the largest device time
    curv = metrics is not None
    sweep_flop = round(CURV_FACTOR * FLOP_SWEEP[case.scheme]) if curv else FLOP_SWEEP[case.scheme]
    visc_flop = 0 if case.visc == W.VISC_NONE else (FLOP_VISCOUS_CURV if curv else FLOP_VISCOUS)
    fused = prof["rk_update"][1] == 0                # the stage update rides on the last sweep when no update kernel ran
    last_sweep = "sweep_z" if case.n[2] > 1 else ("sweep_y" if case.n[1] > 1 else "sweep_x")
    flop_of = {"sweep_x": sweep_flop, "sweep_y": sweep_flop, "sweep_z": sweep_flop, "viscous": visc_flop,
               "primitives": 0, "bc": 0, "rk_update": FLOP_RK}
    if fused:
        flop_of[last_sweep] += FLOP_RK
    dom = max(("sweep_x", "sweep_y", "sweep_z", "viscous"), key=lambda k: prof[k][0])
    dom_ms, dom_cnt = prof[dom]
    dom_avg_s = dom_ms * 1e-3 / max(dom_cnt, 1)
    flop_point = flop_of[dom]
    achieved = flop_point * npts / dom_avg_s * 1e-12
    peaks, peak_src = measured_peaks()
    total_prof_ms = sum(v[0] for v in prof.values())
    nsweeps = sum(1 for d in range(3) if case.n[d] > 1)
    step_flop = nsweeps * sweep_flop + visc_flop + FLOP_RK
    executed = executed_fp64_from_profiles(dom) if cfg == 3 else None
    roofline = {
        "bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved / peak_tflops if peak_tflops > 0 else None,
        "frac_of_nominal_peak": achieved / NOMINAL_FP64_TFLOPS, "nominal_peak": NOMINAL_FP64_TFLOPS,
        "traffic": ncu_traffic_bytes(dom) if cfg == 3 else None,
        "traffic_source": "static: ncu dram__bytes_read.sum + dram__bytes_write.sum per launch of this kernel, committed in "
                          "profiles/dominant_kernel_traffic.txt (not measured in this run)" if cfg == 3 else None,
        "peak_source": "fp64 DFMA micro-benchmark run in this process (osbli_measure_fp64_peak; ncu: profiles/r2_dfma_peak.md); "
                       "nominal 148 SM x 64 lanes x 2 x 1.965 GHz = 37.2",
        "algorithmic_flop_per_point": flop_point,
        "algorithmic_note": "flop of the plain algorithm (SURVEY.md 8(d)); the kernel executes fewer: see executed_fp64",
        "executed_fp64": executed,
        "fused_stage_update": fused,
        "avg_launch_ms": dom_avg_s * 1e3,
        "whole_step_useful_flop_frac": step_flop * value / world * 1e-12 / peak_tflops if peak_tflops > 0 else None,
        "whole_step_useful_flop_frac_of_nominal": step_flop * value / world * 1e-12 / NOMINAL_FP64_TFLOPS,
        "algorithmic_flop_per_point_stage": step_flop,
        "kernel_share_of_step": {k: (v[0] / total_prof_ms if total_prof_ms > 0 else None) for k, v in prof.items()},
        "kernel_ms_per_launch": {k: (v[0] / v[1] if v[1] else None) for k, v in prof.items()},
        "profiled_ms_per_step": ms_prof / args.steps,
        "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src,
    }

    if case.scheme == W.CENTRAL4 and prof["sweep_x"][1] == 0 and prof["viscous"][1] == 0:
        # fused central path (osbli_central.cu): one kernel per stage, bound by HBM.  Algorithmic bytes per point:
        # Q in + dU out + Qout out = 120 in the first stage (dU is not read), 160 in the others.
        zms, zcnt = prof["sweep_z"]
        avg_s = zms * 1e-3 / max(zcnt, 1)
        bytes_point = (120 + 160 + 160) / 3.0
        gbs = bytes_point * npts / avg_s * 1e-9
        roofline.update({"bound": "hbm", "kernel": "central_fused", "achieved": gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                         "frac": gbs / peaks.get("hbm_gbs"), "algorithmic_bytes_per_point": bytes_point, "avg_launch_ms": avg_s * 1e3,
                         "peak_source": peak_src, "traffic": None, "traffic_source": None,
                         "fp64_useful_tflops": step_flop * value / world * 1e-12})

    # the oracle beside it: all cores on a bounded sample of the same workload, and one core on a small one
    cpu_case, cpu_what = cpu_sample_case(args, full=True)
    cpu_rate, cpu_cores, cpu_dt = cpu_oracle_rate(cpu_case)
    small_case, small_what = cpu_sample_case(args, full=False)
    st_rate, _, st_dt = cpu_oracle_rate(small_case, nthreads=1)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": label,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"state {state_bytes / 1e9:.2f} GB per array" + (" >> 126 MB L2 (inputs larger than L2)" if state_bytes > 2.5e8 else
                         " (5 live arrays + metric fields; comparable to the 126 MB L2: side workload, not the headline)")},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 5 * npts * 8, "d2h_bytes_per_step": 5 * npts * 8,
                "ms_per_step": ms_e2e / e2e_steps,
                "api": "osbli_advance_host_batch: every step one pinned host state -> device (interior nodes), 1 RK3 step, device -> host; "
                       "items pipelined over three device states (copy in / compute / copy out overlap across items)",
                "serial_ms_per_step": ms_e2e_serial,
                "serial_api": "osbli_advance_host: the same, one item at a time (copies and compute in series)"},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": cpu_cores, "kind": "oracle",
                         "sample": f"1 RK3 step (3 stage evaluations) of {cpu_what}, {cpu_dt:.1f} s",
                         "single_thread": {"value": st_rate, "unit": UNIT, "cores": 1,
                                           "sample": f"1 RK3 step of {small_what}, {st_dt:.1f} s"}},
    }
    print(json.dumps(line))
    sol.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1,
                    help="number of replicas (one per GPU). bench.py does not spawn ranks: for N > 1 launch it under torchrun "
                         "(python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 ... bench.py --gpus N)")
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[3, 4, 5],
                    help="BASELINE.json configuration: 3 = 256^3 TGV (headline, default), 4 = SBLI slab, 5 = 512^3 TGV")
    ap.add_argument("--perturb", type=float, default=0.0,
                    help="side measurement: seeded perturbation amplitude of the TGV state (non-smooth data takes the full TENO evaluation)")
    ap.add_argument("--n", type=int, default=256, help="grid points per side of the TGV (256 = BASELINE.json config 3)")
    ap.add_argument("--scheme", default="teno5", choices=["wenoz5", "teno5", "teno6", "wenojs5", "central4", "wenoz3", "wenoz7"],
                    help="reconstruction (teno5 = BASELINE.json config 3; the others are side measurements)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
