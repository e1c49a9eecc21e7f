"""Writes the stored oracle samples of the configured-length runs of BASELINE.json configs 3, 4, 5
(tests/golden/config{3,4,5}_oracle_samples.npz).

TEST INFRASTRUCTURE.  Imports only `oracle/` and the seeded input generators
(`paper_2007_14933_b200/workloads.py`, which holds none of the method's arithmetic); nothing here touches the
CUDA path.  The oracle is advanced for the configured number of RK3 steps (200 / 500 / 50) on the host cores
-- about 1 h / 15 min / 2.5 h on 8 cores -- and a strided sample of the interior state is stored at a few
checkpoints (the last one is the configured step count), together with

  * the full-field max-norm of every variable at each checkpoint (the denominators of DESIGN.md Q28),
  * sha256 of the oracle sources (osbli_oracle.cpp + osbli_oracle.h): the GPU test refuses a file whose hash is
    not that of the oracle it sits next to,
  * sha256 of the same strided sample of the initial state: the GPU test checks its own inputs against it.

The sample strides (7, 13, (5, 3, 1)) are coprime to every tile size of the CUDA path, so the sampled nodes
fall on every position inside a tile, including the seams.

    python oracle/make_golden.py --config 3 [--threads 8] [--steps N (debug)] [--out DIR]
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
# run as a script, sys.path[0] is oracle/ itself and `import oracle` would find oracle/oracle.py: drop it
sys.path[:] = [p for p in sys.path if Path(p or ".").resolve() != ROOT / "oracle"]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from oracle import oracle as O                                   # noqa: E402
from paper_2007_14933_b200 import workloads as W                 # noqa: E402

GOLDEN = ROOT / "tests" / "golden"


def use_private_library():
    """Compile the oracle into a private temporary file for this (hours-long) process, so that a rebuild of
    oracle/libosbli_oracle.so by a test session running meanwhile cannot touch the code being executed."""
    import tempfile
    O._LIB = Path(tempfile.mkdtemp(prefix="osbli_golden_")) / "libosbli_oracle_golden.so"
    O.build(force=True)

# config -> (case factory, sample stride per direction (x, y, z), checkpoints in steps)
CONFIGS = {
    3: (lambda: W.tgv(256), (7, 7, 7), (50, 100, 200)),
    4: (lambda: W.sbli_slab(), (5, 3, 1), (100, 250, 500)),
    5: (lambda: W.tgv(512), (13, 13, 13), (10, 25, 50)),
}


def oracle_source_hash() -> str:
    h = hashlib.sha256()
    for name in ("osbli_oracle.cpp", "osbli_oracle.h"):
        h.update((ROOT / "oracle" / name).read_bytes())
    return h.hexdigest()


def sample_of(case, A, stride):
    """Strided sample of the interior nodes of a dense padded array [.., NZ, NY, NX] -> [.., nzs, nys, nxs]."""
    h = case.halo
    n = case.n
    return np.ascontiguousarray(A[..., h[2]:h[2] + n[2]:stride[2], h[1]:h[1] + n[1]:stride[1], h[0]:h[0] + n[0]:stride[0]])


def sample_hash(a) -> str:
    return hashlib.sha256(np.ascontiguousarray(a, dtype=np.float64).tobytes()).hexdigest()


def golden_path(config: int) -> Path:
    return GOLDEN / f"config{config}_oracle_samples.npz"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=sorted(CONFIGS))
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--steps", type=int, default=None, help="debug: stop after this many steps (file marked partial)")
    ap.add_argument("--out", type=str, default=str(GOLDEN))
    ap.add_argument("--resume-dir", type=str, default=None,
                    help="directory for restart files (the state every --resume-every steps); an interrupted run continues from there")
    ap.add_argument("--resume-every", type=int, default=5)
    ap.add_argument("--stop-after-seconds", type=float, default=None,
                    help="write a restart file and exit (status 3) once this much wall time has passed")
    a = ap.parse_args()

    use_private_library()
    make, stride, checkpoints = CONFIGS[a.config]
    case = make()
    assert checkpoints[-1] == case.nsteps, (checkpoints, case.nsteps)
    if a.steps is not None:
        checkpoints = tuple(c for c in checkpoints if c <= a.steps) or (a.steps,)
    metrics = None
    if case.coords is not None:
        metrics = O.metrics_from_coords(case.coords, case.n, case.periodic, delta=case.delta, nthreads=a.threads)
    orc = O.Oracle(metrics=metrics, nthreads=a.threads, **case.physics())
    src_hash = oracle_source_hash()
    q0_hash = sample_hash(sample_of(case, case.Q0, stride))

    Q = case.Q0.copy()
    dU = np.zeros_like(Q)          # dU^(0) is never read (A_1 = 0): the state Q alone restarts a run exactly
    R = np.zeros_like(Q)
    out = {}
    t0 = time.time()
    step = 0
    rdir = Path(a.resume_dir) if a.resume_dir else None
    tag = f"config{a.config}_{src_hash[:12]}_{q0_hash[:12]}"

    def save_restart():
        rdir.mkdir(parents=True, exist_ok=True)
        np.save(rdir / f"{tag}_state.tmp.npy", Q)
        os.replace(rdir / f"{tag}_state.tmp.npy", rdir / f"{tag}_state.npy")
        np.savez(rdir / f"{tag}_samples.tmp.npz", step=step, **out)
        os.replace(rdir / f"{tag}_samples.tmp.npz", rdir / f"{tag}_samples.npz")

    if rdir is not None and (rdir / f"{tag}_samples.npz").exists() and (rdir / f"{tag}_state.npy").exists():
        z = np.load(rdir / f"{tag}_samples.npz")
        step = int(z["step"])
        out = {k: z[k] for k in z.files if k != "step"}
        Q = np.load(rdir / f"{tag}_state.npy")
        print(f"config {a.config}: resuming at step {step} from {rdir}", flush=True)
    for cp in checkpoints:
        while step < cp:
            orc.rk3_step(Q, dU, R, case.dt)
            step += 1
            if rdir is not None and (step % a.resume_every == 0 or (a.stop_after_seconds and time.time() - t0 > a.stop_after_seconds)):
                save_restart()
                if a.stop_after_seconds and time.time() - t0 > a.stop_after_seconds and step < checkpoints[-1]:
                    print(f"config {a.config}: stopped at step {step} after {time.time() - t0:.0f} s (restart file written)", flush=True)
                    sys.exit(3)
            if step % 5 == 0 or step == cp:
                el = time.time() - t0
                print(f"config {a.config}: step {step}/{checkpoints[-1]}  {el:8.1f} s  "
                      f"({3 * case.npoints * step / el:.3e} updates/s, {a.threads} threads)", flush=True)
        if f"state_{cp}" in out:
            continue                                   # checkpoint already sampled before the restart
        assert np.isfinite(Q).all()
        out[f"state_{cp}"] = sample_of(case, Q, stride)
        qi = orc.interior(Q)
        out[f"maxnorm_{cp}"] = np.array([np.abs(qi[c]).max() for c in range(5)])
        out[f"l1norm_{cp}"] = np.array([np.abs(qi[c]).mean() for c in range(5)])
    meta = dict(config=a.config, name=case.name, n=list(case.n), dt=case.dt, nsteps=case.nsteps,
                checkpoints=list(checkpoints), stride=list(stride), scheme=case.scheme, visc=case.visc,
                oracle_sha256=src_hash, q0_sample_sha256=q0_hash, threads=a.threads,
                partial=bool(a.steps is not None and a.steps < case.nsteps),
                seconds=round(time.time() - t0, 1),
                command=f"python oracle/make_golden.py --config {a.config}")
    dest = Path(a.out) / golden_path(a.config).name
    np.savez(dest, meta=json.dumps(meta), **out)
    print(f"wrote {dest} ({dest.stat().st_size / 1e6:.2f} MB)")


if __name__ == "__main__":
    main()
