"""The N > 1 plumbing of bench.py on CPU (gloo, world_size 2): DESIGN.md "Multi-GPU" -- the path does
not shard (north_star: one GPU, no sharding), so `bench.py --gpus N` runs N independent replicas and
the only cross-rank step is the MAX of the device times.  Covered here without a GPU:
  * max_over_ranks / aggregate_updates_per_s under a real 2-process gloo group;
  * `--impl reference` under torchrun: rank 0 alone runs the oracle and prints the one JSON line,
    the other rank exits 0 without work.
"""
import json
import os
import subprocess
import sys
import textwrap
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def _torchrun(args, timeout=600):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="4")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29577"] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_aggregate_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys, json
        sys.path.insert(0, {str(ROOT)!r})
        import torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        ms = bench.max_over_ranks(10.0 * (rank + 1))            # rank 0: 10 ms, rank 1: 20 ms
        dist.barrier()
        if rank == 0:
            print(json.dumps({{"ms": ms, "world": world, "value": bench.aggregate_updates_per_s(1000, 2, world, ms)}}))
        dist.destroy_process_group()
    """))
    res = _torchrun([str(script)])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["world"] == 2 and out["ms"] == 20.0
    assert out["value"] == 2 * 1000 * 3 * 2 / 20e-3              # both replicas' work over the slowest rank's time


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["value"] > 0
    assert out["cpu_baseline"]["kind"] == "oracle" and out["e2e"]["h2d_bytes_per_step"] == 0
    assert out["unit"] == "updates/s" and out["higher_is_better"] is True
