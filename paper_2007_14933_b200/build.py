"""Builds libosbli.so (the C-ABI library of include/osbli.h) in-tree with nvcc for sm_100a.

Run as `python -m paper_2007_14933_b200.build` or through `__graft_entry__.build()`.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libosbli.so"
SOURCES = ["osbli_sweep.cu", "osbli_weno7.cu", "osbli_api.cu", "osbli_visc.cu", "osbli_central.cu", "osbli_bc_rk.cu", "osbli_peak.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + [PKG.parent / "include" / "osbli.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    flags = NVCC_FLAGS + os.environ.get("OSBLI_NVCC_EXTRA", "").split()      # tuning experiments (-D... macros)

    def compile_one(src):
        obj = CSRC / (src[:-3] + ".o")
        cmd = [nvcc(), *flags, "-c", str(CSRC / src), "-o", str(obj)]
        return src, obj, subprocess.run(cmd, capture_output=True, text=True)

    objs = []
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        for src, obj, res in pool.map(compile_one, SOURCES):
            if verbose or res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
            if res.returncode != 0:
                raise RuntimeError(f"nvcc failed on {src}")
            (CSRC / (src[:-3] + ".ptxas.txt")).write_text(res.stderr)
            objs.append(str(obj))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc(), "-shared", "-o", str(tmp), *objs]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
