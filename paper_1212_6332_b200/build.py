"""Build libmd_b200.so (hand-written sm_100a CUDA + the C ABI of include/md.h), in-tree.

    python -m paper_1212_6332_b200.build [--force] [--ptxas-v]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmd_b200.so")
OBJ = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
         "-shared", "-cudart", "static", "--expt-relaxed-constexpr"]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def build(force: bool = False, verbose: bool = False) -> str:
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "md.h")]
    newest = max(os.path.getmtime(p) for p in deps)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    extra = os.environ.get("MD_NVCC_EXTRA", "").split()          # e.g. -DMD_FORCE_MINB=5 (tuning knobs of md_force.cu)
    cflags = [f for f in FLAGS if f != "-shared"] + extra + (["-Xptxas", "-v"] if verbose else [])
    os.makedirs(OBJ, exist_ok=True)
    jobs = []                                                     # one nvcc per translation unit, side by side, then one link
    for src in sources():
        obj = os.path.join(OBJ, os.path.splitext(os.path.basename(src))[0] + ".o")
        cmd = [NVCC, *cflags, "-c", "-o", obj, src]
        jobs.append((cmd, obj, subprocess.Popen(cmd, cwd=CSRC)))
    failed = [(cmd, p.returncode) for cmd, _, p in jobs if p.wait() != 0]
    if failed:
        raise subprocess.CalledProcessError(failed[0][1], failed[0][0])
    subprocess.run([NVCC, *FLAGS, "-o", LIB, *(obj for _, obj, _ in jobs)], check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--ptxas-v" in sys.argv))
