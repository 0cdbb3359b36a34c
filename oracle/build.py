"""Build the CPU oracle shared library (test infrastructure, not the product).

    python -m oracle.build            # -> oracle/libeam_oracle.so
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "eam_oracle.c")
HDR = os.path.join(HERE, "eam_oracle.h")
LIB = os.path.join(HERE, "libeam_oracle.so")
# -ffp-contract=off: no FMA contraction, so every operation rounds once, as written
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    subprocess.run(["gcc", *CFLAGS, "-o", LIB, SRC, "-lm"], check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
