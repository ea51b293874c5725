"""Synchronisation-latency probe (csrc/sync_probe.cu): grid-wide barriers, neighbour flags and a cluster barrier on the GPU it runs on.
`python -m paper_1411_0127_b200.sync_probe` builds the standalone program next to the library and prints its table
(profiles/r2j_launch_floor.md)."""
from __future__ import annotations

import os
import subprocess

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "sync_probe.cu")
EXE = os.path.join(HERE, "sync_probe.bin")


def build(force: bool = False) -> str:
    if force or not os.path.exists(EXE) or os.path.getmtime(EXE) < os.path.getmtime(SRC):
        subprocess.run([_build.nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-rdc=true",
                        "-o", EXE, SRC, "-lcudadevrt"], check=True)
    return EXE


if __name__ == "__main__":
    print(subprocess.run([build()], check=True, capture_output=True, text=True).stdout)
