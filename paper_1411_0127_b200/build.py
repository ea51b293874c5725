"""Build libising_b200.so (the C-ABI library of include/ising.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libising_b200.so")
SOURCES = ["ising_api.cu"]
HEADERS = ["rng.cuh", "update.cuh", "sweep_kernels.cuh", "measure_kernels.cuh", "layout_kernels.cuh",
           os.path.join("..", "..", "include", "ising.h")]


def nvcc_path() -> str:
    return shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"


def nvcc_command(out: str = LIB, extra: list[str] | None = None) -> list[str]:
    return [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            # the threshold table must be plain double arithmetic (R5): no FMA contraction on the host
            "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared", "-o", out,
            *[os.path.join(CSRC, s) for s in SOURCES], *(extra or [])]


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [os.path.join(CSRC, h) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than its sources; returns the path of the .so."""
    if force or is_stale():
        if not os.path.exists(nvcc_path()):
            raise RuntimeError("libising_b200.so is not built and nvcc is not available")
        cmd = nvcc_command(extra=["-Xptxas", "-v"] if verbose else None)
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
