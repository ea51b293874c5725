"""Build libising_b200.so (the C-ABI library of include/ising.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libising_b200.so")
STAMP = LIB + ".srchash"  # git-ignored with the .so; travels with it to the GPU box
SOURCES = ["ising_api.cu"]
HEADERS = ["rng.cuh", "update.cuh", "sweep_kernels.cuh", "batch_kernels.cuh", "cluster_kernels.cuh", "fnv_kernels.cuh", "graph_kernels.cuh", "persistent.cuh", "slab_kernels.cuh", "sliced_kernels.cuh", "measure_kernels.cuh", "layout_kernels.cuh", "lane_rng.cuh",
           os.path.join("..", "..", "include", "ising.h")]


def nvcc_path() -> str:
    return shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"


def nvcc_command(out: str = LIB, extra: list[str] | None = None) -> list[str]:
    return [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            # the threshold table must be plain double arithmetic (R5): no FMA contraction on the host
            "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall,-Wno-unknown-pragmas", "-shared", "-o", out,
            *[os.path.join(CSRC, s) for s in SOURCES], *(extra or [])]


def source_hash() -> str:
    """Hash of every source the library is built from (mtimes do not survive the copy to the GPU box)."""
    import hashlib

    h = hashlib.sha256()
    for d in [os.path.join(CSRC, s) for s in SOURCES] + [os.path.join(CSRC, x) for x in HEADERS]:
        h.update(open(d, "rb").read())
    h.update(" ".join(a for a in nvcc_command(out="-")[1:] if not a.startswith(HERE)).encode())  # flags, not paths
    return h.hexdigest()


def is_stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    return open(STAMP).read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than its sources; returns the path of the .so."""
    if force or is_stale():
        if not os.path.exists(nvcc_path()):
            raise RuntimeError("libising_b200.so is not built and nvcc is not available")
        cmd = nvcc_command(extra=["-Xptxas", "-v"] if verbose else None)
        subprocess.run(cmd, check=True)
        with open(STAMP, "w") as f:
            f.write(source_hash())
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
