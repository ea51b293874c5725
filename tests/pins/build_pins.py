"""Build the test-only pin shims (third-party implementations the oracle is checked against)."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))


def _stale(lib, src):
    return not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src)


def build_minstd() -> str:
    src, lib = os.path.join(HERE, "minstd_shim.cpp"), os.path.join(HERE, "libpin_minstd.so")
    if _stale(lib, src):
        subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", lib, src], check=True)
    return lib


def build_mt19937() -> str:
    src, lib = os.path.join(HERE, "mt19937_shim.cpp"), os.path.join(HERE, "libpin_mt19937.so")
    if _stale(lib, src):
        subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", lib, src], check=True)
    return lib


def build_curand_philox() -> str | None:
    """None when nvcc is not installed (the test then skips)."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        return None
    src, lib = os.path.join(HERE, "curand_philox_shim.cu"), os.path.join(HERE, "libpin_curand_philox.so")
    if _stale(lib, src):
        subprocess.run([nvcc, "-O2", "-shared", "-Xcompiler", "-fPIC", "-o", lib, src], check=True)
    return lib
