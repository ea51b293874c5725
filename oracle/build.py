"""Build the CPU oracle (plain C, gcc) into oracle/libea3d_oracle.so.  TEST INFRASTRUCTURE ONLY."""
from __future__ import annotations

import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ea3d_oracle.c")
LIB = os.path.join(HERE, "libea3d_oracle.so")


def build(force: bool = False) -> str:
    stamp = LIB + ".srchash"  # content hash: mtimes do not survive the copy to the GPU box
    digest = hashlib.sha256(open(SRC, "rb").read()).hexdigest()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read().strip() == digest:
        return LIB
    # -ffp-contract=off: the threshold table must be plain double arithmetic (R5).
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    with open(stamp, "w") as f:
        f.write(digest)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
