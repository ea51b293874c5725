"""Integer issue-rate microbenchmark (csrc/int_peak.cu): measures, on the GPU it runs on, the thread-instructions per
second of the instruction mixes the half-sweep kernel is made of.  `python -m paper_1411_0127_b200.int_peak` prints one
JSON line; DESIGN.md section 6 uses it to check the ALU roofline denominator (148 SMs x 4 schedulers x 32 lanes x clock
for the issue limit, half of that per pipe)."""
from __future__ import annotations

import ctypes as C
import json
import os
import subprocess

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "int_peak.cu")
LIB = os.path.join(HERE, "libint_peak.so")
MIXES = {0: "LOP3 only", 1: "IMAD.WIDE.U32 only", 2: "IMAD.WIDE + LOP3 dependent 1:1", 3: "Philox round (2 IMAD.WIDE + 2 LOP3)",
         4: "ISETP + SEL + LOP3", 5: "IMAD.HI.U32 only", 6: "IMAD (lo) only", 7: "Philox round + 1 LOP3", 8: "Philox round + 2 LOP3",
         9: "Philox round + 3 LOP3", 10: "Philox round + 4 LOP3", 11: "Philox round via DFMA.RM (hi) + IMAD (lo)",
         12: "IMAD (lo) + LOP3 1:1 independent", 13: "FFMA only", 14: "FFMA + LOP3 1:1 independent",
         15: "IMAD (lo) + IADD3 1:1 independent", 16: "IMAD (lo) + FFMA 1:1 independent",
         17: "IMAD.HI + LOP3 1:1 independent", 18: "IMAD.HI + 3 LOP3 independent", 19: "IMAD.WIDE, multiplier in a register",
         20: "DFMA only", 21: "DFMA + LOP3 1:1 independent", 22: "IMAD.WIDE + IMAD (lo) 1:1",
         23: "Philox round from IMAD.HI + IMAD (lo), + 2 LOP3", 24: "Philox round (register multipliers) + 4 LOP3",
         25: "IMAD.WIDE + FFMA 1:1", 26: "IMAD.WIDE + 3 LOP3 independent",
         27: "2 Philox rounds via DFMA.RM + IMAD (lo), state in register pairs", 28: "same + 2 x 2 LOP3", 29: "same + 2 x 4 LOP3",
         30: "2 rounds via IMAD.WIDE + 2 rounds via DFMA.RM, interleaved", 31: "6 rounds via IMAD.WIDE + 2 rounds via DFMA.RM, interleaved"}
# source-level instructions per chain-iteration of each mix (csrc/int_peak.cu)
OPS = {0: 4, 1: 2, 2: 4, 3: 4, 4: 6, 5: 2, 6: 2, 7: 5, 8: 6, 9: 7, 10: 8, 11: 6, 12: 4, 13: 4, 14: 4, 15: 4, 16: 4, 17: 4, 18: 8, 19: 2, 20: 2, 21: 4, 22: 6, 23: 8, 24: 8, 25: 6, 26: 4, 27: 12, 28: 16, 29: 20, 30: 20, 31: 36}


def build(force: bool = False) -> str:
    import hashlib

    stamp = LIB + ".srchash"
    digest = hashlib.sha256(open(SRC, "rb").read()).hexdigest()
    if force or not os.path.exists(LIB) or not os.path.exists(stamp) or open(stamp).read().strip() != digest:
        subprocess.run([_build.nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                        "-Xcompiler", "-fPIC", "-shared", "-o", LIB, SRC], check=True)
        with open(stamp, "w") as f:
            f.write(digest)
    return LIB


def run(ctas_per_sm: int = 8, iters: int = 4096, reps: int = 5, mixes=None) -> dict:
    import torch

    lib = C.CDLL(build())
    lib.int_peak_run.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_double)]
    dev = torch.cuda.current_device()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    scratch = torch.zeros(16, dtype=torch.int32, device=torch.device("cuda", dev))
    out = {"sms": sms, "ctas_per_sm": ctas_per_sm, "threads_per_cta": 256, "mixes": {}}
    for mix, name in MIXES.items():
        if mixes is not None and mix not in mixes:
            continue
        ms, ops = C.c_float(0), C.c_double(0)
        rc = lib.int_peak_run(mix, sms * ctas_per_sm, iters, reps, scratch.data_ptr(), C.byref(ms), C.byref(ops))
        if rc != 0:
            raise RuntimeError(f"int_peak_run({mix}) failed: {rc}")
        rate = ops.value / (ms.value * 1e-3)
        # cycles one SMSP spends per warp on one chain-iteration: 16 warps per SMSP (8 CTAs x 8 warps / 4), 8 chains
        cyc = ms.value * 1e-3 * 1.965e9 / (iters * 8 * (ctas_per_sm * 8 / 4))
        out["mixes"][name] = {"Tinst_per_s": rate / 1e12, "inst_per_clk_per_sm_at_1965MHz": rate / sms / 1.965e9, "ms": ms.value,
                              "cycles_per_warp_iteration": cyc, "instructions_per_iteration": OPS[mix]}
    return out


if __name__ == "__main__":
    print(json.dumps(run()))
