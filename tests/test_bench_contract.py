"""The bench.py contract (-m "not gpu"): the reference arm runs on this CPU box and prints the agreed JSON line; the
last committed GPU line (profiles/*_bench_line.txt, written by `python bench.py` on a B200) carries every agreed key."""
import glob
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches"}


def test_reference_arm_runs_without_a_gpu():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0", "--L", "256"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert BASE_KEYS <= set(line), BASE_KEYS - set(line)
    assert line["impl"] == "reference" and line["metric"] == "ps_per_spin_flip_attempt" and line["unit"] == "ps/flip"
    assert line["higher_is_better"] is False and line["vs_baseline"] is None and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "ps/flip", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in line["config"] and "model" not in line["config"]


def test_last_committed_gpu_line_has_every_agreed_key():
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "*_bench_line.txt")))
    assert files, "no bench line under profiles/"
    line = json.loads(open(files[-1]).read().strip().splitlines()[-1])
    assert BASE_KEYS | {"roofline", "cpu_baseline", "clocks"} <= set(line)
    assert line["metric"] == "ps_per_spin_flip_attempt" and line["dtype"] == "u32" and line["data"] == "synthetic"
    roof = line["roofline"]
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(roof)
    assert roof["bound"] in ("alu", "hbm", "tensor") and abs(roof["frac"] - roof["achieved"] / roof["peak"]) < 1e-9
    assert 0.0 < roof["frac"] < 1.2
    cb = line["cpu_baseline"]
    assert {"value", "unit", "cores", "kind", "sample"} <= set(cb) and cb["kind"] == "oracle"
    e2e = line["e2e"]
    assert e2e["h2d_bytes_per_step"] == 4 * 2**27 and e2e["d2h_bytes_per_step"] == 2**27 + 16  # 512 MiB in, 128 MiB + E, M out
    assert e2e["value"] > line["value"]  # copies inside the timed region
    assert line["gpu_launches"] > 0 and "workload" in line["config"] and "model" not in line["config"]
    assert not set(line["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
