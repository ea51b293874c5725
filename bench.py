#!/usr/bin/env python
"""bench.py -- headline benchmark: ps per spin-flip attempt of the bit-packed checkerboard Metropolis sweep at L=1024.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--L 1024] [--sweeps 20]

One "step" is one pass of the whole hot path over one synthetic lattice of BASELINE.json
config 5: load the canonical packed state into the internal layout (a10), 20 full sweeps = 40 colour half-sweep launches
(a1-a8), energy + magnetisation (a9), canonical spins out (a10).  `value` is measured with the inputs resident in HBM;
`e2e` goes through ising_run_host with pinned HOST buffers (H2D of spins + couplings and D2H of spins, E, M inside the
timed region).  Philox mode is the headline line; the MINSTD mode of the same config is timed too ("minstd").
N > 1 runs N independent replicas (the path does not shard: DESIGN.md section 8), one process per GPU, no collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ps_per_spin_flip_attempt"
UNIT = "ps/flip"
BETA = 1.0 / 1.1

# Algorithmic integer work of one flip attempt on the binding pipe.
#   Philox: fma pipe.  18 wide multiplies per call of 4 sites, IMAD.WIDE = 2 passes of the 32-bit multiplier -> 9.0 slots
#   MINSTD, stateless: 16.69 alu instructions per flip -> 0.896 ps/flip at one 16-lane pipe per SMSP
ALG_SLOTS_PER_FLIP = {0: 18 * 2 / 4}
ALG_INT_OPS_PER_FLIP = 37 / 4 + 2 + 22 / 32
MINSTD_STATELESS_ALU_OPS_PER_FLIP = 16 + 22 / 32
BINDING_PIPE = {0: "fma (IMAD.WIDE)"}
ALG_BYTES_PER_FLIP = 9 / 8  # 9N/16 bytes per half-sweep = 1.125 B per flip attempt, both rng modes
MINSTD_TABLE_BYTES_PER_FLIP = 4.0  # the shipped MINSTD kernel also streams its cached seed states: implementation traffic
# stored-state lane generators (rng modes 3, 4): state words moved per draw, 4 B each.  Parisi-Rapuano reads
# ira[i-24], ira[i-55], ira[i-61] and writes ira[i]; MT19937 in blocks of four draws reads mt[i..i+4], mt[i+397..i+400], writes 4
LANE_STATE_BYTES_PER_DRAW = {3: 16.0, 4: 13.0}
# dram__bytes_read.sum + dram__bytes_write.sum per half-sweep launch at L=1024 from one `ncu --set full` capture.  The figure
# belongs to the kernel sources it was captured on: `kernel_sources_sha256` is kernel_sources_hash() at capture time, and
# the bench line prints `traffic` only while the sources still hash to it (null otherwise, with a note).
NCU_TRAFFIC_L1024 = {
    "kernel_sources_sha256": "d4d8c25eb7ad193dfa890c5abb33e3977afe6a37b478e91ca40ae419a7ead5eb",
    "capture": "profiles/r2n_end_of_round.md",
    0: 537.05e6 + 59.28e6, 1: 2684.53e6 + 61.07e6,
}


def kernel_sources_hash():
    """sha256 of the sources the half-sweep kernel is compiled from (csrc/sweep_kernels.cuh, update.cuh, rng.cuh)."""
    import hashlib

    h = hashlib.sha256()
    for name in ("sweep_kernels.cuh", "update.cuh", "rng.cuh"):
        h.update(open(os.path.join(ROOT, "paper_1411_0127_b200", "csrc", name), "rb").read())
    return h.hexdigest()


def headline_config(L, nsw, world):
    """`config` of the bench line; the reference arm prints the same dict (same workload, same metric)."""
    return {"workload": f"BASELINE.json config 5: L={L} periodic +-J EA cube, 1 sample, random spins, beta=1/1.1, {nsw} sweeps, Philox4x32-10",
            "L": L, "sweeps_per_step": nsw, "rng": "philox4x32-10", "step": "load_state + sweeps + energy + get_spins",
            "l2": "inputs larger than L2 (512 MiB packed state > 126 MB), no flush needed",
            "parallelism": "replicas only" if world > 1 else "1 GPU"}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return float(p.get("hbm_gbs", 6650.0)), float(p.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm = sorted(int(r[1]) for r in self.rows if len(r) >= 9 and r[1].isdigit())
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) >= 9:
                for n, v in zip(names, r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        smax = max((int(r[2]) for r in self.rows if len(r) >= 9 and r[2].isdigit()), default=None)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


class OracleTimer:
    """The oracle as it stands (OpenMP over the planes of one colour) on this host, on the L x L x L lattice of config 5:
    loads the canonical inputs once, then times calls of `sweeps` sweeps (the chain simply continues from call to call)."""

    def __init__(self, L, rng_mode=0, threads=None, spins=None, J=None):
        from oracle import ea3d
        from paper_1411_0127_b200 import synth

        self.ea3d, self.L = ea3d, L
        self.all_threads = ea3d.max_threads()
        self.threads = threads or min(self.all_threads, host_cores())
        ea3d.set_threads(self.threads)
        self.o = ea3d.Oracle(L, 1, synth.DYN_SEED, rng_mode)
        self.o.load_packed(synth.make_spins(L) if spins is None else spins, synth.make_couplings(L) if J is None else J)
        self.o.sweep(BETA, 1)  # touch the pages, warm the cores

    def time(self, sweeps):
        t0 = time.perf_counter()
        self.o.sweep(BETA, sweeps)
        return time.perf_counter() - t0

    def close(self):
        self.ea3d.set_threads(self.all_threads)
        self.o = None


ORACLE_SAMPLE_SWEEPS = 2  # of the 20 sweeps of the workload: about 4 s on 16 cores at L = 1024


def oracle_sample_text(L, sweeps, extra=""):
    return (f"the L={L} lattice of the workload itself (same J / spin recipe, beta=1/1.1, Philox), {sweeps} of its 20 sweeps "
            f"per timed call{extra}")


def run_reference(args):
    """--impl reference: the CPU oracle is the reference arm of this tier (rank 0 only): the same workload (config 5, L = 1024),
    the same metric; a step is a bounded sample of it (2 of the 20 sweeps)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    L, sweeps = args.L, ORACLE_SAMPLE_SWEEPS
    tm = OracleTimer(L)
    times = [tm.time(sweeps) for _ in range(args.warmup + args.steps)][args.warmup:]
    cores = tm.threads
    tm.close()
    total = sum(times)
    flips = len(times) * sweeps * L**3
    ps = 1e12 * total / flips
    med = sorted(times)[len(times) // 2]
    sample = oracle_sample_text(L, sweeps, f"; {len(times)} timed calls, median {med:.2f} s")
    line = {
        "impl": "reference", "metric": METRIC, "value": ps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": headline_config(L, args.sweeps, max(1, args.gpus)), "sample": sample,
        "flips_per_s": flips / total, "value_median": 1e12 * med / (sweeps * L**3),
        "cpu_baseline": {"value": ps, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": ps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default: 20; the reference arm, whose step is 3.4 s of CPU work: 3)")
    ap.add_argument("--warmup", type=int, default=None, help="untimed warm-up steps (default: 5; reference arm: 1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=1024)
    ap.add_argument("--sweeps", type=int, default=20)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-minstd", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-shared", action="store_true", help="skip the shared-random-number (paper's AMSC) timing")
    ap.add_argument("--only-shared", action="store_true", help="time only the shared-random-number mode (for ncu captures)")
    ap.add_argument("--only-lanes", action="store_true", help="time only the stored-state lane generators (sweep and Table II)")
    ap.add_argument("--scan-batches", action="store_true",
                    help="the paper's Fig. 4 study: half-sweep time of small lattices against the number k of coded batches (shared draws)")
    ap.add_argument("--configs", action="store_true",
                    help="the five configurations of BASELINE.json at their full sweep counts, with the outputs each one asks for")
    ap.add_argument("--no-verify", action="store_true", help="--configs: skip the comparison of every output with the CPU oracle")
    ap.add_argument("--aux", action="store_true",
                    help="rows a9 / a10 and the general-L kernels: load_state, energy, get_spins and a half-sweep per layout, with GB/s")
    ap.add_argument("--scan", action="store_true", help="ps/flip of the sweep kernels over lattice sizes and modes (sweeps only)")
    ap.add_argument("--slab-ranks", action="store_true",
                    help="strong scaling instead of replicas: the ONE L^3 lattice of config 5 cut into WORLD_SIZE z-slabs, one per rank / GPU "
                         "(PAPER.md section V), the two boundary planes of every colour half-sweep exchanged with NCCL send / recv "
                         "(paper_1411_0127_b200/slabs.py); prints its own JSON line with \"scaling\": \"strong\"")
    ap.add_argument("--slabs", type=int, default=0,
                    help="z-slab decomposition (PAPER.md section V) of the L^3 lattice into this many slabs, all on this GPU: sweep time "
                         "against the undivided lattice (the cost of the boundary / bulk split and of the plane exchange)")
    ap.add_argument("--sliced", action="store_true",
                    help="the paper's sliced layout (Eq. 4-6) against the rank-linear arrays: half-sweep time, both rng modes (MINSTD "
                         "without the seed table on both sides: same generator work, only the layout differs)")
    ap.add_argument("--sizes", default="", help="--sliced: comma-separated lattice sizes instead of 256,512,1024")
    ap.add_argument("--small", action="store_true",
                    help="small lattices: time per half-sweep with the automatic kernels (0), one launch per half-sweep (3) and the "
                         "persistent kernels everywhere (4), without records and with E and M after every half-sweep")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 3 if args.impl == "reference" else 20
    if args.warmup is None:
        args.warmup = 1 if args.impl == "reference" else 5
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch

    from paper_1411_0127_b200 import MINSTD, PHILOX, Ising, replicas, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        return replicas.max_over_ranks(x, dist, "cuda")

    L, nsw = args.L, args.sweeps
    N = L**3
    # every rank simulates its own disorder sample (replicas): seeds offset by rank
    s_seed, j_seed = replicas.replica_seeds(rank)
    spins = synth.make_spins(L, 1, s_seed)
    J = synth.make_couplings(L, 1, j_seed)
    h_spins = torch.from_numpy(spins.view(np.int32)).pin_memory()
    h_J = torch.from_numpy(J.view(np.int32)).pin_memory()
    h_out = torch.empty_like(h_spins).pin_memory()
    d_spins, d_J = h_spins.cuda(), h_J.cuda()
    d_out = torch.empty_like(d_spins)
    stream = torch.cuda.current_stream()

    def bench_mode(rng_mode):
        g = Ising(L, 1, synth.DYN_SEED, rng_mode)

        def step(ev=None):
            g.ising_set_t(0)  # every step is the same job: the same trajectory from the same state
            g.ising_load_state(d_spins, d_J)
            if ev:
                ev[0].record(stream)
            g.ising_sweep(BETA, nsw)
            if ev:
                ev[1].record(stream)
            E, M = g.ising_energy()
            g.ising_get_spins(d_out)
            return E, M

        for _ in range(args.warmup):
            step()
        barrier()
        l0 = g.ising_kernel_launches()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for k in range(args.steps):
            E, M = step(evs[k])
        e1.record(stream)
        barrier()
        total_ms = max_over_ranks(e0.elapsed_time(e1))
        sweep_ms = max_over_ranks(sum(a.elapsed_time(b) for a, b in evs))
        launches = g.ising_kernel_launches() - l0
        per_step = sorted(a.elapsed_time(b) for a, b in evs)  # this rank's sweep regions (20 sweeps = 40 launches each)
        res = {"total_ms": total_ms, "sweep_ms": sweep_ms, "launches": launches, "E": int(E[0]), "M": int(M[0]),
               "sweep_ms_median": per_step[len(per_step) // 2], "sweep_ms_best": per_step[0]}
        # end to end through host buffers
        if not args.no_e2e:
            for _ in range(2):
                g.ising_set_t(0)
                g.ising_run_host(h_spins, h_J, BETA, nsw, h_out)
            barrier()
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(args.steps):
                g.ising_set_t(0)
                Eh, Mh = g.ising_run_host(h_spins, h_J, BETA, nsw, h_out)
            e1.record(stream)
            barrier()
            res["e2e_ms"] = max_over_ranks(e0.elapsed_time(e1))
            res["e2e_wall_ms"] = 1e3 * (time.perf_counter() - t0)
            assert int(Eh[0]) == res["E"], "e2e path and device path disagree"
            # the same jobs pipelined: NSLOT handles (workspaces) on NSLOT streams through ising_run_host_async, so that the PCIe
            # copies of a job (10 ms in, 2.5 ms out) run under the sweeps of the others (16 ms); every job still copies its own
            # inputs in and its results out.  Two figures: (1) K jobs from an idle device, the fill (first copy in) and the drain
            # (last copy out) inside the timed region: the contract's e2e; (2) the steady state of the same pipeline: the time
            # between the completions of job W - 1 and job W + K - 1 of one continuous stream of W + K jobs.
            NSLOT = 3
            hs = [g] + [Ising(L, 1, synth.DYN_SEED, rng_mode) for _ in range(NSLOT - 1)]
            sts = [torch.cuda.Stream() for _ in range(NSLOT)]
            outs = [h_out] + [torch.empty_like(h_spins).pin_memory() for _ in range(NSLOT - 1)]
            EM = [(torch.zeros(1, dtype=torch.int64).pin_memory(), torch.zeros(1, dtype=torch.int64).pin_memory())
                  for _ in range(NSLOT)]
            done = [torch.cuda.Event() for _ in range(NSLOT)]

            def job(k):
                i = k % NSLOT
                hs[i].ising_set_t(0)
                hs[i].ising_run_host_async(h_spins, h_J, BETA, nsw, outs[i], EM[i][0], EM[i][1], stream=sts[i])

            barrier()
            for k in range(NSLOT):
                job(k)
            barrier()
            e0.record(stream)
            for st in sts:
                st.wait_event(e0)
            for k in range(args.steps):
                job(k)
            for i in range(NSLOT):
                done[i].record(sts[i])
                stream.wait_event(done[i])
            e1.record(stream)
            barrier()
            res["e2e_pipelined_ms"] = max_over_ranks(e0.elapsed_time(e1))
            for i in range(min(NSLOT, args.steps)):
                assert int(EM[i][0][0]) == res["E"] and int(EM[i][1][0]) == res["M"], "pipelined e2e path disagrees"
                assert torch.equal(outs[i], d_out.cpu()), "pipelined e2e spins disagree with the device path"
            # steady state
            Wj = NSLOT + 1
            marks = []
            for k in range(Wj + args.steps):
                job(k)
                ev = torch.cuda.Event(enable_timing=True)
                ev.record(sts[k % NSLOT])
                marks.append(ev)
            barrier()
            res["e2e_steady_ms"] = max_over_ranks(marks[Wj - 1].elapsed_time(marks[Wj + args.steps - 1]))
            res["e2e_slots"] = NSLOT
            for h in hs[1:]:
                h.ising_destroy()
        g.ising_destroy()
        return res

    def bench_shared(Ls, ns, sweeps, mode=2):
        """the paper's own scheme, one draw per 32-sample word (rng_mode 2); rank 2: the same with the
        draws taken from stored-state lane generators (rng_mode 3 Parisi-Rapuano, 4 MT19937); sweeps only."""
        sp = torch.from_numpy(synth.make_spins(Ls, ns).view(np.int32)).cuda()
        Jc = torch.from_numpy(synth.make_couplings(Ls, ns).view(np.int32)).cuda()
        g = Ising(Ls, ns, synth.DYN_SEED, mode)
        g.ising_load_state(sp, Jc)
        g.ising_sweep(BETA, 2)
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        g.ising_sweep(BETA, sweeps)
        b.record(stream)
        barrier()
        ms = a.elapsed_time(b)
        g.ising_destroy()
        flips = sweeps * ns * Ls**3
        bpf = ALG_BYTES_PER_FLIP + LANE_STATE_BYTES_PER_DRAW.get(mode, 0.0) / 32.0  # one draw serves 32 flip attempts
        gbs = bpf * flips / (ms * 1e-3) / 1e9
        gen = {2: "one Philox draw", 3: "one Parisi-Rapuano draw (62-word state per lane, strided)",
               4: "one MT19937 draw (624-word state per lane, strided)"}[mode]
        return {"workload": f"L={Ls} cube x {ns} samples ({ns // 32} coded batches), {sweeps} sweeps, {gen} per 32-sample word",
                "value": 1e9 * ms / flips, "unit": UNIT, "half_sweep_us": 1e3 * ms / (2 * sweeps),
                "roofline": {"bound": "hbm", "achieved": gbs, "unit": "GB/s", "alg_bytes_per_flip": bpf}}

    def bench_table2(kind, nlanes=148 * 1024, ndraws=4096, reps=10):
        """PAPER.md Table II, the device-API generator test: every lane draws numbers and counts the odd ones; instances/s."""
        from paper_1411_0127_b200 import binding

        nbytes = binding.ising_prng_state_bytes(kind, nlanes)
        state = torch.empty(nbytes, dtype=torch.uint8, device="cuda") if nbytes else None
        odd = torch.zeros(nlanes, dtype=torch.int64, device="cuda")
        tot = torch.zeros(nlanes, dtype=torch.int64, device="cuda")
        a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        a.record(stream)
        binding.ising_prng_init(kind, synth.DYN_SEED, nlanes, state)
        b.record(stream)
        binding.ising_prng_count_odd(kind, synth.DYN_SEED, nlanes, 0, ndraws, state, odd, tot)  # warm-up
        torch.cuda.synchronize()
        b2 = torch.cuda.Event(enable_timing=True)
        b2.record(stream)
        for r in range(reps):
            binding.ising_prng_count_odd(kind, synth.DYN_SEED, nlanes, (r + 1) * ndraws, ndraws, state, odd, tot)
        c.record(stream)
        torch.cuda.synchronize()
        ms = b2.elapsed_time(c)
        n = nlanes * ndraws * reps
        frac_odd = float(odd.sum().item()) / (nlanes * ndraws)
        row = {"generator": {0: "philox4x32-10", 1: "minstd", 3: "parisi-rapuano", 4: "mt19937"}[kind], "lanes": nlanes,
               "draws_per_lane": ndraws, "reps": reps, "instances_per_s": n / (ms * 1e-3), "t_init_ms": a.elapsed_time(b),
               "fraction_odd_last_rep": frac_odd}
        bpd = LANE_STATE_BYTES_PER_DRAW.get(kind)
        if bpd:
            row["state_bytes_per_draw"] = bpd
            row["state_GBps"] = bpd * n / (ms * 1e-3) / 1e9
        return row

    def bench_lanes():
        return {"sweep": [bench_shared(512, 32, 4, 3), bench_shared(512, 32, 4, 4), bench_shared(128, 256, 20, 3)],
                "table2_device_api": [bench_table2(k) for k in (0, 1, 3, 4)],
                # the launch configuration of the paper's Table II: 64 blocks x 256 threads, 2^15 draws each, 10 times
                "table2_paper_launch_configuration": [bench_table2(k, nlanes=64 * 256, ndraws=1 << 15, reps=10) for k in (0, 1, 3, 4)]}

    if args.scan:
        from paper_1411_0127_b200 import PHILOX_SHARED

        rows = []
        cases = [(Ls, 1, m) for Ls in (64, 128, 256, 512, 1024, 2048, 3072, 4096) for m in (PHILOX, MINSTD)]
        cases += [(Ls, 32, m) for Ls in (32, 64, 128, 256) for m in (PHILOX, MINSTD)]
        cases += [(64, 32, PHILOX_SHARED), (128, 32, PHILOX_SHARED), (128, 256, PHILOX_SHARED), (256, 32, PHILOX_SHARED),
                  (512, 32, PHILOX_SHARED)]
        for Ls, ns, mode in cases:
            if Ls > 2048:   # 3.4-8.6 GiB of spin bits: random bits drawn on the device (the recipe's SplitMix64 stream on the host takes minutes)
                gen = torch.Generator(device="cuda").manual_seed(Ls)
                sp = torch.randint(-2**31, 2**31 - 1, (1, Ls**3 // 32), dtype=torch.int32, device="cuda", generator=gen)
                Jc = torch.randint(-2**31, 2**31 - 1, (1, 3, Ls**3 // 32), dtype=torch.int32, device="cuda", generator=gen)
            else:
                sp = torch.from_numpy(synth.make_spins(Ls, ns).view(np.int32)).cuda()
                Jc = torch.from_numpy(synth.make_couplings(Ls, ns).view(np.int32)).cuda()
            g = Ising(Ls, ns, synth.DYN_SEED, mode)
            g.ising_load_state(sp, Jc)
            nsweeps = max(2, min(200, int(2e10 / (ns * Ls**3))))
            g.ising_sweep(BETA, nsweeps if ns * Ls**3 <= 256**3 else 2)   # warm-up (small lattices: the same call, so that its CUDA graph exists)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            g.ising_sweep(BETA, nsweeps)
            b.record(stream)
            torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            g.ising_destroy()
            del g, sp, Jc
            rows.append({"L": Ls, "nsamples": ns, "rng_mode": ["philox", "minstd", "philox_shared"][mode], "sweeps": nsweeps,
                         "half_sweep_us": 1e3 * ms / (2 * nsweeps), "ps_per_flip": 1e9 * ms / (nsweeps * ns * Ls**3)})
        print(json.dumps({"scan": rows}))
        return

    if args.slab_ranks:
        # Strong scaling by z-slab decomposition.  Not the default N > 1 path (replicas), and NOT measured on more
        # than one GPU in this build (one GPU per gpurun call): with WORLD_SIZE = 1 the slab is the whole lattice with halos and the
        # exchange is a local copy.
        from paper_1411_0127_b200 import IsingSlab, slabs

        slab = IsingSlab(L, world, rank, synth.DYN_SEED, PHILOX)
        full_spins = torch.from_numpy(synth.make_spins(L).view(np.int32)).cuda()     # every rank builds the same lattice (seeds 2 / 1)
        full_J = torch.from_numpy(synth.make_couplings(L).view(np.int32)).cuda()
        bulk_stream = torch.cuda.Stream()

        def step():
            slab.ising_set_t(0)
            slab.ising_load_state(full_spins, full_J)
            slabs.slab_sweep_distributed(slab, BETA, nsw, dist, rank, world, bulk_stream)
            return slab.ising_energy()

        for _ in range(args.warmup):
            step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            E, M = step()
        e1.record(stream)
        barrier()
        ms = max_over_ranks(e0.elapsed_time(e1))
        Et = torch.tensor([int(E[0]), int(M[0])], dtype=torch.int64, device="cuda")
        if dist is not None:
            dist.all_reduce(Et)
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": 1e9 * ms / (args.steps * nsw * N), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                              "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": False, "scaling": "strong",
                              "vs_baseline": None, "dtype": "u32", "data": "synthetic",
                              "config": {**headline_config(L, nsw, world), "parallelism": f"{world} z-slabs of {L // world} planes, one per GPU",
                                         "step": "load_state of the slab + sweeps (boundary kernel, plane exchange, bulk kernel) + energy share"},
                              "final_energy": int(Et[0]), "final_magnetisation": int(Et[1]),
                              "exchange_bytes_per_half_sweep_per_rank": 2 * L * L // 16}))
        if dist is not None:
            dist.destroy_process_group()
        return

    if args.sliced:
        rows = []
        for Ls in ([int(v) for v in args.sizes.split(",")] if args.sizes else [256, 512, 1024]):
            sp = torch.from_numpy(synth.make_spins(Ls, 1).view(np.int32)).cuda()
            Jc = torch.from_numpy(synth.make_couplings(Ls, 1).view(np.int32)).cuda()
            for mode, choice in ((PHILOX, 3), (MINSTD, 2)):   # one launch per half-sweep on both sides; MINSTD seeds recomputed on both
                g = Ising(Ls, 1, synth.DYN_SEED, mode)
                g.ising_set_kernel(choice)
                g.ising_load_state(sp, Jc)
                nsweeps = max(2, min(50, int(4e9 / Ls**3)))
                res = {}
                for name in ("rank_linear", "sliced"):
                    if name == "sliced":
                        g.ising_sliced_begin()
                    sweep = (lambda n: g.ising_sliced_sweep(BETA, n)) if name == "sliced" else (lambda n: g.ising_sweep(BETA, n))
                    sweep(1)
                    best = None
                    for _ in range(3):
                        torch.cuda.synchronize()
                        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        a.record(stream)
                        sweep(nsweeps)
                        b.record(stream)
                        torch.cuda.synchronize()
                        ms = a.elapsed_time(b)
                        best = ms if best is None or ms < best else best
                    if name == "sliced":
                        g.ising_sliced_end()
                    res[name] = best
                g.ising_destroy()
                rows.append({"L": Ls, "rng_mode": ["philox", "minstd (seeds recomputed)"][mode], "sweeps": nsweeps,
                             "rank_linear_half_sweep_us": 1e3 * res["rank_linear"] / (2 * nsweeps),
                             "sliced_half_sweep_us": 1e3 * res["sliced"] / (2 * nsweeps),
                             "rank_linear_ps_per_flip": 1e9 * res["rank_linear"] / (nsweeps * Ls**3),
                             "sliced_ps_per_flip": 1e9 * res["sliced"] / (nsweeps * Ls**3)})
            del sp, Jc
        print(json.dumps({"sliced": rows}))
        return

    if args.slabs:
        from paper_1411_0127_b200 import IsingSlab, binding

        rows = []
        for mode in (PHILOX, MINSTD):
            ref = Ising(L, 1, synth.DYN_SEED, mode)
            ref.ising_load_state(d_spins, d_J)
            ref.ising_sweep(BETA, 2)
            times, times_push = {}, {}
            for G in sorted({1, args.slabs}):
                hs = [IsingSlab(L, G, r, synth.DYN_SEED, mode) for r in range(G)]
                for h in hs:
                    h.ising_load_state(d_spins, d_J)
                sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
                binding.ising_slab_sweep_local(hs, BETA, 2, sa, sb)
                torch.cuda.synchronize()
                best = None
                for _ in range(3):
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(sa)
                    binding.ising_slab_sweep_local(hs, BETA, nsw, sa, sb)
                    b.record(sa)
                    torch.cuda.synchronize()
                    ms = a.elapsed_time(b)
                    best = ms if best is None or ms < best else best
                times[G] = best
                best = None
                for _ in range(3):   # the exchange fused into the boundary kernels (ising_slab_connect), no copies
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(sa)
                    binding.ising_slab_sweep_local(hs, BETA, nsw, sa, sb, push=True)
                    b.record(sa)
                    torch.cuda.synchronize()
                    ms = a.elapsed_time(b)
                    best = ms if best is None or ms < best else best
                times_push[G] = best
                out = torch.zeros_like(d_out)
                for h in hs:
                    h.ising_get_spins(out)
                del hs
            best = None
            for _ in range(3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                ref.ising_sweep(BETA, nsw)
                b.record(stream)
                torch.cuda.synchronize()
                ms = a.elapsed_time(b)
                best = ms if best is None or ms < best else best
            ref.ising_destroy()
            rows.append({"L": L, "rng_mode": ["philox", "minstd"][mode], "sweeps": nsw, "undivided_ms": best,
                         "undivided_ps_per_flip": 1e9 * best / (nsw * N),
                         **{f"slabs_{G}_ms": t for G, t in times.items()},
                         **{f"slabs_{G}_over_undivided": t / best for G, t in times.items()},
                         **{f"slabs_{G}_fused_exchange_ms": t for G, t in times_push.items()},
                         **{f"slabs_{G}_fused_exchange_over_undivided": t / best for G, t in times_push.items()}})
        print(json.dumps({"slabs": rows}))
        return

    if args.small:
        rows = []
        for Ls in (8, 16, 24, 32, 40, 64, 128, 192, 256, 320, 384, 448):
            sp = torch.from_numpy(synth.make_spins(Ls, 1).view(np.int32)).cuda()
            Jc = torch.from_numpy(synth.make_couplings(Ls, 1).view(np.int32)).cuda()
            for mode in (PHILOX, MINSTD):
                row = {"L": Ls, "rng_mode": ["philox", "minstd"][mode]}
                for every in (0, 1):
                    for choice in (0, 3, 5, 4):
                        g = Ising(Ls, 1, synth.DYN_SEED, mode)
                        g.ising_set_kernel(choice)
                        g.ising_load_state(sp, Jc)
                        g.ising_sweep(BETA, 2)
                        nsweeps = 500 if Ls <= 256 else 100
                        best = None
                        for _ in range(3):
                            torch.cuda.synchronize()
                            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                            a.record(stream)
                            if every:
                                g.ising_sweep_trace(BETA, nsweeps, every_half_sweeps=every)
                            else:
                                g.ising_sweep(BETA, nsweeps)
                            b.record(stream)
                            torch.cuda.synchronize()
                            ms = a.elapsed_time(b)
                            best = ms if best is None or ms < best else best
                        g.ising_destroy()
                        name = {0: "automatic", 3: "launch_per_half_sweep", 5: "automatic_without_cluster_kernel", 4: "persistent"}[choice]
                        row[("recorded_" if every else "") + name + "_us"] = round(1e3 * best / (2 * nsweeps), 3)
                rows.append(row)
        # many samples with their own draws: the paper's sample-packed storage, the batch of site-packed lattices by launches, and the
        # automatic choice (batch; at L = 64 the cluster-resident kernel where it is faster)
        from paper_1411_0127_b200 import LAYOUT_BATCH, LAYOUT_SAMPLE_PACKED
        many = []
        for Ls, ns in ((64, 32), (64, 64), (64, 128), (64, 256), (128, 32), (256, 32)):
            sp = torch.from_numpy(synth.make_spins(Ls, ns).view(np.int32)).cuda()
            Jc = torch.from_numpy(synth.make_couplings(Ls, ns).view(np.int32)).cuda()
            for mode in (PHILOX, MINSTD):
                row = {"L": Ls, "nsamples": ns, "rng_mode": ["philox", "minstd"][mode]}
                for name, layout, choice in (("sample_packed", LAYOUT_SAMPLE_PACKED, 0), ("batch_launches", LAYOUT_BATCH, 3),
                                             ("automatic", 0, 0)):
                    g = Ising(Ls, ns, synth.DYN_SEED, mode, layout=layout)
                    g.ising_set_kernel(choice)
                    g.ising_load_state(sp, Jc)
                    nsweeps = max(4, min(500, int(4e10 / (Ls**3 * ns)) // 2))
                    g.ising_sweep(BETA, nsweeps)
                    for every in (0, 20):
                        best = None
                        for _ in range(3):
                            torch.cuda.synchronize()
                            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                            a.record(stream)
                            if every:
                                g.ising_sweep_trace(BETA, nsweeps, every_half_sweeps=every)
                            else:
                                g.ising_sweep(BETA, nsweeps)
                            b.record(stream)
                            torch.cuda.synchronize()
                            ms = a.elapsed_time(b)
                            best = ms if best is None or ms < best else best
                        row[("recorded_every_20_" if every else "") + name + "_us"] = round(1e3 * best / (2 * nsweeps), 3)
                        row[("recorded_every_20_" if every else "") + name + "_ps_per_flip"] = round(1e9 * best / (nsweeps * ns * Ls**3), 4)
                    g.ising_destroy()
                many.append(row)
            del sp, Jc
        print(json.dumps({"small": rows, "many_samples": many}))
        return

    if args.configs:  # BASELINE.json configs 1-5 as written: sweeps, and the observables each one records, inside the timed region
        from paper_1411_0127_b200 import binding

        def oracle_outputs(idx, cfg, sp_np, J_np):
            """The outputs config `idx` names, from the CPU oracle (outside every timed region; --no-verify skips it)."""
            from oracle import ea3d

            o = ea3d.Oracle(cfg["L"], cfg["nsamples"], synth.DYN_SEED, cfg["rng_mode"])
            o.load_packed(sp_np, J_np)
            beta, nsweeps = cfg["beta"], cfg["sweeps"]
            out = {}
            if idx == 1:
                E = []
                for _ in range(2 * nsweeps):
                    o.half_sweep(beta)
                    E.append(int(o.energy()[0][0]))
                out["E"] = E
                out["spins_fnv"] = ea3d.fnv1a64(o.spins_packed())
            elif idx == 2:
                E = []
                for _ in range(nsweeps // 10):
                    o.sweep(beta, 10)
                    E.append([int(v) for v in o.energy()[0]])
                out["E"] = E
            elif idx == 3:
                E, M = [], []
                for _ in range(nsweeps):
                    o.sweep(beta, 1)
                    e, m = o.energy()
                    E.append(int(e[0]))
                    M.append(int(m[0]))
                out["E"], out["M"] = E, M
            elif idx == 4:
                F = []
                for _ in range(nsweeps // 10):
                    o.sweep(beta, 10)
                    F.append(ea3d.fnv1a64(o.spins_packed()))
                out["fnv"] = F
            else:
                o.sweep(beta, nsweeps)
                out["E"] = [int(o.energy()[0][0])]
                out["spins_fnv"] = ea3d.fnv1a64(o.spins_packed())
            return out

        rows = []
        from paper_1411_0127_b200 import LAYOUT_AUTO, LAYOUT_SAMPLE_PACKED

        # config 2 twice: in the library's own layout for 32 samples with their own draws (a batch of site-packed lattices, run by the
        # cluster-resident kernel) and in the paper's sample-packed storage, "one sample per bit of each uint32"
        for idx, layout in ((1, LAYOUT_AUTO), (2, LAYOUT_AUTO), (2, LAYOUT_SAMPLE_PACKED), (3, LAYOUT_AUTO), (4, LAYOUT_AUTO), (5, LAYOUT_AUTO)):
            cfg, sp_np, J_np = synth.make_config(idx)
            Ls, ns, nsweeps, beta = cfg["L"], cfg["nsamples"], cfg["sweeps"], cfg["beta"]
            sp = torch.from_numpy(sp_np.view(np.int32)).cuda()
            Jc = torch.from_numpy(J_np.view(np.int32)).cuda()
            g = Ising(Ls, ns, synth.DYN_SEED, cfg["rng_mode"], layout=layout)
            out = torch.empty_like(sp)
            if idx == 4:   # the ten checksums are computed on the device (ising_fnv1a64) and read back at the end
                fnv_out = torch.empty(nsweeps // 10, dtype=torch.int64, device="cuda")
                fnv_scratch = torch.empty(binding.ising_fnv1a64_scratch_bytes(sp.numel() * 4), dtype=torch.uint8, device="cuda")

            def run():
                """Returns the device tensors / host values the config asks for (converted to Python after the timed region)."""
                g.ising_set_t(0)
                g.ising_load_state(sp, Jc)
                if idx == 1:      # final spins and energy per half-sweep
                    E, _ = g.ising_sweep_trace(beta, nsweeps, every_half_sweeps=1, want_M=False)
                    g.ising_get_spins(out)
                    return {"E": E, "spins": out}
                if idx == 2:      # energy per site every 10 sweeps
                    E, _ = g.ising_sweep_trace(beta, nsweeps, every_half_sweeps=20, want_M=False)
                    return {"E": E}
                if idx == 3:      # energy and magnetisation per sweep
                    E, M = g.ising_sweep_trace(beta, nsweeps, every_half_sweeps=2)
                    return {"E": E, "M": M}
                if idx == 4:      # 64-bit FNV-1a of the packed spin words every 10 sweeps
                    # FNV-1a looks sequential (h = (h ^ byte) * prime: 17 ms per 16 MiB on a host core, which made this
                    # configuration a hashing benchmark); csrc/fnv_kernels.cuh computes the same number in parallel on the device
                    for k in range(nsweeps // 10):
                        g.ising_sweep(beta, 10)
                        g.ising_get_spins(out)
                        binding.ising_fnv1a64(out, out=fnv_out[k:k + 1], scratch=fnv_scratch)
                    return {"fnv": fnv_out}
                g.ising_sweep(beta, nsweeps)
                E, _ = g.ising_energy()
                g.ising_get_spins(out)
                return {"E": E, "spins": out}

            run()
            torch.cuda.synchronize()
            l0 = g.ising_kernel_launches()
            t0 = time.perf_counter()
            res = run()
            torch.cuda.synchronize()
            wall = time.perf_counter() - t0
            launches = g.ising_kernel_launches() - l0
            got = {}
            if "E" in res:
                Eh = res["E"].cpu().numpy()
                got["E"] = Eh.tolist() if idx == 2 else [int(v) for v in Eh.reshape(-1)]
            if "M" in res:
                got["M"] = [int(v) for v in res["M"].cpu().numpy().reshape(-1)]
            if "spins" in res:
                got["spins_fnv"] = binding.ising_fnv1a64_host(res["spins"].cpu().numpy())
            if "fnv" in res:
                got["fnv"] = [int(v) & (2**64 - 1) for v in res["fnv"].cpu().tolist()]
            g.ising_destroy()
            row = {"config": idx, "layout": "sample-packed (on request)" if layout == LAYOUT_SAMPLE_PACKED else
                   ("batch of site-packed lattices" if ns > 1 else "site-packed"),
                   "L": Ls, "nsamples": ns, "sweeps": nsweeps, "rng_mode": cfg["rng_mode"], "wall_ms": 1e3 * wall,
                   "ps_per_flip_including_outputs": 1e12 * wall / (nsweeps * ns * Ls**3), "kernel_launches": launches,
                   "us_per_half_sweep_including_outputs": 1e6 * wall / (2 * nsweeps),
                   "last_output": got["fnv"][-1] if "fnv" in got else (got["E"][-1] if idx != 2 else got["E"][-1][0])}
            if not args.no_verify:
                want = oracle_outputs(idx, cfg, sp_np, J_np)
                assert got == want, f"config {idx}: outputs differ from the oracle's"
                row["outputs_equal_oracle"] = True
                row["outputs_compared"] = {k: (len(v) if isinstance(v, list) else 1) for k, v in want.items()}
            rows.append(row)
            del sp, Jc, out
        print(json.dumps({"configs": rows}))
        return

    if args.aux:  # measurement of the rows outside the headline step: every layout's load / energy / get and half-sweep
        def avg_ms(fn, n=5):
            fn()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(n):
                fn()
            b.record(stream)
            torch.cuda.synchronize()
            return a.elapsed_time(b) / n

        rows = []
        for Ls, ns, mode, what in ((1024, 1, 0, "site-packed, L multiple of 64 (word-parallel kernels)"),
                                   (1000, 1, 0, "site-packed, general even L (bit-window kernels)"),
                                   (250, 1, 0, "site-packed, general even L (bit-window kernels)"),
                                   (512, 32, 2, "sample-packed, L multiple of 32 (tile load/get, bit-sliced energy)"),
                                   (128, 256, 2, "sample-packed, 8 coded batches"),
                                   (100, 32, 2, "sample-packed, general even L (one bit at a time load/get)")):
            sp = torch.from_numpy(synth.make_spins(Ls, ns).view(np.int32)).cuda()
            Jc = torch.from_numpy(synth.make_couplings(Ls, ns).view(np.int32)).cuda()
            out = torch.empty_like(sp)
            g = Ising(Ls, ns, synth.DYN_SEED, mode)
            state = ns * Ls**3 / 8 * 4  # packed spins + couplings, bytes
            t_load = avg_ms(lambda: g.ising_load_state(sp, Jc))
            t_sweep = avg_ms(lambda: g.ising_sweep(BETA, 2)) / 4
            t_energy = avg_ms(lambda: g.ising_energy())
            t_get = avg_ms(lambda: g.ising_get_spins(out))
            g.ising_destroy()
            rows.append({"L": Ls, "nsamples": ns, "layout": what, "rng_mode": mode,
                         "load_state_ms": t_load, "load_GBps_read_plus_write": 2 * state / t_load / 1e6,
                         "energy_ms": t_energy, "energy_GBps": state / t_energy / 1e6,
                         "get_spins_ms": t_get, "get_GBps_read_plus_write": 2 * state / 4 / t_get / 1e6,
                         "half_sweep_us": 1e3 * t_sweep, "ps_per_flip": 2e9 * t_sweep / (ns * Ls**3)})
            del sp, Jc, out
        print(json.dumps({"aux": rows}))
        return

    if args.scan_batches:  # PAPER.md:308-310, Fig. 4: t_SW stays flat in k until the GPU is full, then grows linearly
        rows = []
        for Ls, ks in ((8, (1, 8, 64, 512, 4096)), (16, (1, 8, 64, 512)), (32, (1, 8, 64)), (64, (1, 8))):
            for k in ks:
                sp = torch.from_numpy(synth.make_spins(Ls, 32 * k).view(np.int32)).cuda()
                Jc = torch.from_numpy(synth.make_couplings(Ls, 32 * k).view(np.int32)).cuda()
                for mode in (2, 3, 4):
                    g = Ising(Ls, 32 * k, synth.DYN_SEED, mode)
                    g.ising_load_state(sp, Jc)
                    g.ising_sweep(BETA, 2)
                    torch.cuda.synchronize()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    g.ising_sweep(BETA, 50)
                    b.record(stream)
                    torch.cuda.synchronize()
                    ms = a.elapsed_time(b)
                    g.ising_destroy()
                    rows.append({"L": Ls, "batches": k, "rng_mode": {2: "philox_shared", 3: "parisi_rapuano_lanes", 4: "mt19937_lanes"}[mode],
                                 "half_sweep_us": 1e3 * ms / 100, "ps_per_flip": 1e9 * ms / (50 * 32 * k * Ls**3)})
        print(json.dumps({"scan_batches": rows}))
        return

    if args.only_shared:
        print(json.dumps({"amsc_shared_random_number": [bench_shared(512, 32, 4)]}))
        return
    if args.only_lanes:
        print(json.dumps({"amsc_lane_generators": bench_lanes()}))
        return

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    philox = bench_mode(PHILOX)
    clocks = sampler.stop() if rank == 0 else None
    minstd = None if args.no_minstd else bench_mode(MINSTD)

    shared = lanes = None
    if world == 1 and not args.no_shared:
        shared = [bench_shared(128, 256, 20), bench_shared(512, 32, 4)]
        lanes = bench_lanes()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    hbm_gbs, sm_max_mhz, peaks_src = measured_peaks()
    flips_per_step = world * nsw * N
    K = args.steps

    traffic_note = None
    traffic_tab = {0: None, 1: None}
    if L == 1024:
        if NCU_TRAFFIC_L1024["kernel_sources_sha256"] == kernel_sources_hash():
            traffic_tab = {0: NCU_TRAFFIC_L1024[0], 1: NCU_TRAFFIC_L1024[1]}
            traffic_note = f"dram__bytes_read.sum + dram__bytes_write.sum per launch, ncu --set full capture {NCU_TRAFFIC_L1024['capture']} of these kernel sources"
        else:
            traffic_note = (f"null: the last ncu capture ({NCU_TRAFFIC_L1024['capture']}) was taken on other kernel sources than the ones "
                            "timed here (kernel_sources_hash differs)")

    # the IMAD.WIDE issue rate of this very part, measured now by the committed microbenchmark (csrc/int_peak.cu, mix 1)
    imad_wide_per_clk_sm = None
    try:
        from paper_1411_0127_b200 import int_peak

        r = int_peak.run(mixes=(1,))["mixes"]["IMAD.WIDE.U32 only"]
        imad_wide_per_clk_sm = r["inst_per_clk_per_sm_at_1965MHz"] * 1965.0 / sm_max_mhz
    except Exception as exc:  # the headline line must not depend on the microbenchmark
        traffic_note = (traffic_note or "") + f" [int_peak unavailable: {exc}]"

    def summarize(res, rng_mode):
        ps = replicas.ps_per_flip(res["total_ms"], K, world, nsw, L)
        half_sweep_ms = res["sweep_ms"] / (K * 2 * nsw)            # average launch duration of the dominant kernel
        flips_per_launch = N / 2
        hbm = ALG_BYTES_PER_FLIP * flips_per_launch / (half_sweep_ms * 1e-3) / 1e9
        hbm_obj = {"achieved": hbm, "peak": hbm_gbs, "unit": "GB/s", "frac": hbm / hbm_gbs, "alg_bytes_per_flip": ALG_BYTES_PER_FLIP,
                   "alg_bytes_per_launch": ALG_BYTES_PER_FLIP * flips_per_launch, "peak_source": peaks_src + " (burst copy)"}
        common = {"traffic": traffic_tab[rng_mode], "traffic_note": traffic_note,
                  "kernel": "half_sweep_site_packed", "kernel_ms": half_sweep_ms, "kernel_ps_per_flip": 1e9 * half_sweep_ms / flips_per_launch,
                  "kernel_ms_median": res["sweep_ms_median"] / (2 * nsw), "kernel_ms_best": res["sweep_ms_best"] / (2 * nsw)}
        peak = 148 * 4 * 16 * sm_max_mhz * 1e6 / 1e12               # one pipe: 148 SMs x 4 SMSPs x 16 lanes x max clock
        if rng_mode == 1:
            # the roofline is the slower of HBM at 1.125 B/flip and the integer bound.  For MINSTD the
            # integer bound is the STATELESS evaluation (16.69 alu instructions per flip on one 16-lane pipe per SMSP).  The
            # shipped kernel trades that work for a stream of cached seed states (4 B per flip, implementation traffic, not
            # algorithmic), so it can run faster than that bound: frac > 1 is annotated, not a roofline violation.
            int_ps = 1e12 * MINSTD_STATELESS_ALU_OPS_PER_FLIP / (peak * 1e12)
            hbm_ps = 1e12 * ALG_BYTES_PER_FLIP / (hbm_gbs * 1e9)
            kernel_ps = 1e9 * half_sweep_ms / flips_per_launch
            impl_bytes = ALG_BYTES_PER_FLIP + MINSTD_TABLE_BYTES_PER_FLIP
            impl_gbs = impl_bytes * flips_per_launch / (half_sweep_ms * 1e-3) / 1e9
            return ps, {"bound": "alu", "achieved": MINSTD_STATELESS_ALU_OPS_PER_FLIP * flips_per_launch / (half_sweep_ms * 1e-3) / 1e12,
                        "peak": peak, "unit": "Tinst/s", "frac": int_ps / kernel_ps,
                        "frac_note": "above 1: the kernel reads cached seed states (implementation_traffic) instead of doing the stateless "
                                     "generator's integer work, which is what the bound counts" if int_ps / kernel_ps > 1 else None,
                        "roofline_ps_per_flip": max(int_ps, hbm_ps), "alg_alu_ops_per_flip_stateless": MINSTD_STATELESS_ALU_OPS_PER_FLIP,
                        "hbm": hbm_obj,
                        "implementation_traffic": {"bytes_per_flip": impl_bytes, "achieved": impl_gbs, "peak": hbm_gbs, "unit": "GB/s",
                                                   "frac": impl_gbs / hbm_gbs,
                                                   "what": "1.125 B lattice + 4 B cached MINSTD seed state per flip attempt"},
                        **common}
        slot_rate = ALG_SLOTS_PER_FLIP[rng_mode] * flips_per_launch / (half_sweep_ms * 1e-3) / 1e12  # T slots/s
        out = {
            "bound": "alu", "achieved": slot_rate, "peak": peak, "unit": "Tinst/s", "frac": slot_rate / peak, **common,
            "binding_pipe": BINDING_PIPE[rng_mode], "alg_slots_per_flip": ALG_SLOTS_PER_FLIP[rng_mode],
            "roofline_ps_per_flip": 1e12 * ALG_SLOTS_PER_FLIP[rng_mode] / (peak * 1e12),
            # BASELINE.json's wording, "integer ops per flip (PRNG + field logic) at the INT32 issue rate": all 11.94 algorithmic
            # integer instructions per flip attempt (37/4 Philox + 2 acceptance + 22/32 field) against one 16-lane pipe per
            # SMSP (the measured LOP3 / IMAD rate) and against both pipes issuing together (the warp scheduler's limit)
            "int32_issue_reading": {"alg_int_ops_per_flip": ALG_INT_OPS_PER_FLIP,
                                    "frac_at_64_lanes_per_sm": ALG_INT_OPS_PER_FLIP * flips_per_launch / (half_sweep_ms * 1e-3) / 1e12 / peak,
                                    "frac_at_128_lanes_per_sm": ALG_INT_OPS_PER_FLIP * flips_per_launch / (half_sweep_ms * 1e-3) / 1e12 / (2 * peak)},
            "peak_source": f"guide unit counts: 148 SM x 4 SMSP x 16 lanes (rt_SMSP=2) x {sm_max_mhz:.0f} MHz ({peaks_src} max clock), per pipe; "
                           "an IMAD.WIDE counts as 2 slots",
            "hbm": hbm_obj,
        }
        if imad_wide_per_clk_sm:
            # the same fraction against what the part delivers: IMAD.WIDE alone, measured in this run (2 slots each)
            pm = 2 * imad_wide_per_clk_sm * 148 * sm_max_mhz * 1e6 / 1e12
            out.update({"peak_measured": pm, "frac_measured": slot_rate / pm,
                        "peak_measured_source": f"int_peak mix 1 in this run: {imad_wide_per_clk_sm:.2f} IMAD.WIDE thread-instructions per clock per SM "
                                                f"(guide-derived: 32), x 2 slots x 148 SMs x {sm_max_mhz:.0f} MHz"})
        return ps, out

    ps, roof = summarize(philox, 0)
    line = {
        "metric": METRIC, "value": ps, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": philox["total_ms"] / K, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic",
        "config": headline_config(L, nsw, world),
        "flips_per_s": 1e12 / ps, "roofline": roof, "gpu_launches": philox["launches"], "clocks": clocks,
        "final_energy": philox["E"],
    }
    spin_bytes, j_bytes = spins.nbytes, J.nbytes
    if "e2e_ms" in philox:
        line["e2e"] = {"value": 1e9 * philox["e2e_ms"] / (K * flips_per_step), "unit": UNIT,
                       "h2d_bytes_per_step": spin_bytes + j_bytes, "d2h_bytes_per_step": spin_bytes + 16,
                       "ms_per_step": philox["e2e_ms"] / K, "api": "ising_run_host"}
        if "e2e_pipelined_ms" in philox:
            # headline e2e = K pipelined jobs from an idle device (fill and drain included); the steady state of the same pipeline
            # and the one-job-at-a-time figure beside it
            ns = philox["e2e_slots"]
            line["e2e"] = {"value": 1e9 * philox["e2e_pipelined_ms"] / (K * flips_per_step), "unit": UNIT,
                           "h2d_bytes_per_step": spin_bytes + j_bytes, "d2h_bytes_per_step": spin_bytes + 16,
                           "ms_per_step": philox["e2e_pipelined_ms"] / K,
                           "api": f"ising_run_host_async, {ns} handles on {ns} streams (copies of one job under the sweeps of the others); "
                                  f"{K} jobs from an idle device: the first copy in (fill) and the last copy out (drain) are inside the timed region",
                           "steady_state": {"value": 1e9 * philox["e2e_steady_ms"] / (K * flips_per_step), "unit": UNIT,
                                            "ms_per_step": philox["e2e_steady_ms"] / K,
                                            "what": f"the same pipeline kept full: time between the completions of job {ns} and job {ns} + {K} of "
                                                    f"{ns + 1 + K} jobs issued back to back; every job copies {spin_bytes + j_bytes} B in and {spin_bytes + 16} B out"},
                           "serial": line["e2e"]}
    if minstd is not None:
        ps_m, roof_m = summarize(minstd, 1)
        line["minstd"] = {"value": ps_m, "unit": UNIT, "ms_per_step": minstd["total_ms"] / K, "roofline": roof_m,
                          "flips_per_s": 1e12 / ps_m}
        if "e2e_ms" in minstd:
            line["minstd"]["e2e"] = 1e9 * minstd["e2e_ms"] / (K * flips_per_step)
        if "e2e_pipelined_ms" in minstd:
            line["minstd"]["e2e_pipelined"] = 1e9 * minstd["e2e_pipelined_ms"] / (K * flips_per_step)
            line["minstd"]["e2e_steady_state"] = 1e9 * minstd["e2e_steady_ms"] / (K * flips_per_step)
    if shared is not None:
        hbm_gbs_, _, src_ = measured_peaks()
        for sh in shared:
            sh["roofline"].update({"peak": hbm_gbs_, "frac": sh["roofline"]["achieved"] / hbm_gbs_, "peak_source": src_ + " (burst copy)"})
        line["amsc_shared_random_number"] = shared
        for sh in lanes["sweep"]:
            sh["roofline"].update({"peak": hbm_gbs_, "frac": sh["roofline"]["achieved"] / hbm_gbs_, "peak_source": src_ + " (burst copy)"})
        line["amsc_lane_generators"] = lanes
    if world == 1 and not args.no_cpu_baseline:
        # the oracle on the workload itself (L = 1024, rank 0's inputs): 2 of its 20 sweeps per call, median of 3 calls
        tm = OracleTimer(L, spins=spins, J=J)
        times = sorted(tm.time(ORACLE_SAMPLE_SWEEPS) for _ in range(3))
        cores = tm.threads
        tm.close()
        line["cpu_baseline"] = {"value": 1e12 * times[1] / (ORACLE_SAMPLE_SWEEPS * L**3), "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": oracle_sample_text(L, ORACLE_SAMPLE_SWEEPS, f"; median of 3 calls ({times[0]:.2f} / {times[1]:.2f} / {times[2]:.2f} s)"),
                                "host_cores_visible": host_cores()}
        t1 = OracleTimer(256, threads=1)   # single-thread figure too (about 4 s)
        t1s = t1.time(8)
        t1.close()
        line["cpu_baseline"]["single_thread"] = {"value": 1e12 * t1s / (8 * 256**3), "unit": UNIT, "cores": 1,
                                                 "sample": f"L=256 cube, 8 sweeps, {t1s:.1f} s"}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
