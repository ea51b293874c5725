"""Host-side logic of the N > 1 path of bench.py: N independent replicas, one process per GPU.

The path does not shard (BASELINE.json: one GPU, no collectives), so there is no data-path collective: every rank sweeps
its own disorder sample, and the only communication is the barrier around the timed region and the max-over-ranks of
the device timings.  Works with the `nccl` backend on GPUs and with `gloo` on CPU (tests/test_multi_rank_cpu.py)."""
from __future__ import annotations


def replica_seeds(rank: int) -> tuple[int, int]:
    """(spin seed, coupling seed) of rank `rank`: rank 0 is exactly BASELINE.json config 5 (seeds 2 and 1)."""
    return 2 + 1000 * rank, 1 + 1000 * rank


def max_over_ranks(x: float, dist=None, device="cpu") -> float:
    """Max of a per-rank timing over all ranks (identity without a process group)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch

    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def ps_per_flip(total_ms: float, steps: int, world: int, sweeps: int, L: int, nsamples: int = 1) -> float:
    """Whole-job ps per spin-flip attempt (R17): the slowest rank's time over the flips all ranks attempted."""
    return 1e9 * total_ms / (steps * world * sweeps * nsamples * L**3)
