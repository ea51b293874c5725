"""world_size-2 gloo test (CPU) of the replicas-only N > 1 path of bench.py: ranks get different
disorder samples, the timing reduction is a max over ranks, and the aggregate metric counts every rank's flips."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1411_0127_b200 import replicas, synth


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s_seed, j_seed = replicas.replica_seeds(rank)
    spins = synth.make_spins(16, 1, s_seed)
    J = synth.make_couplings(16, 1, j_seed)
    my_ms = 10.0 + 5.0 * rank  # rank 1 is the slow one
    dist.barrier()
    total = replicas.max_over_ranks(my_ms, dist)
    digest = torch.tensor([int(spins.view(np.uint32)[:8].sum()), int(J.view(np.uint32)[:8].sum())], dtype=torch.int64)
    gathered = [torch.zeros_like(digest) for _ in range(world)]
    dist.all_gather(gathered, digest)
    if rank == 0:
        out.put((total, [g.tolist() for g in gathered]))
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    total, digests = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert total == 15.0  # max over ranks, not the mean and not rank 0's own time
    assert digests[0] != digests[1]  # the replicas are different disorder samples
    # whole-job metric: both ranks' flips over the slowest rank's time
    one = replicas.ps_per_flip(15.0, 1, 1, 20, 1024)
    two = replicas.ps_per_flip(15.0, 1, 2, 20, 1024)
    assert abs(two - one / 2) < 1e-15


def test_rank0_replica_is_config5():
    assert replicas.replica_seeds(0) == (2, 1)
    assert replicas.max_over_ranks(3.5) == 3.5
