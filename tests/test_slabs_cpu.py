"""z-slab exchange bookkeeping without a GPU: world_size-2 and -3 gloo runs of slabs.exchange_planes on CPU tensors."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_1411_0127_b200 import slabs
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{os.environ['PORT']}", rank=rank, world_size=world)
n = 64
for step in range(3):
    first = torch.full((n,), 1000 * step + 10 * rank + 1, dtype=torch.int32)   # "first owned plane" of this rank
    last = torch.full((n,), 1000 * step + 10 * rank + 2, dtype=torch.int32)    # "last owned plane"
    halo_low, halo_up = torch.zeros(n, dtype=torch.int32), torch.zeros(n, dtype=torch.int32)
    slabs.exchange_planes(dist, rank, world, first, last, halo_low, halo_up)
    below, above = slabs.neighbours(rank, world)
    assert int(halo_low[0]) == 1000 * step + 10 * below + 2, (rank, step, int(halo_low[0]))   # the last plane of the slab below
    assert int(halo_up[0]) == 1000 * step + 10 * above + 1, (rank, step, int(halo_up[0]))     # the first plane of the slab above
    assert bool((halo_low == halo_low[0]).all()) and bool((halo_up == halo_up[0]).all())
dist.destroy_process_group()
print("ok", rank)
''' % ROOT


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_planes_over_gloo(world):
    port = free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    for rank, p in enumerate(procs):
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0 and f"ok {rank}" in out, err[-2000:]


def test_neighbours_and_single_rank():
    import torch

    from paper_1411_0127_b200 import slabs

    assert slabs.neighbours(0, 4) == (3, 1) and slabs.neighbours(3, 4) == (2, 0) and slabs.neighbours(0, 1) == (0, 0)
    first, last = torch.arange(8), torch.arange(8) + 100
    lo, up = torch.zeros(8, dtype=torch.int64), torch.zeros(8, dtype=torch.int64)
    slabs.exchange_planes(None, 0, 1, first, last, lo, up)     # one slab: it is its own neighbour (periodic in z)
    assert torch.equal(up, first) and torch.equal(lo, last)
