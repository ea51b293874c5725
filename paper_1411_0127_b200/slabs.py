"""z-slab domain decomposition across processes (section V; include/ising.h "z-slab domain decomposition").

One process per GPU, rank r owns slab r.  A colour half-sweep is: the boundary kernel, the exchange of the updated colour's two end
planes with the two z-neighbours over torch.distributed point-to-point operations (NCCL over NVLink on GPUs; `gloo` on CPU tensors
in the tests), and the bulk kernel on a second stream meanwhile (the paper's Fig. 10 with send / recv in place of D2H + MPI + H2D).
This module holds the exchange bookkeeping only; every update runs in the library's kernels.
"""
from __future__ import annotations


def neighbours(rank: int, world: int) -> tuple[int, int]:
    """(rank of the slab below, rank of the slab above), periodic in z."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_planes(dist, rank: int, world: int, first, last, halo_low, halo_up):
    """Send `first` (this slab's first owned plane) to the slab below, where it becomes the upper halo, and `last` to the slab above,
    where it becomes the lower halo; receive the neighbours' planes into halo_low / halo_up.  All four are contiguous tensors of the
    same size.  world = 1: the slab is its own neighbour.  world = 2: both neighbours are the same rank, and the two messages of
    each direction pair up in the order they are posted (first plane, then last plane)."""
    below, above = neighbours(rank, world)
    if world == 1:
        halo_up.copy_(first)
        halo_low.copy_(last)
        return
    ops = [dist.P2POp(dist.isend, first, below), dist.P2POp(dist.isend, last, above),
           # the slab above sends its first plane down to me: my upper halo; the slab below sends its last plane up: my lower halo
           dist.P2POp(dist.irecv, halo_up, above), dist.P2POp(dist.irecv, halo_low, below)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()


def slab_sweep_distributed(slab, beta: float, nsweeps: int, dist, rank: int, world: int, bulk_stream):
    """nsweeps sweeps of the lattice whose slab `rank` is `slab` (an IsingSlab on this process's GPU).  Boundary kernel and exchange
    on the current stream, bulk kernel on `bulk_stream`."""
    import torch

    main = torch.cuda.current_stream()
    for _ in range(2 * nsweeps):
        c = slab.ising_get_t() & 1
        bulk_stream.wait_stream(main)
        slab.ising_slab_half_sweep_boundary(beta)
        exchange_planes(dist, rank, world, slab.ising_slab_plane(c, 0), slab.ising_slab_plane(c, 1), slab.ising_slab_plane(c, 2),
                        slab.ising_slab_plane(c, 3))
        slab.ising_slab_half_sweep_bulk(beta, stream=bulk_stream)
        main.wait_stream(bulk_stream)
