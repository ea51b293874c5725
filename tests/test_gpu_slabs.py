"""z-slab domain decomposition (-m gpu): G slabs of one lattice, all on the same GPU, must follow exactly the trajectory of the
undivided lattice and of the CPU oracle (the draws are keyed by the site's position in the whole lattice)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import MINSTD, PHILOX, Ising, IsingSlab, binding, slabs, synth  # noqa: E402

pytestmark = pytest.mark.gpu
SEED = synth.DYN_SEED


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def make_slabs(L, G, rng_mode, d_spins, d_J):
    hs = [IsingSlab(L, G, r, SEED, rng_mode) for r in range(G)]
    for h in hs:
        h.ising_load_state(d_spins, d_J)
    return hs


def gather(hs, W):
    out = torch.zeros(W, dtype=torch.int32, device="cuda")
    for h in hs:
        h.ising_get_spins(out)
    E = sum(int(h.ising_energy()[0][0]) for h in hs)
    M = sum(int(h.ising_energy()[1][0]) for h in hs)
    return out, E, M


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,G", [(64, 1), (64, 2), (64, 4), (64, 8), (128, 2), (192, 3), (256, 2), (256, 4), (320, 5)])
def test_slabs_follow_the_undivided_lattice(L, G, rng_mode):
    spins, J = synth.make_spins(L, 1, 81), synth.make_couplings(L, 1, 82)
    d_spins, d_J = dev(spins), dev(J)
    W = spins.size
    ref = Ising(L, 1, SEED, rng_mode)
    ref.ising_load_state(d_spins, d_J)
    hs = make_slabs(L, G, rng_mode, d_spins, d_J)
    got, E, M = gather(hs, W)
    assert torch.equal(got, d_spins.flatten()), "load / get round trip through the slabs"
    Er, Mr = ref.ising_energy()
    assert (E, M) == (int(Er[0]), int(Mr[0])), "energy shares of the loaded state"
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    o = None
    if L <= 64:
        o = ea3d.Oracle(L, 1, SEED, rng_mode)
        o.load_packed(spins, J)
    for beta, n in ((1 / 1.1, 3), (0.4, 2)):
        ref.ising_sweep(beta, n)
        torch.cuda.synchronize()
        binding.ising_slab_sweep_local(hs, beta, n, sa, sb)
        torch.cuda.synchronize()
        got, E, M = gather(hs, W)
        assert torch.equal(got, ref.ising_get_spins().flatten()), f"L={L}, {G} slabs, beta={beta}"
        Er, Mr = ref.ising_energy()
        assert (E, M) == (int(Er[0]), int(Mr[0]))
        assert all(h.ising_get_t() == ref.ising_get_t() for h in hs)
        if o is not None:
            o.sweep(beta, n)
            assert np.array_equal(got.cpu().numpy().view(np.uint32), o.spins_packed().reshape(-1))
            assert E == int(o.energy()[0][0]) and M == int(o.energy()[1][0])


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_slab_calls_one_by_one_with_the_exchange_done_by_the_caller(rng_mode):
    """The path a multi-GPU run takes (slabs.slab_sweep_distributed), with all ranks played by one process: boundary kernel,
    exchange of the planes ising_slab_plane names (slabs.exchange_planes' bookkeeping, here as tensor copies), bulk kernel."""
    L, G = 128, 4
    spins, J = synth.make_spins(L, 1, 83), synth.make_couplings(L, 1, 84)
    d_spins, d_J = dev(spins), dev(J)
    ref = Ising(L, 1, SEED, rng_mode)
    ref.ising_load_state(d_spins, d_J)
    hs = make_slabs(L, G, rng_mode, d_spins, d_J)
    beta = 1 / 1.1
    for _ in range(6):
        c = hs[0].ising_get_t() & 1
        for h in hs:
            h.ising_slab_half_sweep_boundary(beta)
        for r, h in enumerate(hs):
            below, above = slabs.neighbours(r, G)
            hs[below].ising_slab_plane(c, 3).copy_(h.ising_slab_plane(c, 0))   # my first plane: the upper halo of the slab below
            hs[above].ising_slab_plane(c, 2).copy_(h.ising_slab_plane(c, 1))   # my last plane: the lower halo of the slab above
        for h in hs:
            h.ising_slab_half_sweep_bulk(beta)
    ref.ising_sweep(beta, 3)
    got, E, M = gather(hs, spins.size)
    assert torch.equal(got, ref.ising_get_spins().flatten())
    assert E == int(ref.ising_energy()[0][0])


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,G", [(64, 1), (64, 2), (64, 8), (128, 4), (192, 3), (256, 2), (320, 5)])
def test_slabs_with_the_exchange_fused_into_the_boundary_kernel(L, G, rng_mode):
    """ising_slab_sweep_local_push: no plane copies; the boundary kernels store their end planes into the neighbours' halos
    themselves (ising_slab_connect).  Same trajectory as the undivided lattice (and the oracle at L = 64), for slabs of one CTA
    row (first and last plane in the same row), one slab that is its own neighbour, and every words-per-thread variant."""
    spins, J = synth.make_spins(L, 1, 85), synth.make_couplings(L, 1, 86)
    d_spins, d_J = dev(spins), dev(J)
    ref = Ising(L, 1, SEED, rng_mode)
    ref.ising_load_state(d_spins, d_J)
    hs = make_slabs(L, G, rng_mode, d_spins, d_J)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    o = None
    if L <= 64:
        o = ea3d.Oracle(L, 1, SEED, rng_mode)
        o.load_packed(spins, J)
    for beta, n in ((1 / 1.1, 3), (0.4, 2)):
        ref.ising_sweep(beta, n)
        torch.cuda.synchronize()
        l0 = sum(h.ising_kernel_launches() for h in hs)
        binding.ising_slab_sweep_local(hs, beta, n, sa, sb, push=True)
        torch.cuda.synchronize()
        assert sum(h.ising_kernel_launches() for h in hs) - l0 <= 2 * n * 2 * G     # boundary + bulk per slab and half-sweep, nothing else
        got, E, M = gather(hs, spins.size)
        assert torch.equal(got, ref.ising_get_spins().flatten()), f"L={L}, {G} slabs, beta={beta}"
        Er, Mr = ref.ising_energy()
        assert (E, M) == (int(Er[0]), int(Mr[0]))
        if o is not None:
            o.sweep(beta, n)
            assert np.array_equal(got.cpu().numpy().view(np.uint32), o.spins_packed().reshape(-1))
    # the copies and the fused exchange mix freely: both leave the same halos
    binding.ising_slab_sweep_local(hs, 0.7, 1, sa, sb)
    binding.ising_slab_sweep_local(hs, 0.7, 1, sa, sb, push=True)
    torch.cuda.synchronize()
    ref.ising_sweep(0.7, 2)
    got, E, M = gather(hs, spins.size)
    assert torch.equal(got, ref.ising_get_spins().flatten()) and E == int(ref.ising_energy()[0][0])


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_fused_exchange_call_by_call_as_a_multi_gpu_run_makes_them(rng_mode):
    """The calls of a multi-GPU run with the fused exchange, all ranks played by one process: connect each slab to its
    neighbours' halos once, then per half-sweep the pushing boundary kernel and the bulk kernel -- no exchange step at all.
    An unconnected slab refuses the pushing kernel."""
    L, G = 128, 4
    spins, J = synth.make_spins(L, 1, 87), synth.make_couplings(L, 1, 88)
    d_spins, d_J = dev(spins), dev(J)
    ref = Ising(L, 1, SEED, rng_mode)
    ref.ising_load_state(d_spins, d_J)
    hs = make_slabs(L, G, rng_mode, d_spins, d_J)
    with pytest.raises(binding.IsingError):
        hs[0].ising_slab_half_sweep_boundary_push(1.0)
    for r, h in enumerate(hs):
        below, above = slabs.neighbours(r, G)
        if r % 2 == 0:
            h.ising_slab_connect(hs[below], hs[above])
        else:   # raw addresses, as a process that opened its neighbours' workspaces over CUDA IPC would pass them
            h.ising_slab_connect([hs[below].ising_slab_plane(c, 3).data_ptr() for c in (0, 1)],
                                 [hs[above].ising_slab_plane(c, 2).data_ptr() for c in (0, 1)])
    beta = 1 / 1.1
    for _ in range(6):
        for h in hs:
            h.ising_slab_half_sweep_boundary_push(beta)
        for h in hs:
            h.ising_slab_half_sweep_bulk(beta)
    ref.ising_sweep(beta, 3)
    got, E, M = gather(hs, spins.size)
    assert torch.equal(got, ref.ising_get_spins().flatten())
    assert E == int(ref.ising_energy()[0][0])


def test_slab_argument_checks():
    with pytest.raises(binding.IsingError):
        IsingSlab(100, 2, 0, SEED, PHILOX)        # rows are not whole words
    with pytest.raises(binding.IsingError):
        IsingSlab(64, 16, 0, SEED, PHILOX)        # 4 planes per slab: not a whole row of CTAs
    with pytest.raises(binding.IsingError):
        IsingSlab(64, 2, 2, SEED, PHILOX)         # slab index out of range
    with pytest.raises(binding.IsingError):
        IsingSlab(64, 2, 0, SEED, binding.PHILOX_SHARED)
    h = IsingSlab(64, 2, 0, SEED, PHILOX)
    with pytest.raises(binding.IsingError):
        h.ising_sweep(1.0, 1)                     # a slab cannot sweep on its own
    plane = h.ising_slab_plane(0, 0)
    assert plane.numel() == 64 * 64 // 16
    g = Ising(64, 1, SEED, PHILOX)
    with pytest.raises(binding.IsingError):
        binding.lib() and binding._check(binding.lib().ising_slab_half_sweep_bulk(g._h, 1.0, None), "bulk on a whole-lattice handle")


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_slabs_at_L1024_equal_the_undivided_lattice(rng_mode):
    """The headline lattice cut into 4 slabs: two sweeps, spins and energy against the single handle."""
    L, G = 1024, 4
    cfg, spins, J = synth.make_config(5)
    d_spins, d_J = dev(spins), dev(J)
    ref = Ising(L, 1, SEED, rng_mode)
    ref.ising_load_state(d_spins, d_J)
    ref.ising_sweep(cfg["beta"], 2)
    want = ref.ising_get_spins().flatten().clone()
    Er, Mr = ref.ising_energy()
    Er, Mr = int(Er[0]), int(Mr[0])
    ref.ising_destroy()
    del ref
    hs = make_slabs(L, G, rng_mode, d_spins, d_J)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    binding.ising_slab_sweep_local(hs, cfg["beta"], 2, sa, sb)
    torch.cuda.synchronize()
    got, E, M = gather(hs, spins.size)
    assert torch.equal(got, want) and (E, M) == (Er, Mr)
    # again with the exchange fused into the boundary kernels
    for h in hs:
        h.ising_load_state(d_spins, d_J)
        h.ising_set_t(0)
    binding.ising_slab_sweep_local(hs, cfg["beta"], 2, sa, sb, push=True)
    torch.cuda.synchronize()
    got, E, M = gather(hs, spins.size)
    assert torch.equal(got, want) and (E, M) == (Er, Mr)
