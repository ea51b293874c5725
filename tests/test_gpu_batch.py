"""GPU parity tests (-m gpu) of the two structures that serve many samples with their own random numbers and small lattices:

* the BATCH layout (csrc/batch_kernels.cuh): nsamples site-packed lattices one after the other, every kernel of the one-sample
  path on all of them in one launch -- against the oracle, against the sample-packed layout of the same handle type, and against
  the one-site-at-a-time kernels;
* the CLUSTER-RESIDENT kernel (csrc/cluster_kernels.cuh): one thread-block cluster per sample, the lattice in distributed shared
  memory, all half-sweeps and records of a call in one launch -- against the oracle and against one launch per half-sweep.

All outputs are integers: every comparison is exact (R15).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import (LAYOUT_AUTO, LAYOUT_BATCH, LAYOUT_SAMPLE_PACKED, MINSTD, PHILOX, PHILOX_SHARED, Ising,  # noqa: E402
                                  binding, synth)

pytestmark = pytest.mark.gpu
SEED = synth.DYN_SEED


def dev(a: np.ndarray):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host_u32(t) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def oracle_trace(L, ns, mode, spins, J, beta, nhalf, seed=SEED, t0=0):
    """The oracle's E, M after each of nhalf half-sweeps, and the oracle itself."""
    o = ea3d.Oracle(L, ns, seed, mode)
    o.load_packed(spins, J)
    o.t = t0
    rec = []
    for _ in range(nhalf):
        o.half_sweep(beta)
        rec.append(tuple(x.copy() for x in o.energy()))
    return o, rec


# ------------------------------------------------------------------------------------------------------------ batch layout

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,ns", [(64, 32), (64, 96), (128, 64), (192, 32), (256, 32)])
def test_batch_layout_equals_the_oracle(L, ns, rng_mode):
    """1, 2, 3 and 4 words per thread (L = 64, 128, 192, 256), one and several words of samples: load / get round trip, E and M of
    every sample after every half-sweep from the measuring half-sweeps (kernel choices 0, 2, 3) and from the one-site-at-a-time
    kernels with their own energy kernel (choice 1), final spins, ising_energy."""
    spins, J = synth.make_spins(L, ns, 7), synth.make_couplings(L, ns, 3)
    nsw = 3 if L <= 128 else 2
    o, rec = oracle_trace(L, ns, rng_mode, spins, J, 0.6, 2 * nsw)
    for choice in (0, 1, 2, 3):
        g = Ising(L, ns, SEED, rng_mode, layout=LAYOUT_BATCH)
        g.ising_set_kernel(choice)
        g.ising_load_state(dev(spins), dev(J))
        assert np.array_equal(host_u32(g.ising_get_spins()), spins), "round trip"
        E, M = g.ising_sweep_trace(0.6, nsw, every_half_sweeps=1)
        E, M = E.cpu().numpy(), M.cpu().numpy()
        for k in range(2 * nsw):
            assert np.array_equal(E[k], rec[k][0]) and np.array_equal(M[k], rec[k][1]), (choice, k)
        assert np.array_equal(host_u32(g.ising_get_spins()), o.spins_packed()), choice
        E2, M2 = g.ising_energy()
        assert np.array_equal(E2.cpu().numpy(), rec[-1][0]) and np.array_equal(M2.cpu().numpy(), rec[-1][1]), choice
        assert g.ising_get_t() == 2 * nsw
        g.ising_destroy()


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,ns", [(64, 64), (128, 32)])
def test_the_two_layouts_of_many_samples_agree(L, ns, rng_mode):
    """The automatic layout of these handles is the batch; the sample-packed layout (the paper's AMSC storage) stays available
    on request.  Same spins, records and energies over calls of different lengths, another beta and a counter across 2^32."""
    spins, J = synth.make_spins(L, ns, 17), synth.make_couplings(L, ns, 13)
    a = Ising(L, ns, SEED, rng_mode)                               # automatic = batch
    b = Ising(L, ns, SEED, rng_mode, layout=LAYOUT_SAMPLE_PACKED)
    c = Ising(L, ns, SEED, rng_mode, layout=LAYOUT_BATCH)
    c.ising_set_kernel(3)
    for g in (a, b, c):
        g.ising_load_state(dev(spins), dev(J))
    for beta, n in ((1 / 1.1, 6), (0.4, 1), (1 / 1.1, 9)):
        for g in (a, b, c):
            g.ising_sweep(beta, n)
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins()) and torch.equal(a.ising_get_spins(), c.ising_get_spins()), (beta, n)
    res = [g.ising_sweep_trace(0.8, 6, every_half_sweeps=3) for g in (a, b, c)]
    for r in res[1:]:
        assert torch.equal(res[0][0], r[0]) and torch.equal(res[0][1], r[1])
    for g in (a, b, c):
        g.ising_set_t(2**32 - 5)
        g.ising_sweep(1 / 1.1, 5)
    assert a.ising_get_t() == 2**32 + 5
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins()) and torch.equal(a.ising_get_spins(), c.ising_get_spins())
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0]) and torch.equal(a.ising_energy()[1], c.ising_energy()[1])


def test_layout_rules():
    """A batch needs samples that draw their own numbers and whole-word rows; the shared-draw modes keep the sample-packed arrays."""
    for L, ns, mode, layout in ((64, 32, PHILOX_SHARED, LAYOUT_BATCH), (32, 32, PHILOX, LAYOUT_BATCH), (96, 32, MINSTD, LAYOUT_BATCH),
                                (64, 1, PHILOX, LAYOUT_BATCH), (64, 1, PHILOX, LAYOUT_SAMPLE_PACKED)):
        with pytest.raises(binding.IsingError):
            Ising(L, ns, SEED, mode, layout=layout)
    Ising(32, 32, SEED, PHILOX, layout=LAYOUT_SAMPLE_PACKED).ising_destroy()
    Ising(64, 32, SEED, PHILOX_SHARED, layout=LAYOUT_AUTO).ising_destroy()


def test_batch_overlap_of_replicas_equals_the_oracle():
    L, ns = 64, 64
    W = L**3 // 32
    J = np.tile(synth.make_couplings(L, 1, 33).reshape(1, 3, W), (ns, 1, 1))
    spins = synth.make_spins(L, ns, 34)
    o = ea3d.Oracle(L, ns, SEED, PHILOX)
    o.load_packed(spins, J)
    g = Ising(L, ns, SEED, PHILOX)
    g.ising_load_state(dev(spins), dev(J))
    o.sweep(0.9, 2)
    g.ising_sweep(0.9, 2)
    for a, b in ((0, 0), (0, 1), (5, 31), (31, 5), (ns - 1, 0), (ns - 1, ns - 2), (7, ns - 9)):
        assert int(g.ising_overlap(a, b)[0]) == o.overlap(a, b), (a, b)
    with pytest.raises(binding.IsingError):
        g.ising_overlap(0, ns)


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_batch_run_host_and_guards(rng_mode):
    """ising_run_host on a batch handle whose workspace sits between two guard regions; outputs against the oracle."""
    L, ns = 64, 32
    nbytes = binding.ising_workspace_bytes(L, ns, rng_mode)
    G = 1 << 20
    buf = torch.full((G + nbytes + G,), 0xA5, dtype=torch.uint8, device="cuda")
    spins, J = synth.make_spins(L, ns, 97), synth.make_couplings(L, ns, 98)
    g = Ising(L, ns, SEED, rng_mode, workspace=buf[G:G + nbytes])
    hs = torch.from_numpy(spins.view(np.int32)).pin_memory()
    hJ = torch.from_numpy(J.view(np.int32)).pin_memory()
    out = torch.empty_like(hs).pin_memory()
    E, M = g.ising_run_host(hs, hJ, 1 / 1.1, 5, out)     # 10 half-sweeps: the cluster-resident kernel
    o = ea3d.Oracle(L, ns, SEED, rng_mode)
    o.load_packed(spins, J)
    o.sweep(1 / 1.1, 5)
    assert np.array_equal(out.numpy().view(np.uint32).reshape(ns, -1), o.spins_packed())
    Eo, Mo = o.energy()
    assert np.array_equal(E.numpy(), Eo) and np.array_equal(M.numpy(), Mo)
    g.ising_sweep_trace(1 / 1.1, 2, every_half_sweeps=1)   # launches
    g.ising_overlap(0, 1)
    torch.cuda.synchronize()
    assert bool((buf[:G] == 0xA5).all()) and bool((buf[G + nbytes:] == 0xA5).all()), "workspace guard overwritten"


# ------------------------------------------------------------------------------------------------ cluster-resident kernel

# (L, samples): L = 64: one sample -> clusters of 16 CTAs, 32 samples -> 4, 64 -> 2, 96 -> 1 with four words per thread;
# L = 128 (two words per row): 16 and 8 CTAs.  Kernel choice 4 = this kernel for every call it exists for (by itself the library
# takes it at L = 64 for calls without records or with sparse ones: the next test).
CLUSTER_CASES = [(64, 1), (64, 32), (64, 64), (64, 96), (128, 1), (128, 32)]


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,ns", CLUSTER_CASES)
def test_cluster_resident_kernel_equals_the_oracle(L, ns, rng_mode):
    """Calls of 8 half-sweeps and more run in ONE launch; E and M after every half-sweep, after every third, and none, final spins
    and energies against the oracle; a start at an odd counter (blue first)."""
    choice = 4
    spins, J = synth.make_spins(L, ns, 7), synth.make_couplings(L, ns, 3)
    nsw = 5
    o, rec = oracle_trace(L, ns, rng_mode, spins, J, 0.6, 2 * nsw)
    for every in (1, 3, 0):
        g = Ising(L, ns, SEED, rng_mode)
        g.ising_set_kernel(choice)
        g.ising_load_state(dev(spins), dev(J))
        n0 = g.ising_kernel_launches()
        if every:
            E, M = g.ising_sweep_trace(0.6, nsw, every_half_sweeps=every)
            E, M = E.cpu().numpy(), M.cpu().numpy()
            assert E.shape[0] == 2 * nsw // every
            for i in range(2 * nsw // every):
                k = (i + 1) * every - 1
                assert np.array_equal(E[i], rec[k][0]) and np.array_equal(M[i], rec[k][1]), (every, i)
        else:
            g.ising_sweep(0.6, nsw)
        assert g.ising_kernel_launches() - n0 <= 2, "one launch (plus the pre-set of the records)"
        assert np.array_equal(host_u32(g.ising_get_spins()), o.spins_packed()), every
        E2, M2 = g.ising_energy()
        assert np.array_equal(E2.cpu().numpy(), rec[-1][0]) and np.array_equal(M2.cpu().numpy(), rec[-1][1])
        assert g.ising_get_t() == 2 * nsw
        g.ising_destroy()
    # a start at an odd counter across 2^32 (blue first): against one launch per half-sweep, and with Philox against the oracle
    # (the oracle's MINSTD streams are stored states and cannot jump)
    t0 = 2**32 - 5
    a, b = Ising(L, ns, SEED, rng_mode), Ising(L, ns, SEED, rng_mode)
    a.ising_set_kernel(choice)
    b.ising_set_kernel(3)
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
        g.ising_set_t(t0)
        g.ising_sweep(1 / 1.1, 4)
    assert a.ising_get_t() == t0 + 8 and torch.equal(a.ising_get_spins(), b.ising_get_spins())
    if rng_mode == PHILOX:
        o2, rec2 = oracle_trace(L, ns, rng_mode, spins, J, 1 / 1.1, 8, t0=t0)
        E2, M2 = a.ising_energy()
        assert np.array_equal(E2.cpu().numpy(), rec2[7][0]) and np.array_equal(M2.cpu().numpy(), rec2[7][1])
        assert np.array_equal(host_u32(a.ising_get_spins()), o2.spins_packed())


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,ns,choice", [(64, 1, 0), (64, 32, 0), (64, 128, 0), (128, 32, 4)])
def test_cluster_resident_kernel_equals_one_launch_per_half_sweep(L, ns, choice, rng_mode):
    """Longer calls against kernel choice 3 (one launch per half-sweep): 200 sweeps with records every 20 half-sweeps and every 7,
    calls of different lengths (short ones stay with the launches), another beta, special temperatures.  (MINSTD with many samples:
    clusters of 8 CTAs with the seed states cached in shared memory, more clusters than fit the GPU at once, running in waves.)"""
    spins, J = synth.make_spins(L, ns, 87), synth.make_couplings(L, ns, 88)
    a = Ising(L, ns, SEED, rng_mode)
    a.ising_set_kernel(choice)
    b = Ising(L, ns, SEED, rng_mode)
    b.ising_set_kernel(3)
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
    nsw = 200 if L == 64 and ns <= 32 else 30
    for every in (20, 7):
        n0 = a.ising_kernel_launches()
        Ea, Ma = a.ising_sweep_trace(1 / 1.1, nsw, every_half_sweeps=every)
        if choice == 4 or rng_mode == PHILOX:
            assert a.ising_kernel_launches() - n0 == 2, "the pre-set of the records and ONE launch"
        Eb, Mb = b.ising_sweep_trace(1 / 1.1, nsw, every_half_sweeps=every)
        assert Ea.shape[0] == 2 * nsw // every and torch.equal(Ea, Eb) and torch.equal(Ma, Mb), every
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    for beta, n in ((0.4, 4), (1 / 1.1, 3), (0.0, 4), (float("inf"), 5), (0.9, 17)):
        for g in (a, b):
            g.ising_sweep(beta, n)
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins()), (beta, n)
    Ea, none = a.ising_sweep_trace(0.8, 16, every_half_sweeps=2, want_M=False)
    Eb, _ = b.ising_sweep_trace(0.8, 16, every_half_sweeps=2, want_M=False)
    assert none is None and torch.equal(Ea, Eb)
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0]) and torch.equal(a.ising_energy()[1], b.ising_energy()[1])


def test_cluster_kernel_of_two_handles_on_two_streams():
    """Two handles, two streams, their clusters resident side by side."""
    L = 64
    jobs = []
    for i, (ns, mode) in enumerate(((32, PHILOX), (1, MINSTD))):
        spins, J = synth.make_spins(L, ns, 91 + i), synth.make_couplings(L, ns, 101 + i)
        g, r = Ising(L, ns, SEED + i, mode), Ising(L, ns, SEED + i, mode)
        r.ising_set_kernel(3)
        for h in (g, r):
            h.ising_load_state(dev(spins), dev(J))
        jobs.append((g, r, torch.cuda.Stream()))
    torch.cuda.synchronize()
    for rep in range(3):
        for g, r, st in jobs:
            g.ising_sweep(1 / 1.1 if rep != 1 else 0.4, 40, stream=st)
    torch.cuda.synchronize()
    for g, r, st in jobs:
        for rep in range(3):
            r.ising_sweep(1 / 1.1 if rep != 1 else 0.4, 40)
        assert torch.equal(g.ising_get_spins(), r.ising_get_spins())
