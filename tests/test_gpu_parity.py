"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle -- tolerance 0.

All outputs are integers (spins, energies, magnetisations, checksums), so every comparison is exact (R15).
Every BASELINE.json configuration runs at its stated sweep count against the oracle with the outputs it names
(north_star: "bit-exactly on every config"; PAPER.md:298 + fn. 47: all schemes give the same bits): config 1 E per
half-sweep + final spins; config 2 E of the 32 samples every 10 of 1000 sweeps; config 3 E and M after each of 1000
sweeps; config 4 all ten FNV-1a checksums over 100 sweeps; config 5 (L = 1024, the configuration bench.py times) E and M
after each of the 20 sweeps and the final spins element by element, in both rng modes, plus sampled sites against the
oracle's single-site rule and the word-parallel kernel against the generic one-site-at-a-time kernel.
"""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import LAYOUT_AUTO, LAYOUT_SAMPLE_PACKED, MINSTD, PHILOX, PHILOX_SHARED, Ising, binding, synth  # noqa: E402

pytestmark = pytest.mark.gpu
SEED = synth.DYN_SEED


def dev(a: np.ndarray):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host_u32(t) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def make_pair(L, nsamples, rng_mode, spins, J, seed=SEED, layout=LAYOUT_AUTO):
    o = ea3d.Oracle(L, nsamples, seed, rng_mode)
    o.load_packed(spins, J)
    g = Ising(L, nsamples, seed, rng_mode, layout=layout)
    g.ising_load_state(dev(spins), dev(J))
    return o, g


def assert_same_state(o, g, what=""):
    got = host_u32(g.ising_get_spins())
    want = o.spins_packed()
    assert np.array_equal(got, want), f"{what}: {np.count_nonzero(got != want)} of {want.size} spin words differ"
    E, M = g.ising_energy()
    Eo, Mo = o.energy()
    assert np.array_equal(E.cpu().numpy(), Eo) and np.array_equal(M.cpu().numpy(), Mo), what


# ------------------------------------------------------------------------------------------------ load / get / energy

@pytest.mark.parametrize("L,nsamples", [(4, 1), (6, 1), (16, 1), (24, 1), (64, 1), (128, 1), (256, 1), (4, 32), (6, 32),
                                        (16, 64), (10, 32), (32, 32), (64, 96), (96, 32), (128, 64)])
def test_layout_round_trip_and_energy(L, nsamples):
    """Rows a9 / a10.  Sample-packed: the bit-sliced energy kernel (any L) and, for L a multiple of 32, the register-transpose
    tile kernels of load / get; kernel choice 1 runs the one-bit-at-a-time kernels on the same data."""
    spins, J = synth.make_spins(L, nsamples, 7), synth.make_couplings(L, nsamples, 3)
    # (many samples: the sample-packed arrays, which is what this test is about; L = 64 and 128 would be a batch otherwise)
    o, g = make_pair(L, nsamples, PHILOX, spins, J, layout=LAYOUT_SAMPLE_PACKED if nsamples > 1 else LAYOUT_AUTO)
    assert_same_state(o, g, "after load")
    assert np.array_equal(host_u32(g.ising_get_spins()), spins)
    if nsamples == 1 and L >= 64:  # the generic measurement kernel on the same internal layout
        g.ising_set_kernel(1)
        assert_same_state(o, g, "generic measure")
    if nsamples > 1:
        g.ising_set_kernel(1)      # generic energy and scatter on the arrays the tile kernel wrote
        assert_same_state(o, g, "generic measure / scatter after tile gather")
        g.ising_load_state(dev(spins), dev(J))   # generic gather
        g.ising_set_kernel(0)
        assert_same_state(o, g, "tile scatter / sliced energy after generic gather")
        o.sweep(0.7, 1)
        g.ising_sweep(0.7, 1)
        assert_same_state(o, g, "after a sweep")


def test_energy_closed_forms_on_gpu():
    L = 64
    W = synth.words_per_sample(L)
    up = synth.make_spins(L, 1, init="up")
    ferro = np.zeros((1, 3, W), dtype=np.uint32)
    g = Ising(L, 1, 1, PHILOX)
    g.ising_load_state(dev(up), dev(ferro))
    E, M = g.ising_energy()
    assert int(E[0]) == -3 * L**3 and int(M[0]) == L**3
    J = synth.make_couplings(L, 1, 5)
    g.ising_load_state(dev(up), dev(J))
    E, _ = g.ising_energy()
    nneg = int(np.unpackbits(J.view(np.uint8)).sum())  # all-up: E = -sum J = -(3N - 2 #(J=-1))
    assert int(E[0]) == -(3 * L**3 - 2 * nneg)


# ------------------------------------------------------------------------------------------------ BASELINE.json configs

def test_config1_L16_philox_energy_every_half_sweep():
    cfg, spins, J = synth.make_config(1)
    o, g = make_pair(cfg["L"], 1, cfg["rng_mode"], spins, J)
    E, M = g.ising_sweep_trace(cfg["beta"], cfg["sweeps"], every_half_sweeps=1)
    E, M = E.cpu().numpy()[:, 0], M.cpu().numpy()[:, 0]
    for k in range(2 * cfg["sweeps"]):
        o.half_sweep(cfg["beta"])
        Eo, Mo = o.energy()
        assert (int(E[k]), int(M[k])) == (int(Eo[0]), int(Mo[0])), k
    assert_same_state(o, g, "config 1 final")
    assert g.ising_get_t() == 20


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [4, 6, 10, 16, 18, 22, 24, 32, 34, 62, 64, 66, 70, 96, 100, 126, 128, 130, 190, 250, 256])
def test_site_packed_trajectories(L, rng_mode):
    """Ragged and whole-word half-rows: the word-parallel kernel for L a multiple of 64, the bit-window kernel for every other
    even L (rows shorter than a word, rows of 33 / 62.5 / 125 bits straddling words, a partial last word), and the
    one-site-at-a-time kernel (choice 1) on the same inputs."""
    spins, J = synth.make_spins(L, 1, 11), synth.make_couplings(L, 1, 5)
    o, g = make_pair(L, 1, rng_mode, spins, J)
    nsw = 12 if L <= 64 else 4
    beta = 0.6
    for _ in range(nsw):
        o.sweep(beta, 1)
    E, M = g.ising_sweep_trace(beta, nsw, every_half_sweeps=2 * nsw)
    assert_same_state(o, g, f"L={L}")
    for choice in (1,):     # one site at a time
        g1 = Ising(L, 1, SEED, rng_mode)
        g1.ising_set_kernel(choice)
        g1.ising_load_state(dev(spins), dev(J))
        g1.ising_sweep(beta, nsw)
        assert torch.equal(g.ising_get_spins(), g1.ising_get_spins()), f"L={L}: kernel choice {choice} differs"
    Eo, Mo = o.energy()
    assert int(E[0, 0]) == int(Eo[0]) and int(M[0, 0]) == int(Mo[0])
    assert int(Eo[0]) == int(o.dE_sum[0]) + int(ea3d.Oracle.energy(_loaded(L, 1, rng_mode, spins, J))[0][0])


def _loaded(L, ns, rng_mode, spins, J):
    o = ea3d.Oracle(L, ns, SEED, rng_mode)
    o.load_packed(spins, J)
    return o


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("beta", [0.0, float("inf"), 1 / 1.1])
def test_special_temperatures(rng_mode, beta):
    L = 64
    spins, J = synth.make_spins(L, 1, 4), synth.make_couplings(L, 1, 9)
    o, g = make_pair(L, 1, rng_mode, spins, J)
    E0 = int(g.ising_energy()[0][0])
    for k in range(3):
        o.sweep(beta, 1)
        g.ising_sweep(beta, 1)
        assert_same_state(o, g, f"beta={beta} sweep {k}")
    if beta == 0.0:  # every proposal accepted: three sweeps invert every spin three times
        assert np.array_equal(host_u32(g.ising_get_spins()), ~spins)
        assert int(g.ising_energy()[0][0]) == E0
    if beta == float("inf"):
        assert int(g.ising_energy()[0][0]) <= E0


def test_config2_L64_32_samples_philox():
    cfg, spins, J = synth.make_config(2)
    nsw = cfg["sweeps"]
    assert nsw == 1000
    o, g = make_pair(cfg["L"], 32, cfg["rng_mode"], spins, J)
    E, _ = g.ising_sweep_trace(cfg["beta"], nsw, every_half_sweeps=20, want_M=False)  # every 10 sweeps
    E = E.cpu().numpy()
    for r in range(nsw // 10):
        o.sweep(cfg["beta"], 10)
        assert np.array_equal(E[r], o.energy()[0]), f"record {r}"
    assert_same_state(o, g, "config 2 final")
    assert len(set(E[-1].tolist())) > 16  # the 32 samples really are different systems


def test_config2_in_the_sample_packed_layout_and_by_launches():
    """Config 2 runs, by default, as a batch of 32 site-packed lattices in the cluster-resident kernel (the test above).  The same
    1000 sweeps in the paper's sample-packed storage, and in the batch layout with one launch per half-sweep: same records, same
    spins."""
    cfg, spins, J = synth.make_config(2)
    res = []
    for layout, choice in ((LAYOUT_AUTO, 0), (LAYOUT_SAMPLE_PACKED, 0), (LAYOUT_AUTO, 3)):
        g = Ising(cfg["L"], 32, SEED, cfg["rng_mode"], layout=layout)
        g.ising_set_kernel(choice)
        g.ising_load_state(dev(spins), dev(J))
        E, _ = g.ising_sweep_trace(cfg["beta"], cfg["sweeps"], every_half_sweeps=20, want_M=False)
        res.append((E.clone(), g.ising_get_spins().clone(), g.ising_kernel_launches()))
        g.ising_destroy()
    for r in res[1:]:
        assert torch.equal(res[0][0], r[0]) and torch.equal(res[0][1], r[1])
    assert res[0][2] <= 4 and res[2][2] >= 2000      # one launch against one per half-sweep


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,nsamples", [(4, 32), (6, 32), (10, 32), (16, 64), (8, 160), (24, 96), (64, 64), (10, 64), (6, 96), (12, 160)])
def test_sample_packed_small(L, nsamples, rng_mode):
    spins, J = synth.make_spins(L, nsamples, 21), synth.make_couplings(L, nsamples, 8)
    o, g = make_pair(L, nsamples, rng_mode, spins, J, layout=LAYOUT_SAMPLE_PACKED)
    o.sweep(0.7, 6)
    g.ising_sweep(0.7, 6)
    assert_same_state(o, g, f"L={L} x {nsamples}")


def test_config3_L256_minstd_energy_and_magnetisation_per_sweep():
    cfg, spins, J = synth.make_config(3)
    nsw = cfg["sweeps"]
    assert nsw == 1000
    o, g = make_pair(cfg["L"], 1, cfg["rng_mode"], spins, J)
    E, M = g.ising_sweep_trace(cfg["beta"], nsw, every_half_sweeps=2)
    E, M = E.cpu().numpy()[:, 0], M.cpu().numpy()[:, 0]
    for k in range(nsw):
        o.sweep(cfg["beta"], 1)
        Eo, Mo = o.energy()
        assert (int(E[k]), int(M[k])) == (int(Eo[0]), int(Mo[0])), k
    assert_same_state(o, g, "config 3 final")


def test_config4_L512_philox_fnv_checksums():
    cfg, spins, J = synth.make_config(4)
    nsw = cfg["sweeps"]
    assert nsw == 100
    o, g = make_pair(cfg["L"], 1, cfg["rng_mode"], spins, J)
    for r in range(nsw // 10):
        o.sweep(cfg["beta"], 10)
        g.ising_sweep(cfg["beta"], 10)
        d_spins = g.ising_get_spins()
        got = binding.ising_fnv1a64_host(host_u32(d_spins))
        assert got == ea3d.fnv1a64(o.spins_packed()), f"checksum after {10 * (r + 1)} sweeps"
        assert int(binding.ising_fnv1a64(d_spins)[0]) & (2**64 - 1) == got, "the checksum computed on the device"
    assert_same_state(o, g, "config 4 final")
    # and the remaining sweeps of the config against the generic kernel (second GPU implementation)
    g2 = Ising(cfg["L"], 1, SEED, cfg["rng_mode"])
    g2.ising_load_state(g.ising_get_spins(), dev(J))
    g2.ising_set_t(g.ising_get_t())
    g2.ising_set_kernel(1)
    g.ising_sweep(cfg["beta"], 5)
    g2.ising_sweep(cfg["beta"], 5)
    assert torch.equal(g.ising_get_spins(), g2.ising_get_spins())


# ------------------------------------------------------------------------------------------------ invariances

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_batching_of_sweeps_into_calls_and_resume(rng_mode):
    L = 64
    spins, J = synth.make_spins(L, 1, 2), synth.make_couplings(L, 1, 1)
    a = Ising(L, 1, SEED, rng_mode)
    a.ising_load_state(dev(spins), dev(J))
    a.ising_sweep(0.9, 10)
    b = Ising(L, 1, SEED, rng_mode)
    b.ising_load_state(dev(spins), dev(J))
    for _ in range(10):
        b.ising_sweep(0.9, 1)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    # checkpoint / resume: (spins, t) is the whole dynamic state
    c = Ising(L, 1, SEED, rng_mode)
    c.ising_load_state(dev(spins), dev(J))
    c.ising_sweep(0.9, 4)
    d = Ising(L, 1, SEED, rng_mode)
    d.ising_load_state(c.ising_get_spins(), dev(J))
    d.ising_set_t(c.ising_get_t())
    d.ising_sweep(0.9, 6)
    assert torch.equal(a.ising_get_spins(), d.ising_get_spins())
    # a different seed gives a different trajectory
    e = Ising(L, 1, SEED + 1, rng_mode)
    e.ising_load_state(dev(spins), dev(J))
    e.ising_sweep(0.9, 10)
    assert not torch.equal(a.ising_get_spins(), e.ising_get_spins())


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [64, 128, 256, 512])
def test_word_parallel_kernel_equals_generic_kernel(L, rng_mode):
    spins, J = synth.make_spins(L, 1, 31), synth.make_couplings(L, 1, 32)
    a = Ising(L, 1, SEED, rng_mode)
    b = Ising(L, 1, SEED, rng_mode)
    b.ising_set_kernel(1)
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
        g.ising_sweep(1 / 1.1, 3)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0])


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [192, 320])
def test_word_parallel_layout_for_L_not_a_power_of_two_equals_the_oracle(L, rng_mode):
    """L = 192, 320 (multiples of 64 that are not powers of two: rows of 3 and 5 words, one thread per row):
    layout round trip, trajectory, energy and magnetisation against the oracle."""
    spins, J = synth.make_spins(L, 1, 33), synth.make_couplings(L, 1, 34)
    o, g = make_pair(L, 1, rng_mode, spins, J)
    assert np.array_equal(host_u32(g.ising_get_spins())[0], spins.reshape(-1))
    assert_same_state(o, g, f"L={L} loaded")
    for beta, n in ((1 / 1.1, 2), (1 / 0.7, 1)):
        o.sweep(beta, n)
        g.ising_sweep(beta, n)
        assert_same_state(o, g, f"L={L} rng {rng_mode} beta {beta}")


@pytest.mark.parametrize("rng_mode,kernel", [(PHILOX, 0), (MINSTD, 0), (MINSTD, 2)])
@pytest.mark.parametrize("L", [192, 320, 384, 448, 576, 768, 1280])
def test_word_parallel_kernel_equals_generic_kernel_for_any_multiple_of_64(L, rng_mode, kernel):
    """Rows of 3, 6, 12 words (three words per thread, 1 / 2 / 4 lanes per row), of 5 and 20 words (five words per thread)
    and of 7 and 9 words (one word per thread, the row padded to 8 and 16 lanes, idle lanes store nothing)."""
    W = L**3 // 32
    gen = torch.Generator(device="cuda").manual_seed(L)
    d_spins = torch.randint(-2**31, 2**31 - 1, (W,), dtype=torch.int32, device="cuda", generator=gen)
    d_J = torch.randint(-2**31, 2**31 - 1, (3 * W,), dtype=torch.int32, device="cuda", generator=gen)
    a = Ising(L, 1, SEED, rng_mode)
    a.ising_set_kernel(kernel)
    b = Ising(L, 1, SEED, rng_mode)
    b.ising_set_kernel(1)
    for g in (a, b):
        g.ising_load_state(d_spins, d_J)
        g.ising_sweep(1 / 1.1, 2)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    Ea, Ma = a.ising_energy()
    Eb, Mb = b.ising_energy()
    assert torch.equal(Ea, Eb) and torch.equal(Ma, Mb)


def test_minstd_seed_table_and_recomputed_seeds_at_four_words_per_thread():
    """MINSTD, four words per thread (L = 512 is the smallest such lattice): the automatic choice reads the seed-state table
    for every word, choice 2 recomputes SplitMix64 per draw.  Same bits as the oracle after a sweep, and the recording
    (MEASURE) variant gives the oracle's E and M per half-sweep."""
    L = 512
    spins, J = synth.make_spins(L, 1, 51), synth.make_couplings(L, 1, 52)
    o = _loaded(L, 1, MINSTD, spins, J)
    hs = []
    for choice in (0, 2):
        g = Ising(L, 1, SEED, MINSTD)
        g.ising_set_kernel(choice)
        g.ising_load_state(dev(spins), dev(J))
        g.ising_sweep(1 / 0.7, 1)
        hs.append(g)
    o.sweep(1 / 0.7, 1)
    assert_same_state(o, hs[0], "seed table, L=512")
    for g in hs[1:]:
        assert torch.equal(g.ising_get_spins(), hs[0].ising_get_spins())
    E, M = hs[0].ising_sweep_trace(1 / 0.7, 1, every_half_sweeps=1)
    for r in range(2):
        o.half_sweep(1 / 0.7)
        Eo, Mo = o.energy()
        assert int(E[r, 0]) == int(Eo[0]) and int(M[r, 0]) == int(Mo[0]), r
    assert_same_state(o, hs[0], "seed table after the recording sweep")


@pytest.mark.parametrize("L", [64, 128, 256, 512])
def test_minstd_cached_seed_table_equals_recomputed_seeds(L):
    """MINSTD: the default word-parallel kernel streams the seed states s0 from a table filled once per handle; kernel
    choice 2 recomputes SplitMix64 per draw.  Same bits, also across separate calls (the table is reused) and after a
    reload of the lattice (the table depends on (seed, site) only)."""
    spins, J = synth.make_spins(L, 1, 41), synth.make_couplings(L, 1, 42)
    a = Ising(L, 1, SEED, MINSTD)
    b = Ising(L, 1, SEED, MINSTD)
    b.ising_set_kernel(2)
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
        g.ising_sweep(1 / 0.7, 2)
        g.ising_sweep(1 / 0.7, 1)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert a.ising_kernel_launches() == b.ising_kernel_launches() + 2  # the two table fills
    spins2 = synth.make_spins(L, 1, 43)
    for g in (a, b):
        g.ising_load_state(dev(spins2), dev(J))
        g.ising_sweep(0.5, 2)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0])


# ------------------------------------------------------------------------------------------------ shared-random-number mode

@pytest.mark.parametrize("L,nsamples", [(4, 32), (6, 32), (8, 32), (8, 64), (12, 32), (16, 64), (24, 32), (40, 32), (64, 32),
                                        (8, 320), (16, 160), (32, 96), (6, 64), (10, 160), (12, 96)])
def test_shared_random_number_mode_equals_the_oracle(L, nsamples):
    """rng_mode 2 (R18): one Philox draw per 32-sample word.  The vectorised kernel (L % 8 == 0) and
    the generic sample-packed kernel (kernel choice 1, and every other L) against the oracle, trajectory and energies."""
    spins, J = synth.make_spins(L, nsamples, 51), synth.make_couplings(L, nsamples, 52)
    o, g = make_pair(L, nsamples, PHILOX_SHARED, spins, J)
    g2 = Ising(L, nsamples, SEED, PHILOX_SHARED)
    g2.ising_set_kernel(1)
    g2.ising_load_state(dev(spins), dev(J))
    for beta, n in ((1 / 1.1, 2), (0.3, 1), (1 / 0.7, 2)):
        o.sweep(beta, n)
        g.ising_sweep(beta, n)
        g2.ising_sweep(beta, n)
        assert_same_state(o, g, f"shared mode L={L} beta={beta}")
        assert torch.equal(g.ising_get_spins(), g2.ising_get_spins())


@pytest.mark.parametrize("beta", [0.0, float("inf")])
def test_shared_mode_special_temperatures(beta):
    L, ns = 16, 32
    spins, J = synth.make_spins(L, ns, 53), synth.make_couplings(L, ns, 54)
    o, g = make_pair(L, ns, PHILOX_SHARED, spins, J)
    o.sweep(beta, 2)
    g.ising_sweep(beta, 2)
    assert_same_state(o, g, f"shared mode beta={beta}")


def test_shared_mode_needs_whole_words_of_samples():
    with pytest.raises(binding.IsingError):
        Ising(16, 1, SEED, PHILOX_SHARED)


# ------------------------------------------------------------------------------------------------ edge cases

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_zero_sweeps_is_a_no_op(rng_mode):
    L = 64
    spins, J = synth.make_spins(L, 1, 61), synth.make_couplings(L, 1, 62)
    g = Ising(L, 1, SEED, rng_mode)
    g.ising_load_state(dev(spins), dev(J))
    n0 = g.ising_kernel_launches()
    g.ising_sweep(0.7, 0)
    assert g.ising_get_t() == 0 and g.ising_kernel_launches() == n0
    assert np.array_equal(host_u32(g.ising_get_spins()), spins)
    with pytest.raises(binding.IsingError):
        g.ising_sweep(0.7, -1)
    with pytest.raises(binding.IsingError):
        g.ising_sweep(-0.1, 1)


@pytest.mark.parametrize("L,nsamples,rng_mode", [(64, 1, PHILOX), (6, 1, PHILOX), (8, 32, PHILOX), (10, 32, PHILOX),
                                                  (8, 64, PHILOX_SHARED), (6, 32, PHILOX_SHARED)])
def test_64_bit_seed_and_half_sweep_counter_across_2_to_32(L, nsamples, rng_mode):
    """Philox key and counter are 64-bit quantities split into 32-bit words (R9): a seed with a non-zero high word and a
    half-sweep counter that crosses 2^32 during the run exercise hi32(seed) ^ sample and hi32(t) in every kernel."""
    seed = 0xDEADBEEF12345678
    t0 = 2**32 - 2
    spins, J = synth.make_spins(L, nsamples, 91), synth.make_couplings(L, nsamples, 92)
    o, g = make_pair(L, nsamples, rng_mode, spins, J, seed=seed)
    o.t = t0
    g.ising_set_t(t0)
    o.sweep(1 / 1.1, 2)
    g.ising_sweep(1 / 1.1, 2)
    assert g.ising_get_t() == t0 + 4 == o.t
    assert_same_state(o, g, f"L={L} x {nsamples}, mode {rng_mode}, t across 2^32")


@pytest.mark.parametrize("L,nsamples,rng_mode,kernel", [(64, 1, PHILOX, 0), (128, 1, MINSTD, 0), (512, 1, MINSTD, 0), (64, 1, MINSTD, 2),
                                                         (6, 1, PHILOX, 0), (16, 1, MINSTD, 0), (64, 1, PHILOX, 1), (8, 32, PHILOX, 0),
                                                         (6, 32, MINSTD, 0), (16, 64, PHILOX, 1), (8, 64, PHILOX_SHARED, 0),
                                                         (6, 32, PHILOX_SHARED, 0)])
def test_no_kernel_writes_outside_the_workspace(L, nsamples, rng_mode, kernel):
    """Memory safety without a sanitizer: the workspace sits between two guard regions of 1 MiB filled with a pattern,
    and so do the output buffers; every entry point runs; the guards must be untouched."""
    nbytes = binding.ising_workspace_bytes(L, nsamples, rng_mode)
    G = 1 << 20
    buf = torch.full((G + nbytes + G,), 0xA5, dtype=torch.uint8, device="cuda")
    W = (L**3 + 31) // 32
    out = torch.full((G // 4 + nsamples * W + G // 4,), 0x5A5A5A5A, dtype=torch.int32, device="cuda")
    spins, J = synth.make_spins(L, nsamples, 95), synth.make_couplings(L, nsamples, 96)
    g = Ising(L, nsamples, SEED, rng_mode, workspace=buf[G:G + nbytes])
    g.ising_set_kernel(kernel)
    g.ising_load_state(dev(spins), dev(J))
    g.ising_sweep(1 / 1.1, 2)
    E, M = g.ising_sweep_trace(1 / 1.1, 1, every_half_sweeps=1)
    g.ising_energy()
    g.ising_get_spins(out[G // 4:G // 4 + nsamples * W])
    torch.cuda.synchronize()
    assert bool((buf[:G] == 0xA5).all()) and bool((buf[G + nbytes:] == 0xA5).all()), "workspace guard overwritten"
    assert bool((out[:G // 4] == 0x5A5A5A5A).all()) and bool((out[G // 4 + nsamples * W:] == 0x5A5A5A5A).all()), "output guard"
    # and the run is the same as with a private workspace
    ref = Ising(L, nsamples, SEED, rng_mode)
    ref.ising_set_kernel(kernel)
    ref.ising_load_state(dev(spins), dev(J))
    ref.ising_sweep(1 / 1.1, 3)
    assert torch.equal(ref.ising_get_spins().flatten(), out[G // 4:G // 4 + nsamples * W])


@pytest.mark.parametrize("rng_mode,kernel", [(PHILOX, 0), (MINSTD, 2)])
def test_maximum_size_L2048_word_parallel_equals_generic(rng_mode, kernel):
    """L = 2048 is the largest lattice every layout and mode accepts (tests/test_gpu_large.py goes beyond): 2^33 spins, 1 GiB of spin bits.
    The oracle cannot hold it (34 GB of int8 per array); the word-parallel kernel is compared with the generic
    one-site-at-a-time kernel over one sweep, and the energy bookkeeping with the spin count."""
    L = 2048
    W = L**3 // 32
    gen = torch.Generator(device="cuda").manual_seed(7)
    d_spins = torch.randint(-2**31, 2**31 - 1, (W,), dtype=torch.int32, device="cuda", generator=gen)
    d_J = torch.randint(-2**31, 2**31 - 1, (3 * W,), dtype=torch.int32, device="cuda", generator=gen)
    a = Ising(L, 1, SEED, rng_mode)
    a.ising_set_kernel(kernel)
    a.ising_load_state(d_spins, d_J)
    assert torch.equal(a.ising_get_spins().flatten(), d_spins)
    a.ising_sweep(1 / 1.1, 1)
    out_a = a.ising_get_spins().clone()
    Ea, Ma = a.ising_energy()
    a.ising_destroy()
    del a
    b = Ising(L, 1, SEED, rng_mode)
    b.ising_set_kernel(1)
    b.ising_load_state(d_spins, d_J)
    b.ising_sweep(1 / 1.1, 1)
    assert torch.equal(b.ising_get_spins(), out_a)
    Eb, Mb = b.ising_energy()
    assert int(Ea[0]) == int(Eb[0]) and int(Ma[0]) == int(Mb[0])
    up = int(sum(bin(int(w) & 0xFFFFFFFF).count("1") for w in out_a.flatten()[:4096].cpu().tolist()))  # spot check of the bit order
    assert 0 < up < 32 * 4096
    assert abs(int(Ea[0])) < 3 * L**3 and abs(int(Ma[0])) <= L**3 and int(Ea[0]) % 2 == (3 * L**3) % 2


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,nsamples", [(8, 32), (24, 64), (64, 32), (128, 32)])
def test_sample_packed_vector_kernel_equals_scalar_kernel(L, nsamples, rng_mode):
    """L % 8 == 0: the sample-packed kernel with 128-bit loads (default) against the scalar-load kernel (kernel choice 1),
    both thread-per-group variants (L = 128 x 32 has more than 148 x 1024 groups)."""
    spins, J = synth.make_spins(L, nsamples, 81), synth.make_couplings(L, nsamples, 82)
    a = Ising(L, nsamples, SEED, rng_mode, layout=LAYOUT_SAMPLE_PACKED)
    b = Ising(L, nsamples, SEED, rng_mode, layout=LAYOUT_SAMPLE_PACKED)
    b.ising_set_kernel(1)
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
        g.ising_sweep(1 / 1.1, 2)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0])


@pytest.mark.parametrize("rng_mode,nsamples", [(PHILOX, 32), (PHILOX_SHARED, 32), (PHILOX_SHARED, 96)])
def test_sample_packed_L256_vector_kernels_equal_scalar_kernel(rng_mode, nsamples):
    """The largest sample-packed sizes bench.py times (L = 256 x 32 samples and more): the 128-bit-load kernels (default)
    against the scalar-load kernel (kernel choice 1) over one sweep (the scalar kernel is compared with the oracle at
    small sizes)."""
    L = 256
    gen = torch.Generator(device="cuda").manual_seed(11)
    W = L**3 // 32
    d_spins = torch.randint(-2**31, 2**31 - 1, (nsamples * W,), dtype=torch.int32, device="cuda", generator=gen)
    d_J = torch.randint(-2**31, 2**31 - 1, (nsamples * 3 * W,), dtype=torch.int32, device="cuda", generator=gen)
    a = Ising(L, nsamples, SEED, rng_mode, layout=LAYOUT_SAMPLE_PACKED)
    b = Ising(L, nsamples, SEED, rng_mode, layout=LAYOUT_SAMPLE_PACKED)
    b.ising_set_kernel(1)
    for g in (a, b):
        g.ising_load_state(d_spins, d_J)
        g.ising_sweep(1 / 1.1, 1)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0])


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_sample_packed_large_lattice_one_thread_per_group(rng_mode):
    """L = 128 x 32 samples has more than 148 x 1024 Philox groups, so the one-thread-per-group variant of the
    sample-packed kernel runs (smaller lattices use four threads per group); two batches exercise the batch loop."""
    L, ns = 128, 64
    spins, J = synth.make_spins(L, ns, 71), synth.make_couplings(L, ns, 72)
    o, g = make_pair(L, ns, rng_mode, spins, J, layout=LAYOUT_SAMPLE_PACKED)
    o.sweep(1 / 1.1, 1)
    g.ising_sweep(1 / 1.1, 1)
    assert_same_state(o, g, f"sample-packed L={L} x {ns}")


def test_run_host_equals_device_calls():
    L = 128
    spins, J = synth.make_spins(L, 1, 2), synth.make_couplings(L, 1, 1)
    a = Ising(L, 1, SEED, PHILOX)
    hs = torch.from_numpy(spins.view(np.int32)).pin_memory()
    hJ = torch.from_numpy(J.view(np.int32)).pin_memory()
    out = torch.empty_like(hs).pin_memory()
    E, M = a.ising_run_host(hs, hJ, 1 / 1.1, 5, out)
    o = _loaded(L, 1, PHILOX, spins, J)
    o.sweep(1 / 1.1, 5)
    assert np.array_equal(out.numpy().view(np.uint32), o.spins_packed())
    assert int(E[0]) == int(o.energy()[0][0]) and int(M[0]) == int(o.energy()[1][0])
    assert a.ising_kernel_launches() == 1 + 10 + 1 + 1  # load, 10 half-sweeps, fused energy, get


@pytest.mark.parametrize("L,nsamples,rng_mode", [(64, 1, MINSTD), (16, 1, PHILOX), (8, 32, PHILOX), (6, 64, MINSTD),
                                                  (8, 64, PHILOX_SHARED)])
def test_run_host_every_layout(L, nsamples, rng_mode):
    """ising_run_host (host buffers in, host results out) for the word-parallel, generic, sample-packed and shared-draw
    paths: spins, E and M of every sample against the oracle; without the optional outputs too."""
    spins, J = synth.make_spins(L, nsamples, 97), synth.make_couplings(L, nsamples, 98)
    a = Ising(L, nsamples, SEED, rng_mode)
    hs = torch.from_numpy(spins.view(np.int32)).pin_memory()
    hJ = torch.from_numpy(J.view(np.int32)).pin_memory()
    out = torch.empty_like(hs).pin_memory()
    E, M = a.ising_run_host(hs, hJ, 1 / 1.1, 3, out)
    o = _loaded(L, nsamples, rng_mode, spins, J)
    o.sweep(1 / 1.1, 3)
    assert np.array_equal(out.numpy().view(np.uint32).reshape(nsamples, -1), o.spins_packed())
    Eo, Mo = o.energy()
    assert np.array_equal(E.numpy(), Eo) and np.array_equal(M.numpy(), Mo)
    a.ising_set_t(0)
    E2, _ = a.ising_run_host(hs, hJ, 1 / 1.1, 3, None)  # same job again, spins not wanted
    assert np.array_equal(E2.numpy(), Eo)


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_run_host_async_double_buffered(rng_mode):
    """ising_run_host_async: two handles on two streams with six different jobs in flight alternately (the double buffering of
    bench.py's e2e); every job's spins, E and M against the oracle."""
    L, njobs = 128, 6
    handles = [Ising(L, 1, SEED, rng_mode), Ising(L, 1, SEED, rng_mode)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    jobs = []
    for k in range(njobs):
        spins, J = synth.make_spins(L, 1, 200 + k), synth.make_couplings(L, 1, 300 + k)
        jobs.append(dict(spins=spins, J=J, hs=torch.from_numpy(spins.view(np.int32)).pin_memory(),
                         hJ=torch.from_numpy(J.view(np.int32)).pin_memory(),
                         out=torch.empty(spins.size, dtype=torch.int32).pin_memory(),
                         E=torch.zeros(1, dtype=torch.int64).pin_memory(), M=torch.zeros(1, dtype=torch.int64).pin_memory()))
    torch.cuda.synchronize()
    for k, jb in enumerate(jobs):
        g, st = handles[k % 2], streams[k % 2]
        g.ising_set_t(0)
        g.ising_run_host_async(jb["hs"], jb["hJ"], 1 / 1.1, 2 + k % 3, jb["out"], jb["E"], jb["M"], stream=st)
    for st in streams:
        st.synchronize()
    for k, jb in enumerate(jobs):
        o = _loaded(L, 1, rng_mode, jb["spins"], jb["J"])
        o.sweep(1 / 1.1, 2 + k % 3)
        assert np.array_equal(jb["out"].numpy().view(np.uint32), o.spins_packed().reshape(-1)), f"job {k}"
        Eo, Mo = o.energy()
        assert int(jb["E"][0]) == int(Eo[0]) and int(jb["M"][0]) == int(Mo[0]), f"job {k}"


# ------------------------------------------------------------------------------------------------ config 5, full size

def _avail_gib():
    try:
        import psutil
        return psutil.virtual_memory().available / 2**30
    except Exception:
        return 0.0


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_config5_L1024_all_20_sweeps_against_the_oracle(rng_mode):
    """BASELINE.json config 5 at its stated length, both rng modes: E and M after each of the 20 sweeps (ising_sweep_trace,
    the recording half-sweeps measure inside the kernel) and the final spins element by element against the oracle
    (2 x 10^10 scalar updates per mode; 4 GiB of int8 arrays, 8 GiB with the MINSTD stream states)."""
    cfg, spins, J = synth.make_config(5)
    L, beta, nsw = cfg["L"], cfg["beta"], cfg["sweeps"]
    assert (L, nsw) == (1024, 20)
    if _avail_gib() < 14:
        pytest.skip("not enough host RAM for the int8 oracle arrays at L=1024")
    o, g = make_pair(L, 1, rng_mode, spins, J)
    assert np.array_equal(host_u32(g.ising_get_spins()), spins)
    E, M = g.ising_sweep_trace(beta, nsw, every_half_sweeps=2)
    E, M = E.cpu().numpy()[:, 0], M.cpu().numpy()[:, 0]
    for k in range(nsw):
        o.sweep(beta, 1)
        Eo, Mo = o.energy()
        assert (int(E[k]), int(M[k])) == (int(Eo[0]), int(Mo[0])), f"sweep {k + 1}"
    assert_same_state(o, g, "config 5 after 20 sweeps")
    assert g.ising_get_t() == 2 * nsw
    # the launch pattern bench.py times (one ising_sweep call, no recording half-sweeps) leaves the same bits
    g3 = Ising(L, 1, SEED, rng_mode)
    g3.ising_load_state(dev(spins), dev(J))
    g3.ising_sweep(beta, nsw)
    assert torch.equal(g3.ising_get_spins(), g.ising_get_spins())
    E3, M3 = g3.ising_energy()
    assert (int(E3[0]), int(M3[0])) == (int(E[-1]), int(M[-1]))


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_config5_L1024_kernel_cross_checks(rng_mode):
    """Extra checks at L = 1024 beside the full-length oracle comparison above: the generic one-site-at-a-time kernel
    reproduces the last sweep, and sampled sites of the last sweep obey the oracle's single-site rule."""
    cfg, spins, J = synth.make_config(5)
    L, beta, nsw = cfg["L"], cfg["beta"], cfg["sweeps"]
    dJ = dev(J)
    g = Ising(L, 1, SEED, rng_mode)
    g.ising_load_state(dev(spins), dJ)
    have_ram = _avail_gib() > 14
    g.ising_sweep(beta, nsw - 1)
    t0 = g.ising_get_t()
    assert t0 == 2 * (nsw - 1)
    d_before = g.ising_get_spins().clone()  # state before the last sweep
    E_trace, _ = g.ising_sweep_trace(beta, 1, every_half_sweeps=1, want_M=False)
    d_end = g.ising_get_spins().clone()

    # (1) the generic one-site-at-a-time kernel reproduces the last sweep from the same state
    g2 = Ising(L, 1, SEED, rng_mode)
    g2.ising_set_kernel(1)
    g2.ising_load_state(d_before, dJ)
    g2.ising_set_t(t0)
    g2.ising_sweep(beta, 1)
    assert torch.equal(g2.ising_get_spins(), d_end), "word-parallel vs generic kernel at L=1024"
    assert int(g2.ising_energy()[0][0]) == int(E_trace[-1, 0])
    del g2

    if not have_ram:
        pytest.skip("not enough host RAM for the int8 oracle arrays at L=1024: oracle checks skipped")

    # (2) sampled sites against the oracle's single-site rule.  Red sites change only in the red half-sweep t0, so their
    # final value is before ^ flips(t0).  For blue sites a handle is put at the odd counter t0+1 with the same state, so
    # that its next sweep starts with the blue half-sweep t0+1 (then red t0+2): blue final = before ^ flips(t0+1).
    s_before = host_u32(d_before)
    o = _loaded(L, 1, rng_mode, s_before, J)
    g4 = Ising(L, 1, SEED, rng_mode)
    g4.ising_load_state(d_before, dJ)
    g4.ising_set_t(t0 + 1)
    g4.ising_sweep(beta, 1)
    before_bits = np.unpackbits(s_before.view(np.uint8), bitorder="little")
    finals = {0: np.unpackbits(host_u32(d_end).view(np.uint8), bitorder="little"),
              1: np.unpackbits(host_u32(g4.ising_get_spins()).view(np.uint8), bitorder="little")}
    rng = np.random.default_rng(123)
    for colour in (0, 1):
        n_flipped = 0
        for _ in range(2000):
            x, y, z = (int(v) for v in rng.integers(0, L, 3))
            if ((x + y + z) & 1) != colour:
                x ^= 1
            i = x + L * (y + L * z)
            flips, dE, R = o.site_flips(beta, 0, x, y, z, t0 + colour)
            assert flips in (0, 1)
            assert int(finals[colour][i]) == int(before_bits[i]) ^ flips, (colour, x, y, z, dE, R)
            n_flipped += flips
        assert 0 < n_flipped < 2000


@pytest.mark.parametrize("nsamples,rng_mode", [(1, PHILOX), (1, MINSTD), (32, PHILOX), (96, MINSTD), (96, PHILOX_SHARED)])
def test_automatic_and_one_at_a_time_kernels_agree_over_sizes(nsamples, rng_mode):
    """Every layout-specific kernel family (word-parallel, bit-window with and without the segment loop, vectorised / multi-batch
    sample-packed, tile load / get, bit-sliced energy) against the one-site / one-bit-at-a-time kernels (choice 1) on the same
    inputs: spins, energies and magnetisations after three sweeps, over lattice sizes of every alignment class."""
    sizes = (4, 6, 10, 12, 20, 36, 48, 66, 72, 100, 136, 160, 200) if nsamples == 1 else (4, 6, 10, 12, 20, 36, 40, 48, 66, 72)
    for L in sizes:
        spins, J = synth.make_spins(L, nsamples, 3), synth.make_couplings(L, nsamples, 4)
        res = []
        for choice in (0, 1):
            g = Ising(L, nsamples, 777, rng_mode)
            g.ising_set_kernel(choice)
            g.ising_load_state(dev(spins), dev(J))
            E, M = g.ising_sweep_trace(0.8, 3, every_half_sweeps=3)
            res.append((g.ising_get_spins().clone(), E.clone(), M.clone()))
            g.ising_destroy()
        assert all(torch.equal(a, b) for a, b in zip(res[0], res[1])), f"L={L} x {nsamples}, mode {rng_mode}"


@pytest.mark.parametrize("L,nsamples", [(6, 32), (16, 64), (40, 96)])
def test_overlap_of_replicas_equals_the_oracle(L, nsamples):
    """ising_overlap: q_ab = sum_i sigma^a sigma^b for samples in the same and in different coded batches, on
    replicas (same couplings, different initial spins) after a few sweeps."""
    W = (L**3 + 31) // 32
    J1 = synth.make_couplings(L, 1, 33)
    J = np.tile(J1.reshape(1, 3, W), (nsamples, 1, 1))
    spins = synth.make_spins(L, nsamples, 34)
    o, g = make_pair(L, nsamples, PHILOX, spins, J)
    o.sweep(0.9, 2)
    g.ising_sweep(0.9, 2)
    pairs = [(0, 0), (0, 1), (5, 31), (31, 5), (nsamples - 1, 0), (nsamples - 1, nsamples - 2), (7, nsamples - 9)]
    for a, b in pairs:
        assert int(g.ising_overlap(a, b)[0]) == o.overlap(a, b), (a, b)
    assert int(g.ising_overlap(3, 3)[0]) == L**3
    with pytest.raises(binding.IsingError):
        g.ising_overlap(0, nsamples)
    with pytest.raises(binding.IsingError):
        Ising(64, 1, SEED, PHILOX).ising_overlap(0, 0)


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [64, 128, 192, 256, 320, 448, 66, 100, 126, 250])
def test_energy_measured_inside_the_half_sweep_kernel(L, rng_mode):
    """Trace records of the word-parallel layout come from the half-sweep kernel itself (MEASURE variant: satisfied bonds from
    the field bit planes, n -> 6 - n where the site flipped).  E and M after every half-sweep (red and blue records) against the
    one-site-at-a-time kernels with their separate energy kernel, for 1, 3, 4, 5 words per thread and a padded row (L = 448), and
    for the loop-free bit-window kernel of general L (66, 100, 126, 250: rows straddling words, a partial last word); E-only
    traces; the oracle at the smaller sizes."""
    spins, J = synth.make_spins(L, 1, 91), synth.make_couplings(L, 1, 92)
    g = Ising(L, 1, SEED, rng_mode)
    g.ising_load_state(dev(spins), dev(J))
    r = Ising(L, 1, SEED, rng_mode)
    r.ising_set_kernel(1)
    r.ising_load_state(dev(spins), dev(J))
    E, M = g.ising_sweep_trace(0.8, 3, every_half_sweeps=1)
    Er, Mr = r.ising_sweep_trace(0.8, 3, every_half_sweeps=1)
    assert torch.equal(E, Er) and torch.equal(M, Mr)
    assert torch.equal(g.ising_get_spins(), r.ising_get_spins())
    E2, none = g.ising_sweep_trace(0.8, 1, every_half_sweeps=2, want_M=False)      # E only, and the slots stay clean
    Er2, Mr2 = r.ising_sweep_trace(0.8, 1, every_half_sweeps=2)
    assert none is None and torch.equal(E2, Er2)
    Eg, Mg = g.ising_energy()                                                        # the separate energy kernel agrees
    assert int(Eg[0]) == int(Er2[-1, 0]) and int(Mg[0]) == int(Mr2[-1, 0])
    if L <= 128:
        o = ea3d.Oracle(L, 1, SEED, rng_mode)
        o.load_packed(spins, J)
        for k in range(6):
            o.half_sweep(0.8)
            Eo, Mo = o.energy()
            assert (int(E[k, 0]), int(M[k, 0])) == (int(Eo[0]), int(Mo[0])), k


# ------------------------------------------------------------------------------------------------ persistent kernel

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [64, 128, 192, 256, 320, 448])
def test_persistent_kernel_equals_one_launch_per_half_sweep(L, rng_mode):
    """Lattices with whole-word rows below L = 512 can run all half-sweeps of a call in one cooperative launch, the CTAs
    synchronising tile by tile through epoch counters (persistent.cuh; kernel choice 4, automatic for recorded calls at L = 64
    and 128); kernel choice 3 keeps one launch per half-sweep.  Same spins, E and M records for every record spacing (1, 2, 3, 5
    half-sweeps: records on red and on blue half-sweeps, a spacing that does not divide the call), from an odd starting counter
    (the call begins with a blue half-sweep, and MINSTD changes its multiplier after the first half-sweep), over several
    calls; the launch counts show which path ran; the oracle at the small sizes."""
    spins, J = synth.make_spins(L, 1, 71), synth.make_couplings(L, 1, 72)
    a = Ising(L, 1, SEED, rng_mode)
    a.ising_set_kernel(4)   # the persistent kernel for every call
    b = Ising(L, 1, SEED, rng_mode)
    b.ising_set_kernel(3)
    o = _loaded(L, 1, rng_mode, spins, J) if L <= 128 else None
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
    la, lb = a.ising_kernel_launches(), b.ising_kernel_launches()
    a.ising_sweep(0.8, 3)
    b.ising_sweep(0.8, 3)
    fills = 2 if rng_mode == MINSTD else 0          # the two seed-table launches
    assert a.ising_kernel_launches() - la == 1 + fills and b.ising_kernel_launches() - lb == 6 + (2 if rng_mode == MINSTD else 0)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    if o is not None:
        o.sweep(0.8, 3)
        assert_same_state(o, a, f"persistent L={L}")
    for every, nsw in ((1, 2), (2, 3), (3, 3), (5, 4)):
        Ea, Ma = a.ising_sweep_trace(0.8, nsw, every_half_sweeps=every)
        Eb, Mb = b.ising_sweep_trace(0.8, nsw, every_half_sweeps=every)
        assert Ea.shape[0] == (2 * nsw) // every and torch.equal(Ea, Eb) and torch.equal(Ma, Mb), every
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    if o is not None:
        o.sweep(0.8, 12)
        assert_same_state(o, a, f"persistent L={L} after the traces")
    # odd starting counter
    for g in (a, b):
        g.ising_set_t(7)
        g.ising_load_state(dev(spins), dev(J))
    Ea, Ma = a.ising_sweep_trace(1 / 1.1, 2, every_half_sweeps=1, want_M=False)
    Eb, Mb = b.ising_sweep_trace(1 / 1.1, 2, every_half_sweeps=1, want_M=False)
    assert Ma is None and torch.equal(Ea, Eb) and torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert a.ising_get_t() == 11 == b.ising_get_t()
    if o is not None and rng_mode == PHILOX:   # (the oracle's MINSTD streams are stored states: they cannot jump to t = 7)
        o2 = _loaded(L, 1, rng_mode, spins, J)
        o2.t = 7
        for k in range(4):
            o2.half_sweep(1 / 1.1)
            assert int(Ea[k, 0]) == int(o2.energy()[0][0]), k
        assert_same_state(o2, a, "odd starting counter")
    Eg, Mg = a.ising_energy()           # the separate energy kernel still works on the state the persistent kernel left
    assert int(Eg[0]) == int(Ea[-1, 0])


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_long_recorded_call_through_every_launch_structure(rng_mode):
    """66000 half-sweeps in one call with a record every 1001 (too far apart for a graph with records: one launch per half-sweep),
    the persistent kernel (choice 4: one cooperative launch) and one launch per half-sweep (choice 3): same records and spins."""
    L, nsw, every = 64, 33000, 1001
    spins, J = synth.make_spins(L, 1, 73), synth.make_couplings(L, 1, 74)
    res = []
    for choice in (0, 4, 3):
        g = Ising(L, 1, SEED, rng_mode)
        g.ising_set_kernel(choice)
        g.ising_load_state(dev(spins), dev(J))
        E, M = g.ising_sweep_trace(1 / 1.1, nsw, every_half_sweeps=every)
        res.append((E.clone(), M.clone(), g.ising_get_spins().clone()))
        assert g.ising_get_t() == 2 * nsw
    assert res[0][0].shape[0] == (2 * nsw) // every
    for r in res[1:]:
        assert all(torch.equal(x, y) for x, y in zip(res[0], r))


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L,nsamples", [(64, 1), (128, 1), (192, 1), (64, 32)])
def test_graph_replays_equal_one_launch_per_half_sweep(L, nsamples, rng_mode):
    """Calls of 16 half-sweeps and more on the one-sample lattices L = 64 and 128 replay CUDA graphs of up to 64 half-sweeps whose
    kernels take the half-sweep counter, the thresholds and the record position from a slot of constant memory (graph_kernels.cuh;
    automatic); kernel choice 3 keeps one launch per half-sweep (as does every other geometry: L = 192 and the sample-packed
    lattice are here to show that the same calls go through there too).  Same spins and records: calls of different lengths (graph
    cache, remainders launched), record spacings 1, 2, 3, 7 and 20, another beta, an odd starting counter across 2^32, and the
    oracle at the small sizes."""
    spins, J = synth.make_spins(L, nsamples, 87), synth.make_couplings(L, nsamples, 88)
    a = Ising(L, nsamples, SEED, rng_mode)
    a.ising_set_kernel(5)     # the automatic choice without the cluster-resident kernel, which otherwise takes L = 64
    b = Ising(L, nsamples, SEED, rng_mode)
    b.ising_set_kernel(3)
    small = nsamples * L**3 <= 64**3 * 2
    o = _loaded(L, nsamples, rng_mode, spins, J) if small else None
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
    la = a.ising_kernel_launches()
    for beta, n in ((1 / 1.1, 40), (0.6, 9), (1 / 1.1, 37), (0.6, 40)):     # 80 = 64 + 16 launched; 18; 74 = 64 + 10; again 80
        a.ising_sweep(beta, n)
        b.ising_sweep(beta, n)
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins()), (beta, n)
        if o is not None:
            o.sweep(beta, n)
    if nsamples == 1 and L <= 128:
        assert a.ising_kernel_launches() - la > 4 * 66      # the replays count their kernels (64 half-sweeps + 2 per replay)
    if o is not None:
        assert_same_state(o, a, f"graphs L={L} x {nsamples}")
    for every, n in ((1, 20), (2, 33), (3, 30), (7, 35), (20, 40)):
        Ea, Ma = a.ising_sweep_trace(0.8, n, every_half_sweeps=every)
        Eb, Mb = b.ising_sweep_trace(0.8, n, every_half_sweeps=every)
        assert Ea.shape[0] == (2 * n) // every and torch.equal(Ea, Eb) and torch.equal(Ma, Mb), every
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins()), every
    Ea, none = a.ising_sweep_trace(0.8, 16, every_half_sweeps=2, want_M=False)
    Eb, _ = b.ising_sweep_trace(0.8, 16, every_half_sweeps=2, want_M=False)
    assert none is None and torch.equal(Ea, Eb)
    for g in (a, b):
        g.ising_set_t(2**32 - 21)
        g.ising_sweep(1 / 1.1, 20)
    assert a.ising_get_t() == 2**32 + 19 and torch.equal(a.ising_get_spins(), b.ising_get_spins())
    assert torch.equal(a.ising_energy()[0], b.ising_energy()[0])


def test_graph_replays_of_two_handles_on_two_streams():
    """Every graph-using handle has its own slot of constant memory: two handles replaying graphs concurrently on two streams (and a
    third one created and destroyed in between) do not disturb each other."""
    L = 64
    jobs = []
    for i, (seed_s, mode) in enumerate(((91, PHILOX), (92, MINSTD))):
        spins, J = synth.make_spins(L, 1, seed_s), synth.make_couplings(L, 1, seed_s + 10)
        g = Ising(L, 1, SEED + i, mode)
        g.ising_set_kernel(5)
        r = Ising(L, 1, SEED + i, mode)
        r.ising_set_kernel(3)
        for h in (g, r):
            h.ising_load_state(dev(spins), dev(J))
        jobs.append((g, r, torch.cuda.Stream()))
    torch.cuda.synchronize()
    tmp = Ising(L, 1, 5, PHILOX)
    tmp.ising_load_state(dev(synth.make_spins(L, 1, 1)), dev(synth.make_couplings(L, 1, 2)))
    tmp.ising_sweep(0.5, 20)
    tmp.ising_destroy()
    for rep in range(3):
        for g, r, st in jobs:
            g.ising_sweep(1 / 1.1 if rep != 1 else 0.4, 64, stream=st)
    torch.cuda.synchronize()
    for g, r, st in jobs:
        for rep in range(3):
            r.ising_sweep(1 / 1.1 if rep != 1 else 0.4, 64)
        assert torch.equal(g.ising_get_spins(), r.ising_get_spins())


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [4, 6, 10, 16, 18, 22, 24, 32, 34, 40])
def test_on_chip_kernel_equals_the_oracle_and_one_launch_per_half_sweep(L, rng_mode):
    """Lattices of at most 1024 words per colour (every even L <= 40) run all half-sweeps and records of a call in ONE launch of ONE
    CTA out of shared memory (half_sweeps_on_chip).  Against the oracle half-sweep by half-sweep (E and M records of
    every spacing, red and blue), against one launch per half-sweep (kernel choice 3), from an odd starting counter, across
    several calls (the spins go back to global memory after every call), with the separate energy and get kernels afterwards."""
    spins, J = synth.make_spins(L, 1, 77), synth.make_couplings(L, 1, 78)
    o, a = make_pair(L, 1, rng_mode, spins, J)
    a.ising_set_kernel(4)     # wherever it exists (automatic where it is the faster one: up to L = 32 with records, 24 without)
    b = Ising(L, 1, SEED, rng_mode)
    b.ising_set_kernel(3)
    b.ising_load_state(dev(spins), dev(J))
    la = a.ising_kernel_launches()
    E, M = a.ising_sweep_trace(1 / 1.1, 5, every_half_sweeps=1)
    assert a.ising_kernel_launches() - la == 1
    Eb, Mb = b.ising_sweep_trace(1 / 1.1, 5, every_half_sweeps=1)
    assert torch.equal(E, Eb) and torch.equal(M, Mb)
    for k in range(10):
        o.half_sweep(1 / 1.1)
        Eo, Mo = o.energy()
        assert (int(E[k, 0]), int(M[k, 0])) == (int(Eo[0]), int(Mo[0])), k
    assert_same_state(o, a, f"on-chip L={L}")
    a.ising_sweep(0.5, 7)
    o.sweep(0.5, 7)
    assert_same_state(o, a, f"on-chip L={L}, second call")
    E, none = a.ising_sweep_trace(0.9, 4, every_half_sweeps=3, want_M=False)     # records after half-sweeps 3 and 6 of 8
    o.sweep(0.9, 1)
    o.half_sweep(0.9)
    e3 = int(o.energy()[0][0])
    o.half_sweep(0.9)
    o.sweep(0.9, 1)
    e6 = int(o.energy()[0][0])
    o.sweep(0.9, 1)
    assert none is None and E.shape[0] == 2 and (int(E[0, 0]), int(E[1, 0])) == (e3, e6)
    assert_same_state(o, a, f"on-chip L={L}, third call")
    if rng_mode == PHILOX:   # odd starting counter (the oracle's stored MINSTD streams cannot jump)
        o.t = 2**32 - 1
        a.ising_set_t(2**32 - 1)
        o.sweep(1 / 0.7, 2)
        a.ising_sweep(1 / 0.7, 2)
        assert a.ising_get_t() == 2**32 + 3
        assert_same_state(o, a, "odd starting counter across 2^32")


def test_config1_through_every_launch_structure():
    """BASELINE.json config 1 (L = 16, E per half-sweep): the on-chip kernel (automatic), one launch per half-sweep (choice 3) and
    the one-site-at-a-time kernels (choice 1) give the same 20 energies and the same final spins."""
    cfg, spins, J = synth.make_config(1)
    res = []
    for choice in (0, 3, 1):
        g = Ising(cfg["L"], 1, SEED, cfg["rng_mode"])
        g.ising_set_kernel(choice)
        g.ising_load_state(dev(spins), dev(J))
        E, M = g.ising_sweep_trace(cfg["beta"], cfg["sweeps"], every_half_sweeps=1)
        res.append((E.clone(), M.clone(), g.ising_get_spins().clone(), g.ising_kernel_launches()))
    for r in res[1:]:
        assert all(torch.equal(x, y) for x, y in zip(res[0][:3], r[:3]))
    assert res[0][3] == 1 + 1 + 1 and res[1][3] >= 1 + 20 + 20      # load + one launch + get   against   load + 20 x (sweep + energy) + get


def test_handle_belongs_to_the_current_device():
    """A handle is created on torch's current device and every call runs there (the binding used to default to
    cuda:0 whatever the process had selected).  With a second GPU visible, the same job on device 1 gives the same bits, and the
    library refuses a call made with another device current."""
    g = Ising(64, 1, SEED, PHILOX)
    assert g.device.index == torch.cuda.current_device() and g.workspace.device == g.device
    if torch.cuda.device_count() < 2:
        return
    spins, J = synth.make_spins(64, 1, 2), synth.make_couplings(64, 1, 1)
    g.ising_load_state(dev(spins), dev(J))
    g.ising_sweep(0.9, 3)
    with torch.cuda.device(1):
        h = Ising(64, 1, SEED, PHILOX)
        assert h.device.index == 1 and h.workspace.device.index == 1
        sp1 = torch.from_numpy(spins.view(np.int32)).to("cuda:1")
        J1 = torch.from_numpy(J.view(np.int32)).to("cuda:1")
        h.ising_load_state(sp1, J1)
        h.ising_sweep(0.9, 3)
        out1 = h.ising_get_spins()
        assert out1.device.index == 1
    assert torch.equal(out1.cpu(), g.ising_get_spins().cpu())
    h.ising_sweep(0.9, 1)      # called with device 0 current: the binding switches to the handle's device for the call
    with pytest.raises(AssertionError):
        h.ising_load_state(dev(spins), dev(J))   # tensors of device 0 handed to a handle of device 1
    # the C library itself refuses a launch for a handle of another device than the current one
    assert binding.lib().ising_sweep(h._h, 0.9, 1, None) == binding.EINVAL


# ------------------------------------------------------------------------------------------------ FNV-1a on the device

@pytest.mark.parametrize("nbytes", [0, 1, 2, 3, 4, 5, 255, 256, 257, 1000, 4099, 227328, 227332, 229376, 229380, 1 << 20, (1 << 24) + 4])
def test_fnv1a64_on_the_device_equals_the_definition(nbytes):
    """ising_fnv1a64 (parallel: low-byte maps per chunk, composed, then per-chunk sums) against the byte-by-byte definition as the
    oracle and the host routine compute it: empty input, lengths that are not multiples of 4, one chunk, the chunk boundary, 888
    chunks, random bytes and the all-0xff / all-zero strings."""
    rng = np.random.default_rng(nbytes)
    for kind in ("random", "ff", "zero"):
        if kind == "random":
            host = rng.integers(0, 256, nbytes, dtype=np.uint8)
        else:
            host = np.full(nbytes, 0xFF if kind == "ff" else 0, dtype=np.uint8)
        pad = (-nbytes) % 4
        d = torch.from_numpy(np.concatenate([host, np.zeros(pad, dtype=np.uint8)])).cuda()[:nbytes]
        got = int(binding.ising_fnv1a64(d)[0]) & (2**64 - 1)
        assert got == ea3d.fnv1a64(host) == binding.ising_fnv1a64_host(host), (nbytes, kind)
        if nbytes > 1 << 20 and kind == "random":
            break


@pytest.mark.parametrize("nbytes", [1000, 227332, (1 << 22) + 3])
def test_fnv1a64_scratch_between_guards(nbytes):
    """Memory safety without a sanitizer: the scratch of ising_fnv1a64 sits between two guard regions, and so does the input."""
    G = 1 << 20
    sb = binding.ising_fnv1a64_scratch_bytes(nbytes)
    buf = torch.full((G + sb + G,), 0xA5, dtype=torch.uint8, device="cuda")
    host = np.random.default_rng(nbytes).integers(0, 256, nbytes, dtype=np.uint8)
    data = torch.full((G + nbytes + G,), 0x5A, dtype=torch.uint8, device="cuda")
    data[G:G + nbytes] = torch.from_numpy(host).cuda()
    out = torch.full((3,), 0x1234, dtype=torch.int64, device="cuda")
    binding.ising_fnv1a64(data[G:G + nbytes], out=out[1:2], scratch=buf[G:G + sb])
    torch.cuda.synchronize()
    assert int(out[1]) & (2**64 - 1) == ea3d.fnv1a64(host)
    assert int(out[0]) == 0x1234 and int(out[2]) == 0x1234
    assert bool((buf[:G] == 0xA5).all()) and bool((buf[G + sb:] == 0xA5).all()), "scratch guard overwritten"
    assert bool((data[:G] == 0x5A).all()) and bool((data[G + nbytes:] == 0x5A).all()), "input guard overwritten"


def test_fnv1a64_on_the_device_of_the_spins_of_a_run():
    """The use config 4 makes of it: the checksum of the canonical spins after some sweeps, device routine = host routine."""
    L = 128
    g = Ising(L, 1, SEED, PHILOX)
    g.ising_load_state(dev(synth.make_spins(L, 1, 3)), dev(synth.make_couplings(L, 1, 4)))
    scratch = torch.empty(binding.ising_fnv1a64_scratch_bytes(L**3 // 8), dtype=torch.uint8, device="cuda")
    out = torch.empty(1, dtype=torch.int64, device="cuda")
    for _ in range(3):
        g.ising_sweep(1 / 1.1, 2)
        spins = g.ising_get_spins()
        binding.ising_fnv1a64(spins, out=out, scratch=scratch)
        assert int(out[0]) & (2**64 - 1) == binding.ising_fnv1a64_host(host_u32(spins))
