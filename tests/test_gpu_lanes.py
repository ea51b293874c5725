"""GPU parity tests (-m gpu) of the stored-state lane generators (rng_mode 3 = Parisi-Rapuano, 4 = MT19937; PAPER.md:180-195,
SURVEY.md 8(f) rank 2, R19): the shared-draw sweep driven by them and the Table II odd-count benchmark, through the
C ABI, against the CPU oracle -- tolerance 0 (all outputs are integers)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import MT19937_SHARED, PHILOX, MINSTD, PR_SHARED, Ising, binding, synth  # noqa: E402

pytestmark = pytest.mark.gpu
SEED = synth.DYN_SEED


def dev(a: np.ndarray):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def host_u32(t) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def make_pair(L, ns, mode, nlanes, spins, J):
    g = Ising(L, ns, SEED, mode)
    if nlanes is not None:
        g.ising_set_lanes(nlanes)
    o = ea3d.Oracle(L, ns, SEED, mode, nlanes=g.ising_get_lanes())
    o.load_packed(spins, J)
    g.ising_load_state(dev(spins), dev(J))
    return o, g


def assert_same_state(o, g, what=""):
    got = host_u32(g.ising_get_spins())
    want = o.spins_packed()
    assert np.array_equal(got, want), f"{what}: {np.count_nonzero(got != want)} of {want.size} spin words differ"
    E, M = g.ising_energy()
    Eo, Mo = o.energy()
    assert np.array_equal(E.cpu().numpy(), Eo) and np.array_equal(M.cpu().numpy(), Mo), what


# nlanes None = the default min(N/8, 151552); the others give several rounds per lane and a ragged last round
@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
# (16, 32, 7), (24, 64, 50): many rounds per lane, the ring wraps several times inside one launch; L = 4, 6, 10, 12, 20, 30: groups
# of four sites that straddle rows (L % 8 != 0, per-word neighbour loads)
@pytest.mark.parametrize("L,ns,nlanes", [(8, 32, None), (8, 64, 24), (16, 32, 100), (16, 96, 512), (24, 32, 333), (40, 32, None),
                                         (40, 64, 1000), (64, 32, 4096), (16, 32, 7), (24, 64, 50), (8, 1024, None), (8, 160, 300),
                                         (16, 96, None), (4, 32, None), (6, 64, 5), (10, 32, None), (12, 96, 100), (20, 32, 333),
                                         (30, 64, None)])
def test_lane_mode_sweep_equals_the_oracle(mode, L, ns, nlanes):
    spins, J = synth.make_spins(L, ns, 71), synth.make_couplings(L, ns, 72)
    o, g = make_pair(L, ns, mode, nlanes, spins, J)
    for beta, n in ((1 / 1.1, 2), (0.3, 1), (1 / 0.7, 2)):   # 10 half-sweeps: the ring position wraps (62) on most cases
        o.sweep(beta, n)
        g.ising_sweep(beta, n)
        assert_same_state(o, g, f"lane mode {mode} L={L} ns={ns} nlanes={nlanes} beta={beta}")


@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
def test_lane_mode_with_the_default_wave_of_lanes(mode):
    """The launch configuration bench.py times: 151552 lanes (1184 CTAs of 128, one wave).  L = 128 has 262144 groups per colour:
    two rounds per lane, the second one ragged; 64 samples = two coded batches."""
    L, ns = 128, 64
    spins, J = synth.make_spins(L, ns, 77), synth.make_couplings(L, ns, 78)
    o, g = make_pair(L, ns, mode, None, spins, J)
    assert g.ising_get_lanes() == 148 * 1024
    for beta, n in ((1 / 1.1, 1), (0.5, 1)):
        o.sweep(beta, n)
        g.ising_sweep(beta, n)
        assert_same_state(o, g, f"lane mode {mode}, default lanes, beta={beta}")


@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
def test_lane_mode_many_half_sweeps_cross_the_mt_ring(mode):
    """L = 8, 2 batches, 3 lanes: 4 * ceil(2 * 64 / 3) = 172 draws per lane per half-sweep; 8 half-sweeps = 1376 draws cross the
    624-word MT block twice and the 62-word ring 22 times.  Sweeps split over several calls (the state persists)."""
    L, ns = 8, 64
    spins, J = synth.make_spins(L, ns, 73), synth.make_couplings(L, ns, 74)
    o, g = make_pair(L, ns, mode, 3, spins, J)
    for n in (1, 2, 1):
        o.sweep(0.8, n)
        g.ising_sweep(0.8, n)
        assert_same_state(o, g, f"mode {mode} after {n}")
    E, M = g.ising_sweep_trace(0.8, 1, 1)
    want = []
    for _ in range(2):
        o.half_sweep(0.8)
        want.append(o.energy()[0])
    assert np.array_equal(E.cpu().numpy(), np.stack(want))


@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
@pytest.mark.parametrize("beta", [0.0, float("inf")])
def test_lane_mode_special_temperatures(mode, beta):
    L, ns = 16, 32
    spins, J = synth.make_spins(L, ns, 75), synth.make_couplings(L, ns, 76)
    o, g = make_pair(L, ns, mode, 77, spins, J)
    o.sweep(beta, 2)
    g.ising_sweep(beta, 2)
    assert_same_state(o, g, f"lane mode beta={beta}")


@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
def test_lane_mode_checkpoint_and_resume(mode):
    """The run state is (workspace bytes, t, nlanes): a copy of the workspace taken after 3 sweeps, resumed in a new handle, continues
    exactly like the uninterrupted run (and like the oracle)."""
    L, ns, nlanes = 16, 64, 77
    spins, J = synth.make_spins(L, ns, 81), synth.make_couplings(L, ns, 82)
    o, g = make_pair(L, ns, mode, nlanes, spins, J)
    g.ising_sweep(0.9, 3)
    o.sweep(0.9, 3)
    torch.cuda.synchronize()
    saved, t = g.workspace.clone(), g.ising_get_t()
    g.ising_sweep(0.9, 2)
    o.sweep(0.9, 2)
    r = Ising(L, ns, SEED, mode, workspace=saved)
    r.ising_resume_lanes(t, nlanes)
    r.ising_sweep(0.9, 2)
    assert torch.equal(r.ising_get_spins(), g.ising_get_spins())
    assert_same_state(o, r, "resumed run")
    with pytest.raises(binding.IsingError):
        Ising(16, 32, SEED, PHILOX).ising_resume_lanes(0, 1)


def test_lane_mode_argument_checks():
    for mode in (PR_SHARED, MT19937_SHARED):
        with pytest.raises(binding.IsingError):
            Ising(16, 1, SEED, mode)          # needs whole words of samples
        g = Ising(16, 32, SEED, mode)
        assert g.ising_get_lanes() == 16**3 // 8
        assert Ising(8, 96, SEED, mode).ising_get_lanes() == 3 * 8**3 // 8    # units = batches x groups
        with pytest.raises(binding.IsingError):
            g.ising_set_lanes(0)
        with pytest.raises(binding.IsingError):
            g.ising_set_lanes(16**3 // 8 + 1)
        with pytest.raises(binding.IsingError):
            g.ising_set_t(4)                   # the generator state is not a function of t
        spins, J = synth.make_spins(16, 32, 1), synth.make_couplings(16, 32, 2)
        g.ising_load_state(dev(spins), dev(J))
        g.ising_sweep(0.5, 1)
        with pytest.raises(binding.IsingError):
            g.ising_set_lanes(8)               # only before the first sweep
    with pytest.raises(binding.IsingError):
        Ising(16, 32, SEED, PHILOX).ising_get_lanes()


# ------------------------------------------------------------------------------------------------ Table II: odd count

@pytest.mark.parametrize("kind", [PHILOX, MINSTD, PR_SHARED, MT19937_SHARED])
@pytest.mark.parametrize("nlanes,chunks", [(1, (4, 8)), (37, (64, 700, 1236)), (1000, (2000,)), (300, (60, 64, 4))])
def test_count_odd_equals_the_oracle(kind, nlanes, chunks):
    seed = 99
    nbytes = binding.ising_prng_state_bytes(kind, nlanes)
    state = torch.empty(max(nbytes, 1), dtype=torch.uint8, device="cuda") if nbytes else None
    binding.ising_prng_init(kind, seed, nlanes, state)
    odd = torch.zeros(nlanes, dtype=torch.int64, device="cuda")
    tot = torch.zeros(nlanes, dtype=torch.int64, device="cuda")
    done = 0
    odd_all = np.zeros(nlanes, np.uint64)
    tot_all = np.zeros(nlanes, np.uint64)
    for n in chunks:                      # the state persists between calls: chunks concatenate
        binding.ising_prng_count_odd(kind, seed, nlanes, done, n, state, odd, tot)
        odd_all += odd.cpu().numpy().view(np.uint64)
        tot_all += tot.cpu().numpy().view(np.uint64)
        done += n
    want_odd, want_tot = ea3d.count_odd(kind, seed, nlanes, done)
    assert np.array_equal(odd_all, want_odd)
    assert np.array_equal(tot_all, want_tot)


@pytest.mark.parametrize("kind", [PHILOX, MINSTD, PR_SHARED, MT19937_SHARED])
def test_count_odd_in_the_bench_configuration(kind):
    """bench.py's Table II run: 151552 lanes x 4096 draws per call (two calls here), every lane against the oracle."""
    seed, nlanes, nd = synth.DYN_SEED, 148 * 1024, 4096
    nbytes = binding.ising_prng_state_bytes(kind, nlanes)
    state = torch.empty(nbytes, dtype=torch.uint8, device="cuda") if nbytes else None
    binding.ising_prng_init(kind, seed, nlanes, state)
    odd = torch.zeros(nlanes, dtype=torch.int64, device="cuda")
    tot = torch.zeros(nlanes, dtype=torch.int64, device="cuda")
    odd_all = np.zeros(nlanes, np.uint64)
    tot_all = np.zeros(nlanes, np.uint64)
    for r in range(2):
        binding.ising_prng_count_odd(kind, seed, nlanes, r * nd, nd, state, odd, tot)
        odd_all += odd.cpu().numpy().view(np.uint64)
        tot_all += tot.cpu().numpy().view(np.uint64)
    want_odd, want_tot = ea3d.count_odd(kind, seed, nlanes, 2 * nd)
    assert np.array_equal(odd_all, want_odd)
    assert np.array_equal(tot_all, want_tot)


def test_count_odd_argument_checks():
    odd = torch.zeros(4, dtype=torch.int64, device="cuda")
    with pytest.raises(binding.IsingError):
        binding.ising_prng_count_odd(PHILOX, 1, 4, 0, 6, None, odd, odd)     # not a multiple of 4
    with pytest.raises(binding.IsingError):
        binding.ising_prng_state_bytes(2, 4)                                   # the shared Philox mode has no lanes
    assert binding.ising_prng_state_bytes(PHILOX, 10) == 0
    assert binding.ising_prng_state_bytes(MINSTD, 10) == 40
    assert binding.ising_prng_state_bytes(PR_SHARED, 10) == 62 * 40
    assert binding.ising_prng_state_bytes(MT19937_SHARED, 10) == 624 * 40


# ------------------------------------------------------------------------------------------------ memory safety

@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
@pytest.mark.parametrize("L,ns,nlanes", [(8, 32, None), (16, 64, 100), (24, 32, 7)])
def test_lane_kernels_write_only_inside_their_buffers(mode, L, ns, nlanes):
    """Memory safety without a sanitizer: the workspace (lattice + strided generator state) and the Table II state / result
    buffers sit between guard regions filled with a pattern; after every entry point has run the guards must be untouched."""
    nbytes = binding.ising_workspace_bytes(L, ns, mode)
    G = 1 << 20
    buf = torch.full((G + nbytes + G,), 0xA5, dtype=torch.uint8, device="cuda")
    spins, J = synth.make_spins(L, ns, 95), synth.make_couplings(L, ns, 96)
    g = Ising(L, ns, SEED, mode, workspace=buf[G:G + nbytes])
    if nlanes is not None:
        g.ising_set_lanes(nlanes)
    g.ising_load_state(dev(spins), dev(J))
    g.ising_sweep(1 / 1.1, 3)
    g.ising_sweep_trace(1 / 1.1, 1, every_half_sweeps=1)
    g.ising_get_spins()
    torch.cuda.synchronize()
    assert bool((buf[:G] == 0xA5).all()) and bool((buf[G + nbytes:] == 0xA5).all()), "workspace guard overwritten"
    # Table II kernels: state and per-lane results between guards
    n = 333
    sb = binding.ising_prng_state_bytes(mode, n)
    st = torch.full((G + sb + G,), 0xA5, dtype=torch.uint8, device="cuda")
    res = torch.full((1024 + 2 * n + 1024,), 0x5A5A5A5A5A5A5A5A, dtype=torch.int64, device="cuda")
    binding.ising_prng_init(mode, 5, n, st[G:G + sb])
    for first, nd in ((0, 1000), (1000, 40), (1040, 64)):   # staged (>= 62 draws) and unstaged Parisi-Rapuano kernels
        binding.ising_prng_count_odd(mode, 5, n, first, nd, st[G:G + sb], res[1024:1024 + n], res[1024 + n:1024 + 2 * n])
    torch.cuda.synchronize()
    assert bool((st[:G] == 0xA5).all()) and bool((st[G + sb:] == 0xA5).all()), "state guard overwritten"
    assert bool((res[:1024] == 0x5A5A5A5A5A5A5A5A).all()) and bool((res[1024 + 2 * n:] == 0x5A5A5A5A5A5A5A5A).all()), "result guard"


@pytest.mark.parametrize("mode", [PR_SHARED, MT19937_SHARED])
def test_lane_mode_long_run(mode):
    """200 half-sweeps in uneven calls: the ring position handed to every launch ((t mod ring) * (draws per half-sweep mod ring)
    mod ring) must track the generators exactly; 332 draws per lane and half-sweep, 66400 in total (106 MT19937 blocks)."""
    L, ns, nlanes = 16, 64, 13
    spins, J = synth.make_spins(L, ns, 87), synth.make_couplings(L, ns, 88)
    o, g = make_pair(L, ns, mode, nlanes, spins, J)
    for n in (1, 7, 30, 62):
        o.sweep(1 / 1.1, n)
        g.ising_sweep(1 / 1.1, n)
        assert_same_state(o, g, f"after {n} more sweeps")
    assert g.ising_get_t() == 200
