"""Lattices beyond L = 2048 (-m gpu): L = 2560, 3072 (rows of 5 and 3 x 8 words) and L = 4096, where the Philox group index passes
2^32 and its high word enters the counter (R9), and where the MINSTD seed states are recomputed instead of cached.

The oracle cannot hold these lattices (one int8 per spin: 17-69 GB per array), so the checks are the ones the brief names for full
sizes: sampled sites against the oracle one by one (the oracle's own draw of the site and its own threshold table, the local field
from the canonical bits; both halves of the lattice, its corners and its periodic seams), the word-parallel kernel against the
one-site-at-a-time kernel over a whole sweep, and properties that hold at any size (round trip, records = ising_energy, parity of E).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import MINSTD, PHILOX, Ising, synth  # noqa: E402

pytestmark = pytest.mark.gpu
SEED = synth.DYN_SEED


def _bits(d_words, idx):
    """Bits number idx (int64 array) of a flat int32 CUDA tensor of canonical words, as a numpy array of 0 / 1."""
    idx = np.asarray(idx, dtype=np.int64)
    w = d_words[torch.from_numpy(idx >> 5).cuda()].cpu().numpy().view(np.uint32)
    return ((w >> (idx & 31).astype(np.uint32)) & 1).astype(np.int64)


def _sample_sites(L, colour, n, rng):
    pts = [(0, 0, 0), (L - 1, L - 1, L - 1), (0, L - 1, 0), (L - 1, 0, L // 2), (1, 0, L // 2 - 1), (5, 7, L // 2), (L - 2, 3, L - 1)]
    pts += [tuple(int(v) for v in rng.integers(0, L, 3)) for _ in range(n)]
    return [((x ^ 1) if ((x + y + z) & 1) != colour else x, y, z) for x, y, z in pts]


def _expected_flips(L, rng_mode, beta, t, d_spins, d_J, sites):
    """flip (0 / 1) of every site in `sites` (all of colour t & 1) in half-sweep t from the state d_spins: Eq. 8-9 with the oracle's draw."""
    N = L**3
    T = ea3d.thresholds(beta, rng_mode)
    xs, ys, zs = (np.array(v, dtype=np.int64) for v in zip(*sites))
    i = xs + L * (ys + L * zs)
    s = 2 * _bits(d_spins, i) - 1
    h = np.zeros_like(s)
    for d, (dx, dy, dz) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
        ip = (xs + dx) % L + L * ((ys + dy) % L + L * ((zs + dz) % L))
        im = (xs - dx) % L + L * ((ys - dy) % L + L * ((zs - dz) % L))
        h += (1 - 2 * _bits(d_J, d * N + i)) * (2 * _bits(d_spins, ip) - 1)       # bond (i, i + d), owned by i
        h += (1 - 2 * _bits(d_J, d * N + im)) * (2 * _bits(d_spins, im) - 1)      # bond (i - d, i), owned by the neighbour
    dE = 2 * s * h
    out = []
    for k, (x, y, z) in enumerate(sites):
        if rng_mode == PHILOX:
            R = ea3d.philox_draw(L, SEED, 0, x, y, z, t)
        else:
            R = ea3d.minstd_draw(SEED, int(i[k]), t >> 1)
        out.append(int(dE[k] <= 0 or R < T[int(dE[k]) // 4 - 1]))
    return i, np.array(out)


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [2560, 3072, 4096])
def test_lattices_beyond_L2048(L, rng_mode):
    W = L**3 // 32
    beta = 1 / 1.1
    gen = torch.Generator(device="cuda").manual_seed(L)
    d_spins = torch.randint(-2**31, 2**31 - 1, (W,), dtype=torch.int32, device="cuda", generator=gen)
    d_J = torch.randint(-2**31, 2**31 - 1, (3 * W,), dtype=torch.int32, device="cuda", generator=gen)
    g = Ising(L, 1, SEED, rng_mode)
    out = torch.empty((1, W), dtype=torch.int32, device="cuda")
    g.ising_load_state(d_spins, d_J)
    g.ising_get_spins(out)
    assert torch.equal(out.flatten(), d_spins), "round trip"
    E0 = int(g.ising_energy()[0][0])

    # one sweep with a record after each half-sweep (the measuring variant of the kernel)
    E, M = g.ising_sweep_trace(beta, 1, every_half_sweeps=1)
    g.ising_get_spins(out)
    E1, M1 = g.ising_energy()
    assert int(E[1, 0]) == int(E1[0]) and int(M[1, 0]) == int(M1[0]), "records of the half-sweep kernel = the energy kernel"
    assert E0 % 2 == (3 * L**3) % 2 == int(E1[0]) % 2 and int(E1[0]) < E0, "a quench from random spins lowers the energy"

    rng = np.random.default_rng(L + rng_mode)
    # red sites change in half-sweep 0 only: final = before ^ flips(t = 0)
    sites = _sample_sites(L, 0, 300, rng)
    i, flips = _expected_flips(L, rng_mode, beta, 0, d_spins, d_J, sites)
    assert np.array_equal(_bits(out.flatten(), i), _bits(d_spins, i) ^ flips), "red sites against the oracle's rule"
    assert 0 < flips.sum() < len(sites)
    if L == 4096:   # both sides of the Philox group index 2^32
        zs = np.array([s[2] for s in sites])
        assert (zs >= L // 2).sum() > 50 and (zs < L // 2).sum() > 50

    # the one-site-at-a-time kernel (64-bit indices throughout) over the same sweep, on the same handle
    sweep_out = out.clone()
    g.ising_set_kernel(1)
    g.ising_load_state(d_spins, d_J)
    g.ising_set_t(0)
    g.ising_sweep(beta, 1)
    g.ising_get_spins(out)
    assert torch.equal(out, sweep_out), "word-parallel kernel = one-site-at-a-time kernel"
    assert int(g.ising_energy()[0][0]) == int(E1[0])
    del sweep_out

    # blue sites: the same state at the odd counter 1, so that the next sweep starts with the blue half-sweep t = 1
    g.ising_set_kernel(0)
    g.ising_load_state(d_spins, d_J)
    g.ising_set_t(1)
    g.ising_sweep(beta, 1)
    g.ising_get_spins(out)
    sites = _sample_sites(L, 1, 300, rng)
    i, flips = _expected_flips(L, rng_mode, beta, 1, d_spins, d_J, sites)
    assert np.array_equal(_bits(out.flatten(), i), _bits(d_spins, i) ^ flips), "blue sites against the oracle's rule"
    assert g.ising_get_t() == 3
    g.ising_destroy()


def test_z_slabs_of_the_L4096_lattice():
    """L = 4096 cut into two z-slabs (the upper one holds the Philox groups beyond 2^32): one sweep with the exchange by copies and
    one with the exchange fused into the boundary kernels, against the undivided lattice."""
    from paper_1411_0127_b200 import IsingSlab, binding

    L, G, beta = 4096, 2, 1 / 1.1
    W = L**3 // 32
    gen = torch.Generator(device="cuda").manual_seed(99)
    d_spins = torch.randint(-2**31, 2**31 - 1, (W,), dtype=torch.int32, device="cuda", generator=gen)
    d_J = torch.randint(-2**31, 2**31 - 1, (3 * W,), dtype=torch.int32, device="cuda", generator=gen)
    ref = Ising(L, 1, SEED, PHILOX)
    ref.ising_load_state(d_spins, d_J)
    ref.ising_sweep(beta, 2)
    want = ref.ising_get_spins().flatten()
    Er, Mr = (int(v[0]) for v in ref.ising_energy())
    ref.ising_destroy()
    del ref
    torch.cuda.empty_cache()
    hs = [IsingSlab(L, G, r, SEED, PHILOX) for r in range(G)]
    for h in hs:
        h.ising_load_state(d_spins, d_J)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    binding.ising_slab_sweep_local(hs, beta, 1, sa, sb)
    binding.ising_slab_sweep_local(hs, beta, 1, sa, sb, push=True)
    torch.cuda.synchronize()
    out = torch.zeros(W, dtype=torch.int32, device="cuda")
    for h in hs:
        h.ising_get_spins(out)
    assert torch.equal(out, want)
    assert sum(int(h.ising_energy()[0][0]) for h in hs) == Er and sum(int(h.ising_energy()[1][0]) for h in hs) == Mr
