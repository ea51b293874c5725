"""The paper's sliced layout (Eq. 4-6) as an alternative internal layout (-m gpu): the same trajectory as the
rank-linear arrays and the CPU oracle, bit for bit, in both rng modes (all schemes give the same bits)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import ea3d  # noqa: E402
from paper_1411_0127_b200 import MINSTD, PHILOX, Ising, binding, synth  # noqa: E402

pytestmark = pytest.mark.gpu
SEED = synth.DYN_SEED


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [64, 128, 256, 512])
def test_sliced_layout_follows_the_same_trajectory(L, rng_mode):
    spins, J = synth.make_spins(L, 1, 85), synth.make_couplings(L, 1, 86)
    a = Ising(L, 1, SEED, rng_mode)
    b = Ising(L, 1, SEED, rng_mode)
    for g in (a, b):
        g.ising_load_state(dev(spins), dev(J))
    # round trip of the layout conversion alone
    a.ising_sliced_begin()
    a.ising_sliced_end()
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())
    o = None
    if L <= 128:
        o = ea3d.Oracle(L, 1, SEED, rng_mode)
        o.load_packed(spins, J)
    for beta, n in ((1 / 1.1, 2), (0.5, 1)):
        a.ising_sliced_begin()
        a.ising_sliced_sweep(beta, n)
        a.ising_sliced_end()
        b.ising_sweep(beta, n)
        assert a.ising_get_t() == b.ising_get_t()
        assert torch.equal(a.ising_get_spins(), b.ising_get_spins()), f"L={L} mode {rng_mode} beta {beta}"
        assert torch.equal(a.ising_energy()[0], b.ising_energy()[0])
        if o is not None:
            o.sweep(beta, n)
            assert np.array_equal(a.ising_get_spins().cpu().numpy().view(np.uint32), o.spins_packed())
    # the two layouts can alternate within one run: sweeps in the sliced layout, then in the handle's own
    a.ising_sweep(0.7, 1)
    b.ising_sweep(0.7, 1)
    assert torch.equal(a.ising_get_spins(), b.ising_get_spins())


def test_sliced_layout_argument_checks():
    with pytest.raises(binding.IsingError):
        Ising(192, 1, SEED, PHILOX).ising_sliced_begin()      # rows of 6 words: lanes per row not a power of two
    with pytest.raises(binding.IsingError):
        Ising(16, 1, SEED, PHILOX).ising_sliced_begin()       # rows shorter than a word
    with pytest.raises(binding.IsingError):
        Ising(64, 32, SEED, PHILOX).ising_sliced_begin()      # sample-packed handle
