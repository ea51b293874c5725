"""Pins of the oracle's shared-random-number mode (Eq. 15; R18): the 32
samples coded in one word share one draw per (site, half-sweep).

The mode adds no arithmetic of its own: every sample still follows the scalar rule Eq. 9 with a uniform 32-bit draw, so
  (1) the trajectory of sample s of batch b is, bit for bit, the trajectory of a ONE-sample run of the already pinned
      independent mode with sample index b (same J, same spins): the marginal chain of every sample is the pinned chain;
  (2) what is new is the coupling between samples: two samples of a batch that start from the same state with the same
      couplings stay identical for ever (they see the same draws), which does not hold in the independent mode;
  (3) samples in different batches use different draws.
"""
import numpy as np
import pytest

from oracle import ea3d
from paper_1411_0127_b200 import synth


def _oracle(L, ns, mode, spins, J, seed=77):
    o = ea3d.Oracle(L, ns, seed, mode)
    o.load_packed(spins, J)
    return o


@pytest.mark.parametrize("L", [4, 6, 8])
def test_every_sample_follows_the_pinned_single_sample_chain(L):
    ns = 64
    spins, J = synth.make_spins(L, ns, 5), synth.make_couplings(L, ns, 6)
    W = (L**3 + 31) // 32
    sh = _oracle(L, ns, ea3d.PHILOX_SHARED, spins, J)
    for _ in range(6):
        sh.half_sweep(0.6)
    got = sh.spins_packed()
    J3 = J.reshape(ns, 3, W)
    sp = spins.reshape(ns, W)
    for s in (0, 1, 17, 31, 32, 45, 63):
        # independent mode, one sample: oracle_philox_draw keys sample index 0, so shift the seed's high word by b
        b = s >> 5
        one = ea3d.Oracle(L, 1, 77 ^ (b << 32), ea3d.PHILOX)
        one.load_packed(sp[s], J3[s])
        for _ in range(6):
            one.half_sweep(0.6)
        assert np.array_equal(one.spins_packed()[0], got[s]), s


def test_equal_samples_of_a_batch_stay_equal_and_batches_differ():
    L, ns = 6, 64
    W = (L**3 + 31) // 32
    spins1, J1 = synth.make_spins(L, 1, 9), synth.make_couplings(L, 1, 10)
    spins = np.tile(spins1.reshape(1, W), (ns, 1))
    J = np.tile(J1.reshape(1, 3, W), (ns, 1, 1))
    sh = _oracle(L, ns, ea3d.PHILOX_SHARED, spins, J)
    ind = _oracle(L, ns, ea3d.PHILOX, spins, J)
    for _ in range(8):
        sh.half_sweep(0.5)
        ind.half_sweep(0.5)
    a, b = sh.spins_packed(), ind.spins_packed()
    assert all(np.array_equal(a[0], a[s]) for s in range(32))          # one word, one draw
    assert all(np.array_equal(a[32], a[s]) for s in range(32, 64))
    assert not np.array_equal(a[0], a[32])                              # another batch, other draws
    assert not np.array_equal(b[0], b[1])                               # independent draws decorrelate equal samples


def test_shared_mode_thresholds_are_the_philox_ones():
    for beta in (0.0, 0.3, 1 / 1.1, 5.0, float("inf")):
        assert ea3d.thresholds(beta, ea3d.PHILOX_SHARED) == ea3d.thresholds(beta, ea3d.PHILOX)
