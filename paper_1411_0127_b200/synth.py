"""Seeded synthetic inputs for the 3D +-J Edwards-Anderson sweep (SURVEY.md section 8(c) reading c14).

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path.  It
holds none of the method's arithmetic: it only manufactures the inputs of the paper's
workload -- i.i.d. bimodal couplings J = +-1 with p = 1/2 (Eq. 2) and random or
ordered initial spins (off-equilibrium relaxation from a quench) -- in the
canonical bit-packed format of ``include/ising.h``:

* spins:     ``nsamples x W`` uint32, W = ceil(N/32), N = L**3; bit (i & 31) of word (i >> 5)
             is site i = x + L*(y + L*z); bit 1 <=> sigma = +1          (Eq. 10)
* couplings: ``nsamples x 3 x W`` uint32 ordered [sample][dir x,y,z][word]; the bit of site i
             in direction d is the bond between i and i + d-hat; bit 1 <=> J = -1 (Eq. 10)

Bits above N in the last word are zero.

Recipe (frozen): word k (0-based) of a bit array drawn from
``seed`` is the high 32 bits of the (k+1)-th output of a 64-bit Weyl-sequence generator with a
xor-shift-multiply finaliser, started at ``seed``.  Couplings of sample s use seed
``j_seed0 + s`` with the three directions concatenated; spins of sample s use ``spin_seed``
at word offset s*W.
"""
from __future__ import annotations

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


def words_per_sample(L: int) -> int:
    """Number of uint32 words of one canonical bit array of an L^3 lattice."""
    n = L * L * L
    return (n + 31) // 32


def random_words(seed: int, count: int, offset: int = 0) -> np.ndarray:
    """``count`` uint32 words: word k is the high half of output number (offset + k + 1)."""
    with np.errstate(over="ignore"):
        k = np.arange(offset + 1, offset + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + k * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(32)).astype(np.uint32)


def _mask_tail(words: np.ndarray, L: int) -> np.ndarray:
    n = L * L * L
    tail = n & 31
    if tail:
        words[..., -1] &= np.uint32((1 << tail) - 1)
    return words


def make_couplings(L: int, nsamples: int = 1, j_seed0: int = 1) -> np.ndarray:
    """Canonical couplings, shape (nsamples, 3, W); sample s is drawn from seed j_seed0 + s."""
    W = words_per_sample(L)
    out = np.empty((nsamples, 3, W), dtype=np.uint32)
    for s in range(nsamples):
        out[s] = random_words(j_seed0 + s, 3 * W).reshape(3, W)
    return _mask_tail(out, L)


def make_spins(L: int, nsamples: int = 1, spin_seed: int = 2, init: str = "random") -> np.ndarray:
    """Canonical spins, shape (nsamples, W). ``init``: 'random' | 'up' (all sigma=+1) | 'down'."""
    W = words_per_sample(L)
    if init == "random":
        out = random_words(spin_seed, nsamples * W).reshape(nsamples, W).copy()
    elif init == "up":
        out = np.full((nsamples, W), 0xFFFFFFFF, dtype=np.uint32)
    elif init == "down":
        out = np.zeros((nsamples, W), dtype=np.uint32)
    else:
        raise ValueError(f"unknown init {init!r}")
    return _mask_tail(out, L)


# The five workloads of BASELINE.json "configs".  rng_mode: 0 = Philox4x32-10,
# 1 = MINSTD per-site streams.  ``dyn_seed`` is the seed given to ising_create (not stated in
# BASELINE.json; 12345 everywhere, recorded in BASELINE.md / DESIGN.md).
CONFIGS = {
    1: dict(L=16, nsamples=1, j_seed0=1, spin_seed=2, init="random", beta=1.0 / 1.1, sweeps=10, rng_mode=0),
    2: dict(L=64, nsamples=32, j_seed0=1, spin_seed=2, init="random", beta=1.0 / 1.1, sweeps=1000, rng_mode=0),
    3: dict(L=256, nsamples=1, j_seed0=1, spin_seed=2, init="random", beta=1.0 / 0.7, sweeps=1000, rng_mode=1),
    4: dict(L=512, nsamples=1, j_seed0=1, spin_seed=2, init="up", beta=1.0 / 1.1, sweeps=100, rng_mode=0),
    5: dict(L=1024, nsamples=1, j_seed0=1, spin_seed=2, init="random", beta=1.0 / 1.1, sweeps=20, rng_mode=0),
}
DYN_SEED = 12345


def make_config(idx: int):
    """(cfg dict, spins, couplings) of BASELINE.json config ``idx`` (1-based)."""
    cfg = dict(CONFIGS[idx])
    spins = make_spins(cfg["L"], cfg["nsamples"], cfg["spin_seed"], cfg["init"])
    J = make_couplings(cfg["L"], cfg["nsamples"], cfg["j_seed0"])
    return cfg, spins, J
