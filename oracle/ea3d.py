"""ctypes front end of the CPU oracle (oracle/ea3d_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from the CUDA path; the conversions between the canonical
bit-packed format (include/ising.h) and the oracle's int8 arrays below are the oracle's own.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

PHILOX, MINSTD, PHILOX_SHARED = 0, 1, 2  # PHILOX_SHARED: one draw per 32-sample word (R18)
PR_LANES, MT_LANES = 3, 4  # shared draw from stored-state generators, one per lane (R19)

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        u32p, u64p, i8p, i64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_int8),
                                 C.POINTER(C.c_int64))
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_splitmix64_output.argtypes = [C.c_uint64, C.c_uint64]
        L.oracle_splitmix64_output.restype = C.c_uint64
        L.oracle_minstd_step.argtypes = [C.c_uint32]
        L.oracle_minstd_step.restype = C.c_uint32
        L.oracle_minstd_seed_state.argtypes = [C.c_uint64, C.c_uint64]
        L.oracle_minstd_seed_state.restype = C.c_uint32
        L.oracle_minstd_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        L.oracle_minstd_draw.restype = C.c_uint32
        L.oracle_philox_draw.argtypes = [C.c_int, C.c_uint64, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint64]
        L.oracle_philox_draw.restype = C.c_uint32
        L.oracle_thresholds.argtypes = [C.c_double, C.c_int, u64p]
        L.oracle_thresholds.restype = C.c_int
        L.oracle_energy.argtypes = [C.c_int, C.c_int, i8p, i8p, i8p, i8p, i64p, i64p]
        L.oracle_energy.restype = None
        L.oracle_overlap.argtypes = [C.c_int, i8p, i8p]
        L.oracle_overlap.restype = C.c_int64
        L.oracle_minstd_init.argtypes = [C.c_int, C.c_int, C.c_uint64, u32p]
        L.oracle_minstd_init.restype = None
        L.oracle_half_sweep.argtypes = [C.c_int, C.c_int, i8p, i8p, i8p, i8p, C.c_uint64, C.c_int, C.c_uint64,
                                        u64p, u32p, i64p, i64p]
        L.oracle_half_sweep.restype = C.c_int
        L.oracle_site_flips.argtypes = [C.c_int, i8p, i8p, i8p, i8p, C.c_int, C.c_uint64, C.c_int, C.c_uint64,
                                        u64p, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), u64p]
        L.oracle_site_flips.restype = C.c_int
        L.oracle_fnv1a64.argtypes = [C.c_void_p, C.c_uint64]
        L.oracle_fnv1a64.restype = C.c_uint64
        L.oracle_pr_next.argtypes = [u32p, u64p]
        L.oracle_pr_next.restype = C.c_uint32
        L.oracle_pr_seed.argtypes = [C.c_uint64, C.c_uint64, u32p]
        L.oracle_pr_seed.restype = None
        L.oracle_mt_seed.argtypes = [C.c_uint32, u32p]
        L.oracle_mt_seed.restype = None
        L.oracle_mt_next.argtypes = [u32p, u64p]
        L.oracle_mt_next.restype = C.c_uint32
        L.oracle_mt_lane_seed.argtypes = [C.c_uint64, C.c_uint64]
        L.oracle_mt_lane_seed.restype = C.c_uint32
        L.oracle_lane_state_words.argtypes = [C.c_int]
        L.oracle_lane_state_words.restype = C.c_int
        L.oracle_lanes_init.argtypes = [C.c_int, C.c_uint64, C.c_int64, u32p, u64p]
        L.oracle_lanes_init.restype = C.c_int
        L.oracle_lanes_draw_table.argtypes = [C.c_int, C.c_int64, u32p, u64p, C.c_int64, C.c_int, u32p]
        L.oracle_lanes_draw_table.restype = C.c_int
        L.oracle_half_sweep_lanes.argtypes = [C.c_int, C.c_int, i8p, i8p, i8p, i8p, C.c_int, C.c_int64, u32p, u64p,
                                              C.c_uint64, u64p, u32p, i64p, i64p]
        L.oracle_half_sweep_lanes.restype = C.c_int
        L.oracle_count_odd.argtypes = [C.c_int, C.c_uint64, C.c_int64, C.c_int64, u64p, u64p]
        L.oracle_count_odd.restype = C.c_int
        L.oracle_set_threads.argtypes = [C.c_int]
        L.oracle_get_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


# ---- thin scalar wrappers ------------------------------------------------------------------

def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(o, C.c_uint32))
    return tuple(int(v) for v in o)


def splitmix64_output(seed, n):
    return int(lib().oracle_splitmix64_output(seed & (2**64 - 1), n))


def minstd_step(r):
    return int(lib().oracle_minstd_step(r))


def minstd_seed_state(seed, q):
    return int(lib().oracle_minstd_seed_state(seed, q))


def minstd_draw(seed, q, n):
    return int(lib().oracle_minstd_draw(seed, q, n))


def philox_draw(L, seed, sample, x, y, z, t):
    return int(lib().oracle_philox_draw(L, seed, sample, x, y, z, t))


def pr_sequence(seed_words, n):
    """n draws of the Parisi-Rapuano generator from the 62 seed words ira[0..61]."""
    ring = np.asarray(seed_words, dtype=np.uint32).copy()
    assert ring.size == 62
    nd = C.c_uint64(0)
    return [int(lib().oracle_pr_next(_p(ring, C.c_uint32), C.byref(nd))) for _ in range(n)]


def pr_seed_words(seed, lane):
    ring = np.zeros(62, dtype=np.uint32)
    lib().oracle_pr_seed(seed, lane, _p(ring, C.c_uint32))
    return ring


def mt_sequence(s, n):
    """n draws of MT19937 seeded by init_genrand(s)."""
    mt = np.zeros(624, dtype=np.uint32)
    lib().oracle_mt_seed(s, _p(mt, C.c_uint32))
    nd = C.c_uint64(0)
    return [int(lib().oracle_mt_next(_p(mt, C.c_uint32), C.byref(nd))) for _ in range(n)]


def mt_state_after_seed(s):
    mt = np.zeros(624, dtype=np.uint32)
    lib().oracle_mt_seed(s, _p(mt, C.c_uint32))
    return mt


def mt_lane_seed(seed, lane):
    return int(lib().oracle_mt_lane_seed(seed, lane))


def count_odd(kind, seed, nlanes, ndraws):
    """(odd[q], sum[q]) of `ndraws` numbers of every lane (Table II)."""
    odd = np.zeros(nlanes, dtype=np.uint64)
    sm = np.zeros(nlanes, dtype=np.uint64)
    rc = lib().oracle_count_odd(kind, seed, nlanes, ndraws, _p(odd, C.c_uint64), _p(sm, C.c_uint64))
    if rc != 0:
        raise ValueError("bad arguments")
    return odd, sm


def thresholds(beta, rng_mode):
    T = np.zeros(3, dtype=np.uint64)
    rc = lib().oracle_thresholds(float(beta), int(rng_mode), _p(T, C.c_uint64))
    if rc != 0:
        raise ValueError("bad beta or rng_mode")
    return tuple(int(v) for v in T)


def fnv1a64(buf) -> int:
    a = np.ascontiguousarray(buf)
    return int(lib().oracle_fnv1a64(a.ctypes.data, a.nbytes))


def set_threads(n: int):
    lib().oracle_set_threads(int(n))


def max_threads() -> int:
    return int(lib().oracle_get_max_threads())


# ---- canonical packed format <-> int8 arrays (the oracle's own conversions) ------------------

def unpack_bits(words: np.ndarray, n: int) -> np.ndarray:
    """uint32 words (little-endian bit order: bit i&31 of word i>>5) -> uint8 array of n bits."""
    w = np.ascontiguousarray(words, dtype="<u4")
    return np.unpackbits(w.view(np.uint8), bitorder="little")[:n]


def pack_bits(bits: np.ndarray) -> np.ndarray:
    n = bits.size
    nw = (n + 31) // 32
    b = np.zeros(nw * 32, dtype=np.uint8)
    b[:n] = bits
    return np.packbits(b, bitorder="little").view("<u4").astype(np.uint32)


def spins_from_packed(words: np.ndarray, n: int) -> np.ndarray:
    """PAPER.md:246-249 Eq. 10: bit 1 <=> sigma = +1, bit 0 <=> sigma = -1."""
    bits = unpack_bits(words, n)
    out = bits.astype(np.int8)
    out *= 2
    out -= 1
    return out


def couplings_from_packed(words: np.ndarray, n: int) -> np.ndarray:
    """PAPER.md:246-249 Eq. 10: bit 1 <=> J = -1, bit 0 <=> J = +1."""
    bits = unpack_bits(words, n)
    out = bits.astype(np.int8)
    out *= -2
    out += 1
    return out


def spins_to_packed(sigma: np.ndarray) -> np.ndarray:
    return pack_bits((sigma > 0).astype(np.uint8))


class Oracle:
    """The reference chain: state in int8 arrays, half-sweep counter t, red (even t) then blue."""

    def __init__(self, L: int, nsamples: int, seed: int, rng_mode: int, nlanes: int | None = None):
        if L < 2 or L % 2:
            raise ValueError("L must be even and >= 2")
        self.nlanes = None
        self.L, self.nsamples, self.seed, self.rng_mode = L, nsamples, int(seed), int(rng_mode)
        self.N = L ** 3
        self.t = 0
        self.sigma = np.ones((nsamples, self.N), dtype=np.int8)
        self.Jx = np.ones((nsamples, self.N), dtype=np.int8)
        self.Jy = np.ones((nsamples, self.N), dtype=np.int8)
        self.Jz = np.ones((nsamples, self.N), dtype=np.int8)
        self.dE_sum = np.zeros(nsamples, dtype=np.int64)
        self.stats = np.zeros(11, dtype=np.int64)
        self.minstd_state = None
        if rng_mode == MINSTD:
            self.minstd_state = np.zeros(nsamples * self.N, dtype=np.uint32)
            lib().oracle_minstd_init(L, nsamples, self.seed, _p(self.minstd_state, C.c_uint32))
        if rng_mode in (PR_LANES, MT_LANES):
            if nlanes is None or nlanes < 1 or nsamples % 32 or self.N % 8:
                raise ValueError("lane modes need nlanes, nsamples = 32k and N a multiple of 8")
            self.nlanes = int(nlanes)
            w = lib().oracle_lane_state_words(rng_mode)
            self.lane_state = np.zeros(self.nlanes * w, dtype=np.uint32)
            self.lane_ndrawn = np.zeros(self.nlanes, dtype=np.uint64)
            self.lane_scratch = np.zeros((nsamples // 32) * (self.N // 2), dtype=np.uint32)
            lib().oracle_lanes_init(rng_mode, self.seed, self.nlanes, _p(self.lane_state, C.c_uint32),
                                    _p(self.lane_ndrawn, C.c_uint64))

    # -- state I/O in the canonical packed format
    def load_packed(self, spins_words: np.ndarray, J_words: np.ndarray):
        sw = np.asarray(spins_words).reshape(self.nsamples, -1)
        jw = np.asarray(J_words).reshape(self.nsamples, 3, -1)
        for s in range(self.nsamples):
            self.sigma[s] = spins_from_packed(sw[s], self.N)
            self.Jx[s] = couplings_from_packed(jw[s, 0], self.N)
            self.Jy[s] = couplings_from_packed(jw[s, 1], self.N)
            self.Jz[s] = couplings_from_packed(jw[s, 2], self.N)

    def load_arrays(self, sigma, Jx, Jy, Jz):
        self.sigma[...] = np.asarray(sigma, dtype=np.int8).reshape(self.nsamples, self.N)
        self.Jx[...] = np.asarray(Jx, dtype=np.int8).reshape(self.nsamples, self.N)
        self.Jy[...] = np.asarray(Jy, dtype=np.int8).reshape(self.nsamples, self.N)
        self.Jz[...] = np.asarray(Jz, dtype=np.int8).reshape(self.nsamples, self.N)

    def spins_packed(self) -> np.ndarray:
        return np.stack([spins_to_packed(self.sigma[s]) for s in range(self.nsamples)])

    # -- dynamics
    def half_sweep(self, beta: float):
        T = np.array(thresholds(beta, self.rng_mode), dtype=np.uint64)
        if self.nlanes is not None:
            rc = lib().oracle_half_sweep_lanes(self.L, self.nsamples, _p(self.sigma, C.c_int8), _p(self.Jx, C.c_int8),
                                               _p(self.Jy, C.c_int8), _p(self.Jz, C.c_int8), self.rng_mode, self.nlanes,
                                               _p(self.lane_state, C.c_uint32), _p(self.lane_ndrawn, C.c_uint64), self.t,
                                               _p(T, C.c_uint64), _p(self.lane_scratch, C.c_uint32),
                                               _p(self.dE_sum, C.c_int64), _p(self.stats, C.c_int64))
            if rc != 0:
                raise RuntimeError("oracle_half_sweep_lanes failed")
            self.t += 1
            return
        ms = _p(self.minstd_state, C.c_uint32) if self.minstd_state is not None else None
        rc = lib().oracle_half_sweep(self.L, self.nsamples, _p(self.sigma, C.c_int8), _p(self.Jx, C.c_int8),
                                     _p(self.Jy, C.c_int8), _p(self.Jz, C.c_int8), self.seed, self.rng_mode,
                                     self.t, _p(T, C.c_uint64), ms, _p(self.dE_sum, C.c_int64),
                                     _p(self.stats, C.c_int64))
        if rc != 0:
            raise RuntimeError("oracle_half_sweep failed")
        self.t += 1

    def sweep(self, beta: float, nsweeps: int = 1):
        for _ in range(2 * nsweeps):
            self.half_sweep(beta)

    def energy(self):
        E = np.zeros(self.nsamples, dtype=np.int64)
        M = np.zeros(self.nsamples, dtype=np.int64)
        lib().oracle_energy(self.L, self.nsamples, _p(self.sigma, C.c_int8), _p(self.Jx, C.c_int8),
                            _p(self.Jy, C.c_int8), _p(self.Jz, C.c_int8), _p(E, C.c_int64), _p(M, C.c_int64))
        return E, M

    def overlap(self, a: int, b: int) -> int:
        """q_ab = sum_i sigma_i^a sigma_i^b (replicas)."""
        return int(lib().oracle_overlap(self.L, _p(self.sigma[a], C.c_int8), _p(self.sigma[b], C.c_int8)))

    def site_flips(self, beta: float, sample: int, x: int, y: int, z: int, t: int | None = None):
        """(flips, dE, R) for one site of the active colour of half-sweep t, from the CURRENT state."""
        T = np.array(thresholds(beta, self.rng_mode), dtype=np.uint64)
        dE = C.c_int(0)
        R = C.c_uint64(0)
        tt = self.t if t is None else t
        rc = lib().oracle_site_flips(self.L, _p(self.sigma[sample], C.c_int8), _p(self.Jx[sample], C.c_int8),
                                     _p(self.Jy[sample], C.c_int8), _p(self.Jz[sample], C.c_int8), sample,
                                     self.seed, self.rng_mode, tt, _p(T, C.c_uint64), x, y, z, C.byref(dE),
                                     C.byref(R))
        return rc, dE.value, R.value
