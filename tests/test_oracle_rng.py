"""Pins of the oracle's random number generators, thresholds and checksum (CPU only).

Each test compares oracle/ with something the oracle did not produce: a published known-answer vector
(tests/golden/), a third-party implementation (cuRAND's header, libstdc++'s std::minstd_rand0), exact decimal
arithmetic, an algebraic inverse written here, or the independent pure-Python implementation.
"""
import ctypes as C
import os
import zlib

import numpy as np
import pytest

from oracle import ea3d, ea3d_py
from tests.pins import build_pins

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


# ---------------------------------------------------------------- Philox4x32-10 (R10)

def test_philox_known_answers():
    for row in _rows("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row]
        assert ea3d.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])
        assert ea3d_py.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_philox_against_curand_header():
    lib_path = build_pins.build_curand_philox()
    if lib_path is None:
        pytest.skip("nvcc not installed")
    lib = C.CDLL(lib_path)
    u32p = C.POINTER(C.c_uint32)
    lib.pin_curand_philox4x32_10.argtypes = [u32p, u32p, u32p]
    rng = np.random.default_rng(7)
    cases = rng.integers(0, 2**32, size=(2000, 6), dtype=np.uint64).astype(np.uint32)
    # plus structured counters like the ones the sweep uses: (t, 0, g, 0), key (seed, sample)
    structured = np.array([[t, 0, g, 0, 12345, s] for t in (0, 1, 39) for g in (0, 1, 2**27 - 1) for s in (0, 31)],
                          dtype=np.uint32)
    for row in np.concatenate([cases, structured]):
        c, k, o = row[:4].copy(), row[4:6].copy(), np.zeros(4, np.uint32)
        lib.pin_curand_philox4x32_10(c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), o.ctypes.data_as(u32p))
        assert ea3d.philox4x32_10(c, k) == tuple(int(v) for v in o)


def _philox_round_inverse(c, k):
    """Inverse of one Philox round (written here, not in the oracle): the multipliers are odd, hence invertible
    mod 2^32; (n0,n1,n2,n3) = (hi1^c1^k0, lo1, hi0^c3^k1, lo0)."""
    M0, M1, m = 0xD2511F53, 0xCD9E8D57, 0xFFFFFFFF
    n0, n1, n2, n3 = c
    c0 = (n3 * pow(M0, -1, 2**32)) & m
    c2 = (n1 * pow(M1, -1, 2**32)) & m
    hi0, hi1 = (M0 * c0) >> 32, (M1 * c2) >> 32
    return (c0, n0 ^ hi1 ^ k[0], c2, n2 ^ hi0 ^ k[1])


def test_philox_is_a_bijection_round_trip():
    rng = np.random.default_rng(11)
    for _ in range(200):
        ctr = tuple(int(v) for v in rng.integers(0, 2**32, 4))
        key = tuple(int(v) for v in rng.integers(0, 2**32, 2))
        out = ea3d.philox4x32_10(ctr, key)
        c = out
        for r in reversed(range(10)):
            kr = ((key[0] + r * 0x9E3779B9) & 0xFFFFFFFF, (key[1] + r * 0xBB67AE85) & 0xFFFFFFFF)
            c = _philox_round_inverse(c, kr)
        assert c == ctr


def test_philox_draw_keying():
    """DESIGN.md R9: key (lo32 seed, hi32 seed ^ sample); counter (lo t, hi t, lo g, hi g); g = j>>2; word j&3."""
    L, seed = 8, (0xABCDEF01 << 32) | 0x12345678
    for (s, x, y, z, t) in [(0, 0, 0, 0, 0), (3, 5, 2, 7, 9), (31, 7, 7, 7, 2**33 + 1), (1, 2, 3, 4, 1)]:
        j = (x >> 1) + (L // 2) * (y + L * z)
        key = (seed & 0xFFFFFFFF, (seed >> 32) ^ s)
        ctr = (t & 0xFFFFFFFF, t >> 32, (j >> 2) & 0xFFFFFFFF, (j >> 2) >> 32)
        want = ea3d.philox4x32_10(ctr, key)[j & 3]
        assert ea3d.philox_draw(L, seed, s, x, y, z, t) == want


def test_philox_equidistribution_smoke():
    out = np.array([ea3d.philox4x32_10((n, 0, 0, 0), (1, 2)) for n in range(4000)], dtype=np.uint64).ravel()
    assert abs(out.mean() / 2**32 - 0.5) < 0.01
    bits = ((out[:, None] >> np.arange(32, dtype=np.uint64)) & 1).mean(axis=0)
    assert np.all(np.abs(bits - 0.5) < 0.02)


# ---------------------------------------------------------------- SplitMix64 (R11)

def test_splitmix64_published_sequence():
    want = [int(r[0]) for r in _rows("splitmix64_seed1234567.txt")]
    assert [ea3d.splitmix64_output(1234567, n) for n in range(1, 6)] == want
    assert [ea3d_py.splitmix64_output(1234567, n) for n in range(1, 6)] == want


def test_splitmix64_finaliser_inverse_round_trip():
    rng = np.random.default_rng(5)
    for seed, n in zip(rng.integers(0, 2**63, 100), rng.integers(1, 2**40, 100)):
        z = ea3d.splitmix64_output(int(seed), int(n))
        assert ea3d_py.splitmix64_unmix(z) == (int(seed) + int(n) * 0x9E3779B97F4A7C15) % 2**64


def test_minstd_seed_state_is_legal_and_matches_python():
    for q in list(range(64)) + [2**30 - 1, 2**35 + 17]:
        s0 = ea3d.minstd_seed_state(12345, q)
        assert 1 <= s0 <= 2**30
        assert s0 == ea3d_py.minstd_seed_state(12345, q)
        assert s0 == (ea3d.splitmix64_output(12345, q + 1) >> 34) + 1


# ---------------------------------------------------------------- MINSTD (Eq. 7)

def _minstd_lib():
    lib = C.CDLL(build_pins.build_minstd())
    lib.pin_minstd_rand0_sequence.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32)]
    lib.pin_minstd_rand0_discard.argtypes = [C.c_uint32, C.c_uint64]
    lib.pin_minstd_rand0_discard.restype = C.c_uint32
    return lib


def test_minstd_park_miller_check_value():
    want = int(_rows("minstd_park_miller.txt")[0][0])
    r = 1
    for _ in range(10000):
        r = ea3d.minstd_step(r)
    assert r == want
    assert ea3d_py.minstd_draw.__doc__  # stateless form: 16807^10000 mod M
    assert pow(16807, 10000, 2**31 - 1) == want


def test_minstd_against_std_minstd_rand0():
    lib = _minstd_lib()
    for s0 in (1, 2, 16807, 2**30, 2**31 - 2, 123456789):
        buf = np.zeros(500, np.uint32)
        lib.pin_minstd_rand0_sequence(s0, 500, buf.ctypes.data_as(C.POINTER(C.c_uint32)))
        r, seq = s0, []
        for _ in range(500):
            r = ea3d.minstd_step(r)
            seq.append(r)
        assert seq == [int(v) for v in buf]


def test_minstd_draw_is_nth_state_of_the_site_stream():
    """DESIGN.md R12: draw of sweep n = (n+1)-th value after the seed state; the stateless (jump-ahead) form of the
    Python implementation and libstdc++'s discard() must agree with the oracle's plain iteration."""
    lib = _minstd_lib()
    for q in (0, 1, 77, 2**24 + 5):
        s0 = ea3d.minstd_seed_state(99, q)
        for n in (0, 1, 2, 10, 999):
            d = ea3d.minstd_draw(99, q, n)
            assert d == ea3d_py.minstd_draw(99, q, n)
            assert d == lib.pin_minstd_rand0_discard(s0, n)
            assert 1 <= d <= 2**31 - 2


# ---------------------------------------------------------------- thresholds (R5/R6)

def test_thresholds_against_exact_decimal_arithmetic():
    for mode, num, den, t4, t8, t12 in _rows("thresholds.txt"):
        beta = float(num) / float(den)
        got = ea3d.thresholds(beta, int(mode))
        assert got == (int(t4), int(t8), int(t12)), (mode, num, den)
        assert ea3d_py.thresholds(beta, int(mode)) == got


def test_thresholds_are_nested_and_reject_bad_beta():
    for beta in (0.0, 0.05, 0.5, 1 / 1.1, 1 / 0.7, 3.0, 1e3, float("inf")):
        for mode in (0, 1):
            t4, t8, t12 = ea3d.thresholds(beta, mode)
            assert t12 <= t8 <= t4 <= (2**32 if mode == 0 else 2**31 - 1)
    assert ea3d.thresholds(float("inf"), 0) == (0, 0, 0)
    for bad in (-0.1, float("nan")):
        with pytest.raises(ValueError):
            ea3d.thresholds(bad, 0)
    with pytest.raises(ValueError):
        ea3d.thresholds(1.0, 7)


# ---------------------------------------------------------------- FNV-1a 64 (config 4 checksum)

def _fnv1a64_py(data: bytes) -> int:
    h = 0xCBF29CE484222325
    for b in data:
        h = ((h ^ b) * 0x100000001B3) % 2**64
    return h


def test_fnv1a64():
    assert ea3d.fnv1a64(np.zeros(0, np.uint8)) == 0xCBF29CE484222325          # empty input -> offset basis
    assert ea3d.fnv1a64(np.frombuffer(b"a", np.uint8)) == 0xAF63DC4C8601EC8C  # published FNV-1a test vector
    assert ea3d.fnv1a64(np.frombuffer(b"foobar", np.uint8)) == 0x85944171F73967E8
    rng = np.random.default_rng(3)
    w = rng.integers(0, 2**32, 257, dtype=np.uint64).astype(np.uint32)
    assert ea3d.fnv1a64(w) == _fnv1a64_py(w.astype("<u4").tobytes())
    assert zlib.crc32(w.tobytes()) != ea3d.fnv1a64(w)  # (sanity: not accidentally another checksum)
