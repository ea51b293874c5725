"""Pins of the oracle's stored-state lane generators and of the lane-driven shared-draw sweep (rng_mode 3 = Parisi-Rapuano,
4 = MT19937; R19).  CPU only.

  MT19937          the ISO C++ check value (tests/golden/mt19937_std_check.txt), libstdc++'s std::mt19937 and numpy's legacy
                   RandomState (both third-party implementations, both seeded by init_genrand)
  Parisi-Rapuano   the paper's two lines restated here on an unbounded history list (no ring, no modulo)
  lane order       the draw table rebuilt here from per-lane sequences with the order of R19 written out
  sweep            every sample follows the scalar rule of the pinned independent oracle when that oracle is fed the same
                   numbers; beta = 0 and beta = inf special cases; incremental energy
"""
import ctypes as C
import os

import numpy as np
import pytest

from oracle import ea3d, ea3d_py
from paper_1411_0127_b200 import synth
from tests.pins import build_pins

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M32 = 0xFFFFFFFF


# ---------------------------------------------------------------- MT19937

def test_mt19937_iso_cpp_check_value():
    with open(os.path.join(GOLD, "mt19937_std_check.txt")) as f:
        seed, n, want = [int(v) for v in [l for l in f if l.strip() and not l.startswith("#")][0].split()]
    assert ea3d.mt_sequence(seed, n)[-1] == want


def test_mt19937_against_std_mt19937_and_numpy():
    lib = C.CDLL(build_pins.build_mt19937())
    lib.pin_mt19937_sequence.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(C.c_uint32)]
    for s in (0, 1, 5489, 19650218, 0xFFFFFFFF, 123456789):
        n = 2000  # crosses three regenerations of the 624-word block
        buf = np.zeros(n, np.uint32)
        lib.pin_mt19937_sequence(s, n, buf.ctypes.data_as(C.POINTER(C.c_uint32)))
        got = ea3d.mt_sequence(s, n)
        assert got == [int(v) for v in buf]
        rs = np.random.RandomState(s)
        assert np.array_equal(ea3d.mt_state_after_seed(s), rs.get_state()[1])  # init_genrand itself
        assert got == [int(v) for v in rs._bit_generator.random_raw(n)]


# ---------------------------------------------------------------- Parisi-Rapuano

def _pr_history(seed_words, n):
    """ira[i] = ira[i-24] + ira[i-55]; R = ira[i] ^ ira[i-61], on an ever-growing list."""
    ira = [int(v) for v in seed_words]
    out = []
    for _ in range(n):
        i = len(ira)
        ira.append((ira[i - 24] + ira[i - 55]) & M32)
        out.append(ira[i] ^ ira[i - 61])
    return out


def test_parisi_rapuano_against_the_unbounded_history_form():
    rng = np.random.RandomState(3)
    for _ in range(3):
        seed_words = rng.randint(0, 2**32, size=62, dtype=np.uint64).astype(np.uint32)
        assert ea3d.pr_sequence(seed_words, 1000) == _pr_history(seed_words, 1000)


def test_parisi_rapuano_lags_are_24_55_61():
    """A single set bit in seed word r shows up in the first draws exactly where the lags say: draw n reads the words
    62+n-24, 62+n-55, 62+n-61, i.e. seed word r is read by draws n = r-38 (lag 24), r-7 (lag 55) and r-1 (lag 61)."""
    for r in (1, 7, 38, 45, 61):
        w = np.zeros(62, np.uint32)
        w[r] = 1
        seq = ea3d.pr_sequence(w, 24)  # before any generated word feeds back (lag 24)
        hit = {n for n, v in enumerate(seq) if v}
        want = {n for n in (r - 38, r - 7, r - 1) if 0 <= n < 24}
        assert hit == want, (r, hit, want)


def test_lane_seeds_are_splitmix_words():
    for q in (0, 1, 5, 1000):
        ring = ea3d.pr_seed_words(99, q)
        assert [int(v) for v in ring] == [ea3d_py.splitmix64_output(99, q * 62 + r + 1) >> 32 for r in range(62)]
        assert ea3d.mt_lane_seed(99, q) == ea3d_py.splitmix64_output(99, q + 1) >> 32


# ---------------------------------------------------------------- lane order of a half-sweep (R19)

def _lane_sequences(mode, seed, nlanes, n):
    if mode == ea3d.PR_LANES:
        return [ea3d.pr_sequence(ea3d.pr_seed_words(seed, q), n) for q in range(nlanes)]
    return [ea3d.mt_sequence(ea3d.mt_lane_seed(seed, q), n) for q in range(nlanes)]


@pytest.mark.parametrize("mode", [ea3d.PR_LANES, ea3d.MT_LANES])
@pytest.mark.parametrize("ngroups,nlanes,k", [(8, 8, 1), (8, 3, 1), (27, 5, 2), (64, 24, 3), (8, 16, 2), (8, 13, 5)])
def test_draw_table_follows_the_lane_order(mode, ngroups, nlanes, k):
    lib = ea3d.lib()
    w = lib.oracle_lane_state_words(mode)
    state = np.zeros(nlanes * w, np.uint32)
    nd = np.zeros(nlanes, np.uint64)
    u32, u64 = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    lib.oracle_lanes_init(mode, 4242, nlanes, state.ctypes.data_as(u32), nd.ctypes.data_as(u64))
    rounds = -(-(k * ngroups) // nlanes)
    per_hs = 4 * rounds
    seqs = _lane_sequences(mode, 4242, nlanes, 3 * per_hs)
    for hs in range(3):
        table = np.zeros(k * 4 * ngroups, np.uint32)
        assert lib.oracle_lanes_draw_table(mode, nlanes, state.ctypes.data_as(u32), nd.ctypes.data_as(u64), ngroups, k,
                                           table.ctypes.data_as(u32)) == 0
        assert all(int(v) == (hs + 1) * per_hs for v in nd)          # every lane advances by the same amount
        for b in range(k):
            for j in range(4 * ngroups):
                g, wd = j >> 2, j & 3
                u = b * ngroups + g                      # unit = (batch, group), batch-major
                q, m = u % nlanes, u // nlanes
                assert int(table[b * 4 * ngroups + j]) == seqs[q][hs * per_hs + m * 4 + wd], (hs, b, j)


# ---------------------------------------------------------------- the sweep

def _packed(L, ns, a=5, b=6):
    return synth.make_spins(L, ns, a), synth.make_couplings(L, ns, b)


@pytest.mark.parametrize("mode", [ea3d.PR_LANES, ea3d.MT_LANES])
def test_every_sample_follows_the_scalar_rule_with_the_lane_draws(mode):
    """Second implementation of the sweep (oracle/ea3d_py.py's scalar rule on Python integers) fed with the lane draws
    rebuilt from per-lane sequences."""
    L, ns, nlanes, seed, beta, nhs = 4, 64, 3, 31, 0.55, 4
    spins, J = _packed(L, ns)
    o = ea3d.Oracle(L, ns, seed, mode, nlanes=nlanes)
    o.load_packed(spins, J)
    for _ in range(nhs):
        o.half_sweep(beta)
    got = o.spins_packed()
    N, ngroups, k = L**3, L**3 // 8, ns // 32
    per_hs = 4 * -(-(k * ngroups) // nlanes)
    seqs = _lane_sequences(mode, seed, nlanes, nhs * per_hs)
    T = ea3d.thresholds(beta, mode)
    W = (N + 31) // 32
    for s in (0, 13, 31, 32, 63):
        b = s >> 5
        sg = [int(v) for v in ea3d.spins_from_packed(spins.reshape(ns, W)[s], N)]
        Jw = J.reshape(ns, 3, W)[s]
        Jd = [[int(v) for v in ea3d.couplings_from_packed(Jw[d], N)] for d in range(3)]
        for t in range(nhs):
            for z in range(L):
                for y in range(L):
                    for x in range(L):
                        if (x + y + z) & 1 != t & 1:
                            continue
                        i = x + L * (y + L * z)
                        def at(xx, yy, zz):
                            return (xx % L) + L * ((yy % L) + L * (zz % L))
                        h = (Jd[0][i] * sg[at(x + 1, y, z)] + Jd[0][at(x - 1, y, z)] * sg[at(x - 1, y, z)]
                             + Jd[1][i] * sg[at(x, y + 1, z)] + Jd[1][at(x, y - 1, z)] * sg[at(x, y - 1, z)]
                             + Jd[2][i] * sg[at(x, y, z + 1)] + Jd[2][at(x, y, z - 1)] * sg[at(x, y, z - 1)])
                        dE = 2 * sg[i] * h
                        j = (x >> 1) + (L // 2) * (y + L * z)
                        g, wd = j >> 2, j & 3
                        u = b * ngroups + g
                        R = seqs[u % nlanes][t * per_hs + (u // nlanes) * 4 + wd]
                        if dE <= 0 or R < T[dE // 4 - 1]:
                            sg[i] = -sg[i]
        want = ea3d.spins_to_packed(np.array(sg, dtype=np.int8))
        assert np.array_equal(want, got[s]), s


@pytest.mark.parametrize("mode", [ea3d.PR_LANES, ea3d.MT_LANES])
def test_lane_modes_special_temperatures_and_energy_bookkeeping(mode):
    L, ns = 4, 32
    spins, J = _packed(L, ns, 7, 8)
    # beta = 0: every proposal accepted, a full sweep inverts every spin
    o = ea3d.Oracle(L, ns, 1, mode, nlanes=5)
    o.load_packed(spins, J)
    before = o.sigma.copy()
    o.sweep(0.0, 1)
    assert np.array_equal(o.sigma, -before)
    # beta = inf: energy never increases; incremental dE bookkeeping equals the recomputed energy
    o = ea3d.Oracle(L, ns, 1, mode, nlanes=5)
    o.load_packed(spins, J)
    E0, _ = o.energy()
    prev = E0.copy()
    for _ in range(6):
        o.half_sweep(float("inf"))
        E, _ = o.energy()
        assert np.all(E <= prev)
        assert np.array_equal(E, E0 + o.dE_sum)
        prev = E
    assert o.stats[2] == 0 and o.stats[3] == 0
    # finite beta: bookkeeping again, and equal samples of a batch stay equal
    W = (L**3 + 31) // 32
    sp1 = np.tile(spins.reshape(ns, W)[:1], (ns, 1))
    J1 = np.tile(J.reshape(ns, 3, W)[:1], (ns, 1, 1))
    o = ea3d.Oracle(L, ns, 1, mode, nlanes=8)
    o.load_packed(sp1, J1)
    E0, _ = o.energy()
    o.sweep(0.4, 3)
    E, _ = o.energy()
    assert np.array_equal(E, E0 + o.dE_sum)
    a = o.spins_packed()
    assert all(np.array_equal(a[0], a[s]) for s in range(ns))
    assert not np.array_equal(a[0], sp1[0])


def test_lane_mode_thresholds_are_the_philox_ones():
    for beta in (0.0, 0.3, 1 / 1.1, float("inf")):
        assert ea3d.thresholds(beta, ea3d.PR_LANES) == ea3d.thresholds(beta, ea3d.PHILOX)
        assert ea3d.thresholds(beta, ea3d.MT_LANES) == ea3d.thresholds(beta, ea3d.PHILOX)


# ---------------------------------------------------------------- Table II: counting odd numbers

@pytest.mark.parametrize("kind", [ea3d.PHILOX, ea3d.MINSTD, ea3d.PR_LANES, ea3d.MT_LANES])
def test_count_odd_against_per_lane_sequences(kind):
    nl, nd, seed = 7, 700, 2024
    odd, sm = ea3d.count_odd(kind, seed, nl, nd)
    for q in range(nl):
        if kind == ea3d.PR_LANES:
            seq = ea3d.pr_sequence(ea3d.pr_seed_words(seed, q), nd)
        elif kind == ea3d.MT_LANES:
            seq = ea3d.mt_sequence(ea3d.mt_lane_seed(seed, q), nd)
        elif kind == ea3d.MINSTD:
            seq = [ea3d_py.minstd_draw(seed, q, n) for n in range(nd)]
        else:
            seq = []
            for n in range(nd):
                c = n >> 2
                seq.append(ea3d_py.philox4x32_10([c & M32, c >> 32, q, 0], [seed & M32, seed >> 32])[n & 3])
        assert int(odd[q]) == sum(v & 1 for v in seq)
        assert int(sm[q]) == sum(seq) % 2**64
    # roughly half of the numbers are odd
    assert abs(float(odd.sum()) / (nl * nd) - 0.5) < 0.03
