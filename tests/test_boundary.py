"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds, loads and exports every symbol that
include/ising.h declares; its host-only entry points (thresholds, FNV-1a, argument validation) agree with the
oracle; and the word update of the word-parallel kernels -- run on the host through the test hook
ising_hostcheck_update_word, i.e. the same __host__ __device__ code as the kernels (folded Philox, stateless MINSTD,
Eq. 11-13 adder, per-bit acceptance, reconstructed Eq. 17) -- reproduces the oracle's scalar rule site by site.
No compute call needs a GPU here.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import ea3d
from paper_1411_0127_b200 import binding, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "ising.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(ising_[a-z0-9_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    lib = binding.lib()
    for name in declared:
        assert hasattr(lib, name), name


@pytest.mark.parametrize("rng_mode", [0, 1])
def test_thresholds_equal_the_oracle_table(rng_mode):
    betas = [0.0, 1e-9, 0.05, 0.1732, 0.3, 1 / 1.1, 1.0, 1 / 0.7, 2.5, 7.0, 30.0, 1e3, float("inf")]
    for beta in betas:
        assert binding.ising_thresholds(beta, rng_mode) == ea3d.thresholds(beta, rng_mode), beta
    # the values DESIGN.md quotes
    assert binding.ising_thresholds(1 / 1.1, 0) == (113163715, 2981635, 78560)
    assert binding.ising_thresholds(1 / 0.7, 1) == (7083487, 23364, 77)
    assert binding.ising_thresholds(0.0, 0) == (2**32, 2**32, 2**32)
    for bad in (-1.0, float("nan")):
        with pytest.raises(binding.IsingError):
            binding.ising_thresholds(bad, rng_mode)


def test_lane_modes_host_side():
    """rng modes 3, 4 (R19): thresholds are the Philox table; the workspace grows by the strided generator state
    (62 / 624 words per lane; min(k N/8, 148*1024) lanes: one wave of threads);
    nsamples % 32 is required."""
    lib = binding.lib()
    out = C.c_size_t(0)
    for mode, ring, cap in ((binding.PR_SHARED, 62, 148 * 1024), (binding.MT19937_SHARED, 624, 148 * 1024)):
        for beta in (0.0, 0.4, 1 / 1.1, float("inf")):
            assert binding.ising_thresholds(beta, mode) == ea3d.thresholds(beta, mode) == ea3d.thresholds(beta, 0)
        assert lib.ising_workspace_bytes(16, 1, mode, C.byref(out)) == binding.EINVAL
        assert lib.ising_workspace_bytes(12, 32, mode, C.byref(out)) == binding.OK      # any even L
        for L, ns in ((8, 32), (64, 64), (256, 32)):
            lanes = min((ns // 32) * L**3 // 8, cap)
            extra = binding.ising_workspace_bytes(L, ns, mode) - binding.ising_workspace_bytes(L, ns, binding.PHILOX_SHARED)
            assert 0 <= extra - 4 * ring * lanes < 256
        assert binding.ising_prng_state_bytes(mode, 1000) == 4 * ring * 1000
    assert binding.ising_prng_state_bytes(binding.PHILOX, 5) == 0 and binding.ising_prng_state_bytes(binding.MINSTD, 5) == 20
    assert lib.ising_prng_state_bytes(binding.PHILOX_SHARED, 5, C.byref(out)) == binding.EINVAL
    assert lib.ising_prng_state_bytes(0, 0, C.byref(out)) == binding.EINVAL


def test_fnv1a64_host():
    rng = np.random.default_rng(5)
    for n in (0, 1, 7, 4096):
        buf = rng.integers(0, 256, n, dtype=np.uint8)
        assert binding.ising_fnv1a64_host(buf) == ea3d.fnv1a64(buf)
    assert binding.ising_fnv1a64_host(np.zeros(0, dtype=np.uint8)) == 0xCBF29CE484222325
    assert binding.ising_fnv1a64_host(np.frombuffer(b"foobar", dtype=np.uint8)) == 0x85944171F73967E8


def test_argument_validation_without_a_gpu():
    lib = binding.lib()
    out = C.c_size_t(0)
    for L, ns in ((3, 1), (2, 1), (0, 1), (-4, 1), (8192, 1), (4098, 1), (2050, 1), (2112, 1), (4096, 32), (16, 2), (16, 0), (16, 48)):
        assert lib.ising_workspace_bytes(L, ns, 0, C.byref(out)) == binding.EINVAL, (L, ns)
    assert lib.ising_workspace_bytes(16, 1, 7, C.byref(out)) == binding.EINVAL
    assert lib.ising_workspace_bytes(16, 1, 2, C.byref(out)) == binding.EINVAL   # shared draws need 32-sample words
    assert lib.ising_workspace_bytes(16, 32, 2, C.byref(out)) == binding.OK
    assert lib.ising_workspace_bytes(16, 1, 0, None) == binding.EINVAL
    # sizes: 8 internal bit arrays + canonical staging + accumulators
    for L, ns in ((16, 1), (64, 32), (256, 1), (1024, 1), (6, 1), (4, 64), (192, 1), (768, 1), (448, 1), (576, 1)):
        nbytes = binding.ising_workspace_bytes(L, ns, 0)
        N = L**3
        assert nbytes >= ns * (N // 8) * 8 and nbytes % 256 == 0
        # MINSTD adds the seed-state table (4 bytes per site) where the word-parallel layout applies
        # (word-parallel layout: L a multiple of 64; rows whose lane count is not a power of two are padded)
        # (many samples with L a multiple of 64 are stored as a batch of such lattices: one table per sample)
        table = 0
        if L % 64 == 0:
            wpr = odd = L // 64
            while odd % 2 == 0:
                odd //= 2
            W = odd if odd in (3, 5) else (4 if odd == 1 and wpr >= 8 else 1)  # words per thread
            if ns > 1 and odd == 1 and wpr >= 2:
                W = 4 if wpr >= 4 else 2
            pad = 1
            while pad < wpr // W:
                pad *= 2
            table = 4 * 2 * L * L * pad * W * 32 * ns
            assert table >= 4 * N * ns and (table == 4 * N * ns) == (odd in (1, 3, 5))
        assert binding.ising_workspace_bytes(L, ns, 1) == nbytes + table
    assert binding.ising_workspace_bytes(1024, 1, 0) < 1100 * 2**20
    # beyond 2^32 Philox groups (L > 2048): one sample, rows of 1, 3, 5 x 2^e words; no MINSTD seed table there
    for L in (2560, 3072, 4096):
        nbytes = binding.ising_workspace_bytes(L, 1, 0)
        assert 8 * L**3 // 8 <= nbytes < 8 * L**3 // 8 + 2**20 and binding.ising_workspace_bytes(L, 1, 1) == nbytes
    h = C.c_void_p()
    assert lib.ising_create(16, 1, 1, 0, None, 1 << 20, C.byref(h)) == binding.EINVAL
    assert lib.ising_create(16, 1, 1, 0, C.c_void_p(256), 16, C.byref(h)) == binding.EINVAL      # too small
    assert lib.ising_create(16, 1, 1, 0, C.c_void_p(260), 1 << 20, C.byref(h)) == binding.EINVAL  # misaligned
    assert lib.ising_sweep(None, 1.0, 1, None) == binding.EINVAL
    assert lib.ising_strerror(binding.ECUDA) == b"CUDA error"
    # a handle on a fake (never dereferenced on the host) workspace: host-side checks only
    assert lib.ising_create(16, 1, 1, 0, C.c_void_p(1 << 20), 1 << 20, C.byref(h)) == binding.OK
    assert lib.ising_sweep(h, -1.0, 1, None) == binding.EINVAL
    assert lib.ising_sweep(h, float("nan"), 1, None) == binding.EINVAL
    assert lib.ising_sweep(h, 1.0, -1, None) == binding.EINVAL
    assert lib.ising_sweep(h, 1.0, 0, None) == binding.OK  # nothing to launch
    assert lib.ising_load_state(h, None, None, None) == binding.EINVAL
    t = C.c_uint64(99)
    assert lib.ising_get_t(h, C.byref(t)) == binding.OK and t.value == 0
    assert lib.ising_set_t(h, 6) == binding.OK and lib.ising_get_t(h, C.byref(t)) == binding.OK and t.value == 6
    assert lib.ising_set_kernel(h, 5) == binding.OK and lib.ising_set_kernel(h, 6) == binding.EINVAL
    # layouts (ising_create_layout): a batch of site-packed lattices only for many samples with their own draws and whole-word rows
    h2 = C.c_void_p()
    big = C.c_void_p(1 << 20)
    assert lib.ising_create_layout(64, 32, 1, 0, binding.LAYOUT_BATCH, big, 1 << 30, C.byref(h2)) == binding.OK
    assert lib.ising_destroy(h2) == binding.OK
    assert lib.ising_create_layout(64, 32, 1, 1, binding.LAYOUT_SAMPLE_PACKED, big, 1 << 30, C.byref(h2)) == binding.OK
    assert lib.ising_destroy(h2) == binding.OK
    for L, ns, mode, layout in ((64, 32, 2, binding.LAYOUT_BATCH), (32, 32, 0, binding.LAYOUT_BATCH), (64, 1, 0, binding.LAYOUT_BATCH),
                                (64, 1, 0, binding.LAYOUT_SAMPLE_PACKED), (64, 32, 0, 3), (64, 32, 0, -1)):
        assert lib.ising_create_layout(L, ns, 1, mode, layout, big, 1 << 30, C.byref(h2)) == binding.EINVAL, (L, ns, mode, layout)
    assert lib.ising_kernel_launches(h) == 0
    assert lib.ising_destroy(h) == binding.OK


def test_no_cpu_fallback_device_calls_fail_loudly_without_a_gpu():
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    lib = binding.lib()
    h = C.c_void_p()
    assert lib.ising_create(16, 1, 1, 0, C.c_void_p(1 << 20), 1 << 20, C.byref(h)) == binding.OK
    assert lib.ising_sweep(h, 1.0, 1, None) == binding.ECUDA
    lib.ising_destroy(h)


# ---------------------------------------------------------------------------------------------------------------
# word update on the host vs the oracle's scalar rule
# ---------------------------------------------------------------------------------------------------------------

def _operand_words(o: ea3d.Oracle, colour: int, k: int, y: int, z: int):
    """The 13 operand words of the active word k of half-row (y,z), built site by site from the oracle's int8 arrays
    (bit conventions of Eq. 10): s, six neighbour spins (+x,-x,+y,-y,+z,-z), six couplings (same order)."""
    L = o.L
    sg, Jx, Jy, Jz = (a[0].reshape(L, L, L) for a in (o.sigma, o.Jx, o.Jy, o.Jz))  # [z][y][x]
    xodd = (y + z + colour) & 1
    ops = [0] * 13
    sites = []
    for b in range(32):
        x = 2 * (32 * k + b) + xodd
        xp, xm, yp, ym, zp, zm = (x + 1) % L, (x - 1) % L, (y + 1) % L, (y - 1) % L, (z + 1) % L, (z - 1) % L
        nb = [sg[z, y, xp], sg[z, y, xm], sg[z, yp, x], sg[z, ym, x], sg[zp, y, x], sg[zm, y, x]]
        J = [Jx[z, y, x], Jx[z, y, xm], Jy[z, y, x], Jy[z, ym, x], Jz[z, y, x], Jz[zm, y, x]]
        ops[0] |= int(sg[z, y, x] > 0) << b
        for d in range(6):
            ops[1 + d] |= int(nb[d] > 0) << b
            ops[7 + d] |= int(J[d] < 0) << b
        sites.append((x, y, z))
    return ops, sites, xodd


@pytest.mark.parametrize("rng_mode", [0, 1])
@pytest.mark.parametrize("beta", [1 / 1.1, 0.25, 0.0, float("inf")])
def test_host_word_update_equals_oracle_site_rule(rng_mode, beta):
    L, seed = 64, 12345
    o = ea3d.Oracle(L, 1, seed, rng_mode)
    o.load_packed(synth.make_spins(L, 1, 2), synth.make_couplings(L, 1, 1))
    rng = np.random.default_rng(17 + rng_mode)
    wpr = L // 64
    nflip = 0
    for trial in range(40):
        t = int(rng.integers(0, 50))
        if trial == 0 and rng_mode == 0:
            t = 2**33 + 5  # exercises the high counter word (the oracle's MINSTD draw iterates t/2 times: keep t small there)
        colour = t & 1
        k, y, z = int(rng.integers(0, wpr)), int(rng.integers(0, L)), int(rng.integers(0, L))
        ops, sites, xodd = _operand_words(o, colour, k, y, z)
        word_index = k + wpr * (y + L * z)
        site0 = L * (y + L * z) + xodd + 64 * k
        got = binding.ising_hostcheck_update_word(rng_mode, seed, t, beta, ops, word_index, site0, 2)
        want = 0
        for b, (x, yy, zz) in enumerate(sites):
            flips, dE, R = o.site_flips(beta, 0, x, yy, zz, t)
            assert flips in (0, 1)
            new = int(o.sigma[0].reshape(L, L, L)[zz, yy, x] > 0) ^ flips
            want |= new << b
            nflip += flips
        assert got == want, (trial, t, k, y, z, hex(got), hex(want))
    if beta == 0.0:
        assert nflip == 40 * 32


def test_host_word_update_all_bond_patterns_and_draw_levels():
    """Exhaustive over the 64 neighbour-bond patterns of a site x both spin values, at a beta where all of
    cond4 / cond8 / cond12 occur often: the bit-sliced adder (Eq. 12-13) and the reconstructed mask (Eq. 17, R1)
    must equal 'flip iff dE <= 0 or R < T[dE]' with dE = 2 sigma h (Eq. 8-9)."""
    seed, beta, t = 99, 0.05, 7
    T = ea3d.thresholds(beta, 0)
    rng = np.random.default_rng(3)
    for word_index in range(24):
        ops = [int(v) for v in rng.integers(0, 2**32, 13, dtype=np.uint64)]
        got = binding.ising_hostcheck_update_word(0, seed, t, beta, ops, word_index)
        for b in range(32):
            s = 2 * ((ops[0] >> b) & 1) - 1
            h = 0
            for d in range(6):
                sk = 2 * ((ops[1 + d] >> b) & 1) - 1
                J = 1 - 2 * ((ops[7 + d] >> b) & 1)
                h += J * sk
            dE = 2 * s * h
            j = 32 * word_index + b
            R = ea3d.philox4x32_10((t, 0, j >> 2, 0), (seed, 0))[j & 3]
            flip = dE <= 0 or R < T[dE // 4 - 1]
            assert ((got >> b) & 1) == (((ops[0] >> b) & 1) ^ int(flip)), (word_index, b, dE, R)


def test_host_word_update_with_a_group_index_beyond_2_to_32():
    """L = 4096 has Philox group indices g = j >> 2 of 2^32 and more, whose high word is the counter word c3 (R9); the other sizes
    beyond 2048 (2560, 3072) stay below.  The kernels' word update (folded constants for c3 = 0 and c3 = 1) against 'flip iff
    dE <= 0 or R < T[dE]' with R from the oracle's draw of the site at its coordinates, for words on both sides of g = 2^32, the
    two words next to it, and the last word of the array."""
    seed, beta = 0xABCDEF0123456789, 0.05
    T = ea3d.thresholds(beta, 0)
    rng = np.random.default_rng(5)
    for L in (4096, 3072, 2560):
        wpr = L // 64
        n_words = wpr * L * L                      # words of one colour array
        assert (n_words > 2**29) == (L == 4096) and n_words <= 2**30
        picks = [n_words - 1, 0] + [int(v) for v in rng.integers(0, n_words, 5)]
        if L == 4096:
            picks += [2**29 - 1, 2**29, 2**29 + 1]
        for word_index in picks:
            t = int(rng.integers(0, 2**34))
            colour = t & 1
            k, row = word_index % wpr, word_index // wpr
            y, z = row % L, row // L
            xodd = (y + z + colour) & 1
            ops = [int(v) for v in rng.integers(0, 2**32, 13, dtype=np.uint64)]
            got = binding.ising_hostcheck_update_word(0, seed, t, beta, ops, word_index)
            for b in range(32):
                s = 2 * ((ops[0] >> b) & 1) - 1
                h = sum((1 - 2 * ((ops[7 + d] >> b) & 1)) * (2 * ((ops[1 + d] >> b) & 1) - 1) for d in range(6))
                dE = 2 * s * h
                x = 2 * (32 * k + b) + xodd       # bit b of word k of the half-row
                j = (x >> 1) + (L // 2) * (y + L * z)
                assert j == 32 * word_index + b and (j >> 2 >= 2**32) == (word_index >= 2**29)
                R = ea3d.philox_draw(L, seed, 0, x, y, z, t)
                flip = dE <= 0 or R < T[dE // 4 - 1]
                assert ((got >> b) & 1) == (((ops[0] >> b) & 1) ^ int(flip)), (L, word_index, b, dE, R)
