"""Second, independent CPU implementation in pure Python integers (small L only).  TEST INFRASTRUCTURE ONLY.

Written separately from oracle/ea3d_oracle.c so that the two can be checked against each other:
different data structures (lists of tuples, explicit bond list), stateless MINSTD through modular
exponentiation, arbitrary-precision integers, and the energy change computed as an energy difference
of the bonds touching the site rather than as 2*sigma*h.  Citations as in ea3d_oracle.c.
"""
from __future__ import annotations

import math

MASK32 = 0xFFFFFFFF
MASK64 = 0xFFFFFFFFFFFFFFFF
MINSTD_A = 16807
MINSTD_M = 2**31 - 1
PHILOX, MINSTD = 0, 1


def philox4x32_10(ctr, key):
    """Philox4x32-10 (R10) on Python integers."""
    c = [int(v) & MASK32 for v in ctr]
    k = [int(v) & MASK32 for v in key]
    for r in range(10):
        kr0 = (k[0] + r * 0x9E3779B9) & MASK32
        kr1 = (k[1] + r * 0xBB67AE85) & MASK32
        prod0 = 0xD2511F53 * c[0]
        prod1 = 0xCD9E8D57 * c[2]
        c = [((prod1 >> 32) ^ c[1] ^ kr0) & MASK32, prod1 & MASK32,
             ((prod0 >> 32) ^ c[3] ^ kr1) & MASK32, prod0 & MASK32]
    return tuple(c)


def splitmix64_output(seed, n):
    z = (seed + n * 0x9E3779B97F4A7C15) & MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
    return z ^ (z >> 31)


def splitmix64_unmix(z):
    """Inverse of the SplitMix64 finaliser (each xor-shift and odd multiply is a bijection of 2^64)."""
    def unxorshift(v, s):
        r = v
        for _ in range(64 // s + 1):
            r = v ^ (r >> s)
        return r
    z = unxorshift(z, 31)
    z = (z * pow(0x94D049BB133111EB, -1, 2**64)) & MASK64
    z = unxorshift(z, 27)
    z = (z * pow(0xBF58476D1CE4E5B9, -1, 2**64)) & MASK64
    z = unxorshift(z, 30)
    return z


def minstd_seed_state(seed, q):
    return (splitmix64_output(seed, q + 1) >> 34) + 1


def minstd_draw(seed, q, n):
    """Stateless: R_n = 16807^(n+1) * s0 mod (2^31-1)  (Eq. 7 iterated n+1 times)."""
    return (pow(MINSTD_A, n + 1, MINSTD_M) * minstd_seed_state(seed, q)) % MINSTD_M


def thresholds(beta, rng_mode):
    scale = 2.0**32 if rng_mode == PHILOX else 2147483647.0
    return tuple(int(math.floor(scale * math.exp(-(beta * dE)))) for dE in (4.0, 8.0, 12.0))


class PyChain:
    """One sample of the chain on Python lists.  spins[i] in {-1,+1}; J[d][i] in {-1,+1}."""

    def __init__(self, L, seed, rng_mode, sample=0, nsites_all=None):
        self.L, self.seed, self.rng_mode, self.sample = L, seed, rng_mode, sample
        self.N = L**3
        self.t = 0
        self.spins = [1] * self.N
        self.J = [[1] * self.N for _ in range(3)]

    def idx(self, x, y, z):
        L = self.L
        return (x % L) + L * ((y % L) + L * (z % L))

    def bonds_of(self, x, y, z):
        """The six (coupling, neighbour index) pairs of site (x,y,z) (PAPER.md:105 cubic stencil)."""
        i = self.idx(x, y, z)
        out = []
        for d, (dx, dy, dz) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
            out.append((self.J[d][i], self.idx(x + dx, y + dy, z + dz)))
            m = self.idx(x - dx, y - dy, z - dz)
            out.append((self.J[d][m], m))
        return i, out

    def local_energy(self, i, bonds, s_i):
        return -sum(Jb * s_i * self.spins[k] for Jb, k in bonds)

    def draw(self, x, y, z):
        L = self.L
        if self.rng_mode == PHILOX:
            j = (x >> 1) + (L // 2) * (y + L * z)
            g = j >> 2
            key = (self.seed & MASK32, ((self.seed >> 32) & MASK32) ^ self.sample)
            ctr = (self.t & MASK32, (self.t >> 32) & MASK32, g & MASK32, (g >> 32) & MASK32)
            return philox4x32_10(ctr, key)[j & 3]
        q = self.sample * self.N + self.idx(x, y, z)
        return minstd_draw(self.seed, q, self.t >> 1)

    def half_sweep(self, beta):
        T = thresholds(beta, self.rng_mode)
        colour = self.t & 1
        L = self.L
        flips = []
        for z in range(L):
            for y in range(L):
                for x in range(L):
                    if (x + y + z) & 1 != colour:
                        continue
                    i, bonds = self.bonds_of(x, y, z)
                    s = self.spins[i]
                    dE = self.local_energy(i, bonds, -s) - self.local_energy(i, bonds, s)
                    assert dE in (-12, -8, -4, 0, 4, 8, 12)  # PAPER.md:234 Eq. 8
                    R = self.draw(x, y, z)
                    if dE <= 0 or R < T[dE // 4 - 1]:
                        flips.append(i)
        # same-colour sites share no bond: applying the flips afterwards is equivalent
        for i in flips:
            self.spins[i] = -self.spins[i]
        self.t += 1

    def energy(self):
        L = self.L
        e = 0
        for z in range(L):
            for y in range(L):
                for x in range(L):
                    i = self.idx(x, y, z)
                    for d, (dx, dy, dz) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
                        e -= self.J[d][i] * self.spins[i] * self.spins[self.idx(x + dx, y + dy, z + dz)]
        return e
