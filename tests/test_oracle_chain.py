"""Pins of the oracle's Markov chain (CPU only): what the paper and the mathematics fix.

(a) L=2 exact enumeration: Gibbs stationarity of the red-then-blue Metropolis sweep and the oracle's empirical
    one-sweep transition frequencies / long-run histogram        (Eq. 3, Eq. 9)
(b) beta = inf: only dE <= 0 moves, energy non-increasing         (Eq. 9)
(c) beta = 0: every proposal accepted                             (Eq. 9)
(d) incremental dE bookkeeping == energy recomputed from Eq. 1
(e) gauge invariance of the trajectory                            (site-keyed draws)
plus closed forms of Eq. 1, the dE set of Eq. 8, an independent pure-Python implementation, and the
high-temperature expansion of the energy.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import ea3d, ea3d_py

PHILOX, MINSTD = 0, 1
DIRS = ((1, 0, 0), (0, 1, 0), (0, 0, 1))


# ---------------------------------------------------------------- helpers written for the tests only

def idx(L, x, y, z):
    return (x % L) + L * ((y % L) + L * (z % L))


def random_pm1(rng, shape):
    return (2 * rng.integers(0, 2, shape) - 1).astype(np.int8)


def energy_np(L, sigma, Jx, Jy, Jz):
    """Eq. 1 with numpy rolls (each bond once)."""
    s = sigma.reshape(L, L, L).astype(np.int64)  # [z][y][x]
    e = 0
    for J, axis in ((Jx, 2), (Jy, 1), (Jz, 0)):
        e -= int((J.reshape(L, L, L) * s * np.roll(s, -1, axis=axis)).sum())
    return e


def make_oracle(L, rng_mode, seed=12345, nsamples=1, rng=None, J=None, sigma=None):
    rng = rng or np.random.default_rng(L * 7 + rng_mode)
    o = ea3d.Oracle(L, nsamples, seed, rng_mode)
    N = L**3
    if J is None:
        J = [random_pm1(rng, (nsamples, N)) for _ in range(3)]
    if sigma is None:
        sigma = random_pm1(rng, (nsamples, N))
    o.load_arrays(sigma, *J)
    return o


# ---------------------------------------------------------------- (a) exact L=2 model

class ExactL2:
    """The 256-state chain of the L=2 cube written out from Eq. 1, Eq. 3 and Eq. 9 (no oracle code).

    With L=2 the +d and -d neighbours coincide but the two couplings Jd[i] and Jd[i-d] are distinct bonds
    (R13), 24 bonds in all."""

    def __init__(self, Jx, Jy, Jz, beta, accept_prob=None):
        self.J = (Jx, Jy, Jz)
        self.beta = beta
        self.states = np.array(list(itertools.product((-1, 1), repeat=8)), dtype=np.int64)  # state id -> spins[8]
        self.ids = {tuple(s): k for k, s in enumerate(self.states)}
        self.colour = np.array([(x + y + z) & 1 for z in range(2) for y in range(2) for x in range(2)])
        self.accept_prob = accept_prob or (lambda dE: 1.0 if dE <= 0 else math.exp(-beta * dE))

    def H(self, s):
        e = 0
        for z in range(2):
            for y in range(2):
                for x in range(2):
                    i = idx(2, x, y, z)
                    for d, (dx, dy, dz) in enumerate(DIRS):
                        e -= self.J[d][i] * s[i] * s[idx(2, x + dx, y + dy, z + dz)]
        return int(e)

    def gibbs(self):
        w = np.array([math.exp(-self.beta * self.H(s)) for s in self.states])
        return w / w.sum()

    def half_sweep_matrix(self, colour):
        P = np.zeros((256, 256))
        sites = [i for i in range(8) if self.colour[i] == colour]
        for a, s in enumerate(self.states):
            p_flip = []
            for i in sites:
                t = s.copy()
                t[i] = -t[i]
                p_flip.append(self.accept_prob(self.H(t) - self.H(s)))
            for pattern in itertools.product((0, 1), repeat=len(sites)):
                t, p = s.copy(), 1.0
                for i, f, pf in zip(sites, pattern, p_flip):
                    p *= pf if f else 1.0 - pf
                    if f:
                        t[i] = -t[i]
                P[a, self.ids[tuple(t)]] += p
        return P

    def sweep_matrix(self):
        return self.half_sweep_matrix(0) @ self.half_sweep_matrix(1)  # red first (R8)


def _l2_couplings(seed=4):
    rng = np.random.default_rng(seed)
    return [random_pm1(rng, 8) for _ in range(3)]


@pytest.mark.parametrize("beta", [0.2, 0.45, 1 / 1.1])
def test_L2_gibbs_is_stationary_under_red_then_blue_metropolis(beta):
    """the sequential checkerboard update satisfies balance; Eq. 3 is its fixed point."""
    Jx, Jy, Jz = _l2_couplings()
    m = ExactL2(Jx, Jy, Jz, beta)
    P, pi = m.sweep_matrix(), m.gibbs()
    assert np.allclose(P.sum(axis=1), 1.0, atol=1e-13)
    assert np.abs(pi @ P - pi).max() < 1e-13
    # and the half-sweeps separately (each is a product of single-site Metropolis kernels)
    assert np.abs(pi @ m.half_sweep_matrix(0) - pi).max() < 1e-13
    assert np.abs(pi @ m.half_sweep_matrix(1) - pi).max() < 1e-13


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_L2_oracle_one_sweep_transition_frequencies(rng_mode):
    """Many independent samples (distinct Philox keys / MINSTD streams), same J and start state: the empirical
    distribution after ONE oracle sweep must match the exact row of P built with p = T/scale (strict <)."""
    beta, S = 0.35, 40000
    Jx, Jy, Jz = _l2_couplings()
    scale = 2.0**32 if rng_mode == PHILOX else 2.0**31 - 2  # MINSTD: R uniform on [1, 2^31-2]
    T = ea3d.thresholds(beta, rng_mode)

    def p_acc(dE):
        if dE <= 0:
            return 1.0
        t = T[dE // 4 - 1]
        return t / scale if rng_mode == PHILOX else (t - 1) / scale  # #{R in [1,2^31-2]: R < t}
    m = ExactL2(Jx, Jy, Jz, beta, accept_prob=p_acc)
    P = m.sweep_matrix()
    start = np.array([1, -1, -1, 1, 1, 1, -1, 1], dtype=np.int8)
    o = ea3d.Oracle(2, S, 2024, rng_mode)
    o.load_arrays(np.tile(start, (S, 1)), np.tile(Jx, (S, 1)), np.tile(Jy, (S, 1)), np.tile(Jz, (S, 1)))
    o.sweep(beta, 1)
    ids = np.array([m.ids[tuple(int(v) for v in row)] for row in o.sigma])
    counts = np.bincount(ids, minlength=256).astype(float)
    expect = P[m.ids[tuple(int(v) for v in start)]] * S
    assert counts[expect == 0].sum() == 0
    big = expect >= 5
    chi2 = ((counts[big] - expect[big]) ** 2 / expect[big]).sum()
    dof = big.sum() - 1
    assert chi2 < dof + 5 * math.sqrt(2 * dof), (chi2, dof)
    # a chain with the acceptance of dE=4 moves off by 10% would fail: sanity-check the test's power
    wrong = ExactL2(Jx, Jy, Jz, beta, accept_prob=lambda dE: p_acc(dE) * (0.9 if dE == 4 else 1.0)).sweep_matrix()
    ew = wrong[m.ids[tuple(int(v) for v in start)]] * S
    bw = ew >= 5
    assert ((counts[bw] - ew[bw]) ** 2 / ew[bw]).sum() > bw.sum() + 5 * math.sqrt(2 * bw.sum())


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_L2_oracle_long_run_histogram_is_gibbs(rng_mode):
    """BASELINE.json check (a): long-run state histogram vs exp(-beta H)/Z."""
    beta, S, burn, keep = 0.4, 512, 30, 60
    Jx, Jy, Jz = _l2_couplings(9)
    m = ExactL2(Jx, Jy, Jz, beta)
    pi = m.gibbs()
    rng = np.random.default_rng(1)
    o = ea3d.Oracle(2, S, 777, rng_mode)
    o.load_arrays(random_pm1(rng, (S, 8)), np.tile(Jx, (S, 1)), np.tile(Jy, (S, 1)), np.tile(Jz, (S, 1)))
    o.sweep(beta, burn)
    counts = np.zeros(256)
    weights = 2 ** np.arange(7, -1, -1)  # itertools.product order: first spin is the most significant
    for _ in range(keep):
        o.sweep(beta, 3)  # thinning; the L=2 chain decorrelates in a few sweeps at this beta
        ids = ((o.sigma.astype(np.int64) + 1) // 2) @ weights
        counts += np.bincount(ids, minlength=256)
    n = counts.sum()
    tv = 0.5 * np.abs(counts / n - pi).sum()
    assert tv < 0.03, tv  # sampling noise alone gives ~0.5*sqrt(2*256/(pi*n)) ~ 0.016 at n = 30720
    e_emp = sum(c * m.H(s) for c, s in zip(counts, m.states)) / n
    e_exact = sum(p * m.H(s) for p, s in zip(pi, m.states))
    assert abs(e_emp - e_exact) < 0.15


# ---------------------------------------------------------------- (b) (c) (d) special cases

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_beta_infinity_only_downhill_moves(rng_mode):
    o = make_oracle(8, rng_mode)
    E_prev = o.energy()[0][0]
    for _ in range(12):
        o.half_sweep(float("inf"))
        E = o.energy()[0][0]
        assert E <= E_prev
        E_prev = E
    assert o.stats[2] == 0 and o.stats[3] == 0  # no accepted dE>0 move, no dE outside Eq. 8
    # the very large finite beta behaves the same (T = 0)
    assert ea3d.thresholds(50.0, rng_mode) == (0, 0, 0)


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_beta_zero_flips_every_spin_of_the_colour(rng_mode):
    L = 6
    o = make_oracle(L, rng_mode)
    s0 = o.sigma.copy()
    E0 = o.energy()[0][0]
    colour = np.array([(x + y + z) & 1 for z in range(L) for y in range(L) for x in range(L)])
    o.half_sweep(0.0)
    assert np.array_equal(o.sigma[0][colour == 0], -s0[0][colour == 0])
    assert np.array_equal(o.sigma[0][colour == 1], s0[0][colour == 1])
    o.half_sweep(0.0)
    assert np.array_equal(o.sigma, -s0)
    assert o.energy()[0][0] == E0  # global flip leaves Eq. 1 unchanged
    assert o.stats[0] == o.stats[1] == L**3


@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [4, 6, 10])
def test_incremental_energy_equals_recomputed_and_dE_set(rng_mode, L):
    o = make_oracle(L, rng_mode, nsamples=2)
    E0 = o.energy()[0].copy()
    for _ in range(10):
        o.half_sweep(1 / 1.1)
        E, M = o.energy()
        assert np.array_equal(E, E0 + o.dE_sum)
        for s in range(2):
            assert E[s] == energy_np(L, o.sigma[s], o.Jx[s], o.Jy[s], o.Jz[s])
            assert M[s] == int(o.sigma[s].astype(np.int64).sum())
    assert o.stats[3] == 0 and o.stats[4:11].sum() == o.stats[0] == 10 * 2 * L**3 // 2  # Eq. 8 set only


def test_energy_closed_forms():
    L = 6
    N = L**3
    rng = np.random.default_rng(0)
    o = ea3d.Oracle(L, 1, 1, PHILOX)
    ones = np.ones((1, N), np.int8)
    o.load_arrays(ones, ones, ones, ones)
    assert o.energy()[0][0] == -3 * N and o.energy()[1][0] == N  # ferromagnet, all up
    J = [random_pm1(rng, (1, N)) for _ in range(3)]
    o.load_arrays(ones, *J)
    assert o.energy()[0][0] == -int(sum(j.astype(np.int64).sum() for j in J))  # all up: E = -sum J
    o.load_arrays(-ones, *J)
    assert o.energy()[0][0] == -int(sum(j.astype(np.int64).sum() for j in J)) and o.energy()[1][0] == -N
    # Neel state on the ferromagnet: every bond unsatisfied
    neel = np.array([1 - 2 * ((x + y + z) & 1) for z in range(L) for y in range(L) for x in range(L)], np.int8)
    o.load_arrays(neel[None], ones, ones, ones)
    assert o.energy()[0][0] == 3 * N and o.energy()[1][0] == 0
    # a single -J bond in direction y at one site raises the ferromagnetic energy by 2
    Jy = ones.copy()
    Jy[0, idx(L, 1, 2, 3)] = -1
    o.load_arrays(ones, ones, Jy, ones)
    assert o.energy()[0][0] == -3 * N + 2


def test_dE_uses_the_six_right_bonds():
    """One antiparallel neighbour at a time on the ferromagnet: dE of the centre spin must be 12 - 2*2 = 8 for each
    of the six neighbours and 12 otherwise; one flipped coupling likewise -- catches wrong index / transposed J."""
    L, beta = 6, 0.3
    N = L**3
    ones = np.ones((1, N), np.int8)
    c = (2, 3, 4)
    nbrs = [(c[0] + s * d[0], c[1] + s * d[1], c[2] + s * d[2]) for d in DIRS for s in (1, -1)]
    for site in nbrs + [(0, 0, 0)]:
        sg = ones.copy()
        sg[0, idx(L, *site)] = -1
        o = ea3d.Oracle(L, 1, 1, PHILOX)
        o.load_arrays(sg, ones, ones, ones)
        _, dE, _ = o.site_flips(beta, 0, *c, t=(sum(c) & 1))
        assert dE == (8 if site in nbrs else 12)
    # bonds: J_d at the centre couples to +d, J_d at (centre - d) couples to -d
    for d, dv in enumerate(DIRS):
        for at, hits in ((c, True), (tuple(ci - di for ci, di in zip(c, dv)), True),
                         (tuple(ci + di for ci, di in zip(c, dv)), False)):
            J = [ones.copy() for _ in range(3)]
            J[d][0, idx(L, *at)] = -1
            o = ea3d.Oracle(L, 1, 1, PHILOX)
            o.load_arrays(ones, *J)
            _, dE, _ = o.site_flips(beta, 0, *c, t=(sum(c) & 1))
            assert dE == (8 if hits else 12), (d, at)


# ---------------------------------------------------------------- (e) gauge invariance

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
def test_gauge_invariance_of_the_trajectory(rng_mode):
    """sigma_i -> s_i sigma_i, J_ik -> s_i J_ik s_k leaves dE of every site unchanged, hence (draws being keyed on
    the site, not on the state) the same sites flip: E'(t) = E(t), sigma'(t) = s sigma(t)."""
    L, beta = 8, 1 / 1.1
    N = L**3
    rng = np.random.default_rng(42)
    sigma = random_pm1(rng, (1, N))
    J = [random_pm1(rng, (1, N)) for _ in range(3)]
    g = random_pm1(rng, N)
    g3 = g.reshape(L, L, L)
    Jg = [(J[d][0].reshape(L, L, L) * g3 * np.roll(g3, -1, axis=2 - d)).reshape(1, N).astype(np.int8) for d in range(3)]
    a = make_oracle(L, rng_mode, J=J, sigma=sigma)
    b = make_oracle(L, rng_mode, J=Jg, sigma=(sigma * g).astype(np.int8))
    for _ in range(16):
        a.half_sweep(beta)
        b.half_sweep(beta)
        assert a.energy()[0][0] == b.energy()[0][0]
        assert np.array_equal(b.sigma[0], a.sigma[0] * g)
    assert a.stats[2] > 0  # some uphill moves were accepted: the thresholds were exercised


# ---------------------------------------------------------------- independent second implementation

@pytest.mark.parametrize("rng_mode", [PHILOX, MINSTD])
@pytest.mark.parametrize("L", [2, 4, 6])
def test_c_oracle_equals_pure_python_chain(rng_mode, L):
    N = L**3
    rng = np.random.default_rng(100 + L)
    sigma = random_pm1(rng, (2, N))
    J = [random_pm1(rng, (2, N)) for _ in range(3)]
    seed = (0x1234 << 32) | 0x9ABCDEF0
    o = make_oracle(L, rng_mode, seed=seed, nsamples=2, J=J, sigma=sigma)
    chains = []
    for s in range(2):
        c = ea3d_py.PyChain(L, seed, rng_mode, sample=s)
        c.spins = [int(v) for v in sigma[s]]
        c.J = [[int(v) for v in J[d][s]] for d in range(3)]
        chains.append(c)
    for beta in (0.3, 1 / 1.1, 1 / 0.7):
        for _ in range(4):
            o.half_sweep(beta)
            for s, c in enumerate(chains):
                c.half_sweep(beta)
                assert c.spins == [int(v) for v in o.sigma[s]]
                assert c.energy() == o.energy()[0][s]


def test_site_flips_agrees_with_half_sweep():
    L, beta = 6, 0.5
    for rng_mode in (PHILOX, MINSTD):
        o = make_oracle(L, rng_mode)
        o.sweep(beta, 2)
        before = o.sigma.copy()
        pred = {}
        for z in range(L):
            for y in range(L):
                for x in range(L):
                    if (x + y + z) & 1 == 0:
                        pred[(x, y, z)] = o.site_flips(beta, 0, x, y, z)[0]
        o.half_sweep(beta)
        for (x, y, z), f in pred.items():
            i = idx(L, x, y, z)
            assert (o.sigma[0, i] != before[0, i]) == bool(f)


def test_packed_round_trip_and_bit_conventions():
    """Eq. 10: spin bit 1 <=> +1; coupling bit 1 <=> -1; site i is bit i&31 of word i>>5."""
    L = 4
    N = L**3
    sw = np.zeros(N // 32, np.uint32)
    sw[1] = 1 << 3  # site 35 up, all others down
    s = ea3d.spins_from_packed(sw, N)
    assert s[35] == 1 and s.sum() == -(N - 2)
    jw = np.zeros(N // 32, np.uint32)
    jw[0] = 1 << 31
    j = ea3d.couplings_from_packed(jw, N)
    assert j[31] == -1 and j.sum() == N - 2
    rng = np.random.default_rng(2)
    sig = random_pm1(rng, N)
    assert np.array_equal(ea3d.spins_from_packed(ea3d.spins_to_packed(sig), N), sig)


# ---------------------------------------------------------------- statistical sanity of the whole dynamics

def test_high_temperature_energy_of_the_ferromagnet_and_of_pm_J():
    """Simple-cubic Ising high-temperature series e/N = -3 (v + 4 v^3 + O(v^5)), v = tanh(beta); for +-J, p=1/2, the
    disorder average is -3 tanh(beta) + O(v^5)... both catch a wrong sign or a wrong threshold scale."""
    L, beta = 12, 0.1
    N = L**3
    v = math.tanh(beta)
    rng = np.random.default_rng(8)
    ones = np.ones((1, N), np.int8)
    for J, expect in (([ones, ones, ones], -3 * (v + 4 * v**3)),
                      ([random_pm1(rng, (1, N)) for _ in range(3)], -3 * v)):
        o = make_oracle(L, PHILOX, J=J, sigma=random_pm1(rng, (1, N)))
        o.sweep(beta, 20)
        acc = []
        for _ in range(60):
            o.sweep(beta, 1)
            acc.append(o.energy()[0][0] / N)
        assert abs(np.mean(acc) - expect) < 0.02, (np.mean(acc), expect)


def test_overlap_against_closed_forms_and_a_library_dot_product():
    """q_ab = sum_i sigma^a_i sigma^b_i: q_aa = N, q(a, -a) = -N, symmetry, and numpy's dot product."""
    L, ns = 6, 4
    o = ea3d.Oracle(L, ns, 1, ea3d.PHILOX)
    rng = np.random.default_rng(9)
    sg = (2 * rng.integers(0, 2, size=(ns, L**3)) - 1).astype(np.int8)
    sg[3] = -sg[0]
    o.load_arrays(sg, np.ones_like(sg), np.ones_like(sg), np.ones_like(sg))
    N = L**3
    assert o.overlap(0, 0) == N and o.overlap(0, 3) == -N
    for a in range(ns):
        for b in range(ns):
            assert o.overlap(a, b) == o.overlap(b, a) == int(np.dot(sg[a].astype(np.int64), sg[b].astype(np.int64)))
