/*
 * ea3d_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct implementation of what the hot path of arXiv 1411.0127
 * computes: the checkerboard (red/blue) Metropolis sweep of the 3D +-J Edwards-Anderson model.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this file.  It shares no code with the CUDA path (paper_1411_0127_b200/csrc/); the two
 * were written separately from the same paper passages, which are cited beside each function as
 * PAPER.md:<line> (file /root/reference/PAPER.md) or as a DESIGN.md reading (R-numbers).
 *
 * State: one int8 per spin (sigma = +-1) and one int8 per coupling (J = +-1), per sample:
 *     sigma[s*N + i], Jx[s*N + i], Jy[..], Jz[..],   N = L^3,  i = x + L*(y + L*z)
 * Jd[i] couples site i with site i + d-hat (periodic).  There is no bit packing, no blocking and
 * no reordering here: every site of the active colour is visited with the scalar rule.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): exact Gibbs stationarity and transition rows at L=2,
 * beta=inf / beta=0 special cases, incremental-vs-recomputed energy, gauge invariance, closed-form
 * energies, cuRAND's host Philox4_32_10 generator, C++ std::minstd_rand0 and the Park-Miller
 * 10000th-value check, an independent pure-Python big-integer implementation (oracle/ea3d_py.py).
 * SplitMix64: the generator's published check sequence for seed 1234567 (tests/golden/splitmix64_seed1234567.txt),
 * two independent implementations and an inverse round trip of the finaliser.  The shared-random-number mode
 * (rng_mode 2) is pinned sample by sample against the independent mode (tests/test_oracle_shared.py).
 * The stored-state lane generators (rng_mode 3, 4; R19): MT19937 against C++ std::mt19937 (whose 10000th value
 * the C++ standard fixes) and numpy's legacy RandomState; Parisi-Rapuano against an unbounded-history restatement of the
 * paper's two lines in the test; the lane-driven sweep against a per-sample run fed with the same
 * draw table (tests/test_oracle_lanes.py).  The replica overlap: closed forms and a library dot product (tests/test_oracle_chain.py).
 * No function is left "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_RNG_PHILOX 0
#define ORACLE_RNG_MINSTD 1
/* The paper's own asynchronous multispin coding (Eq. 15): the 32 samples coded in
 * one word share ONE random number per (site, half-sweep).  DESIGN.md R18: the shared draw of the samples 32b..32b+31
 * (coded batch b) is the Philox draw of "sample" b, i.e. oracle_philox_draw(..., sample >> 5, ...). */
#define ORACLE_RNG_PHILOX_SHARED 2
/* Shared draw per 32-sample word as in mode 2, but the numbers come from generators with STORED state, one per "lane"
 * (the paper's one generator per thread), R19: Parisi-Rapuano and
 * MT19937. */
#define ORACLE_RNG_PR_LANES 3
#define ORACLE_RNG_MT_LANES 4

/* ------------------------------------------------------------------------------------------ */
/* Random number generators                                                                    */
/* ------------------------------------------------------------------------------------------ */

/* Philox4x32-10 (Salmon et al., SC'11; R10).  Ten rounds; in each round
 *   (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2 as 32x32->64 products,
 *   (c0,c1,c2,c3) <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0);
 * the key is bumped by (W0,W1) between rounds (9 bumps; round 1 uses the key as given). */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += W0;
            k1 += W1;
        }
        uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* n-th output (n >= 1) of SplitMix64 started at `seed` (R11). */
uint64_t oracle_splitmix64_output(uint64_t seed, uint64_t n)
{
    uint64_t z = seed + n * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z = z ^ (z >> 31);
    return z;
}

/* MINSTD, Eq. 7:  R_{n+1} = 16807 * R_n mod (2^31 - 1). */
uint32_t oracle_minstd_step(uint32_t r)
{
    return (uint32_t)(((uint64_t)16807u * (uint64_t)r) % 2147483647ull);
}

/* Seed state of MINSTD stream q = sample*N + i (R11): (splitmix64 output q+1 >> 34) + 1,
 * a value in [1, 2^30], hence a legal MINSTD state. */
uint32_t oracle_minstd_seed_state(uint64_t seed, uint64_t q)
{
    return (uint32_t)(oracle_splitmix64_output(seed, q + 1) >> 34) + 1u;
}

/* The draw of stream q in sweep n (n = t >> 1, from 0) is the (n+1)-th state after the seed state:
 * the generator is advanced, then used (R12).  Plain iteration. */
uint32_t oracle_minstd_draw(uint64_t seed, uint64_t q, uint64_t n)
{
    uint32_t r = oracle_minstd_seed_state(seed, q);
    for (uint64_t k = 0; k <= n; ++k) r = oracle_minstd_step(r);
    return r;
}

/* Philox draw of (sample, site, half-sweep t) (R9): key = (lo32(seed), hi32(seed)^sample),
 * counter = (lo32(t), hi32(t), lo32(g), hi32(g)), g = j >> 2, output word j & 3, where
 * j = (x >> 1) + (L/2)*(y + L*z) is the rank of the site within its colour. */
uint32_t oracle_philox_draw(int L, uint64_t seed, int sample, int x, int y, int z, uint64_t t)
{
    uint64_t j = (uint64_t)(x >> 1) + (uint64_t)(L / 2) * ((uint64_t)y + (uint64_t)L * (uint64_t)z);
    uint64_t g = j >> 2;
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) ^ (uint32_t)sample };
    uint32_t ctr[4] = { (uint32_t)t, (uint32_t)(t >> 32), (uint32_t)g, (uint32_t)(g >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[j & 3];
}

/* ------------------------------------------------------------------------------------------ */
/* Acceptance thresholds                                                                       */
/* ------------------------------------------------------------------------------------------ */

/* PAPER.md:242 ("R_max exp(-beta dE) = EXP12, EXP8, EXP4") with the scale of DESIGN.md R5/R6:
 *   Philox:  T[dE] = floor(2^32 * exp(-beta*dE))           in [0, 2^32]   (R uniform in [0, 2^32))
 *   MINSTD:  T[dE] = floor((2^31 - 1) * exp(-beta*dE))     in [0, 2^31-1] (R in [1, 2^31-2])
 *   Parisi-Rapuano and MT19937 give uniform 32-bit words: the Philox scale.
 * T[0],T[1],T[2] are for dE = 4, 8, 12.  Returns 0, or -1 for beta < 0 / NaN / unknown mode. */
int oracle_thresholds(double beta, int rng_mode, uint64_t T[3])
{
    if (!(beta >= 0.0)) return -1;
    if (rng_mode < ORACLE_RNG_PHILOX || rng_mode > ORACLE_RNG_MT_LANES) return -1;
    for (int k = 0; k < 3; ++k) {
        double dE = 4.0 * (double)(k + 1);
        double x = beta * dE;
        double p = exp(-x);
        double scaled = (rng_mode != ORACLE_RNG_MINSTD) ? ldexp(p, 32) : 2147483647.0 * p;
        T[k] = (uint64_t)floor(scaled);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* The model                                                                                   */
/* ------------------------------------------------------------------------------------------ */

static inline int wrap_up(int a, int L) { return (a + 1 == L) ? 0 : a + 1; }
static inline int wrap_dn(int a, int L) { return (a == 0) ? L - 1 : a - 1; }
static inline int64_t site_index(int L, int x, int y, int z)
{
    return (int64_t)x + (int64_t)L * ((int64_t)y + (int64_t)L * (int64_t)z);
}

/* dE of flipping sigma_i, Eq. 8:  dE = H[-sigma_i] - H[sigma_i] = 2 sigma_i h_i with
 * h_i = sum over the six neighbours k of J_ik sigma_k   (H from PAPER.md:25 Eq. 1). */
static inline int local_dE(int L, const int8_t *sg, const int8_t *Jx, const int8_t *Jy, const int8_t *Jz,
                           int x, int y, int z)
{
    int64_t i = site_index(L, x, y, z);
    int64_t ixp = site_index(L, wrap_up(x, L), y, z), ixm = site_index(L, wrap_dn(x, L), y, z);
    int64_t iyp = site_index(L, x, wrap_up(y, L), z), iym = site_index(L, x, wrap_dn(y, L), z);
    int64_t izp = site_index(L, x, y, wrap_up(z, L)), izm = site_index(L, x, y, wrap_dn(z, L));
    int h = Jx[i] * sg[ixp] + Jx[ixm] * sg[ixm]
          + Jy[i] * sg[iyp] + Jy[iym] * sg[iym]
          + Jz[i] * sg[izp] + Jz[izm] * sg[izm];
    return 2 * sg[i] * h;
}

/* Metropolis rule, Eq. 9 with the integer compare of PAPER.md:242 / Eq. 15 (strict <,
 * DESIGN.md R4):  accept iff dE <= 0 or R < T[dE].  Returns 1 = flip, 0 = keep, -1 = dE outside Eq. 8. */
static inline int metropolis_accept(int dE, uint64_t R, const uint64_t T[3])
{
    if (dE <= 0) return (dE == 0 || dE == -4 || dE == -8 || dE == -12) ? 1 : -1;
    if (dE == 4) return R < T[0];
    if (dE == 8) return R < T[1];
    if (dE == 12) return R < T[2];
    return -1;
}

/* Energy and magnetisation from scratch, Eq. 1 (every bond once):
 *   E[s] = - sum_i ( Jx[i] s_i s_{i+x} + Jy[i] s_i s_{i+y} + Jz[i] s_i s_{i+z} ),   M[s] = sum_i s_i. */
void oracle_energy(int L, int nsamples, const int8_t *sigma, const int8_t *Jx, const int8_t *Jy,
                   const int8_t *Jz, int64_t *E, int64_t *M)
{
    int64_t N = (int64_t)L * L * L;
    for (int s = 0; s < nsamples; ++s) {
        const int8_t *sg = sigma + (int64_t)s * N;
        const int8_t *jx = Jx + (int64_t)s * N, *jy = Jy + (int64_t)s * N, *jz = Jz + (int64_t)s * N;
        int64_t e = 0, m = 0;
#pragma omp parallel for reduction(+ : e, m) schedule(static)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    int64_t i = site_index(L, x, y, z);
                    int64_t ixp = site_index(L, wrap_up(x, L), y, z);
                    int64_t iyp = site_index(L, x, wrap_up(y, L), z);
                    int64_t izp = site_index(L, x, y, wrap_up(z, L));
                    e -= jx[i] * sg[i] * sg[ixp] + jy[i] * sg[i] * sg[iyp] + jz[i] * sg[i] * sg[izp];
                    m += sg[i];
                }
        E[s] = e;
        if (M) M[s] = m;
    }
}

/* Overlap of two replicas (samples with the same couplings, "we simulate four replicas at once"):
 *   q_ab = sum_i sigma_i^a sigma_i^b,   an integer in [-N, N]; q_aa = N. */
int64_t oracle_overlap(int L, const int8_t *sigma_a, const int8_t *sigma_b)
{
    int64_t N = (int64_t)L * L * L, q = 0;
    for (int64_t i = 0; i < N; ++i) q += (int64_t)sigma_a[i] * (int64_t)sigma_b[i];
    return q;
}

/* Fill the per-site MINSTD stream states with their seed states (R11). */
void oracle_minstd_init(int L, int nsamples, uint64_t seed, uint32_t *state)
{
    int64_t N = (int64_t)L * L * L;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < (int64_t)nsamples * N; ++q)
        state[q] = oracle_minstd_seed_state(seed, (uint64_t)q);
}

/* One colour half-sweep: every site of colour c = t & 1 (c = (x+y+z) & 1; red = 0 is
 * the colour of even t, R8) is visited once with the Metropolis rule.  Same-colour sites
 * have no bond in common, so the visiting order is irrelevant and the loop over planes
 * may run on several cores.  The draw R(sample, site, t) is consumed whether or not it is needed.
 *
 *   minstd_state : nsamples*N stream states (MINSTD mode; advanced in place), unused for Philox
 *   dE_sum       : nsamples running sums, += dE of every accepted flip (incremental energy)
 *   stats[0..10] : += {proposals, accepted, accepted with dE > 0, proposals with dE outside Eq. 8,
 *                      histogram of proposals over dE = -12,-8,-4,0,4,8,12 (stats[4..10])}
 * Returns 0, or -1 on bad arguments. */
static int half_sweep_core(int L, int nsamples, int8_t *sigma, const int8_t *Jx, const int8_t *Jy, const int8_t *Jz,
                           uint64_t seed, int rng_mode, uint64_t t, const uint64_t T[3], uint32_t *minstd_state,
                           const uint32_t *draw_table, int64_t *dE_sum, int64_t *stats)
{
    if (L < 2 || (L & 1) || nsamples < 1) return -1;
    if (rng_mode == ORACLE_RNG_MINSTD && !minstd_state) return -1;
    if ((rng_mode == ORACLE_RNG_PR_LANES || rng_mode == ORACLE_RNG_MT_LANES) && !draw_table) return -1;
    int64_t N = (int64_t)L * L * L;
    int colour = (int)(t & 1);
    int64_t st_prop = 0, st_acc = 0, st_up = 0, st_bad = 0;
    int64_t h0 = 0, h1 = 0, h2 = 0, h3 = 0, h4 = 0, h5 = 0, h6 = 0;
    for (int s = 0; s < nsamples; ++s) {
        int8_t *sg = sigma + (int64_t)s * N;
        const int8_t *jx = Jx + (int64_t)s * N, *jy = Jy + (int64_t)s * N, *jz = Jz + (int64_t)s * N;
        int64_t dsum = 0;
#pragma omp parallel for reduction(+ : dsum, st_prop, st_acc, st_up, st_bad, h0, h1, h2, h3, h4, h5, h6) schedule(static)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != colour) continue;
                    int64_t i = site_index(L, x, y, z);
                    int dE = local_dE(L, sg, jx, jy, jz, x, y, z);
                    uint64_t R;
                    if (rng_mode == ORACLE_RNG_PHILOX) {
                        R = oracle_philox_draw(L, seed, s, x, y, z, t);
                    } else if (rng_mode == ORACLE_RNG_PHILOX_SHARED) {
                        R = oracle_philox_draw(L, seed, s >> 5, x, y, z, t);
                    } else if (rng_mode == ORACLE_RNG_PR_LANES || rng_mode == ORACLE_RNG_MT_LANES) {
                        /* DESIGN.md R19: the draw of (coded batch s>>5, colour rank j) of this half-sweep */
                        int64_t j = (int64_t)(x >> 1) + (int64_t)(L / 2) * ((int64_t)y + (int64_t)L * (int64_t)z);
                        R = draw_table[(int64_t)(s >> 5) * (N / 2) + j];
                    } else {
                        uint32_t *st = &minstd_state[(int64_t)s * N + i];
                        *st = oracle_minstd_step(*st);
                        R = *st;
                    }
                    int acc = metropolis_accept(dE, R, T);
                    st_prop++;
                    switch (dE) {
                        case -12: h0++; break;
                        case -8: h1++; break;
                        case -4: h2++; break;
                        case 0: h3++; break;
                        case 4: h4++; break;
                        case 8: h5++; break;
                        case 12: h6++; break;
                        default: break;
                    }
                    if (acc < 0) { st_bad++; continue; }
                    if (acc) {
                        sg[i] = (int8_t)(-sg[i]);
                        dsum += dE;
                        st_acc++;
                        if (dE > 0) st_up++;
                    }
                }
        if (dE_sum) dE_sum[s] += dsum;
    }
    if (stats) {
        stats[0] += st_prop; stats[1] += st_acc; stats[2] += st_up; stats[3] += st_bad;
        stats[4] += h0; stats[5] += h1; stats[6] += h2; stats[7] += h3; stats[8] += h4; stats[9] += h5;
        stats[10] += h6;
    }
    return 0;
}

int oracle_half_sweep(int L, int nsamples, int8_t *sigma, const int8_t *Jx, const int8_t *Jy, const int8_t *Jz,
                      uint64_t seed, int rng_mode, uint64_t t, const uint64_t T[3], uint32_t *minstd_state,
                      int64_t *dE_sum, int64_t *stats)
{
    if (rng_mode == ORACLE_RNG_PR_LANES || rng_mode == ORACLE_RNG_MT_LANES) return -1; /* use oracle_half_sweep_lanes */
    return half_sweep_core(L, nsamples, sigma, Jx, Jy, Jz, seed, rng_mode, t, T, minstd_state, NULL, dE_sum, stats);
}

/* The single-site rule on its own, for checks of sampled sites at sizes where a whole oracle
 * trajectory is too slow: given the configuration BEFORE half-sweep t, would site (x,y,z) of
 * `sample` flip?  sigma/J point at that sample's arrays.  MINSTD draws are recomputed from the seed
 * state by plain iteration.  Returns 1 = flips, 0 = stays, -1 = site not of colour t&1 or bad dE;
 * *dE_out and *R_out receive dE and the draw. */
int oracle_site_flips(int L, const int8_t *sigma, const int8_t *Jx, const int8_t *Jy, const int8_t *Jz,
                      int sample, uint64_t seed, int rng_mode, uint64_t t, const uint64_t T[3],
                      int x, int y, int z, int *dE_out, uint64_t *R_out)
{
    if (((x + y + z) & 1) != (int)(t & 1)) return -1;
    int64_t N = (int64_t)L * L * L;
    int dE = local_dE(L, sigma, Jx, Jy, Jz, x, y, z);
    uint64_t R;
    if (rng_mode == ORACLE_RNG_PHILOX)
        R = oracle_philox_draw(L, seed, sample, x, y, z, t);
    else if (rng_mode == ORACLE_RNG_PHILOX_SHARED)
        R = oracle_philox_draw(L, seed, sample >> 5, x, y, z, t);
    else
        R = oracle_minstd_draw(seed, (uint64_t)sample * (uint64_t)N + (uint64_t)site_index(L, x, y, z), t >> 1);
    if (dE_out) *dE_out = dE;
    if (R_out) *R_out = R;
    return metropolis_accept(dE, R, T);
}

/* 64-bit FNV-1a over a byte string (checksum of BASELINE.json config 4; public constants). */
uint64_t oracle_fnv1a64(const uint8_t *data, uint64_t nbytes)
{
    uint64_t h = 0xcbf29ce484222325ull;
    for (uint64_t k = 0; k < nbytes; ++k) {
        h ^= (uint64_t)data[k];
        h *= 0x100000001b3ull;
    }
    return h;
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int oracle_get_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* Generators with stored state, one per lane (R19)           */
/* ------------------------------------------------------------------------------------------ */

#define ORACLE_PR_RING 62
#define ORACLE_MT_N 624

/* Parisi-Rapuano: "a lagged-Fibonacci-like PRNG with a minimal state of 62 words",
 *     ira[i] = ira[i-24] + ira[i-55];   R = ira[i] ^ ira[i-61];
 * on 32-bit words (the sum is mod 2^32).  The state is the last 62 words; they are kept in a ring indexed by
 * i mod 62.  The seed words are ira[0..61], so draw number n (from 0) is R of i = 62 + n. */
uint32_t oracle_pr_next(uint32_t ring[ORACLE_PR_RING], uint64_t *ndrawn)
{
    uint64_t i = (uint64_t)ORACLE_PR_RING + *ndrawn;
    uint32_t v = ring[(i - 24) % ORACLE_PR_RING] + ring[(i - 55) % ORACLE_PR_RING];
    uint32_t R = v ^ ring[(i - 61) % ORACLE_PR_RING];
    ring[i % ORACLE_PR_RING] = v;
    *ndrawn += 1;
    return R;
}

/* Seed words of lane q (R19): ira[r] = high 32 bits of SplitMix64 output number q*62 + r + 1 from `seed`. */
void oracle_pr_seed(uint64_t seed, uint64_t lane, uint32_t ring[ORACLE_PR_RING])
{
    for (int r = 0; r < ORACLE_PR_RING; ++r)
        ring[r] = (uint32_t)(oracle_splitmix64_output(seed, lane * ORACLE_PR_RING + (uint64_t)r + 1) >> 32);
}

/* MT19937 (Matsumoto & Nishimura 1998; "the widely known Mersenne Twister MT19937"): seeding by
 * init_genrand(s), mt[0] = s, mt[i] = 1812433253 * (mt[i-1] ^ (mt[i-1] >> 30)) + i. */
void oracle_mt_seed(uint32_t s, uint32_t mt[ORACLE_MT_N])
{
    mt[0] = s;
    for (uint32_t i = 1; i < ORACLE_MT_N; ++i) mt[i] = 1812433253u * (mt[i - 1] ^ (mt[i - 1] >> 30)) + i;
}

/* The textbook generator: when the 624 words are used up the whole block is regenerated,
 *   y = (mt[k] & UPPER) | (mt[k+1] & LOWER);  mt[k] = mt[k+397] ^ (y >> 1) ^ (y odd ? 0x9908b0df : 0)   (indices mod 624),
 * and output number n is the tempered word n mod 624 of the current block. */
uint32_t oracle_mt_next(uint32_t mt[ORACLE_MT_N], uint64_t *ndrawn)
{
    uint32_t pos = (uint32_t)(*ndrawn % ORACLE_MT_N);
    if (pos == 0) {
        for (int k = 0; k < ORACLE_MT_N; ++k) {
            uint32_t y = (mt[k] & 0x80000000u) | (mt[(k + 1) % ORACLE_MT_N] & 0x7fffffffu);
            mt[k] = mt[(k + 397) % ORACLE_MT_N] ^ (y >> 1) ^ ((y & 1u) ? 0x9908b0dfu : 0u);
        }
    }
    uint32_t y = mt[pos];
    y ^= y >> 11;
    y ^= (y << 7) & 0x9d2c5680u;
    y ^= (y << 15) & 0xefc60000u;
    y ^= y >> 18;
    *ndrawn += 1;
    return y;
}

/* init_genrand seed of lane q (R19): high 32 bits of SplitMix64 output number q + 1 from `seed`. */
uint32_t oracle_mt_lane_seed(uint64_t seed, uint64_t lane)
{
    return (uint32_t)(oracle_splitmix64_output(seed, lane + 1) >> 32);
}

int oracle_lane_state_words(int rng_mode)
{
    return rng_mode == ORACLE_RNG_PR_LANES ? ORACLE_PR_RING : rng_mode == ORACLE_RNG_MT_LANES ? ORACLE_MT_N : 0;
}

/* state: nlanes * oracle_lane_state_words(mode) words, lane-major; ndrawn: nlanes counters. */
int oracle_lanes_init(int rng_mode, uint64_t seed, int64_t nlanes, uint32_t *state, uint64_t *ndrawn)
{
    const int W = oracle_lane_state_words(rng_mode);
    if (W == 0 || nlanes < 1) return -1;
    for (int64_t q = 0; q < nlanes; ++q) {
        if (rng_mode == ORACLE_RNG_PR_LANES) oracle_pr_seed(seed, (uint64_t)q, state + q * W);
        else oracle_mt_seed(oracle_mt_lane_seed(seed, (uint64_t)q), state + q * W);
        ndrawn[q] = 0;
    }
    return 0;
}

static inline uint32_t lane_next(int rng_mode, uint32_t *lane_state, uint64_t *ndrawn)
{
    return rng_mode == ORACLE_RNG_PR_LANES ? oracle_pr_next(lane_state, ndrawn) : oracle_mt_next(lane_state, ndrawn);
}

/* The draws of one colour half-sweep (R19).  The N/2 sites of the colour are numbered by their colour rank j and
 * taken in groups of four, g = j >> 2 (ngroups = N/8 groups); with k coded batches of 32 samples there are k * ngroups
 * units u = b * ngroups + g, b = batch.  Lane q serves the units u = q, q + nlanes, q + 2 nlanes, ... in that order, and for
 * each unit the four sites w = 0..3 of its group: the next number of the lane is the draw shared by the 32 samples of
 * batch b at site j = 4g + w.  Every lane takes the same number of draws per half-sweep,
 * 4 ceil(k ngroups / nlanes): a lane whose last unit does not exist draws and discards.  Small lattices fill the machine
 * with many coded batches, which is why the units, not the groups, are dealt to the lanes.
 * table[b * (N/2) + j] receives the draw. */
int oracle_lanes_draw_table(int rng_mode, int64_t nlanes, uint32_t *state, uint64_t *ndrawn, int64_t ngroups, int k,
                            uint32_t *table)
{
    const int W = oracle_lane_state_words(rng_mode);
    if (W == 0 || nlanes < 1 || ngroups < 1 || k < 1) return -1;
    const int64_t units = (int64_t)k * ngroups;
    const int64_t rounds = (units + nlanes - 1) / nlanes;
    for (int64_t q = 0; q < nlanes; ++q)
        for (int64_t m = 0; m < rounds; ++m) {
            const int64_t u = q + m * nlanes;
            for (int w = 0; w < 4; ++w) {
                const uint32_t R = lane_next(rng_mode, state + q * W, &ndrawn[q]);
                if (u < units) table[4 * u + w] = R;   /* 4u + w = b * (N/2) + 4g + w */
            }
        }
    return 0;
}

/* One colour half-sweep in a lane mode: the draw table of this half-sweep, then the scalar rule of oracle_half_sweep
 * with R = table[batch][colour rank].  nsamples must be a multiple of 32, L a multiple of 4 (so that N/2 is a multiple of 4).
 * scratch: (nsamples/32) * N/2 words. */
int oracle_half_sweep_lanes(int L, int nsamples, int8_t *sigma, const int8_t *Jx, const int8_t *Jy, const int8_t *Jz,
                            int rng_mode, int64_t nlanes, uint32_t *state, uint64_t *ndrawn, uint64_t t,
                            const uint64_t T[3], uint32_t *scratch, int64_t *dE_sum, int64_t *stats)
{
    if (nsamples < 32 || nsamples % 32 || L < 2 || ((int64_t)L * L * L) % 8) return -1;
    const int64_t ngroups = (int64_t)L * L * L / 8;
    if (oracle_lanes_draw_table(rng_mode, nlanes, state, ndrawn, ngroups, nsamples / 32, scratch) != 0) return -1;
    return half_sweep_core(L, nsamples, sigma, Jx, Jy, Jz, 0, rng_mode, t, T, NULL, scratch, dE_sum, stats);
}

/* PAPER.md:196-197 and Table II: "its kernel version counting the fraction of odd numbers".  Every lane
 * draws `ndraws` numbers; odd[q] = how many were odd, sum[q] = their sum mod 2^64 (a checksum of the whole sequence).
 * Kinds: 3 = Parisi-Rapuano, 4 = MT19937 (lanes seeded as above), 1 = MINSTD with the seed state of stream q (R11) advanced
 * ndraws times (Eq. 7), 0 = Philox4x32-10 with key (lo32 seed, hi32 seed) and counter (lo32 c, hi32 c, lo32 q, hi32 q) for call
 * number c = n >> 2, output word n & 3. */
int oracle_count_odd(int kind, uint64_t seed, int64_t nlanes, int64_t ndraws, uint64_t *odd, uint64_t *sum)
{
    if (nlanes < 1 || ndraws < 0) return -1;
    if (kind != ORACLE_RNG_PHILOX && kind != ORACLE_RNG_MINSTD && kind != ORACLE_RNG_PR_LANES && kind != ORACLE_RNG_MT_LANES)
        return -1;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < nlanes; ++q) {
        uint64_t o = 0, s = 0;
        if (kind == ORACLE_RNG_PR_LANES || kind == ORACLE_RNG_MT_LANES) {
            uint32_t st[ORACLE_MT_N];
            uint64_t nd = 0;
            if (kind == ORACLE_RNG_PR_LANES) oracle_pr_seed(seed, (uint64_t)q, st);
            else oracle_mt_seed(oracle_mt_lane_seed(seed, (uint64_t)q), st);
            for (int64_t n = 0; n < ndraws; ++n) {
                const uint32_t R = lane_next(kind, st, &nd);
                o += R & 1u;
                s += R;
            }
        } else if (kind == ORACLE_RNG_MINSTD) {
            uint32_t r = oracle_minstd_seed_state(seed, (uint64_t)q);
            for (int64_t n = 0; n < ndraws; ++n) {
                r = oracle_minstd_step(r);
                o += r & 1u;
                s += r;
            }
        } else {
            const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
            for (int64_t n = 0; n < ndraws; ++n) {
                const uint64_t c = (uint64_t)n >> 2;
                const uint32_t ctr[4] = { (uint32_t)c, (uint32_t)(c >> 32), (uint32_t)q, (uint32_t)((uint64_t)q >> 32) };
                uint32_t out[4];
                oracle_philox4x32_10(ctr, key, out);
                o += out[n & 3] & 1u;
                s += out[n & 3];
            }
        }
        odd[q] = o;
        sum[q] = s;
    }
    return 0;
}
