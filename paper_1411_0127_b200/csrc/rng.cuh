// rng.cuh -- the two in-register random number generators of the CUDA path.
//
// Nothing here is shared with oracle/: this file was written from the same definitions (R9-R12).
// All functions are __host__ __device__ so that the host-only test hook ising_hostcheck_update_word can
// run the very code the kernels run.
#pragma once
#include <stdint.h>

#ifdef __CUDACC__
#define ISING_HD __host__ __device__ __forceinline__
#else
#define ISING_HD inline
#endif

namespace isingk {

// ---------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11; R10).  Round r = 0..9 with round key
// (K0_r, K1_r) = (k0 + r*W0, k1 + r*W1):
//     (hi0:lo0) = M0*c0,  (hi1:lo1) = M1*c2,   (c0,c1,c2,c3) <- (hi1^c1^K0_r, lo1, hi0^c3^K1_r, lo0)
// Keying (R9): key = (lo32 seed, hi32 seed ^ sample); counter = (lo32 t, hi32 t, lo32 g, hi32 g) with g = j>>2 the
// colour rank of the site divided by 4 (g = N/8 at most: below 2^32 up to L = 3250, below 2^33 up to L = 4096); output word j&3 is site j's draw.
// ---------------------------------------------------------------------------------------------------
constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

// Plain, unfolded form: used by the generic one-site-at-a-time kernel and to fold the constants below.
ISING_HD void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                            uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Within one half-sweep launch t and the key are the same for every call, and only c2 = g varies.  Hence
// in round 0 the product M0*c0 is a launch constant, which makes c2 after round 0 a launch constant, which
// makes the product M1*c2 of round 1 a launch constant.  The host folds these (fold_philox) so that a call
// costs 18 wide multiplies and 19 XORs instead of 20 + 20 + 18 key bumps.  With X_r the state after round r:
//     X1 = (Qhi ^ a, Qlo, A2, A3)                 Q = M1*g,  a = thi^K0_0,  A2 = P0hi^K1_0,  A3 = P0lo,  P0 = M0*tlo
//     X2 = (Qlo ^ b, Blo, Phi ^ d, Plo)           P = M0*X1.c0,  B = M1*A2,  b = Bhi^K0_1,  d = A3^K1_1
//     X3 = (Q'hi ^ e, Q'lo, P'hi ^ Plo ^ K1_2, P'lo)     P' = M0*X2.c0,  Q' = M1*X2.c2,  e = Blo^K0_2
//     rounds 3..9 as written above.
struct PhiloxSampleConst {
    uint32_t b, d, e;
    uint32_t k1[8];  // K1_2 .. K1_9
};
struct PhiloxCommonConst {
    uint32_t a;
    uint32_t k0[7];  // K0_3 .. K0_9
};

// c3 = hi32(g): 0 for every group index below 2^32 (every lattice up to L = 3250); L = 4096 has g < 2^33 and folds a
// second set for c3 = 1, which differs in b and e only (c3 enters round 0 through A2, and A2 only through B).
ISING_HD void fold_philox(uint64_t seed, uint32_t sample, uint64_t t, PhiloxCommonConst *cc, PhiloxSampleConst *sc, uint32_t c3 = 0u)
{
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32) ^ sample;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);
    const uint64_t P0 = (uint64_t)PHILOX_M0 * tlo;
    const uint32_t A2 = (uint32_t)(P0 >> 32) ^ c3 ^ k1;
    const uint32_t A3 = (uint32_t)P0;
    const uint64_t B = (uint64_t)PHILOX_M1 * A2;
    cc->a = thi ^ k0;
    for (int r = 3; r < 10; ++r) cc->k0[r - 3] = k0 + (uint32_t)r * PHILOX_W0;
    sc->b = (uint32_t)(B >> 32) ^ (k0 + PHILOX_W0);
    sc->d = A3 ^ (k1 + PHILOX_W1);
    sc->e = (uint32_t)B ^ (k0 + 2u * PHILOX_W0);
    for (int r = 2; r < 10; ++r) sc->k1[r - 2] = k1 + (uint32_t)r * PHILOX_W1;
}

// The same in two steps, for kernels that run many half-sweeps: the round keys depend on (seed, sample) only, the four words
// a, b, d, e on t as well.
ISING_HD void fold_philox_keys(uint64_t seed, uint32_t sample, PhiloxCommonConst *cc, PhiloxSampleConst *sc)
{
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32) ^ sample;
    for (int r = 3; r < 10; ++r) cc->k0[r - 3] = k0 + (uint32_t)r * PHILOX_W0;
    for (int r = 2; r < 10; ++r) sc->k1[r - 2] = k1 + (uint32_t)r * PHILOX_W1;
}
ISING_HD void fold_philox_time(uint64_t seed, uint32_t sample, uint64_t t, PhiloxCommonConst *cc, PhiloxSampleConst *sc)
{
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32) ^ sample;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);
    const uint64_t P0 = (uint64_t)PHILOX_M0 * tlo;
    const uint32_t A2 = (uint32_t)(P0 >> 32) ^ k1;
    const uint64_t B = (uint64_t)PHILOX_M1 * A2;
    cc->a = thi ^ k0;
    sc->b = (uint32_t)(B >> 32) ^ (k0 + PHILOX_W0);
    sc->d = (uint32_t)P0 ^ (k1 + PHILOX_W1);
    sc->e = (uint32_t)B ^ (k0 + 2u * PHILOX_W0);
}

ISING_HD void philox_folded(const PhiloxCommonConst &cc, const PhiloxSampleConst &sc, uint32_t g, uint32_t out[4])
{
    // round 0.  (Forming M1 * g for the calls of a thread as M1 * g_base + a compile-time constant turns 31 of 32 of these
    // multiplies into 64-bit adds; measured at L = 1024: 0.3912 against 0.3868 ms per half-sweep, two adds on the alu pipe cost
    // more than the multiply on the fma pipe they replace.  Not used.)
    const uint64_t Q = (uint64_t)PHILOX_M1 * g;
    // round 0
    uint32_t c0 = (uint32_t)(Q >> 32) ^ cc.a;
    // round 1
    const uint64_t P = (uint64_t)PHILOX_M0 * c0;
    c0 = (uint32_t)Q ^ sc.b;
    uint32_t c2 = (uint32_t)(P >> 32) ^ sc.d;
    // round 2
    const uint64_t P2 = (uint64_t)PHILOX_M0 * c0;
    const uint64_t Q2 = (uint64_t)PHILOX_M1 * c2;
    c0 = (uint32_t)(Q2 >> 32) ^ sc.e;
    uint32_t c1 = (uint32_t)Q2;
    c2 = (uint32_t)(P2 >> 32) ^ (uint32_t)P ^ sc.k1[0];
    uint32_t c3 = (uint32_t)P2;
    // rounds 3..9
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ cc.k0[r - 3];
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ sc.k1[r - 2];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ---------------------------------------------------------------------------------------------------
// MINSTD (Eq. 7: R <- 16807 R mod 2^31-1) with one stream per site (R11, R12).
// Stream q = sample*N + i.  Seed state s0 = (z >> 34) + 1 with z the (q+1)-th SplitMix64 output from `seed`;
// the draw of sweep n is R_n = 16807^(n+1) * s0 mod (2^31-1), evaluated statelessly with A = 16807^(n+1) mod M
// supplied by the host.  No PRNG state is ever stored.
// ---------------------------------------------------------------------------------------------------
constexpr uint64_t SPLITMIX_GAMMA = 0x9E3779B97F4A7C15ull;
constexpr uint32_t MINSTD_M = 2147483647u;

// w = seed + (q+1)*GAMMA, the SplitMix64 state whose finalised value is output number q+1.
ISING_HD uint32_t minstd_seed_state_from_weyl(uint64_t w)
{
    uint64_t z = w;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    // (z ^ (z >> 31)) >> 34 == z >> 34: the last xor-shift cannot reach the top 30 bits.
    return (uint32_t)(z >> 34) + 1u;
}

// A * s0 mod (2^31 - 1) for 1 <= A, s0 < 2^31 - 1, by folding the 62-bit product twice (2^31 = 1 mod M).
// The result is never 0 or M because M is prime, so no final conditional subtraction is needed:
// x1 = lo31 + (p >> 31) < 2^31 + 2^30 is either already in [1, M-1] or in [M+1, 2^31 + 2^30), and the second
// fold maps the latter to x1 - M.
ISING_HD uint32_t minstd_mulmod(uint32_t A, uint32_t s0)
{
    const uint64_t p = (uint64_t)A * s0;
    const uint32_t x1 = ((uint32_t)p & MINSTD_M) + (uint32_t)(p >> 31);
    return (x1 & MINSTD_M) + (x1 >> 31);
}

// The same with the multiplier doubled (A2 = 2A < 2^32): the 63-bit product 2*A*s0 has (A*s0) >> 31 in its high word
// and (A*s0) & M in bits 1..31 of its low word, so the first fold needs no funnel shift and no mask.
ISING_HD uint32_t minstd_mulmod2(uint32_t A2, uint32_t s0)
{
    const uint64_t p = (uint64_t)A2 * s0;
    const uint32_t x1 = ((uint32_t)p >> 1) + (uint32_t)(p >> 32);
    return (x1 & MINSTD_M) + (x1 >> 31);
}

ISING_HD uint32_t minstd_power(uint64_t n_plus_1)
{  // 16807^(n+1) mod M by square-and-multiply (host: once per sweep; device: graph_kernels.cuh, once per graph replay)
    uint64_t base = 16807u, acc = 1u, e = n_plus_1;
    while (e) {
        if (e & 1) acc = (acc * base) % MINSTD_M;
        base = (base * base) % MINSTD_M;
        e >>= 1;
    }
    return (uint32_t)acc;
}

}  // namespace isingk
