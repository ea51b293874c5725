// update.cuh -- the word-wise Metropolis update: bond bits, bit-sliced adder, per-bit acceptance masks, flip mask
// (SURVEY.md 8(a) rows a4, a5, a7, a8).  __host__ __device__ so that ising_hostcheck_update_word runs the same code.
#pragma once
#include <stdint.h>

#include "rng.cuh"

namespace isingk {

// Acceptance thresholds as the kernels use them ("EXP4, EXP8, EXP12"; R4-R6).
// Philox: accept dE iff R < T[dE] with T in [0, 2^32]; T = 2^32 does not fit a 32-bit compare, so the table holds
// min(T, 2^32-1) plus an all-ones "always" mask for T = 2^32 (beta = 0).  MINSTD: T in [0, 2^31-1], plain compare.
struct Thresholds {
    uint32_t t4, t8, t12;
    uint32_t always4, always8, always12;  // 0 or 0xFFFFFFFF
};

// Per-bit number n of SATISFIED bonds among the six of each site (R2), as three bit planes (Eq. 12-13,
// PAPER.md:258-271).  b_k = J_k ^ s_k ^ s is the bond bit of Eq. 11; under the encoding of Eq. 10 it
// marks an UNSATISFIED bond, so a_k = ~b_k is summed.  Two full adders, a half adder and a full adder.  Written with
// three-input functions throughout so that every line is one LOP3: 6 bond bits + 8 adder ops.
ISING_HD void satisfied_bond_count(uint32_t s, const uint32_t J[6], const uint32_t nb[6], uint32_t &sum2, uint32_t &sum1,
                                   uint32_t &sum0)
{
    const uint32_t a0 = ~(J[0] ^ nb[0] ^ s), a1 = ~(J[1] ^ nb[1] ^ s), a2 = ~(J[2] ^ nb[2] ^ s);
    const uint32_t a3 = ~(J[3] ^ nb[3] ^ s), a4 = ~(J[4] ^ nb[4] ^ s), a5 = ~(J[5] ^ nb[5] ^ s);
    const uint32_t sA = a0 ^ a1 ^ a2, cA = (a0 & a1) | (a2 & (a0 | a1));
    const uint32_t sB = a3 ^ a4 ^ a5, cB = (a3 & a4) | (a5 & (a3 | a4));
    sum0 = sA ^ sB;
    const uint32_t cC = sA & sB;
    sum1 = cA ^ cB ^ cC;
    sum2 = (cA & cB) | (cC & (cA | cB));
}

// Flip mask, Eq. 16-17 (Eq. 17 itself is lost in the text and reconstructed from the prose, R1):
// n <= 3 (sum2 = 0, dE <= 0) always flips; n = 4, 5, 6 (dE = 4, 8, 12) flip where cond4, cond8, cond12 is set.
// Here the cond masks are per bit (every site has its own draw) instead of the paper's all-or-nothing words (Eq. 15).
ISING_HD uint32_t flip_mask(uint32_t sum2, uint32_t sum1, uint32_t sum0, uint32_t cond4, uint32_t cond8, uint32_t cond12)
{
    return cond12 | ~sum2 | (sum2 & (sum2 ^ sum1) & (cond8 | (cond4 & ~sum0)));
}

// acc |= bit where R < T: one compare and one predicated OR, both on the integer ALU.
ISING_HD void or_if_lt(uint32_t &acc, uint32_t R, uint32_t T, uint32_t bit)
{
#ifdef __CUDA_ARCH__
    asm("{ .reg .pred p; setp.lt.u32 p, %1, %2; @p or.b32 %0, %0, %3; }" : "+r"(acc) : "r"(R), "r"(T), "r"(bit));
#else
    if (R < T) acc |= bit;
#endif
}

ISING_HD uint32_t min_u32(uint32_t a, uint32_t b) { return a < b ? a : b; }

// Acceptance bits of NR draws for the sites bit0 .. bit0+NR-1 of a word.  cond4 is needed for every draw.  R < T8
// happens for < 0.1 % of the draws at the temperatures of interest, so cond8 / cond12 are filled in a rarely taken,
// warp-uniform branch guarded by the minimum of the draws (one VIMNMX3 per two draws).
// VOTE = false: the rare branch is taken per thread (for callers whose warps are not converged here, e.g. inside a loop
// with a per-thread trip count, where a full-mask vote would be undefined).
template <int NR, bool VOTE = true>
ISING_HD void accumulate_cond(const uint32_t *R, int bit0, const Thresholds &T, uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    uint32_t mn = 0xFFFFFFFFu;
#pragma unroll
    for (int w = 0; w < NR; ++w) {
        or_if_lt(c4, R[w], T.t4, 1u << (bit0 + w));
        mn = min_u32(mn, R[w]);
    }
#ifdef __CUDA_ARCH__
    if (VOTE ? __any_sync(0xFFFFFFFFu, mn < T.t8) != 0 : mn < T.t8) {
#else
    if (mn < T.t8) {
#endif
#pragma unroll
        for (int w = 0; w < NR; ++w) or_if_lt(c8, R[w], T.t8, 1u << (bit0 + w));
#ifdef __CUDA_ARCH__
        if (VOTE ? __any_sync(0xFFFFFFFFu, mn < T.t12) != 0 : mn < T.t12) {
#else
        if (mn < T.t12) {
#endif
#pragma unroll
            for (int w = 0; w < NR; ++w) or_if_lt(c12, R[w], T.t12, 1u << (bit0 + w));
        }
    }
}

ISING_HD void finish_cond(const Thresholds &T, uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    c4 |= T.always4;
    c8 |= T.always8;
    c12 |= T.always12;
}

// Site-packed word (bits = 32 consecutive sites of one colour of one lattice): colour rank of bit b is
// j = 32*word_index + b, so Philox call q = 0..7 has counter g = 8*word_index + q and serves bits 4q..4q+3 (R9).
// Two calls are generated together: four independent multiply chains hide the IMAD.WIDE latency at any occupancy.
template <bool VOTE = true>
ISING_HD void cond_masks_site_packed_philox(const PhiloxCommonConst &cc, const PhiloxSampleConst &sc, uint32_t word_index,
                                            const Thresholds &T, uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    c4 = 0; c8 = 0; c12 = 0;
    const uint32_t g0 = 8u * word_index;
#pragma unroll
    for (int q = 0; q < 8; q += 2) {
        uint32_t R[8];
        philox_folded(cc, sc, g0 + (uint32_t)q, R);
        philox_folded(cc, sc, g0 + (uint32_t)q + 1u, R + 4);
        accumulate_cond<8, VOTE>(R, 4 * q, T, c4, c8, c12);
    }
    finish_cond(T, c4, c8, c12);
}

// MINSTD, site-packed word: the stream id of bit b is q_b = site0 + b*site_stride (canonical site index, sample 0),
// i.e. the SplitMix64 Weyl state advances by site_stride*GAMMA per bit.  `weyl0` = seed + (site0+1)*GAMMA.
template <bool VOTE = true>
ISING_HD void cond_masks_site_packed_minstd(uint64_t weyl0, uint64_t weyl_step, uint32_t A2, const Thresholds &T,
                                            uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    c4 = 0; c8 = 0; c12 = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        uint32_t R[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) R[w] = minstd_mulmod2(A2, minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + w) * weyl_step));
        accumulate_cond<4, VOTE>(R, 4 * q, T, c4, c8, c12);
    }
    finish_cond(T, c4, c8, c12);
}

// The same for a word whose bits 0..k-1 and k..31 lie in two different rows (general L): bit b uses the Weyl state
// (b < k ? weylA : weylB) + b * weyl_step, where weylA / weylB are referred to bit 0 of the word.
ISING_HD void cond_masks_site_packed_minstd_two(uint64_t weylA, uint64_t weylB, uint32_t k, uint64_t weyl_step, uint32_t A2,
                                                const Thresholds &T, uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    c4 = 0; c8 = 0; c12 = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        uint32_t R[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t b = (uint32_t)(4 * q + w);
            R[w] = minstd_mulmod2(A2, minstd_seed_state_from_weyl((b < k ? weylA : weylB) + (uint64_t)b * weyl_step));
        }
        accumulate_cond<4>(R, 4 * q, T, c4, c8, c12);
    }
    finish_cond(T, c4, c8, c12);
}

}  // namespace isingk
