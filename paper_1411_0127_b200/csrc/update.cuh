// update.cuh -- the word-wise Metropolis update: bond bits, bit-sliced adder, per-bit acceptance masks, flip mask
// (SURVEY.md 8(a) rows a4, a5, a7, a8).  __host__ __device__ so that ising_hostcheck_update_word runs the same code.
#pragma once
#include <stdint.h>

#include "rng.cuh"

namespace isingk {

// Acceptance thresholds as the kernels use them ("EXP4, EXP8, EXP12"; R4-R6).
// Philox: accept dE iff R < T[dE] with T in [0, 2^32]; T = 2^32 does not fit a 32-bit compare, so the table holds
// min(T, 2^32-1) plus an all-ones "always" mask for T = 2^32 (beta = 0).  MINSTD: T in [0, 2^31-1], plain compare.
// For dE = 4, the test every site needs, the table also holds k4 = (2^32 - T4) mod 2^32: the 33-bit sum R + k4 carries
// into bit 32 exactly when R >= T4 (for T4 = 2^32 it never does; for T4 = 0 the carry is lost, hence `never4`).
struct Thresholds {
    uint32_t t4, t8, t12;
    uint32_t always4, always8, always12;  // 0 or 0xFFFFFFFF
    uint32_t k4;
    uint32_t never4;  // 0xFFFFFFFF iff T4 = 0 (beta = infinity)
};

// Per-bit number n of SATISFIED bonds among the six of each site (R2), as three bit planes (Eq. 12-13,
// PAPER.md:258-271).  u_k = J_k ^ s_k is the neighbour part of the bond bit of Eq. 11;
// J ^ s_i ^ s_k = 1 marks an unsatisfied bond under the encoding of Eq. 10, so a_k = ~(u_k ^ s) counts satisfied ones.
// Two full adders, a half adder and a full adder: 8 three-input logic ops on top of the 6 bond XORs.
ISING_HD void satisfied_bond_count(uint32_t s, const uint32_t u[6], uint32_t &sum2, uint32_t &sum1, uint32_t &sum0)
{
    const uint32_t a0 = ~(u[0] ^ s), a1 = ~(u[1] ^ s), a2 = ~(u[2] ^ s);
    const uint32_t a3 = ~(u[3] ^ s), a4 = ~(u[4] ^ s), a5 = ~(u[5] ^ s);
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

// 2*acc + (R >= T4): shifts the next "not accepted at dE = 4" bit into the accumulator.  On the device this is a carry
// chain of two instructions: IADD3 (R + k4, carry out = R >= T4) and an add-with-carry acc + acc + C, which ptxas is
// free to issue as IMAD.X on the FMA pipe, off the ALU pipe that the Philox XORs load.
ISING_HD uint32_t shift_in_ge(uint32_t acc, uint32_t R, const Thresholds &T)
{
#ifdef __CUDA_ARCH__
    uint32_t out;
    asm("{ .reg .u32 t; add.cc.u32 t, %1, %2; addc.u32 %0, %3, %3; }" : "=r"(out) : "r"(R), "r"(T.k4), "r"(acc));
    return out;
#else
    const uint64_t t = (uint64_t)R + T.k4;
    return 2u * acc + (uint32_t)(t >> 32);
#endif
}

// The acceptance bits of four draws (sites bit0+3 .. bit0, in this order, so that shifting left leaves site b at bit b
// once all 32 sites of a word have been shifted in from the top bit down).  nc4 collects R >= T4 (the complement of
// cond4).  R < T8 happens for < 0.1 % of the draws at the temperatures of interest, so cond8 / cond12 are filled in a
// rarely taken branch guarded by the minimum of the four draws.
ISING_HD void accumulate_cond(const uint32_t R[4], int bit0, const Thresholds &T, uint32_t &nc4, uint32_t &c8, uint32_t &c12)
{
#pragma unroll
    for (int w = 3; w >= 0; --w) nc4 = shift_in_ge(nc4, R[w], T);
    uint32_t mn = R[0] < R[1] ? R[0] : R[1];
    const uint32_t mn2 = R[2] < R[3] ? R[2] : R[3];
    mn = mn < mn2 ? mn : mn2;
#ifdef __CUDA_ARCH__
    if (__any_sync(0xFFFFFFFFu, mn < T.t8)) {
#else
    if (mn < T.t8) {
#endif
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            c8 |= (R[w] < T.t8 ? 1u : 0u) << (bit0 + w);
            c12 |= (R[w] < T.t12 ? 1u : 0u) << (bit0 + w);
        }
    }
}

ISING_HD void finish_cond(const Thresholds &T, uint32_t nc4, uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    c4 = ~(nc4 | T.never4);
    c8 |= T.always8;
    c12 |= T.always12;
}

// Site-packed word (bits = 32 consecutive sites of one colour of one lattice): colour rank of bit b is
// j = 32*word_index + b, so Philox call q = 0..7 has counter g = 8*word_index + q and serves bits 4q..4q+3 (R9).
ISING_HD void cond_masks_site_packed_philox(const PhiloxCommonConst &cc, const PhiloxSampleConst &sc, uint32_t word_index,
                                            const Thresholds &T, uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    uint32_t nc4 = 0;
    c8 = 0; c12 = 0;
#pragma unroll
    for (int q = 7; q >= 0; --q) {
        uint32_t R[4];
        philox_folded(cc, sc, 8u * word_index + (uint32_t)q, R);
        accumulate_cond(R, 4 * q, T, nc4, c8, c12);
    }
    finish_cond(T, nc4, c4, c8, c12);
}

// MINSTD, site-packed word: the stream id of bit b is q_b = site0 + b*site_stride (canonical site index, sample 0),
// i.e. the SplitMix64 Weyl state advances by site_stride*GAMMA per bit.  `weyl0` = seed + (site0+1)*GAMMA.
ISING_HD void cond_masks_site_packed_minstd(uint64_t weyl0, uint64_t weyl_step, uint32_t A, const Thresholds &T,
                                            uint32_t &c4, uint32_t &c8, uint32_t &c12)
{
    uint32_t nc4 = 0;
    c8 = 0; c12 = 0;
#pragma unroll
    for (int q = 7; q >= 0; --q) {
        uint32_t R[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) R[w] = minstd_mulmod(A, minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + w) * weyl_step));
        accumulate_cond(R, 4 * q, T, nc4, c8, c12);
    }
    finish_cond(T, nc4, c4, c8, c12);
}

}  // namespace isingk
