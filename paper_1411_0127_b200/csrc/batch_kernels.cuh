// batch_kernels.cuh -- many disorder samples with their OWN random numbers as a batch of site-packed lattices
// (multispin coding over the sites of one sample, "SMSC", against coding over samples, "AMSC"; PAPER.md:151-153,
// 308-310: many small systems in one launch to fill the GPU).
//
// With one draw per (sample, site, half-sweep) (R9, R11) the samples of a handle share nothing: sample s of a Philox handle is
// exactly the one-sample lattice with the key word k1 ^ s (R9), sample s of a MINSTD handle exactly the one-sample lattice whose
// SplitMix64 seed is advanced by s N steps (stream q = s N + i, R11: seed + (q + 1) GAMMA = (seed + s N GAMMA) + (i + 1) GAMMA).
// Storing such samples bit-interleaved (32 samples per word, the paper's AMSC storage) buys nothing -- there is no shared draw to
// amortise -- and costs a thread 32 different sets of Philox constants (measured: 0.78-0.84 against 0.72 ps per flip attempt at the
// large sizes, 6.2 against about 4 us per half-sweep for 32 samples of L = 64).  So for nsamples = 32k, rng modes 0 and 1 and L a
// multiple of 64 the internal layout is nsamples site-packed lattices one after the other (the eight colour arrays of sample s at
// s * lattice_stride), and every kernel of the one-sample path runs on all of them in one launch with blockIdx.z = sample: the word-
// parallel tile update, its measuring variant (the records E[r * nsamples + s] receive their counts by atomics), the fused energy
// kernel, the colour split / merge, the MINSTD seed table.  The canonical format at the boundary (ising.h) is per sample already.
// The shared-draw modes 2-4 keep the sample-packed arrays: there one draw serves the 32 samples of a word, which is the point of AMSC.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "measure_kernels.cuh"
#include "sweep_kernels.cuh"

namespace isingk {

struct BatchInfo {
    size_t lattice_stride;   // words between the arrays of consecutive samples (8 arrays of one lattice)
    size_t tab_stride;       // MINSTD seed table: uint4 elements per sample and colour
    uint64_t N;              // sites of one lattice
    uint64_t t;              // half-sweep counter of this launch
    uint32_t nsamples;
    uint32_t sample0;        // sample of blockIdx.z = 0 (launches are cut at 65535 samples)
};

// The operands and generator constants of sample s from those of sample 0.  Everything here is CTA-uniform.
__device__ __forceinline__ SweepArgs sample_operands(const SweepArgs &a0, size_t off)
{
    SweepArgs a = a0;
    a.S_act = a0.S_act + off;
    a.S_oth = a0.S_oth + off;
#pragma unroll
    for (int d = 0; d < 3; ++d) { a.J_act[d] = a0.J_act[d] + off; a.J_oth[d] = a0.J_oth[d] + off; }
    return a;
}

template <int RNG>
__device__ __forceinline__ SiteRng sample_generator(const SiteRng &r0, const BatchInfo &b, uint32_t s)
{
    SiteRng r = r0;
    if (RNG == 0) fold_philox(r0.seed, s, b.t, &r.pc, &r.ps);                    // key (k0, k1 ^ s)  (R9)
    else r.seed = r0.seed + (uint64_t)s * b.N * SPLITMIX_GAMMA;                  // streams s N .. s N + N - 1  (R11)
    if (RNG == 2) r.s0tab = r0.s0tab + (size_t)s * b.tab_stride;
    return r;
}

// grid = (L / (32 / tpr_pad), L / 8, samples of this launch), as half_sweep_site_packed.  MEASURE: E / M point at the record's first
// sample; sample s adds to E[s], M[s] (pre-set to -3N, -N by init_records).
template <int RNG, int W, bool MEASURE>
__global__ void __launch_bounds__(SWEEP_THREADS, RNG == 0 && W == 4 && !MEASURE ? 4 : 0)
half_sweep_site_packed_batch(const __grid_constant__ SweepArgs a0, const __grid_constant__ SiteRng rng0, const __grid_constant__ BatchInfo b,
                             long long *E, long long *M)
{
    const uint32_t s = b.sample0 + blockIdx.z;
    const SweepArgs a = sample_operands(a0, (size_t)s * b.lattice_stride);
    const SiteRng rng = sample_generator<RNG>(rng0, b, s);
    unsigned long long unsat = 0, up = 0;
    site_packed_tile<RNG, W, MEASURE, false>(a, rng, blockIdx.x, blockIdx.y, gridDim.x, unsat, up);
    if (MEASURE) add_to_record(unsat, up, E ? E + s : nullptr, M ? M + s : nullptr);
}

// The seed tables of all samples, colour `colour` (thread mapping of minstd_fill_s0).
template <int W>
__global__ void __launch_bounds__(SWEEP_THREADS) minstd_fill_s0_batch(uint4 *tab, int L, int colour, uint64_t seed, BatchInfo b)
{
    const uint32_t s = b.sample0 + blockIdx.z;
    const RowMap rm = row_map<W>(L, blockIdx.x, blockIdx.y);
    const int lane = rm.lane, warp = rm.warp, y = rm.y, z = rm.z, k0 = rm.k0;
    const int xodd = (y + z + colour) & 1;
    const uint64_t row_site0 = (uint64_t)s * b.N + (uint64_t)L * ((uint64_t)y + (uint64_t)L * z) + (uint64_t)xodd;
    const uint32_t warp_global = (blockIdx.y * gridDim.x + blockIdx.x) * (SWEEP_THREADS / 32) + warp;
    uint4 *out = tab + (size_t)s * b.tab_stride;
#pragma unroll 1
    for (int k = 0; k < W; ++k) {
        const uint64_t weyl0 = seed + (row_site0 + 64ull * (uint64_t)(k0 + k) + 1) * SPLITMIX_GAMMA;
#pragma unroll 1
        for (int q = 0; q < 8; ++q) {
            uint4 v;
            v.x = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 0) * (2 * SPLITMIX_GAMMA));
            v.y = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 1) * (2 * SPLITMIX_GAMMA));
            v.z = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 2) * (2 * SPLITMIX_GAMMA));
            v.w = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 3) * (2 * SPLITMIX_GAMMA));
            __stcs(out + minstd_s0_index<W>(warp_global, k, q, lane), v);
        }
    }
}

// E[s], M[s] of every sample in one launch: the tile counts of energy_site_packed, added to the pre-set E[s] = -3N, M[s] = -N (R16).
template <int W>
__global__ void __launch_bounds__(SWEEP_THREADS)
energy_site_packed_batch(const MeasureArgs a0, BatchInfo b, long long *E, long long *M)
{
    const uint32_t s = b.sample0 + blockIdx.z;
    const size_t off = (size_t)s * b.lattice_stride;
    MeasureArgs a = a0;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        a.S[c] = a0.S[c] + off;
#pragma unroll
        for (int d = 0; d < 3; ++d) a.J[d][c] = a0.J[d][c] + off;
    }
    unsigned int unsat, up;
    energy_tile<W>(a, blockIdx.x, blockIdx.y, unsat, up);
    add_to_record(unsat, up, E ? E + s : nullptr, M ? M + s : nullptr);
}

// Overlap of two samples (replicas): q = N - 2 D, D = differing spins = popcount of the XOR of their spin arrays.
// Sa / Sb: colour-0 arrays of the two lattices; the colour-1 arrays follow at `colour_stride` words.  *cnt zero on entry.
__global__ void __launch_bounds__(256)
overlap_site_packed(const uint32_t *__restrict__ Sa, const uint32_t *__restrict__ Sb, size_t colour_stride, uint32_t n_words,
                    unsigned long long *cnt)
{
    unsigned long long d = 0, unused = 0;
    for (uint32_t w = blockIdx.x * 256u + threadIdx.x; w < n_words; w += gridDim.x * 256u)
        d += __popc(__ldg(Sa + w) ^ __ldg(Sb + w)) + __popc(__ldg(Sa + colour_stride + w) ^ __ldg(Sb + colour_stride + w));
    block_accumulate2(d, unused, cnt);
}

}  // namespace isingk
