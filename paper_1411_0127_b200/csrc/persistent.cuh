// persistent.cuh -- many half-sweeps in ONE launch, for small lattices ("a CUDA graph or a persistent
// cooperative kernel is used for small L"; the paper's small-L saturation study).
//
// The paper launches two kernels per sweep.  On a B200 a half-sweep of a small lattice is 0.3-6 us of work, while a
// launch into a stream costs the host 2.35 us and any synchronisation that crosses the L2 about 1.4 us
// (profiles/r2j_launch_floor.md: a grid-wide release / acquire barrier over 148-296 co-resident CTAs 1.3-1.4 us, a flag handed from
// one CTA to its neighbours 1.45 us, a graph edge 0.5-0.9 us, a cluster barrier 0.23 us, a CTA barrier 0.02 us).  Two kernels:
//
// half_sweeps_on_chip<RNG> -- lattices of at most 1024 words per colour (every even L <= 40; config 1, L = 16).  ONE CTA stages
//   the eight bit arrays in shared memory, runs ALL half-sweeps of the call there with a CTA barrier between them (the bit-window
//   word update of half_sweep_site_packed_rows on shared-memory operands), computes the records (E, M per recorded half-sweep)
//   itself, and writes the spins back at the end: no launch, no L2 round trip between half-sweeps.
//
// persistent_site_packed<RNG, W, RECORDS> -- one-sample lattices with whole-word rows below L = 512, ON REQUEST only (kernel
//   choice 4).  A grid of co-resident CTAs (cudaLaunchCooperativeKernel) runs as a dataflow over TILES (the rows of one CTA of the
//   per-launch kernel): the update of a tile at half-sweep k + 1 reads only the tile itself and its four neighbours in the (y, z)
//   tile grid as half-sweep k left them, so
//   * every tile has an epoch counter in global memory = the number of half-sweeps it has completed in this launch;
//   * a CTA owns the tiles b, b + G, b + 2G, ... and walks over them half-sweep after half-sweep; before tile X of half-sweep k
//     it waits until the four neighbours of X show epoch >= k (ld.acquire.gpu): they have written what X reads now, and they have
//     finished reading the bits X overwrites now; after the tile it publishes epoch[X] = k + 1 (st.release.gpu behind a CTA barrier);
//   * neighbouring tiles never drift apart by more than one half-sweep, distant ones may, and nobody waits for the slowest CTA of
//     the grid (the boundary / bulk idea of the paper's section V, applied between the SMs of one GPU);
//   * the per-half-sweep constants (colour, operand arrays, Philox round constants, MINSTD multiplier) are recomputed on the device
//     from the half-sweep counter t0 + k; spins are read with ld.global.cg (the L2 is the point of coherence);
//   * recording half-sweeps use the MEASURE variant of the tile update and add their counts straight into the record: E[r] and M[r]
//     are pre-set to -3N and -N by init_records and receive 2 x (unsatisfied bonds) and 2 x (up spins) (R16) by one atomic pair
//     per CTA; nothing waits for a record.
//   Measured (profiles/r2n_small.md): never the fastest.  The flag latency is paid per tile and is as long as a launch: 2.3-2.6 us
//   per half-sweep at L = 64 and 128 where graph replays (graph_kernels.cuh) take 2.1-2.3 and the cluster-resident kernel (cluster_kernels.cuh) 0.9-1.2 at L = 64, 10.3 against
//   8.1 us at L = 256.  A first version with a grid-wide barrier per half-sweep was slower still, and the sample-packed variant of
//   the dataflow ran config 2 at 9.1 against 5.8 us per half-sweep and is not in the library.  The kernel is kept, tested, as the
//   reproducible record of that result.
// The results are bit-identical to one launch per half-sweep: the draws are keyed by (site, t), not by the thread mapping.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "measure_kernels.cuh"
#include "sweep_kernels.cuh"

namespace isingk {

// Wait until the neighbours of tile (bx, by) of a periodic gx x gy tile grid (epochs at `epoch`, row-major) have completed k
// half-sweeps.  Called by all threads of the CTA; k is CTA-uniform.
__device__ __forceinline__ void wait_for_neighbour_tiles(const unsigned int *epoch, uint32_t gx, uint32_t gy, uint32_t bx, uint32_t by,
                                                         uint32_t k)
{
    if (k != 0 && threadIdx.x < 4) {
        uint32_t nx = bx, ny = by;
        if (threadIdx.x == 0) nx = bx + 1 == gx ? 0 : bx + 1;
        else if (threadIdx.x == 1) nx = bx == 0 ? gx - 1 : bx - 1;
        else if (threadIdx.x == 2) ny = by + 1 == gy ? 0 : by + 1;
        else ny = by == 0 ? gy - 1 : by - 1;
        const unsigned int *p = epoch + (size_t)ny * gx + nx;
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        } while ((int)(v - k) < 0);
    }
    __syncthreads();   // the acquires above are ordered before every thread's loads of this tile
}

// The tile is done: all stores of the CTA are ordered before the epoch by the CTA barrier and the release.
__device__ __forceinline__ void publish_tile(unsigned int *epoch_of_tile, uint32_t value)
{
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(epoch_of_tile), "r"(value) : "memory");
}

struct PersistArgs {
    LatticeArrays A;            // the 8 bit arrays of the lattice
    int L;
    Thresholds T;
    uint64_t seed;
    uint64_t t0;                // half-sweep counter of the first half-sweep of this launch
    uint32_t nhalf;             // half-sweeps to run
    uint32_t every;             // record E / M after every `every`-th half-sweep of this launch (0: never)
    uint32_t A_first;           // MINSTD: 16807^(n+1) mod M for the sweep n = t0 >> 1
    uint4 *s0tab[2];            // MINSTD with cached seed states: the tables of the two colours (else null)
    unsigned int *epoch;        // one counter per tile, zero on entry
    long long *E, *M;           // records r = 0, 1, ...: E[r], M[r] (either may be null); persistent_site_packed: pre-set by init_records
    uint64_t N;                 // sites
};

// Site-packed, L a multiple of 64 (the word-parallel tile update of sweep_kernels.cuh), RNG 0 = Philox, 1 = MINSTD stateless,
// 2 = MINSTD with the seed table.  grid = co-resident CTAs <= tiles; gx x gy tiles per half-sweep.  RECORDS = false leaves the
// measuring variant of the tile update out of the kernel (fewer registers, more resident CTAs).
template <int RNG, int W, bool RECORDS>
__global__ void __launch_bounds__(SWEEP_THREADS)
persistent_site_packed(const __grid_constant__ PersistArgs p, uint32_t gx, uint32_t gy)
{
    uint32_t rec = 0;
    uint32_t A = p.A_first;
    const uint32_t ntiles = gx * gy;
    for (uint32_t k = 0; k < p.nhalf; ++k) {
        const uint64_t t = p.t0 + k;
        const int c = (int)(t & 1);
        SweepArgs a;
        a.S_act = p.A.S[c];
        a.S_oth = p.A.S[1 - c];
#pragma unroll
        for (int d = 0; d < 3; ++d) { a.J_act[d] = p.A.J[d][c]; a.J_oth[d] = p.A.J[d][1 - c]; }
        a.L = p.L;
        a.colour = c;
        a.T = p.T;
        SiteRng sr;
        sr.seed = p.seed;
        sr.A2 = 2u * A;
        sr.s0tab = p.s0tab[c];
        if (RNG == 0) fold_philox(p.seed, 0u, t, &sr.pc, &sr.ps);
        const bool record = RECORDS && p.every != 0 && (k + 1) % p.every == 0;
        unsigned long long unsat = 0, up = 0;
        for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const uint32_t by = tile / gx, bx = tile - by * gx;
            wait_for_neighbour_tiles(p.epoch, gx, gy, bx, by, k);
            if (RECORDS && record) site_packed_tile<RNG, W, true, true>(a, sr, bx, by, gx, unsat, up);
            else site_packed_tile<RNG, W, false, true>(a, sr, bx, by, gx, unsat, up);
            publish_tile(p.epoch + tile, k + 1);
        }
        if (RECORDS && record) {
            add_to_record(unsat, up, p.E ? p.E + rec : nullptr, p.M ? p.M + rec : nullptr);
            ++rec;
        }
        if (RNG != 0 && c == 1) A = minstd_mulmod(16807u, A);   // the next half-sweep belongs to the next sweep: 16807^(n+2)
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// One CTA, the whole lattice in shared memory, all half-sweeps of the call (see the head of this file).  Any even L with
// n_words = ceil(L^3 / 64) <= ONCHIP_MAX_WORDS.  Dynamic shared memory: 8 arrays of `stride` = n_words + 1 words (the bit windows
// read one word past their last one), in the order S[0], S[1], Jx[0], Jx[1], Jy[0], Jy[1], Jz[0], Jz[1] of LatticeArrays.
// RNG 0 = Philox, 1 = MINSTD (stateless: SplitMix64 seed state per site and draw, R11, R12).
// ---------------------------------------------------------------------------------------------------------------------
constexpr uint32_t ONCHIP_MAX_WORDS = 1024;
constexpr int ONCHIP_THREADS = 512;

template <int RNG>
__global__ void __launch_bounds__(ONCHIP_THREADS)
half_sweeps_on_chip(const __grid_constant__ PersistArgs p, uint32_t n_words, uint32_t Hc)
{
    extern __shared__ uint32_t sm[];
    __shared__ unsigned long long cta_sum[2];
    const uint32_t stride = n_words + 1;
    // array (kind, colour) at sm + (2 * kind + colour) * stride, kind 0 = spins, 1 + d = couplings of direction d: pointer
    // arithmetic, not pointer tables, so that nothing is indexed at run time out of local memory
    for (uint32_t w = threadIdx.x; w < stride; w += ONCHIP_THREADS) {
        const bool in = w < n_words;
        sm[w] = in ? p.A.S[0][w] : 0u;
        sm[stride + w] = in ? p.A.S[1][w] : 0u;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            sm[(size_t)(2 + 2 * d) * stride + w] = in ? p.A.J[d][0][w] : 0u;
            sm[(size_t)(3 + 2 * d) * stride + w] = in ? p.A.J[d][1][w] : 0u;
        }
    }
    __syncthreads();
    uint32_t rec = 0, A = p.A_first;
    MeasureArgs m;
    m.L = p.L;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        m.S[c] = sm + (size_t)c * stride;
#pragma unroll
        for (int d = 0; d < 3; ++d) m.J[d][c] = sm + (size_t)(2 + 2 * d + c) * stride;
    }
    for (uint32_t k = 0; k < p.nhalf; ++k) {
        const uint64_t t = p.t0 + k;
        const int c = (int)(t & 1);
        SweepArgs a;
        a.S_act = sm + (size_t)c * stride;
        a.S_oth = sm + (size_t)(1 - c) * stride;
#pragma unroll
        for (int d = 0; d < 3; ++d) { a.J_act[d] = sm + (size_t)(2 + 2 * d + c) * stride; a.J_oth[d] = sm + (size_t)(3 + 2 * d - c) * stride; }
        a.L = p.L;
        a.colour = c;
        a.T = p.T;
        SiteRng sr;
        sr.seed = p.seed;
        sr.A2 = 2u * A;
        sr.s0tab = nullptr;
        if (RNG == 0) fold_philox(p.seed, 0u, t, &sr.pc, &sr.ps);
        // a thread writes only its own words of the active colour and reads the other colour and the couplings: in place
        for (uint32_t w = threadIdx.x; w < n_words; w += ONCHIP_THREADS) a.S_act[w] = rows_word_update<RNG, true, false>(a, sr, w, Hc);
        __syncthreads();
        if (p.every != 0 && (k + 1) % p.every == 0) {
            unsigned long long unsat = 0, up = 0;
            if (threadIdx.x == 0) { cta_sum[0] = 0; cta_sum[1] = 0; }
            for (uint32_t item = threadIdx.x; item < 2 * n_words; item += ONCHIP_THREADS) rows_energy_item<true>(m, item, n_words, Hc, unsat, up);
            __syncthreads();
            block_accumulate2(unsat, up, cta_sum);   // (has a CTA barrier inside; warp 0 adds to cta_sum)
            if (threadIdx.x == 0) {
                if (p.E) p.E[rec] = 2 * (long long)cta_sum[0] - 3 * (long long)p.N;   // R16
                if (p.M) p.M[rec] = 2 * (long long)cta_sum[1] - (long long)p.N;
            }
            ++rec;
        }
        if (RNG != 0 && c == 1) A = minstd_mulmod(16807u, A);
    }
    for (uint32_t w = threadIdx.x; w < n_words; w += ONCHIP_THREADS) {
        p.A.S[0][w] = sm[w];
        p.A.S[1][w] = sm[stride + w];
    }
}

}  // namespace isingk
