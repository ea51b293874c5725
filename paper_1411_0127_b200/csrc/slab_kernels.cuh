// slab_kernels.cuh -- z-slab domain decomposition (section V; Fig. 10, Fig. 11 PAPER.md:394;
// SURVEY.md 8(f) rank 3).  The lattice is cut along z into G slabs of Lz = L/G planes, one handle (one GPU) per slab.
//
// Storage of a slab: the same eight colour-separated bit arrays as the whole lattice (sweep_kernels.cuh), but with Lz + 2 planes:
// local plane 0 is a copy of the plane below the slab (lattice plane z0 - 1, periodic), local planes 1 .. Lz are the slab's own,
// local plane Lz + 1 is a copy of the plane above (z0 + Lz).  The word-parallel tile update runs unchanged on it (SLAB = true:
// z-neighbours are the planes below and above in the array, no wrap; colours, Philox counters and MINSTD stream ids use the
// plane's z in the lattice), so a slab's trajectory is bit-identical to the same planes of the undivided lattice.
//
// One colour half-sweep of a slab (the paper's Fig. 10, with a peer copy in place of D2H + MPI + H2D):
//   boundary launch   the CTA rows that hold the slab's first and last planes (8 planes each)         -- stream A
//   exchange          the updated colour's first owned plane -> upper halo of the slab below,
//                     its last owned plane -> lower halo of the slab above (L^2/16 bytes each: 64 KiB at L = 1024)  -- stream A
//   bulk launch       all other CTA rows, concurrently                                                  -- stream B
// With the standard checkerboard every plane holds both colours, so each colour update sends in both directions (PAPER.md:394:
// "two-ways for the standard implementation"; the paper's one-directional exchange is a property of its sliced layout).
// Couplings never move: the halo planes of the coupling arrays are filled once by the loader.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "layout_kernels.cuh"
#include "measure_kernels.cuh"
#include "sweep_kernels.cuh"

namespace isingk {

// grid = (L / (32 / tpr_pad), number of CTA rows of this launch); the CTA row is a.by_first + blockIdx.y * a.by_stride.
template <int RNG, int W, bool BIG = false>
__global__ void __launch_bounds__(SWEEP_THREADS)
half_sweep_site_packed_slab(const __grid_constant__ SweepArgs a, const __grid_constant__ SiteRng rng)
{
    unsigned long long unused0 = 0, unused1 = 0;
    site_packed_tile<RNG, W, false, false, true, BIG>(a, rng, blockIdx.x, (uint32_t)a.by_first + blockIdx.y * (uint32_t)a.by_stride, gridDim.x,
                                                 unused0, unused1);
}

// The same with the exchange fused into the kernel (SURVEY.md section 5 "direct remote stores into the neighbour's halo buffer"): the
// threads whose rows lie in the slab's first / last owned plane store their updated words a second time, into the upper halo of the
// slab below / the lower halo of the slab above -- plain stores to addresses that are valid on this device: the neighbour's workspace
// on the same GPU, or on a peer GPU mapped over NVLink (peer access / CUDA IPC), where they travel as the kernel runs instead of
// as a separate copy after it.  The words are read back from the thread's own store (L2, coherent load) so that the tile update of
// sweep_kernels.cuh stays as it is.  Nobody reads the halos of the ACTIVE colour during this half-sweep (z-neighbours are of the
// other colour), so the remote stores race with nothing; the next half-sweep must wait for this kernel on every slab, as it must
// for the copies.
struct SlabPush {
    uint32_t *dn, *up;   // active colour: upper halo plane of the slab below, lower halo plane of the slab above
    int Lz;
};

template <int RNG, int W, bool BIG = false>
__global__ void __launch_bounds__(SWEEP_THREADS)
half_sweep_site_packed_slab_push(const __grid_constant__ SweepArgs a, const __grid_constant__ SiteRng rng, const SlabPush p)
{
    unsigned long long unused0 = 0, unused1 = 0;
    const uint32_t by = (uint32_t)a.by_first + blockIdx.y * (uint32_t)a.by_stride;
    site_packed_tile<RNG, W, false, false, true, BIG>(a, rng, blockIdx.x, by, gridDim.x, unused0, unused1);
    const RowMap rm = row_map<W>(a.L, blockIdx.x, by);
    const int zl = rm.z + 1;   // plane in the slab's arrays (plane 0 is the lower halo)
    if (rm.active && (zl == 1 || zl == p.Lz)) {
        const uint32_t wpr = (uint32_t)a.L >> 6;
        const uint32_t in_plane = wpr * (uint32_t)rm.y + (uint32_t)rm.k0;
        uint32_t s[W];
        load_spin_words<W, true>(a.S_act, (size_t)wpr * (uint32_t)a.L * (uint32_t)zl + in_plane, s);
        if (zl == 1) store_words<W>(p.dn, in_plane, s);
        if (zl == p.Lz) store_words<W>(p.up, in_plane, s);
    }
}

// Unsatisfied bonds (+x, +y, +z bond of every owned site; the +z bond of the last owned plane reaches into the upper halo) and up
// spins of the slab's own planes, added to acc[0], acc[1]: the slab's share of E and M; the shares of all slabs add up to the
// lattice's (R16: E = 2 * unsatisfied - 3N, M = 2 * up - N).  grid = (L / (32 / tpr_pad), Lz / 8).
template <int W>
__global__ void __launch_bounds__(SWEEP_THREADS)
energy_site_packed_slab(const MeasureArgs a, int z0, unsigned long long *acc)
{
    const int L = a.L, wpr = L >> 6;
    const RowMap rm = row_map<W>(L, blockIdx.x, blockIdx.y);
    const int tpr = rm.tpr, y = rm.y, z = rm.z + 1, zg = rm.z + z0, k0 = rm.k0;
    const int yp = y + 1 == L ? 0 : y + 1;
    const uint32_t row = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * z) + k0;
    const uint32_t row_yp = (uint32_t)wpr * ((uint32_t)yp + (uint32_t)L * z) + k0;
    const uint32_t row_zp = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * (z + 1)) + k0;
    unsigned long long unsat = 0, up = 0;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        uint32_t s[W], o[W], oyp[W], ozp[W], jx[W], jy[W], jz[W];
        load_words<W>(a.S[c], row, s);
        load_words<W>(a.S[1 - c], row, o);
        load_words<W>(a.S[1 - c], row_yp, oyp);
        load_words<W>(a.S[1 - c], row_zp, ozp);
        load_words<W>(a.J[0][c], row, jx);
        load_words<W>(a.J[1][c], row, jy);
        load_words<W>(a.J[2][c], row, jz);
        const uint32_t xodd = (uint32_t)((y + zg + c) & 1);
        uint32_t edge = o[0];
        if (tpr > 1) edge = __shfl_sync(0xFFFFFFFFu, edge, rm.next_lane);
#pragma unroll
        for (int k = 0; k < W; ++k) {
            const uint32_t nx = __funnelshift_r(o[k], (k + 1 < W) ? o[(k + 1) % W] : edge, xodd);
            if (rm.active) {
                unsat += __popc(jx[k] ^ s[k] ^ nx) + __popc(jy[k] ^ s[k] ^ oyp[k]) + __popc(jz[k] ^ s[k] ^ ozp[k]);
                up += __popc(s[k]);
            }
        }
    }
    block_accumulate2(unsat, up, acc);
}

// Canonical arrays of the WHOLE lattice -> the slab's arrays (all Lz + 2 local planes, halos included), for `narrays` canonical bit
// arrays at once; one thread per internal word.  Local plane zl holds lattice plane (z0 - 1 + zl) mod L.
__global__ void __launch_bounds__(256) split_colours_slab(const __grid_constant__ SplitArgs a, int z0, int planes /* Lz + 2 */)
{
    const int L = a.L, wpr = L >> 6;
    const uint64_t n = (uint64_t)wpr * L * planes;
    const uint64_t widx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (widx >= n) return;
    const uint64_t r = widx / (unsigned)wpr;          // local row = y + L * zl
    const int k = (int)(widx - r * (unsigned)wpr);
    const int y = (int)(r % (unsigned)L), zl = (int)(r / (unsigned)L);
    const int zg = (z0 - 1 + zl + L) % L;
    const int p = (y + zg) & 1;
    const uint64_t cw = 2 * ((uint64_t)wpr * ((uint64_t)y + (uint64_t)L * zg) + k);   // the two canonical words of this internal word
    for (int q = 0; q < a.narrays; ++q) {
        const uint32_t c0 = __ldg(a.canon[q] + cw), c1 = __ldg(a.canon[q] + cw + 1);
        a.out[q][p][widx] = compress_even_bits(c0) | (compress_even_bits(c1) << 16);
        a.out[q][1 - p][widx] = compress_even_bits(c0 >> 1) | (compress_even_bits(c1 >> 1) << 16);
    }
}

// The slab's own planes -> their words of the canonical spin array of the whole lattice (the other words are not touched).
__global__ void __launch_bounds__(256)
merge_colours_slab(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon, int L, int z0, int Lz)
{
    const int wpr = L >> 6;
    const uint64_t n = (uint64_t)wpr * L * Lz;
    const uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    const uint64_t r = idx / (unsigned)wpr;            // y + L * (zl - 1)
    const int k = (int)(idx - r * (unsigned)wpr);
    const int y = (int)(r % (unsigned)L), zl = (int)(r / (unsigned)L) + 1, zg = z0 + zl - 1;
    const int p = (y + zg) & 1;
    const uint64_t widx = (uint64_t)wpr * ((uint64_t)y + (uint64_t)L * zl) + k;
    const uint32_t even = (p ? S1 : S0)[widx], odd = (p ? S0 : S1)[widx];
    const uint64_t cw = 2 * ((uint64_t)wpr * ((uint64_t)y + (uint64_t)L * zg) + k);
    canon[cw] = spread_to_even_bits(even) | (spread_to_even_bits(odd) << 1);
    canon[cw + 1] = spread_to_even_bits(even >> 16) | (spread_to_even_bits(odd >> 16) << 1);
}

}  // namespace isingk
