// measure_kernels.cuh -- energy and magnetisation.
//
//   E = - sum over the 3N bonds of J sigma sigma (Eq. 1, each bond once).  With the encoding of Eq. 10 the
//   bond bit e = J ^ s_i ^ s_k (Eq. 11) is 1 exactly when -J sigma_i sigma_k = +1, so E = 2*popc(e over all bonds) - 3N,
//   and M = 2*popc(s) - N.  The kernels accumulate the two popcounts per sample into uint64 counters (warp shuffle
//   reduction, one atomic per warp); finalize_energy turns them into int64 E and M.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sweep_kernels.cuh"

namespace isingk {

struct MeasureArgs {
    const uint32_t *S[2];
    const uint32_t *J[3][2];
    int L;
};

__device__ __forceinline__ void warp_reduce_add2(unsigned long long &a, unsigned long long &b)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_down_sync(0xFFFFFFFFu, a, off);
        b += __shfl_down_sync(0xFFFFFFFFu, b, off);
    }
}

// Block-level sum of two counters, then one atomic pair per block.
__device__ __forceinline__ void block_accumulate2(unsigned long long a, unsigned long long b, unsigned long long *acc)
{
    __shared__ unsigned long long sh[2][32];
    warp_reduce_add2(a, b);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sh[0][warp] = a; sh[1][warp] = b; }
    __syncthreads();
    if (warp == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        a = lane < nw ? sh[0][lane] : 0;
        b = lane < nw ? sh[1][lane] : 0;
        warp_reduce_add2(a, b);
        if (lane == 0) {
            atomicAdd(&acc[0], a);
            atomicAdd(&acc[1], b);
        }
    }
}

// Site-packed, L = 64*2^k: a grid-stride loop over the words of both colours.  The +x neighbour of the colour-c site
// with bit m is bit m (xodd = 0) or bit m+1 (xodd = 1) of the other colour's half-row; +y / +z neighbours are the same
// bit one row up.  Every word is read once from HBM (the neighbour reads hit L1/L2): 512 MiB at L = 1024.
__global__ void __launch_bounds__(256)
energy_site_packed(const MeasureArgs a, unsigned long long *acc /* [0] = unsatisfied bonds, [1] = up spins */)
{
    const int L = a.L, wpr = L >> 6;
    const uint64_t words_per_colour = (uint64_t)wpr * L * L;
    unsigned long long unsat = 0, up = 0;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const uint32_t *__restrict__ Sc = a.S[c], *__restrict__ So = a.S[1 - c];
        const uint32_t *__restrict__ Jx = a.J[0][c], *__restrict__ Jy = a.J[1][c], *__restrict__ Jz = a.J[2][c];
        for (uint64_t widx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; widx < words_per_colour;
             widx += (uint64_t)gridDim.x * blockDim.x) {
            const int k = (int)(widx % wpr);
            const uint64_t r = widx / wpr;
            const int y = (int)(r % L), z = (int)(r / L);
            const int yp = (y + 1) & (L - 1), zp = (z + 1) & (L - 1);
            const int xodd = (y + z + c) & 1;
            const uint32_t s = Sc[widx];
            const size_t rowbase = (size_t)wpr * r;
            uint32_t nx = So[rowbase + k];
            if (xodd) nx = __funnelshift_r(nx, So[rowbase + ((k + 1) % wpr)], 1);
            const uint32_t ny = So[(size_t)wpr * ((size_t)yp + (size_t)L * z) + k];
            const uint32_t nz = So[(size_t)wpr * ((size_t)y + (size_t)L * zp) + k];
            unsat += __popc(Jx[widx] ^ s ^ nx) + __popc(Jy[widx] ^ s ^ ny) + __popc(Jz[widx] ^ s ^ nz);
            up += __popc(s);
        }
    }
    block_accumulate2(unsat, up, acc);
}

// Site-packed, any even L: one thread per word, one site at a time.
__global__ void __launch_bounds__(256)
energy_site_packed_generic(const MeasureArgs a, unsigned long long *acc, uint64_t n_words, uint64_t Hc)
{
    const int L = a.L, H = L >> 1;
    const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long unsat = 0, up = 0;
    if (tid < 2 * n_words) {
        const int c = tid >= n_words;
        const uint64_t widx = tid - (c ? n_words : 0);
        for (int b = 0; b < 32; ++b) {
            const uint64_t j = 32 * widx + b;
            if (j >= Hc) break;
            const int m = (int)(j % H);
            const uint64_t r = j / H;
            const int y = (int)(r % L), z = (int)(r / L);
            const int x = 2 * m + ((y + z + c) & 1);
            const int xp = (x + 1 == L) ? 0 : x + 1, yp = (y + 1 == L) ? 0 : y + 1, zp = (z + 1 == L) ? 0 : z + 1;
            const int s = get_bit(a.S[c], j);
            unsat += get_bit(a.J[0][c], j) ^ s ^ get_bit(a.S[1 - c], colour_rank(L, xp, y, z));
            unsat += get_bit(a.J[1][c], j) ^ s ^ get_bit(a.S[1 - c], colour_rank(L, x, yp, z));
            unsat += get_bit(a.J[2][c], j) ^ s ^ get_bit(a.S[1 - c], colour_rank(L, x, y, zp));
            up += s;
        }
    }
    block_accumulate2(unsat, up, acc);
}

// Sample-packed: one thread per site (either colour); bit b of every word belongs to sample b, so the per-sample counts
// are the column sums of the bond words.  Each thread adds the bits of its words into shared per-sample counters.
__global__ void __launch_bounds__(256)
energy_sample_packed(const MeasureArgs a, unsigned long long *acc /* [32][2] */, uint64_t Hc)
{
    __shared__ unsigned int sh_unsat[32], sh_up[32];
    if (threadIdx.x < 32) { sh_unsat[threadIdx.x] = 0; sh_up[threadIdx.x] = 0; }
    __syncthreads();
    const int L = a.L, H = L >> 1;
    const uint64_t tid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t ex = 0, ey = 0, ez = 0, s = 0;
    if (tid < 2 * Hc) {
        const int c = tid >= Hc;
        const uint64_t j = tid - (c ? Hc : 0);
        const int m = (int)(j % H);
        const uint64_t r = j / H;
        const int y = (int)(r % L), z = (int)(r / L);
        const int x = 2 * m + ((y + z + c) & 1);
        const int xp = (x + 1 == L) ? 0 : x + 1, yp = (y + 1 == L) ? 0 : y + 1, zp = (z + 1 == L) ? 0 : z + 1;
        s = a.S[c][j];
        ex = a.J[0][c][j] ^ s ^ a.S[1 - c][colour_rank(L, xp, y, z)];
        ey = a.J[1][c][j] ^ s ^ a.S[1 - c][colour_rank(L, x, yp, z)];
        ez = a.J[2][c][j] ^ s ^ a.S[1 - c][colour_rank(L, x, y, zp)];
    }
    // Column sums over the warp: lane b collects bit b of every lane's words with ballots.
    const int lane = threadIdx.x & 31;
    unsigned int my_unsat = 0, my_up = 0;
#pragma unroll
    for (int b = 0; b < 32; ++b) {
        const unsigned int cnt = __popc(__ballot_sync(0xFFFFFFFFu, (ex >> b) & 1u)) +
                                 __popc(__ballot_sync(0xFFFFFFFFu, (ey >> b) & 1u)) +
                                 __popc(__ballot_sync(0xFFFFFFFFu, (ez >> b) & 1u));
        const unsigned int cup = __popc(__ballot_sync(0xFFFFFFFFu, (s >> b) & 1u));
        if (lane == b) { my_unsat = cnt; my_up = cup; }
    }
    atomicAdd(&sh_unsat[lane], my_unsat);
    atomicAdd(&sh_up[lane], my_up);
    __syncthreads();
    if (threadIdx.x < 32) {
        atomicAdd(&acc[2 * threadIdx.x], (unsigned long long)sh_unsat[threadIdx.x]);
        atomicAdd(&acc[2 * threadIdx.x + 1], (unsigned long long)sh_up[threadIdx.x]);
    }
}

// E = 2*unsat - 3N, M = 2*up - N  (R16), one thread per sample.
__global__ void finalize_energy(const unsigned long long *acc, int nsamples, long long N, long long *E, long long *M)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsamples) return;
    if (E) E[s] = 2 * (long long)acc[2 * s] - 3 * N;
    if (M) M[s] = 2 * (long long)acc[2 * s + 1] - N;
}

}  // namespace isingk
