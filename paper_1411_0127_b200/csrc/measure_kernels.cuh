// measure_kernels.cuh -- energy and magnetisation.
//
//   E = - sum over the 3N bonds of J sigma sigma (Eq. 1, each bond once).  With the encoding of Eq. 10 the
//   bond bit e = J ^ s_i ^ s_k (Eq. 11) is 1 exactly when -J sigma_i sigma_k = +1, so E = 2*popc(e over all bonds) - 3N,
//   and M = 2*popc(s) - N.  The kernels accumulate the two popcounts per sample into uint64 counters (warp shuffle
//   reduction, then a block reduction and one atomic pair per CTA); finalize_energy turns them into int64 E and M.
//   Kernels: energy_site_packed<W> (L a multiple of 64, fused finalisation), energy_site_packed_rows (every other even L, bit
//   windows), energy_sample_packed_sliced (sample-packed: bit-sliced column sums, all batches, fused finalisation), and the
//   one-bit-at-a-time energy_site_packed_generic / energy_sample_packed (kernel choice 1).
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

// Site-packed, L a multiple of 64: the thread mapping of the half-sweep kernel (a thread owns W consecutive words of a half-row,
// for both colours).  The +x neighbour of the colour-c site with bit m is bit m (xodd = 0) or bit m+1 (xodd = 1) of the
// other colour's half-row (a funnel shift by xodd; the bit entering at the end of the thread's words comes from the
// next lane of the row); +y / +z neighbours are the same bit one row up.  Every word is read once from HBM with 128-bit
// loads (the neighbour reads hit L1/L2): 512 MiB at L = 1024.
// One launch does everything: the CTAs add their counts to the slots, and the last CTA to finish (a ticket counter
// behind the slots) sums the slots, writes E and M (R16), and clears slots and counter for the next call, so a trace of
// E per half-sweep costs one small launch per record instead of memset + kernel + finalize.
// The counts of one tile = the rows of CTA (bx, by) of the grid (L / (32 / tpr_pad), L / 8): this thread's unsatisfied bonds and up
// spins are returned in unsat / up.
template <int W>
__device__ __forceinline__ void energy_tile(const MeasureArgs &a, uint32_t bx, uint32_t by, unsigned int &unsat, unsigned int &up)
{
    const int L = a.L, wpr = L >> 6;
    const RowMap rm = row_map<W>(L, bx, by);
    const int tpr = rm.tpr, y = rm.y, z = rm.z, k0 = rm.k0;
    const int yp = y + 1 == L ? 0 : y + 1, zp = z + 1 == L ? 0 : z + 1;
    const uint32_t row = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * z) + k0;
    const uint32_t row_yp = (uint32_t)wpr * ((uint32_t)yp + (uint32_t)L * z) + k0;
    const uint32_t row_zp = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * zp) + k0;
    const int next_lane = rm.next_lane;
    unsat = 0;
    up = 0;
    wait_for_previous_kernel();
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
        const uint32_t xodd = (uint32_t)((y + z + c) & 1);
        uint32_t edge = o[0];
        if (tpr > 1) edge = __shfl_sync(0xFFFFFFFFu, edge, next_lane);
#pragma unroll
        for (int k = 0; k < W; ++k) {
            const uint32_t nx = __funnelshift_r(o[k], (k + 1 < W) ? o[(k + 1) % W] : edge, xodd);
            if (rm.active) {  // idle lanes of a padded row shadow lane 0: count nothing twice
                unsat += __popc(jx[k] ^ s[k] ^ nx) + __popc(jy[k] ^ s[k] ^ oyp[k]) + __popc(jz[k] ^ s[k] ^ ozp[k]);
                up += __popc(s[k]);
            }
        }
    }
}

template <int W>
__global__ void __launch_bounds__(SWEEP_THREADS)
energy_site_packed(const MeasureArgs a, unsigned long long *acc /* ACC_SLOTS x {unsatisfied bonds, up spins}, then the ticket */,
                   long long N, long long *E, long long *M)
{
    unsigned int unsat, up;
    energy_tile<W>(a, blockIdx.x, blockIdx.y, unsat, up);
    block_accumulate2(unsat, up, acc + 2 * ((blockIdx.x + blockIdx.y * gridDim.x) & (ACC_SLOTS - 1)));
    finalize_slots_last_cta(acc, N, E, M);
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

// Site-packed, any even L: one thread per word; the +x / +y / +z neighbours of its row segments are unaligned bit windows
// of the other colour's array (bit_window, as in half_sweep_site_packed_rows); three popcounts per segment.
// item = word w of colour 0 (item < n_words) or of colour 1; adds the word's unsatisfied +x / +y / +z bonds and up spins.
template <bool PLAIN>
__device__ __forceinline__ void rows_energy_item(const MeasureArgs &a, uint32_t item, uint32_t n_words, uint32_t Hc, unsigned long long &unsat,
                                                 unsigned long long &up)
{
    const uint32_t L = (uint32_t)a.L, H = L >> 1, LH = L * H;
    const int c = item >= n_words;
    const uint32_t w = item - (c ? n_words : 0u), j0 = 32u * w;
    uint32_t remaining = Hc - j0 < 32u ? Hc - j0 : 32u, bitoff = 0;
    uint32_t r = j0 / H, m = j0 - r * H, z = r / L, y = r - z * L;
    // (selects, not run-time indices into the argument struct: a local copy of it would otherwise live in local memory)
    const uint32_t *So = c ? a.S[0] : a.S[1], *Sc = c ? a.S[1] : a.S[0];
    const uint32_t *Jxc = c ? a.J[0][1] : a.J[0][0], *Jyc = c ? a.J[1][1] : a.J[1][0], *Jzc = c ? a.J[2][1] : a.J[2][0];
    const uint32_t s = load_word<PLAIN>(Sc, w), jx = load_word<PLAIN>(Jxc, w), jy = load_word<PLAIN>(Jyc, w), jz = load_word<PLAIN>(Jzc, w);
    uint32_t nx = 0, ny = 0, nz = 0;
    while (remaining > 0) {
        const uint32_t len = remaining < H - m ? remaining : H - m;
        const uint32_t segmask = (len == 32u ? 0xFFFFFFFFu : ((1u << len) - 1u)) << bitoff;
        const uint32_t xodd = (y + z + (uint32_t)c) & 1u;
        const uint32_t P = r * H;
        const uint32_t Pyp = (y + 1 == L) ? P - (LH - H) : P + H, Pzp = (z + 1 == L) ? P - (Hc - LH) : P + LH;
        uint32_t wpx = bit_window<PLAIN>(So, P + m + xodd);
        if (xodd && m + len == H) wpx = (wpx & ~(1u << (len - 1))) | (bit_at<PLAIN>(So, P) << (len - 1));
        nx |= (wpx << bitoff) & segmask;
        ny |= (bit_window<PLAIN>(So, Pyp + m) << bitoff) & segmask;
        nz |= (bit_window<PLAIN>(So, Pzp + m) << bitoff) & segmask;
        bitoff += len;
        remaining -= len;
        m += len;
        if (m == H) {
            m = 0;
            ++r;
            if (++y == L) { y = 0; ++z; }
        }
    }
    const uint32_t valid = bitoff == 32u ? 0xFFFFFFFFu : (1u << bitoff) - 1u;
    unsat += __popc((jx ^ s ^ nx) & valid) + __popc((jy ^ s ^ ny) & valid) + __popc((jz ^ s ^ nz) & valid);
    up += __popc(s & valid);
}

__global__ void __launch_bounds__(256)
energy_site_packed_rows(const __grid_constant__ MeasureArgs a, unsigned long long *acc, uint32_t n_words, uint32_t Hc)
{
    unsigned long long unsat = 0, up = 0;
    for (uint32_t tid = blockIdx.x * 256u + threadIdx.x; tid < 2 * n_words; tid += gridDim.x * 256u)   // persistent grid
        rows_energy_item<false>(a, tid, n_words, Hc, unsat, up);
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

// Sample-packed, bit-sliced: the per-sample counts are the column sums of the bond words (and of the spin words).  A thread
// adds the words of its sites into vertical counters, i.e. bit planes of weight 1, 2, 4, ...: eight words at a time go
// through a carry-save adder tree (Harley-Seal: 7 full adders = 14 LOP3 per 8 words, the carry of weight 8 ripples into the
// upper planes), about 4 logic operations per word instead of 32 ballots.  At the end of its chunk the warp transposes
// every plane across its lanes (5 shuffle stages), after which lane b holds column b of all 32 lanes, i.e. sample b, and a
// popcount per plane gives the counts.  A warp owns one chunk of nblocks x 8 x 32 consecutive sites of one colour
// (coalesced loads: lane l takes the sites l, l + 32, ...); any even L.
constexpr int EN_MAX_BLOCKS = 64;   // 8 sites x 64 blocks x 3 bonds = 1536 < 2^11 (bond planes), 512 spins < 2^10

// (carry, sum) = a + b + c per bit: two LOP3
__device__ __forceinline__ void full_add(uint32_t &carry, uint32_t &sum, uint32_t a, uint32_t b, uint32_t c)
{
    const uint32_t u = a ^ b;
    carry = (a & b) | (u & c);
    sum = u ^ c;
}

template <int KH>
struct VerticalCounter {   // planes of weight 1, 2, 4 and KH planes of weight 8, 16, ...
    uint32_t ones = 0, twos = 0, fours = 0, hi[KH] = {};
    __device__ __forceinline__ void add8(const uint32_t *w)
    {
        uint32_t twosA, twosB, foursA, foursB, eights;
        full_add(twosA, ones, ones, w[0], w[1]);
        full_add(twosB, ones, ones, w[2], w[3]);
        full_add(foursA, twos, twos, twosA, twosB);
        full_add(twosA, ones, ones, w[4], w[5]);
        full_add(twosB, ones, ones, w[6], w[7]);
        full_add(foursB, twos, twos, twosA, twosB);
        full_add(eights, fours, fours, foursA, foursB);
#pragma unroll
        for (int p = 0; p < KH; ++p) {
            const uint32_t c = hi[p] & eights;
            hi[p] ^= eights;
            eights = c;
        }
    }
};

template <int J>
__device__ __forceinline__ uint32_t warp_transpose32_stage(uint32_t x, int lane)
{
    constexpr uint32_t m = J == 16 ? 0x0000FFFFu : J == 8 ? 0x00FF00FFu : J == 4 ? 0x0F0F0F0Fu : J == 2 ? 0x33333333u : 0x55555555u;
    const uint32_t other = __shfl_xor_sync(0xFFFFFFFFu, x, J);
    return (lane & J) ? (((other >> J) & m) | (x & ~m)) : ((x & m) | ((other & m) << J));
}
// Lane i holds row i of a 32 x 32 bit matrix; returns column `lane` (bit i = bit `lane` of row i).
__device__ __forceinline__ uint32_t warp_transpose32(uint32_t x, int lane)
{
    x = warp_transpose32_stage<16>(x, lane);
    x = warp_transpose32_stage<8>(x, lane);
    x = warp_transpose32_stage<4>(x, lane);
    x = warp_transpose32_stage<2>(x, lane);
    return warp_transpose32_stage<1>(x, lane);
}

template <int KH>
__device__ __forceinline__ unsigned int column_count(const VerticalCounter<KH> &v, int lane)
{   // the count of column `lane` summed over the 32 lanes of the warp
    unsigned int n = __popc(warp_transpose32(v.ones, lane)) + 2u * __popc(warp_transpose32(v.twos, lane)) +
                     4u * __popc(warp_transpose32(v.fours, lane));
#pragma unroll
    for (int p = 0; p < KH; ++p) n += (unsigned int)__popc(warp_transpose32(v.hi[p], lane)) << (3 + p);
    return n;
}

// grid = (ceil(2 * chunks_per_colour / 8), batches) CTAs of 8 warps, one chunk per warp; blockIdx.y = coded batch, whose arrays
// start batch_stride words after those of batch 0 (a holds batch 0) and whose counters are acc[64 b .. 64 b + 63].
// One launch does everything, as in energy_site_packed: the counters are zero on entry, and the last CTA to finish (ticket)
// turns them into E and M of all samples (R16) and clears counters and ticket for the next call.
__global__ void __launch_bounds__(256, 3)
energy_sample_packed_sliced(const __grid_constant__ MeasureArgs a, size_t batch_stride, unsigned long long *acc /* [batch][32][2] */,
                            unsigned int *ticket, uint32_t Hc, uint32_t chunks_per_colour, int nblocks, int nsamples, long long N,
                            long long *E, long long *M)
{
    __shared__ unsigned int sh_unsat[32], sh_up[32];
    if (threadIdx.x < 32) { sh_unsat[threadIdx.x] = 0; sh_up[threadIdx.x] = 0; }
    __syncthreads();
    const uint32_t L = (uint32_t)a.L, H = L >> 1, HL = H * L;
    const int lane = threadIdx.x & 31;
    const uint32_t chunk = blockIdx.x * 8u + (threadIdx.x >> 5);
    const size_t boff = (size_t)blockIdx.y * batch_stride;
    acc += 64u * blockIdx.y;
    wait_for_previous_kernel();
    if (chunk < 2u * chunks_per_colour) {   // warp-uniform
        // neighbouring warps take the two colours of the same stretch of ranks: the spin words one colour reads as neighbours
        // are the other's own words and meet in the L2 (colour-major order read both spin arrays twice from HBM)
        const int c = chunk & 1u;
        uint32_t j = (chunk >> 1) * (256u * (uint32_t)nblocks) + (uint32_t)lane;
        uint32_t m = j % H, r = j / H, y = r % L, z = r / L;
        const uint32_t *__restrict__ S = a.S[c] + boff, *__restrict__ So = a.S[1 - c] + boff;
        const uint32_t *__restrict__ Jx = a.J[0][c] + boff, *__restrict__ Jy = a.J[1][c] + boff, *__restrict__ Jz = a.J[2][c] + boff;
        VerticalCounter<8> bonds;   // 11 planes
        VerticalCounter<7> spins;   // 10 planes
        for (int blk = 0; blk < nblocks; ++blk) {
            uint32_t e[24], s[8];
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                // indices of four sites first, then their 28 loads back to back, then the bond words: nothing between the
                // loads depends on a loaded value, so all of them are in flight together
                uint32_t js[4], jx[4], jy[4], jz[4], ok[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const bool valid = j < Hc;
                    const uint32_t xodd = (y + z + (uint32_t)c) & 1u;
                    ok[i] = valid ? 0xFFFFFFFFu : 0u;
                    js[i] = valid ? j : 0u;
                    jx[i] = valid ? j - m + (xodd ? (m + 1 == H ? 0u : m + 1) : m) : 0u;
                    jy[i] = valid ? ((y + 1 == L) ? j - (HL - H) : j + H) : 0u;
                    jz[i] = valid ? ((z + 1 == L) ? j - (Hc - HL) : j + HL) : 0u;
                    j += 32u;
                    m += 32u;
                    while (m >= H) {
                        m -= H;
                        if (++y == L) { y = 0; ++z; }
                    }
                }
                uint32_t rs[4], rjx[4], rjy[4], rjz[4], rox[4], roy[4], roz[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    rs[i] = __ldg(S + js[i]);
                    rjx[i] = __ldg(Jx + js[i]);
                    rjy[i] = __ldg(Jy + js[i]);
                    rjz[i] = __ldg(Jz + js[i]);
                    rox[i] = __ldg(So + jx[i]);
                    roy[i] = __ldg(So + jy[i]);
                    roz[i] = __ldg(So + jz[i]);
                }
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int k = 4 * half + i;
                    s[k] = rs[i] & ok[i];
                    e[3 * k] = (rjx[i] ^ rs[i] ^ rox[i]) & ok[i];
                    e[3 * k + 1] = (rjy[i] ^ rs[i] ^ roy[i]) & ok[i];
                    e[3 * k + 2] = (rjz[i] ^ rs[i] ^ roz[i]) & ok[i];
                }
            }
            bonds.add8(e);
            bonds.add8(e + 8);
            bonds.add8(e + 16);
            spins.add8(s);
        }
        atomicAdd(&sh_unsat[lane], column_count(bonds, lane));
        atomicAdd(&sh_up[lane], column_count(spins, lane));
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        atomicAdd(&acc[2 * threadIdx.x], (unsigned long long)sh_unsat[threadIdx.x]);
        atomicAdd(&acc[2 * threadIdx.x + 1], (unsigned long long)sh_up[threadIdx.x]);
    }
    __shared__ bool is_last;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        is_last = atomicAdd(ticket, 1u) == gridDim.x * gridDim.y - 1;  // every other CTA's atomics are visible then
    }
    __syncthreads();
    if (is_last) {
        acc -= 64u * blockIdx.y;
        for (int sidx = threadIdx.x; sidx < nsamples; sidx += 256) {   // read and clear
            const unsigned long long tu = atomicExch(&acc[2 * sidx], 0ull), tp = atomicExch(&acc[2 * sidx + 1], 0ull);
            if (E) E[sidx] = 2 * (long long)tu - 3 * N;
            if (M) M[sidx] = 2 * (long long)tp - N;
        }
        if (threadIdx.x == 0) *ticket = 0u;
    }
}

// Overlap of two samples of a sample-packed handle (replicas): q = sum_i sigma^a_i sigma^b_i = N - 2 D with D the
// number of sites where bit ia of sample a's word differs from bit ib of sample b's word.  Wa / Wb: the spin arrays (one
// colour) of the batches holding a and b.  Persistent grid, one atomic per CTA; *cnt must be zero on entry.
__global__ void __launch_bounds__(256)
overlap_sample_packed(const uint32_t *__restrict__ Wa0, const uint32_t *__restrict__ Wb0, const uint32_t *__restrict__ Wa1,
                      const uint32_t *__restrict__ Wb1, int ia, int ib, uint32_t Hc, unsigned long long *cnt)
{
    unsigned long long d = 0, unused = 0;
    for (uint32_t j = blockIdx.x * 256u + threadIdx.x; j < Hc; j += gridDim.x * 256u)
        d += (((__ldg(Wa0 + j) >> ia) ^ (__ldg(Wb0 + j) >> ib)) & 1u) + (((__ldg(Wa1 + j) >> ia) ^ (__ldg(Wb1 + j) >> ib)) & 1u);
    block_accumulate2(d, unused, cnt);
}

__global__ void finalize_overlap(unsigned long long *cnt, long long N, long long *q)
{
    *q = N - 2 * (long long)cnt[0];
    cnt[0] = 0;
    cnt[1] = 0;
}

// E = 2*unsat - 3N, M = 2*up - N  (R16), one thread per sample (sample-packed and generic paths).
__global__ void finalize_energy(const unsigned long long *acc, int nsamples, long long N, long long *E, long long *M)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nsamples) return;
    if (E) E[s] = 2 * (long long)acc[2 * s] - 3 * N;
    if (M) M[s] = 2 * (long long)acc[2 * s + 1] - N;
}

}  // namespace isingk
