// layout_kernels.cuh -- canonical packed format <-> internal colour-separated layout.
//
// Canonical: bit (i&31) of word (i>>5), i = x + L*(y + L*z), one bit array per sample (spins) or per (sample, dir).
// Internal:  bit arrays indexed by the colour rank j = (x>>1) + (L/2)*(y + L*z), one per colour (sweep_kernels.cuh).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sweep_kernels.cuh"

namespace isingk {

// keep the even-position bits of v, packed into the low 16 bits
__device__ __forceinline__ uint32_t compress_even_bits(uint32_t v)
{
    v &= 0x55555555u;
    v = (v | (v >> 1)) & 0x33333333u;
    v = (v | (v >> 2)) & 0x0F0F0F0Fu;
    v = (v | (v >> 4)) & 0x00FF00FFu;
    v = (v | (v >> 8)) & 0x0000FFFFu;
    return v;
}

// spread the low 16 bits of v to the even positions
__device__ __forceinline__ uint32_t spread_to_even_bits(uint32_t v)
{
    v &= 0x0000FFFFu;
    v = (v | (v << 8)) & 0x00FF00FFu;
    v = (v | (v << 4)) & 0x0F0F0F0Fu;
    v = (v | (v << 2)) & 0x33333333u;
    v = (v | (v << 1)) & 0x55555555u;
    return v;
}

// Site-packed, L a multiple of 64.  A canonical row (fixed y,z) is L/32 words; its even-x bits belong to colour p = (y+z)&1
// and its odd-x bits to colour 1-p.  One thread de-interleaves canonical words 2k, 2k+1 of a row into word k of the
// half-row of both colours, for `narrays` canonical bit arrays at once (spins, Jx, Jy, Jz).
struct SplitArgs {
    const uint32_t *canon[4];
    uint32_t *out[4][2];  // [array][colour]
    int narrays;
    int L;
    // a batch of lattices (batch_kernels.cuh), blockIdx.y = sample: words between consecutive samples in canon[q] / in out[q][c]
    size_t canon_stride[4], out_stride;
};

template <int V>  // V internal words (2V canonical words) per thread, V <= L/64
__global__ void __launch_bounds__(256) split_colours_site_packed(const __grid_constant__ SplitArgs a)
{
    typedef typename WordVec<V>::type Vec;
    const int L = a.L, wpr = L >> 6;
    const uint64_t n = (uint64_t)wpr * L * L;
    const uint64_t widx = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * V;
    if (widx >= n) return;
    const uint64_t r = widx / (unsigned)wpr;
    const int p = (int)((r % (unsigned)L) + (r / (unsigned)L)) & 1;
    for (int q = 0; q < a.narrays; ++q) {
        uint32_t c[2 * V], even[V], odd[V];
        const uint32_t *canon = a.canon[q] + (size_t)blockIdx.y * a.canon_stride[q];
        const Vec lo = __ldcs(reinterpret_cast<const Vec *>(canon + 2 * widx));
        const Vec hi = __ldcs(reinterpret_cast<const Vec *>(canon + 2 * widx + V));
#pragma unroll
        for (int k = 0; k < V; ++k) {
            c[k] = reinterpret_cast<const uint32_t *>(&lo)[k];
            c[V + k] = reinterpret_cast<const uint32_t *>(&hi)[k];
        }
#pragma unroll
        for (int k = 0; k < V; ++k) {
            even[k] = compress_even_bits(c[2 * k]) | (compress_even_bits(c[2 * k + 1]) << 16);
            odd[k] = compress_even_bits(c[2 * k] >> 1) | (compress_even_bits(c[2 * k + 1] >> 1) << 16);
        }
        // the VALUE is selected by the row's parity, not the array: every store instruction of a warp then writes one array, its
        // lanes' rows back to back (512 contiguous bytes), instead of alternating between the two arrays row by row, which
        // left half-written lines behind (739 MB of DRAM writes for 537 MB of output at L = 1024, profiles/r1p_aux_kernels.md)
        uint32_t for0[V], for1[V];
#pragma unroll
        for (int k = 0; k < V; ++k) {
            for0[k] = p ? odd[k] : even[k];
            for1[k] = p ? even[k] : odd[k];
        }
        const size_t so = (size_t)blockIdx.y * a.out_stride;
        __stcs(reinterpret_cast<Vec *>(a.out[q][0] + so + widx), *reinterpret_cast<const Vec *>(for0));
        __stcs(reinterpret_cast<Vec *>(a.out[q][1] + so + widx), *reinterpret_cast<const Vec *>(for1));
    }
}

template <int V>
__global__ void __launch_bounds__(256)
merge_colours_site_packed(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon, int L,
                          size_t in_stride = 0, size_t canon_stride = 0)   // a batch of lattices: blockIdx.y = sample
{
    typedef typename WordVec<V>::type Vec;
    const int wpr = L >> 6;
    S0 += (size_t)blockIdx.y * in_stride;
    S1 += (size_t)blockIdx.y * in_stride;
    canon += (size_t)blockIdx.y * canon_stride;
    const uint64_t n = (uint64_t)wpr * L * L;
    const uint64_t widx = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * V;
    if (widx >= n) return;
    const uint64_t r = widx / (unsigned)wpr;
    const int p = (int)((r % (unsigned)L) + (r / (unsigned)L)) & 1;
    const Vec v0 = *reinterpret_cast<const Vec *>(S0 + widx), v1 = *reinterpret_cast<const Vec *>(S1 + widx);   // contiguous per warp
    const Vec ve = p ? v1 : v0, vo = p ? v0 : v1;
    uint32_t out[2 * V];
#pragma unroll
    for (int k = 0; k < V; ++k) {
        const uint32_t even = reinterpret_cast<const uint32_t *>(&ve)[k], odd = reinterpret_cast<const uint32_t *>(&vo)[k];
        out[2 * k] = spread_to_even_bits(even) | (spread_to_even_bits(odd) << 1);
        out[2 * k + 1] = spread_to_even_bits(even >> 16) | (spread_to_even_bits(odd >> 16) << 1);
    }
    __stcs(reinterpret_cast<Vec *>(canon + 2 * widx), *reinterpret_cast<const Vec *>(out));
    __stcs(reinterpret_cast<Vec *>(canon + 2 * widx + V), *reinterpret_cast<const Vec *>(out + V));
}

// Site-packed, any even L: one thread per internal word of one colour array, one bit at a time.
__global__ void __launch_bounds__(256)
gather_site_packed_generic(const uint32_t *__restrict__ canon, uint32_t *__restrict__ out, int colour, int L,
                           uint64_t n_words, uint64_t Hc)
{
    const uint64_t widx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (widx >= n_words) return;
    const int H = L >> 1;
    uint32_t w = 0;
    for (int b = 0; b < 32; ++b) {
        const uint64_t j = 32 * widx + b;
        if (j >= Hc) break;
        const int m = (int)(j % H);
        const uint64_t r = j / H;
        const int y = (int)(r % L), z = (int)(r / L);
        const int x = 2 * m + ((y + z + colour) & 1);
        const uint64_t i = (uint64_t)x + (uint64_t)L * r;
        w |= ((canon[i >> 5] >> (i & 31)) & 1u) << b;
    }
    out[widx] = w;
}

// Site-packed, any even L: one thread per canonical word.
__global__ void __launch_bounds__(256)
scatter_site_packed_generic(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon,
                            int L, uint64_t n_canon_words, uint64_t N)
{
    const uint64_t cw = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cw >= n_canon_words) return;
    uint32_t w = 0;
    for (int b = 0; b < 32; ++b) {
        const uint64_t i = 32 * cw + b;
        if (i >= N) break;
        const int x = (int)(i % L);
        const uint64_t r = i / L;
        const int y = (int)(r % L), z = (int)(r / L);
        const int c = (x + y + z) & 1;
        const uint64_t j = (uint64_t)(x >> 1) + (uint64_t)(L >> 1) * r;
        w |= (uint32_t)get_bit(c ? S1 : S0, j) << b;
    }
    canon[cw] = w;
}

// Site-packed, any even L, word at a time (the bit windows of half_sweep_site_packed_rows).  gather: the row segments of an
// output word are every second bit of a canonical bit range (a 64-bit window, even bits compressed); scatter: the row
// segments of a canonical word interleave a bit range of each colour array (16-bit windows spread to alternate bits).
__device__ __forceinline__ uint32_t canon_window(const uint32_t *__restrict__ a, uint64_t pos, uint64_t n_words)
{   // bits pos .. pos+31 of a caller-owned array of n_words words; words past its end read as zero
    const uint64_t w = pos >> 5;
    const uint32_t sh = (uint32_t)pos & 31u;
    const uint32_t lo = w < n_words ? __ldg(a + w) : 0u;
    const uint32_t hi = (sh && w + 1 < n_words) ? __ldg(a + w + 1) : 0u;
    return __funnelshift_r(lo, hi, sh);
}

// grid = (ceil(n_words / 128), 4 arrays).  Word w of BOTH colour arrays comes from the same canonical sites (colour ranks
// 32 w .. 32 w + 31 of either colour are the 64 sites 64 w .. 64 w + 63 of the rows they lie in): the even sites of a row segment
// belong to the colour with xodd = 0 there, the odd ones to the other, so one pass over the canonical windows fills both words
// (one pass per colour read every canonical word twice from HBM: 996 MB for 500 MB at L = 1000).
__global__ void __launch_bounds__(128)
gather_site_packed_rows(const __grid_constant__ SplitArgs a, uint32_t n_words, uint32_t Hc, uint64_t n_canon_words)
{
    const uint32_t w = blockIdx.x * 128u + threadIdx.x;
    if (w >= n_words) return;
    const int arr = blockIdx.y;
    const uint32_t *__restrict__ canon = a.canon[arr];
    const uint32_t L = (uint32_t)a.L, H = L >> 1;
    const uint32_t j0 = 32u * w;
    uint32_t remaining = Hc - j0 < 32u ? Hc - j0 : 32u, bitoff = 0;
    uint32_t r = j0 / H, m = j0 - r * H, z = r / L, y = r - z * L;
    uint32_t out0 = 0, out1 = 0;   // colour 0 / colour 1
    while (remaining > 0) {
        const uint32_t len = remaining < H - m ? remaining : H - m;
        const uint32_t segmask = (len == 32u ? 0xFFFFFFFFu : ((1u << len) - 1u)) << bitoff;
        const uint32_t p = (y + z) & 1u;                          // colour of the even sites of this row
        const uint64_t base = (uint64_t)L * r + 2u * m;          // canonical index of the segment's first pair of sites
        const uint32_t w0 = canon_window(canon, base, n_canon_words);
        uint32_t even = compress_even_bits(w0), odd = compress_even_bits(w0 >> 1);
        if (len > 16u) {
            const uint32_t w1 = canon_window(canon, base + 32u, n_canon_words);
            even |= compress_even_bits(w1) << 16;
            odd |= compress_even_bits(w1 >> 1) << 16;
        }
        out0 |= ((p ? odd : even) << bitoff) & segmask;
        out1 |= ((p ? even : odd) << bitoff) & segmask;
        bitoff += len;
        remaining -= len;
        m += len;
        if (m == H) {
            m = 0;
            ++r;
            if (++y == L) { y = 0; ++z; }
        }
    }
    a.out[arr][0][w] = out0;
    a.out[arr][1][w] = out1;
}

__global__ void __launch_bounds__(128)
scatter_site_packed_rows(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon, int L_,
                         uint64_t n_canon_words, uint64_t N)
{
    const uint64_t cw = (uint64_t)blockIdx.x * 128u + threadIdx.x;
    if (cw >= n_canon_words) return;
    const uint32_t L = (uint32_t)L_, H = L >> 1;
    const uint64_t i0 = 32u * cw;
    uint32_t remaining = N - i0 < 32u ? (uint32_t)(N - i0) : 32u, bitoff = 0;
    uint32_t r = (uint32_t)(i0 / L), x = (uint32_t)(i0 - (uint64_t)r * L), z = r / L, y = r - z * L;
    uint32_t out = 0;
    while (remaining > 0) {
        const uint32_t len = remaining < L - x ? remaining : L - x;
        const uint32_t segmask = (len == 32u ? 0xFFFFFFFFu : ((1u << len) - 1u)) << bitoff;
        const uint32_t xodd0 = (y + z) & 1u;                       // x parity of colour 0 in this row
        const uint32_t xa0 = x + ((x ^ xodd0) & 1u), xa1 = x + ((x ^ xodd0 ^ 1u) & 1u);   // first x of either colour in the segment
        const uint32_t P = r * H;
        const uint32_t v = (spread_to_even_bits(bit_window(S0, P + (xa0 >> 1))) << (xa0 - x)) |
                           (spread_to_even_bits(bit_window(S1, P + (xa1 >> 1))) << (xa1 - x));
        out |= (v << bitoff) & segmask;
        bitoff += len;
        remaining -= len;
        x += len;
        if (x == L) {
            x = 0;
            ++r;
            if (++y == L) { y = 0; ++z; }
        }
    }
    canon[cw] = out;
}

// Sample-packed, one bit at a time (any even L): word j of the colour-c array of a batch collects bit i(j,c) of the 32 samples'
// canonical arrays, for all coded batches, the four bit arrays and both colours in one launch: blockIdx.y = 8 * batch + 2 * array + colour
// (array 0 = spins, 1..3 = Jx, Jy, Jz).  ws = the internal arrays (8 per batch, array_words each, S[0], S[1], Jx[0], Jx[1], ...).
__global__ void __launch_bounds__(256)
gather_sample_packed_all(const uint32_t *__restrict__ d_spins, const uint32_t *__restrict__ d_J, uint32_t *__restrict__ ws,
                         uint64_t array_words, uint64_t W, int L, uint64_t Hc, uint32_t batch0)
{
    const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Hc) return;
    const uint32_t b = batch0 + blockIdx.y / 8u, arr = (blockIdx.y & 7u) >> 1, colour = blockIdx.y & 1u;
    const uint32_t *__restrict__ canon = arr == 0 ? d_spins + (uint64_t)b * 32 * W : d_J + (uint64_t)b * 32 * 3 * W + (uint64_t)(arr - 1) * W;
    const uint64_t sample_stride = arr == 0 ? W : 3 * W;
    uint32_t *__restrict__ out = ws + ((uint64_t)b * 8 + 2 * arr + colour) * array_words;
    const int H = L >> 1;
    const int m = (int)(j % H);
    const uint64_t r = j / H;
    const int x = 2 * m + (((int)(r % L) + (int)(r / L) + (int)colour) & 1);
    const uint64_t i = (uint64_t)x + (uint64_t)L * r;
    uint32_t w = 0;
#pragma unroll 8
    for (int s = 0; s < 32; ++s) w |= ((canon[s * sample_stride + (i >> 5)] >> (i & 31)) & 1u) << s;
    out[j] = w;
}

// Sample-packed -> canonical spins: one thread per canonical word of one sample.
// blockIdx.z = coded batch: its colour arrays start batch_stride words after S0 / S1, its canonical words 32 * sample_stride
// words after canon.
__global__ void __launch_bounds__(256)
scatter_sample_packed(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon,
                      uint64_t sample_stride, int L, uint64_t n_canon_words, uint64_t N, uint64_t batch_stride)
{
    const uint64_t cw = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int sample = blockIdx.y;  // within the batch
    if (cw >= n_canon_words) return;
    S0 += (uint64_t)blockIdx.z * batch_stride;
    S1 += (uint64_t)blockIdx.z * batch_stride;
    canon += (uint64_t)blockIdx.z * 32 * sample_stride;
    uint32_t w = 0;
    for (int b = 0; b < 32; ++b) {
        const uint64_t i = 32 * cw + b;
        if (i >= N) break;
        const int x = (int)(i % L);
        const uint64_t r = i / L;
        const int c = (x + (int)(r % L) + (int)(r / L)) & 1;
        const uint64_t j = (uint64_t)(x >> 1) + (uint64_t)(L >> 1) * r;
        w |= (((c ? S1 : S0)[j] >> sample) & 1u) << b;
    }
    canon[sample * sample_stride + cw] = w;
}

// ---------------------------------------------------------------------------------------------------
// Sample-packed, L a multiple of 32 (a canonical word = 32 consecutive x of one row): tile kernels.  One thread owns one
// canonical word index cw of all 32 samples of a batch: 32 words (lane l reads word cw0 + l of sample s: 128 contiguous
// bytes per warp load), transposed in registers as a 32 x 32 bit matrix (5 x 16 masked swaps), are the 32 site words of
// the row segment; the 16 of each colour go out as four 128-bit stores.  The scatter kernel is the inverse.
// ---------------------------------------------------------------------------------------------------
template <int J>
__device__ __forceinline__ void transpose32_stage(uint32_t (&A)[32])
{
    constexpr uint32_t m = J == 16 ? 0x0000FFFFu : J == 8 ? 0x00FF00FFu : J == 4 ? 0x0F0F0F0Fu : J == 2 ? 0x33333333u : 0x55555555u;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        if ((k & J) == 0) {
            const uint32_t t = ((A[k] >> J) ^ A[k + J]) & m;
            A[k] ^= t << J;
            A[k + J] ^= t;
        }
    }
}

__device__ __forceinline__ void transpose32_in_registers(uint32_t (&A)[32])
{  // bit b of A[s]  <->  bit s of A[b]
    transpose32_stage<16>(A);
    transpose32_stage<8>(A);
    transpose32_stage<4>(A);
    transpose32_stage<2>(A);
    transpose32_stage<1>(A);
}

struct GatherTileArgs {
    const uint32_t *canon[4];  // first sample of the batch: spins, Jx, Jy, Jz
    uint64_t stride[4];        // words between consecutive samples
    uint32_t *out[4][2];       // sample-packed arrays of the two colours
};

// grid = (ceil(ncw / 128), 4 arrays)
__global__ void __launch_bounds__(128) gather_sample_packed_tiles(const __grid_constant__ GatherTileArgs a, int L, uint32_t ncw)
{
    const int arr = blockIdx.y;
    const uint32_t cw = blockIdx.x * 128u + threadIdx.x;
    if (cw >= ncw) return;
    const uint32_t wpr = (uint32_t)L >> 5, r = cw / wpr, y = r % (uint32_t)L, z = r / (uint32_t)L;
    const uint32_t base = ((uint32_t)L >> 1) * r + (cw - r * wpr) * 16u;   // colour rank of the first site of either colour
    const uint32_t *__restrict__ src = a.canon[arr] + cw;
    const uint64_t stride = a.stride[arr];
    uint32_t A[32];
#pragma unroll
    for (int s = 0; s < 32; ++s) A[s] = __ldg(src + (uint64_t)s * stride);
    transpose32_in_registers(A);   // A[b] = the 32 samples of site 32 cw + b
    const bool odd0 = ((y + z) & 1u) != 0;   // colour 0 holds the odd x of this row
    uint32_t *o0 = a.out[arr][0] + base, *o1 = a.out[arr][1] + base;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        uint4 v0, v1;
        v0.x = odd0 ? A[8 * q + 1] : A[8 * q];     v1.x = odd0 ? A[8 * q] : A[8 * q + 1];
        v0.y = odd0 ? A[8 * q + 3] : A[8 * q + 2]; v1.y = odd0 ? A[8 * q + 2] : A[8 * q + 3];
        v0.z = odd0 ? A[8 * q + 5] : A[8 * q + 4]; v1.z = odd0 ? A[8 * q + 4] : A[8 * q + 5];
        v0.w = odd0 ? A[8 * q + 7] : A[8 * q + 6]; v1.w = odd0 ? A[8 * q + 6] : A[8 * q + 7];
        reinterpret_cast<uint4 *>(o0)[q] = v0;
        reinterpret_cast<uint4 *>(o1)[q] = v1;
    }
}

// grid = ceil(ncw / 128): canonical spins of the 32 samples of a batch from the two colour arrays
__global__ void __launch_bounds__(128)
scatter_sample_packed_tiles(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon,
                            uint64_t sample_stride, int L, uint32_t ncw)
{
    const uint32_t cw = blockIdx.x * 128u + threadIdx.x;
    if (cw >= ncw) return;
    const uint32_t wpr = (uint32_t)L >> 5, r = cw / wpr, y = r % (uint32_t)L, z = r / (uint32_t)L;
    const uint32_t base = ((uint32_t)L >> 1) * r + (cw - r * wpr) * 16u;
    const bool odd0 = ((y + z) & 1u) != 0;
    uint32_t A[32];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const uint4 v0 = __ldg(reinterpret_cast<const uint4 *>(S0 + base) + q);
        const uint4 v1 = __ldg(reinterpret_cast<const uint4 *>(S1 + base) + q);
        A[8 * q] = odd0 ? v1.x : v0.x;     A[8 * q + 1] = odd0 ? v0.x : v1.x;
        A[8 * q + 2] = odd0 ? v1.y : v0.y; A[8 * q + 3] = odd0 ? v0.y : v1.y;
        A[8 * q + 4] = odd0 ? v1.z : v0.z; A[8 * q + 5] = odd0 ? v0.z : v1.z;
        A[8 * q + 6] = odd0 ? v1.w : v0.w; A[8 * q + 7] = odd0 ? v0.w : v1.w;
    }
    transpose32_in_registers(A);   // A[s] = canonical word cw of sample s
#pragma unroll
    for (int s = 0; s < 32; ++s) canon[(uint64_t)s * sample_stride + cw] = A[s];
}

}  // namespace isingk
