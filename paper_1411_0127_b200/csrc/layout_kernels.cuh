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
};

template <int V>  // V internal words (2V canonical words) per thread, V <= L/64
__global__ void __launch_bounds__(256) split_colours_site_packed(const SplitArgs a)
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
        const Vec lo = __ldcs(reinterpret_cast<const Vec *>(a.canon[q] + 2 * widx));
        const Vec hi = __ldcs(reinterpret_cast<const Vec *>(a.canon[q] + 2 * widx + V));
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
        *reinterpret_cast<Vec *>(a.out[q][p] + widx) = *reinterpret_cast<const Vec *>(even);
        *reinterpret_cast<Vec *>(a.out[q][1 - p] + widx) = *reinterpret_cast<const Vec *>(odd);
    }
}

template <int V>
__global__ void __launch_bounds__(256)
merge_colours_site_packed(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon, int L)
{
    typedef typename WordVec<V>::type Vec;
    const int wpr = L >> 6;
    const uint64_t n = (uint64_t)wpr * L * L;
    const uint64_t widx = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * V;
    if (widx >= n) return;
    const uint64_t r = widx / (unsigned)wpr;
    const int p = (int)((r % (unsigned)L) + (r / (unsigned)L)) & 1;
    const Vec ve = *reinterpret_cast<const Vec *>((p ? S1 : S0) + widx);
    const Vec vo = *reinterpret_cast<const Vec *>((p ? S0 : S1) + widx);
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

// Sample-packed: word j of the colour-c array of a batch collects bit i(j,c) of the 32 samples' canonical arrays.
// canon points at the first sample of the batch; consecutive samples are `sample_stride` words apart.
__global__ void __launch_bounds__(256)
gather_sample_packed(const uint32_t *__restrict__ canon, uint64_t sample_stride, uint32_t *__restrict__ out, int colour, int L,
                     uint64_t Hc)
{
    const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Hc) return;
    const int H = L >> 1;
    const int m = (int)(j % H);
    const uint64_t r = j / H;
    const int x = 2 * m + (((int)(r % L) + (int)(r / L) + colour) & 1);
    const uint64_t i = (uint64_t)x + (uint64_t)L * r;
    uint32_t w = 0;
#pragma unroll 8
    for (int b = 0; b < 32; ++b) w |= ((canon[b * sample_stride + (i >> 5)] >> (i & 31)) & 1u) << b;
    out[j] = w;
}

// Sample-packed -> canonical spins: one thread per canonical word of one sample.
__global__ void __launch_bounds__(256)
scatter_sample_packed(const uint32_t *__restrict__ S0, const uint32_t *__restrict__ S1, uint32_t *__restrict__ canon,
                      uint64_t sample_stride, int L, uint64_t n_canon_words, uint64_t N)
{
    const uint64_t cw = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int sample = blockIdx.y;  // within the batch
    if (cw >= n_canon_words) return;
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

}  // namespace isingk
