// fnv_kernels.cuh -- the 64-bit FNV-1a checksum of BASELINE.json config 4 computed on the device, in parallel.
//
// FNV-1a is defined byte by byte, h <- (h ^ b) * P mod 2^64 (offset basis 0xcbf29ce484222325, P = 0x100000001b3), and looks
// sequential: on a host core it takes 17 ms per 16 MiB, which made config 4 (ten checksums of the L = 512 spins in 100 sweeps) a
// hashing benchmark (31 ms, of which 10 ms sweeps).  It is not:
//   * the XOR touches the low byte only, so  h ^ b = h + d  with  d = (l ^ b) - l,  l = h & 0xff,  and  h' = (h + d) * P;
//   * the low byte follows its own recurrence  l' = ((l ^ b) * 0xb3) & 0xff  (0xb3 = P & 0xff), closed on 8 bits.
// Hence for a chunk of n bytes  h_end = h_start * P^n + sum_i d_i * P^(n - i),  where the d_i depend on the data and on the low
// byte at the start of the chunk only.  Three small steps:
//   1. fnv_low_byte_maps: for every sub-chunk (a chunk = 32 sub-chunks), the map (low byte at its start) -> (low byte at its end),
//      by running the 8-bit recurrence from all 256 starting values (one integer instruction per value and byte: two values share
//      a register in 16-bit lanes); the 32 maps of a chunk are composed into the chunk's map;
//   2. fnv_chunk_starts: one CTA composes the chunk maps in order (they sit in shared memory): the low byte at every chunk's start;
//   3. fnv_chunk_sums: every sub-chunk runs once more from its actual start (a walk through the chunk's 32 maps) and accumulates
//      acc <- (acc + d) * P;  the chunk folds its 32 parts, and fnv_combine folds the chunks,  h <- h * P^n_c + acc_c,  as a tree
//      of compositions of affine maps.
// All arithmetic is mod 2^64 as in the definition; the result is the same 64-bit number, bit for bit (tests: published vectors, the
// host routine, the oracle's).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace isingk {

constexpr uint64_t FNV_OFFSET = 0xcbf29ce484222325ull, FNV_PRIME = 0x100000001b3ull;
constexpr int FNV_MAX_CHUNKS = 888;     // 888 x 256 bytes of maps = 222 KiB fit the shared memory of one CTA (step 2); 888 = 3 x 2 x 148:
                                        // three full waves of step 1 at two CTAs of 1024 threads per SM (896 would leave a fourth wave of 8)
constexpr int FNV_SUB = 32;             // sub-chunks per chunk: the unit of steps 1 and 3
constexpr int FNV_STARTS_PER_THREAD = 8;

struct FnvPlan {
    uint64_t nbytes;
    uint32_t nchunks, chunk_bytes;   // chunk_bytes = FNV_SUB * sub_bytes, sub_bytes a multiple of 4; the last chunk holds the rest
    uint32_t sub_bytes;
};

inline FnvPlan fnv_plan(uint64_t nbytes)
{
    FnvPlan p;
    p.nbytes = nbytes;
    uint64_t sb = (nbytes + (uint64_t)FNV_MAX_CHUNKS * FNV_SUB - 1) / ((uint64_t)FNV_MAX_CHUNKS * FNV_SUB);
    sb = (sb + 3) / 4 * 4;
    if (sb < 64) sb = 64;
    p.sub_bytes = (uint32_t)sb;
    p.chunk_bytes = (uint32_t)(sb * FNV_SUB);
    p.nchunks = (uint32_t)((nbytes + p.chunk_bytes - 1) / p.chunk_bytes);
    return p;
}

// scratch: [nchunks][256] chunk maps, [nchunks][FNV_SUB][256] sub-chunk maps, [nchunks] start bytes (padded), [nchunks] uint64 sums
inline size_t fnv_scratch_bytes(const FnvPlan &p)
{
    return (size_t)p.nchunks * 256 * (1 + FNV_SUB) + ((size_t)p.nchunks + 7) / 8 * 8 + (size_t)p.nchunks * 8 + 256;
}

// bytes [begin, begin + n) of sub-chunk (c, j): n = 0 past the end of the data
__device__ __forceinline__ void fnv_sub_range(const FnvPlan &p, uint32_t c, uint32_t j, uint64_t &begin, uint64_t &n)
{
    begin = (uint64_t)c * p.chunk_bytes + (uint64_t)j * p.sub_bytes;
    n = begin >= p.nbytes ? 0 : (p.nbytes - begin < p.sub_bytes ? p.nbytes - begin : p.sub_bytes);
}

// Step 1.  grid = nchunks, block = FNV_SUB x 32 threads: thread (j, g) runs the starting values 8g .. 8g + 7 through sub-chunk j;
// then thread s composes the FNV_SUB maps of the chunk in order.  Both the chunk's map and its sub-chunk maps are kept.
__global__ void __launch_bounds__(FNV_SUB * 32) fnv_low_byte_maps(const uint8_t *__restrict__ data, FnvPlan p, uint8_t *__restrict__ chunk_maps,
                                                                  uint8_t *__restrict__ sub_maps)
{
    __shared__ uint8_t sm[FNV_SUB][256];
    const uint32_t c = blockIdx.x, j = threadIdx.x >> 5, g = threadIdx.x & 31u;
    uint64_t begin, n;
    fnv_sub_range(p, c, j, begin, n);
    // two starting values per register, in 16-bit lanes: a lane holds a byte, byte * 0xb3 < 2^16 stays in its lane, and the mask
    // that cuts it back to a byte is folded into the XOR of the next step: one LOP3 and one IMAD per byte and TWO values
    constexpr int NREG = FNV_STARTS_PER_THREAD / 2;
    uint32_t x[NREG];
#pragma unroll
    for (int k = 0; k < NREG; ++k) x[k] = (g * FNV_STARTS_PER_THREAD + 2 * k) | ((g * FNV_STARTS_PER_THREAD + 2 * k + 1) << 16);
    const uint32_t *words = reinterpret_cast<const uint32_t *>(data + begin);   // begin is a multiple of 4, data 4-byte aligned
    const uint32_t nwords = (uint32_t)(n / 4);
    for (uint32_t w = 0; w < nwords; ++w) {
        const uint32_t v = __ldg(words + w);
#pragma unroll
        for (int b4 = 0; b4 < 4; ++b4) {
            const uint32_t bb = __byte_perm(v, 0u, 0x4040u | (uint32_t)b4 | ((uint32_t)b4 << 8));   // byte b4 of v in both lanes
#pragma unroll
            for (int k = 0; k < NREG; ++k) x[k] = ((x[k] & 0x00ff00ffu) ^ bb) * 0xb3u;
        }
    }
    for (uint64_t i = 4ull * nwords; i < n; ++i) {   // the last bytes of data whose length is not a multiple of 4
        const uint32_t bb = (uint32_t)data[begin + i] * 0x00010001u;
#pragma unroll
        for (int k = 0; k < NREG; ++k) x[k] = ((x[k] & 0x00ff00ffu) ^ bb) * 0xb3u;
    }
#pragma unroll
    for (int k = 0; k < NREG; ++k) {
        sm[j][g * FNV_STARTS_PER_THREAD + 2 * k] = (uint8_t)x[k];
        sm[j][g * FNV_STARTS_PER_THREAD + 2 * k + 1] = (uint8_t)(x[k] >> 16);
    }
    __syncthreads();
    uint32_t *out = reinterpret_cast<uint32_t *>(sub_maps + (size_t)c * FNV_SUB * 256);
    for (uint32_t i = threadIdx.x; i < FNV_SUB * 64; i += FNV_SUB * 32) out[i] = reinterpret_cast<const uint32_t *>(&sm[0][0])[i];
    if (threadIdx.x < 256) {
        uint32_t v = threadIdx.x;
#pragma unroll 1
        for (int jj = 0; jj < FNV_SUB; ++jj) v = sm[jj][v];
        chunk_maps[(size_t)c * 256 + threadIdx.x] = (uint8_t)v;
    }
}

// Step 2.  <<<1, 256, nchunks * 256>>>: the chunk maps into shared memory, then one thread walks through them.
__global__ void __launch_bounds__(256) fnv_chunk_starts(const uint8_t *__restrict__ maps, uint32_t nchunks, uint8_t *__restrict__ start)
{
    extern __shared__ uint8_t sm_maps[];
    const uint32_t nwords = nchunks * 64u;
    for (uint32_t i = threadIdx.x; i < nwords; i += 256u) reinterpret_cast<uint32_t *>(sm_maps)[i] = reinterpret_cast<const uint32_t *>(maps)[i];
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t l = (uint32_t)(FNV_OFFSET & 0xffu);
        for (uint32_t c = 0; c < nchunks; ++c) {
            start[c] = (uint8_t)l;
            l = sm_maps[c * 256u + l];
        }
    }
}

__device__ __forceinline__ uint64_t fnv_prime_power(uint64_t n)
{
    uint64_t base = FNV_PRIME, acc = 1;
    while (n) {
        if (n & 1) acc *= base;
        base *= base;
        n >>= 1;
    }
    return acc;
}

// Step 3.  grid = nchunks, block = FNV_SUB threads: the starting low byte of every sub-chunk from the chunk's (a walk through its
// sub-chunk maps), then thread j runs sub-chunk j once: acc = sum_i d_i P^(n - i); the chunk's sum folds them in order.
__global__ void __launch_bounds__(FNV_SUB) fnv_chunk_sums(const uint8_t *__restrict__ data, FnvPlan p, const uint8_t *__restrict__ start,
                                                          const uint8_t *__restrict__ sub_maps, unsigned long long *__restrict__ sums)
{
    __shared__ uint8_t sm[FNV_SUB][256];
    __shared__ uint8_t sub_start[FNV_SUB];
    __shared__ unsigned long long part[FNV_SUB], pw[FNV_SUB];
    const uint32_t c = blockIdx.x, j = threadIdx.x;
    const uint32_t *in = reinterpret_cast<const uint32_t *>(sub_maps + (size_t)c * FNV_SUB * 256);
    for (uint32_t i = threadIdx.x; i < FNV_SUB * 64; i += FNV_SUB) reinterpret_cast<uint32_t *>(&sm[0][0])[i] = in[i];
    __syncthreads();
    if (j == 0) {
        uint32_t l = start[c];
        for (int jj = 0; jj < FNV_SUB; ++jj) {
            sub_start[jj] = (uint8_t)l;
            l = sm[jj][l];
        }
    }
    __syncthreads();
    uint64_t begin, n;
    fnv_sub_range(p, c, j, begin, n);
    uint32_t l = sub_start[j];
    uint64_t acc = 0;
    const uint32_t *words = reinterpret_cast<const uint32_t *>(data + begin);
    const uint32_t nwords = (uint32_t)(n / 4);
    for (uint32_t w = 0; w < nwords; ++w) {
        const uint32_t v = __ldg(words + w);
#pragma unroll
        for (int b4 = 0; b4 < 4; ++b4) {
            const uint32_t y = (l ^ (v >> (8 * b4))) & 0xffu;                   // low byte of h ^ b
            acc = (acc + (uint64_t)(int64_t)((int32_t)y - (int32_t)l)) * FNV_PRIME;
            l = (y * 0xb3u) & 0xffu;
        }
    }
    for (uint64_t i = 4ull * nwords; i < n; ++i) {
        const uint32_t y = (l ^ (uint32_t)data[begin + i]) & 0xffu;
        acc = (acc + (uint64_t)(int64_t)((int32_t)y - (int32_t)l)) * FNV_PRIME;
        l = (y * 0xb3u) & 0xffu;
    }
    part[j] = acc;
    pw[j] = fnv_prime_power(n);
    __syncthreads();
    if (j == 0) {   // the chunk as one affine map h -> h * A + B, with A = P^(bytes of the chunk) implied by the plan
        uint64_t B = 0;
        for (int jj = 0; jj < FNV_SUB; ++jj) B = B * pw[jj] + part[jj];
        sums[c] = B;
    }
}

// <<<1, 1024>>>: h = h * P^n_c + acc_c over the chunks in order, as a tree of compositions of affine maps h -> h A + B.
__global__ void __launch_bounds__(1024) fnv_combine(FnvPlan p, const unsigned long long *__restrict__ sums, unsigned long long *out)
{
    __shared__ unsigned long long A[1024], B[1024];
    const uint32_t c = threadIdx.x;
    uint64_t a = 1, b = 0;
    if (c < p.nchunks) {
        const uint64_t begin = (uint64_t)c * p.chunk_bytes;
        const uint64_t n = p.nbytes - begin < p.chunk_bytes ? p.nbytes - begin : p.chunk_bytes;
        a = fnv_prime_power(n);
        b = sums[c];
    }
    A[c] = a;
    B[c] = b;
    __syncthreads();
    for (uint32_t step = 1; step < 1024; step <<= 1) {   // element c absorbs element c + step (the later bytes): (A1, B1) then (A2, B2)
        uint64_t a2 = 1, b2 = 0;
        const bool take = (c % (2 * step)) == 0 && c + step < 1024;
        if (take) { a2 = A[c + step]; b2 = B[c + step]; }
        __syncthreads();
        if (take) { B[c] = B[c] * a2 + b2; A[c] = A[c] * a2; }
        __syncthreads();
    }
    if (c == 0) *out = FNV_OFFSET * A[0] + B[0];
}

}  // namespace isingk
