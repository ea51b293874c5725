// int_peak.cu -- integer issue-rate microbenchmark for the ALU roofline of the half-sweep kernel (SURVEY.md 8(d):
// "the INT32 peak of sm_100 is not in MEASURED_PEAKS.json; it must be measured on the box").
//
// Each kernel runs, per thread, ITERS iterations of 8 independent dependency chains of one instruction mix, so that the
// result is bound by issue / pipe throughput and not by latency.  The host entry returns thread-instructions per second.
//   mix 0: LOP3 only (alu pipe)            mix 1: IMAD.WIDE.U32 only (fma pipe)
//   mix 2: LOP3 + IMAD.WIDE.U32 1:1        mix 3: the Philox round (2 IMAD.WIDE + 2 LOP3 on two chains)
//   mix 4: ISETP + SEL pairs (an acceptance-bit insert)
//   mix 5: IMAD.HI.U32 only           mix 6: IMAD (lo) only
//   mix 7..10: the Philox round plus 1..4 extra independent LOP3 (do the alu and fma pipes overlap?)
//   mix 11: the Philox round with hi32 of the products from the FP64 pipe (DFMA.RM of (2^52 + c) * M*2^-32 + 2^52 - M*2^20,
//           exact) and lo32 from IMAD: the variant DESIGN.md section 6 lists as tried and rejected
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int CHAINS = 8;

__device__ __forceinline__ uint32_t lop3_xor3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ void mul_wide(uint32_t a, uint32_t m, uint32_t &hi, uint32_t &lo)
{
    uint64_t p;
    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(m));
    hi = (uint32_t)(p >> 32);
    lo = (uint32_t)p;
}
__device__ __forceinline__ uint32_t setp_sel(uint32_t r, uint32_t t, uint32_t bit)
{
    uint32_t d;
    asm volatile("{ .reg .pred p; setp.lt.u32 p, %1, %2; selp.u32 %0, %3, 0, p; }" : "=r"(d) : "r"(r), "r"(t), "r"(bit));
    return d;
}

// Instructions per chain per iteration (fixed by the inline PTX; verified with cuobjdump):
//   mix 0: 4 LOP3    mix 1: 2 IMAD.WIDE    mix 2: 2 IMAD.WIDE + 2 LOP3 (two dependent steps)
//   mix 3: 2 IMAD.WIDE + 2 LOP3 (one Philox round)    mix 4: 2 x (ISETP + SEL) + 2 LOP3
//   mix 5: 2 IMAD.HI    mix 6: 2 IMAD    mix 7..10: 2 IMAD.WIDE + (3..6) LOP3    mix 11: 2 DFMA + 2 IMAD + 2 LOP3
template <int MIX>
__global__ void __launch_bounds__(256) int_mix_kernel(uint32_t *out, int iters, uint32_t k0, uint32_t k1)
{
    uint32_t a[CHAINS], b[CHAINS], e[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) {
        a[c] = threadIdx.x * 2654435761u + c * 40503u + blockIdx.x;
        b[c] = a[c] ^ 0x9E3779B9u;
        e[c] = a[c] + 17u;
    }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < CHAINS; ++c) {
            if (MIX == 0) {
                a[c] = lop3_xor3(a[c], b[c], k0);
                b[c] = lop3_xor3(b[c], a[c], k1);
                a[c] = lop3_xor3(a[c], b[c], k1);
                b[c] = lop3_xor3(b[c], a[c], k0);
            } else if (MIX == 1) {
                uint32_t h, l;
                mul_wide(a[c], 0xD2511F53u, h, l);
                mul_wide(h, 0xCD9E8D57u, a[c], b[c]);
            } else if (MIX == 2) {
                uint32_t h, l;
                mul_wide(a[c], 0xD2511F53u, h, l);
                a[c] = lop3_xor3(h, l, k0);
                mul_wide(a[c], 0xCD9E8D57u, h, l);
                a[c] = lop3_xor3(h, l, k1);
            } else if (MIX == 3) {
                uint32_t h0, l0, h1, l1;
                mul_wide(a[c], 0xD2511F53u, h0, l0);
                mul_wide(b[c], 0xCD9E8D57u, h1, l1);
                a[c] = lop3_xor3(h1, l0, k0);
                b[c] = lop3_xor3(h0, l1, k1);
            } else if (MIX == 4) {
                b[c] = lop3_xor3(b[c], setp_sel(a[c], k0, 4u), k1);
                a[c] = lop3_xor3(a[c], setp_sel(b[c], k1, 8u), k0);
            } else if (MIX == 5) {
                asm volatile("mul.hi.u32 %0, %0, 0xD2511F53;" : "+r"(a[c]));
                asm volatile("mul.hi.u32 %0, %0, 0xCD9E8D57;" : "+r"(b[c]));
            } else if (MIX == 6) {
                asm volatile("mul.lo.u32 %0, %0, 0xD2511F53;" : "+r"(a[c]));
                asm volatile("mul.lo.u32 %0, %0, 0xCD9E8D57;" : "+r"(b[c]));
            } else if (MIX >= 7 && MIX <= 10) {
                uint32_t h0, l0, h1, l1;
                mul_wide(a[c], 0xD2511F53u, h0, l0);
                mul_wide(b[c], 0xCD9E8D57u, h1, l1);
                a[c] = lop3_xor3(h1, l0, k0);
                b[c] = lop3_xor3(h0, l1, k1);
#pragma unroll
                for (int x = 0; x < MIX - 6; ++x) e[c] = lop3_xor3(e[c], k0, k1);
            } else {
                const double Ms0 = 3528531795.0 * 0x1p-32, K0 = 0x1p52 - 3528531795.0 * 0x1p20;   // M0 = 0xD2511F53
                const double Ms1 = 3449720151.0 * 0x1p-32, K1 = 0x1p52 - 3449720151.0 * 0x1p20;   // M1 = 0xCD9E8D57
                const uint32_t h0 = (uint32_t)__double2loint(__fma_rd(__hiloint2double(0x43300000, (int)a[c]), Ms0, K0));
                const uint32_t h1 = (uint32_t)__double2loint(__fma_rd(__hiloint2double(0x43300000, (int)b[c]), Ms1, K1));
                const uint32_t l0 = a[c] * 0xD2511F53u, l1 = b[c] * 0xCD9E8D57u;
                a[c] = lop3_xor3(h1, l0, k0);
                b[c] = lop3_xor3(h0, l1, k1);
            }
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) r ^= a[c] ^ b[c] ^ e[c];
    if (r == 0x12345u) out[0] = r;  // never true in practice; keeps the results observable
}

}  // namespace

extern "C" {

// Runs mix `mix` on `ctas` CTAs of 256 threads for `iters` iterations, `reps` times; returns the best launch time in ms
// in *ms_out.  d_scratch: >= 4 bytes of device memory.  Source-level operations per thread per iteration are returned
// in *ops_out (the SASS count is checked with cuobjdump; see profiles/).
int int_peak_run(int mix, int ctas, int iters, int reps, uint32_t *d_scratch, float *ms_out, double *ops_out)
{
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -2;
    float best = 1e30f;
    const double ops_per_iter[12] = {4.0 * CHAINS, 2.0 * CHAINS, 4.0 * CHAINS, 4.0 * CHAINS, 6.0 * CHAINS, 2.0 * CHAINS,
                                     2.0 * CHAINS, 5.0 * CHAINS, 6.0 * CHAINS, 7.0 * CHAINS, 8.0 * CHAINS, 6.0 * CHAINS};
    if (mix < 0 || mix > 11) return -1;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0);
        switch (mix) {
            case 0: int_mix_kernel<0><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 1: int_mix_kernel<1><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 2: int_mix_kernel<2><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 3: int_mix_kernel<3><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 4: int_mix_kernel<4><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 5: int_mix_kernel<5><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 6: int_mix_kernel<6><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 7: int_mix_kernel<7><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 8: int_mix_kernel<8><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 9: int_mix_kernel<9><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 10: int_mix_kernel<10><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            default: int_mix_kernel<11><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
        }
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) return -2;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms_out = best;
    *ops_out = ops_per_iter[mix] * (double)iters * 256.0 * (double)ctas;
    return 0;
}
}
