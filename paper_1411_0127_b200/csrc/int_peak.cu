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
//   mix 12: IMAD (lo) + LOP3 1:1 on independent chains   mix 13: FFMA only   mix 14: FFMA + LOP3 1:1
//   mix 15: IMAD (lo) + IADD3 1:1   mix 16: IMAD (lo) + FFMA 1:1   (12-16: can the fma and alu pipes issue in the same cycles?)
//   mix 17: IMAD.HI + LOP3 1:1   mix 18: IMAD.HI + 3 LOP3   mix 19: IMAD.WIDE with the multiplier in a register
//   mix 20: DFMA only   mix 21: DFMA + LOP3 1:1   mix 22: IMAD.WIDE + IMAD (lo) 1:1   mix 23: Philox round from IMAD.HI + IMAD (lo)
//   plus 2 LOP3   mix 24: Philox round (register multipliers) + 4 LOP3   mix 25: IMAD.WIDE + FFMA 1:1
//   mix 26: IMAD.WIDE + 3 LOP3, all independent (17-26: which form of the 64-bit product overlaps with alu work?)
//   mix 27..29: the Philox round with hi32 from DFMA.RM and the state kept in register pairs whose high word is the
//           0x43300000 the DFMA result already carries (no moves), plus 0, 2, 4 extra LOP3
//   mix 30: 2 Philox rounds via IMAD.WIDE on one state + 2 rounds via DFMA.RM + IMAD (lo) on another (do the fma-heavy and
//           fp64 pipes take the two kinds of rounds side by side?)   mix 31: 3 IMAD.WIDE rounds per DFMA round (6 + 2)
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

// low word of the pair ^= x ^ k, in place (the high word, 0x43300000 from the DFMA, stays where it is)
__device__ __forceinline__ void xor_low_word(double &q, uint32_t x, uint32_t k)
{
    asm volatile("{ .reg .b32 lo, hi; mov.b64 {lo, hi}, %0; lop3.b32 lo, lo, %1, %2, 0x96; mov.b64 %0, {lo, hi}; }"
                 : "+d"(q) : "r"(x), "r"(k));
}

// Instructions per chain per iteration (fixed by the inline PTX; verified with cuobjdump):
//   mix 0: 4 LOP3    mix 1: 2 IMAD.WIDE    mix 2: 2 IMAD.WIDE + 2 LOP3 (two dependent steps)
//   mix 3: 2 IMAD.WIDE + 2 LOP3 (one Philox round)    mix 4: 2 x (ISETP + SEL) + 2 LOP3
//   mix 5: 2 IMAD.HI    mix 6: 2 IMAD    mix 7..10: 2 IMAD.WIDE + (3..6) LOP3    mix 11: 2 DFMA + 2 IMAD + 2 LOP3
//   mix 12: 2 IMAD + 2 LOP3    mix 13: 4 FFMA    mix 14: 2 FFMA + 2 LOP3    mix 15: 2 IMAD + 2 IADD3    mix 16: 2 IMAD + 2 FFMA
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
    double d[CHAINS], g[CHAINS];   // mixes 20, 21, 27-29 only
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) {
        d[c] = __hiloint2double(0x43300000, (int)a[c]);
        g[c] = __hiloint2double(0x43300000, (int)b[c]);
    }
    const double d0 = __hiloint2double(0x3ff00000, (int)k0), d1 = __hiloint2double(0x3fe00000, (int)k1);
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
            } else if (MIX == 12) {
                asm volatile("mad.lo.u32 %0, %0, 0xD2511F53, %1;" : "+r"(a[c]) : "r"(k0));
                b[c] = lop3_xor3(b[c], k0, k1);
                asm volatile("mad.lo.u32 %0, %0, 0xCD9E8D57, %1;" : "+r"(a[c]) : "r"(k1));
                e[c] = lop3_xor3(e[c], k1, k0);
            } else if (MIX == 13) {
                float fa = __uint_as_float(a[c]), fb = __uint_as_float(b[c]);
                const float f0 = __uint_as_float(k0), f1 = __uint_as_float(k1);
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fa) : "f"(f0), "f"(f1));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fb) : "f"(f1), "f"(f0));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fa) : "f"(f1), "f"(f0));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fb) : "f"(f0), "f"(f1));
                a[c] = __float_as_uint(fa);
                b[c] = __float_as_uint(fb);
            } else if (MIX == 14) {
                float fa = __uint_as_float(a[c]);
                const float f0 = __uint_as_float(k0), f1 = __uint_as_float(k1);
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fa) : "f"(f0), "f"(f1));
                b[c] = lop3_xor3(b[c], k0, k1);
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fa) : "f"(f1), "f"(f0));
                e[c] = lop3_xor3(e[c], k1, k0);
                a[c] = __float_as_uint(fa);
            } else if (MIX == 15) {
                asm volatile("mad.lo.u32 %0, %0, 0xD2511F53, %1;" : "+r"(a[c]) : "r"(k0));
                asm volatile("{ .reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2; }" : "+r"(b[c]) : "r"(k0), "r"(k1));
                asm volatile("mad.lo.u32 %0, %0, 0xCD9E8D57, %1;" : "+r"(a[c]) : "r"(k1));
                asm volatile("{ .reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2; }" : "+r"(e[c]) : "r"(k1), "r"(k0));
            } else if (MIX == 16) {
                float fb = __uint_as_float(b[c]);
                const float f0 = __uint_as_float(k0), f1 = __uint_as_float(k1);
                asm volatile("mad.lo.u32 %0, %0, 0xD2511F53, %1;" : "+r"(a[c]) : "r"(k0));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fb) : "f"(f0), "f"(f1));
                asm volatile("mad.lo.u32 %0, %0, 0xCD9E8D57, %1;" : "+r"(a[c]) : "r"(k1));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fb) : "f"(f1), "f"(f0));
                b[c] = __float_as_uint(fb);
            } else if (MIX == 17 || MIX == 18) {
                asm volatile("mul.hi.u32 %0, %0, 0xD2511F53;" : "+r"(a[c]));
                b[c] = lop3_xor3(b[c], k0, k1);
                if (MIX == 18) { b[c] = lop3_xor3(b[c], k1, k0); b[c] = lop3_xor3(b[c], k0, k1); }
                asm volatile("mul.hi.u32 %0, %0, 0xCD9E8D57;" : "+r"(a[c]));
                e[c] = lop3_xor3(e[c], k1, k0);
                if (MIX == 18) { e[c] = lop3_xor3(e[c], k0, k1); e[c] = lop3_xor3(e[c], k1, k0); }
            } else if (MIX == 19) {
                uint32_t h, l;
                mul_wide(a[c], k0, h, l);
                mul_wide(h, k1, a[c], b[c]);
            } else if (MIX == 20) {
                asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[c]) : "d"(d0), "d"(d1));
                asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[c]) : "d"(d1), "d"(d0));
            } else if (MIX == 21) {
                asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[c]) : "d"(d0), "d"(d1));
                b[c] = lop3_xor3(b[c], k0, k1);
                asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[c]) : "d"(d1), "d"(d0));
                e[c] = lop3_xor3(e[c], k1, k0);
            } else if (MIX == 22) {
                uint32_t h, l;
                mul_wide(a[c], 0xD2511F53u, h, l);
                asm volatile("mad.lo.u32 %0, %0, 0xD2511F53, %1;" : "+r"(b[c]) : "r"(k0));
                mul_wide(h ^ l, 0xCD9E8D57u, h, l);
                a[c] = h ^ l;
                asm volatile("mad.lo.u32 %0, %0, 0xCD9E8D57, %1;" : "+r"(e[c]) : "r"(k1));
            } else if (MIX == 23) {
                uint32_t h0, h1, l0, l1;
                asm volatile("mul.hi.u32 %0, %1, 0xD2511F53;" : "=r"(h0) : "r"(a[c]));
                asm volatile("mul.lo.u32 %0, %1, 0xD2511F53;" : "=r"(l0) : "r"(b[c]));
                asm volatile("mul.hi.u32 %0, %1, 0xCD9E8D57;" : "=r"(h1) : "r"(b[c]));
                asm volatile("mul.lo.u32 %0, %1, 0xCD9E8D57;" : "=r"(l1) : "r"(a[c]));
                a[c] = lop3_xor3(h1, l0, k0);
                b[c] = lop3_xor3(h0, l1, k1);
                e[c] = lop3_xor3(e[c], k0, k1);
                e[c] = lop3_xor3(e[c], k1, k0);
            } else if (MIX == 24) {
                uint32_t h0, l0, h1, l1;
                mul_wide(a[c], k0, h0, l0);
                mul_wide(b[c], k1, h1, l1);
                a[c] = lop3_xor3(h1, l0, k0);
                b[c] = lop3_xor3(h0, l1, k1);
#pragma unroll
                for (int x = 0; x < 4; ++x) e[c] = lop3_xor3(e[c], k0, k1);
            } else if (MIX == 25) {
                uint32_t h, l;
                float fb = __uint_as_float(b[c]);
                const float f0 = __uint_as_float(k0), f1 = __uint_as_float(k1);
                mul_wide(a[c], 0xD2511F53u, h, l);
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fb) : "f"(f0), "f"(f1));
                mul_wide(h ^ l, 0xCD9E8D57u, h, l);
                a[c] = h ^ l;
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(fb) : "f"(f1), "f"(f0));
                b[c] = __float_as_uint(fb);
            } else if (MIX == 26) {
                uint32_t h, l;
                mul_wide(a[c], 0xD2511F53u, h, l);
                a[c] = h;
                b[c] = lop3_xor3(b[c], k0, k1);
                b[c] = lop3_xor3(b[c], k1, k0);
                e[c] = lop3_xor3(e[c], k1, k0);
            } else if (MIX >= 27 && MIX <= 29) {
                const double Ms0 = 3528531795.0 * 0x1p-32, K0 = 0x1p52 - 3528531795.0 * 0x1p20;   // M0 = 0xD2511F53
                const double Ms1 = 3449720151.0 * 0x1p-32, K1 = 0x1p52 - 3449720151.0 * 0x1p20;   // M1 = 0xCD9E8D57
#pragma unroll
                for (int rr = 0; rr < 2; ++rr) {   // two rounds, so that the register pairs return to their places
                    double P = __fma_rd(d[c], Ms0, K0), Q = __fma_rd(g[c], Ms1, K1);
                    const uint32_t l0 = (uint32_t)__double2loint(d[c]) * 0xD2511F53u, l1 = (uint32_t)__double2loint(g[c]) * 0xCD9E8D57u;
                    xor_low_word(Q, l0, k0);
                    xor_low_word(P, l1, k1);
                    d[c] = Q;
                    g[c] = P;
#pragma unroll
                    for (int x = 0; x < 2 * (MIX - 27); ++x) e[c] = lop3_xor3(e[c], k0, k1);
                }
            } else if (MIX == 30 || MIX == 31) {
                const double Ms0 = 3528531795.0 * 0x1p-32, K0 = 0x1p52 - 3528531795.0 * 0x1p20;   // M0 = 0xD2511F53
                const double Ms1 = 3449720151.0 * 0x1p-32, K1 = 0x1p52 - 3449720151.0 * 0x1p20;   // M1 = 0xCD9E8D57
#pragma unroll
                for (int rr = 0; rr < 2; ++rr) {
                    double P = __fma_rd(d[c], Ms0, K0), Q = __fma_rd(g[c], Ms1, K1);
                    const uint32_t l0 = (uint32_t)__double2loint(d[c]) * 0xD2511F53u, l1 = (uint32_t)__double2loint(g[c]) * 0xCD9E8D57u;
                    xor_low_word(Q, l0, k0);
                    xor_low_word(P, l1, k1);
                    d[c] = Q;
                    g[c] = P;
#pragma unroll
                    for (int ww = 0; ww < (MIX == 30 ? 1 : 3); ++ww) {
                        uint32_t h0, l0w, h1, l1w;
                        mul_wide(a[c], 0xD2511F53u, h0, l0w);
                        mul_wide(b[c], 0xCD9E8D57u, h1, l1w);
                        a[c] = lop3_xor3(h1, l0w, k0);
                        b[c] = lop3_xor3(h0, l1w, k1);
                    }
                }
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
    for (int c = 0; c < CHAINS; ++c) r ^= a[c] ^ b[c] ^ e[c] ^ (uint32_t)__double2loint(d[c]) ^ (uint32_t)__double2loint(g[c]);
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
    const double ops_per_iter[32] = {4.0 * CHAINS, 2.0 * CHAINS, 4.0 * CHAINS, 4.0 * CHAINS, 6.0 * CHAINS, 2.0 * CHAINS,
                                     2.0 * CHAINS, 5.0 * CHAINS, 6.0 * CHAINS, 7.0 * CHAINS, 8.0 * CHAINS, 6.0 * CHAINS,
                                     4.0 * CHAINS, 4.0 * CHAINS, 4.0 * CHAINS, 4.0 * CHAINS, 4.0 * CHAINS,
                                     4.0 * CHAINS, 8.0 * CHAINS, 2.0 * CHAINS, 2.0 * CHAINS, 4.0 * CHAINS, 6.0 * CHAINS,
                                     8.0 * CHAINS, 8.0 * CHAINS, 6.0 * CHAINS, 4.0 * CHAINS,
                                     12.0 * CHAINS, 16.0 * CHAINS, 20.0 * CHAINS, 20.0 * CHAINS, 36.0 * CHAINS};
    if (mix < 0 || mix > 31) return -1;
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
            case 11: int_mix_kernel<11><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 12: int_mix_kernel<12><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 13: int_mix_kernel<13><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 14: int_mix_kernel<14><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 15: int_mix_kernel<15><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 16: int_mix_kernel<16><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 17: int_mix_kernel<17><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 18: int_mix_kernel<18><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 19: int_mix_kernel<19><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 20: int_mix_kernel<20><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 21: int_mix_kernel<21><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 22: int_mix_kernel<22><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 23: int_mix_kernel<23><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 24: int_mix_kernel<24><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 25: int_mix_kernel<25><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 26: int_mix_kernel<26><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 27: int_mix_kernel<27><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 28: int_mix_kernel<28><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 29: int_mix_kernel<29><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            case 30: int_mix_kernel<30><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
            default: int_mix_kernel<31><<<ctas, 256>>>(d_scratch, iters, 0x1234567u, 0x89abcdefu); break;
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
