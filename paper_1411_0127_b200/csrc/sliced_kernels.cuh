// sliced_kernels.cuh -- the paper's SLICED layout (Eq. 4-6; half-z labelling PAPER.md:150; neighbour index code
// Appendix A) as an alternative internal layout of the one-sample lattice, built to decide SURVEY.md 8(f) rank 4
// by measurement (profiles/r2f_sliced_layout.md).
//
//   x' = x,  y' = y - x,  z' = x - y + z   (mod L)        <=>        x = x',  y = y' + x',  z = z' + y'                     (Eq. 4)
// Planes of constant z' are one-coloured: (x + y + z) = z' (mod 2).  The two colours are separate arrays of L/2 planes of L x L
// sites, plane zz of colour c being z' = 2 zz + c (the pair of planes 2 zz, 2 zz + 1 shares the label zz), one bit per
// site, bit (r & 31) of word (r >> 5) with r = x' + L (y' + L zz): a row (fixed y', zz) is L/32 whole words of 32 consecutive x.
// The six neighbours of a site lie in TWO rows of the plane above and TWO rows of the plane below (Eq. 5):
//   +z (x', y', z'+1)    -y (x', y'-1, z'+1)    +x (x'+1, y'-1, z'+1)         -z (x', y', z'-1)    +y (x', y'+1, z'-1)    -x (x'-1, y'+1, z'-1)
// so a word needs the four aligned words U0 (y', up), U1 (y'-1, up), D0 (y', down), D1 (y'+1, down) of the other colour, U1 shifted
// down and D1 shifted up by one bit for the x neighbours (the bit that crosses a word comes from the neighbouring lane), where
// up / down = plane zz / zz - 1 of the other colour for a red word and zz + 1 / zz for a blue one.  Couplings sit at the site that
// owns them (bond (i, i + d)), as in the rank-linear layout: three own words, J-y at U1, J-z at D0, J-x at D1 (shifted with it).
//
// What the layout cannot do is carry the draw definition R9 cheaply: one Philox call serves four consecutive sites of a colour in
// CANONICAL row order (x, x+2, x+4, x+6 at fixed y, z), and consecutive bits of a sliced word are consecutive x at y = y' + x:
// 32 different canonical rows, hence 32 calls per word, each used for one of its four outputs (the paper's own remark: all
// schemes give the same bits only "after remapping all random numbers", fn. 47).  MINSTD, keyed per site (R11), is indifferent
// to the layout.  Both are implemented so that the cost is a number, not an argument.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sweep_kernels.cuh"

namespace isingk {

struct SlicedArrays {     // the eight sliced bit arrays, same sizes as LatticeArrays' (N/2 bits each)
    uint32_t *S[2];
    uint32_t *J[3][2];
};

// rank-linear position of the site with sliced coordinates (x', y', zz) of colour c: colour rank j (R9) and canonical index q
__device__ __forceinline__ void sliced_to_site(int L, int c, uint32_t xs, uint32_t ys, uint32_t zz, uint32_t &j, uint64_t &q)
{
    const uint32_t Lm = (uint32_t)L - 1u;   // L is a power of two times 64... any multiple of 32 works with % below; use & for 2^e
    const uint32_t x = xs, y = (ys + xs) % (uint32_t)L, z = (2u * zz + (uint32_t)c + ys) % (uint32_t)L;
    (void)Lm;
    j = (x >> 1) + (uint32_t)(L >> 1) * (y + (uint32_t)L * z);
    q = (uint64_t)x + (uint64_t)L * ((uint64_t)y + (uint64_t)L * z);
}

// rank-linear arrays -> sliced arrays, all eight; one thread per sliced word, one bit at a time (layout conversion of the
// experiment, not a hot path).  grid = ceil(8 * words / 256).
__global__ void __launch_bounds__(256) to_sliced_layout(const LatticeArrays A, const SlicedArrays B, int L)
{
    const uint32_t words = (uint32_t)(((uint64_t)L * L * L) >> 6);
    const uint32_t t = blockIdx.x * 256u + threadIdx.x;
    if (t >= 8u * words) return;
    const uint32_t arr = t / words, w = t - arr * words;
    const int kind = (int)(arr >> 1), c = (int)(arr & 1u);
    const uint32_t *src = kind == 0 ? A.S[c] : A.J[kind - 1][c];
    uint32_t *dst = kind == 0 ? B.S[c] : B.J[kind - 1][c];
    const uint32_t wpr = (uint32_t)L >> 5, row = w / wpr, k = w - row * wpr, zz = row / (uint32_t)L, ys = row - zz * (uint32_t)L;
    uint32_t out = 0;
    for (uint32_t b = 0; b < 32; ++b) {
        uint32_t j;
        uint64_t q;
        sliced_to_site(L, c, 32u * k + b, ys, zz, j, q);
        out |= ((__ldg(src + (j >> 5)) >> (j & 31u)) & 1u) << b;
    }
    dst[w] = out;
}

// sliced spins -> rank-linear spins; one thread per rank-linear word of either colour.
__global__ void __launch_bounds__(256) from_sliced_layout(const SlicedArrays B, const LatticeArrays A, int L)
{
    const uint32_t words = (uint32_t)(((uint64_t)L * L * L) >> 6);
    const uint32_t t = blockIdx.x * 256u + threadIdx.x;
    if (t >= 2u * words) return;
    const int c = t >= words;
    const uint32_t w = t - (c ? words : 0u);
    const uint32_t H = (uint32_t)L >> 1;
    uint32_t out = 0;
    for (uint32_t b = 0; b < 32; ++b) {
        const uint32_t j = 32u * w + b, m = j % H, r = j / H, y = r % (uint32_t)L, z = r / (uint32_t)L;
        const uint32_t x = 2u * m + ((y + z + (uint32_t)c) & 1u);
        const uint32_t xs = x, ys = (y + (uint32_t)L - x) % (uint32_t)L, zs = (x + (uint32_t)L - y + z) % (uint32_t)L;   // Eq. 4; zs = 2 zz + c
        const uint32_t rs = xs + (uint32_t)L * (ys + (uint32_t)L * (zs >> 1));
        out |= ((__ldg(B.S[c] + (rs >> 5)) >> (rs & 31u)) & 1u) << b;
    }
    A.S[c][w] = out;
}

// One colour half-sweep in the sliced layout.  A thread owns W consecutive words of a row; TPR = (L/32)/W lanes own a row (a
// power of two <= 32), a warp covers 32/TPR consecutive rows y' of a plane, the 8 warps of a CTA the next rows.
// grid = (L/2) * L * (L/32) / W / 256.  RNG 0 = Philox (R9: one call per site here), 1 = MINSTD stateless (R11, R12).
template <int RNG, int W>
__global__ void __launch_bounds__(256)
half_sweep_sliced(const __grid_constant__ SlicedArrays B, const __grid_constant__ SiteRng rng, int L, int colour, Thresholds T)
{
    const uint32_t wpr = (uint32_t)L >> 5, tpr = wpr / W, lane = threadIdx.x & 31u;
    const uint32_t tid = blockIdx.x * 256u + threadIdx.x;
    const uint32_t row = tid / tpr, lir = tid - row * tpr;          // row = y' + L zz
    const uint32_t zz = row / (uint32_t)L, ys = row - zz * (uint32_t)L, k0 = lir * W;
    const uint32_t Hz = (uint32_t)L >> 1;
    const int c = colour;
    const uint32_t z_up = c ? (zz + 1 == Hz ? 0u : zz + 1) : zz, z_dn = c ? zz : (zz == 0 ? Hz - 1 : zz - 1);
    const uint32_t y_m = ys == 0 ? (uint32_t)L - 1 : ys - 1, y_p = ys + 1 == (uint32_t)L ? 0u : ys + 1;
    const uint32_t w_own = wpr * (ys + (uint32_t)L * zz) + k0;
    const uint32_t w_u0 = wpr * (ys + (uint32_t)L * z_up) + k0, w_u1 = wpr * (y_m + (uint32_t)L * z_up) + k0;
    const uint32_t w_d0 = wpr * (ys + (uint32_t)L * z_dn) + k0, w_d1 = wpr * (y_p + (uint32_t)L * z_dn) + k0;
    const uint32_t *So = B.S[1 - c];
    wait_for_previous_kernel();
    uint32_t s[W], u0[W], u1[W], d0[W], d1[W], jxa[W], jya[W], jza[W], jyo[W], jzo[W], jxo[W];
    load_words<W>(B.S[c], w_own, s);
    load_words<W>(So, w_u0, u0);
    load_words<W>(So, w_u1, u1);
    load_words<W>(So, w_d0, d0);
    load_words<W>(So, w_d1, d1);
    load_words<W>(B.J[0][c], w_own, jxa);
    load_words<W>(B.J[1][c], w_own, jya);
    load_words<W>(B.J[2][c], w_own, jza);
    load_words<W>(B.J[1][1 - c], w_u1, jyo);
    load_words<W>(B.J[2][1 - c], w_d0, jzo);
    load_words<W>(B.J[0][1 - c], w_d1, jxo);
    uint32_t Bm[W];
#pragma unroll
    for (int k = 0; k < W; ++k) Bm[k] = jxo[k] ^ d1[k];
    // the bits that cross the thread's words: +x takes bit 0 of the next word of row (y'-1, up), -x bit 31 of the previous word
    // of row (y'+1, down); both periodic within the row
    uint32_t next_u1 = u1[0], prev_B = Bm[W - 1];
    if (tpr > 1) {
        const uint32_t base = lane & ~(tpr - 1u), l = lane & (tpr - 1u);
        next_u1 = __shfl_sync(0xFFFFFFFFu, next_u1, base | ((l + 1) & (tpr - 1u)));
        prev_B = __shfl_sync(0xFFFFFFFFu, prev_B, base | ((l + tpr - 1) & (tpr - 1u)));
    }
    uint32_t out[W];
#pragma unroll
    for (int k = 0; k < W; ++k) {
        const uint32_t up1_next = (k + 1 < W) ? u1[(k + 1) % W] : next_u1;
        const uint32_t B_prev = (k > 0) ? Bm[(k + W - 1) % W] : prev_B;
        const uint32_t J[6] = {jxa[k], 0u, jya[k], jyo[k], jza[k], jzo[k]};
        const uint32_t nb[6] = {__funnelshift_r(u1[k], up1_next, 1), __funnelshift_l(B_prev, Bm[k], 1), d1[k], u1[k], u0[k], d0[k]};
        uint32_t sum2, sum1, sum0, c4 = 0, c8 = 0, c12 = 0;
        satisfied_bond_count(s[k], J, nb, sum2, sum1, sum0);
        // bit b of this word: x = 32 (k0 + k) + b, y = (y' + x) mod L, z = (2 zz + c + y') mod L.  y wraps once at most inside a word
        // (at x = L - y'), so the canonical index q = x + L y + L^2 z and the colour rank j = (x >> 1) + (L/2)(y + L z) are
        // linear in b on each side of the wrap.
        const uint32_t x0 = 32u * (k0 + (uint32_t)k);
        const uint32_t z = (2u * zz + (uint32_t)c + ys) % (uint32_t)L;
        const uint32_t y0 = (ys + x0) % (uint32_t)L;                      // y of bit 0
        const uint32_t kw = (uint32_t)L - y0;                             // bits kw .. 31 (if kw < 32) have y = y0 + b - L
        if (RNG == 1) {
            const uint64_t qA = (uint64_t)x0 + (uint64_t)L * ((uint64_t)y0 + (uint64_t)L * z);
            const uint64_t qB = qA - (uint64_t)L * (uint64_t)L;          // referred to bit 0: q(b) = qB + b (1 + L) for b >= kw
            cond_masks_site_packed_minstd_two(rng.seed + (qA + 1) * SPLITMIX_GAMMA, rng.seed + (qB + 1) * SPLITMIX_GAMMA, kw < 32u ? kw : 32u,
                                              (uint64_t)(1 + L) * SPLITMIX_GAMMA, rng.A2, T, c4, c8, c12);
        } else {
            // R9: the draw of a site is output word j & 3 of the Philox call g = j >> 2.  Consecutive bits are in different canonical
            // rows: no two of them share a call.
#pragma unroll 4
            for (uint32_t b = 0; b < 32; ++b) {
                const uint32_t x = x0 + b, y = b < kw ? y0 + b : y0 + b - (uint32_t)L;
                const uint32_t j = (x >> 1) + ((uint32_t)L >> 1) * (y + (uint32_t)L * z);
                uint32_t R4[4];
                philox_folded(rng.pc, rng.ps, j >> 2, R4);
                const uint32_t R = (j & 2u) ? ((j & 1u) ? R4[3] : R4[2]) : ((j & 1u) ? R4[1] : R4[0]);
                if (R < T.t4) c4 |= 1u << b;
                if (R < T.t8) c8 |= 1u << b;
                if (R < T.t12) c12 |= 1u << b;
            }
            finish_cond(T, c4, c8, c12);
        }
        out[k] = s[k] ^ flip_mask(sum2, sum1, sum0, c4, c8, c12);
    }
    store_words<W>(B.S[c], w_own, out);
}

}  // namespace isingk
