// sweep_kernels.cuh -- the colour half-sweep kernels.
//
// Internal layout.  Sites are split by colour c = (x+y+z)&1 and numbered within their colour by
// the colour rank j = (x>>1) + (L/2)*(y + L*z)  (the same j that keys the Philox counter, R9).  Per lattice there are
// 8 bit arrays indexed by j: spins S[c] and couplings Jd[c], d = x,y,z, where Jd[c] holds the bond (i, i+d-hat) of
// the colour-c site i.
//   site-packed   (nsamples = 1):  bit (j&31) of word (j>>5); for L a multiple of 64 a half-row (fixed y,z) is L/64 words.
//   sample-packed (nsamples = 32k): word j of batch b holds samples 32b..32b+31 of site j.
// An active site of colour c in a row of parity p = (y+z)&1 has x = 2m + xodd, xodd = c^p.  Its +-y and +-z neighbours
// have the same m in the other colour's arrays; its two x-neighbours are bits m and m-1 (xodd = 0) or m and m+1
// (xodd = 1) of the other colour's half-row.
//
// Kernels: half_sweep_site_packed<RNG, W> (L a multiple of 64; RNG 0 = Philox, 1 = MINSTD stateless, 2 = MINSTD with cached
// seed states), minstd_fill_s0<W>, half_sweep_site_packed_rows<RNG> (every other even L: operands gathered as bit windows),
// half_sweep_site_packed_generic<RNG> (one site at a time; kernel choice 1), half_sweep_sample_packed<RNG, PARTS> (any L;
// RNG 2 = shared draw, R18), half_sweep_sample_packed_vec<RNG, PARTS, MULTI> (L % 8 == 0, 128-bit loads, optionally all coded
// batches in one launch), half_sweep_shared_vec<FLAT> (shared draw, 128-bit loads, all coded batches in one launch).
// The lane-generator kernels (rng modes 3, 4) are in lane_rng.cuh.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "update.cuh"

namespace isingk {

struct LatticeArrays {  // one lattice (site-packed) or one batch of 32 samples (sample-packed)
    uint32_t *S[2];
    uint32_t *J[3][2];
};

struct RngLaunch {  // per-launch PRNG constants, passed by value (constant bank)
    PhiloxCommonConst pc;
    PhiloxSampleConst ps[32];  // one per sample of the batch; the generic site-packed and the shared-draw kernels use ps[0] only
    uint64_t seed;             // MINSTD
    uint32_t A;                // MINSTD: 16807^(n+1) mod M for the sweep n = t>>1 of this launch
    uint32_t tlo, thi;         // half-sweep counter (generic kernel: unfolded Philox)
    uint32_t k0, k1base;       // Philox key: k1 = k1base ^ sample
    uint32_t sample_base;      // first sample of this batch (sample-packed)
};

struct SweepArgs {
    uint32_t *S_act;           // active colour spins (read + written)
    const uint32_t *S_oth;     // other colour spins
    const uint32_t *J_act[3];  // couplings owned by the active colour: bonds (i, i+d)
    const uint32_t *J_oth[3];  // couplings owned by the other colour: bonds (i-d, i) seen from the active site i
    int L;
    int colour;
    Thresholds T;
    // z-slab handles only (SLAB variants of the kernels; slab_kernels.cuh): the arrays hold the planes z0 - 1 .. z0 + Lz of the
    // lattice (local plane 0 and Lz + 1 are halos), and a launch covers the rows of CTAs by_first + blockIdx.y * by_stride
    int z0, by_first, by_stride;
};

// ---------------------------------------------------------------------------------------------------
// Word-parallel kernel, site-packed, L a multiple of 64.  One thread owns W consecutive words of one half-row
// (W = 4: one 128-bit load per operand array); TPR = (L/64)/W consecutive lanes own a row, and the bit that crosses
// a word boundary in x comes from the neighbouring lane by a warp shuffle (or from the thread's own words when it
// owns the whole row).  A warp covers 32/TPR consecutive y, the 8 warps of a CTA cover 8 consecutive z, so most
// +-y / +-z operand words are L1 hits and every word leaves HBM once per half-sweep (profiles/: DRAM bytes per launch
// = 9N/16).  The kernel is bound by integer issue (Philox: 18 IMAD.WIDE + 19 LOP3 per 4 sites), so it is laid out to
// execute as few other instructions as possible: the 12 operand vectors are loaded first, the field sums of all W
// words are reduced to three bit planes each (22 logic ops per 32 sites), and only then the random numbers are drawn.
// ---------------------------------------------------------------------------------------------------
// The word-parallel site-packed kernel spreads its per-CTA atomics over ACC_SLOTS counter pairs (one address would
// serialise 16384 atomics in L2 at L = 1024); the last CTA adds them up.
constexpr int ACC_SLOTS = 64;

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

// Last-CTA finalisation shared by energy_site_packed and the measuring half-sweep: the CTAs have added their counts to the
// slots; the last one to finish (ticket counter behind the slots) sums them, writes E = 2 * unsatisfied - 3N and
// M = 2 * up - N (R16) and clears slots and ticket for the next call.
__device__ __forceinline__ void finalize_slots_last_cta(unsigned long long *acc, long long N, long long *E, long long *M)
{
    __shared__ bool is_last;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(acc + 2 * ACC_SLOTS);
    if (threadIdx.x == 0) {
        __threadfence();
        is_last = atomicAdd(ticket, 1u) == gridDim.x * gridDim.y - 1;  // every other CTA's atomics are visible then
    }
    __syncthreads();
    if (is_last && threadIdx.x < 32) {  // warp 0 of the last CTA: read-and-clear the slots, two per lane
        unsigned long long tu = 0, tp = 0;
        for (int k = threadIdx.x; k < ACC_SLOTS; k += 32) {
            tu += atomicExch(&acc[2 * k], 0ull);
            tp += atomicExch(&acc[2 * k + 1], 0ull);
        }
        warp_reduce_add2(tu, tp);
        if (threadIdx.x == 0) {
            if (E) E[0] = 2 * (long long)tu - 3 * N;
            if (M) M[0] = 2 * (long long)tp - N;
            *ticket = 0u;
        }
    }
}

// A recording half-sweep adds its counts straight into the record: E[0] and M[0] were pre-set to -3N and -N (init_records) and
// receive 2 x (unsatisfied bonds) and 2 x (up spins) (R16) by one atomic pair per CTA.  Nothing waits for the sum: no ticket, no
// last-CTA pass (that tail cost a recording launch 1.5 us at L = 256).
__device__ __forceinline__ void add_to_record(unsigned long long unsat, unsigned long long up, long long *E, long long *M)
{
    __shared__ unsigned long long cta_sum[2];
    if (threadIdx.x == 0) { cta_sum[0] = 0; cta_sum[1] = 0; }
    __syncthreads();
    block_accumulate2(unsat, up, cta_sum);   // warp 0 adds the CTA's totals to cta_sum; thread 0 then sees its own adds
    if (threadIdx.x == 0) {
        if (E) atomicAdd(reinterpret_cast<unsigned long long *>(E), 2ull * cta_sum[0]);
        if (M) atomicAdd(reinterpret_cast<unsigned long long *>(M), 2ull * cta_sum[1]);
    }
}

__global__ void init_records(long long *E, long long *M, uint32_t n, long long N)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    if (E) E[r] = -3 * N;
    if (M) M[r] = -N;
}

template <int W> struct WordVec;
template <> struct WordVec<1> { typedef uint32_t type; };
template <> struct WordVec<2> { typedef uint2 type; };
template <> struct WordVec<4> { typedef uint4 type; };
template <int W> struct IsVectorWidth { static constexpr bool value = W == 1 || W == 2 || W == 4; };

// W = 3 or 5 words per thread (rows of 3 * 2^e or 5 * 2^e words, L = 192, 320, 384, 640, 768, 1280, ...): the thread's
// words are not a power-of-two vector, so they move as W 32-bit accesses.
template <int W>
__device__ __forceinline__ void load_words_scalar(const uint32_t *__restrict__ p, size_t word_off, uint32_t out[W])
{
#pragma unroll
    for (int k = 0; k < W; ++k) out[k] = __ldg(p + word_off + k);
}

template <int W>
__device__ __forceinline__ void load_words(const uint32_t *__restrict__ p, size_t word_off, uint32_t out[W])
{
    if constexpr (!IsVectorWidth<W>::value) {
        load_words_scalar<W>(p, word_off, out);
    } else {
        typedef typename WordVec<W>::type V;
        const V v = __ldg(reinterpret_cast<const V *>(p + word_off));
        const uint32_t *pv = reinterpret_cast<const uint32_t *>(&v);
#pragma unroll
        for (int k = 0; k < W; ++k) out[k] = pv[k];
    }
}

// Spin words.  COHERENT = false: the read-only path (ld.global.nc), for kernels that run one half-sweep per launch.
// COHERENT = true: ld.global.cg (served by the L2, the point of coherence), for the persistent kernels in which other CTAs
// rewrite the spin arrays between the half-sweeps of ONE launch: neither the non-coherent path nor a stale L1 line may
// serve such a load.  (Couplings never change during a launch and always take the read-only path.)
template <int W, bool COHERENT>
__device__ __forceinline__ void load_spin_words(const uint32_t *p, size_t word_off, uint32_t out[W])
{
    if constexpr (!COHERENT) {
        load_words<W>(p, word_off, out);
    } else if constexpr (!IsVectorWidth<W>::value) {
#pragma unroll
        for (int k = 0; k < W; ++k) out[k] = __ldcg(p + word_off + k);
    } else {
        typedef typename WordVec<W>::type V;
        const V v = __ldcg(reinterpret_cast<const V *>(p + word_off));
        const uint32_t *pv = reinterpret_cast<const uint32_t *>(&v);
#pragma unroll
        for (int k = 0; k < W; ++k) out[k] = pv[k];
    }
}

// 128-bit load of words that are read exactly once per half-sweep (couplings, the active spins): ld.global.cs, evict-first,
// so that they do not displace what is re-read (the other colour's spins, the lane generators' state) from the L2.
__device__ __forceinline__ void load_words4_streaming(const uint32_t *__restrict__ p, size_t word_off, uint32_t out[4])
{
    const uint4 v = __ldcs(reinterpret_cast<const uint4 *>(p + word_off));
    out[0] = v.x; out[1] = v.y; out[2] = v.z; out[3] = v.w;
}

template <int W>
__device__ __forceinline__ void store_words(uint32_t *p, size_t word_off, const uint32_t in[W])
{
    if constexpr (!IsVectorWidth<W>::value) {
#pragma unroll
        for (int k = 0; k < W; ++k) p[word_off + k] = in[k];
    } else {
        typedef typename WordVec<W>::type V;
        V out;
        uint32_t *po = reinterpret_cast<uint32_t *>(&out);
#pragma unroll
        for (int k = 0; k < W; ++k) po[k] = in[k];
        *reinterpret_cast<V *>(p + word_off) = out;
    }
}

struct SiteRng {  // per-launch PRNG constants of the site-packed kernel (one sample)
    PhiloxCommonConst pc;
    PhiloxSampleConst ps;
    uint64_t seed;  // MINSTD
    uint32_t A2;    // MINSTD: 2 * (16807^(n+1) mod M) for the sweep n = t>>1 of this launch
    uint4 *s0tab;   // MINSTD with cached seeds (RNG = 2): seed states s0 of the active colour, see minstd_s0_index
    uint32_t b_hi, e_hi;   // Philox, lattices beyond L = 2048 (BIG): ps.b, ps.e for the groups g >= 2^32 (counter word c3 = 1, R9)
};

// Cached MINSTD seed states (RNG = 2).  s0 = (SplitMix64(seed, site) >> 34) + 1 (R11) does not depend on time, so it
// can be computed once per handle and streamed from HBM (4 B per site per sweep) instead of being recomputed (about
// 17 integer instructions per site per sweep).  The table is laid out for the thread mapping of the kernel: the
// 16-byte element (warp w of the grid, word k of the thread, bits 4q..4q+3, lane l) is at ((w*W + k)*8 + q)*32 + l,
// so every load instruction of a warp reads 512 contiguous bytes.
template <int W>
__device__ __forceinline__ size_t minstd_s0_index(uint32_t warp_global, int k, int q, int lane)
{
    return (((size_t)warp_global * W + k) * 8 + q) * 32 + lane;
}

constexpr int SWEEP_THREADS = 256;

// Programmatic dependent launch: a half-sweep launched with the programmatic-stream-serialization attribute may start
// its CTAs (index arithmetic) while the previous half-sweep drains; it must not touch the lattice before this point.
// Without the attribute this is a no-op.
__device__ __forceinline__ void wait_for_previous_kernel() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Eq. 15 for the shared-random-number mode (R18): one draw per site decides for all 32 samples of
// the word, so cond4 / cond8 / cond12 are all-ones or zero words.
__device__ __forceinline__ void shared_cond_words(const uint32_t R[4], const Thresholds &T, uint32_t c4[4], uint32_t c8[4],
                                                  uint32_t c12[4])
{
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        c4[w] = R[w] < T.t4 ? 0xFFFFFFFFu : 0u;
        c8[w] = R[w] < T.t8 ? 0xFFFFFFFFu : 0u;
        c12[w] = R[w] < T.t12 ? 0xFFFFFFFFu : 0u;
    }
}

// Thread mapping of the word-parallel kernels (half-sweep, seed table, energy), any L that is a multiple of 64: a row of
// wpr = L/64 words is owned by tpr = wpr/W consecutive lanes.  When tpr is not a power of two (L = 192, 320, 384, ...)
// the row is padded to tpr_pad = the next power of two lanes; the idle lanes shadow lane 0 of the row (their loads stay
// in bounds) and store nothing.  grid = (L / (32 / tpr_pad), L / 8), 256 threads.
struct RowMap {
    int lane, warp, tpr, tpr_pad, lane_in_row, y, z, k0;
    int next_lane, prev_lane;  // lanes owning the next / previous words of the row (periodic)
    bool active;
};

inline int row_map_tpr_pad(int tpr)
{
    int p = 1;
    while (p < tpr) p <<= 1;
    return p;
}

template <int W>
__device__ __forceinline__ RowMap row_map(int L, uint32_t bx, uint32_t by)
{
    RowMap m;
    m.tpr = (L >> 6) / W;
    const int lg = m.tpr <= 1 ? 0 : 32 - __clz(m.tpr - 1);
    m.tpr_pad = 1 << lg;
    m.lane = threadIdx.x & 31;
    m.warp = threadIdx.x >> 5;
    const int lir = m.lane & (m.tpr_pad - 1);
    m.active = lir < m.tpr;
    m.lane_in_row = m.active ? lir : 0;
    m.y = (int)bx * (32 >> lg) + (m.lane >> lg);
    m.z = (int)by * (SWEEP_THREADS / 32) + m.warp;
    m.k0 = m.lane_in_row * W;
    const int base = m.lane & ~(m.tpr_pad - 1);
    m.next_lane = base | (m.lane_in_row + 1 == m.tpr ? 0 : m.lane_in_row + 1);
    m.prev_lane = base | (m.lane_in_row == 0 ? m.tpr - 1 : m.lane_in_row - 1);
    return m;
}

// MEASURE: the half-sweep also returns E and M of the configuration it leaves (row a9 fused into rows a2-a8).  Every bond has
// exactly one end in the active colour, so the number of satisfied bonds of the whole lattice is the sum over the active
// sites of their count n (already in the three bit planes), with n -> 6 - n where the site flipped; the up spins are those of
// the new active words plus the other colour's words of the same rows, which are loaded anyway.  About 15 popcounts per
// word, then the slot accumulation and last-CTA finalisation of energy_site_packed: a trace of E and M per sweep costs no
// extra launch and no extra pass over the 512 MiB (L = 1024: 78 us per record saved).
// Four CTAs per SM (64 registers) for the Philox kernel the L = 1024 numbers are quoted on (0.3899 -> 0.3868 ms per half-sweep, 8 bytes
// of spill); the other variants keep ptxas' own choice (W = 5 would spill 40 bytes).
// The update of one tile = the rows of one (virtual) CTA (bx, by) of the grid (L / (32 / tpr_pad), L / 8): the body of
// half_sweep_site_packed (one tile per CTA) and of persistent_site_packed (a CTA walks over tiles, half-sweep after
// half-sweep; COHERENT spin loads, see load_spin_words).  gx = x extent of that grid.  m_unsat / m_up (MEASURE): this
// thread's unsatisfied bonds and up spins are ADDED to them.
// SLAB: the arrays are those of a z-slab (see SweepArgs): the tile's planes are stored one plane up (the lower halo is plane 0),
// their z-neighbours are simply the planes below and above (halos at the ends, no wrap), and everything keyed by the site -- the
// colour of a row, the Philox counter, the MINSTD stream ids -- uses the plane's z in the whole lattice.
// BIG: lattices beyond L = 2048, whose Philox group index g = 8 x (word index) + q reaches 2^32: the words from index 2^29 on
// take the constants folded for the counter word c3 = hi32(g) = 1 (R9; fold_philox).  Nothing else changes: the word index itself
// stays below 2^30 up to L = 4096, and the MINSTD stream ids are 64-bit anyway.
template <int RNG, int W, bool MEASURE, bool COHERENT, bool SLAB = false, bool BIG = false>
__device__ __forceinline__ void site_packed_tile(const SweepArgs &a, const SiteRng &rng, uint32_t bx, uint32_t by, uint32_t gx,
                                                 unsigned long long &m_unsat, unsigned long long &m_up_out)
{
    const int L = a.L;
    const int wpr = L >> 6;                 // words per half-row
    const RowMap rm = row_map<W>(L, bx, by);
    const int tpr = rm.tpr, lane = rm.lane, warp = rm.warp, y = rm.y, k0 = rm.k0;
    const int z = SLAB ? rm.z + 1 : rm.z;          // plane in the arrays
    const int zg = SLAB ? rm.z + a.z0 : rm.z;      // plane in the lattice

    const int yp = y + 1 == L ? 0 : y + 1, ym = y == 0 ? L - 1 : y - 1;
    const int zp = SLAB ? z + 1 : (z + 1 == L ? 0 : z + 1), zm = SLAB ? z - 1 : (z == 0 ? L - 1 : z - 1);
    const uint32_t row = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * z) + k0;   // < 2^27 words for L <= 2048
    const uint32_t row_yp = (uint32_t)wpr * ((uint32_t)yp + (uint32_t)L * z) + k0;
    const uint32_t row_ym = (uint32_t)wpr * ((uint32_t)ym + (uint32_t)L * z) + k0;
    const uint32_t row_zp = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * zp) + k0;
    const uint32_t row_zm = (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * zm) + k0;
    const uint32_t row_g = SLAB ? (uint32_t)wpr * ((uint32_t)y + (uint32_t)L * zg) + k0 : row;   // the row's words in the lattice

    uint32_t s[W], sum2[W], sum1[W], sum0[W];
    unsigned int m_sat = 0, m_up = 0;   // MEASURE: satisfied bonds of this thread's sites, up spins of both colours
    const int xodd = (y + zg + a.colour) & 1;
    if (!COHERENT) wait_for_previous_kernel();
    {
        uint32_t o[W], oyp[W], oym[W], ozp[W], ozm[W];
        uint32_t jxa[W], jya[W], jza[W], jxo[W], jyo[W], jzo[W];
        load_spin_words<W, COHERENT>(a.S_act, row, s);
        load_spin_words<W, COHERENT>(a.S_oth, row, o);
        load_words<W>(a.J_oth[0], row, jxo);
        load_words<W>(a.J_act[0], row, jxa);
        load_spin_words<W, COHERENT>(a.S_oth, row_yp, oyp);
        load_spin_words<W, COHERENT>(a.S_oth, row_ym, oym);
        load_spin_words<W, COHERENT>(a.S_oth, row_zp, ozp);
        load_spin_words<W, COHERENT>(a.S_oth, row_zm, ozm);
        load_words<W>(a.J_act[1], row, jya);
        load_words<W>(a.J_act[2], row, jza);
        load_words<W>(a.J_oth[1], row_ym, jyo);
        load_words<W>(a.J_oth[2], row_zm, jzo);

        // x-neighbours (row a3).  An active site with bit m has x = 2m + xodd.  xodd = 0: its +x neighbour is bit m of
        // the other colour's half-row and its -x neighbour bit m-1, whose coupling is owned by that neighbour, so the
        // word B = jxo ^ o is shifted up by one bit.  xodd = 1: -x is bit m (word B unshifted) and +x is bit m+1, so
        // the word o is shifted down by one bit.  Both are funnel shifts by xodd / 1 - xodd; the bit entering at the
        // end of the thread's words comes from the neighbouring lane of the row (periodic).
        uint32_t B[W];
#pragma unroll
        for (int k = 0; k < W; ++k) B[k] = jxo[k] ^ o[k];
        uint32_t edge = xodd ? o[0] : B[W - 1];
        if (tpr > 1) edge = __shfl_sync(0xFFFFFFFFu, edge, xodd ? rm.next_lane : rm.prev_lane);
        const uint32_t sh_r = (uint32_t)xodd, sh_l = 1u - (uint32_t)xodd;
#pragma unroll
        for (int k = 0; k < W; ++k) {
            const uint32_t o_next = (k + 1 < W) ? o[(k + 1) % W] : edge;
            const uint32_t B_prev = (k > 0) ? B[(k + W - 1) % W] : edge;
            const uint32_t J[6] = {jxa[k], 0u, jya[k], jyo[k], jza[k], jzo[k]};
            const uint32_t nb[6] = {__funnelshift_r(o[k], o_next, sh_r), __funnelshift_l(B_prev, B[k], sh_l), oyp[k], oym[k], ozp[k],
                                    ozm[k]};
            satisfied_bond_count(s[k], J, nb, sum2[k], sum1[k], sum0[k]);
            if (MEASURE) m_up += __popc(o[k]);
        }
    }
    // after the flips f of a word: sum of n' = sum of n + 6 popc(f) - 2 (sum of n over the flipped bits)
    auto measure_word = [&](int k, uint32_t f) {
        m_sat += __popc(sum0[k]) + 2 * __popc(sum1[k]) + 4 * __popc(sum2[k]) + 6 * __popc(f);
        m_sat -= 2 * (__popc(sum0[k] & f) + 2 * __popc(sum1[k] & f) + 4 * __popc(sum2[k] & f));
        m_up += __popc(s[k]);
    };

    const uint64_t row_site0 = (uint64_t)L * ((uint64_t)y + (uint64_t)L * zg) + (uint64_t)xodd;  // MINSTD stream ids
    // RNG = 2: the seed states of all W words come from the table; RNG = 0, 1: every word draws in registers.
    constexpr int WC = RNG == 2 ? W : 0;
    // seeds from the table, two groups of 16 sites in flight: while one half-word's draws are compared, the next
    // half-word's four 16-byte loads are outstanding (about 2 KB per warp, enough to keep HBM busy)
    const uint32_t warp_global = (by * gx + bx) * (SWEEP_THREADS / 32) + warp;
    const uint4 *tab = rng.s0tab;
    uint4 cur[4], nxt[4];
    if (WC > 0) {
#pragma unroll
        for (int i = 0; i < 4; ++i) cur[i] = __ldcs(tab + minstd_s0_index<W>(warp_global, 0, i, lane));
    }
    // The two thresholds every draw is compared with live in ordinary registers (row < 2^27, so the OR adds nothing; it
    // only keeps them out of the uniform register file, which the 19 Philox constants fill: ptxas otherwise reloads
    // them from the constant bank after every rare-path branch).
    Thresholds Tr = a.T;
    Tr.t4 |= row >> 31;
    Tr.t8 |= row >> 31;
    PhiloxCommonConst pcr = rng.pc;
    PhiloxSampleConst psr = rng.ps;
    if (RNG == 0) {  // likewise the round keys of the last two rounds
        pcr.k0[5] |= row >> 31;
        pcr.k0[6] |= row >> 31;
        psr.k1[5] |= row >> 31;
        psr.k1[6] |= row >> 31;
        psr.k1[7] |= row >> 31;
    }
#pragma unroll
    for (int k = WC; k < W; ++k) {
        uint32_t c4, c8, c12;
        if (RNG == 0) {
            if (BIG) {
                PhiloxSampleConst psw = psr;
                const bool hi = ((row_g + (uint32_t)k) >> 29) != 0u;
                psw.b = hi ? rng.b_hi : psr.b;
                psw.e = hi ? rng.e_hi : psr.e;
                cond_masks_site_packed_philox(pcr, psw, row_g + (uint32_t)k, Tr, c4, c8, c12);
            } else {
                cond_masks_site_packed_philox(pcr, psr, row_g + (uint32_t)k, Tr, c4, c8, c12);
            }
        } else {
            const uint64_t site0 = row_site0 + 64ull * (uint64_t)(k0 + k);
            cond_masks_site_packed_minstd(rng.seed + (site0 + 1) * SPLITMIX_GAMMA, 2 * SPLITMIX_GAMMA, rng.A2, a.T, c4, c8, c12);
        }
        const uint32_t f = flip_mask(sum2[k], sum1[k], sum0[k], c4, c8, c12);
        s[k] ^= f;
        if (MEASURE) measure_word(k, f);
    }

    if (WC > 0) {
        uint32_t c4 = 0, c8 = 0, c12 = 0;
#pragma unroll
        for (int h = 0; h < 2 * WC; ++h) {
            const int k = h >> 1, half = h & 1;
            if (h + 1 < 2 * WC) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    nxt[i] = __ldcs(tab + minstd_s0_index<W>(warp_global, (h + 1) >> 1, 4 * ((h + 1) & 1) + i, lane));
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint32_t R[4] = {minstd_mulmod2(rng.A2, cur[i].x), minstd_mulmod2(rng.A2, cur[i].y),
                                       minstd_mulmod2(rng.A2, cur[i].z), minstd_mulmod2(rng.A2, cur[i].w)};
                accumulate_cond<4>(R, 16 * half + 4 * i, a.T, c4, c8, c12);
            }
            if (half) {
                finish_cond(a.T, c4, c8, c12);
                const uint32_t f = flip_mask(sum2[k], sum1[k], sum0[k], c4, c8, c12);
                s[k] ^= f;
                if (MEASURE) measure_word(k, f);
                c4 = 0; c8 = 0; c12 = 0;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) cur[i] = nxt[i];
        }
    }
    if (rm.active) store_words<W>(a.S_act, row, s);
    if (MEASURE && rm.active) {
        // unsatisfied bonds = 6 per active site - satisfied; idle lanes of a padded row shadow lane 0 and count nothing
        m_unsat += 192ull * W - m_sat;
        m_up_out += m_up;
    }
}

template <int RNG, int W, bool MEASURE, bool BIG = false>
__global__ void __launch_bounds__(SWEEP_THREADS, RNG == 0 && W == 4 && !MEASURE ? 4 : 0)
half_sweep_site_packed(const __grid_constant__ SweepArgs a, const __grid_constant__ SiteRng rng, unsigned long long *acc, long long N,
                       long long *E, long long *M)
{
    unsigned long long unsat = 0, up = 0;
    site_packed_tile<RNG, W, MEASURE, false, false, BIG>(a, rng, blockIdx.x, blockIdx.y, gridDim.x, unsat, up);
    if (MEASURE) add_to_record(unsat, up, E, M);
}

// Fills the seed table of colour `colour` with the thread mapping of half_sweep_site_packed<2, W> (same grid).
// z0: the lattice plane of the grid's first plane (0, or the first owned plane of a z-slab, whose table covers its own planes).
template <int W>
__global__ void __launch_bounds__(SWEEP_THREADS) minstd_fill_s0(uint4 *tab, int L, int colour, uint64_t seed, int z0 = 0)
{
    const RowMap rm = row_map<W>(L, blockIdx.x, blockIdx.y);
    const int lane = rm.lane, warp = rm.warp, y = rm.y, z = rm.z + z0, k0 = rm.k0;
    const int xodd = (y + z + colour) & 1;
    const uint64_t row_site0 = (uint64_t)L * ((uint64_t)y + (uint64_t)L * z) + (uint64_t)xodd;
    const uint32_t warp_global = (blockIdx.y * gridDim.x + blockIdx.x) * (SWEEP_THREADS / 32) + warp;
#pragma unroll 1
    for (int k = 0; k < W; ++k) {
        const uint64_t weyl0 = seed + (row_site0 + 64ull * (uint64_t)(k0 + k) + 1) * SPLITMIX_GAMMA;
#pragma unroll 1
        for (int q = 0; q < 8; ++q) {
            uint4 v;
            v.x = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 0) * (2 * SPLITMIX_GAMMA));
            v.y = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 1) * (2 * SPLITMIX_GAMMA));
            v.z = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 2) * (2 * SPLITMIX_GAMMA));
            v.w = minstd_seed_state_from_weyl(weyl0 + (uint64_t)(4 * q + 3) * (2 * SPLITMIX_GAMMA));
            __stcs(tab + minstd_s0_index<W>(warp_global, k, q, lane), v);
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Generic kernel, site-packed, any even L >= 4: one thread per word of the active colour, one site at a time with
// the scalar rule (dE = 2 sigma_i h_i, Eq. 8) and the unfolded Philox.  Slow; it serves lattices whose half-rows
// are not whole words (L = 16) and, in the tests, as a second GPU implementation with a different layout access
// and thread mapping (all schemes must give the same bits).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ int get_bit(const uint32_t *__restrict__ p, uint64_t j)
{
    return (int)((p[j >> 5] >> (j & 31)) & 1u);
}

__device__ __forceinline__ uint64_t colour_rank(int L, int x, int y, int z)
{
    return (uint64_t)(x >> 1) + (uint64_t)(L >> 1) * ((uint64_t)y + (uint64_t)L * (uint64_t)z);
}

template <int RNG>
__global__ void __launch_bounds__(256)
half_sweep_site_packed_generic(const SweepArgs a, const __grid_constant__ RngLaunch rng, uint64_t n_words, uint64_t Hc)
{
    const uint64_t widx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (widx >= n_words) return;
    const int L = a.L, H = L >> 1;
    wait_for_previous_kernel();
    uint32_t word = a.S_act[widx];
    uint32_t flips = 0;
    uint32_t R4[4] = {0, 0, 0, 0};
    for (int b = 0; b < 32; ++b) {
        const uint64_t j = 32 * widx + b;
        if (j >= Hc) break;
        const int m = (int)(j % H);
        const uint64_t r = j / H;
        const int y = (int)(r % L), z = (int)(r / L);
        const int x = 2 * m + ((y + z + a.colour) & 1);
        const int xp = (x + 1 == L) ? 0 : x + 1, xm = (x == 0) ? L - 1 : x - 1;
        const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
        const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
        const uint64_t jn[6] = {colour_rank(L, xp, y, z), colour_rank(L, xm, y, z), colour_rank(L, x, yp, z),
                                colour_rank(L, x, ym, z), colour_rank(L, x, y, zp), colour_rank(L, x, y, zm)};
        int h = 0;  // local field sum_k J_ik sigma_k, sigma = 2 bit - 1, J = 1 - 2 bit (Eq. 10)
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            const int sk = 2 * get_bit(a.S_oth, jn[d]) - 1;
            const int Jb = (d & 1) ? get_bit(a.J_oth[d >> 1], jn[d]) : get_bit(a.J_act[d >> 1], j);
            h += (1 - 2 * Jb) * sk;
        }
        const int si = 2 * (int)((word >> b) & 1u) - 1;
        const int dE = 2 * si * h;
        uint32_t R;
        if (RNG == 0) {
            if ((b & 3) == 0)
                philox4x32_10(rng.tlo, rng.thi, (uint32_t)(j >> 2), (uint32_t)(j >> 34), rng.k0, rng.k1base, R4);
            R = R4[b & 3];
        } else {
            const uint64_t q = (uint64_t)x + (uint64_t)L * ((uint64_t)y + (uint64_t)L * (uint64_t)z);
            R = minstd_mulmod(rng.A, minstd_seed_state_from_weyl(rng.seed + (q + 1) * SPLITMIX_GAMMA));
        }
        bool acc;
        if (dE <= 0) acc = true;
        else if (dE == 4) acc = (R < a.T.t4) || a.T.always4;
        else if (dE == 8) acc = (R < a.T.t8) || a.T.always8;
        else acc = (R < a.T.t12) || a.T.always12;
        if (acc) flips |= 1u << b;
    }
    a.S_act[widx] = word ^ flips;
}

// ---------------------------------------------------------------------------------------------------
// Site-packed, any even L (rows of L/2 bits that do not fill whole words: L = 16, 96, 250, ...): the word update of the
// word-parallel kernel on operands gathered as bit windows.  The colour arrays are rank-linear (bit j of the array =
// colour rank j), so a word covers 32 consecutive ranks, i.e. one or more row segments; within a segment every neighbour
// set is a contiguous bit range of the other colour's array (the same columns of the row y+-1 / z+-1, or the row itself
// shifted by one bit for +-x, with the periodic bit patched in), fetched as an unaligned 32-bit window (two loads and a
// funnel shift).  The draws are those of cond_masks_site_packed_philox (word w = ranks 32w .. 32w+31, R9) or, for
// MINSTD, one evaluation per segment with the canonical site index of its first bit (R11).  The paper's point that the
// scheme must work for every L = 2n, not only powers of two, is what this kernel is for: about
// 1 ps/flip instead of 12-55 for the one-site-at-a-time kernel it replaces (kernel choice 1 still selects that one).
// ---------------------------------------------------------------------------------------------------
// PLAIN = false: loads through the read-only path (global arrays that no one writes during the launch); PLAIN = true: ordinary
// loads through a generic pointer (arrays staged in shared memory by half_sweeps_on_chip, which are rewritten between half-sweeps).
template <bool PLAIN>
__device__ __forceinline__ uint32_t load_word(const uint32_t *a, uint32_t w)
{
    if constexpr (PLAIN) return a[w];
    else return __ldg(a + w);
}
template <bool PLAIN = false>
__device__ __forceinline__ uint32_t bit_window(const uint32_t *a, uint32_t pos)
{   // bits pos .. pos+31 of the bit array (bits past the array's end are garbage that the caller masks out)
    const uint32_t w = pos >> 5, sh = pos & 31u;
    const uint32_t lo = load_word<PLAIN>(a, w);
    const uint32_t hi = sh ? load_word<PLAIN>(a, w + 1) : 0u;
    return __funnelshift_r(lo, hi, sh);
}
template <bool PLAIN = false>
__device__ __forceinline__ uint32_t bit_at(const uint32_t *a, uint32_t pos) { return (load_word<PLAIN>(a, pos >> 5) >> (pos & 31u)) & 1u; }

// The update of word w (colour ranks 32 w .. 32 w + 31); returns the new word.  PLAIN: see load_word.  VOTE: the rare branch of
// the acceptance is taken after a warp vote (all 32 lanes of the warp must be here) or per thread.
template <int RNG, bool PLAIN, bool VOTE>
__device__ __forceinline__ uint32_t rows_word_update(const SweepArgs &a, const SiteRng &rng, uint32_t w, uint32_t Hc)
{
    const uint32_t L = (uint32_t)a.L, H = L >> 1, LH = L * H;
    const uint32_t j0 = 32u * w;
    uint32_t remaining = Hc - j0 < 32u ? Hc - j0 : 32u, bitoff = 0;
    uint32_t r = j0 / H, m = j0 - r * H, z = r / L, y = r - z * L;
    const uint32_t s = load_word<PLAIN>(a.S_act, w);
    uint32_t J[6] = {load_word<PLAIN>(a.J_act[0], w), 0u, load_word<PLAIN>(a.J_act[1], w), 0u, load_word<PLAIN>(a.J_act[2], w), 0u};
    uint32_t nb[6] = {0u, 0u, 0u, 0u, 0u, 0u};
    uint32_t c4 = 0, c8 = 0, c12 = 0;
    while (remaining > 0) {
        const uint32_t len = remaining < H - m ? remaining : H - m;
        const uint32_t segmask = (len == 32u ? 0xFFFFFFFFu : ((1u << len) - 1u)) << bitoff;
        const uint32_t xodd = (y + z + (uint32_t)a.colour) & 1u;
        const uint32_t P = r * H;                                   // rank of the first site of this row
        const uint32_t Pyp = (y + 1 == L) ? P - (LH - H) : P + H, Pym = (y == 0) ? P + (LH - H) : P - H;
        const uint32_t Pzp = (z + 1 == L) ? P - (Hc - LH) : P + LH, Pzm = (z == 0) ? P + (Hc - LH) : P - LH;
        // +x: column m + xodd of the same row; the last column wraps to column 0 when xodd = 1
        uint32_t wpx = bit_window<PLAIN>(a.S_oth, P + m + xodd);
        if (xodd && m + len == H) wpx = (wpx & ~(1u << (len - 1))) | (bit_at<PLAIN>(a.S_oth, P) << (len - 1));
        // -x: column m - 1 + xodd with its own coupling; column 0 wraps to column H-1 when xodd = 0
        uint32_t wmx, jmx;
        if (xodd) {
            wmx = bit_window<PLAIN>(a.S_oth, P + m);
            jmx = bit_window<PLAIN>(a.J_oth[0], P + m);
        } else if (m == 0) {
            wmx = (bit_window<PLAIN>(a.S_oth, P) << 1) | bit_at<PLAIN>(a.S_oth, P + H - 1);
            jmx = (bit_window<PLAIN>(a.J_oth[0], P) << 1) | bit_at<PLAIN>(a.J_oth[0], P + H - 1);
        } else {
            wmx = bit_window<PLAIN>(a.S_oth, P + m - 1);
            jmx = bit_window<PLAIN>(a.J_oth[0], P + m - 1);
        }
        nb[0] |= (wpx << bitoff) & segmask;
        nb[1] |= (wmx << bitoff) & segmask;
        J[1] |= (jmx << bitoff) & segmask;
        nb[2] |= (bit_window<PLAIN>(a.S_oth, Pyp + m) << bitoff) & segmask;
        nb[3] |= (bit_window<PLAIN>(a.S_oth, Pym + m) << bitoff) & segmask;
        J[3] |= (bit_window<PLAIN>(a.J_oth[1], Pym + m) << bitoff) & segmask;
        nb[4] |= (bit_window<PLAIN>(a.S_oth, Pzp + m) << bitoff) & segmask;
        nb[5] |= (bit_window<PLAIN>(a.S_oth, Pzm + m) << bitoff) & segmask;
        J[5] |= (bit_window<PLAIN>(a.J_oth[2], Pzm + m) << bitoff) & segmask;
        if (RNG == 1) {   // MINSTD: stream id = canonical site index; bit b of the word is site0 + 2 (b - bitoff)
            const uint64_t site0 = (uint64_t)L * r + 2u * m + xodd - 2ull * bitoff;
            uint32_t d4, d8, d12;
            // no warp vote here: the threads of a warp run this loop a different number of times when L/2 does not divide 32
            cond_masks_site_packed_minstd<false>(rng.seed + (site0 + 1) * SPLITMIX_GAMMA, 2 * SPLITMIX_GAMMA, rng.A2, a.T, d4, d8, d12);
            c4 |= d4 & segmask;
            c8 |= d8 & segmask;
            c12 |= d12 & segmask;
        }
        bitoff += len;
        remaining -= len;
        m += len;
        if (m == H) {
            m = 0;
            ++r;
            if (++y == L) { y = 0; ++z; }
        }
    }
    if (RNG == 0) cond_masks_site_packed_philox<VOTE>(rng.pc, rng.ps, w, a.T, c4, c8, c12);
    uint32_t sum2, sum1, sum0;
    satisfied_bond_count(s, J, nb, sum2, sum1, sum0);
    const uint32_t valid = bitoff == 32u ? 0xFFFFFFFFu : (1u << bitoff) - 1u;   // the last word of the array may be partial
    return s ^ (flip_mask(sum2, sum1, sum0, c4, c8, c12) & valid);
}

template <int RNG>
__global__ void __launch_bounds__(128)
half_sweep_site_packed_rows(const SweepArgs a, const __grid_constant__ SiteRng rng, uint32_t n_words, uint32_t Hc)
{
    const uint32_t w = blockIdx.x * 128u + threadIdx.x;
    if (w >= n_words) return;
    wait_for_previous_kernel();
    a.S_act[w] = rows_word_update<RNG, false, true>(a, rng, w, Hc);
}

// ---------------------------------------------------------------------------------------------------
// The same for rows of at least 32 bits (L >= 64), without the segment loop: a word then lies in one row or straddles two
// (bits 0..k-1 in row A, bits k..31 in row B), and in rank space its neighbour sets are ALMOST contiguous over both:
//   +-y, +-z: rank j + off with the same offset for both rows unless one of them sits at a periodic boundary (3 of L
//             straddling words): one unaligned window, a second one only in that rare case;
//   +-x:      ranks j-1, j, j+1 of the other colour are the aligned word itself and its two one-bit shifts; which of them a
//             bit takes depends on the x parity of its row (mask X); the periodic bit at a row end / row start inside the
//             word is patched in.
// The segment loop of half_sweep_site_packed_rows makes every warp pay for two segments as soon as one of its 32 words
// straddles (always, for L < 2048); here the straddle costs a few mask operations: 933 -> 711 instructions per word (ncu).
// ---------------------------------------------------------------------------------------------------
// MEASURE: E and M of the resulting configuration, as in half_sweep_site_packed<.., MEASURE = true>.
template <int RNG, bool MEASURE>
__global__ void __launch_bounds__(128)
half_sweep_site_packed_rows2(const SweepArgs a, const __grid_constant__ SiteRng rng, uint32_t n_words, uint32_t Hc,
                             unsigned long long *acc, long long N, long long *E, long long *M)
{
    const uint32_t w_raw = blockIdx.x * 128u + threadIdx.x;
    if (!MEASURE && w_raw >= n_words) return;
    const bool live = w_raw < n_words;                 // MEASURE: every thread reaches the block reduction
    const uint32_t w = live ? w_raw : n_words - 1;
    const uint32_t L = (uint32_t)a.L, H = L >> 1, LH = L * H;
    const uint32_t j0 = 32u * w;
    const uint32_t rA = j0 / H, m0 = j0 - rA * H, zA = rA / L, yA = rA - zA * L;
    const uint32_t nvalid = Hc - j0 < 32u ? Hc - j0 : 32u;
    const uint32_t k = H - m0;                                   // bits 0..k-1 are in row A
    const bool two = k < nvalid;                                 // bits k.. are in row B = the next row
    uint32_t yB = yA + 1, zB = zA;
    if (yB == L) { yB = 0; ++zB; }
    const uint32_t xoddA = (yA + zA + (uint32_t)a.colour) & 1u, xoddB = (yB + zB + (uint32_t)a.colour) & 1u;
    const uint32_t maskA = k >= 32u ? 0xFFFFFFFFu : (1u << k) - 1u, maskB = ~maskA;
    const uint32_t X = (xoddA ? maskA : 0u) | (xoddB ? maskB : 0u);   // x parity of every bit's site
    const uint32_t PA = rA * H;                                  // rank of the first site of row A; row B starts at PA + H
    wait_for_previous_kernel();
    const uint32_t s = __ldg(a.S_act + w);
    uint32_t J[6], nb[6];
    J[0] = __ldg(a.J_act[0] + w);
    J[2] = __ldg(a.J_act[1] + w);
    J[4] = __ldg(a.J_act[2] + w);
    uint32_t other_word;                               // the other colour's word of the same ranks (MEASURE: its up spins)
    {   // +-x
        const uint32_t lo = __ldg(a.S_oth + w), hi = __ldg(a.S_oth + w + 1), prev = w ? __ldg(a.S_oth + w - 1) : 0u;
        other_word = lo;
        const uint32_t jlo = __ldg(a.J_oth[0] + w), jprev = w ? __ldg(a.J_oth[0] + w - 1) : 0u;
        nb[0] = (X & __funnelshift_r(lo, hi, 1)) | (~X & lo);
        nb[1] = (X & lo) | (~X & __funnelshift_l(prev, lo, 1));
        J[1] = (X & jlo) | (~X & __funnelshift_l(jprev, jlo, 1));
        if (k <= 32u && xoddA) nb[0] = (nb[0] & ~(1u << (k - 1))) | (bit_at(a.S_oth, PA) << (k - 1));   // row A ends here: +x wraps
        if (m0 == 0 && !xoddA) {                                                                        // row A starts here: -x wraps
            nb[1] = (nb[1] & ~1u) | bit_at(a.S_oth, PA + H - 1);
            J[1] = (J[1] & ~1u) | bit_at(a.J_oth[0], PA + H - 1);
        }
        if (two && !xoddB) {                                                                            // row B starts at bit k
            nb[1] = (nb[1] & ~(1u << k)) | (bit_at(a.S_oth, PA + 2 * H - 1) << k);
            J[1] = (J[1] & ~(1u << k)) | (bit_at(a.J_oth[0], PA + 2 * H - 1) << k);
        }
    }
    {   // +-y, +-z: offsets in rank space (mod 2^32), per row
        const uint32_t ypA = (yA + 1 == L) ? 0u - (LH - H) : H, ypB = (yB + 1 == L) ? 0u - (LH - H) : H;
        const uint32_t ymA = (yA == 0) ? LH - H : 0u - H, ymB = (yB == 0) ? LH - H : 0u - H;
        const uint32_t zpA = (zA + 1 == L) ? 0u - (Hc - LH) : LH, zpB = (zB + 1 == L) ? 0u - (Hc - LH) : LH;
        const uint32_t zmA = (zA == 0) ? Hc - LH : 0u - LH, zmB = (zB == 0) ? Hc - LH : 0u - LH;
        nb[2] = bit_window(a.S_oth, j0 + ypA);
        nb[3] = bit_window(a.S_oth, j0 + ymA);
        J[3] = bit_window(a.J_oth[1], j0 + ymA);
        nb[4] = bit_window(a.S_oth, j0 + zpA);
        nb[5] = bit_window(a.S_oth, j0 + zmA);
        J[5] = bit_window(a.J_oth[2], j0 + zmA);
        if (two && (ypA != ypB || ymA != ymB || zpA != zpB || zmA != zmB)) {   // a periodic boundary between the two rows: rare
            // row B's windows start at its first bit k (j0 + offset alone may lie before the array)
            const uint32_t jB = j0 + k;
            nb[2] = (nb[2] & maskA) | (bit_window(a.S_oth, jB + ypB) << k);
            nb[3] = (nb[3] & maskA) | (bit_window(a.S_oth, jB + ymB) << k);
            J[3] = (J[3] & maskA) | (bit_window(a.J_oth[1], jB + ymB) << k);
            nb[4] = (nb[4] & maskA) | (bit_window(a.S_oth, jB + zpB) << k);
            nb[5] = (nb[5] & maskA) | (bit_window(a.S_oth, jB + zmB) << k);
            J[5] = (J[5] & maskA) | (bit_window(a.J_oth[2], jB + zmB) << k);
        }
    }
    uint32_t c4, c8, c12;
    if (RNG == 0) {
        cond_masks_site_packed_philox(rng.pc, rng.ps, w, a.T, c4, c8, c12);
    } else {   // MINSTD: canonical site index of bit b = site0 + 2b within its row; both bases are referred to bit 0
        const uint64_t siteA = (uint64_t)L * rA + 2u * m0 + xoddA;
        const uint64_t siteB = (uint64_t)L * (rA + 1) + xoddB - 2ull * k;
        cond_masks_site_packed_minstd_two(rng.seed + (siteA + 1) * SPLITMIX_GAMMA, rng.seed + (siteB + 1) * SPLITMIX_GAMMA, k,
                                          2 * SPLITMIX_GAMMA, rng.A2, a.T, c4, c8, c12);
    }
    uint32_t sum2, sum1, sum0;
    satisfied_bond_count(s, J, nb, sum2, sum1, sum0);
    const uint32_t valid = nvalid == 32u ? 0xFFFFFFFFu : (1u << nvalid) - 1u;
    const uint32_t f = flip_mask(sum2, sum1, sum0, c4, c8, c12) & valid;
    if (live) a.S_act[w] = s ^ f;
    if (MEASURE) {
        sum0 &= valid;
        sum1 &= valid;
        sum2 &= valid;
        const unsigned sat = __popc(sum0) + 2 * __popc(sum1) + 4 * __popc(sum2) + 6 * __popc(f) -
                             2 * (__popc(sum0 & f) + 2 * __popc(sum1 & f) + 4 * __popc(sum2 & f));
        const unsigned long long unsat = live ? 6ull * nvalid - sat : 0ull;
        const unsigned long long up = live ? (unsigned long long)(__popc((s ^ f) & valid) + __popc(other_word & valid)) : 0ull;
        add_to_record(unsat, up, E, M);
    }
}

// ---------------------------------------------------------------------------------------------------
// Sample-packed kernel (nsamples = 32 per batch), any even L >= 4.  A Philox group g = 4 consecutive same-colour sites
// j = 4g..4g+3 needs one call per sample (bit), keyed by the sample (R9).  Neighbours are whole words, so no
// x-alignment is needed.  A CTA has 4 warps.  PARTS = 1: one thread per group, all 32 samples (large lattices: index
// arithmetic, 52 loads and the field logic are paid once per 32 calls).  PARTS = 4: lane = group, warp p = samples
// 8p..8p+7 (warp-uniform Philox constants), each warp updates byte p of its groups' words; the loads of the four warps
// coincide (L1 hits).  This spreads a small lattice (config 2: 32768 groups) over every SM.
// ---------------------------------------------------------------------------------------------------
// Loads and field sums of the group g (colour ranks 4g .. 4g+3), sample-packed, any even L: the four sites may lie in
// different rows, so every site computes its own six neighbour ranks.  site[w] = canonical index of site w (MINSTD ids).
__device__ __forceinline__ void group_sums_any_L(const SweepArgs &a, uint32_t g, uint32_t s[4], uint32_t sum2[4], uint32_t sum1[4],
                                                 uint32_t sum0[4], uint64_t site[4])
{
    const uint32_t L = (uint32_t)a.L, H = L >> 1, HL = H * L, Hc = HL * L;  // Hc = N/2 < 2^32 for L <= 2048
    const uint32_t j0 = 4u * g;
    uint32_t m = j0 % H;
    const uint32_t r0 = j0 / H;
    uint32_t y = r0 % L, z = r0 / L;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t j = j0 + w;
        const uint32_t xodd = (y + z + (uint32_t)a.colour) & 1u;
        // colour ranks of the six neighbours (other colour): same row for +-x, rows y+-1 and planes z+-1 otherwise
        const uint32_t rowbase = j - m;
        const uint32_t m_other = xodd ? (m + 1 == H ? 0u : m + 1) : (m == 0 ? H - 1 : m - 1);
        const uint32_t jxp = rowbase + (xodd ? m_other : m), jxm = rowbase + (xodd ? m : m_other);
        const uint32_t jyp = (y + 1 == L) ? j - (HL - H) : j + H, jym = (y == 0) ? j + (HL - H) : j - H;
        const uint32_t jzp = (z + 1 == L) ? j - (Hc - HL) : j + HL, jzm = (z == 0) ? j + (Hc - HL) : j - HL;
        const uint32_t jn[6] = {jxp, jxm, jyp, jym, jzp, jzm};
        uint32_t Jw[6], nb[6];
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            Jw[d] = (d & 1) ? __ldg(a.J_oth[d >> 1] + jn[d]) : __ldg(a.J_act[d >> 1] + j);
            nb[d] = __ldg(a.S_oth + jn[d]);
        }
        s[w] = a.S_act[j];
        satisfied_bond_count(s[w], Jw, nb, sum2[w], sum1[w], sum0[w]);
        site[w] = (uint64_t)(2u * m + xodd) + (uint64_t)L * ((uint64_t)y + (uint64_t)L * (uint64_t)z);
        if (++m == H) {  // next site of the colour: next row
            m = 0;
            if (++y == L) { y = 0; ++z; }
        }
    }
}

// MULTI: all coded batches in one launch (blockIdx.y = batch, arrays batch_stride words apart, plain Philox rounds keyed per
// sample or, for the shared draw, per batch), as in half_sweep_sample_packed_vec.
template <int RNG, int PARTS, bool MULTI>
__global__ void __launch_bounds__(128)
half_sweep_sample_packed(SweepArgs a, const __grid_constant__ RngLaunch rng, uint32_t n_groups, uint64_t N, size_t batch_stride)
{
    constexpr int SPT = 32 / PARTS;  // samples per thread
    const uint32_t sample0 = MULTI ? 32u * blockIdx.y : rng.sample_base;
    if (MULTI) {
        const size_t off = (size_t)blockIdx.y * batch_stride;
        a.S_act += off;
        a.S_oth += off;
#pragma unroll
        for (int d = 0; d < 3; ++d) { a.J_act[d] += off; a.J_oth[d] += off; }
    }
    const int part = PARTS == 1 ? 0 : (int)(threadIdx.x >> 5);  // warp-uniform
    const uint32_t g_raw = PARTS == 1 ? blockIdx.x * 128u + threadIdx.x : blockIdx.x * 32u + (threadIdx.x & 31u);
    const bool valid = g_raw < n_groups;
    const uint32_t g = valid ? g_raw : n_groups - 1;  // keep the warp converged for the votes below
    uint32_t s[4], sum2[4], sum1[4], sum0[4];
    uint64_t site[4];
    const uint32_t j0 = 4u * g;
    wait_for_previous_kernel();
    group_sums_any_L(a, g, s, sum2, sum1, sum0, site);
    uint32_t c4[4] = {0, 0, 0, 0}, c8[4] = {0, 0, 0, 0}, c12[4] = {0, 0, 0, 0};
    if (RNG == 2) {  // shared draw: Eq. 15 verbatim, the cond words are all ones or zero
        uint32_t R[4];
        if (MULTI) philox4x32_10(rng.tlo, rng.thi, g, 0u, rng.k0, rng.k1base ^ blockIdx.y, R);   // R18: key field = batch
        else philox_folded(rng.pc, rng.ps[0], g, R);
        shared_cond_words(R, a.T, c4, c8, c12);
    }
    // PARTS = 1: a rolled loop over the 16 sample pairs (the unrolled body of 32 calls is 40 KB of code that every warp
    // walks through once, and the instruction cache misses showed up as the top stall); PARTS = 4: 4 pairs, unrolled.
    uint32_t bit_lo = 1u;  // 1 << i
#pragma unroll(PARTS == 1 ? 1 : 4)
    for (int i = 0; i < SPT && RNG != 2; i += 2) {
        const int b = SPT * part + i;
        uint32_t R[8];
        if (RNG == 0 && MULTI) {
            philox4x32_10(rng.tlo, rng.thi, g, 0u, rng.k0, rng.k1base ^ (sample0 + (uint32_t)b), R);
            philox4x32_10(rng.tlo, rng.thi, g, 0u, rng.k0, rng.k1base ^ (sample0 + (uint32_t)b + 1u), R + 4);
        } else if (RNG == 0) {
            philox_folded(rng.pc, rng.ps[b], g, R);
            philox_folded(rng.pc, rng.ps[b + 1], g, R + 4);
        } else {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const uint64_t qs = (uint64_t)(sample0 + b + e) * N;
#pragma unroll
                for (int w = 0; w < 4; ++w)
                    R[4 * e + w] = minstd_mulmod(rng.A, minstd_seed_state_from_weyl(rng.seed + (qs + site[w] + 1) * SPLITMIX_GAMMA));
            }
        }
        const uint32_t bit_hi = bit_lo << 1;
        uint32_t mn = 0xFFFFFFFFu;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            or_if_lt(c4[e & 3], R[e], a.T.t4, e < 4 ? bit_lo : bit_hi);
            mn = min_u32(mn, R[e]);
        }
        if (__any_sync(0xFFFFFFFFu, mn < a.T.t8)) {
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                or_if_lt(c8[e & 3], R[e], a.T.t8, e < 4 ? bit_lo : bit_hi);
                or_if_lt(c12[e & 3], R[e], a.T.t12, e < 4 ? bit_lo : bit_hi);
            }
        }
        bit_lo <<= 2;
    }
    if (!valid) return;
    const int sh = SPT * part;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t f = flip_mask(sum2[w] >> sh, sum1[w] >> sh, sum0[w] >> sh, c4[w] | a.T.always4, c8[w] | a.T.always8,
                                     c12[w] | a.T.always12);
        if (PARTS == 1) a.S_act[j0 + w] = s[w] ^ f;
        else reinterpret_cast<unsigned char *>(a.S_act + j0 + w)[part] = (unsigned char)((s[w] >> sh) ^ f);  // little-endian
    }
}

// Loads and field sums of one group of four consecutive same-colour sites of a row, sample-packed, L % 8 == 0 (so that
// L/2 is a multiple of 4 and a group never leaves its row): own spins and couplings, the y+-1 / z+-1 neighbours and their
// couplings are 128-bit loads; the two x-neighbours are the same four words of the other colour shifted by one word
// (one extra 32-bit load each for spins and couplings).  p = index of the group within the plane z (y = p / gpr).
// COHERENT: spin words through the L2 (persistent kernels, see load_spin_words).
template <bool STREAM = false, bool COHERENT = false>
__device__ __forceinline__ void vec_group_sums(const SweepArgs &a, uint32_t gpr, uint32_t gpr_inv, uint32_t p, uint32_t z,
                                               uint32_t &j0, uint64_t &site0, uint32_t s[4], uint32_t sum2[4], uint32_t sum1[4],
                                               uint32_t sum0[4])
{
    const uint32_t L = (uint32_t)a.L, H = L >> 1;
    const uint32_t y = gpr == 1 ? p : __umulhi(p, gpr_inv);   // exact: p < 2^19, 2 <= gpr <= 2^8
    const uint32_t m0 = 4u * (p - y * gpr);
    const uint32_t rowbase = H * (y + L * z);
    j0 = rowbase + m0;
    const uint32_t HL = H * L, Hc = HL * L;
    const uint32_t jyp = (y + 1 == L) ? j0 - (HL - H) : j0 + H, jym = (y == 0) ? j0 + (HL - H) : j0 - H;
    const uint32_t jzp = (z + 1 == L) ? j0 - (Hc - HL) : j0 + HL, jzm = (z == 0) ? j0 + (Hc - HL) : j0 - HL;
    const uint32_t xodd = (y + z + (uint32_t)a.colour) & 1u;
    site0 = (uint64_t)(2u * m0 + xodd) + (uint64_t)L * ((uint64_t)y + (uint64_t)L * (uint64_t)z);
    // the word next to the four: m0+4 (xodd = 1, +x neighbour of the last site) or m0-1 (xodd = 0, -x of the first)
    const uint32_t m_extra = xodd ? (m0 + 4 == H ? 0u : m0 + 4) : (m0 == 0 ? H - 1 : m0 - 1);

    uint32_t o[4], oyp[4], oym[4], ozp[4], ozm[4], jxa[4], jya[4], jza[4], jxo[4], jyo[4], jzo[4];
    if (!COHERENT) wait_for_previous_kernel();
    if (STREAM) {
        load_words4_streaming(a.S_act, j0, s);
        load_words<4>(a.S_oth, j0, o);
        load_words4_streaming(a.J_oth[0], j0, jxo);
    } else {
        load_spin_words<4, COHERENT>(a.S_act, j0, s);
        load_spin_words<4, COHERENT>(a.S_oth, j0, o);
        load_words<4>(a.J_oth[0], j0, jxo);
    }
    const uint32_t o_extra = COHERENT ? __ldcg(a.S_oth + rowbase + m_extra) : __ldg(a.S_oth + rowbase + m_extra);
    const uint32_t jxo_extra = __ldg(a.J_oth[0] + rowbase + m_extra);
    load_spin_words<4, COHERENT>(a.S_oth, jyp, oyp);
    load_spin_words<4, COHERENT>(a.S_oth, jym, oym);
    load_spin_words<4, COHERENT>(a.S_oth, jzp, ozp);
    load_spin_words<4, COHERENT>(a.S_oth, jzm, ozm);
    if (STREAM) {
        load_words4_streaming(a.J_act[0], j0, jxa);
        load_words4_streaming(a.J_act[1], j0, jya);
        load_words4_streaming(a.J_act[2], j0, jza);
        load_words4_streaming(a.J_oth[1], jym, jyo);
        load_words4_streaming(a.J_oth[2], jzm, jzo);
    } else {
        load_words<4>(a.J_act[0], j0, jxa);
        load_words<4>(a.J_act[1], j0, jya);
        load_words<4>(a.J_act[2], j0, jza);
        load_words<4>(a.J_oth[1], jym, jyo);
        load_words<4>(a.J_oth[2], jzm, jzo);
    }
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        // xodd = 0: +x is word m (own coupling), -x is word m-1 with that neighbour's coupling;
        // xodd = 1: -x is word m with its coupling, +x is word m+1 (own coupling)
        const uint32_t o_up = (w < 3) ? o[(w + 1) & 3] : o_extra;                    // word m+1 (xodd = 1)
        const uint32_t o_dn = (w > 0) ? o[(w + 3) & 3] : o_extra;                    // word m-1 (xodd = 0)
        const uint32_t jx_dn = (w > 0) ? jxo[(w + 3) & 3] : jxo_extra;
        const uint32_t J[6] = {jxa[w], xodd ? jxo[w] : jx_dn, jya[w], jyo[w], jza[w], jzo[w]};
        const uint32_t nb[6] = {xodd ? o_up : o[w], xodd ? o[w] : o_dn, oyp[w], oym[w], ozp[w], ozm[w]};
        satisfied_bond_count(s[w], J, nb, sum2[w], sum1[w], sum0[w]);
    }
}

// ---------------------------------------------------------------------------------------------------
// Shared-random-number mode (rng_mode 2, R18), sample-packed, L % 8 == 0: the paper's own asynchronous multispin
// coding.  One Philox call per group of 4 consecutive sites serves 4 x 32 flip attempts, so the
// kernel is bound by HBM (1.125 B per flip attempt), not by the generator.  With L/2 a multiple of 4 a group never
// leaves its row: own spins and couplings, the y+-1 / z+-1 neighbours and their couplings are 128-bit loads, the two
// x-neighbours are the same four words of the other colour shifted by one word (one extra 32-bit load).
// grid = (ceil(L * L/8 / 128), L, batches): blockIdx.y = z, the x index runs over (y, group in row), blockIdx.z is the
// coded batch (k batches of 32 samples in one launch); the arrays of batch b start b * batch_stride
// words after those of batch 0, and its draws use the key (k0, k1base ^ b) (R18).  With several batches per launch the
// launch constants cannot be folded per batch, so the plain ten rounds are run (the kernel is HBM-bound either way).
// ---------------------------------------------------------------------------------------------------
struct SharedRng {
    uint32_t tlo, thi, k0, k1base;
};

// FLAT (L < 32, where a plane has fewer than 128 groups): grid = ceil(batches * L * L * L/8 / 128), the thread index runs
// over the units u = b * ngroups + g of all batches, so that small lattices with many coded batches (PAPER.md:151-153,
// 308-310) keep every thread busy (L = 8 x 4096 batches: 0.58 -> 0.17 ps/flip).
template <bool FLAT>
__global__ void __launch_bounds__(128)
half_sweep_shared_vec(SweepArgs a, const SharedRng rng, uint32_t gpr /* groups per row = L/8 */,
                      uint32_t gpr_inv /* ceil(2^32 / gpr) */, size_t batch_stride, uint32_t nbatches,
                      uint32_t batch0 /* first batch of this launch (launches are chunked to 65535 batches) */)
{
    const uint32_t L = (uint32_t)a.L;
    uint32_t p = blockIdx.x * 128u + threadIdx.x, z = blockIdx.y, batch = batch0 + blockIdx.z;
    if (FLAT) {
        const uint32_t per_plane = L * gpr, ngroups = per_plane * L;
        if (p >= nbatches * ngroups) return;
        batch = p / ngroups;
        const uint32_t g = p - batch * ngroups;
        z = g / per_plane;
        p = g - z * per_plane;
    } else if (p >= L * gpr) {
        return;
    }
    {
        const size_t off = (size_t)batch * batch_stride;
        a.S_act += off;
        a.S_oth += off;
#pragma unroll
        for (int d = 0; d < 3; ++d) { a.J_act[d] += off; a.J_oth[d] += off; }
    }
    uint32_t j0, s[4], sum2[4], sum1[4], sum0[4];
    uint64_t site0;
    vec_group_sums(a, gpr, gpr_inv, p, z, j0, site0, s, sum2, sum1, sum0);

    uint32_t R[4], c4[4], c8[4], c12[4];
    philox4x32_10(rng.tlo, rng.thi, j0 >> 2, 0u, rng.k0, rng.k1base ^ batch, R);
    shared_cond_words(R, a.T, c4, c8, c12);

    uint32_t out[4];
#pragma unroll
    for (int w = 0; w < 4; ++w)
        out[w] = s[w] ^ flip_mask(sum2[w], sum1[w], sum0[w], c4[w] | a.T.always4, c8[w] | a.T.always8, c12[w] | a.T.always12);
    *reinterpret_cast<uint4 *>(a.S_act + j0) = *reinterpret_cast<const uint4 *>(out);
}

// ---------------------------------------------------------------------------------------------------
// Independent draws (Philox or MINSTD per sample), sample-packed, L % 8 == 0: the loads and field sums of
// half_sweep_shared_vec, then one Philox call per sample as in half_sweep_sample_packed (same PARTS scheme: PARTS = 4
// spreads the 32 samples of a group over the four warps of the CTA, each updating one byte of the four words).
// grid = (ceil(L * L/8 / (128 / PARTS)), L), one launch per batch of 32 samples.
// ---------------------------------------------------------------------------------------------------
// MULTI: all coded batches in one launch (blockIdx.z = batch, arrays batch_stride words apart).  The launch constants
// cannot be folded per (batch, sample) then, so the plain ten Philox rounds are run with the key (k0, k1base ^ sample);
// a small lattice with many batches is one launch instead of one per batch.
// The body of half_sweep_sample_packed_vec (one launch per half-sweep) and of half_sweep_sample_packed_vec_graph (graph_kernels.cuh);
// RL = RngLaunch, or any struct with the fields the chosen variant reads (MULTI: tlo, thi, k0, k1base, seed, A only).
template <int RNG, int PARTS, bool MULTI, typename RL>
__device__ __forceinline__ void sample_packed_vec_body(SweepArgs a, const RL &rng, uint32_t gpr, uint32_t gpr_inv, uint64_t N, size_t batch_stride)
{
    constexpr int SPT = 32 / PARTS;
    const uint32_t L = (uint32_t)a.L;
    const uint32_t sample0 = MULTI ? 32u * blockIdx.z : rng.sample_base;
    if (MULTI) {
        const size_t off = (size_t)blockIdx.z * batch_stride;
        a.S_act += off;
        a.S_oth += off;
#pragma unroll
        for (int d = 0; d < 3; ++d) { a.J_act[d] += off; a.J_oth[d] += off; }
    }
    const int part = PARTS == 1 ? 0 : (int)(threadIdx.x >> 5);  // warp-uniform
    const uint32_t p_raw = PARTS == 1 ? blockIdx.x * 128u + threadIdx.x : blockIdx.x * 32u + (threadIdx.x & 31u);
    const bool valid = p_raw < L * gpr;
    const uint32_t p = valid ? p_raw : L * gpr - 1;  // keep the warp converged for the votes below
    uint32_t j0, s[4], sum2[4], sum1[4], sum0[4];
    uint64_t site0;
    vec_group_sums(a, gpr, gpr_inv, p, blockIdx.y, j0, site0, s, sum2, sum1, sum0);
    const uint32_t g = j0 >> 2;

    uint32_t c4[4] = {0, 0, 0, 0}, c8[4] = {0, 0, 0, 0}, c12[4] = {0, 0, 0, 0};
    uint32_t bit_lo = 1u;  // 1 << i
#pragma unroll(PARTS == 1 ? 1 : 4)
    for (int i = 0; i < SPT; i += 2) {
        const int b = SPT * part + i;
        uint32_t R[8];
        if constexpr (RNG == 0 && MULTI) {
            philox4x32_10(rng.tlo, rng.thi, g, 0u, rng.k0, rng.k1base ^ (sample0 + (uint32_t)b), R);
            philox4x32_10(rng.tlo, rng.thi, g, 0u, rng.k0, rng.k1base ^ (sample0 + (uint32_t)b + 1u), R + 4);
        } else if constexpr (RNG == 0) {
            philox_folded(rng.pc, rng.ps[b], g, R);
            philox_folded(rng.pc, rng.ps[b + 1], g, R + 4);
        } else {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const uint64_t w0 = rng.seed + ((uint64_t)(sample0 + b + e) * N + site0 + 1) * SPLITMIX_GAMMA;
#pragma unroll
                for (int w = 0; w < 4; ++w)  // consecutive sites of the colour are 2 apart in the canonical index
                    R[4 * e + w] = minstd_mulmod(rng.A, minstd_seed_state_from_weyl(w0 + (uint64_t)w * (2 * SPLITMIX_GAMMA)));
            }
        }
        const uint32_t bit_hi = bit_lo << 1;
        uint32_t mn = 0xFFFFFFFFu;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            or_if_lt(c4[e & 3], R[e], a.T.t4, e < 4 ? bit_lo : bit_hi);
            mn = min_u32(mn, R[e]);
        }
        if (__any_sync(0xFFFFFFFFu, mn < a.T.t8)) {
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                or_if_lt(c8[e & 3], R[e], a.T.t8, e < 4 ? bit_lo : bit_hi);
                or_if_lt(c12[e & 3], R[e], a.T.t12, e < 4 ? bit_lo : bit_hi);
            }
        }
        bit_lo <<= 2;
    }
    if (!valid) return;
    const int sh = SPT * part;
    uint32_t out[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t f = flip_mask(sum2[w] >> sh, sum1[w] >> sh, sum0[w] >> sh, c4[w] | a.T.always4, c8[w] | a.T.always8,
                                     c12[w] | a.T.always12);
        out[w] = (s[w] >> sh) ^ f;
    }
    if (PARTS == 1) {
        *reinterpret_cast<uint4 *>(a.S_act + j0) = *reinterpret_cast<const uint4 *>(out);
    } else {
#pragma unroll
        for (int w = 0; w < 4; ++w) reinterpret_cast<unsigned char *>(a.S_act + j0 + w)[part] = (unsigned char)out[w];  // little-endian
    }
}

template <int RNG, int PARTS, bool MULTI>
__global__ void __launch_bounds__(128)
half_sweep_sample_packed_vec(SweepArgs a, const __grid_constant__ RngLaunch rng, uint32_t gpr, uint32_t gpr_inv, uint64_t N,
                             size_t batch_stride)
{
    sample_packed_vec_body<RNG, PARTS, MULTI>(a, rng, gpr, gpr_inv, N, batch_stride);
}

}  // namespace isingk
