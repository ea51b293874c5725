// lane_rng.cuh -- generators with STORED state, one per "lane" (the paper's one generator per thread),
// SURVEY.md 8(f) rank 2, R19 / section 11:
//   Parisi-Rapuano:  ira[i] = ira[i-24] + ira[i-55];  R = ira[i] ^ ira[i-61];   62-word ring
//   MT19937, incremental form: y = (mt[i] & UPPER) | (mt[i+1] & LOWER); mt[i] = mt[i+397] ^ (y >> 1) ^ (y odd ?
//   MATRIX : 0); R = temper(mt[i]);  624-word ring, seeded by init_genrand.
// State layout = the paper's strided scheme: word r of lane q is at state[r * nlanes + q], so the 32
// lanes of a warp read 128 contiguous bytes per ring position and "only O(1) memory transactions" are needed per draw
// (PAPER.md:370).  Every lane is at the same ring position, which the host passes in (pos0 = draws so far mod ring).
// Draws are produced four at a time: within four consecutive draws no read position equals an earlier write position
// (the shortest lag is 24, resp. 1 for MT where the word read ahead is the OLD one), so all loads are issued first.
//
// Kernels: lanes_init<GEN>, half_sweep_shared_lanes<GEN> (rng_mode 3, 4: the shared-draw sweep of sweep_kernels.cuh with
// these generators), count_odd_lanes<GEN>, count_odd_minstd, count_odd_philox (Table II).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sweep_kernels.cuh"

namespace isingk {

constexpr int GEN_PR = 0, GEN_MT = 1;
template <int GEN> struct LaneRing { static constexpr uint32_t size = GEN == GEN_PR ? 62u : 624u; };

struct LaneArgs {
    uint32_t *state;   // ring * nlanes words, strided
    uint32_t nlanes;
    uint32_t pos0;     // ring position of the first draw of this launch
};

template <uint32_t RING>
__device__ __forceinline__ uint32_t ring_add(uint32_t pos, uint32_t c)
{  // (pos + c) mod RING for pos, c < RING
    const uint32_t p = pos + c;
    return p >= RING ? p - RING : p;
}

__device__ __forceinline__ uint32_t mt_temper(uint32_t y)
{
    y ^= y >> 11;
    y ^= (y << 7) & 0x9d2c5680u;
    y ^= (y << 15) & 0xefc60000u;
    y ^= y >> 18;
    return y;
}

// Four consecutive draws of the lane whose words are st[r * stride], in two steps so that a kernel can put other loads
// between them: lane_load4 issues every state load of the four draws and advances pos by 4, lane_finish4 computes the
// draws and stores the four new state words.
template <int GEN> struct LaneOperands {
    uint32_t v[GEN == GEN_PR ? 12 : 9];
    uint32_t p[4];   // ring positions of the four draws (the words they overwrite)
};

template <int GEN>
__device__ __forceinline__ void lane_load4(const uint32_t *st, size_t stride, uint32_t &pos, LaneOperands<GEN> &o)
{
    constexpr uint32_t RING = LaneRing<GEN>::size;
    uint32_t p[5];
#pragma unroll
    for (int d = 0; d < 5; ++d) p[d] = ring_add<RING>(pos, (uint32_t)d);
#pragma unroll
    for (int d = 0; d < 4; ++d) o.p[d] = p[d];
    if (GEN == GEN_PR) {
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            o.v[d] = st[(size_t)ring_add<RING>(p[d], RING - 24) * stride];
            o.v[4 + d] = st[(size_t)ring_add<RING>(p[d], RING - 55) * stride];
            o.v[8 + d] = st[(size_t)p[d + 1] * stride];   // i - 61 = i + 1 (mod 62)
        }
    } else {
#pragma unroll
        for (int d = 0; d < 5; ++d) o.v[d] = st[(size_t)p[d] * stride];
#pragma unroll
        for (int d = 0; d < 4; ++d) o.v[5 + d] = st[(size_t)ring_add<RING>(p[d], 397) * stride];
    }
    pos = p[4];
}

template <int GEN>
__device__ __forceinline__ void lane_finish4(uint32_t *st, size_t stride, const LaneOperands<GEN> &o, uint32_t R[4])
{
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        if (GEN == GEN_PR) {
            const uint32_t v = o.v[d] + o.v[4 + d];
            st[(size_t)o.p[d] * stride] = v;
            R[d] = v ^ o.v[8 + d];
        } else {
            const uint32_t y = (o.v[d] & 0x80000000u) | (o.v[d + 1] & 0x7fffffffu);
            const uint32_t v = o.v[5 + d] ^ (y >> 1) ^ ((y & 1u) ? 0x9908b0dfu : 0u);
            st[(size_t)o.p[d] * stride] = v;
            R[d] = mt_temper(v);
        }
    }
}

template <int GEN>
__device__ __forceinline__ void lane_next4(uint32_t *st, size_t stride, uint32_t &pos, uint32_t R[4])
{
    LaneOperands<GEN> o;
    lane_load4<GEN>(st, stride, pos, o);
    lane_finish4<GEN>(st, stride, o, R);
}

__device__ __forceinline__ uint64_t splitmix64_output_dev(uint64_t seed, uint64_t n)
{
    uint64_t z = seed + n * SPLITMIX_GAMMA;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// Seeding (R19).  PR: ring word r of lane q = high word of SplitMix64 output q*62 + r + 1.  MT: init_genrand of the high
// word of SplitMix64 output q + 1.
template <int GEN>
__global__ void __launch_bounds__(128) lanes_init(uint32_t *state, uint32_t nlanes, uint64_t seed)
{
    const uint32_t q = blockIdx.x * 128u + threadIdx.x;
    if (q >= nlanes) return;
    uint32_t *st = state + q;
    if (GEN == GEN_PR) {
        for (uint32_t r = 0; r < 62u; ++r)
            st[(size_t)r * nlanes] = (uint32_t)(splitmix64_output_dev(seed, (uint64_t)q * 62u + r + 1) >> 32);
    } else {
        uint32_t v = (uint32_t)(splitmix64_output_dev(seed, (uint64_t)q + 1) >> 32);
        st[0] = v;
        for (uint32_t i = 1; i < 624u; ++i) {
            v = 1812433253u * (v ^ (v >> 30)) + i;
            st[(size_t)i * nlanes] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Shared-draw half-sweep driven by lane generators (rng_mode 3, 4), sample-packed.  Thread = lane q.  It
// serves the units u = q + m * nlanes, m = 0 .. rounds-1, where unit u = b * ngroups + g is group g (four consecutive
// same-colour sites of a row, the unit of half_sweep_shared_vec) of coded batch b, and takes four draws per unit (R19); a
// lane whose last unit does not exist still draws.  Consecutive lanes hold consecutive groups of one batch, so the
// lattice loads of a warp are the same coalesced 512-byte rows as in half_sweep_shared_vec; small lattices with many
// batches fill the machine because the units, not the groups, are dealt to the lanes.
// (Holding the twelve state operands in registers across the lattice loads, so that both round trips overlap, spills at 64
// registers and was slower: 0.249 against 0.239 ps/flip.)
// ---------------------------------------------------------------------------------------------------
// VEC = false (L % 8 != 0): a group may straddle rows, its sums come from group_sums_any_L (one load per word).
// STREAM (host: lattices larger than the L2): the couplings and the active spins, read once per half-sweep, are loaded
// evict-first so that they do not push the generator state and the other colour's spins out of the L2 -- Parisi-Rapuano
// at L = 512 x 32 samples: 0.231 -> 0.212 ps/flip; on lattices that fit the L2 the same hint costs 10-20 % (their couplings
// would have stayed resident), hence the switch.
template <int GEN, bool VEC, bool STREAM>
__global__ void __launch_bounds__(128, 8)
half_sweep_shared_lanes(const SweepArgs a0, const LaneArgs ln, uint32_t gpr, uint32_t gpr_inv, size_t batch_stride,
                        uint32_t ngroups, uint64_t units, uint32_t rounds)
{
    const uint32_t q = blockIdx.x * 128u + threadIdx.x;
    if (q >= ln.nlanes) return;
    uint32_t *st = ln.state + q;
    const size_t stride = ln.nlanes;
    uint32_t pos = ln.pos0;
    const uint32_t per_plane = (uint32_t)a0.L * gpr;
    wait_for_previous_kernel();   // the state was written by the previous half-sweep
    for (uint32_t m = 0; m < rounds; ++m) {
        const uint64_t u = (uint64_t)q + (uint64_t)m * ln.nlanes;
        uint32_t R[4];
        lane_next4<GEN>(st, stride, pos, R);
        if (u >= units) continue;
        const uint32_t b = (uint32_t)(u / ngroups), g = (uint32_t)(u - (uint64_t)b * ngroups);
        SweepArgs a = a0;
        const size_t off = (size_t)b * batch_stride;
        a.S_act += off;
        a.S_oth += off;
#pragma unroll
        for (int d = 0; d < 3; ++d) { a.J_act[d] += off; a.J_oth[d] += off; }
        uint32_t j0, s[4], sum2[4], sum1[4], sum0[4], c4[4], c8[4], c12[4];
        if (VEC) {
            const uint32_t z = g / per_plane, p = g - z * per_plane;
            uint64_t site0;
            vec_group_sums<STREAM>(a, gpr, gpr_inv, p, z, j0, site0, s, sum2, sum1, sum0);
        } else {
            uint64_t site[4];
            j0 = 4u * g;
            group_sums_any_L(a, g, s, sum2, sum1, sum0, site);
        }
        shared_cond_words(R, a.T, c4, c8, c12);
        uint32_t out[4];
#pragma unroll
        for (int w = 0; w < 4; ++w)
            out[w] = s[w] ^ flip_mask(sum2[w], sum1[w], sum0[w], c4[w] | a.T.always4, c8[w] | a.T.always8, c12[w] | a.T.always12);
        *reinterpret_cast<uint4 *>(a.S_act + j0) = *reinterpret_cast<const uint4 *>(out);
    }
}

// ---------------------------------------------------------------------------------------------------
// PAPER.md:196-197, Table II: "its kernel version counting the fraction of odd numbers".  Every lane draws ndraws numbers
// (a multiple of 4) continuing from ring position pos0; odd[q] = how many were odd, sum[q] = their sum mod 2^64.
// ---------------------------------------------------------------------------------------------------
// STAGE (Parisi-Rapuano only): the 62-word rings of the CTA's 128 lanes are copied to shared memory (31 KB, word r of thread i
// at ring[r * 128 + i]: conflict-free) for the duration of the launch and written back at the end: 852 -> 1313 G numbers/s.
// (The same staging in the half-sweep kernel was slower than global-memory rings at every lane count -- 0.283 against 0.239
// ps/flip at best: 7 x 31 KB of shared memory leave almost no L1 for the lattice loads -- and is not used there.)
template <int GEN, bool STAGE>
__global__ void __launch_bounds__(128)
count_odd_lanes(const LaneArgs ln, uint64_t ndraws, unsigned long long *odd, unsigned long long *sum)
{
    static_assert(!STAGE || GEN == GEN_PR, "only the 62-word ring fits shared memory");
    __shared__ uint32_t ring[STAGE ? 62 * 128 : 1];
    const uint32_t q = blockIdx.x * 128u + threadIdx.x;
    if (q >= ln.nlanes) return;
    uint32_t *gst = ln.state + q;
    uint32_t *st = STAGE ? ring + threadIdx.x : gst;
    const size_t stride = STAGE ? 128u : ln.nlanes;
    if (STAGE)
        for (uint32_t r = 0; r < 62u; ++r) st[r * 128u] = gst[(size_t)r * ln.nlanes];
    uint32_t pos = ln.pos0;
    unsigned long long o = 0, s = 0;
    for (uint64_t n = 0; n < ndraws; n += 4) {
        uint32_t R[4];
        lane_next4<GEN>(st, stride, pos, R);
        o += (R[0] & 1u) + (R[1] & 1u) + (R[2] & 1u) + (R[3] & 1u);
        s += (unsigned long long)R[0] + R[1] + R[2] + R[3];
    }
    if (STAGE)
        for (uint32_t r = 0; r < 62u; ++r) gst[(size_t)r * ln.nlanes] = st[r * 128u];
    odd[q] = o;
    sum[q] = s;
}

// MINSTD (Eq. 7): one state word per lane, state[q]; init = seed state of stream q (R11).
__global__ void __launch_bounds__(128) minstd_lanes_init(uint32_t *state, uint32_t nlanes, uint64_t seed)
{
    const uint32_t q = blockIdx.x * 128u + threadIdx.x;
    if (q < nlanes) state[q] = minstd_seed_state_from_weyl(seed + ((uint64_t)q + 1) * SPLITMIX_GAMMA);
}

__global__ void __launch_bounds__(128)
count_odd_minstd(uint32_t *state, uint32_t nlanes, uint64_t ndraws, unsigned long long *odd, unsigned long long *sum)
{
    const uint32_t q = blockIdx.x * 128u + threadIdx.x;
    if (q >= nlanes) return;
    uint32_t r = state[q];
    unsigned long long o = 0, s = 0;
    for (uint64_t n = 0; n < ndraws; ++n) {
        r = minstd_mulmod(16807u, r);
        o += r & 1u;
        s += r;
    }
    state[q] = r;
    odd[q] = o;
    sum[q] = s;
}

// Philox4x32-10, no state: key (lo32 seed, hi32 seed), counter (lo32 c, hi32 c, q, 0), c = call number = draw number >> 2.
__global__ void __launch_bounds__(128)
count_odd_philox(uint32_t nlanes, uint64_t seed, uint64_t first_call, uint64_t ncalls, unsigned long long *odd, unsigned long long *sum)
{
    const uint32_t q = blockIdx.x * 128u + threadIdx.x;
    if (q >= nlanes) return;
    unsigned long long o = 0, s = 0;
    for (uint64_t c = first_call; c < first_call + ncalls; ++c) {
        uint32_t R[4];
        philox4x32_10((uint32_t)c, (uint32_t)(c >> 32), q, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), R);
        o += (R[0] & 1u) + (R[1] & 1u) + (R[2] & 1u) + (R[3] & 1u);
        s += (unsigned long long)R[0] + R[1] + R[2] + R[3];
    }
    odd[q] = o;
    sum[q] = s;
}

}  // namespace isingk
