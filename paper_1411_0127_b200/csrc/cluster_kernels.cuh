// cluster_kernels.cuh -- whole trajectories of small lattices out of distributed shared memory: one thread-block cluster per
// sample, all half-sweeps of a call in one launch (many small systems to fill the GPU; SURVEY.md section 3:
// "a persistent kernel is used for small L").
//
// A lattice with whole-word rows whose eight bit arrays fit the shared memory of a cluster (L = 64: 128 KiB, L = 128: 1 MiB) never
// has to leave the SMs between half-sweeps.  The cluster of C CTAs cuts it along z: CTA r holds the planes r L/C .. (r + 1) L/C - 1
// of all eight arrays and updates them; the planes below and above its own live in the neighbouring CTAs' shared memory and are read
// there directly (distributed shared memory, ld through mapa-translated addresses) -- the paper's slab decomposition of section V
// with the SMs of one cluster in the place of the GPUs, and without the exchange step, since a remote plane can be
// read in place.  Between two half-sweeps there is ONE cluster barrier (all stores of the active colour before any load of the next
// half-sweep, which also orders the remote reads of the colour that is overwritten next), and it is split: a thread arrives when its
// store is done, then draws the random numbers of its first word of the NEXT half-sweep -- the acceptance masks depend on
// (site, t) only, not on the spins, and are three quarters of the work -- and only then waits.  The barrier's latency (0.23 us,
// profiles/r2j_launch_floor.md) and the skew between the CTAs disappear behind the generator; nothing crosses the L2 and no launch
// happens until the call's last half-sweep.  Samples are independent (batch_kernels.cuh), so a grid is one cluster per sample and
// clusters never talk to each other; C is chosen so that samples x C fills the 148 SMs (32 samples: C = 4; one sample: C = 16,
// the non-portable maximum).
//   Records (ising_sweep_trace): a recording half-sweep runs a second copy of the update that counts, as the measuring tile update
// does, the satisfied bonds from the field sums it holds and the up spins of both colours, and adds the CTA's totals to the
// pre-set record (R16, as add_to_record does) behind the arrive; the other half-sweeps run the plain copy.
//   The bits are those of one launch per half-sweep: the draws are keyed by (sample, site, t), not by the thread mapping (R9, R11).
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "sweep_kernels.cuh"

namespace isingk {

namespace cg = cooperative_groups;

constexpr int CLUSTER_MAX_THREADS = 1024;
constexpr int CLUSTER_SEED_CACHE_MAX_NW = 512;   // MINSTD: cached seed states need 256 bytes of shared memory per thread

struct ClusterArgs {
    LatticeArrays A;         // the arrays of sample 0
    size_t lattice_stride;   // words between the arrays of consecutive samples
    int L;
    Thresholds T;
    uint64_t seed, t0, N;
    uint32_t nhalf, every;   // half-sweeps of this launch; record after every `every`-th (0: never)
    uint32_t A_first;        // MINSTD: 16807^(n+1) mod M of the sweep n = t0 >> 1
    uint32_t nsamples, sample0;
    long long *E, *M;        // record r of sample s at E[r * nsamples + s] (pre-set by init_records); either may be null
};

__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// Addresses in the shared::cluster window (32 bits): a CTA's own shared memory and its neighbours' are read the same way.
__device__ __forceinline__ uint32_t cluster_address(const void *smem_ptr, uint32_t rank)
{
    uint32_t a;
    asm("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(a) : "r"((uint32_t)__cvta_generic_to_shared(smem_ptr)), "r"(rank));
    return a;
}
__device__ __forceinline__ uint32_t cluster_load(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
template <int BYTE_OFFSET>   // the same with a compile-time offset in the instruction
__device__ __forceinline__ uint32_t cluster_load_at(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1+%2];" : "=r"(v) : "r"(addr), "n"(BYTE_OFFSET) : "memory");
    return v;
}

struct false_type_tag { static constexpr bool value = false; };
struct true_type_tag { static constexpr bool value = true; };

// What the update of one word needs to know about its place and does not change from one half-sweep to the next.
struct WordPlace {
    uint32_t wl;                 // index of the word in the CTA's slab of each array
    uint32_t w_yp, w_ym;         // the same bit one row up / down (periodic within the plane)
    uint32_t zp_addr, zm_addr;   // shared::cluster address of the word one plane up / down IN ARRAY 0 (this slab's or a neighbour's)
    uint32_t w_next, w_prev;     // next / previous word of the row (periodic); WPR > 1 only
    uint32_t xodd0;              // (y + z) & 1: a site of colour c with bit m has x = 2m + (xodd0 ^ c)
    uint32_t wg;                 // index of the word in the lattice's colour array (Philox counter, R9)
    uint64_t site_even;          // canonical site of bit 0 if xodd were 0 (MINSTD stream ids, R11)
};

template <int WPR>
__device__ __forceinline__ WordPlace place_word(uint32_t wl, uint32_t L, uint32_t Lz, uint32_t z0, uint32_t a_self, uint32_t a_up, uint32_t a_dn)
{
    const uint32_t plane = L * WPR;
    const uint32_t k = WPR == 1 ? 0u : wl % WPR, row = wl / WPR, y = row % L, zl = row / L;
    WordPlace w;
    w.wl = wl;
    w.w_yp = y + 1 == L ? wl - (plane - WPR) : wl + WPR;
    w.w_ym = y == 0 ? wl + plane - WPR : wl - WPR;
    // z neighbours: in this slab, or the first / last plane of the slab above / below
    const bool top = zl + 1 == Lz, bot = zl == 0;
    w.zp_addr = (top ? a_up : a_self) + 4u * (top ? wl - (Lz - 1) * plane : wl + plane);
    w.zm_addr = (bot ? a_dn : a_self) + 4u * (bot ? wl + (Lz - 1) * plane : wl - plane);
    w.w_next = k + 1 == WPR ? wl - (WPR - 1) : wl + 1;
    w.w_prev = k == 0 ? wl + (WPR - 1) : wl - 1;
    w.xodd0 = (y + z0 + zl) & 1u;
    w.wg = z0 * plane + wl;
    w.site_even = (uint64_t)L * ((uint64_t)y + (uint64_t)L * (z0 + zl)) + 64ull * k;
    return w;
}

// RNG 0 = Philox, 1 = MINSTD (stateless, R11 / R12).  WPR = words per half-row = L / 64.  Cluster of C = gridDim.x / samples CTAs
// (cluster dimension attribute of the launch); blockDim.x = min(1024, words per colour and CTA), a thread owns the words
// tid, tid + blockDim.x, ... of its CTA's slab.  NW > 0: exactly one word per thread and NW = blockDim.x = words per colour and CTA
// known at compile time (L = 64 in clusters of 16, 8, 4 CTAs: 256, 512, 1024): the thread's place is computed once, before the
// first half-sweep, and the twelve operand loads of a half-sweep are four base addresses plus offsets in the instructions (a
// twelfth of the update's instructions were address arithmetic otherwise).  NW = 0: any slab size, several words per thread.
// Dynamic shared memory: 8 arrays of L^2 WPR (L / C) words in the order S[0], S[1], Jx[0], Jx[1], Jy[0], Jy[1], Jz[0], Jz[1].
template <int RNG, int WPR, bool RECORDS, int NW>
__global__ void __launch_bounds__(NW > 0 ? NW : CLUSTER_MAX_THREADS, 1)
half_sweeps_cluster(const __grid_constant__ ClusterArgs p)
{
    extern __shared__ uint32_t sm[];
    constexpr bool SINGLE = NW > 0;
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t C = cluster.num_blocks(), r = cluster.block_rank();
    const uint32_t sample = p.sample0 + blockIdx.x / C;
    const uint32_t L = (uint32_t)p.L, Lz = L / C;
    const uint32_t plane = L * WPR;              // words of one plane of one array
    const uint32_t nw = SINGLE ? (uint32_t)NW : plane * Lz;   // words of one array in this CTA
    const uint32_t z0 = r * Lz;

    // ---- load the slab -------------------------------------------------------------------------------------------------
    {
        const size_t goff = (size_t)sample * p.lattice_stride + (size_t)z0 * plane;
        for (uint32_t i = threadIdx.x; i < nw; i += blockDim.x) {
            sm[i] = p.A.S[0][goff + i];
            sm[nw + i] = p.A.S[1][goff + i];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                sm[(2 + 2 * d) * nw + i] = p.A.J[d][0][goff + i];
                sm[(3 + 2 * d) * nw + i] = p.A.J[d][1][goff + i];
            }
        }
    }
    // this slab and the slabs above and below (periodic) in the shared::cluster window: the same offsets in every CTA
    const uint32_t a_self = cluster_address(sm, r);
    const uint32_t a_up = cluster_address(sm, r + 1 == C ? 0 : r + 1), a_dn = cluster_address(sm, r == 0 ? C - 1 : r - 1);

    const uint64_t seed = RNG == 0 ? p.seed : p.seed + (uint64_t)sample * p.N * SPLITMIX_GAMMA;   // R11: streams s N .. s N + N - 1
    uint32_t A = p.A_first, rec = 0;
    PhiloxCommonConst pc;
    PhiloxSampleConst ps;
    // MINSTD with one word per thread and at most 512 threads: the thread's 2 x 32 seed states s0 (R11: they depend on the site only)
    // are computed once per launch and kept in shared memory behind the arrays, [colour][bit][thread]; a draw is then one
    // multiplication mod 2^31 - 1 (R12) instead of a SplitMix64 evaluation and that multiplication.
    constexpr bool SEED_CACHE = RNG == 1 && NW > 0 && NW <= CLUSTER_SEED_CACHE_MAX_NW;
    uint32_t *const seeds = sm + 8 * nw;
    // the masks of word `w` for colour c with the constants of the current half-sweep
    auto masks = [&](const WordPlace &w, int c, uint32_t &c4, uint32_t &c8, uint32_t &c12) {
        if (RNG == 0) {
            cond_masks_site_packed_philox(pc, ps, w.wg, p.T, c4, c8, c12);
        } else if (SEED_CACHE) {
            c4 = 0; c8 = 0; c12 = 0;
            const uint32_t *sc = seeds + (uint32_t)c * 32u * (uint32_t)NW + threadIdx.x;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                uint32_t R[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) R[i] = minstd_mulmod2(2u * A, sc[(4 * q + i) * NW]);
                accumulate_cond<4>(R, 4 * q, p.T, c4, c8, c12);
            }
            finish_cond(p.T, c4, c8, c12);
        } else {
            cond_masks_site_packed_minstd(seed + (w.site_even + (w.xodd0 ^ (uint32_t)c) + 1) * SPLITMIX_GAMMA, 2 * SPLITMIX_GAMMA, 2u * A, p.T, c4, c8, c12);
        }
    };

    // first word of the thread, half-sweep 0: masks before the barrier that ends the load
    const WordPlace first = place_word<WPR>(threadIdx.x, L, Lz, z0, a_self, a_up, a_dn);
    if (SEED_CACHE) {
#pragma unroll 1
        for (uint32_t c = 0; c < 2; ++c) {
            const uint64_t weyl0 = seed + (first.site_even + (first.xodd0 ^ c) + 1) * SPLITMIX_GAMMA;
#pragma unroll 4
            for (uint32_t b = 0; b < 32; ++b)
                seeds[(c * 32u + b) * (uint32_t)NW + threadIdx.x] = minstd_seed_state_from_weyl(weyl0 + (uint64_t)b * (2 * SPLITMIX_GAMMA));
        }
    }
    uint32_t c4 = 0, c8 = 0, c12 = 0;
    if (RNG == 0) fold_philox_keys(p.seed, sample, &pc, &ps);
    if (p.nhalf) {
        if (RNG == 0) fold_philox_time(p.seed, sample, p.t0, &pc, &ps);
        masks(first, (int)(p.t0 & 1), c4, c8, c12);
    }
    cluster_arrive();
    cluster_wait();

    // One half-sweep kk of the launch.  MEAS (the last half-sweep of a run that ends at a record): the thread also counts, as the
    // measuring tile update of sweep_kernels.cuh does, the satisfied bonds of the configuration it leaves -- every bond has exactly
    // one end in the active colour, so they are the sum over the active sites of the count n in the three bit planes, with
    // n -> 6 - n where the site flipped -- and the up spins of its word of either colour; after the arrive the CTA's totals go to
    // the record (R16, pre-set by init_records) by one atomic pair, which completes under the draws of the next half-sweep.  The
    // plain copy of the body is the same code as in the kernel without records.
    __shared__ unsigned long long rec_sum[2];
    auto half_sweep = [&](uint32_t kk, auto meas) {
        constexpr bool MEAS = decltype(meas)::value;
        const uint64_t t = p.t0 + kk;
        const int c = (int)(t & 1);
        const uint32_t act = (uint32_t)c * nw, oth = nw - act;   // offsets of the active / other colour within a pair of arrays
        unsigned int m_sat = 0, m_up = 0, m_words = 0;
        for (uint32_t wl = threadIdx.x; wl < nw; wl += blockDim.x) {
            WordPlace w = first;
            if (!SINGLE && wl != threadIdx.x) {   // later words of the thread: place and masks now
                w = place_word<WPR>(wl, L, Lz, z0, a_self, a_up, a_dn);
                masks(w, c, c4, c8, c12);
            }
            const uint32_t xodd = w.xodd0 ^ (uint32_t)c;
            // four bases in this CTA's arrays, two in the window of the cluster; everything else is a fixed distance away
            uint32_t *const pa = sm + act + w.wl;
            const uint32_t *const po = sm + oth + w.wl, *const pyp = sm + oth + w.w_yp, *const pym = sm + oth + w.w_ym;
            const uint32_t zp = w.zp_addr + 4u * oth, zm = w.zm_addr + 4u * oth;
            uint32_t s = pa[0];
            const uint32_t o = po[0];
            const uint32_t jxo = po[2 * nw], jxa = pa[2 * nw];
            const uint32_t oyp = pyp[0], oym = pym[0];
            const uint32_t ozp = cluster_load(zp), ozm = cluster_load(zm);
            const uint32_t jya = pa[4 * nw], jza = pa[6 * nw];
            const uint32_t jyo = pym[4 * nw], jzo = SINGLE ? cluster_load_at<24 * NW>(zm) : cluster_load(zm + 24u * nw);
            // x neighbours (row a3; see site_packed_tile): the bit that crosses the word boundary comes from the row's next /
            // previous word (periodic), which for WPR = 1 is the word itself
            const uint32_t B = jxo ^ o;
            uint32_t o_next = o, B_prev = B;
            if (WPR > 1) {
                const uint32_t *const pp = sm + oth + w.w_prev;
                o_next = sm[oth + w.w_next];
                B_prev = pp[2 * nw] ^ pp[0];
            }
            const uint32_t J[6] = {jxa, 0u, jya, jyo, jza, jzo};
            const uint32_t nb[6] = {__funnelshift_r(o, o_next, xodd), __funnelshift_l(B_prev, B, 1u - xodd), oyp, oym, ozp, ozm};
            uint32_t sum2, sum1, sum0;
            satisfied_bond_count(s, J, nb, sum2, sum1, sum0);
            const uint32_t f = flip_mask(sum2, sum1, sum0, c4, c8, c12);
            s ^= f;
            pa[0] = s;
            if (MEAS) {
                m_sat += __popc(sum0) + 2 * __popc(sum1) + 4 * __popc(sum2) + 6 * __popc(f);
                m_sat -= 2 * (__popc(sum0 & f) + 2 * __popc(sum1 & f) + 4 * __popc(sum2 & f));
                m_up += __popc(s) + __popc(o);
                ++m_words;
            }
            if (SINGLE) break;
        }
        cluster_arrive();
        if (MEAS) {
            if (threadIdx.x == 0) { rec_sum[0] = 0; rec_sum[1] = 0; }
            __syncthreads();
            block_accumulate2(192ull * m_words - m_sat, m_up, rec_sum);   // (a CTA barrier inside; warp 0 adds the totals)
            if (threadIdx.x == 0) {
                if (p.E) atomicAdd(reinterpret_cast<unsigned long long *>(p.E + (size_t)rec * p.nsamples + sample), 2ull * rec_sum[0]);
                if (p.M) atomicAdd(reinterpret_cast<unsigned long long *>(p.M + (size_t)rec * p.nsamples + sample), 2ull * rec_sum[1]);
            }
            ++rec;
        }
        if (RNG != 0 && c == 1) A = minstd_mulmod(16807u, A);   // the next half-sweep belongs to the next sweep
        if (kk + 1 < p.nhalf) {   // the draws of the thread's first word for the next half-sweep, under the barrier
            if (RNG == 0) fold_philox_time(p.seed, sample, t + 1, &pc, &ps);
            masks(first, 1 - c, c4, c8, c12);
        }
        cluster_wait();
    };
    // Half-sweeps in runs that end at a record (RECORDS) or at the end of the call
    const uint32_t run = RECORDS && p.every != 0 ? p.every : p.nhalf;
    for (uint32_t k0 = 0; k0 < p.nhalf; k0 += run) {
        const uint32_t k1 = k0 + run < p.nhalf ? k0 + run : p.nhalf;
        const bool record = RECORDS && k1 == k0 + run;
        const uint32_t k_plain = record ? k1 - 1 : k1;
        for (uint32_t kk = k0; kk < k_plain; ++kk) half_sweep(kk, false_type_tag());
        if (record) half_sweep(k1 - 1, true_type_tag());
    }

    // ---- store the spins (every remote read of this slab is complete: its reader has passed the last barrier) -----------
    {
        const size_t goff = (size_t)sample * p.lattice_stride + (size_t)z0 * plane;
        for (uint32_t i = threadIdx.x; i < nw; i += blockDim.x) {
            p.A.S[0][goff + i] = sm[i];
            p.A.S[1][goff + i] = sm[nw + i];
        }
    }
}

}  // namespace isingk
