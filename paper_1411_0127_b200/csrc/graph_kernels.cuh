// graph_kernels.cuh -- half-sweeps of small lattices replayed from a CUDA graph ("a CUDA graph or a persistent
// cooperative kernel is used for small L"; saturating the GPU at small L).
//
// Measured on this part (profiles/r2j_launch_floor.md): a kernel launched into a stream costs at least 2.35 us, with or without
// programmatic dependent launch, whatever it does -- that is the rate at which the host can submit launches -- while empty kernels
// replayed from an instantiated graph follow each other every 0.5-0.9 us.  For the one-sample lattices L = 64 and 128 (L = 64 is since served by the cluster-resident kernel of cluster_kernels.cuh, and comes
// here only under kernel choice 5), whose
// half-sweep kernel runs for about 2 us, graph replays are 10-25 % faster than launches (2.1-2.3 against 2.6-2.7 us per half-sweep);
// from L = 192 on the kernels are longer than a launch and the stream launches, which overlap consecutive kernels by programmatic
// dependent launch, are as fast or faster, and the sample-packed variant lost at every size (its per-sample Philox constants do not
// fit the constant slot, so it ran the plain ten rounds): graphs are used for L <= 128, one sample.  A graph is replayed unchanged, so nothing a
// half-sweep needs may sit in its launch parameters if it changes from one half-sweep to the next or from one call to the next:
// the half-sweep counter t (colour, Philox counter, MINSTD multiplier), the thresholds of beta, where the records go.  Those live in
// a slot of constant memory, c_dyn[slot]:
//   * ising_sweep / ising_sweep_trace write the call's values to a device copy of the slot (dyn_begin);
//   * a graph is [dyn_prepare: MINSTD multipliers of the coming sweeps] -> [copy of the device copy into the constant slot] ->
//     K half-sweep kernels, the k-th working at t + k with k a launch parameter -> [dyn_advance: t += K, record index += records];
//   * the kernels derive everything else from t + k with uniform (per-warp) arithmetic: the operand arrays of the colour, the folded
//     Philox constants (fold_philox), the multiplier A[(t + k >> 1) - (t >> 1)].  Being read from the constant bank and kernel
//     parameters, all of it stays in the uniform datapath: no registers, no per-thread work.
// Recording half-sweeps add into pre-set records as everywhere (add_to_record).  The bits are those of one launch per half-sweep.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sweep_kernels.cuh"

namespace isingk {

constexpr int DYN_SLOTS = 16;          // graph-using handles alive at the same time (others fall back to launches)
constexpr int DYN_MAX_STEPS = 128;     // half-sweeps per graph
constexpr int DYN_MAX_SWEEPS = DYN_MAX_STEPS / 2 + 2;

struct DynConst {
    unsigned long long t;     // half-sweep counter of the first step of the replay in flight
    unsigned int rec;         // index of the first record of this replay
    unsigned int minstd;      // fill A[] (rng mode MINSTD)
    long long *E, *M;         // the call's record arrays (null: none)
    Thresholds T;
    uint32_t A[DYN_MAX_SWEEPS];   // MINSTD: 16807^(n+1) mod M for the sweeps n = (t >> 1) + i
};

__constant__ DynConst c_dyn[DYN_SLOTS];

__global__ void dyn_begin(DynConst *d, unsigned long long t, unsigned int minstd, long long *E, long long *M, Thresholds T)
{
    d->t = t;
    d->rec = 0;
    d->minstd = minstd;
    d->E = E;
    d->M = M;
    d->T = T;
}

// <<<1, DYN_MAX_SWEEPS>>>
__global__ void dyn_prepare(DynConst *d)
{
    if (d->minstd) d->A[threadIdx.x] = minstd_power((d->t >> 1) + threadIdx.x + 1);
}

__global__ void dyn_advance(DynConst *d, unsigned int nsteps, unsigned int nrec)
{
    d->t += nsteps;
    d->rec += nrec;
}

// Step k of a replay, site-packed lattices with whole-word rows (the word-parallel tile update).  grid as half_sweep_site_packed.
template <int RNG, int W, bool MEASURE>
__global__ void __launch_bounds__(SWEEP_THREADS)
half_sweep_site_packed_graph(const __grid_constant__ LatticeArrays A, int L, uint64_t seed, uint4 *tab0, uint4 *tab1, int slot, uint32_t k,
                             uint32_t rec_off)
{
    const DynConst &d = c_dyn[slot];
    const uint64_t t = d.t + k;
    const int c = (int)(t & 1);
    SweepArgs a;
    a.S_act = A.S[c];
    a.S_oth = A.S[1 - c];
#pragma unroll
    for (int dd = 0; dd < 3; ++dd) { a.J_act[dd] = A.J[dd][c]; a.J_oth[dd] = A.J[dd][1 - c]; }
    a.L = L;
    a.colour = c;
    a.T = d.T;
    SiteRng sr;
    sr.seed = seed;
    sr.A2 = RNG == 0 ? 0u : 2u * d.A[(uint32_t)((t >> 1) - (d.t >> 1))];
    sr.s0tab = c ? tab1 : tab0;
    if (RNG == 0) fold_philox(seed, 0u, t, &sr.pc, &sr.ps);
    unsigned long long unsat = 0, up = 0;
    site_packed_tile<RNG, W, MEASURE, false>(a, sr, blockIdx.x, blockIdx.y, gridDim.x, unsat, up);
    if (MEASURE) add_to_record(unsat, up, d.E ? d.E + d.rec + rec_off : nullptr, d.M ? d.M + d.rec + rec_off : nullptr);
}

}  // namespace isingk
