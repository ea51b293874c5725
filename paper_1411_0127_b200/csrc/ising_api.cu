// ising_api.cu -- the C ABI of include/ising.h: handle, workspace carving, threshold table (row a1) and launches.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <mutex>
#include <new>

#include "../../include/ising.h"
#include "batch_kernels.cuh"
#include "cluster_kernels.cuh"
#include "fnv_kernels.cuh"
#include "graph_kernels.cuh"
#include "lane_rng.cuh"
#include "layout_kernels.cuh"
#include "measure_kernels.cuh"
#include "persistent.cuh"
#include "slab_kernels.cuh"
#include "sliced_kernels.cuh"
#include "sweep_kernels.cuh"

using namespace isingk;

namespace {

constexpr size_t ALIGN_WORDS = 64;  // 256-byte alignment of every internal array
constexpr int MAX_L = 4096;         // Philox group index g = j>>2 below 2^33: counter word c3 = hi32(g) is 0 or 1 (rng.cuh, R9)
constexpr int MAX_L_32BIT_GROUPS = 2048;   // up to here every layout is available (and g < 2^32; g passes 2^32 from L = 3252 on)

inline size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Geometry {
    int L, nsamples, nbatches;  // nbatches = 0: site-packed
    bool batched;               // nsamples > 1 site-packed lattices one after the other (batch_kernels.cuh); then nbatches = 0
    int nlat;                   // site-packed lattices in the workspace: 1, or nsamples when batched (0: sample-packed)
    uint64_t N, Hc;             // sites, sites per colour
    size_t canon_words;         // W = ceil(N/32)
    size_t array_words;         // words of one internal bit array (padded)
    size_t arrays_total_words;  // 8 arrays per lattice / batch
    size_t staging_words;       // canonical spins + couplings of all samples
    size_t acc_bytes;
    size_t s0_words;            // cached MINSTD seed states: 32 words per word of each colour array (fast layout only)
    size_t epoch_words;         // tile epochs of the persistent kernels (0: this geometry has no persistent path)
    uint32_t pgx, pgy;          // their tile grid
    bool onchip;                // small enough for half_sweeps_on_chip (one CTA, the lattice in shared memory)
    bool fast;                  // half-rows are whole words: L is a multiple of 64
    int W;                      // words per thread of the word-parallel kernel (fast layout)
};

// Lane modes (R19): default number of generator lanes = min(k N/8 units, one wave of threads on the 148 SMs: 8 CTAs of 128
// threads at 64 registers).
constexpr uint32_t MAX_LANES = 148u * 1024u;

inline bool lane_mode(int rng_mode) { return rng_mode == ISING_RNG_PR_SHARED || rng_mode == ISING_RNG_MT19937_SHARED; }
inline bool shared_mode(int rng_mode) { return rng_mode == ISING_RNG_PHILOX_SHARED || lane_mode(rng_mode); }
inline bool known_mode(int rng_mode) { return rng_mode >= ISING_RNG_PHILOX && rng_mode <= ISING_RNG_MT19937_SHARED; }
inline uint32_t lanes_default(const Geometry &g, int rng_mode)
{
    (void)rng_mode;
    const uint64_t units = (g.N / 8) * (uint64_t)(g.nbatches > 0 ? g.nbatches : 1);
    return (uint32_t)(units < MAX_LANES ? units : MAX_LANES);
}
inline uint32_t lane_ring(int rng_mode) { return rng_mode == ISING_RNG_PR_SHARED ? 62u : rng_mode == ISING_RNG_MT19937_SHARED ? 624u : 0u; }

// Which (L, nsamples, rng_mode) can be stored as a batch of site-packed lattices: independent draws (modes 0, 1), whole-word rows.
inline bool batch_layout_possible(int L, int nsamples, int rng_mode)
{
    return nsamples > 1 && L % 64 == 0 && (rng_mode == ISING_RNG_PHILOX || rng_mode == ISING_RNG_MINSTD);
}

// batched: nsamples > 1 as a batch of site-packed lattices (the caller has checked batch_layout_possible)
bool make_geometry(int L, int nsamples, Geometry *g, bool batched = false)
{
    if (L < 4 || (L & 1) || L > MAX_L) return false;
    if (!(nsamples == 1 || (nsamples > 0 && nsamples % 32 == 0))) return false;
    if (L > MAX_L_32BIT_GROUPS) {   // beyond 2^32 groups: one sample, the word-parallel layout with a row in at most 32 lanes
        const int wpr = L >> 6;     // (L = 2560, 3072, 4096: rows of 5, 3, 1 x 2^e words)
        int odd = wpr;
        while (odd % 2 == 0) odd /= 2;
        if (nsamples != 1 || L % 64 != 0 || !(odd == 1 || odd == 3 || odd == 5)) return false;
    }
    const bool site = nsamples == 1 || batched;
    g->L = L;
    g->nsamples = nsamples;
    g->batched = batched && nsamples > 1;
    g->nlat = site ? nsamples : 0;
    g->nbatches = site ? 0 : nsamples / 32;
    g->N = (uint64_t)L * L * L;
    g->Hc = g->N / 2;
    g->canon_words = (size_t)((g->N + 31) / 32);
    const size_t raw = site ? (size_t)((g->Hc + 31) / 32) : (size_t)g->Hc;
    g->array_words = round_up(raw, ALIGN_WORDS);
    g->arrays_total_words = 8 * g->array_words * (site ? (size_t)nsamples : (size_t)g->nbatches);
    g->staging_words = round_up((size_t)nsamples * 4 * g->canon_words, ALIGN_WORDS);
    // popcounts + E, M of ising_run_host, then the ACC_SLOTS counter pairs and the ticket of the word-parallel energy kernel
    // ... + overlap counter (2), then (256-byte aligned) the device copy of the handle's slot of graph constants (graph_kernels.cuh)
    g->acc_bytes = round_up(((size_t)nsamples * 4 + 2 * ACC_SLOTS + 1 + 2) * sizeof(unsigned long long), 256) + round_up(sizeof(DynConst), 256);
    g->fast = site && L % 64 == 0;
    // Words per thread of the word-parallel kernel: 4 (one 128-bit load per operand array) from L = 512 on; below that
    // the lattice is a fraction of one wave of CTAs and one word per thread gives the most parallelism (measured).
    g->W = 1;
    if (g->fast) {
        const int wpr = L >> 6;
        int odd = wpr;
        while (odd % 2 == 0) odd /= 2;
        if (odd == 3 || odd == 5) g->W = odd;  // rows of 3 * 2^e or 5 * 2^e words: 3 or 5 words per thread, no idle lanes
        else if (odd == 1 && wpr >= 8) g->W = 4;
        // other odd parts (7, 9, 11, ...): one word per thread, the row padded to a power of two of lanes
        // a batch of lattices has the samples for parallelism: as many words per thread as the row allows (L = 128: 2, L = 256: 4)
        if (g->batched && odd == 1 && wpr >= 2) g->W = wpr >= 4 ? 4 : 2;
    }
    // cached MINSTD seed states: 2 colours x one 4-byte word per site of every thread of the word-parallel grid (rows
    // whose lane count is not a power of two are padded, RowMap in sweep_kernels.cuh); N words when L = 64*2^k
    // (a batch: one table per sample, as long as all of them stay below 4 GiB; beyond that the seeds are recomputed)
    g->s0_words = g->fast ? 2 * (size_t)L * L * row_map_tpr_pad((L >> 6) / g->W) * g->W * 32 : 0;
    if (g->batched) g->s0_words = g->s0_words * (size_t)nsamples <= (1ull << 30) ? g->s0_words * (size_t)nsamples : 0;
    if (L > MAX_L_32BIT_GROUPS) g->s0_words = 0;   // 67-275 GB of table: the seeds are recomputed
    // persistent paths (persistent.cuh): one-sample lattices with whole-word rows below L = 512 get a tile grid with epoch counters
    // (used automatically up to L = 128, where it beats the launches); one-sample lattices of at most 1024 words per colour that
    // are not of that kind (every other even L <= 40) run on one SM out of shared memory
    g->epoch_words = 0;
    g->pgx = g->pgy = 0;
    if (g->fast && g->W != 4 && L <= MAX_L_32BIT_GROUPS) {
        g->pgx = (uint32_t)(L / (32 / row_map_tpr_pad((L >> 6) / g->W)));
        g->pgy = (uint32_t)(L / (SWEEP_THREADS / 32));
        g->epoch_words = g->batched ? 0 : (size_t)g->pgx * g->pgy;
    }
    g->onchip = nsamples == 1 && !g->fast && (g->Hc + 31) / 32 <= ONCHIP_MAX_WORDS;
    return true;
}

}  // namespace

struct ising {
    Geometry g;
    uint64_t seed;
    int rng_mode;
    uint64_t t;
    int kernel_choice;
    uint64_t launches;
    uint32_t *ws;
    uint32_t *staging;
    unsigned long long *acc;
    uint32_t *s0tab;   // MINSTD mode, fast layout: seed-state tables of the two colours (nullptr otherwise)
    bool s0_ready;
    uint32_t *lane_state;  // lane modes: ring * nlanes words, strided (lane_rng.cuh)
    uint32_t nlanes;
    bool lanes_ready;
    bool slots_clean;  // the slots and the ticket of the fused energy kernel are zero (it leaves them so)
    bool overlap_clean;  // the counter of ising_overlap is zero
    int device;          // CUDA device the workspace lives on (-1: unknown, e.g. no device present)
    // CUDA-graph path (graph_kernels.cuh): the handle's constant slot (-1: none yet / none free), the device copy of its contents, a
    // private stream to capture on (the caller's may be the legacy default stream), and the instantiated graphs
    struct GraphEntry { cudaGraphExec_t exec; uint32_t K, every; bool records; uint64_t last_use; };
    int dyn_slot;
    DynConst *dyn;
    cudaStream_t cap_stream;
    GraphEntry graphs[8];
    int ngraphs;
    uint64_t graph_clock;
    uint32_t *push_dn[2], *push_up[2];   // z-slab handles, per colour: the neighbours' halo planes this slab's boundary kernel stores into (ising_slab_connect)
    int nslabs, slab, z0, Lz;  // z-slab handles (ising_create_slab): this handle owns the planes z0 .. z0 + Lz - 1; nslabs = 0 otherwise
    unsigned int *epochs;  // tile epochs of the persistent kernels (nullptr: no persistent path for this geometry / mode)
    bool no_cluster;       // kernel choice 5: the automatic choice without the cluster-resident kernels
    int cluster_size;      // CTAs per cluster of the cluster-resident kernel (0: not asked yet, -1: none for this handle / device)
    int persist_grid[2];   // co-resident CTAs of this handle's persistent kernel without / with records (0: not asked yet, -1: none)

    LatticeArrays arrays(int batch) const
    {
        LatticeArrays A;
        uint32_t *base = ws + (size_t)batch * 8 * g.array_words;
        A.S[0] = base;
        A.S[1] = base + g.array_words;
        for (int d = 0; d < 3; ++d)
            for (int c = 0; c < 2; ++c) A.J[d][c] = base + (size_t)(2 + 2 * d + c) * g.array_words;
        return A;
    }
};

namespace {

thread_local bool g_launch_failed = false;  // set by launch_pdl when cudaLaunchKernelEx itself reports a failure

int check_launch(ising_t *h, int n = 1)
{
    h->launches += (uint64_t)n;
    const bool failed = g_launch_failed;
    g_launch_failed = false;
    return cudaGetLastError() == cudaSuccess && !failed ? ISING_OK : ISING_ECUDA;
}

// The workspace of a handle lives on one device (recorded by ising_create); every launch must be made with that device
// current, or the kernels would dereference another GPU's memory (peer access) or fault (none).
bool on_own_device(const ising_t *h);
void release_graphs(ising_t *h);
int slab_load_state(ising_t *h, const uint32_t *d_spins, const uint32_t *d_J, cudaStream_t st);
int slab_get_spins(ising_t *h, uint32_t *d_out, cudaStream_t st);
int slab_energy(ising_t *h, long long *d_E, long long *d_M, cudaStream_t st);

// Row a1 (R5, R6).  Plain double arithmetic with the C library's exp; compiled without FMA contraction.
int compute_thresholds(double beta, int rng_mode, uint64_t out[3])
{
    if (!(beta >= 0.0)) return ISING_EINVAL;
    if (!known_mode(rng_mode)) return ISING_EINVAL;
    for (int k = 0; k < 3; ++k) {
        const double dE = 4.0 * (double)(k + 1);
        const double x = beta * dE;
        const double p = exp(-x);
        const double scaled = rng_mode != ISING_RNG_MINSTD ? ldexp(p, 32) : 2147483647.0 * p;
        out[k] = (uint64_t)floor(scaled);
    }
    return ISING_OK;
}

Thresholds kernel_thresholds(const uint64_t T[3])
{
    Thresholds k;
    uint32_t *t = &k.t4, *al = &k.always4;
    for (int i = 0; i < 3; ++i) {
        const bool always = T[i] > 0xFFFFFFFFull;
        t[i] = always ? 0xFFFFFFFFu : (uint32_t)T[i];
        al[i] = always ? 0xFFFFFFFFu : 0u;
    }
    return k;
}

void fill_rng_launch(const ising_t *h, int batch, RngLaunch *r)
{
    memset(r, 0, sizeof(*r));
    // (a batch of site-packed lattices: `batch` is the sample, a one-sample lattice whose key / seed is that of the sample)
    const uint32_t sample_base = h->g.batched ? (uint32_t)batch : (uint32_t)(batch * 32);
    r->seed = h->g.batched ? h->seed + (uint64_t)batch * h->g.N * SPLITMIX_GAMMA : h->seed;
    r->tlo = (uint32_t)h->t;
    r->thi = (uint32_t)(h->t >> 32);
    r->k0 = (uint32_t)h->seed;
    r->k1base = (uint32_t)(h->seed >> 32) ^ (h->g.batched ? sample_base : 0u);
    r->sample_base = sample_base;
    if (h->rng_mode == ISING_RNG_PHILOX) {
        const int ns = h->g.nbatches == 0 ? 1 : 32;
        for (int s = 0; s < ns; ++s) fold_philox(h->seed, sample_base + (uint32_t)s, h->t, &r->pc, &r->ps[s]);
    } else if (h->rng_mode == ISING_RNG_PHILOX_SHARED) {
        fold_philox(h->seed, (uint32_t)batch, h->t, &r->pc, &r->ps[0]);  // R18: the sample field of the key is the batch
    } else {
        r->A = minstd_power((h->t >> 1) + 1);
    }
}

// Launch with programmatic stream serialization (the kernel calls wait_for_previous_kernel() before its first load).
template <typename... KArgs, typename... Args>
void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    // a failed launch leaves its code in the runtime's last-error slot too, which check_launch reads; the return value is kept
    // so that a failure is never lost between the two
    if (cudaLaunchKernelEx(&cfg, kernel, args...) != cudaSuccess) g_launch_failed = true;
}

// The constants of the word-parallel kernels from the launch block; beyond L = 2048 also Philox's b, e for the counter word c3 = 1.
SiteRng site_rng_of(const ising_t *h, const RngLaunch &r)
{
    SiteRng sr;
    sr.pc = r.pc;
    sr.ps = r.ps[0];
    sr.seed = r.seed;
    sr.A2 = 2u * r.A;
    sr.s0tab = nullptr;
    sr.b_hi = sr.e_hi = 0u;
    if (h->rng_mode == ISING_RNG_PHILOX && h->g.L > MAX_L_32BIT_GROUPS) {
        PhiloxCommonConst pc1;
        PhiloxSampleConst ps1;
        fold_philox(h->seed, 0u, h->t, &pc1, &ps1, 1u);
        sr.b_hi = ps1.b;
        sr.e_hi = ps1.e;
    }
    return sr;
}

// The word-parallel kernel for W words per thread, plain or with E and M of the resulting configuration (MEASURE).
template <int RNG, int W>
void launch_site_packed_w(bool measure, dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr, unsigned long long *slots,
                          long long N, long long *mE, long long *mM)
{
    // lattices beyond L = 2048 with Philox: the instance that knows about the counter word c3 (sweep_kernels.cuh, BIG)
    if (RNG == 0 && W >= 3 && a.L > MAX_L_32BIT_GROUPS) {
        constexpr int WB = W >= 3 ? W : 4;
        if (measure) launch_pdl(half_sweep_site_packed<0, WB, true, true>, grid, dim3(SWEEP_THREADS), st, a, sr, slots, N, mE, mM);
        else launch_pdl(half_sweep_site_packed<0, WB, false, true>, grid, dim3(SWEEP_THREADS), st, a, sr, (unsigned long long *)nullptr, 0ll,
                        (long long *)nullptr, (long long *)nullptr);
        return;
    }
    if (measure) launch_pdl(half_sweep_site_packed<RNG, W, true>, grid, dim3(SWEEP_THREADS), st, a, sr, slots, N, mE, mM);
    else launch_pdl(half_sweep_site_packed<RNG, W, false>, grid, dim3(SWEEP_THREADS), st, a, sr, (unsigned long long *)nullptr, 0ll,
                    (long long *)nullptr, (long long *)nullptr);
}
template <int RNG>
void launch_site_packed(int W, bool measure, dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr, unsigned long long *slots,
                        long long N, long long *mE, long long *mM)
{
    if (W == 4) launch_site_packed_w<RNG, 4>(measure, grid, st, a, sr, slots, N, mE, mM);
    else if (W == 3) launch_site_packed_w<RNG, 3>(measure, grid, st, a, sr, slots, N, mE, mM);
    else if (W == 5) launch_site_packed_w<RNG, 5>(measure, grid, st, a, sr, slots, N, mE, mM);
    else launch_site_packed_w<RNG, 1>(measure, grid, st, a, sr, slots, N, mE, mM);
}

// The same for a batch of lattices (batch_kernels.cuh): grid.z = samples of this launch.
template <int RNG, int W>
void launch_batch_w(bool measure, dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr, const BatchInfo &bi, long long *mE,
                    long long *mM)
{
    if (measure) launch_pdl(half_sweep_site_packed_batch<RNG, W, true>, grid, dim3(SWEEP_THREADS), st, a, sr, bi, mE, mM);
    else launch_pdl(half_sweep_site_packed_batch<RNG, W, false>, grid, dim3(SWEEP_THREADS), st, a, sr, bi, (long long *)nullptr,
                    (long long *)nullptr);
}
template <int RNG>
void launch_batch(int W, bool measure, dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr, const BatchInfo &bi, long long *mE,
                  long long *mM)
{
    if (W == 4) launch_batch_w<RNG, 4>(measure, grid, st, a, sr, bi, mE, mM);
    else if (W == 2) launch_batch_w<RNG, 2>(measure, grid, st, a, sr, bi, mE, mM);
    else if (W == 3) launch_batch_w<RNG, 3>(measure, grid, st, a, sr, bi, mE, mM);
    else if (W == 5) launch_batch_w<RNG, 5>(measure, grid, st, a, sr, bi, mE, mM);
    else launch_batch_w<RNG, 1>(measure, grid, st, a, sr, bi, mE, mM);
}

BatchInfo batch_info(const ising_t *h, uint32_t sample0)
{
    BatchInfo bi;
    bi.lattice_stride = 8 * h->g.array_words;
    bi.tab_stride = h->g.s0_words / 2 / (size_t)h->g.nsamples / 4;   // uint4 elements of one sample's table of one colour
    bi.N = h->g.N;
    bi.t = h->t;
    bi.nsamples = (uint32_t)h->g.nsamples;
    bi.sample0 = sample0;
    return bi;
}

// MINSTD, batch of lattices: the seed tables of all samples (colour c of sample s at tab[c] + s * tab_stride), once per handle.
int batch_fill_seed_tables(ising_t *h, cudaStream_t st)
{
    const Geometry &g = h->g;
    if (h->s0_ready) return ISING_OK;
    uint4 *tab[2] = {(uint4 *)h->s0tab, (uint4 *)(h->s0tab + g.s0_words / 2)};
    for (int s0 = 0; s0 < g.nsamples; s0 += 65535) {
        const int ns = g.nsamples - s0 < 65535 ? g.nsamples - s0 : 65535;
        const dim3 grid(g.pgx ? g.pgx : (unsigned)(g.L / (32 / row_map_tpr_pad((g.L >> 6) / g.W))), (unsigned)(g.L / (SWEEP_THREADS / 32)), (unsigned)ns);
        const BatchInfo bi = batch_info(h, (uint32_t)s0);
        for (int cc = 0; cc < 2; ++cc) {
            if (g.W == 4) minstd_fill_s0_batch<4><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, bi);
            else if (g.W == 2) minstd_fill_s0_batch<2><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, bi);
            else if (g.W == 3) minstd_fill_s0_batch<3><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, bi);
            else if (g.W == 5) minstd_fill_s0_batch<5><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, bi);
            else minstd_fill_s0_batch<1><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, bi);
        }
        const int rc = check_launch(h, 2);
        if (rc != ISING_OK) return rc;
    }
    h->s0_ready = true;
    return ISING_OK;
}

// mE / mM (device, may be null): where the half-sweep itself writes E and M of the configuration it leaves; honoured by the
// word-parallel site-packed kernel only (see can_measure_in_sweep), ignored elsewhere.
template <int RNG>
int launch_half_sweep(ising_t *h, const Thresholds &T, cudaStream_t st, long long *mE = nullptr, long long *mM = nullptr)
{
    const Geometry &g = h->g;
    const int c = (int)(h->t & 1);
    const int nb = g.nbatches == 0 ? g.nlat : g.nbatches;
    for (int b = 0; b < nb; ++b) {
        const LatticeArrays A = h->arrays(b);
        SweepArgs a{};
        a.S_act = A.S[c];
        a.S_oth = A.S[1 - c];
        for (int d = 0; d < 3; ++d) { a.J_act[d] = A.J[d][c]; a.J_oth[d] = A.J[d][1 - c]; }
        a.L = g.L;
        a.colour = c;
        a.T = T;
        RngLaunch r;
        fill_rng_launch(h, b, &r);
        if (RNG == 2) {
            const uint64_t ngroups = g.Hc / 4;
            if (g.L % 8 == 0 && h->kernel_choice != 1) {
                // all coded batches in one launch (blockIdx.z = batch): a is batch 0 here, b == 0
                SharedRng sr;
                sr.tlo = r.tlo; sr.thi = r.thi; sr.k0 = r.k0; sr.k1base = r.k1base;
                const uint32_t gpr = (uint32_t)g.L / 8;
                const uint32_t gpr_inv = (uint32_t)((0x100000000ull + gpr - 1) / gpr);
                if (g.L < 32) {  // fewer than 128 groups per plane: the thread index runs over (batch, group)
                    const uint64_t units = (uint64_t)nb * (g.N / 8);
                    launch_pdl(half_sweep_shared_vec<true>, dim3((unsigned)((units + 127) / 128)), dim3(128), st, a, sr, gpr, gpr_inv,
                               (size_t)(8 * g.array_words), (uint32_t)nb, 0u);
                } else {
                    // blockIdx.z = batch: at most 65535 per launch (more than that is 2 M samples, still within a B200's HBM at L = 32)
                    for (int b0 = 0; b0 < nb; b0 += 65535) {
                        const int nbh = nb - b0 < 65535 ? nb - b0 : 65535;
                        const dim3 grid((unsigned)(((uint64_t)g.L * gpr + 127) / 128), (unsigned)g.L, (unsigned)nbh);
                        launch_pdl(half_sweep_shared_vec<false>, grid, dim3(128), st, a, sr, gpr, gpr_inv, (size_t)(8 * g.array_words),
                                   (uint32_t)nbh, (uint32_t)b0);
                        if (b0 + nbh < nb) {
                            const int rc = check_launch(h);
                            if (rc != ISING_OK) return rc;
                        }
                    }
                }
                const int rc = check_launch(h);
                if (rc != ISING_OK) return rc;
                break;
            }
            if (nb > 1 && nb <= 65535 && h->kernel_choice != 1) {  // all coded batches in one launch (a is batch 0, b == 0)
                launch_pdl(half_sweep_sample_packed<2, 1, true>, dim3((unsigned)((ngroups + 127) / 128), (unsigned)nb), dim3(128), st, a, r,
                           (uint32_t)ngroups, (uint64_t)g.N, (size_t)(8 * g.array_words));
                const int rc = check_launch(h);
                if (rc != ISING_OK) return rc;
                break;
            }
            launch_pdl(half_sweep_sample_packed<2, 1, false>, dim3((unsigned)((ngroups + 127) / 128)), dim3(128), st, a, r, (uint32_t)ngroups,
                       (uint64_t)g.N, (size_t)0);
        } else if (g.nbatches != 0) {
            const uint64_t ngroups = g.Hc / 4;
            // small lattices: 4 threads per group (8 samples each) so that the grid covers the 148 SMs
            if (g.L % 8 == 0 && h->kernel_choice != 1) {  // 128-bit loads
                const uint32_t gpr = (uint32_t)g.L / 8, inv = (uint32_t)((0x100000000ull + gpr - 1) / gpr);
                const uint64_t per_plane = (uint64_t)g.L * gpr;
                const size_t bstride = (size_t)(8 * g.array_words);
                if (nb > 1 && nb <= 65535) {  // all coded batches in one launch (a is batch 0 here, b == 0)
                    if (ngroups * (uint64_t)nb < 148u * 1024u)
                        launch_pdl(half_sweep_sample_packed_vec<RNG, 4, true>, dim3((unsigned)((per_plane + 31) / 32), (unsigned)g.L, (unsigned)nb), dim3(128), st, a, r, gpr, inv, (uint64_t)g.N, bstride);
                    else
                        launch_pdl(half_sweep_sample_packed_vec<RNG, 1, true>, dim3((unsigned)((per_plane + 127) / 128), (unsigned)g.L, (unsigned)nb), dim3(128), st, a, r, gpr, inv, (uint64_t)g.N, bstride);
                    const int rc = check_launch(h);
                    if (rc != ISING_OK) return rc;
                    break;
                }
                if (ngroups < 148u * 1024u)
                    launch_pdl(half_sweep_sample_packed_vec<RNG, 4, false>, dim3((unsigned)((per_plane + 31) / 32), (unsigned)g.L), dim3(128), st, a, r, gpr, inv, (uint64_t)g.N, bstride);
                else
                    launch_pdl(half_sweep_sample_packed_vec<RNG, 1, false>, dim3((unsigned)((per_plane + 127) / 128), (unsigned)g.L), dim3(128), st, a, r, gpr, inv, (uint64_t)g.N, bstride);
            } else if (nb > 1 && nb <= 65535 && h->kernel_choice != 1) {  // any even L, all coded batches in one launch
                const size_t bstride = (size_t)(8 * g.array_words);
                if (ngroups * (uint64_t)nb < 148u * 1024u)
                    launch_pdl(half_sweep_sample_packed<RNG, 4, true>, dim3((unsigned)((ngroups + 31) / 32), (unsigned)nb), dim3(128), st, a, r, (uint32_t)ngroups, (uint64_t)g.N, bstride);
                else
                    launch_pdl(half_sweep_sample_packed<RNG, 1, true>, dim3((unsigned)((ngroups + 127) / 128), (unsigned)nb), dim3(128), st, a, r, (uint32_t)ngroups, (uint64_t)g.N, bstride);
                const int rc = check_launch(h);
                if (rc != ISING_OK) return rc;
                break;
            } else if (ngroups < 148u * 1024u)
                launch_pdl(half_sweep_sample_packed<RNG, 4, false>, dim3((unsigned)((ngroups + 31) / 32)), dim3(128), st, a, r, (uint32_t)ngroups, (uint64_t)g.N, (size_t)0);
            else
                launch_pdl(half_sweep_sample_packed<RNG, 1, false>, dim3((unsigned)((ngroups + 127) / 128)), dim3(128), st, a, r, (uint32_t)ngroups, (uint64_t)g.N, (size_t)0);
        } else if (g.fast && h->kernel_choice != 1) {
            const int wpr = g.L >> 6;
            const int W = g.W;
            unsigned long long *slots = nullptr;   // (the measuring variant adds to the pre-set record itself: add_to_record)
            const int tpr_pad = row_map_tpr_pad(wpr / W);
            const dim3 grid((unsigned)(g.L / (32 / tpr_pad)), (unsigned)(g.L / (SWEEP_THREADS / 32)));
            SiteRng sr = site_rng_of(h, r);
            // MINSTD: the seed states s0(seed, site) come from the table unless kernel choice 2 asks for recomputation
            const bool cached = RNG == 1 && h->kernel_choice != 2 && h->s0tab != nullptr;
            if (g.batched) {   // all samples in one launch (blockIdx.z = sample; a, sr are sample 0 here, b == 0)
                sr.seed = h->seed;
                if (cached) {
                    const int rc = batch_fill_seed_tables(h, st);
                    if (rc != ISING_OK) return rc;
                    sr.s0tab = (uint4 *)(h->s0tab + (c ? g.s0_words / 2 : 0));
                }
                for (int s0 = 0; s0 < g.nsamples; s0 += 65535) {
                    const int ns = g.nsamples - s0 < 65535 ? g.nsamples - s0 : 65535;
                    const BatchInfo bi = batch_info(h, (uint32_t)s0);
                    const dim3 gridb(grid.x, grid.y, (unsigned)ns);
                    if (cached) launch_batch<2>(W, mE != nullptr || mM != nullptr, gridb, st, a, sr, bi, mE, mM);
                    else launch_batch<RNG>(W, mE != nullptr || mM != nullptr, gridb, st, a, sr, bi, mE, mM);
                    if (s0 + ns < g.nsamples) {
                        const int rc = check_launch(h);
                        if (rc != ISING_OK) return rc;
                    }
                }
                const int rc = check_launch(h);
                if (rc != ISING_OK) return rc;
                break;
            }
            if (cached) {
                uint4 *tab[2] = {(uint4 *)h->s0tab, (uint4 *)(h->s0tab + g.s0_words / 2)};
                if (!h->s0_ready) {  // once per handle: the seed states depend on (seed, site) only (R11)
                    for (int cc = 0; cc < 2; ++cc) {
                        if (W == 4) minstd_fill_s0<4><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
                        else if (W == 3) minstd_fill_s0<3><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
                        else if (W == 5) minstd_fill_s0<5><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
                        else minstd_fill_s0<1><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
                    }
                    const int rc = check_launch(h, 2);
                    if (rc != ISING_OK) return rc;
                    h->s0_ready = true;
                }
                sr.s0tab = tab[c];
                launch_site_packed<2>(W, mE != nullptr || mM != nullptr, grid, st, a, sr, slots, (long long)g.N, mE, mM);
            } else {
                launch_site_packed<RNG>(W, mE != nullptr || mM != nullptr, grid, st, a, sr, slots, (long long)g.N, mE, mM);
            }
        } else if (h->kernel_choice != 1 && g.Hc < (1ull << 32)) {  // any even L: the word update on operands gathered as bit windows
            const uint64_t nw = (g.Hc + 31) / 32;
            SiteRng sr;   // the small per-launch constant block (the 1.4 KB RngLaunch doubles the enqueue cost of a tiny launch)
            sr.pc = r.pc;
            sr.ps = r.ps[0];
            sr.seed = r.seed;
            sr.A2 = 2u * r.A;
            sr.s0tab = nullptr;
            if (g.L >= 64) {  // rows of at least 32 bits: no segment loop
                unsigned long long *slots = nullptr;
                if (mE || mM) {
                    launch_pdl(half_sweep_site_packed_rows2<RNG, true>, dim3((unsigned)((nw + 127) / 128)), dim3(128), st, a, sr, (uint32_t)nw,
                               (uint32_t)g.Hc, slots, (long long)g.N, mE, mM);
                } else {
                    launch_pdl(half_sweep_site_packed_rows2<RNG, false>, dim3((unsigned)((nw + 127) / 128)), dim3(128), st, a, sr, (uint32_t)nw,
                               (uint32_t)g.Hc, (unsigned long long *)nullptr, 0ll, (long long *)nullptr, (long long *)nullptr);
                }
            } else
                launch_pdl(half_sweep_site_packed_rows<RNG>, dim3((unsigned)((nw + 127) / 128)), dim3(128), st, a, sr, (uint32_t)nw, (uint32_t)g.Hc);
        } else {
            const uint64_t nw = (g.Hc + 31) / 32;
            launch_pdl(half_sweep_site_packed_generic<RNG>, dim3((unsigned)((nw + 255) / 256)), dim3(256), st, a, r, (uint64_t)nw, (uint64_t)g.Hc);
        }
        const int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
    }
    h->t += 1;
    return ISING_OK;
}

// Lane modes (R19): one launch per half-sweep, thread = lane; the lane state is seeded by the first launch of the handle.
template <int GEN>
int launch_half_sweep_lanes(ising_t *h, const Thresholds &T, cudaStream_t st)
{
    const Geometry &g = h->g;
    const unsigned blocks = (h->nlanes + 127u) / 128u;
    if (!h->lanes_ready) {
        lanes_init<GEN><<<blocks, 128, 0, st>>>(h->lane_state, h->nlanes, h->seed);
        const int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
        h->lanes_ready = true;
    }
    const int c = (int)(h->t & 1);
    const LatticeArrays A = h->arrays(0);
    SweepArgs a{};
    a.S_act = A.S[c];
    a.S_oth = A.S[1 - c];
    for (int d = 0; d < 3; ++d) { a.J_act[d] = A.J[d][c]; a.J_oth[d] = A.J[d][1 - c]; }
    a.L = g.L;
    a.colour = c;
    a.T = T;
    const uint32_t ngroups = (uint32_t)(g.N / 8);
    const uint64_t units = (uint64_t)g.nbatches * ngroups;   // (batch, group) pairs, batch-major (R19)
    const uint32_t rounds = (uint32_t)((units + h->nlanes - 1) / h->nlanes);
    const uint64_t per_half_sweep = 4ull * rounds;
    LaneArgs ln;
    ln.state = h->lane_state;
    ln.nlanes = h->nlanes;
    ln.pos0 = (uint32_t)((h->t % LaneRing<GEN>::size) * (per_half_sweep % LaneRing<GEN>::size) % LaneRing<GEN>::size);
    if (g.L % 8 == 0) {
        const uint32_t gpr = (uint32_t)g.L / 8, gpr_inv = (uint32_t)((0x100000000ull + gpr - 1) / gpr);
        // lattices beyond the L2 (126 MB): stream the read-once arrays past it (lane_rng.cuh)
        if (g.arrays_total_words * sizeof(uint32_t) > (96u << 20))
            launch_pdl(half_sweep_shared_lanes<GEN, true, true>, dim3(blocks), dim3(128), st, a, ln, gpr, gpr_inv, (size_t)(8 * g.array_words),
                       ngroups, units, rounds);
        else
            launch_pdl(half_sweep_shared_lanes<GEN, true, false>, dim3(blocks), dim3(128), st, a, ln, gpr, gpr_inv, (size_t)(8 * g.array_words),
                       ngroups, units, rounds);
    } else {  // groups that straddle rows: per-word neighbour loads
        launch_pdl(half_sweep_shared_lanes<GEN, false, false>, dim3(blocks), dim3(128), st, a, ln, 1u, 0u, (size_t)(8 * g.array_words), ngroups,
                   units, rounds);
    }
    const int rc = check_launch(h);
    if (rc != ISING_OK) return rc;
    h->t += 1;
    return ISING_OK;
}

// Can the half-sweep kernel of this handle return E and M itself (half_sweep_site_packed<.., MEASURE = true>)?
bool can_measure_in_sweep(const ising_t *h)
{
    if (h->g.nbatches != 0 || (h->rng_mode != ISING_RNG_PHILOX && h->rng_mode != ISING_RNG_MINSTD)) return false;
    if (h->g.fast) return h->kernel_choice != 1;                                                              // word-parallel kernel
    return h->g.L >= 64 && h->kernel_choice != 1 && h->g.Hc < (1ull << 32);                                   // loop-free bit-window kernel
}

int half_sweep(ising_t *h, const Thresholds &T, cudaStream_t st, long long *mE = nullptr, long long *mM = nullptr)
{
    if (h->rng_mode == ISING_RNG_PR_SHARED) return launch_half_sweep_lanes<GEN_PR>(h, T, st);
    if (h->rng_mode == ISING_RNG_MT19937_SHARED) return launch_half_sweep_lanes<GEN_MT>(h, T, st);
    if (h->rng_mode == ISING_RNG_PHILOX_SHARED) return launch_half_sweep<2>(h, T, st);
    return h->rng_mode == ISING_RNG_PHILOX ? launch_half_sweep<0>(h, T, st, mE, mM) : launch_half_sweep<1>(h, T, st, mE, mM);
}

// ---------------------------------------------------------------------------------------------------------------------
// Persistent path (persistent.cuh): all half-sweeps of a call in one cooperative launch, the CTAs synchronising tile by tile
// through epoch counters.  Automatic (kernel choice 0 or 2) for the geometries make_geometry gives a tile grid.
// ---------------------------------------------------------------------------------------------------------------------
// `records`: the call records E / M (ising_sweep_trace).
bool persistent_available(const ising_t *h, bool records)
{
    if (h->g.nsamples != 1 || (h->rng_mode != ISING_RNG_PHILOX && h->rng_mode != ISING_RNG_MINSTD)) return false;
    if (h->g.onchip) {
        if (h->kernel_choice == 4) return true;
        if (h->kernel_choice != 0 && h->kernel_choice != 2) return false;
        // automatic: where one SM beats a launch per half-sweep on all of them (profiles/r2n_small.md): with records up to 512
        // words per colour (L <= 32: 3.8-5.5 against 10.8-12.3 us per recorded half-sweep), without up to 216 (L <= 24)
        const uint64_t nw = (h->g.Hc + 31) / 32;
        return records ? nw <= 512 : nw <= 216;
    }
    if (!h->epochs) return false;
    // the dataflow kernel: on request only (kernel choice 4).  Its tile flags cost 1.4 us per half-sweep where a graph replay
    // (graph_kernels.cuh, the automatic choice for these lattices) costs 0.5-0.9 us (profiles/r2j_launch_floor.md)
    return h->kernel_choice == 4;
}

template <typename Kernel>
int launch_cooperative(ising_t *h, Kernel kernel, int threads, int which, const PersistArgs &p, uint32_t ntiles, cudaStream_t st)
{
    if (h->persist_grid[which] == 0) {   // once per handle: how many CTAs of this kernel are resident at once
        int per_sm = 0, sms = 0, dev = 0, coop = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, 0) != cudaSuccess)
            return ISING_ECUDA;
        h->persist_grid[which] = coop && per_sm > 0 ? per_sm * sms : -1;
    }
    if (h->persist_grid[which] < 0) return ISING_EINVAL;
    // every CTA walks over the same number of tiles (1024 tiles on 740 resident CTAs: 512 CTAs x 2 tiles, not 740 x 1.4)
    const uint32_t cap = (uint32_t)h->persist_grid[which], rounds = (ntiles + cap - 1) / cap;
    const unsigned grid = (ntiles + rounds - 1) / rounds;
    uint32_t gx = h->g.pgx, gy = h->g.pgy;
    void *args[] = {(void *)&p, (void *)&gx, (void *)&gy};
    if (cudaLaunchCooperativeKernel((const void *)kernel, dim3(grid), dim3((unsigned)threads), args, 0, st) != cudaSuccess) {
        cudaGetLastError();
        return ISING_ECUDA;
    }
    return check_launch(h);
}

template <int RNG, int W>
int launch_persistent_site(ising_t *h, const PersistArgs &p, bool records, cudaStream_t st)
{
    const uint32_t ntiles = h->g.pgx * h->g.pgy;
    if (records) return launch_cooperative(h, persistent_site_packed<RNG, W, true>, SWEEP_THREADS, 1, p, ntiles, st);
    return launch_cooperative(h, persistent_site_packed<RNG, W, false>, SWEEP_THREADS, 0, p, ntiles, st);
}
template <int RNG>
int launch_persistent_site(ising_t *h, const PersistArgs &p, bool records, cudaStream_t st)
{
    switch (h->g.W) {
        case 1: return launch_persistent_site<RNG, 1>(h, p, records, st);
        case 3: return launch_persistent_site<RNG, 3>(h, p, records, st);
        case 5: return launch_persistent_site<RNG, 5>(h, p, records, st);
        default: return ISING_EINVAL;
    }
}

// nhalf half-sweeps from the handle's counter on; site-packed handles record E / M after every `every`-th (0: none) into d_E / d_M.
int sweep_persistent(ising_t *h, const Thresholds &T, uint32_t nhalf, uint32_t every, long long *d_E, long long *d_M, cudaStream_t st)
{
    const Geometry &g = h->g;
    if (g.onchip) {   // one CTA, the lattice in shared memory, every half-sweep and record of the call in one launch
        PersistArgs p;
        memset(&p, 0, sizeof(p));
        p.A = h->arrays(0);
        p.L = g.L;
        p.T = T;
        p.seed = h->seed;
        p.t0 = h->t;
        p.nhalf = nhalf;
        p.every = (d_E || d_M) ? every : 0u;
        p.A_first = h->rng_mode == ISING_RNG_MINSTD ? minstd_power((h->t >> 1) + 1) : 0u;
        p.E = d_E;
        p.M = d_M;
        p.N = g.N;
        const uint32_t nw = (uint32_t)((g.Hc + 31) / 32);
        const size_t smem = 8 * (size_t)(nw + 1) * sizeof(uint32_t);
        if (h->rng_mode == ISING_RNG_PHILOX) half_sweeps_on_chip<0><<<1, ONCHIP_THREADS, smem, st>>>(p, nw, (uint32_t)g.Hc);
        else half_sweeps_on_chip<1><<<1, ONCHIP_THREADS, smem, st>>>(p, nw, (uint32_t)g.Hc);
        const int rc = check_launch(h);
        if (rc == ISING_OK) h->t += nhalf;
        return rc;
    }
    const bool site = true;
    const bool table = site && h->rng_mode == ISING_RNG_MINSTD && h->kernel_choice != 2 && h->s0tab != nullptr;
    uint4 *tab[2] = {nullptr, nullptr};
    if (table) {
        tab[0] = (uint4 *)h->s0tab;
        tab[1] = (uint4 *)(h->s0tab + g.s0_words / 2);
        if (!h->s0_ready) {
            const dim3 grid(g.pgx, g.pgy);
            for (int cc = 0; cc < 2; ++cc) {
                if (g.W == 3) minstd_fill_s0<3><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
                else if (g.W == 5) minstd_fill_s0<5><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
                else minstd_fill_s0<1><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed);
            }
            const int rc = check_launch(h, 2);
            if (rc != ISING_OK) return rc;
            h->s0_ready = true;
        }
    }
    const bool records = site && every != 0 && (d_E || d_M);
    if (records) {   // the records receive their counts by atomics: preset them to -3N / -N
        const uint32_t nrec = nhalf / every;
        if (nrec) {
            init_records<<<(nrec + 255) / 256, 256, 0, st>>>(d_E, d_M, nrec, (long long)g.N);
            const int rc = check_launch(h);
            if (rc != ISING_OK) return rc;
        }
    }
    // epochs are 32-bit and restart with every launch: at most 2^30 half-sweeps per launch; a chunk ends on a record boundary so
    // that `every` keeps its phase
    uint32_t chunk_max = 1u << 30;
    if (records) chunk_max -= chunk_max % every;
    uint32_t done = 0, rec = 0;
    while (done < nhalf) {
        const uint32_t n = nhalf - done < chunk_max ? nhalf - done : chunk_max;
        PersistArgs p;
        memset(&p, 0, sizeof(p));
        p.A = h->arrays(0);
        p.L = g.L;
        p.T = T;
        p.seed = h->seed;
        p.t0 = h->t;
        p.nhalf = n;
        p.every = records ? every : 0u;
        p.A_first = h->rng_mode == ISING_RNG_MINSTD ? minstd_power((h->t >> 1) + 1) : 0u;
        p.s0tab[0] = tab[0];
        p.s0tab[1] = tab[1];
        p.epoch = h->epochs;
        p.E = records && d_E ? d_E + rec : nullptr;
        p.M = records && d_M ? d_M + rec : nullptr;
        p.N = g.N;
        if (cudaMemsetAsync(h->epochs, 0, g.epoch_words * sizeof(uint32_t), st) != cudaSuccess) return ISING_ECUDA;
        int rc;
        if (h->rng_mode == ISING_RNG_PHILOX) rc = launch_persistent_site<0>(h, p, records, st);
        else if (table) rc = launch_persistent_site<2>(h, p, records, st);
        else rc = launch_persistent_site<1>(h, p, records, st);
        if (rc != ISING_OK) return rc;
        h->t += n;
        done += n;
        if (records) rec += n / every;
    }
    return ISING_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// Cluster-resident path (cluster_kernels.cuh): one thread-block cluster per sample, the lattice in distributed shared memory, all
// half-sweeps of the call in one launch.  L = 64 and 128, one sample or a batch of lattices, Philox or MINSTD.
// ---------------------------------------------------------------------------------------------------------------------
template <int RNG, int WPR>
auto cluster_kernel(bool records, int nw_fixed)
{
    // one word per thread with the slab size known at compile time (L = 64 in clusters of 16, 8, 4 CTAs), or the general kernel
    if (WPR == 1 && nw_fixed == 256) return records ? half_sweeps_cluster<RNG, 1, true, 256> : half_sweeps_cluster<RNG, 1, false, 256>;
    if (WPR == 1 && nw_fixed == 512) return records ? half_sweeps_cluster<RNG, 1, true, 512> : half_sweeps_cluster<RNG, 1, false, 512>;
    if (WPR == 1 && nw_fixed == 1024) return records ? half_sweeps_cluster<RNG, 1, true, 1024> : half_sweeps_cluster<RNG, 1, false, 1024>;
    return records ? half_sweeps_cluster<RNG, WPR, true, 0> : half_sweeps_cluster<RNG, WPR, false, 0>;
}

// nw_fixed: words per colour and CTA when every thread has exactly one of them (0: several words per thread)
void (*cluster_kernel_of(const ising_t *h, bool records, int nw_fixed))(const ClusterArgs)
{
    const bool philox = h->rng_mode == ISING_RNG_PHILOX;
    if (h->g.L == 64) return philox ? cluster_kernel<0, 1>(records, nw_fixed) : cluster_kernel<1, 1>(records, nw_fixed);
    return philox ? cluster_kernel<0, 2>(records, 0) : cluster_kernel<1, 2>(records, 0);
}

struct ClusterShape { int C, threads; size_t smem; int nw_fixed; };

ClusterShape cluster_shape(const ising_t *h, int C)
{
    const Geometry &g = h->g;
    const size_t nw = (size_t)g.L * (size_t)(g.L >> 6) * (size_t)(g.L / C);   // words of one array in one CTA
    ClusterShape s;
    s.C = C;
    s.threads = nw < (size_t)CLUSTER_MAX_THREADS ? (int)nw : CLUSTER_MAX_THREADS;
    s.smem = 8 * nw * sizeof(uint32_t);
    s.nw_fixed = nw <= (size_t)CLUSTER_MAX_THREADS ? (int)nw : 0;
    // MINSTD, one word per thread, at most 512 threads (and L = 64, where those kernels exist): the cached seed states of the thread
    if (h->rng_mode == ISING_RNG_MINSTD && g.L == 64 && s.nw_fixed && s.nw_fixed <= CLUSTER_SEED_CACHE_MAX_NW) s.smem += 256 * nw;
    return s;
}

// CTAs per cluster for this handle (0: no cluster path): the largest power of two up to 16 with samples x C <= the SMs of the
// device, at least what the shared memory asks for; checked once per handle against what the device can co-schedule.
int cluster_size_of(ising_t *h)
{
    if (h->cluster_size != 0) return h->cluster_size > 0 ? h->cluster_size : 0;
    h->cluster_size = -1;
    const Geometry &g = h->g;
    if (h->nslabs || !g.fast || g.nbatches != 0 || (g.L != 64 && g.L != 128)) return 0;
    if (h->rng_mode != ISING_RNG_PHILOX && h->rng_mode != ISING_RNG_MINSTD) return 0;
    int dev = 0, sms = 0, smem_max = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    int pref = 16;
    while (pref > 1 && (long long)g.nsamples * pref > sms) pref >>= 1;
    // MINSTD: clusters of 8 CTAs of 512 threads keep the seed states in shared memory; the clusters of many samples then run in waves
    // MINSTD at L = 64: clusters of at least 8 CTAs (at most 512 threads each) keep the seed states of their words in shared memory,
    // which is worth more than having all clusters resident at once: the clusters of many samples then run in waves, each through
    // all half-sweeps of the call (samples are independent)
    if (h->rng_mode == ISING_RNG_MINSTD && pref < 8 && g.L == 64) pref = 8;
    // Philox at L = 64: not below 4 CTAs (one word per thread, slab size a compile-time constant); more samples run in waves
    if (h->rng_mode == ISING_RNG_PHILOX && pref < 4 && g.L == 64) pref = 4;
    while (pref <= 16 && cluster_shape(h, pref).smem > (size_t)smem_max) pref <<= 1;
    // the preferred size, then smaller ones (a device that cannot co-schedule 16 CTAs), then larger ones: the first the device accepts
    int order[10], n = 0;
    for (int c = pref; c >= 1; c >>= 1) order[n++] = c;
    for (int c = 2 * pref; c <= 16; c <<= 1) order[n++] = c;
    for (int k = 0; k < n; ++k) {
        const int C = order[k];
        if (C > 16) continue;
        const ClusterShape cs = cluster_shape(h, C);
        if (cs.smem > (size_t)smem_max) continue;
        bool ok = true;
        for (int records = 0; records < 2 && ok; ++records) {
            auto kernel = cluster_kernel_of(h, records != 0, cs.nw_fixed);
            ok = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cs.smem) == cudaSuccess &&
                 (C <= 8 || cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess);
            if (!ok) break;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)C);
            cfg.blockDim = dim3((unsigned)cs.threads);
            cfg.dynamicSmemBytes = cs.smem;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = (unsigned)C;
            attr[0].val.clusterDim.y = 1;
            attr[0].val.clusterDim.z = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
            int nclusters = 0;
            ok = cudaOccupancyMaxActiveClusters(&nclusters, kernel, &cfg) == cudaSuccess && nclusters >= 1;
        }
        if (ok) {
            h->cluster_size = C;
            return C;
        }
        cudaGetLastError();
    }
    return 0;
}

// Which calls run there.  Automatic (kernel choice 0 / 2): where it was measured faster than the launches (profiles/r2n_small.md):
// L = 64 with Philox up to 256 samples (one sample: 1.15 against 2.2 us per half-sweep; 32 samples: 3.6 against 5.2; 64 / 128 / 256
// samples in clusters of 4 CTAs running in waves: 7.3 / 14.5 / 28.9 against 8.4 / 15.6 / 29.9; from 512 samples on the launches fill
// the GPU as well), with MINSTD any number of samples (seed states cached in shared memory, clusters of 8 CTAs
// running in waves: 32 samples 3.8 against 4.0 us, 128 samples 11.3 against 13.7, 512 samples 0.655 against 0.725 ps per flip
// attempt -- no seed table goes through HBM).  On request (choice 4): every case it exists for, L = 128 included.  Short calls stay
// with the launches (the slab is loaded and stored once per call).
// `every`: record spacing of the call in half-sweeps (0: no records).  A recording half-sweep runs the measuring copy of the update
// and costs 0.6 us more than a plain one, so the kernel wins at every spacing (one sample, a record after EVERY half-sweep: 1.75
// against 2.8 us by graph replays with Philox, 2.5 against 2.8 with MINSTD; 32 samples: 3.7 against 5.3 us by launches).
bool cluster_available(ising_t *h, uint32_t nhalf, uint32_t every)
{
    (void)every;
    if (h->kernel_choice == 1 || h->kernel_choice == 3 || h->no_cluster || nhalf < 8) return false;
    if (h->kernel_choice != 4) {
        if (h->g.L != 64) return false;
        if (h->rng_mode == ISING_RNG_PHILOX && h->g.nsamples > 256) return false;
    }
    return cluster_size_of(h) > 0;
}

// records: E / M pre-set by the caller (init_records), record r of sample s at [r * nsamples + s].
int sweep_cluster(ising_t *h, const Thresholds &T, uint32_t nhalf, uint32_t every, long long *d_E, long long *d_M, cudaStream_t st)
{
    const Geometry &g = h->g;
    const bool records = every != 0 && (d_E || d_M);
    const ClusterShape cs = cluster_shape(h, h->cluster_size);
    ClusterArgs p;
    memset(&p, 0, sizeof(p));
    p.A = h->arrays(0);
    p.lattice_stride = 8 * g.array_words;
    p.L = g.L;
    p.T = T;
    p.seed = h->seed;
    p.t0 = h->t;
    p.N = g.N;
    p.nhalf = nhalf;
    p.every = records ? every : 0u;
    p.A_first = h->rng_mode == ISING_RNG_MINSTD ? minstd_power((h->t >> 1) + 1) : 0u;
    p.nsamples = (uint32_t)g.nsamples;
    p.sample0 = 0;
    p.E = records ? d_E : nullptr;
    p.M = records ? d_M : nullptr;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((size_t)g.nsamples * cs.C));
    cfg.blockDim = dim3((unsigned)cs.threads);
    cfg.dynamicSmemBytes = cs.smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cs.C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, cluster_kernel_of(h, records, cs.nw_fixed), p) != cudaSuccess) g_launch_failed = true;
    const int rc = check_launch(h);
    if (rc == ISING_OK) h->t += nhalf;
    return rc;
}

// ---------------------------------------------------------------------------------------------------------------------
// CUDA-graph path (graph_kernels.cuh): K half-sweeps per replay, for lattices whose half-sweep is shorter than a launch.
// ---------------------------------------------------------------------------------------------------------------------
std::mutex g_slot_mutex;
bool g_slot_used[DYN_SLOTS] = {};

void release_graphs(ising_t *h)
{
    for (int i = 0; i < h->ngraphs; ++i) cudaGraphExecDestroy(h->graphs[i].exec);
    h->ngraphs = 0;
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    h->cap_stream = nullptr;
    if (h->dyn_slot >= 0) {
        std::lock_guard<std::mutex> lock(g_slot_mutex);
        g_slot_used[h->dyn_slot] = false;
        h->dyn_slot = -1;
    }
}

// Which calls replay graphs: automatic kernels (choice 0 / 2), one-sample lattices with whole-word rows up to L = 128 (where a
// half-sweep kernel is shorter than a launch: profiles/r2j_launch_floor.md), Philox or MINSTD.
bool graph_geometry(const ising_t *h)
{
    const Geometry &g = h->g;
    if (h->nslabs || (h->kernel_choice != 0 && h->kernel_choice != 2)) return false;
    if (h->rng_mode != ISING_RNG_PHILOX && h->rng_mode != ISING_RNG_MINSTD) return false;
    return g.nsamples == 1 && g.fast && g.L <= 128;
}

bool acquire_slot(ising_t *h)
{
    if (h->dyn_slot >= 0) return true;
    std::lock_guard<std::mutex> lock(g_slot_mutex);
    for (int i = 0; i < DYN_SLOTS; ++i)
        if (!g_slot_used[i]) {
            g_slot_used[i] = true;
            h->dyn_slot = i;
            return true;
        }
    return false;
}

template <int RNG, int W>
void capture_site_step(ising_t *h, bool rec, uint4 *tab0, uint4 *tab1, uint32_t k, uint32_t rec_off)
{
    const Geometry &g = h->g;
    const dim3 grid(g.pgx, g.pgy);
    const LatticeArrays A = h->arrays(0);
    // captured with the programmatic-stream-serialization attribute: the edges between the half-sweeps of the graph become
    // programmatic dependencies, i.e. the next kernel's CTAs start while the previous one drains, as in the stream launches
    if (rec) launch_pdl(half_sweep_site_packed_graph<RNG, W, true>, grid, dim3(SWEEP_THREADS), h->cap_stream, A, g.L, h->seed, tab0, tab1, h->dyn_slot, k, rec_off);
    else launch_pdl(half_sweep_site_packed_graph<RNG, W, false>, grid, dim3(SWEEP_THREADS), h->cap_stream, A, g.L, h->seed, tab0, tab1, h->dyn_slot, k, rec_off);
}
template <int RNG>
void capture_site_step(ising_t *h, bool rec, uint4 *tab0, uint4 *tab1, uint32_t k, uint32_t rec_off)
{
    if (h->g.W == 3) capture_site_step<RNG, 3>(h, rec, tab0, tab1, k, rec_off);
    else if (h->g.W == 5) capture_site_step<RNG, 5>(h, rec, tab0, tab1, k, rec_off);
    else capture_site_step<RNG, 1>(h, rec, tab0, tab1, k, rec_off);
}

// The instantiated graph of K half-sweeps with a record after every `every`-th, built on first use.
cudaGraphExec_t get_graph(ising_t *h, uint32_t K, uint32_t every, bool records)
{
    ++h->graph_clock;
    for (int i = 0; i < h->ngraphs; ++i)
        if (h->graphs[i].K == K && h->graphs[i].records == records && (!records || h->graphs[i].every == every)) {
            h->graphs[i].last_use = h->graph_clock;
            return h->graphs[i].exec;
        }
    if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return nullptr;
    DynConst *slot_addr = nullptr;
    if (cudaGetSymbolAddress((void **)&slot_addr, c_dyn) != cudaSuccess) return nullptr;
    slot_addr += h->dyn_slot;
    const Geometry &g = h->g;
    const bool table = g.nsamples == 1 && h->rng_mode == ISING_RNG_MINSTD && h->kernel_choice != 2 && h->s0tab != nullptr;
    uint4 *tab0 = table ? (uint4 *)h->s0tab : nullptr, *tab1 = table ? (uint4 *)(h->s0tab + g.s0_words / 2) : nullptr;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return nullptr;
    dyn_prepare<<<1, DYN_MAX_SWEEPS, 0, h->cap_stream>>>(h->dyn);
    cudaMemcpyAsync(slot_addr, h->dyn, sizeof(DynConst), cudaMemcpyDeviceToDevice, h->cap_stream);
    uint32_t rec_off = 0;
    for (uint32_t k = 0; k < K; ++k) {
        const bool rec = records && (k + 1) % every == 0;
        if (h->rng_mode == ISING_RNG_PHILOX) capture_site_step<0>(h, rec, tab0, tab1, k, rec_off);
        else if (table) capture_site_step<2>(h, rec, tab0, tab1, k, rec_off);
        else capture_site_step<1>(h, rec, tab0, tab1, k, rec_off);
        if (rec) ++rec_off;
    }
    dyn_advance<<<1, 1, 0, h->cap_stream>>>(h->dyn, K, rec_off);
    const bool launch_failed = g_launch_failed;
    g_launch_failed = false;
    const bool captured = cudaStreamEndCapture(h->cap_stream, &graph) == cudaSuccess && graph != nullptr && !launch_failed;
    cudaGraphExec_t exec = nullptr;
    if (captured && cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) exec = nullptr;
    if (graph) cudaGraphDestroy(graph);
    if (!exec) {
        cudaGetLastError();
        return nullptr;
    }
    int at = h->ngraphs;
    if (at == 8) {   // evict the least recently used
        at = 0;
        for (int i = 1; i < 8; ++i)
            if (h->graphs[i].last_use < h->graphs[at].last_use) at = i;
        cudaGraphExecDestroy(h->graphs[at].exec);
    } else {
        ++h->ngraphs;
    }
    h->graphs[at] = {exec, K, every, records, h->graph_clock};
    return exec;
}

// Replays graphs for as many whole chunks of K half-sweeps as fit into nhalf; returns the number of half-sweeps done (0: none, the
// caller launches them), *nrec = records written.  Records (site-packed only): E / M pre-set by the caller.
int sweep_graphs(ising_t *h, const Thresholds &T, uint32_t nhalf, uint32_t every, long long *d_E, long long *d_M, cudaStream_t st,
                 uint32_t *done, uint32_t *nrec)
{
    *done = 0;
    *nrec = 0;
    const bool records = every != 0 && (d_E || d_M);
    if (!graph_geometry(h)) return ISING_OK;
    uint32_t K;
    if (records) {
        if (every > 64) return ISING_OK;
        const uint32_t cap = nhalf < 64 ? nhalf : 64;
        K = every * (cap / every);
    } else {
        K = nhalf < 64 ? nhalf : 64;
    }
    if (K < 16 || !acquire_slot(h)) return ISING_OK;   // short calls are not worth a graph (building one costs a few hundred launches)
    if (h->rng_mode == ISING_RNG_MINSTD && h->g.nsamples == 1 && h->kernel_choice != 2 && h->s0tab && !h->s0_ready) {
        uint4 *tab[2] = {(uint4 *)h->s0tab, (uint4 *)(h->s0tab + h->g.s0_words / 2)};
        const dim3 grid(h->g.pgx, h->g.pgy);
        for (int cc = 0; cc < 2; ++cc) {
            if (h->g.W == 3) minstd_fill_s0<3><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], h->g.L, cc, h->seed);
            else if (h->g.W == 5) minstd_fill_s0<5><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], h->g.L, cc, h->seed);
            else minstd_fill_s0<1><<<grid, SWEEP_THREADS, 0, st>>>(tab[cc], h->g.L, cc, h->seed);
        }
        const int rc = check_launch(h, 2);
        if (rc != ISING_OK) return rc;
        h->s0_ready = true;
    }
    cudaGraphExec_t exec = get_graph(h, K, every, records);
    if (!exec) return ISING_OK;   // no graph: the caller's launches do the work
    dyn_begin<<<1, 1, 0, st>>>(h->dyn, (unsigned long long)h->t, h->rng_mode == ISING_RNG_MINSTD ? 1u : 0u, records ? d_E : nullptr,
                               records ? d_M : nullptr, T);
    int rc = check_launch(h);
    if (rc != ISING_OK) return rc;
    const uint32_t nrep = nhalf / K;
    for (uint32_t r = 0; r < nrep; ++r)
        if (cudaGraphLaunch(exec, st) != cudaSuccess) {
            cudaGetLastError();
            return ISING_ECUDA;
        }
    h->launches += (uint64_t)nrep * (K + 2);
    h->t += (uint64_t)nrep * K;
    *done = nrep * K;
    *nrec = records ? nrep * (K / every) : 0;
    return ISING_OK;
}

int measure(ising_t *h, long long *d_E, long long *d_M, cudaStream_t st)
{
    const Geometry &g = h->g;
    unsigned long long *slots = h->acc + 4 * (size_t)g.nsamples;
    if (g.batched && h->kernel_choice != 1) {   // every sample in one launch, the counts added to the pre-set E[s], M[s]
        init_records<<<(unsigned)((g.nsamples + 255) / 256), 256, 0, st>>>(d_E, d_M, (uint32_t)g.nsamples, (long long)g.N);
        int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
        const LatticeArrays A = h->arrays(0);
        MeasureArgs m;
        for (int c = 0; c < 2; ++c) {
            m.S[c] = A.S[c];
            for (int d = 0; d < 3; ++d) m.J[d][c] = A.J[d][c];
        }
        m.L = g.L;
        const int tpr_pad = row_map_tpr_pad((g.L >> 6) / g.W);
        for (int s0 = 0; s0 < g.nsamples; s0 += 65535) {
            const int ns = g.nsamples - s0 < 65535 ? g.nsamples - s0 : 65535;
            const dim3 grid((unsigned)(g.L / (32 / tpr_pad)), (unsigned)(g.L / (SWEEP_THREADS / 32)), (unsigned)ns);
            const BatchInfo bi = batch_info(h, (uint32_t)s0);
            if (g.W == 4) launch_pdl(energy_site_packed_batch<4>, grid, dim3(SWEEP_THREADS), st, m, bi, d_E, d_M);
            else if (g.W == 2) launch_pdl(energy_site_packed_batch<2>, grid, dim3(SWEEP_THREADS), st, m, bi, d_E, d_M);
            else if (g.W == 3) launch_pdl(energy_site_packed_batch<3>, grid, dim3(SWEEP_THREADS), st, m, bi, d_E, d_M);
            else if (g.W == 5) launch_pdl(energy_site_packed_batch<5>, grid, dim3(SWEEP_THREADS), st, m, bi, d_E, d_M);
            else launch_pdl(energy_site_packed_batch<1>, grid, dim3(SWEEP_THREADS), st, m, bi, d_E, d_M);
            rc = check_launch(h);
            if (rc != ISING_OK) return rc;
        }
        return ISING_OK;
    }
    if (g.nsamples == 1 && g.fast && h->kernel_choice != 1) {  // one fused launch (measure_kernels.cuh)
        if (!h->slots_clean) {
            if (cudaMemsetAsync(slots, 0, (2 * ACC_SLOTS + 1) * sizeof(unsigned long long), st) != cudaSuccess) return ISING_ECUDA;
            h->slots_clean = true;
        }
        const LatticeArrays A = h->arrays(0);
        MeasureArgs m;
        for (int c = 0; c < 2; ++c) {
            m.S[c] = A.S[c];
            for (int d = 0; d < 3; ++d) m.J[d][c] = A.J[d][c];
        }
        m.L = g.L;
        const int tpr_pad = row_map_tpr_pad((g.L >> 6) / g.W);
        const dim3 grid((unsigned)(g.L / (32 / tpr_pad)), (unsigned)(g.L / (SWEEP_THREADS / 32)));
        if (g.W == 4) launch_pdl(energy_site_packed<4>, grid, dim3(SWEEP_THREADS), st, m, slots, (long long)g.N, d_E, d_M);
        else if (g.W == 3) launch_pdl(energy_site_packed<3>, grid, dim3(SWEEP_THREADS), st, m, slots, (long long)g.N, d_E, d_M);
        else if (g.W == 5) launch_pdl(energy_site_packed<5>, grid, dim3(SWEEP_THREADS), st, m, slots, (long long)g.N, d_E, d_M);
        else launch_pdl(energy_site_packed<1>, grid, dim3(SWEEP_THREADS), st, m, slots, (long long)g.N, d_E, d_M);
        return check_launch(h);
    }
    if (g.nbatches != 0 && g.Hc < (1ull << 31) && h->kernel_choice != 1) {  // bit-sliced column sums, one fused launch
        if (!h->slots_clean) {
            if (cudaMemsetAsync(h->acc, 0, (size_t)g.nsamples * 2 * sizeof(unsigned long long), st) != cudaSuccess ||
                cudaMemsetAsync(slots, 0, (2 * ACC_SLOTS + 1) * sizeof(unsigned long long), st) != cudaSuccess)
                return ISING_ECUDA;
            h->slots_clean = true;
        }
        const LatticeArrays A = h->arrays(0);
        MeasureArgs m;
        for (int c = 0; c < 2; ++c) {
            m.S[c] = A.S[c];
            for (int d = 0; d < 3; ++d) m.J[d][c] = A.J[d][c];
        }
        m.L = g.L;
        // chunk = nblocks x 256 sites per warp: long enough to amortise the 21 plane transposes at its end, short enough for
        // several waves of CTAs (16 blocks = 4096 sites per warp from L = 256 x 32 samples on)
        int nblocks = (int)(g.Hc / (256u * 2048u));
        nblocks = nblocks < 1 ? 1 : nblocks > 16 ? 16 : nblocks;
        static_assert(16 <= EN_MAX_BLOCKS, "counter planes");
        const uint32_t cpc = (uint32_t)((g.Hc + 256u * nblocks - 1) / (256u * nblocks));
        launch_pdl(energy_sample_packed_sliced, dim3((2 * cpc + 7) / 8, (unsigned)g.nbatches), dim3(256), st, m,
                   (size_t)(8 * g.array_words), h->acc, (unsigned int *)(slots + 2 * ACC_SLOTS), (uint32_t)g.Hc, cpc, nblocks,
                   g.nsamples, (long long)g.N, d_E, d_M);
        return check_launch(h);
    }
    h->slots_clean = false;  // the generic kernels below leave their counts in acc
    if (cudaMemsetAsync(h->acc, 0, (size_t)g.nsamples * 2 * sizeof(unsigned long long), st) != cudaSuccess)
        return ISING_ECUDA;
    const int nb = g.nbatches == 0 ? g.nlat : g.nbatches;
    for (int b = 0; b < nb; ++b) {
        const LatticeArrays A = h->arrays(b);
        MeasureArgs m;
        for (int c = 0; c < 2; ++c) {
            m.S[c] = A.S[c];
            for (int d = 0; d < 3; ++d) m.J[d][c] = A.J[d][c];
        }
        m.L = g.L;
        if (g.nbatches != 0) {
            energy_sample_packed<<<(unsigned)((2 * g.Hc + 255) / 256), 256, 0, st>>>(m, h->acc + (size_t)b * 64, g.Hc);
        } else if (h->kernel_choice != 1 && g.Hc < (1ull << 31)) {
            const uint32_t nw = (uint32_t)((g.Hc + 31) / 32);
            const unsigned need = (2 * nw + 255) / 256;
            energy_site_packed_rows<<<need < 148u * 8u ? need : 148u * 8u, 256, 0, st>>>(m, h->acc, nw, (uint32_t)g.Hc);
        } else {   // (a batch of lattices under kernel choice 1: lattice b counts into the pair of sample b)
            const uint64_t nw = (g.Hc + 31) / 32;
            energy_site_packed_generic<<<(unsigned)((2 * nw + 255) / 256), 256, 0, st>>>(m, h->acc + 2 * (size_t)b, nw, g.Hc);
        }
        const int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
    }
    finalize_energy<<<(g.nsamples + 127) / 128, 128, 0, st>>>(h->acc, g.nsamples, (long long)g.N, d_E, d_M);
    return check_launch(h);
}

// ---------------------------------------------------------------------------------------------------------------------
// z-slab handles (slab_kernels.cuh)
// ---------------------------------------------------------------------------------------------------------------------
bool make_slab_geometry(int L, int nslabs, Geometry *g, int *Lz)
{
    if (!make_geometry(L, 1, g) || !g->fast) return false;                    // whole-word rows: L a multiple of 64
    if (nslabs < 1 || L % nslabs != 0 || (L / nslabs) % (SWEEP_THREADS / 32) != 0) return false;   // a CTA row is 8 planes
    *Lz = L / nslabs;
    const size_t plane_words = (size_t)(L >> 6) * L;
    g->array_words = round_up(plane_words * (size_t)(*Lz + 2), ALIGN_WORDS);
    g->arrays_total_words = 8 * g->array_words;
    g->staging_words = ALIGN_WORDS;                                            // no host-buffer path for slabs
    g->s0_words = 2 * (size_t)L * (size_t)*Lz * row_map_tpr_pad((L >> 6) / g->W) * g->W * 32;   // seed table of the slab's own planes
    if (L > MAX_L_32BIT_GROUPS) g->s0_words = 0;                                                 // (recomputed beyond L = 2048, as for the whole lattice)
    g->epoch_words = 0;
    g->onchip = false;
    return true;
}

SplitArgs slab_split_args(const ising_t *h, const uint32_t *d_spins, const uint32_t *d_J)
{
    const LatticeArrays A = h->arrays(0);
    SplitArgs s = {};
    s.narrays = 4;
    s.L = h->g.L;
    s.canon[0] = d_spins;
    s.out[0][0] = A.S[0];
    s.out[0][1] = A.S[1];
    for (int d = 0; d < 3; ++d) {
        s.canon[1 + d] = d_J + (size_t)d * h->g.canon_words;
        s.out[1 + d][0] = A.J[d][0];
        s.out[1 + d][1] = A.J[d][1];
    }
    return s;
}

dim3 slab_grid(const ising_t *h, unsigned rows);

// MINSTD: the seed-state table of the slab's own planes (R11), once per handle.  It is filled by ising_load_state, not by the first
// half-sweep, because the two parts of a half-sweep run on two streams and both read it: everything a handle does is ordered
// after its load anyway.
int slab_fill_seed_table(ising_t *h, cudaStream_t st)
{
    const Geometry &g = h->g;
    if (h->rng_mode != ISING_RNG_MINSTD || !h->s0tab || h->s0_ready) return ISING_OK;
    uint4 *tab[2] = {(uint4 *)h->s0tab, (uint4 *)(h->s0tab + g.s0_words / 2)};
    const dim3 all = slab_grid(h, (unsigned)(h->Lz / (SWEEP_THREADS / 32)));
    for (int cc = 0; cc < 2; ++cc) {
        if (g.W == 4) minstd_fill_s0<4><<<all, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, h->z0);
        else if (g.W == 3) minstd_fill_s0<3><<<all, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, h->z0);
        else if (g.W == 5) minstd_fill_s0<5><<<all, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, h->z0);
        else minstd_fill_s0<1><<<all, SWEEP_THREADS, 0, st>>>(tab[cc], g.L, cc, h->seed, h->z0);
    }
    const int rc = check_launch(h, 2);
    if (rc == ISING_OK) h->s0_ready = true;
    return rc;
}

int slab_load_state(ising_t *h, const uint32_t *d_spins, const uint32_t *d_J, cudaStream_t st)
{
    const uint64_t n = (uint64_t)(h->g.L >> 6) * h->g.L * (h->Lz + 2);
    split_colours_slab<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(slab_split_args(h, d_spins, d_J), h->z0, h->Lz + 2);
    const int rc = check_launch(h);
    return rc == ISING_OK ? slab_fill_seed_table(h, st) : rc;
}

int slab_get_spins(ising_t *h, uint32_t *d_out, cudaStream_t st)
{
    const LatticeArrays A = h->arrays(0);
    const uint64_t n = (uint64_t)(h->g.L >> 6) * h->g.L * h->Lz;
    merge_colours_slab<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(A.S[0], A.S[1], d_out, h->g.L, h->z0, h->Lz);
    return check_launch(h);
}

dim3 slab_grid(const ising_t *h, unsigned rows)
{
    const int tpr_pad = row_map_tpr_pad((h->g.L >> 6) / h->g.W);
    return dim3((unsigned)(h->g.L / (32 / tpr_pad)), rows);
}

int slab_energy(ising_t *h, long long *d_E, long long *d_M, cudaStream_t st)
{
    const Geometry &g = h->g;
    if (cudaMemsetAsync(h->acc, 0, 2 * sizeof(unsigned long long), st) != cudaSuccess) return ISING_ECUDA;
    const LatticeArrays A = h->arrays(0);
    MeasureArgs m;
    for (int c = 0; c < 2; ++c) {
        m.S[c] = A.S[c];
        for (int d = 0; d < 3; ++d) m.J[d][c] = A.J[d][c];
    }
    m.L = g.L;
    const dim3 grid = slab_grid(h, (unsigned)(h->Lz / (SWEEP_THREADS / 32)));
    if (g.W == 4) energy_site_packed_slab<4><<<grid, SWEEP_THREADS, 0, st>>>(m, h->z0, h->acc);
    else if (g.W == 3) energy_site_packed_slab<3><<<grid, SWEEP_THREADS, 0, st>>>(m, h->z0, h->acc);
    else if (g.W == 5) energy_site_packed_slab<5><<<grid, SWEEP_THREADS, 0, st>>>(m, h->z0, h->acc);
    else energy_site_packed_slab<1><<<grid, SWEEP_THREADS, 0, st>>>(m, h->z0, h->acc);
    // the slab's share: E = 2 * unsatisfied - 3 N_slab, M = 2 * up - N_slab; the shares of all slabs add up to the lattice's (R16)
    finalize_energy<<<1, 32, 0, st>>>(h->acc, 1, (long long)g.L * g.L * h->Lz, d_E, d_M);
    return check_launch(h, 2);
}

template <int RNG, int W>
void launch_slab_w(const dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr)
{
    if (RNG == 0 && W >= 3 && a.L > MAX_L_32BIT_GROUPS) {
        constexpr int WB = W >= 3 ? W : 4;
        half_sweep_site_packed_slab<0, WB, true><<<grid, SWEEP_THREADS, 0, st>>>(a, sr);
        return;
    }
    half_sweep_site_packed_slab<RNG, W><<<grid, SWEEP_THREADS, 0, st>>>(a, sr);
}
template <int RNG, int W>
void launch_slab_push_w(const dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr, const SlabPush &p)
{
    if (RNG == 0 && W >= 3 && a.L > MAX_L_32BIT_GROUPS) {
        constexpr int WB = W >= 3 ? W : 4;
        half_sweep_site_packed_slab_push<0, WB, true><<<grid, SWEEP_THREADS, 0, st>>>(a, sr, p);
        return;
    }
    half_sweep_site_packed_slab_push<RNG, W><<<grid, SWEEP_THREADS, 0, st>>>(a, sr, p);
}
template <int RNG>
void launch_slab(int W, const dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr)
{
    if (W == 4) launch_slab_w<RNG, 4>(grid, st, a, sr);
    else if (W == 3) launch_slab_w<RNG, 3>(grid, st, a, sr);
    else if (W == 5) launch_slab_w<RNG, 5>(grid, st, a, sr);
    else launch_slab_w<RNG, 1>(grid, st, a, sr);
}
// the boundary kernel that also stores its end planes into the neighbours' halos (slab_kernels.cuh)
template <int RNG>
void launch_slab_push(int W, const dim3 grid, cudaStream_t st, const SweepArgs &a, const SiteRng &sr, const SlabPush &p)
{
    if (W == 4) launch_slab_push_w<RNG, 4>(grid, st, a, sr, p);
    else if (W == 3) launch_slab_push_w<RNG, 3>(grid, st, a, sr, p);
    else if (W == 5) launch_slab_push_w<RNG, 5>(grid, st, a, sr, p);
    else launch_slab_push_w<RNG, 1>(grid, st, a, sr, p);
}

// part 0: the CTA rows holding the first and the last 8 planes of the slab (the paper's boundary kernel); part 1: the rows in
// between (its bulk kernel).  Neither advances the counter.  A part without rows launches nothing.
// push: the boundary part also stores the slab's end planes into the neighbours' halos (ising_slab_connect), fusing the exchange.
int slab_half_sweep_part(ising_t *h, const Thresholds &T, int part, cudaStream_t st, bool push = false)
{
    const Geometry &g = h->g;
    const int nby = h->Lz / (SWEEP_THREADS / 32);
    const int c = (int)(h->t & 1);
    const LatticeArrays A = h->arrays(0);
    SweepArgs a{};
    a.S_act = A.S[c];
    a.S_oth = A.S[1 - c];
    for (int d = 0; d < 3; ++d) { a.J_act[d] = A.J[d][c]; a.J_oth[d] = A.J[d][1 - c]; }
    a.L = g.L;
    a.colour = c;
    a.T = T;
    a.z0 = h->z0;
    unsigned rows;
    if (part == 0) {
        a.by_first = 0;
        a.by_stride = nby > 1 ? nby - 1 : 0;
        rows = nby > 1 ? 2u : 1u;
    } else {
        if (nby <= 2) return ISING_OK;
        a.by_first = 1;
        a.by_stride = 1;
        rows = (unsigned)(nby - 2);
    }
    RngLaunch r;
    fill_rng_launch(h, 0, &r);
    SiteRng sr = site_rng_of(h, r);
    const dim3 grid = slab_grid(h, rows);
    const bool table = h->rng_mode == ISING_RNG_MINSTD && h->kernel_choice != 2 && h->s0tab != nullptr && h->s0_ready;   // (filled by the loader)
    if (table) sr.s0tab = (uint4 *)(h->s0tab + (c ? g.s0_words / 2 : 0));
    if (push && part == 0) {
        if (!h->push_dn[c] || !h->push_up[c]) return ISING_EINVAL;   // not connected
        SlabPush p;
        p.dn = h->push_dn[c];
        p.up = h->push_up[c];
        p.Lz = h->Lz;
        if (h->rng_mode == ISING_RNG_PHILOX) launch_slab_push<0>(g.W, grid, st, a, sr, p);
        else if (table) launch_slab_push<2>(g.W, grid, st, a, sr, p);
        else launch_slab_push<1>(g.W, grid, st, a, sr, p);
        return check_launch(h);
    }
    if (h->rng_mode == ISING_RNG_PHILOX) launch_slab<0>(g.W, grid, st, a, sr);
    else if (table) launch_slab<2>(g.W, grid, st, a, sr);
    else launch_slab<1>(g.W, grid, st, a, sr);
    return check_launch(h);
}

// which: 0 = first owned plane, 1 = last owned plane, 2 = lower halo, 3 = upper halo
uint32_t *slab_plane_ptr(const ising_t *h, int colour, int which)
{
    const size_t plane_words = (size_t)(h->g.L >> 6) * h->g.L;
    const int zl = which == 0 ? 1 : which == 1 ? h->Lz : which == 2 ? 0 : h->Lz + 1;
    return h->arrays(0).S[colour] + plane_words * (size_t)zl;
}

bool on_own_device(const ising_t *h)
{
    int cur = -1;
    if (h->device < 0 || cudaGetDevice(&cur) != cudaSuccess) {
        cudaGetLastError();
        return true;   // nothing known to compare with; a launch on a machine without a device fails with ISING_ECUDA anyway
    }
    return cur == h->device;
}

}  // namespace

extern "C" {

// Workspace of one geometry: arrays, staging, accumulators, seed table / lane state, tile epochs.
static size_t geometry_bytes(const Geometry &g, int rng_mode)
{
    size_t n = (g.arrays_total_words + g.staging_words) * sizeof(uint32_t) + g.acc_bytes;
    if (rng_mode == ISING_RNG_MINSTD) n += g.s0_words * sizeof(uint32_t);
    n += round_up(g.epoch_words * sizeof(uint32_t), 256);   // tile epochs of the persistent kernels (unused by the lane modes)
    if (lane_mode(rng_mode)) n += round_up((size_t)lane_ring(rng_mode) * lanes_default(g, rng_mode) * sizeof(uint32_t), 256);
    return n;
}

int ising_workspace_bytes(int L, int nsamples, int rng_mode, size_t *out)
{
    Geometry g;
    if (!out || !make_geometry(L, nsamples, &g)) return ISING_EINVAL;
    if (!known_mode(rng_mode)) return ISING_EINVAL;
    if (shared_mode(rng_mode) && nsamples % 32 != 0) return ISING_EINVAL;  // one draw per 32-sample word
    *out = geometry_bytes(g, rng_mode);
    if (batch_layout_possible(L, nsamples, rng_mode)) {   // enough for either layout (ising_create_layout)
        make_geometry(L, nsamples, &g, true);
        const size_t nb = geometry_bytes(g, rng_mode);
        if (nb > *out) *out = nb;
    }
    return ISING_OK;
}

int ising_create(int L, int nsamples, uint64_t seed, int rng_mode, void *d_workspace, size_t workspace_bytes,
                 ising_t **out)
{
    return ising_create_layout(L, nsamples, seed, rng_mode, ISING_LAYOUT_AUTO, d_workspace, workspace_bytes, out);
}

int ising_create_layout(int L, int nsamples, uint64_t seed, int rng_mode, int layout, void *d_workspace, size_t workspace_bytes,
                        ising_t **out)
{
    size_t need = 0;
    if (!out || !d_workspace) return ISING_EINVAL;
    if (layout != ISING_LAYOUT_AUTO && layout != ISING_LAYOUT_SAMPLE_PACKED && layout != ISING_LAYOUT_BATCH) return ISING_EINVAL;
    if (ising_workspace_bytes(L, nsamples, rng_mode, &need) != ISING_OK) return ISING_EINVAL;
    if (workspace_bytes < need || ((uintptr_t)d_workspace & 255u)) return ISING_EINVAL;
    const bool can_batch = batch_layout_possible(L, nsamples, rng_mode);
    if (layout == ISING_LAYOUT_BATCH && !can_batch) return ISING_EINVAL;
    if (layout == ISING_LAYOUT_SAMPLE_PACKED && nsamples == 1) return ISING_EINVAL;
    const bool batched = can_batch && layout != ISING_LAYOUT_SAMPLE_PACKED;
    ising_t *h = new (std::nothrow) ising_t;
    if (!h) return ISING_EINVAL;
    make_geometry(L, nsamples, &h->g, batched);
    h->seed = seed;
    h->rng_mode = rng_mode;
    h->t = 0;
    h->kernel_choice = 0;
    h->launches = 0;
    h->ws = (uint32_t *)d_workspace;
    h->staging = h->ws + h->g.arrays_total_words;
    h->acc = (unsigned long long *)(h->staging + h->g.staging_words);
    h->s0tab = (rng_mode == ISING_RNG_MINSTD && h->g.s0_words) ? (uint32_t *)((char *)h->acc + h->g.acc_bytes) : nullptr;
    h->s0_ready = false;
    h->slots_clean = false;
    h->overlap_clean = false;
    h->lane_state = lane_mode(rng_mode) ? (uint32_t *)((char *)h->acc + h->g.acc_bytes) : nullptr;
    h->nlanes = lane_mode(rng_mode) ? lanes_default(h->g, rng_mode) : 0;
    h->lanes_ready = false;
    h->persist_grid[0] = h->persist_grid[1] = 0;
    h->cluster_size = 0;
    h->no_cluster = false;
    h->nslabs = h->slab = h->z0 = h->Lz = 0;
    h->push_dn[0] = h->push_dn[1] = h->push_up[0] = h->push_up[1] = nullptr;
    h->dyn_slot = -1;
    h->dyn = (DynConst *)((char *)h->acc + h->g.acc_bytes - round_up(sizeof(DynConst), 256));
    h->cap_stream = nullptr;
    h->ngraphs = 0;
    h->graph_clock = 0;
    h->epochs = nullptr;
    if (h->g.epoch_words && !lane_mode(rng_mode)) {   // the last area of the workspace
        h->epochs = (unsigned int *)((char *)d_workspace + need - round_up(h->g.epoch_words * sizeof(uint32_t), 256));
    }
    // the device the workspace belongs to; a workspace of another device than the current one is refused
    h->device = -1;
    {
        int cur = -1;
        cudaPointerAttributes pa;
        if (cudaGetDevice(&cur) == cudaSuccess && cudaPointerGetAttributes(&pa, d_workspace) == cudaSuccess &&
            (pa.type == cudaMemoryTypeDevice || pa.type == cudaMemoryTypeManaged)) {
            if (pa.device != cur) {
                delete h;
                return ISING_EINVAL;
            }
            h->device = pa.device;
        }
        cudaGetLastError();
    }
    *out = h;
    return ISING_OK;
}

int ising_destroy(ising_t *h)
{
    if (h) release_graphs(h);
    delete h;
    return ISING_OK;
}

int ising_load_state(ising_t *h, const uint32_t *d_spins, const uint32_t *d_J, void *stream)
{
    if (!h || !d_spins || !d_J || !on_own_device(h)) return ISING_EINVAL;
    if (h->nslabs) return slab_load_state(h, d_spins, d_J, (cudaStream_t)stream);
    cudaStream_t st = (cudaStream_t)stream;
    const Geometry &g = h->g;
    const size_t W = g.canon_words;
    if (g.nbatches == 0) {
        const LatticeArrays A = h->arrays(0);
        // the padding words of the arrays must not hold garbage (generic kernels read whole words); when L is a multiple of 64
        // the arrays have no padding (L^3/64 words each) and the split kernel writes every word
        if (g.array_words * 32 != g.Hc &&
            cudaMemsetAsync(h->ws, 0, g.arrays_total_words * sizeof(uint32_t), st) != cudaSuccess)
            return ISING_ECUDA;
        if (g.fast) {   // (a batch of lattices: blockIdx.y = sample, at most 65535 per launch)
            for (int s0 = 0; s0 < g.nlat; s0 += 65535) {
                const int ns = g.nlat - s0 < 65535 ? g.nlat - s0 : 65535;
                const LatticeArrays As = h->arrays(s0);
                SplitArgs s = {};
                s.narrays = 4;
                s.L = g.L;
                s.canon[0] = d_spins + (size_t)s0 * W;
                s.canon_stride[0] = W;
                s.out[0][0] = As.S[0];
                s.out[0][1] = As.S[1];
                for (int d = 0; d < 3; ++d) {
                    s.canon[1 + d] = d_J + ((size_t)s0 * 3 + (size_t)d) * W;
                    s.canon_stride[1 + d] = 3 * W;
                    s.out[1 + d][0] = As.J[d][0];
                    s.out[1 + d][1] = As.J[d][1];
                }
                s.out_stride = 8 * g.array_words;
                const uint64_t n = (uint64_t)(g.L >> 6) * g.L * g.L;
                if (g.W == 4) split_colours_site_packed<4><<<dim3((unsigned)((n / 4 + 255) / 256), (unsigned)ns), 256, 0, st>>>(s);
                else split_colours_site_packed<1><<<dim3((unsigned)((n + 255) / 256), (unsigned)ns), 256, 0, st>>>(s);
                const int rc = check_launch(h);
                if (rc != ISING_OK) return rc;
            }
            return ISING_OK;
        }
        const uint64_t nw = (g.Hc + 31) / 32;
        if (h->kernel_choice != 1 && g.Hc < (1ull << 32)) {  // word at a time, all four arrays and both colours in one launch
            SplitArgs s = {};
            s.narrays = 4;
            s.L = g.L;
            s.canon[0] = d_spins;
            s.out[0][0] = A.S[0];
            s.out[0][1] = A.S[1];
            for (int d = 0; d < 3; ++d) {
                s.canon[1 + d] = d_J + (size_t)d * W;
                s.out[1 + d][0] = A.J[d][0];
                s.out[1 + d][1] = A.J[d][1];
            }
            gather_site_packed_rows<<<dim3((unsigned)((nw + 127) / 128), 4), 128, 0, st>>>(s, (uint32_t)nw, (uint32_t)g.Hc, (uint64_t)W);
            return check_launch(h);
        }
        const unsigned grid = (unsigned)((nw + 255) / 256);
        for (int c = 0; c < 2; ++c) {
            gather_site_packed_generic<<<grid, 256, 0, st>>>(d_spins, A.S[c], c, g.L, nw, g.Hc);
            for (int d = 0; d < 3; ++d)
                gather_site_packed_generic<<<grid, 256, 0, st>>>(d_J + (size_t)d * W, A.J[d][c], c, g.L, nw, g.Hc);
        }
        return check_launch(h, 8);
    }
    const unsigned grid = (unsigned)((g.Hc + 255) / 256);
    if (!(g.L % 32 == 0 && h->kernel_choice != 1)) {  // one bit at a time, all batches / arrays / colours per launch (<= 8191 batches each)
        for (int b0 = 0; b0 < g.nbatches; b0 += 8191) {
            const int nbh = g.nbatches - b0 < 8191 ? g.nbatches - b0 : 8191;
            gather_sample_packed_all<<<dim3(grid, (unsigned)(8 * nbh)), 256, 0, st>>>(d_spins, d_J, h->ws, (uint64_t)g.array_words, (uint64_t)W,
                                                                                 g.L, g.Hc, (uint32_t)b0);
            const int rc = check_launch(h);
            if (rc != ISING_OK) return rc;
        }
        return ISING_OK;
    }
    for (int b = 0; b < g.nbatches; ++b) {
        const LatticeArrays A = h->arrays(b);
        const uint32_t *sp = d_spins + (size_t)b * 32 * W;
        const uint32_t *jp = d_J + (size_t)b * 32 * 3 * W;
        GatherTileArgs t;   // tile kernel: one launch per batch, all four arrays, both colours
        t.canon[0] = sp;
        t.stride[0] = W;
        t.out[0][0] = A.S[0];
        t.out[0][1] = A.S[1];
        for (int d = 0; d < 3; ++d) {
            t.canon[1 + d] = jp + (size_t)d * W;
            t.stride[1 + d] = 3 * W;
            t.out[1 + d][0] = A.J[d][0];
            t.out[1 + d][1] = A.J[d][1];
        }
        gather_sample_packed_tiles<<<dim3((unsigned)((W + 127) / 128), 4), 128, 0, st>>>(t, g.L, (uint32_t)W);
        const int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
    }
    return ISING_OK;
}

int ising_get_spins(ising_t *h, uint32_t *d_out, void *stream)
{
    if (!h || !d_out || !on_own_device(h)) return ISING_EINVAL;
    if (h->nslabs) return slab_get_spins(h, d_out, (cudaStream_t)stream);
    cudaStream_t st = (cudaStream_t)stream;
    const Geometry &g = h->g;
    const size_t W = g.canon_words;
    if (g.nbatches == 0) {
        const LatticeArrays A = h->arrays(0);
        if (g.fast) {   // (a batch of lattices: blockIdx.y = sample)
            const uint64_t n = (uint64_t)(g.L >> 6) * g.L * g.L;
            const size_t in_stride = 8 * g.array_words;
            for (int s0 = 0; s0 < g.nlat; s0 += 65535) {
                const int ns = g.nlat - s0 < 65535 ? g.nlat - s0 : 65535;
                const LatticeArrays As = h->arrays(s0);
                uint32_t *out = d_out + (size_t)s0 * W;
                if (g.W == 4) merge_colours_site_packed<4><<<dim3((unsigned)((n / 4 + 255) / 256), (unsigned)ns), 256, 0, st>>>(As.S[0], As.S[1], out, g.L, in_stride, W);
                else merge_colours_site_packed<1><<<dim3((unsigned)((n + 255) / 256), (unsigned)ns), 256, 0, st>>>(As.S[0], As.S[1], out, g.L, in_stride, W);
                if (s0 + ns < g.nlat) {
                    const int rc = check_launch(h);
                    if (rc != ISING_OK) return rc;
                }
            }
        } else if (h->kernel_choice != 1 && g.Hc < (1ull << 32)) {
            scatter_site_packed_rows<<<(unsigned)((W + 127) / 128), 128, 0, st>>>(A.S[0], A.S[1], d_out, g.L, W, g.N);
        } else {
            scatter_site_packed_generic<<<(unsigned)((W + 255) / 256), 256, 0, st>>>(A.S[0], A.S[1], d_out, g.L, W, g.N);
        }
        return check_launch(h);
    }
    for (int b = 0; b < g.nbatches; ++b) {
        const LatticeArrays A = h->arrays(b);
        if (g.L % 32 == 0 && h->kernel_choice != 1) {
            scatter_sample_packed_tiles<<<(unsigned)((W + 127) / 128), 128, 0, st>>>(A.S[0], A.S[1], d_out + (size_t)b * 32 * W, W, g.L,
                                                                                  (uint32_t)W);
            const int rc = check_launch(h);
            if (rc != ISING_OK) return rc;
            continue;
        }
        const int nbh = g.nbatches - b < 65535 ? g.nbatches - b : 65535;   // all remaining batches in one launch (blockIdx.z)
        const dim3 grid((unsigned)((W + 255) / 256), 32, (unsigned)nbh);
        scatter_sample_packed<<<grid, 256, 0, st>>>(A.S[0], A.S[1], d_out + (size_t)b * 32 * W, W, g.L, W, g.N, (uint64_t)(8 * g.array_words));
        b += nbh - 1;
        const int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
    }
    return ISING_OK;
}

int ising_sweep(ising_t *h, double beta, int nsweeps, void *stream)
{
    return ising_sweep_trace(h, beta, nsweeps, nullptr, nullptr, 0, stream);
}

int ising_sweep_trace(ising_t *h, double beta, int nsweeps, int64_t *d_E, int64_t *d_M, int every_half_sweeps, void *stream)
{
    if (!h || nsweeps < 0 || !on_own_device(h)) return ISING_EINVAL;
    if (h->nslabs) return ISING_EINVAL;   // a slab does not sweep on its own: ising_slab_half_sweep_* / ising_slab_sweep_local
    const bool trace = d_E != nullptr || d_M != nullptr;
    if (trace && every_half_sweeps < 1) return ISING_EINVAL;
    uint64_t T[3];
    if (compute_thresholds(beta, h->rng_mode, T) != ISING_OK) return ISING_EINVAL;
    const Thresholds kt = kernel_thresholds(T);
    cudaStream_t st = (cudaStream_t)stream;
    const bool fused = trace && can_measure_in_sweep(h);   // the recording half-sweeps add E and M to the records themselves
    // small lattices whose arrays fit a cluster's shared memory: the whole call in one launch (cluster_kernels.cuh), below
    const bool in_cluster = nsweeps >= 1 && (!trace || fused) && cluster_available(h, 2u * (uint32_t)nsweeps, trace ? (uint32_t)every_half_sweeps : 0u);
    if (!in_cluster && nsweeps >= 1 && persistent_available(h, trace)) {   // all half-sweeps of the call in one launch (persistent.cuh)
        const uint32_t nhalf = 2u * (uint32_t)nsweeps;
        const int rc = sweep_persistent(h, kt, nhalf, trace ? (uint32_t)every_half_sweeps : 0u, (long long *)d_E, (long long *)d_M, st);
        if (rc != ISING_EINVAL) return rc;   // EINVAL (before anything ran): no cooperative launch on this device; use the launches
    }
    size_t rec = 0;
    int k_first = 1;
    if (fused) {   // the records are pre-set to -3N / -N here (add_to_record)
        const uint32_t nrec = (uint32_t)((2 * (size_t)nsweeps) / (size_t)every_half_sweeps);
        if (nrec) {
            const uint32_t n = nrec * (uint32_t)h->g.nsamples;   // (a batch of lattices: one entry per record and sample)
            init_records<<<(n + 255) / 256, 256, 0, st>>>((long long *)d_E, (long long *)d_M, n, (long long)h->g.N);
            const int rc = check_launch(h);
            if (rc != ISING_OK) return rc;
        }
    }
    if (in_cluster)
        return sweep_cluster(h, kt, 2u * (uint32_t)nsweeps, trace ? (uint32_t)every_half_sweeps : 0u, (long long *)d_E, (long long *)d_M, st);
    // whole chunks of half-sweeps replayed from a graph where a half-sweep is shorter than a launch (graph_kernels.cuh) ...
    if (nsweeps >= 1 && (!trace || fused)) {
        uint32_t done = 0, nrec = 0;
        const int rc = sweep_graphs(h, kt, 2u * (uint32_t)nsweeps, trace ? (uint32_t)every_half_sweeps : 0u, (long long *)d_E, (long long *)d_M, st,
                                    &done, &nrec);
        if (rc != ISING_OK) return rc;
        k_first += (int)done;
        rec += nrec;
    }
    // ... the rest (or everything) one launch per half-sweep
    for (int k = k_first; k <= 2 * nsweeps; ++k) {
        const bool record = trace && k % every_half_sweeps == 0;
        long long *rE = record && d_E ? (long long *)d_E + rec * h->g.nsamples : nullptr;
        long long *rM = record && d_M ? (long long *)d_M + rec * h->g.nsamples : nullptr;
        int rc = fused && record ? half_sweep(h, kt, st, rE, rM) : half_sweep(h, kt, st);
        if (rc != ISING_OK) return rc;
        if (record) {
            if (!fused) {
                rc = measure(h, rE, rM, st);
                if (rc != ISING_OK) return rc;
            }
            ++rec;
        }
    }
    return ISING_OK;
}

int ising_energy(ising_t *h, int64_t *d_E, int64_t *d_M, void *stream)
{
    if (!h || !d_E || !on_own_device(h)) return ISING_EINVAL;
    if (h->nslabs) return slab_energy(h, (long long *)d_E, (long long *)d_M, (cudaStream_t)stream);
    return measure(h, (long long *)d_E, (long long *)d_M, (cudaStream_t)stream);
}

int ising_overlap(ising_t *h, int sample_a, int sample_b, int64_t *d_q, void *stream)
{
    if (!h || !d_q || h->g.nsamples == 1 || sample_a < 0 || sample_b < 0 || sample_a >= h->g.nsamples || sample_b >= h->g.nsamples)
        return ISING_EINVAL;
    if (h->g.Hc >= (1ull << 32) || !on_own_device(h)) return ISING_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const Geometry &g = h->g;
    // the counter pair lives behind the ticket of the energy kernels
    unsigned long long *cnt = h->acc + 4 * (size_t)g.nsamples + 2 * ACC_SLOTS + 1;
    if (!h->overlap_clean) {
        if (cudaMemsetAsync(cnt, 0, 2 * sizeof(unsigned long long), st) != cudaSuccess) return ISING_ECUDA;
        h->overlap_clean = true;   // finalize_overlap leaves it zero
    }
    if (g.batched) {   // two site-packed lattices: popcount of the XOR of their spin arrays
        const LatticeArrays A = h->arrays(sample_a), B = h->arrays(sample_b);
        const uint32_t nw = (uint32_t)(g.Hc / 32);
        const unsigned need = (nw + 255) / 256;
        overlap_site_packed<<<need < 148u * 8u ? need : 148u * 8u, 256, 0, st>>>(A.S[0], B.S[0], g.array_words, nw, cnt);
        finalize_overlap<<<1, 1, 0, st>>>(cnt, (long long)g.N, (long long *)d_q);
        return check_launch(h, 2);
    }
    const LatticeArrays A = h->arrays(sample_a >> 5), B = h->arrays(sample_b >> 5);
    const unsigned need = (unsigned)((g.Hc + 255) / 256);
    overlap_sample_packed<<<need < 148u * 8u ? need : 148u * 8u, 256, 0, st>>>(A.S[0], B.S[0], A.S[1], B.S[1], sample_a & 31, sample_b & 31,
                                                                         (uint32_t)g.Hc, cnt);
    finalize_overlap<<<1, 1, 0, st>>>(cnt, (long long)g.N, (long long *)d_q);
    return check_launch(h, 2);
}

int ising_run_host_async(ising_t *h, const uint32_t *h_spins, const uint32_t *h_J, double beta, int nsweeps,
                         uint32_t *h_spins_out, int64_t *h_E, int64_t *h_M, void *stream)
{
    if (!h || !h_spins || !h_J || !h_E || nsweeps < 0 || !(beta >= 0.0) || !on_own_device(h) || h->nslabs) return ISING_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const Geometry &g = h->g;
    const size_t spin_words = (size_t)g.nsamples * g.canon_words, j_words = 3 * spin_words;
    uint32_t *d_spins = h->staging, *d_J = h->staging + spin_words;
    if (cudaMemcpyAsync(d_spins, h_spins, spin_words * sizeof(uint32_t), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d_J, h_J, j_words * sizeof(uint32_t), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return ISING_ECUDA;
    int rc = ising_load_state(h, d_spins, d_J, stream);
    if (rc != ISING_OK) return rc;
    rc = ising_sweep(h, beta, nsweeps, stream);
    if (rc != ISING_OK) return rc;
    long long *d_E = (long long *)(h->acc + 2 * (size_t)g.nsamples), *d_M = d_E + g.nsamples;
    rc = measure(h, d_E, d_M, st);
    if (rc != ISING_OK) return rc;
    if (h_spins_out) {
        rc = ising_get_spins(h, d_spins, stream);
        if (rc != ISING_OK) return rc;
        if (cudaMemcpyAsync(h_spins_out, d_spins, spin_words * sizeof(uint32_t), cudaMemcpyDeviceToHost, st) != cudaSuccess)
            return ISING_ECUDA;
    }
    if (cudaMemcpyAsync(h_E, d_E, (size_t)g.nsamples * sizeof(int64_t), cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return ISING_ECUDA;
    if (h_M && cudaMemcpyAsync(h_M, d_M, (size_t)g.nsamples * sizeof(int64_t), cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return ISING_ECUDA;
    return ISING_OK;
}

int ising_run_host(ising_t *h, const uint32_t *h_spins, const uint32_t *h_J, double beta, int nsweeps, uint32_t *h_spins_out,
                   int64_t *h_E, int64_t *h_M, void *stream)
{
    const int rc = ising_run_host_async(h, h_spins, h_J, beta, nsweeps, h_spins_out, h_E, h_M, stream);
    if (rc != ISING_OK) return rc;
    return cudaStreamSynchronize((cudaStream_t)stream) == cudaSuccess ? ISING_OK : ISING_ECUDA;
}

int ising_thresholds(double beta, int rng_mode, uint64_t out[3])
{
    if (!out) return ISING_EINVAL;
    return compute_thresholds(beta, rng_mode, out);
}

uint64_t ising_fnv1a64_host(const void *h_data, size_t nbytes)
{
    const unsigned char *p = (const unsigned char *)h_data;
    uint64_t hsh = 0xcbf29ce484222325ull;
    for (size_t k = 0; k < nbytes; ++k) {
        hsh ^= (uint64_t)p[k];
        hsh *= 0x100000001b3ull;
    }
    return hsh;
}

int ising_fnv1a64_scratch_bytes(size_t nbytes, size_t *out)
{
    if (!out) return ISING_EINVAL;
    *out = fnv_scratch_bytes(fnv_plan(nbytes));
    return ISING_OK;
}

int ising_fnv1a64(const void *d_data, size_t nbytes, void *d_scratch, size_t scratch_bytes, uint64_t *d_out, void *stream)
{
    if (!d_out || (nbytes && !d_data) || ((uintptr_t)d_data & 3u)) return ISING_EINVAL;
    const FnvPlan p = fnv_plan(nbytes);
    if (nbytes && (!d_scratch || scratch_bytes < fnv_scratch_bytes(p) || ((uintptr_t)d_scratch & 7u))) return ISING_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t *maps = (uint8_t *)d_scratch, *sub_maps = maps + (size_t)p.nchunks * 256, *start = sub_maps + (size_t)p.nchunks * FNV_SUB * 256;
    unsigned long long *sums = (unsigned long long *)(start + ((size_t)p.nchunks + 7) / 8 * 8);
    if (p.nchunks) {
        static std::mutex once;
        static bool smem_set[64] = {};
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return ISING_ECUDA;
        {
            std::lock_guard<std::mutex> lock(once);
            if (!smem_set[dev]) {   // once per device: the maps of all chunks in the shared memory of one CTA
                if (cudaFuncSetAttribute(fnv_chunk_starts, cudaFuncAttributeMaxDynamicSharedMemorySize, FNV_MAX_CHUNKS * 256) != cudaSuccess) return ISING_ECUDA;
                smem_set[dev] = true;
            }
        }
        fnv_low_byte_maps<<<p.nchunks, FNV_SUB * 32, 0, st>>>((const uint8_t *)d_data, p, maps, sub_maps);
        fnv_chunk_starts<<<1, 256, (size_t)p.nchunks * 256, st>>>(maps, p.nchunks, start);
        fnv_chunk_sums<<<p.nchunks, FNV_SUB, 0, st>>>((const uint8_t *)d_data, p, start, sub_maps, sums);
    }
    fnv_combine<<<1, 1024, 0, st>>>(p, sums, (unsigned long long *)d_out);
    return cudaGetLastError() == cudaSuccess ? ISING_OK : ISING_ECUDA;
}

int ising_get_t(const ising_t *h, uint64_t *t)
{
    if (!h || !t) return ISING_EINVAL;
    *t = h->t;
    return ISING_OK;
}

int ising_set_t(ising_t *h, uint64_t t)
{
    if (!h || lane_mode(h->rng_mode)) return ISING_EINVAL;
    h->t = t;
    return ISING_OK;
}

int ising_get_lanes(const ising_t *h, uint32_t *nlanes)
{
    if (!h || !nlanes || !lane_mode(h->rng_mode)) return ISING_EINVAL;
    *nlanes = h->nlanes;
    return ISING_OK;
}

int ising_set_lanes(ising_t *h, uint32_t nlanes)
{
    if (!h || !lane_mode(h->rng_mode) || h->lanes_ready || nlanes < 1 || nlanes > lanes_default(h->g, h->rng_mode)) return ISING_EINVAL;
    h->nlanes = nlanes;
    return ISING_OK;
}

int ising_resume_lanes(ising_t *h, uint64_t t, uint32_t nlanes)
{
    if (!h || !lane_mode(h->rng_mode) || nlanes < 1 || nlanes > lanes_default(h->g, h->rng_mode)) return ISING_EINVAL;
    h->t = t;
    h->nlanes = nlanes;
    h->lanes_ready = true;  // the generator state in the workspace is the checkpoint's
    return ISING_OK;
}

int ising_prng_state_bytes(int kind, uint32_t nlanes, size_t *out)
{
    if (!out || !known_mode(kind) || kind == ISING_RNG_PHILOX_SHARED || nlanes < 1) return ISING_EINVAL;
    const size_t words = kind == ISING_RNG_PHILOX ? 0 : kind == ISING_RNG_MINSTD ? 1 : lane_ring(kind);
    *out = words * nlanes * sizeof(uint32_t);
    return ISING_OK;
}

int ising_prng_init(int kind, uint64_t seed, uint32_t nlanes, void *d_state, void *stream)
{
    size_t bytes;
    if (ising_prng_state_bytes(kind, nlanes, &bytes) != ISING_OK || (bytes && !d_state)) return ISING_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned blocks = (nlanes + 127u) / 128u;
    if (kind == ISING_RNG_MINSTD) minstd_lanes_init<<<blocks, 128, 0, st>>>((uint32_t *)d_state, nlanes, seed);
    else if (kind == ISING_RNG_PR_SHARED) lanes_init<GEN_PR><<<blocks, 128, 0, st>>>((uint32_t *)d_state, nlanes, seed);
    else if (kind == ISING_RNG_MT19937_SHARED) lanes_init<GEN_MT><<<blocks, 128, 0, st>>>((uint32_t *)d_state, nlanes, seed);
    return cudaGetLastError() == cudaSuccess ? ISING_OK : ISING_ECUDA;
}

int ising_prng_count_odd(int kind, uint64_t seed, uint32_t nlanes, uint64_t ndrawn_before, uint64_t ndraws, void *d_state,
                         uint64_t *d_odd, uint64_t *d_sum, void *stream)
{
    size_t bytes;
    if (ising_prng_state_bytes(kind, nlanes, &bytes) != ISING_OK || (bytes && !d_state) || !d_odd || !d_sum) return ISING_EINVAL;
    if ((ndrawn_before & 3u) || (ndraws & 3u)) return ISING_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned blocks = (nlanes + 127u) / 128u;
    unsigned long long *odd = (unsigned long long *)d_odd, *sum = (unsigned long long *)d_sum;
    LaneArgs ln;
    ln.state = (uint32_t *)d_state;
    ln.nlanes = nlanes;
    if (kind == ISING_RNG_PHILOX) {
        count_odd_philox<<<blocks, 128, 0, st>>>(nlanes, seed, ndrawn_before >> 2, ndraws >> 2, odd, sum);
    } else if (kind == ISING_RNG_MINSTD) {
        count_odd_minstd<<<blocks, 128, 0, st>>>((uint32_t *)d_state, nlanes, ndraws, odd, sum);
    } else if (kind == ISING_RNG_PR_SHARED) {
        ln.pos0 = (uint32_t)(ndrawn_before % 62u);
        if (ndraws >= 62) count_odd_lanes<GEN_PR, true><<<blocks, 128, 0, st>>>(ln, ndraws, odd, sum);
        else count_odd_lanes<GEN_PR, false><<<blocks, 128, 0, st>>>(ln, ndraws, odd, sum);
    } else {
        ln.pos0 = (uint32_t)(ndrawn_before % 624u);
        count_odd_lanes<GEN_MT, false><<<blocks, 128, 0, st>>>(ln, ndraws, odd, sum);
    }
    return cudaGetLastError() == cudaSuccess ? ISING_OK : ISING_ECUDA;
}

int ising_slab_workspace_bytes(int L, int nslabs, int rng_mode, size_t *out)
{
    Geometry g;
    int Lz;
    if (!out || !make_slab_geometry(L, nslabs, &g, &Lz)) return ISING_EINVAL;
    if (rng_mode != ISING_RNG_PHILOX && rng_mode != ISING_RNG_MINSTD) return ISING_EINVAL;
    *out = (g.arrays_total_words + g.staging_words) * sizeof(uint32_t) + g.acc_bytes;
    if (rng_mode == ISING_RNG_MINSTD) *out += g.s0_words * sizeof(uint32_t);
    return ISING_OK;
}

int ising_create_slab(int L, int nslabs, int slab, uint64_t seed, int rng_mode, void *d_workspace, size_t workspace_bytes, ising_t **out)
{
    size_t need = 0;
    if (!out || !d_workspace || slab < 0 || slab >= nslabs) return ISING_EINVAL;
    if (ising_slab_workspace_bytes(L, nslabs, rng_mode, &need) != ISING_OK) return ISING_EINVAL;
    if (workspace_bytes < need || ((uintptr_t)d_workspace & 255u)) return ISING_EINVAL;
    // a whole-lattice handle on a small dummy geometry gives every field its default; then the slab geometry replaces it
    ising_t *h = nullptr;
    {
        size_t small = 0;
        if (ising_workspace_bytes(4, 1, rng_mode, &small) != ISING_OK || small > workspace_bytes) return ISING_EINVAL;
        const int rc = ising_create(4, 1, seed, rng_mode, d_workspace, workspace_bytes, &h);
        if (rc != ISING_OK) return rc;
    }
    make_slab_geometry(L, nslabs, &h->g, &h->Lz);
    h->nslabs = nslabs;
    h->slab = slab;
    h->z0 = slab * h->Lz;
    h->staging = h->ws + h->g.arrays_total_words;
    h->acc = (unsigned long long *)(h->staging + h->g.staging_words);
    h->s0tab = rng_mode == ISING_RNG_MINSTD && h->g.s0_words ? (uint32_t *)((char *)h->acc + h->g.acc_bytes) : nullptr;
    h->epochs = nullptr;
    *out = h;
    return ISING_OK;
}

int ising_slab_half_sweep_boundary(ising_t *h, double beta, void *stream)
{
    if (!h || !h->nslabs || !on_own_device(h)) return ISING_EINVAL;
    uint64_t T[3];
    if (compute_thresholds(beta, h->rng_mode, T) != ISING_OK) return ISING_EINVAL;
    return slab_half_sweep_part(h, kernel_thresholds(T), 0, (cudaStream_t)stream);
}

int ising_slab_connect(ising_t *h, void *const d_below_upper_halo[2], void *const d_above_lower_halo[2])
{
    if (!h || !h->nslabs || !d_below_upper_halo || !d_above_lower_halo) return ISING_EINVAL;
    for (int c = 0; c < 2; ++c)
        if (!d_below_upper_halo[c] || !d_above_lower_halo[c] || ((uintptr_t)d_below_upper_halo[c] & 15u) || ((uintptr_t)d_above_lower_halo[c] & 15u))
            return ISING_EINVAL;
    for (int c = 0; c < 2; ++c) {
        h->push_dn[c] = (uint32_t *)d_below_upper_halo[c];
        h->push_up[c] = (uint32_t *)d_above_lower_halo[c];
    }
    return ISING_OK;
}

int ising_slab_half_sweep_boundary_push(ising_t *h, double beta, void *stream)
{
    if (!h || !h->nslabs || !on_own_device(h)) return ISING_EINVAL;
    uint64_t T[3];
    if (compute_thresholds(beta, h->rng_mode, T) != ISING_OK) return ISING_EINVAL;
    return slab_half_sweep_part(h, kernel_thresholds(T), 0, (cudaStream_t)stream, true);
}

int ising_slab_half_sweep_bulk(ising_t *h, double beta, void *stream)
{
    if (!h || !h->nslabs || !on_own_device(h)) return ISING_EINVAL;
    uint64_t T[3];
    if (compute_thresholds(beta, h->rng_mode, T) != ISING_OK) return ISING_EINVAL;
    const int rc = slab_half_sweep_part(h, kernel_thresholds(T), 1, (cudaStream_t)stream);
    if (rc == ISING_OK) h->t += 1;
    return rc;
}

int ising_slab_plane(ising_t *h, int colour, int which, void **d_ptr, size_t *bytes)
{
    if (!h || !h->nslabs || (colour != 0 && colour != 1) || which < 0 || which > 3 || !d_ptr || !bytes) return ISING_EINVAL;
    *d_ptr = slab_plane_ptr(h, colour, which);
    *bytes = (size_t)(h->g.L >> 6) * h->g.L * sizeof(uint32_t);
    return ISING_OK;
}

static int slab_sweep_local(ising_t **slabs, int nslabs, double beta, int nsweeps, void *stream_a, void *stream_b, bool push);

int ising_slab_sweep_local(ising_t **slabs, int nslabs, double beta, int nsweeps, void *stream_a, void *stream_b)
{
    return slab_sweep_local(slabs, nslabs, beta, nsweeps, stream_a, stream_b, false);
}

int ising_slab_sweep_local_push(ising_t **slabs, int nslabs, double beta, int nsweeps, void *stream_a, void *stream_b)
{
    return slab_sweep_local(slabs, nslabs, beta, nsweeps, stream_a, stream_b, true);
}

// push: the boundary kernels store their end planes into the neighbours' halos themselves (the slabs are connected here: all of
// them live on this device), and there are no copies.
static int slab_sweep_local(ising_t **slabs, int nslabs, double beta, int nsweeps, void *stream_a, void *stream_b, bool push)
{
    if (!slabs || nslabs < 1 || nsweeps < 0 || !stream_a || !stream_b || stream_a == stream_b) return ISING_EINVAL;
    for (int s = 0; s < nslabs; ++s)
        if (!slabs[s] || slabs[s]->nslabs != nslabs || slabs[s]->slab != s || slabs[s]->g.L != slabs[0]->g.L ||
            slabs[s]->t != slabs[0]->t || slabs[s]->rng_mode != slabs[0]->rng_mode || slabs[s]->seed != slabs[0]->seed ||
            !on_own_device(slabs[s]))
            return ISING_EINVAL;
    uint64_t T[3];
    if (compute_thresholds(beta, slabs[0]->rng_mode, T) != ISING_OK) return ISING_EINVAL;
    const Thresholds kt = kernel_thresholds(T);
    cudaStream_t sa = (cudaStream_t)stream_a, sb = (cudaStream_t)stream_b;
    if (push)
        for (int s = 0; s < nslabs; ++s) {
            ising_t *below = slabs[(s + nslabs - 1) % nslabs], *above = slabs[(s + 1) % nslabs];
            void *dn[2] = {slab_plane_ptr(below, 0, 3), slab_plane_ptr(below, 1, 3)}, *up[2] = {slab_plane_ptr(above, 0, 2), slab_plane_ptr(above, 1, 2)};
            if (ising_slab_connect(slabs[s], dn, up) != ISING_OK) return ISING_EINVAL;
        }
    cudaEvent_t ea, eb;
    if (cudaEventCreateWithFlags(&ea, cudaEventDisableTiming) != cudaSuccess) return ISING_ECUDA;
    if (cudaEventCreateWithFlags(&eb, cudaEventDisableTiming) != cudaSuccess) { cudaEventDestroy(ea); return ISING_ECUDA; }
    const size_t plane_bytes = (size_t)(slabs[0]->g.L >> 6) * slabs[0]->g.L * sizeof(uint32_t);
    int rc = ISING_OK;
    // stream B first waits for whatever stream A holds on entry (the loader, a previous call)
    if (cudaEventRecord(ea, sa) != cudaSuccess || cudaStreamWaitEvent(sb, ea, 0) != cudaSuccess) rc = ISING_ECUDA;
    for (int k = 0; rc == ISING_OK && k < 2 * nsweeps; ++k) {
        const int c = (int)(slabs[0]->t & 1);
        // boundary kernels of all slabs, then the exchange of the updated colour's end planes: stream A
        for (int s = 0; rc == ISING_OK && s < nslabs; ++s) rc = slab_half_sweep_part(slabs[s], kt, 0, sa, push);
        for (int s = 0; rc == ISING_OK && !push && s < nslabs; ++s) {
            ising_t *below = slabs[(s + nslabs - 1) % nslabs], *above = slabs[(s + 1) % nslabs];
            if (cudaMemcpyAsync(slab_plane_ptr(below, c, 3), slab_plane_ptr(slabs[s], c, 0), plane_bytes, cudaMemcpyDeviceToDevice, sa) != cudaSuccess ||
                cudaMemcpyAsync(slab_plane_ptr(above, c, 2), slab_plane_ptr(slabs[s], c, 1), plane_bytes, cudaMemcpyDeviceToDevice, sa) != cudaSuccess)
                rc = ISING_ECUDA;
        }
        // bulk kernels, concurrently: stream B (they touch neither the end planes nor the halos)
        for (int s = 0; rc == ISING_OK && s < nslabs; ++s) rc = slab_half_sweep_part(slabs[s], kt, 1, sb);
        // the next half-sweep starts when both streams are done with this one
        if (rc == ISING_OK && (cudaEventRecord(ea, sa) != cudaSuccess || cudaEventRecord(eb, sb) != cudaSuccess ||
                               cudaStreamWaitEvent(sb, ea, 0) != cudaSuccess || cudaStreamWaitEvent(sa, eb, 0) != cudaSuccess))
            rc = ISING_ECUDA;
        for (int s = 0; s < nslabs; ++s) slabs[s]->t += 1;
    }
    cudaEventDestroy(ea);
    cudaEventDestroy(eb);
    return rc;
}

// ---- the paper's sliced layout as an alternative internal layout (sliced_kernels.cuh) ----
static bool sliced_ok(const ising_t *h)
{
    if (!h || h->nslabs || h->g.nsamples != 1 || !h->g.fast || h->g.L > MAX_L_32BIT_GROUPS) return false;
    if (h->rng_mode != ISING_RNG_PHILOX && h->rng_mode != ISING_RNG_MINSTD) return false;
    const int wpr = h->g.L >> 5;                     // words per sliced row; lanes per row must be a power of two
    return (wpr & (wpr - 1)) == 0;
}
static SlicedArrays sliced_arrays(const ising_t *h, void *d_scratch)
{
    SlicedArrays B;
    uint32_t *base = (uint32_t *)d_scratch;
    B.S[0] = base;
    B.S[1] = base + h->g.array_words;
    for (int d = 0; d < 3; ++d)
        for (int c = 0; c < 2; ++c) B.J[d][c] = base + (size_t)(2 + 2 * d + c) * h->g.array_words;
    return B;
}

int ising_sliced_scratch_bytes(const ising_t *h, size_t *out)
{
    if (!out || !sliced_ok(h)) return ISING_EINVAL;
    *out = h->g.arrays_total_words * sizeof(uint32_t);
    return ISING_OK;
}

int ising_sliced_begin(ising_t *h, void *d_scratch, void *stream)
{
    if (!sliced_ok(h) || !d_scratch || ((uintptr_t)d_scratch & 255u) || !on_own_device(h)) return ISING_EINVAL;
    const uint32_t words = (uint32_t)(h->g.N >> 6);
    to_sliced_layout<<<(8u * words + 255u) / 256u, 256, 0, (cudaStream_t)stream>>>(h->arrays(0), sliced_arrays(h, d_scratch), h->g.L);
    return check_launch(h);
}

int ising_sliced_sweep(ising_t *h, void *d_scratch, double beta, int nsweeps, void *stream)
{
    if (!sliced_ok(h) || !d_scratch || nsweeps < 0 || !on_own_device(h)) return ISING_EINVAL;
    uint64_t T[3];
    if (compute_thresholds(beta, h->rng_mode, T) != ISING_OK) return ISING_EINVAL;
    const Thresholds kt = kernel_thresholds(T);
    const SlicedArrays B = sliced_arrays(h, d_scratch);
    const int L = h->g.L, wpr = L >> 5, W = wpr >= 8 ? 4 : 1;
    const unsigned grid = (unsigned)(((uint64_t)(L >> 1) * L * (wpr / W)) / 256u);
    for (int k = 0; k < 2 * nsweeps; ++k) {
        RngLaunch r;
        fill_rng_launch(h, 0, &r);
        SiteRng sr;
        sr.pc = r.pc;
        sr.ps = r.ps[0];
        sr.seed = r.seed;
        sr.A2 = 2u * r.A;
        sr.s0tab = nullptr;
        const int c = (int)(h->t & 1);
        if (h->rng_mode == ISING_RNG_PHILOX) {
            if (W == 4) launch_pdl(half_sweep_sliced<0, 4>, dim3(grid), dim3(256), (cudaStream_t)stream, B, sr, L, c, kt);
            else launch_pdl(half_sweep_sliced<0, 1>, dim3(grid), dim3(256), (cudaStream_t)stream, B, sr, L, c, kt);
        } else {
            if (W == 4) launch_pdl(half_sweep_sliced<1, 4>, dim3(grid), dim3(256), (cudaStream_t)stream, B, sr, L, c, kt);
            else launch_pdl(half_sweep_sliced<1, 1>, dim3(grid), dim3(256), (cudaStream_t)stream, B, sr, L, c, kt);
        }
        const int rc = check_launch(h);
        if (rc != ISING_OK) return rc;
        h->t += 1;
    }
    return ISING_OK;
}

int ising_sliced_end(ising_t *h, void *d_scratch, void *stream)
{
    if (!sliced_ok(h) || !d_scratch || !on_own_device(h)) return ISING_EINVAL;
    const uint32_t words = (uint32_t)(h->g.N >> 6);
    from_sliced_layout<<<(2u * words + 255u) / 256u, 256, 0, (cudaStream_t)stream>>>(sliced_arrays(h, d_scratch), h->arrays(0), h->g.L);
    return check_launch(h);
}

int ising_set_kernel(ising_t *h, int which)
{
    if (!h || which < 0 || which > 5) return ISING_EINVAL;
    h->no_cluster = which == 5;               // 5 = 0 without the cluster-resident kernels
    h->kernel_choice = which == 5 ? 0 : which;
    return ISING_OK;
}

uint64_t ising_kernel_launches(const ising_t *h) { return h ? h->launches : 0; }

int ising_hostcheck_update_word(int rng_mode, uint64_t seed, uint64_t t, double beta, const uint32_t ops[13],
                                uint64_t word_index, uint64_t site0, uint64_t site_stride, uint32_t *out)
{
    if (!ops || !out || shared_mode(rng_mode)) return ISING_EINVAL;  // a site-packed word has no shared draw
    uint64_t T[3];
    if (compute_thresholds(beta, rng_mode, T) != ISING_OK) return ISING_EINVAL;
    const Thresholds kt = kernel_thresholds(T);
    uint32_t sum2, sum1, sum0, c4, c8, c12;
    satisfied_bond_count(ops[0], ops + 7, ops + 1, sum2, sum1, sum0);
    if (rng_mode == ISING_RNG_PHILOX) {
        PhiloxCommonConst pc;
        PhiloxSampleConst ps;
        fold_philox(seed, 0, t, &pc, &ps, (uint32_t)((8 * word_index) >> 32));   // counter word c3 = hi32(g), g = 8 x word index + q (R9)
        cond_masks_site_packed_philox(pc, ps, (uint32_t)word_index, kt, c4, c8, c12);
    } else {
        cond_masks_site_packed_minstd(seed + (site0 + 1) * SPLITMIX_GAMMA, site_stride * SPLITMIX_GAMMA,
                                      2u * minstd_power((t >> 1) + 1), kt, c4, c8, c12);
    }
    *out = ops[0] ^ flip_mask(sum2, sum1, sum0, c4, c8, c12);
    return ISING_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// ising_energy_static: E and M of a canonical packed configuration with NO caller workspace and no allocation of any kind
// (include/ising.h).  The scratch -- the eight colour-separated bit arrays the energy kernel reads, and its counter slots -- lives
// in a file-scope device array of fixed size, which every GPU that loads the library holds until the process exits.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int STATIC_MAX_L = ISING_STATIC_MAX_L;
constexpr size_t STATIC_ARRAY_WORDS = (size_t)STATIC_MAX_L * STATIC_MAX_L * STATIC_MAX_L / 64;   // one colour array at the largest L
constexpr size_t STATIC_SLOT_WORDS = 2 * (2 * ACC_SLOTS + 2);                                      // counter pairs + ticket, as uint32 words
constexpr size_t STATIC_SCRATCH_WORDS = 8 * STATIC_ARRAY_WORDS + STATIC_SLOT_WORDS;                // 1 MiB + 1040 B at L = 128

// In host code this name is a host-side stand-in, not a device address: the kernels get the address cudaGetSymbolAddress returns.
static __device__ __align__(256) uint32_t g_static_scratch[STATIC_SCRATCH_WORDS];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
uint32_t *g_static_ptr[STATIC_MAX_DEVICES] = {};   // device address of g_static_scratch on each device, looked up once per device

// The scratch of the CURRENT device (nullptr: no device / lookup failed).  Every device has its own copy of a __device__ variable,
// so the address is taken once per device, with that device current.
uint32_t *static_scratch_of_current_device()
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= STATIC_MAX_DEVICES) {
        cudaGetLastError();
        return nullptr;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) {
            cudaGetLastError();
            return nullptr;
        }
        g_static_ptr[dev] = (uint32_t *)p;
    }
    return g_static_ptr[dev];
}

}  // namespace

int ising_energy_static(int L, const uint32_t *d_spins, const uint32_t *d_J, int64_t *d_E, int64_t *d_M, void *stream)
{
    if (!d_spins || !d_J || !d_E || L < 64 || L % 64 != 0) return ISING_EINVAL;
    if (L > STATIC_MAX_L) return ISING_ELIMIT;
    uint32_t *scratch = static_scratch_of_current_device();
    if (!scratch) return ISING_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t aw = (size_t)L * L * L / 64;   // words of one colour array (no padding when L is a multiple of 64)
    const size_t W = (size_t)L * L * L / 32;    // canonical words per bit array
    unsigned long long *slots = (unsigned long long *)(scratch + 8 * STATIC_ARRAY_WORDS);
    // the array keeps the last call's contents: the counters and the ticket must start at zero (the arrays are overwritten whole)
    if (cudaMemsetAsync(slots, 0, STATIC_SLOT_WORDS * sizeof(uint32_t), st) != cudaSuccess) return ISING_ECUDA;
    SplitArgs s = {};
    MeasureArgs m;
    s.narrays = 4;
    s.L = L;
    m.L = L;
    for (int q = 0; q < 4; ++q) {       // q = 0: spins, 1 + d: couplings of direction d
        s.canon[q] = q == 0 ? d_spins : d_J + (size_t)(q - 1) * W;
        for (int c = 0; c < 2; ++c) {
            s.out[q][c] = scratch + (size_t)(2 * q + c) * aw;
            if (q == 0) m.S[c] = s.out[q][c];
            else m.J[q - 1][c] = s.out[q][c];
        }
    }
    // words per thread as make_geometry chooses them for L <= 128: one
    const uint64_t n = (uint64_t)(L >> 6) * L * L;
    split_colours_site_packed<1><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(s);
    const int tpr_pad = row_map_tpr_pad(L >> 6);
    const dim3 grid((unsigned)(L / (32 / tpr_pad)), (unsigned)(L / (SWEEP_THREADS / 32)));
    energy_site_packed<1><<<grid, SWEEP_THREADS, 0, st>>>(m, slots, (long long)L * L * L, (long long *)d_E, (long long *)d_M);
    return cudaGetLastError() == cudaSuccess ? ISING_OK : ISING_ECUDA;
}

const char *ising_strerror(int code)
{
    switch (code) {
        case ISING_OK: return "ok";
        case ISING_EINVAL: return "invalid argument";
        case ISING_ECUDA: return "CUDA error";
        case ISING_ELIMIT: return "size beyond the fixed scratch of ising_energy_static (L <= ISING_STATIC_MAX_L)";
        default: return "unknown error";
    }
}

}  // extern "C"
