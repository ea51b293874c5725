/*
 * ising.h -- C ABI of libising_b200: the bit-packed checkerboard (red/blue) Metropolis sweep of the
 * 3D +-J Edwards-Anderson spin glass on one NVIDIA B200 (sm_100a).
 *
 * Method: arXiv 1411.0127 (Lulli, Bernaschi, Parisi).  Citations are PAPER.md:<line> of the paper text
 * plus the section / equation; "R<n>" are the readings listed in DESIGN.md section 2.
 *
 *   H = - sum_<ik> J_ik sigma_i sigma_k   on an L^3 periodic cubic lattice, J = +-1        (Eq. 1-2)
 *   one sweep = Metropolis update (Eq. 9) of all red sites ((x+y+z) even), then of all blue
 *   sites; spins and couplings are one bit each (Eq. 10); the energy
 *   change of a flip is computed word-wise from bond bits (Eq. 11) with a bit-sliced adder (Eq. 12-13)
 *   and turned into a flip mask (Eq. 14-17).  Every (sample, site, half-sweep) has its
 *   own 32-bit draw (R9-R12); the paper's one draw per 32-sample word is the separate
 *   mode ISING_RNG_PHILOX_SHARED (R18).
 *
 * Conventions
 *   N = L^3, site i = x + L*(y + L*z), colour (x+y+z)&1, red = 0 is updated at even half-sweep index t (R8).
 *   Sizes: every even L from 4 to 2048 (all layouts and modes); one-sample lattices also L = 2560, 3072 and 4096, where the
 *   Philox group index passes 2^32 (at L = 4096) and its high word enters the counter (R9), the MINSTD seed states are recomputed instead of
 *   cached, and the workspace is 15.6, 27 and 64 GiB (L = 4096: 32 GiB of bit arrays + 32 GiB of canonical staging).
 *   The half-sweep counter t starts at 0 in ising_create and keeps counting over all sweep calls, so a
 *   trajectory does not depend on how sweeps are batched into calls.
 *   Canonical packed format (the only format that crosses this boundary):
 *     spins      nsamples x W uint32, W = ceil(N/32); bit (i&31) of word (i>>5) is site i; 1 <=> sigma=+1
 *     couplings  nsamples x 3 x W uint32, [sample][dir x,y,z][word]; the bit of site i in direction d is the
 *                bond (i, i+d-hat); 1 <=> J=-1                                              (Eq. 10)
 *     bits above N in the last word are ignored on input and zero on output.
 *   nsamples = 1 uses a site-packed internal layout (bits of a word = 32 sites of one lattice, "SMSC",
 *   PAPER.md:227); nsamples = 32*k uses a sample-packed layout (bits of a word = 32 disorder samples at
 *   one site, "AMSC" storage, with k coded batches) or, where every sample draws
 *   its own random numbers and L is a multiple of 64, a batch of nsamples site-packed lattices (ising_create_layout).
 *
 * Devices: a handle belongs to the CUDA device its workspace lives on.  ising_create refuses a workspace of another
 *   device than the current one, and every call that launches work returns ISING_EINVAL when made with a different
 *   device current (cudaSetDevice): the kernels would otherwise dereference another GPU's memory.  All d_* buffers of
 *   a call must live on the handle's device.
 *
 * Pointers: every pointer named d_* is DEVICE memory owned by the caller (e.g. a torch CUDA tensor), every
 *   h_* pointer is HOST memory owned by the caller.  The handle owns host metadata only; the workspace
 *   passed to ising_create must stay alive, and must not be written by the caller, until ising_destroy.
 *   `stream` is a cudaStream_t passed as void* (0 = the legacy default stream).  Calls taking a stream are
 *   asynchronous on it unless stated otherwise.
 *
 * Errors: every int-returning call returns ISING_OK (0) or a negative code; nothing throws or aborts.
 *   There is no CPU fallback: without a CUDA device the device calls return ISING_ECUDA.
 */
#ifndef ISING_B200_H
#define ISING_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ISING_OK 0
#define ISING_EINVAL (-1) /* bad argument: L odd or < 4 or > 4096 (beyond 2048: one sample and L = 2560, 3072 or 4096 only), nsamples not 1 or a multiple of 32, unknown
                             rng_mode, a mode that does not support (L, nsamples), null pointer, workspace too small /
                             misaligned, beta < 0 or NaN, nsweeps < 0 */
#define ISING_ECUDA (-2)  /* a CUDA runtime call or kernel launch failed (sticky errors surface here too) */
#define ISING_ELIMIT (-3) /* ising_energy_static only: L beyond ISING_STATIC_MAX_L, the size its fixed scratch is built for */

#define ISING_RNG_PHILOX 0 /* Philox4x32-10, key (lo32 seed, hi32 seed ^ sample), counter (t, colour-rank>>2)  (R9, R10).
                              Because the sample index is XORed into the high key word, (seed, sample) and
                              (seed ^ (x << 32), sample ^ x) name the same stream: runs that must be independent need
                              seeds that differ in their LOW 32 bits (the same holds for the batch index in mode 2). */
#define ISING_RNG_MINSTD 1 /* MINSTD 16807 mod 2^31-1 (Eq. 7), one stream per site seeded by
                              SplitMix64 (R11), draw of sweep n = 16807^(n+1) * s0 mod (2^31-1) (R12) */

#define ISING_RNG_PHILOX_SHARED 2 /* the paper's asynchronous multispin coding proper (Eq. 15): the 32
                              samples of a word share ONE Philox draw per (site, half-sweep); nsamples = 32k only; the draw
                              of the samples 32b..32b+31 is the ISING_RNG_PHILOX draw with the key's sample field = b (R18) */

/* The same shared draw, taken from generators with STORED state, one per lane -- the paper's own scheme of one generator
 * per thread with a strided state array (R19).  nsamples = 32k only.
 *   The N/2 sites of a colour are numbered by their colour rank j and taken in groups of four, g = j >> 2 (N/8 groups); with k
 *   coded batches there are k N/8 units u = b * (N/8) + g.  Lane q serves the units q, q + nlanes, q + 2 nlanes, ... in that order,
 *   for each the four sites w = 0..3 of its group; the next number of the lane is the draw of (batch b, site 4g + w).  Every lane
 *   takes 4 ceil(k (N/8) / nlanes) draws per half-sweep (a lane whose last unit does not exist draws and discards).  Thresholds as
 *   for Philox (R5).  nlanes defaults to min(k N/8, 151552 = one wave of threads) (ising_get_lanes / ising_set_lanes); the state
 *   lives in the workspace. */
#define ISING_RNG_PR_SHARED 3      /* Parisi-Rapuano: ira[i] = ira[i-24] + ira[i-55]; R = ira[i] ^ ira[i-61];
                              seed words ira[0..61] of lane q = high words of SplitMix64 outputs q*62 + 1 .. q*62 + 62 of `seed` */
#define ISING_RNG_MT19937_SHARED 4 /* MT19937, lane q seeded by init_genrand(high word of SplitMix64 output q + 1) */

typedef struct ising ising_t; /* opaque */

/* Size in bytes of the device workspace ising_create needs for (L, nsamples, rng_mode): the internal spin and
 * coupling arrays (8 bit arrays per lattice), a canonical staging area used by
 * ising_run_host, the int64 accumulators of the measurement kernel and, in MINSTD mode with nsamples = 1 and
 * L a multiple of 64, a table of the per-site seed states s0 (4 bytes per site, R11).  In modes 0-2 no PRNG *state* is stored:
 * both generators are evaluated statelessly from (seed, sample, site, t) (R9, R12); the table only caches the
 * time-independent SplitMix64 seeding of the MINSTD streams and is filled by the first sweep call.  The lane modes 3, 4 add
 * the strided generator state (62 or 624 words per lane, R19), seeded by the first sweep call. */
int ising_workspace_bytes(int L, int nsamples, int rng_mode, size_t *out);

/* Create a handle.  d_workspace: device memory, >= ising_workspace_bytes, 256-byte aligned.  The lattice
 * content is undefined until ising_load_state.  seed keys the dynamics' random numbers (R9, R11). */
int ising_create(int L, int nsamples, uint64_t seed, int rng_mode, void *d_workspace, size_t workspace_bytes,
                 ising_t **out);

/* The same with the internal layout of a many-sample handle chosen by the caller (ising_create = ISING_LAYOUT_AUTO).
 *   ISING_LAYOUT_SAMPLE_PACKED  bits of a word = 32 samples at one site, the paper's AMSC storage; nsamples = 32k.
 *   ISING_LAYOUT_BATCH          nsamples site-packed lattices one after the other (bits of a word = 32 sites of one sample, the
 *                               paper's SMSC coding, for every sample), all samples in every launch.  Only where the
 *                               samples draw their own numbers (rng modes 0, 1) and L is a multiple of 64: there sample s IS the
 *                               one-sample lattice with the Philox key word k1 ^ s (R9) / the MINSTD streams s N .. s N + N - 1
 *                               (R11), the sample-packed storage has no shared draw to amortise, and this layout is the faster one
 *                               (DESIGN.md section 6).  ISING_EINVAL elsewhere.
 *   ISING_LAYOUT_AUTO           ISING_LAYOUT_BATCH where it is allowed, else sample-packed (nsamples = 1: site-packed).
 * The layout changes no result and nothing at this boundary: the canonical format is per sample in either case, and
 * ising_workspace_bytes is enough for both. */
#define ISING_LAYOUT_AUTO 0
#define ISING_LAYOUT_SAMPLE_PACKED 1
#define ISING_LAYOUT_BATCH 2
int ising_create_layout(int L, int nsamples, uint64_t seed, int rng_mode, int layout, void *d_workspace, size_t workspace_bytes,
                        ising_t **out);

/* Load spins and couplings given in the canonical packed format (device pointers) into the internal
 * layout.  Does not change the half-sweep counter. */
int ising_load_state(ising_t *h, const uint32_t *d_spins, const uint32_t *d_J, void *stream);

/* nsweeps full sweeps at inverse temperature beta = 2*nsweeps colour half-sweeps, red first (rows a1-a8):
 * threshold table T[dE] = floor(2^32 exp(-beta dE)) (Philox, R5) or floor((2^31-1) exp(-beta dE)) (MINSTD,
 * R6) for dE = 4, 8, 12, then per half-sweep the bond bits / adder / flip mask of Eq. 11-17
 * with acceptance R < T[dE] (strict, R4) applied per bit.  Advances t by 2*nsweeps. */
int ising_sweep(ising_t *h, double beta, int nsweeps, void *stream);

/* As ising_sweep, and after every `every_half_sweeps`-th half-sweep of this call (counted from 1) writes the
 * energy (and magnetisation if d_M != NULL) of every sample to record r = 0,1,...:
 * d_E[r*nsamples + s].  d_E / d_M must hold (2*nsweeps / every_half_sweeps) * nsamples int64.  (With nsamples = 1 and L >= 64
 * the recording half-sweeps compute E and M themselves, from the field sums they already hold; otherwise a record is one
 * launch of the energy kernel.) */
int ising_sweep_trace(ising_t *h, double beta, int nsweeps, int64_t *d_E, int64_t *d_M, int every_half_sweeps,
                      void *stream);

/* E[s] = - sum over the 3N bonds of J sigma sigma (Eq. 1, each bond once; R16) and M[s] = sum_i sigma_i for
 * every sample (row a9).  d_E: nsamples int64; d_M: nsamples int64 or NULL. */
int ising_energy(ising_t *h, int64_t *d_E, int64_t *d_M, void *stream);

/* The same E and M (row a9; Eq. 1, R16) for ONE sample given in the canonical packed format, for callers that cannot allocate: no
 * handle, no workspace, and the library calls no cudaMalloc / cudaFree / allocating routine on this path (code under CUDA graph
 * capture, serving loops, harnesses that forbid allocation).  d_spins: L^3/32 uint32, d_J: 3 x L^3/32 uint32 (device, read only);
 * d_E: one int64; d_M: one int64 or NULL (device, written); asynchronous on `stream`, on the CURRENT device.
 *   The scratch the kernels need -- the eight colour-separated bit arrays (row a10) and the counter slots of the energy kernel --
 * is a fixed array in the library's device image: 8 x ISING_STATIC_MAX_L^3 / 16 bytes + 1040 = 1 MiB + 1 KiB, held by every GPU
 * that loads the library until the process exits.  Hence the limits: L a multiple of 64 (else ISING_EINVAL) and
 * L <= ISING_STATIC_MAX_L (else ISING_ELIMIT: use a handle).  ALL calls on a device share that array: calls that overlap on the
 * GPU (two streams, two host threads) race and give wrong results; calls on one stream are safe, each one clears the counters it
 * needs zeroed and overwrites the arrays whole, so nothing of an earlier call is seen. */
#define ISING_STATIC_MAX_L 128
int ising_energy_static(int L, const uint32_t *d_spins, const uint32_t *d_J, int64_t *d_E, int64_t *d_M, void *stream);

/* Overlap of two samples of one handle, q = sum_i sigma_i^a sigma_i^b in [-N, N] (one int64 at d_q): the spin-glass order
 * parameter when the two samples are replicas, i.e. were loaded with the same couplings.  nsamples = 32k only. */
int ising_overlap(ising_t *h, int sample_a, int sample_b, int64_t *d_q, void *stream);

/* Write the spins in the canonical packed format: nsamples x W uint32 (row a10). */
int ising_get_spins(ising_t *h, uint32_t *d_out, void *stream);

/* The whole path on HOST buffers, for end-to-end timing: copies h_spins / h_J (canonical packed, ideally
 * pinned) to the staging area of the workspace, loads them, runs nsweeps sweeps, computes E and M, copies
 * the canonical spins back to h_spins_out (may be NULL) and E / M to h_E / h_M (nsamples int64 each; h_M
 * may be NULL), and synchronises the stream before returning. */
int ising_run_host(ising_t *h, const uint32_t *h_spins, const uint32_t *h_J, double beta, int nsweeps,
                   uint32_t *h_spins_out, int64_t *h_E, int64_t *h_M, void *stream);

/* The same job enqueued on `stream` without the final synchronisation: returns as soon as the copies and launches are queued.
 * All host buffers must be pinned (cudaHostAlloc / torch pin_memory; with pageable memory the copies are staged by the driver
 * and the call is no longer asynchronous) and must stay valid and untouched until the caller has synchronised the stream;
 * h_spins_out / h_E / h_M hold the results only after that.  Meant for double buffering: two handles (two workspaces) on two
 * streams, so that the PCIe copies of one job run under the sweeps of the other (bench.py's `e2e`).  One handle must not have two
 * jobs in flight on different streams: its staging area and lattice arrays are reused by every call. */
int ising_run_host_async(ising_t *h, const uint32_t *h_spins, const uint32_t *h_J, double beta, int nsweeps,
                         uint32_t *h_spins_out, int64_t *h_E, int64_t *h_M, void *stream);

/* Host only.  The acceptance thresholds for dE = 4, 8, 12 exactly as the kernels receive them (R5, R6):
 * out[k] in [0, 2^32] (Philox) or [0, 2^31-1] (MINSTD). */
int ising_thresholds(double beta, int rng_mode, uint64_t out[3]);

/* Host only.  64-bit FNV-1a (offset basis 0xcbf29ce484222325, prime 0x100000001b3) of nbytes bytes: the
 * checksum of BASELINE.json config 4 over the canonical packed spin words (little-endian bytes). */
uint64_t ising_fnv1a64_host(const void *h_data, size_t nbytes);

/* The same checksum of `nbytes` bytes of DEVICE memory (4-byte aligned), computed on the device in parallel and written to *d_out
 * (device, one uint64), asynchronously on `stream`: the value is the one the byte-by-byte definition gives, bit for bit.  (The XOR of
 * FNV-1a touches the low byte only, h ^ b = h + d with d from the low byte, and the low byte follows an 8-bit recurrence of its own;
 * so the hash of a chunk is h_start P^n + sum_i d_i P^(n-i), and chunks are processed in parallel once the low byte at each
 * chunk's start is known: csrc/fnv_kernels.cuh.  16 MiB take 0.2 ms instead of 17 ms on a host core.)  d_scratch: device memory of
 * ising_fnv1a64_scratch_bytes(nbytes) bytes (7.6 MB at most), 8-byte aligned, owned by the caller, overwritten. */
int ising_fnv1a64_scratch_bytes(size_t nbytes, size_t *out);
int ising_fnv1a64(const void *d_data, size_t nbytes, void *d_scratch, size_t scratch_bytes, uint64_t *d_out, void *stream);

/* Half-sweep counter t of the handle (get / set): with ising_get_spins + ising_load_state this makes a run
 * resumable bit-exactly, because no PRNG state exists outside (seed, t). */
int ising_get_t(const ising_t *h, uint64_t *t);
int ising_set_t(ising_t *h, uint64_t t); /* ISING_EINVAL in the lane modes 3, 4: their generator state is not a function of t */

/* Lane modes (3, 4) only.  Number of generator lanes; ising_set_lanes is allowed before the first sweep only, with
 * 1 <= nlanes <= the default (the workspace is sized for the default).  Other modes: ISING_EINVAL. */
int ising_get_lanes(const ising_t *h, uint32_t *nlanes);
int ising_set_lanes(ising_t *h, uint32_t nlanes);

/* Lane modes only: resume from a checkpoint.  The whole run state is (the workspace bytes, t, nlanes): save a copy of the
 * workspace with ising_get_t and ising_get_lanes; to resume, create a handle on a workspace holding those bytes and call
 * ising_resume_lanes(h, t, nlanes), which sets the half-sweep counter and keeps the generator state found in the workspace
 * instead of seeding it.  (In the other modes ising_get_spins + ising_load_state + ising_set_t do the same.) */
int ising_resume_lanes(ising_t *h, uint64_t t, uint32_t nlanes);

/* The paper's device-API generator benchmark (Table II): every lane draws numbers and counts the odd ones.
 * kind: ISING_RNG_PHILOX (no state; key (lo32 seed, hi32 seed), counter (lo32 c, hi32 c, lane, 0), c = draw number >> 2, output
 * word = draw number & 3), ISING_RNG_MINSTD (one word per lane, the seed state of stream `lane`, R11, advanced once per draw),
 * ISING_RNG_PR_SHARED, ISING_RNG_MT19937_SHARED (62 / 624 words per lane, strided: word r of lane q at d_state[r*nlanes + q],
 * seeded as above).
 *   ising_prng_state_bytes  bytes of d_state for (kind, nlanes); 0 for Philox.
 *   ising_prng_init         seeds the state of every lane.
 *   ising_prng_count_odd    every lane takes draws number ndrawn_before .. ndrawn_before + ndraws - 1 of its sequence (both
 *                           multiples of 4; the caller keeps count) and writes d_odd[lane] = how many were odd and d_sum[lane] =
 *                           their sum mod 2^64 (nlanes uint64 each, overwritten). */
int ising_prng_state_bytes(int kind, uint32_t nlanes, size_t *out);
int ising_prng_init(int kind, uint64_t seed, uint32_t nlanes, void *d_state, void *stream);
int ising_prng_count_odd(int kind, uint64_t seed, uint32_t nlanes, uint64_t ndrawn_before, uint64_t ndraws, void *d_state,
                         uint64_t *d_odd, uint64_t *d_sum, void *stream);

/* ---- z-slab domain decomposition (section V; Fig. 10) --------------------
 * The lattice is cut along z into `nslabs` slabs of Lz = L / nslabs planes, one handle -- one GPU, in a multi-GPU run -- per slab;
 * slab r owns the planes r Lz .. (r + 1) Lz - 1.  nsamples = 1, L a multiple of 64, Lz a multiple of 8, rng modes 0 and 1.
 * A slab stores its own planes plus one halo plane below and above (copies of the neighbouring slabs' end planes, periodic), and
 * a colour half-sweep of the lattice is, for every slab: the BOUNDARY kernel (the rows of CTAs that hold the first and last 8
 * planes), then the exchange -- the updated colour's first owned plane goes to the upper halo of the slab below, its last owned
 * plane to the lower halo of the slab above, L^2/16 bytes each (64 KiB at L = 1024), in both directions for each colour because
 * in the standard checkerboard every plane holds both colours -- while the BULK kernel updates all other planes on
 * a second stream (the paper's boundary / bulk overlap).  The library does the kernels; the exchange is the caller's (a peer
 * cudaMemcpyAsync, NCCL send / recv, ...) between the buffers ising_slab_plane names, except for ising_slab_sweep_local, which
 * drives all slabs of one process on one device itself.  Every draw is keyed by the site's position in the whole lattice (R9,
 * R11), so the slabs together follow exactly the trajectory of the undivided lattice.
 *
 * On a slab handle: ising_load_state / ising_get_spins take the canonical arrays of the WHOLE lattice (the slab reads its planes
 * and halos / writes its planes only); ising_energy gives the slab's share, E_r = 2 (unsatisfied +x,+y,+z bonds of its sites)
 * - 3 L^2 Lz and M_r likewise, and sum_r E_r = E, sum_r M_r = M; ising_get_t / ising_set_t as usual; ising_sweep,
 * ising_sweep_trace, ising_run_host* return ISING_EINVAL (a slab cannot sweep without its neighbours). */
int ising_slab_workspace_bytes(int L, int nslabs, int rng_mode, size_t *out);
int ising_create_slab(int L, int nslabs, int slab, uint64_t seed, int rng_mode, void *d_workspace, size_t workspace_bytes,
                      ising_t **out);
/* The two parts of the colour half-sweep t & 1 (thresholds as in ising_sweep).  The boundary part must see the halos of the
 * previous half-sweep's exchange; the bulk part may run concurrently with the boundary part and the exchange on another stream,
 * and advances t by one.  The next half-sweep needs both parts and the exchange complete, on this slab and its two neighbours. */
int ising_slab_half_sweep_boundary(ising_t *h, double beta, void *stream);
int ising_slab_half_sweep_bulk(ising_t *h, double beta, void *stream);
/* Where the planes of the exchange live: *d_ptr = device address, *bytes = L^2/16.  which: 0 = first owned plane, 1 = last owned
 * plane (to send down / up after a half-sweep of `colour`), 2 = lower halo, 3 = upper halo (to receive the plane 1 of the slab
 * below / the plane 0 of the slab above). */
int ising_slab_plane(ising_t *h, int colour, int which, void **d_ptr, size_t *bytes);
/* The exchange fused into the boundary kernel.  ising_slab_connect tells a slab where its neighbours' halos are: for each colour c,
 * d_below_upper_halo[c] = plane 3 (upper halo) of colour c of the slab BELOW, d_above_lower_halo[c] = plane 2 (lower halo) of the
 * slab ABOVE, as ising_slab_plane of those handles names them -- device addresses valid on THIS slab's device: the same GPU, or a
 * peer GPU's memory mapped into this process (cudaDeviceEnablePeerAccess, or cudaIpcOpenMemHandle of the neighbour process's
 * workspace); 16-byte aligned; the handle keeps the pointers, not the memory.  ising_slab_half_sweep_boundary_push is the boundary
 * part whose threads store the updated words of the first / last owned plane a second time, into those halos: over NVLink the
 * planes travel while the kernel runs, and no copy is launched.  Ordering is as for the copies: the next half-sweep may start on a
 * slab only when this kernel has completed on the slab itself AND on its two neighbours (an event per half-sweep between the
 * devices' streams; a kernel's peer stores are visible when it has completed).  ISING_EINVAL if the slab is not connected. */
int ising_slab_connect(ising_t *h, void *const d_below_upper_halo[2], void *const d_above_lower_halo[2]);
int ising_slab_half_sweep_boundary_push(ising_t *h, double beta, void *stream);

/* nsweeps sweeps of a lattice whose `nslabs` slab handles (slabs[r] = slab r, all at the same counter t, same seed and mode) live
 * in this process on the current device: boundary kernels and plane copies (cudaMemcpyAsync) on stream_a, bulk kernels on
 * stream_b, an event pair between half-sweeps.  The two streams must differ; on return both have been made to wait for each other. */
int ising_slab_sweep_local(ising_t **slabs, int nslabs, double beta, int nsweeps, void *stream_a, void *stream_b);
/* The same with the fused exchange: connects every slab to its neighbours and runs the _push boundary kernels; no copies. */
int ising_slab_sweep_local_push(ising_t **slabs, int nslabs, double beta, int nsweeps, void *stream_a, void *stream_b);

/* ---- the paper's sliced layout (Eq. 4-6; Appendix A) ----
 * An alternative internal layout of a one-sample lattice, kept beside the handle's own arrays in a caller-owned scratch buffer:
 * x' = x, y' = y - x, z' = x - y + z; planes of constant z' are one-coloured; the colours are separate arrays of L/2 planes of L x L
 * sites, rows of 32-site words along x.  L must be 64 * 2^e, rng modes 0 and 1.  It exists to MEASURE the layout against the
 * rank-linear arrays: the trajectory is the same bit for bit, but the Philox draws of R9, four consecutive
 * canonical sites per call, cost one call per site here.
 *   ising_sliced_scratch_bytes  size of the scratch (the eight sliced arrays; 256-byte aligned device memory)
 *   ising_sliced_begin          handle's spins and couplings -> sliced arrays
 *   ising_sliced_sweep          nsweeps sweeps on the sliced arrays (one launch per colour half-sweep); advances t
 *   ising_sliced_end            sliced spins -> the handle's arrays (after which ising_energy / ising_get_spins see them) */
int ising_sliced_scratch_bytes(const ising_t *h, size_t *out);
int ising_sliced_begin(ising_t *h, void *d_scratch, void *stream);
int ising_sliced_sweep(ising_t *h, void *d_scratch, double beta, int nsweeps, void *stream);
int ising_sliced_end(ising_t *h, void *d_scratch, void *stream);

/* Select the kernels: 0 = automatic (site-packed lattices, one sample or a batch: the word-parallel kernel when L is a multiple of
 * 64, with the cached seed table in MINSTD mode, the bit-window kernel for every other even L; sample-packed: the vectorised /
 * tile / bit-sliced kernels where L allows them), 1 = force the generic one-site- or one-bit-at-a-time kernels (half-sweep,
 * energy, load, get), 2 = the word-parallel kernel without the seed table (MINSTD seeds recomputed per draw), 3 = as 0 but always
 * one launch per colour half-sweep, 4 = as 0 but the persistent kernels wherever they exist, 5 = as 0 without the cluster-resident
 * kernel.  0 runs all half-sweeps of a call in ONE launch where that is faster: one-sample lattices of at most 1024 words per
 * colour (every even L <= 40) on one SM out of shared memory; L = 64 (one sample, or many: up to 256 with Philox, any number with MINSTD) with one
 * thread-block cluster per sample and the lattice in distributed shared memory; and replays CUDA graphs of up to 64 half-sweeps at
 * L = 128, one sample (and at L = 64 under choice 5).  4 extends the cluster-resident kernel to L = 128 and to any number of samples
 * and adds the dataflow kernel of co-resident CTAs for one-sample multiples of 64 below 512.  All give the same bits; the tests use
 * this to show that results do not depend on layout, thread mapping, caching or launch structure. */
int ising_set_kernel(ising_t *h, int which);

/* Number of kernels this handle has launched so far. */
uint64_t ising_kernel_launches(const ising_t *h);

/* Host only, test hook: run the word update of the word-parallel kernels (the same __host__ __device__
 * code: Philox / MINSTD draws, Eq. 11-13 adder, per-bit acceptance, Eq. 17 mask) on ONE 32-site word given
 * its 13 operand words.  It exists so that the bit logic can be checked without a GPU; it is not a sweep.
 *   ops[0] = active spins s; ops[1..6] = neighbour spin words already aligned under s in the order
 *   +x,-x,+y,-y,+z,-z; ops[7..12] = the matching coupling words (same order).
 *   word_index: index of the word in its colour array (site-packed: colour rank j = 32*word_index + bit);
 *   site0 / site_stride: canonical site index of bit 0 and its increment per bit (MINSTD stream ids).
 * Returns the updated word in *out. */
int ising_hostcheck_update_word(int rng_mode, uint64_t seed, uint64_t t, double beta, const uint32_t ops[13],
                                uint64_t word_index, uint64_t site0, uint64_t site_stride, uint32_t *out);

int ising_destroy(ising_t *h);

const char *ising_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_H */
