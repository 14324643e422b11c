/* ising.h — C ABI of libising_b200: the double-checkerboard Metropolis sweep of
 * arXiv 1006.3865 (M. Weigel, "Simulating spin models on GPU") on one B200 (sm_100a).
 *
 * Citations: P:n = line n of the paper text; S8c.k = item k of the normative
 * specification in SURVEY.md §8(c), restated with every reading in DESIGN.md §3.
 *
 * Model (eq. (1)): spins s_i = ±1 on a periodic square (dim 2) or simple cubic
 * (dim 3) lattice of edge L, H = -Σ_<ij> J_ij s_i s_j.  A proposed flip is accepted with
 * p = min[1, exp(-β ΔE)] (eq. (2)).  The update order is the double checkerboard of
 * tiles of T^dim sites coloured even/odd, sites coloured even/odd, even first at
 * both levels, k inner sweeps per tile visit ("multi-hit").
 *
 * Conventions common to every call
 *   - Site index i = x + L*(y + L*z); canonical spin array = N = L^dim int8 values ±1 in
 *     index order, replica-major when the handle holds R > 1 replicas (R*N bytes).
 *   - Every pointer argument marked [host|device] may be either; the library asks the CUDA
 *     runtime which it is.  Caller owns all argument buffers; the library owns the handle.
 *   - Return value 0 = success, negative ISING_E* = failure (message: ising_last_error()).
 *     ising_create* return NULL on failure.  No C++ exception crosses this boundary.
 *   - All work is issued on the stream set by ising_set_device_hooks (default stream 0).
 *     ising_sweep is asynchronous; calls that hand data back to the caller synchronise that
 *     stream before returning.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with
 *     ISING_ECUDA.
 */
#ifndef ISING_B200_H
#define ISING_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ising_ctx* ising_handle;

enum {
    ISING_OK = 0,
    ISING_EINVAL = -1,       /* bad argument (message says which)                    */
    ISING_ENOMEM = -2,       /* device allocation failed                              */
    ISING_ECUDA = -3,        /* CUDA runtime / launch error, or no device            */
    ISING_EUNSUPPORTED = -4  /* valid request this library has no kernel for         */
};

enum {
    ISING_LAYOUT_I8 = 0,     /* one byte per spin in HBM (default)                    */
    ISING_LAYOUT_BITS = 1    /* one bit per spin in HBM (synchronous multi-spin form) */
};

enum {
    ISING_RNG_WORDS = 0,     /* one Philox4x32-10 output word per site          */
    ISING_RNG_PLANES = 1     /* default: 12 bit-plane bits per 32-site block + 20 per-site bits */
};

/* ising_create — P:53-57; S8c.1-3.
 * dim ∈ {2,3}; L even, ≥ 2, N = L^dim ≤ 2^32.  coupling_or_null [host|device]: NULL ⇒
 * J = +1 on every bond (eq. (1)); otherwise int8 J[dim][N], J[d][i] = bond between site i
 * and i + e_d, every value ±1 (else NULL is returned); the array is copied.  seed = 64-bit
 * Philox4x32-10 key: the hot start s_i = sign bit of Philox(ctr={i>>2,1,0,0})[i&3] and the
 * sweep stream both derive from it.  The inner-sweep counter t starts at 0. */
ising_handle ising_create(int dim, int L, const int8_t* coupling_or_null, uint64_t seed);

/* ising_create_batch — P:100 ("many disorder realizations concurrently"); S8c item 12.
 * n_replicas ≥ 1 independent spin systems (seeds[r], host pointer) sharing one coupling
 * array, advanced together by every ising_sweep (one batched launch per phase). */
ising_handle ising_create_batch(int dim, int L, const int8_t* coupling_or_null,
                                const uint64_t* seeds, int n_replicas);

/* ising_create_multi — P:100 ("asynchronous multi-spin coding", many disorder realisations at once); DESIGN.md
 * §3.6 R17.  R >= 1 realisations of the +-J model, each with its own couplings (couplings = int8 J[R][dim][N],
 * [host|device]) and its own hot start (init_seeds[r], host pointer), all driven by ONE sweep random stream
 * r(i, H) keyed by sweep_seed: realisation r is exactly an ordinary run with couplings J[r] whose random stream
 * happens to be shared with the others.  Everything else (sweep, observables per realisation, copy_spins R*N bytes,
 * overlap) is as for ising_create_batch.  The RNG mapping of a multi handle starts as ISING_RNG_WORDS (one random
 * word per site serves all realisations); with it, n_realisations <= 256 and tile 32 / 64 (dim 2) or tile 8 (dim 3: the
 * Edwards-Anderson glass of P:100) the sweep runs on the multi-spin-coded kernels (32 realisations per machine word; more
 * than 32 as several word lattices driven by the same random numbers). */
ising_handle ising_create_multi(int dim, int L, const int8_t* couplings, const uint64_t* init_seeds, int n_realisations,
                                uint64_t sweep_seed);

void ising_destroy(ising_handle h);

/* ising_sweep — P:64-74 (steps 1-7 and the k-fold multi-hit); S8c.4-6.
 * n_sweeps ≥ 0 outer passes.  One pass = all tiles of coarse colour 0, then colour 1; each
 * tile visit runs k_inner ≥ 1 times (even sites, then odd sites) with its halo frozen.
 * tile = edge T: T even, T | L, and L/T even or T == L; 0 means T = L (the single
 * checkerboard of P:62).  beta finite, ≥ 0.  Acceptance is the integer test
 * r < floor(exp(-β ΔE)·2^32), table built in double on the host (S8c.4).  The 32-bit uniform r of site i in
 * half-sweep H = 2t + colour comes from Philox4x32-10 keyed by the seed, under the handle's RNG mapping (ising_set_rng):
 *   ISING_RNG_PLANES (default): the 12 leading bits of r are bit j of the planes
 *     Philox(ctr={g, 3 + 256 (q>>2), lo32 H, hi32 H})[q&3], q = 0..11, of the site's 32-site block g (bit j = the site's place in
 *     the block), the 20 trailing bits are Philox(ctr={i>>1, 4, lo32 H, hi32 H})[0] >> 12;
 *   ISING_RNG_WORDS: r = Philox(ctr={p>>2, 0, lo32 H, hi32 H})[p&3], p = i>>1.
 * Both give every (site, half-sweep) its own uniform r; the trajectories differ.  Advances t by n_sweeps·k_inner.
 * Asynchronous.  Which kernel runs (a launch per coarse colour, one persistent launch per call for HBM-resident
 * lattices, one cooperative launch with the lattice on chip for smaller ones, ...) never changes the result:
 * ising_sweep_path.  A change of `tile` between calls re-lays the spins out in HBM (through the canonical array,
 * one extra pass over the lattice in each direction). */
int ising_sweep(ising_handle h, double beta, int n_sweeps, int tile, int k_inner);

/* ising_sweep_series — same as ising_sweep, and after every outer pass writes
 * E[pass*R + r], M[pass*R + r] (n_sweeps·R int64 each, [host|device], either may be NULL).
 * Synchronises when an output is a host pointer. */
int ising_sweep_series(ising_handle h, double beta, int n_sweeps, int tile, int k_inner,
                       int64_t* E, int64_t* M);

/* ising_observables — P:86 (E and M are measured but not timed); S8c.7.
 * E[r] = -Σ_i Σ_{d<dim} J_d(i) s_i s_(i+e_d),  M[r] = Σ_i s_i, exact int64, r < R.
 * E, M [host|device], either may be NULL.  Synchronises. */
int ising_observables(ising_handle h, int64_t* E, int64_t* M);

/* ising_overlap — replica overlap Q_ab = Σ_i s_i^a s_i^b (q = Q/N); S8c.7. */
int ising_overlap(ising_handle h, int a, int b, int64_t* Q);

/* ising_overlap_all — all pairwise overlaps of the R replicas of the handle in one call (BASELINE config 5: "per-replica E
 * and pairwise overlap q"; replicas of the +-J glass; S8c.7): Q[a*R + b] = Σ_i s_i^a s_i^b for every a, b
 * (symmetric, Q[a*R + a] = N), R·R int64 values to Q [host|device], caller-owned.  Computed where the spins currently live
 * (XOR + popcount on the bit / byte tile records, no conversion to the canonical array).  Synchronises. */
int ising_overlap_all(ising_handle h, int64_t* Q);

/* ising_overlap_all_static — the same R x R table of overlaps (S8c.7) for callers that may not allocate device
 * memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Takes no handle and calls
 * no cudaMalloc / cudaFree / allocating library routine: its scratch (R·R difference counts) is a file-scope __device__
 * array of ISING_STATIC_MAX_REPLICAS^2 x 8 bytes = 32 KiB that every GPU which loads the library holds until exit.
 *   d_spins [device]  n_replicas · n_sites canonical int8 ±1 spins, replica-major (what ising_copy_spins writes), 4-byte
 *                     aligned; n_sites a positive multiple of 4.  Caller-owned, read only.
 *   d_Q     [device]  n_replicas · n_replicas int64, 8-byte aligned, caller-owned: Q[a*R + b] = Σ_i s_i^a s_i^b.
 *   cuda_stream       the cudaStream_t to enqueue on; NULL = the library's stream (ising_set_device_hooks).
 * Asynchronous: the work is enqueued and the call returns; nothing is copied to the host.  n_replicas < 1 or
 * > ISING_STATIC_MAX_REPLICAS, NULL or misaligned pointers, bad n_sites ⇒ ISING_EINVAL, nothing enqueued.  ALL calls share
 * the one array, which keeps the last call's contents (each call clears the part it uses first): calls that overlap on
 * the GPU (different streams or host threads) race; serialise them.  The first call on a device resolves the array's
 * device address (cudaGetSymbolAddress, once per device): make it before, not under, a graph capture. */
#define ISING_STATIC_MAX_REPLICAS 64
int ising_overlap_all_static(const int8_t* d_spins, int n_replicas, uint64_t n_sites, int64_t* d_Q, void* cuda_stream);

/* ising_copy_spins — canonical int8 ±1 spins, R·N bytes, to dst [host|device]. Synchronises. */
int ising_copy_spins(ising_handle h, int8_t* dst);

/* ising_set_spins — overwrite the spins from canonical int8 ±1 (R·N bytes, [host|device]);
 * any other value ⇒ ISING_EINVAL and the state is unchanged.  Does not touch t. */
int ising_set_spins(ising_handle h, const int8_t* src);

/* ising_copy_spins_bits / ising_set_spins_bits — the same state as one bit per site (eight times fewer bytes over
 * PCIe; the spin is all the model has): word (r·N + i) >> 5, bit i & 31, set ⇔ s_i = +1; R·N/32 uint32
 * words [host|device].  Needs N % 32 == 0 (else ISING_EUNSUPPORTED).  Every bit pattern is a valid state.
 * Synchronise; do not touch t. */
int ising_copy_spins_bits(ising_handle h, uint32_t* dst);
int ising_set_spins_bits(ising_handle h, const uint32_t* src);

/* ising_set_layout — ISING_LAYOUT_I8 or ISING_LAYOUT_BITS: how spins are held in HBM between
 * sweeps.  The trajectory does not depend on it (S8c: both layouts give the same bits). */
int ising_set_layout(ising_handle h, int layout);

/* ising_set_rng — which RNG->site mapping the sweeps use (the paper names no generator, P:78,
 * P:84; DESIGN.md §3 R6 defines both).  Every (site, half-sweep) gets its own uniform 32-bit r
 * from Philox4x32-10 keyed by the seed, compared with the same uint32 thresholds:
 *   ISING_RNG_WORDS   r = Philox(ctr={p>>2, 0, lo32 H, hi32 H})[p&3], p = i>>1 (S8c.3).
 *   ISING_RNG_PLANES  (default) sites of one colour are cut into blocks of 32 (16 pairs x 2 rows
 *     in 2D, 4 pairs x 8 rows in 3D); bit j of plane q = Philox(ctr={g, 3+256*(q>>2), lo32 H,
 *     hi32 H})[q&3] is bit (11-q) of the 12-bit head of site j of block g; the 20-bit tail is
 *     Philox(ctr={i>>1, 4, lo32 H, hi32 H})[0] >> 12; r = head<<20 | tail.
 * The two mappings are different valid Markov chains (different trajectories).  May be called
 * at any time; spins and t are untouched. */
int ising_set_rng(ising_handle h, int mode);

enum {
    ISING_JIT_AUTO = 0,      /* specialise on big calls only (>= 2^27 attempted flips per ising_sweep)   */
    ISING_JIT_OFF = 1,       /* always the pre-compiled kernels                                          */
    ISING_JIT_ON = 2         /* specialise whenever a specialisable kernel is used                       */
};

/* ising_set_jit — run-time specialisation of the 2D multi-spin tile kernel (a2 + a5).  The thresholds of
 * S8c.4 depend on beta only; with their 12 head bits as compile-time constants the bit-serial compare of
 * r with thr[a/2] needs half the instructions.  The library can compile its own kernel source for the
 * current thresholds with NVRTC (first use of a beta: about a second; cached per process).  Results are
 * bit-identical either way; if NVRTC is missing the pre-compiled kernel is used.
 * ising_last_sweep_specialized returns 1 if the last ising_sweep on h ran a specialised kernel. */
int ising_set_jit(ising_handle h, int mode);
int ising_last_sweep_specialized(ising_handle h);

/* The state of a run is (spins, t, seed): the random stream is stateless (S8c.3), so
 * copy_spins + get_counter / set_spins + set_counter resume a run bit-exactly. */
int ising_get_counter(ising_handle h, uint64_t* t);
int ising_set_counter(ising_handle h, uint64_t t);

/* ising_thresholds — the acceptance table of S8c.4 as the library builds it:
 * out[m-1] = floor(exp(-β·4m)·2^32) for m = 1..dim, 0 beyond (host pointer, 3 entries). */
int ising_thresholds(double beta, int dim, uint64_t* out);

/* ising_set_device_hooks — process-wide.  alloc(bytes) returns a device pointer (or NULL),
 * dealloc(ptr) releases it; cuda_stream is a cudaStream_t.  NULL alloc/dealloc restore
 * cudaMalloc/cudaFree.  Existing handles keep (and later release through dealloc at the
 * time of destroy) what they already hold, so set the hooks before creating handles. */
int ising_set_device_hooks(void* (*alloc)(size_t), void (*dealloc)(void*), void* cuda_stream);

/* ising_synchronize — wait for all work issued for this handle. */
int ising_synchronize(ising_handle h);

/* ising_kernel_launches — number of kernels this library has launched in this process
 * (bench.py's gpu_launches). */
uint64_t ising_kernel_launches(void);

/* ising_sweep_path — name of the kernel family the last ising_sweep on h used; static string, never NULL.  Every
 * family computes the same trajectory; names end in _i8 or _bits (the HBM layout) where both exist.
 *   generic                 global-memory kernels, one launch per half-sweep: any valid (dim, L, tile, J)
 *   tile_i8                 2D tiles 32 / 64, RNG mapping "words"
 *   tile_planes_*           2D tiles 32 / 64, J = +1 or +-J, replicas: a launch per coarse colour (the headline kernel)
 *   tile3d_planes_*         3D tiles 8, J = +1 or +-J, replicas
 *   plain64_planes_*        L = 64 plain checkerboard, the whole call in one launch of one warp per replica
 *   resident_planes_*       2D, at most 64 warp jobs per coarse colour (L <= 512), n_sweeps >= 2: the whole call in one
 *                           launch of one thread-block cluster per replica, lattice in registers, tile boundaries through
 *                           distributed shared memory, E / M of ising_sweep_series counted on the registers
 *   resident3d_planes_*     the same in 3D, L <= 64
 *   resident_plain_*, tile_plain_*, resident3d_plain_*, tile3d_plain_*
 *                           the plain checkerboard (tile == L) on the cluster-resident kernels (2D 64 < L <= 512, 3D L <= 64)
 *                           or, for larger lattices, with a launch per half-sweep
 *   resident_masked_*, tile_masked_*, resident3d_masked_*, tile3d_masked_*
 *                           double checkerboard with power-of-two tiles other than the register tiles (2D: 2, 4, 8, 16 —
 *                           the paper's sizes, P:86 — and 128, 256, ...; 3D: 2, 4, 16, 32, ...) as masked half-sweeps
 *   grid_plain_*, grid_masked_*   the same two schemes for 2D lattices beyond the cluster, up to 2^24 sites, in calls of four
 *                           sweeps or more: every half-sweep of the call in one cooperative launch, the lattice on chip on all
 *                           SMs, every tile exchanging its boundary after every half-sweep (k_grid_plain)
 *   grid_planes_{i8,bits}, grid3d_planes_{i8,bits}   lattices beyond the cluster that fit in the shared memory of the GPU (2D
 *                           512 < L, up to 2^28 sites on a B200 where measured to pay: DESIGN.md §6.1g; 3D 64 < L): the whole
 *                           call in one cooperative launch, the lattice read from and written to HBM once per call, boundary
 *                           words exchanged through L2
 *   flow_planes_{i8,bits}   HBM-resident 2D lattices (and calls too short to pay for putting the lattice on chip): all passes in
 *                           one persistent launch, coarse colours ordered by per-tile progress counters
 *   amsc                    asynchronous multi-spin coding of a multi-realisation batch (ising_create_multi)
 * The fast 2D families need L % 32 == 0 (L % 64 for tile 64) and an even number of register tiles per side, the 3D ones
 * L % 8 == 0 and L / 8 even. */
const char* ising_sweep_path(ising_handle h);

/* ising_force_path — testing / measuring aid: 0 = automatic kernel choice, 1 = always the generic global-memory kernels,
 * 2 = a launch per coarse colour (never a cluster-resident, grid-resident or data-flow kernel), 3 = never the persistent
 * data-flow kernel, 4 = never the cluster / grid resident kernels (the data-flow kernel may then run at any size and k). */
int ising_force_path(ising_handle h, int generic_only);

const char* ising_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_H */
