/*
 * wolff.h -- C-ABI boundary of the B200-native Wolff single-cluster hot path.
 *
 * Method: Y. Komura, Y. Okabe, "GPU-based single-cluster algorithm for the
 * simulation of the Ising model", arXiv 1110.0899.  Citations below are
 * "PAPER.md:<line> (section)" into the paper text this build was written from.
 * DESIGN.md section 3 lists the readings (R1..R15) taken where the paper is
 * silent; they are the same on both sides of the parity tests.
 *
 * What one update computes (section 2, steps i-v; Hamiltonian and
 * periodic boundaries PAPER.md:36-40, Eq. 2; wave-front parallel growth
 * PAPER.md:84-98, section 4): choose a site i0; let s0 be its spin; the cluster is
 * the connected component of i0 in the graph whose edges are the lattice bonds
 * between two spins equal to s0 whose bond variable is active (probability
 * p = 1 - exp(-2J/T)); flip every spin of the cluster.  Bond
 * variables are a pure function of (seed, update index, undirected edge), so the
 * result does not depend on traversal order or thread schedule.
 *
 * Conventions
 *   - Lattice: N = L^dim sites, int8 spins +1 / -1, site id i = x + L*y (+ L*L*z),
 *     x fastest; periodic in every direction.
 *   - All device state is owned by the library and lives on the CUDA device that is
 *     current when wolff_create is called.  Every output buffer and the stream are
 *     owned by the caller.  Pointers marked "host or device" may be either (they are
 *     classified with cudaPointerGetAttributes); pageable host memory is allowed.
 *   - Every call returns 0 (WOLFF_OK) or a negative error code; the reason is kept in
 *     a thread-local string returned by wolff_last_error().  Nothing aborts, throws or
 *     prints.  A CUDA error is sticky on the handle (later calls return WOLFF_ECUDA).
 *     A device-side watchdog abort is sticky on the device: launches queued behind the
 *     aborted one do nothing, and the next synchronising call returns WOLFF_EINTERNAL.
 *   - Calls make the handle's device current for their own duration and restore the
 *     caller's current device before they return.
 *   - A handle is not thread-safe; distinct handles are independent, also when different host threads drive handles
 *     of different lattice sizes: the one piece of per-process kernel state, the dynamic shared-memory limit of each
 *     kernel, is only ever set to a single value (the device's maximum), never to a handle's own need.
 *   - There is no CPU fallback: without a usable CUDA device wolff_create fails.
 */
#ifndef WOLFF_B200_H
#define WOLFF_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define WOLFF_API __attribute__((visibility("default")))
#else
#define WOLFF_API
#endif

#define WOLFF_OK      0
#define WOLFF_EINVAL (-1)   /* bad argument */
#define WOLFF_ENOMEM (-2)   /* device or host allocation failed */
#define WOLFF_ECUDA  (-3)   /* CUDA runtime error (sticky on the handle) */
#define WOLFF_EINTERNAL (-4) /* device-side watchdog fired (a barrier did not complete) */

typedef struct wolff_ctx *wolff_handle;   /* opaque, library-owned */

/* Create a chain.  dim = 2 (square) or 3 (simple cubic); L >= 2; N = L^dim <= 2^31;
 * J >= 0 and T > 0 finite (J and T act only through the integer bond
 * threshold floor((1 - exp(-2J/T)) * 2^32)).  Allocates the lattice, the
 * cluster list (uint32 x N, the "ic/in" list of PAPER.md:50) and control words on the
 * current device, fills the lattice with the seed-derived random +/-1 start
 * (BASELINE.json configs: "random start from seed"), sets the update index to 0.
 * Returns NULL on failure (see wolff_last_error). */
WOLFF_API wolff_handle wolff_create(int dim, int L, double J, double T, uint64_t seed);

/* Enqueue n_updates single-cluster updates (PAPER.md:42-48 steps i-v, grown wave-front
 * parallel as in PAPER.md:84-98) on cuda_stream (a cudaStream_t passed as void*; NULL =
 * the legacy default stream) as ONE persistent kernel launch, and return without waiting.
 * Update indices continue from the handle's counter: run(a); run(b) equals run(a+b).
 * n_updates == 0 is a no-op.  The per-update cluster sizes of this call are kept on the
 * device until the next wolff_run (see wolff_observables). */
WOLFF_API int wolff_run(wolff_handle h, uint64_t n_updates, void *cuda_stream);

/* Wait for the handle's queued work, then compute on the device, from the CURRENT lattice,
 * E = - sum over bonds s_i s_j (each bond once, units of J; Eq. 2) and
 * M = sum s_i ("measurement of energy and magnetization"), and, if
 * cluster_sizes != NULL, copy the n_updates cluster sizes of the MOST RECENT wolff_run
 * (uint32 each; the final value of the counter "ic" of PAPER.md:50).  Any of the three
 * pointers may be NULL; each may be host or device memory.  Blocks until done. */
WOLFF_API int wolff_observables(wolff_handle h, int64_t *E, int64_t *M, uint32_t *cluster_sizes);

/* Copy the lattice (N bytes, +1/-1, x fastest) to dst (host or device).  Blocks.  The spins S_i = +/-1 of PAPER.md:36-40
 * (Eq. 2), one int8 each (the paper packs spin and in-cluster flag into one word; here
 * the flip itself is the claim, so the byte is the spin and nothing else). */
WOLFF_API int wolff_get_spins(wolff_handle h, int8_t *dst);

/* Load a lattice (N bytes, each +1 or -1; host or device).  Used for cold starts (the
 * "equilibrated" benchmark variant; PAPER.md:126 measures at T_c), crafted
 * cases and resuming.  Values other than +/-1 give WOLFF_EINVAL and leave the lattice
 * unchanged.  Blocks. */
WOLFF_API int wolff_set_spins(wolff_handle h, const int8_t *src);

/* Update index (number of updates done since creation, or as set: the count of step (v) of
 * PAPER.md:48, which keys the site draw and the bond variables, R8/R10) and the integer bond
 * threshold in [0, 2^32] (p = 1 - exp(-2J/T); R7).  Either pointer may be NULL (host pointers). */
WOLFF_API int wolff_get_state(wolff_handle h, uint64_t *update_index, uint64_t *threshold);

/* Set the update index (to resume a chain: lattice + index + seed is the whole state). */
WOLFF_API int wolff_set_update_index(wolff_handle h, uint64_t update_index);

/* In-kernel measurement -- the paper's "+ measurement" columns ("the time for only spin-update and that
 * including the measurement of energy and magnetization"; Tables 1-2) and its Binder ratio (Eq. 3,
 * PAPER.md:159-164).  With wolff_set_option(h, "measure", 1) every wolff_run evaluates E and M after EVERY update
 * without leaving the persistent kernel, logs them on the device, and adds them to exact integer accumulators:
 *   - shared-memory-resident kernel: after each update every CTA sums the tiles it holds (the low faces of the tiles are
 *     exchanged through global memory); cost per update independent of the cluster, a few microseconds;
 *   - cluster-resident kernel (L a multiple of 32): after each update every CTA of the cluster counts the negative spins
 *     and the unequal forward bonds of its slab of the bit lattice (32 spins per population count) and sends its sums to
 *     CTA 0 in one reduction; cost per update independent of the cluster;
 *   - level-synchronous kernel: M changes by -2 s0 |C|; E by 2 * sum over the cluster's boundary bonds (member i,
 *     non-member j) of s0 s_j, counted in a pass over the update's member list while every member still carries a mark
 *     in bit 1 of its byte (the role of the flag the paper packs into the spin word); cost
 *     proportional to the cluster.
 * All give exactly the values wolff_observables would return after each update.
 *
 * wolff_get_series: the per-update series of the MOST RECENT wolff_run, n_updates entries each: E and M after each
 * update (needs "measure" = 1 during that run, else WOLFF_EINVAL) and the duration of each update in nanoseconds as
 * the kernel saw it (always recorded; saturates at 2^32 - 1).  Any pointer may be NULL; host or device.  Blocks. */
WOLFF_API int wolff_get_series(wolff_handle h, int64_t *E_series, int64_t *M_series, uint32_t *update_ns);

/* Accumulated over all measured updates since creation or the last reset, ten 64-bit words (host pointer):
 *   [0] n   [1] sum E (two's complement)   [2] sum |M|   [3],[4] sum E^2 (low, high word)
 *   [5],[6] sum M^2   [7],[8] sum M^4   [9] 0
 * exact integers (M^4 reaches 2^96 at 2^24 spins, hence 128 bits).  They stay exact while samples x N^4 < 2^128: any
 * number of samples up to N = 2^16, 2^32 samples at N = 2^24, 2^16 at N = 2^28, 16 at N = 2^31; a measured wolff_run
 * (or wolff_batch_run) that would take the count past that bound is refused with WOLFF_EINVAL before anything is
 * launched (reset the moments to go on).  And the Binder ratio of PAPER.md Eq. 3,
 * U = 1 - <M^4> / (3 <M^2>^2), from them (NaN without samples).  Either pointer may be NULL.  Blocks. */
WOLFF_API int wolff_get_moments(wolff_handle h, uint64_t *moments, double *binder);
WOLFF_API int wolff_reset_moments(wolff_handle h);

/* Tuning / test knobs; never change the result.  Three growth kernels implement wolff_run:
 *  - the shared-memory-resident, barrier-free kernel of all SMs (int8 lattice tiles live in the CTAs' shared memory
 *    for the launch, claims across CTAs travel as messages, bond variables come from tables filled ahead of time):
 *    applies when L is a power of two >= 4 and the lattice fits the chip's shared memory; the fastest on clusters of
 *    tens of thousands of spins and more (the BASELINE lattices at T_c);
 *  - the cluster-resident, bit-packed, barrier-free kernel (one bit per spin in the distributed shared memory of ONE
 *    thread-block cluster of up to 16 CTAs; a claim is one atomic on the word that holds the spin, in whichever CTA
 *    holds it; the warp that draws the seed site expands it itself): applies to any L with N <= 2^24 (N / 8 bytes fit
 *    one cluster); the fastest on small and medium clusters (the literal random start of the BASELINE configs, T above
 *    T_c, 3D L = 128) and on every lattice the first kernel does not apply to (L not a power of two);
 *  - the level-synchronous kernel, which runs each BFS level in one of three tiers by frontier width n: one
 *    CTA (n <= up), one thread-block cluster (n <= cluster_up), the whole grid (above): any L.
 * Keys:
 *   "mode"                 0 = chosen by the lattice and the mean cluster size of the last finished run, see
 *                          "small_cluster" (default);
 *                          5 = the cluster-resident kernel whenever it applies (else as mode 0);
 *                          level-synchronous kernel only: 4 = tiers by frontier width, 1 = every level
 *                          grid-wide, 2 = one CTA whenever the frontier fits its shared-memory queue, 3 = the
 *                          cluster whenever it fits
 *   "measure"              1 = E and M after every update inside the kernel (see wolff_get_series); default 0.  The
 *                          cluster-resident kernel measures when L is a multiple of 32 (population counts over its bit
 *                          lattice after each update: cost independent of the cluster); otherwise, and for clusters of
 *                          a handful of spins, a measured run uses one of the other two
 *   "small_cluster"        mode 0: when the last finished run (seen at the caller's next synchronising call) had a mean
 *                          cluster below this size, the next run uses the cluster-resident kernel (default: the measured
 *                          crossover, 8192 in 2D and 32768 in 3D; 0 = never) -- unless the call is for fewer than N / 2^20
 *                          updates, which the launch of that kernel (it packs the lattice with 16 SMs) would dominate;
 *                          where that kernel does not apply, runs with a mean cluster below min(16, this) use
 *                          the level-synchronous kernel, whose fixed cost per update is lower than the first kernel's
 *   "resident_ctas"        cluster-resident kernel: CTAs of the cluster, at most (1, 2, 4, 8 or 16; default 16)
 *   "tile_log"             shared-memory-resident kernel: log2 of the tile side (0 = auto: 6 in 2D, 4 in 3D)
 *   "tile_ctas"            ... CTAs that share the lattice (0 = one per SM)
 *   "ring_cap"             ... entries of a CTA's shared-memory work ring (power of two; overflow spills to global memory);
 *                          also the ring of the cluster-resident kernel
 *   "inbox_log"            ... log2 of the entries of a CTA's inbox, the global-memory queue of claims other CTAs send it
 *                          (0 = auto: what one update can send at most, no capacity checks; 5..24: a smaller inbox --
 *                          a sender that finds it full waits for the receiver, which never waits for anybody)
 *   "fill"                 ... bond tables: 0 = never (Philox inline), 1 = filled by idle warps when updates are long
 *                          enough to pay for it (default), 2 = always
 *   "fill_bufs"            ... bond-table buffers: 0 = two (the running update and the next one) when they fit beside the
 *                          lattice, else one (default); 1 = one
 *   "fill_min_us"          ... fill = 1: mean time per update above which tables are filled (default 30)
 *   "idle_ns"              ... longest sleep of an idle worker warp between two polls of the ring
 *   "watchdog_ms"          ... an update that takes longer aborts the launch (WOLFF_EINTERNAL at the next call)
 *   "up_threshold"         frontier width above which growth leaves one-CTA mode and wakes the cluster
 *   "down_threshold"       frontier width at or below which cluster growth returns to one CTA
 *   "cluster_up_threshold" frontier width above which growth leaves cluster mode for a grid phase
 *   "grid_down_threshold"  frontier width at or below which a grid phase returns to cluster mode
 *   "balance_min"          cluster mode: a CTA holding more than max(balance_min, 2 x fair share) entries
 *                          makes the level redistribute the frontier through distributed shared memory
 *   "cluster_ctas"         CTAs per thread-block cluster: 1, 2, 4, 8 or 16 (default 16)
 *   "grid_ctas"            total CTAs of the persistent kernel (0 = as many clusters as can be co-resident)
 *   "cooperative"          1 (default) = cooperative launch, 0 = plain launch of a grid sized to be co-resident
 *   "speculative"          level-synchronous kernel: 1 = no neighbour gather, the claim atomic is issued for every active
 *                          bond and its returned byte says whether the neighbour was parallel (default 0)
 *   "check_selftest"       bounds-checked builds only (-DWOLFF_CHECKED, libwolff_b200_checked.so): makes one check fail on
 *                          purpose, so that a test can see the report arrive (WOLFF_EINTERNAL at the next call)
 * Thresholds are clamped to what the shared-memory queues can hold.  Unknown key or out-of-range
 * value: WOLFF_EINVAL. */
WOLFF_API int wolff_set_option(wolff_handle h, const char *key, int64_t value);

/* Counters of the most recent wolff_run, for the latency roofline (host pointer, WOLFF_NSTATS values):
 *   [0] updates            [1] flipped spins        [2] one-CTA levels       [3] cluster levels
 *   [4] grid-wide levels   [5] cluster wake-ups     [6] rebalanced cluster levels
 *   [7] claim attempts (atomics)                    [8] widest frontier seen
 * shared-memory-resident kernel ([2]-[6], [8] stay 0):
 *   [9] termination polls of the monitor            [10] passes with a Philox block evaluated inline
 *   [11] messages between CTAs                      [12] sites handed over through the ring
 *   [13] warp passes (profiling builds)             [14] sites spilled to global memory
 *   [15] bond-table chunks filled (32 sites each)
 * cluster-resident kernel: [0], [1], [7], [9], [12], [13], [14] as above; [11] sites taken out of another CTA's ring
 * Blocks until the run has finished. */
#define WOLFF_NSTATS 16
WOLFF_API int wolff_get_stats(wolff_handle h, uint64_t *stats);

/* Dependent-latency microbenchmarks on the current device (the links of one BFS level of the
 * growth kernel, timed in isolation; they define the latency roofline bench.py reports).  Writes
 * WOLFF_NMICRO doubles, nanoseconds each, to a host pointer:
 *   [0] dependent L2 load, one lane (ld.global.cg over an L2-resident 16 MiB buffer)
 *   [1] dependent L2 load, one warp, 32 scattered lines   [2] dependent atom.or with return, one lane
 *   [3] dependent atom.or, one warp, 32 scattered words   [4] __syncthreads at 512 threads
 *   [5] three Philox4x32-10 blocks, one warp              [6] the library's grid barrier, one CTA per SM
 *   [7] one pass of the minimal dependent chain of the shared-memory-resident kernel, one warp alone on an SM:
 *       ld.shared (spin, bond bit) -> atom.shared (claim) -> ballot/popc -> st.shared -> __syncwarp -> ld.shared;
 *       this is the floor of t_pass in the latency roofline T_update >= depth x t_pass
 *   [8] fraction of lanes that won their claim in [7] (1.0 when the chain ran as intended; not a time)
 * between two CTAs of one thread-block cluster (the links of the cluster-resident kernel):
 *   [9] dependent ld.shared::cluster on the peer's shared memory, one lane    [10] dependent atom.shared::cluster.or with
 *   return on the peer, one lane    [11] ... one warp, 32 scattered words    [12] a word stored into the peer's shared
 *   memory until a warp polling there sees it, one way
 * Not part of the measured path. */
#define WOLFF_NMICRO 13
WOLFF_API int wolff_microbench(double *out_ns, int n_out);

/* Free everything wolff_create allocated (lattice, cluster list of PAPER.md:50, control block, logs).  NULL is allowed. */
WOLFF_API int wolff_destroy(wolff_handle h);

/* ------------------------------------------------------------------------------------------------------------------
 * A BATCH of R independent chains in one launch.
 *
 * The paper's physics results are sweeps over temperatures and lattice sizes (the temperature
 * dependence of the timings, Fig. 1, and the Binder ratio U(T) for several L, Fig. 2, Eq. 3): many independent chains.
 * A batch holds R chains of the same dim and L, chain r with its own J[r], T[r] and seed[r]; wolff_batch_run performs
 * n_updates updates of EVERY chain in ONE persistent launch, one CTA per chain at a time (a CTA takes the next chain
 * when it has finished one), so up to 8-16 chains per SM are in flight (or, "resident" = 3, one thread-block cluster per
 * chain: one launch per chain, seven side by side).  Chain r computes, bit for bit, what a single
 * chain made by wolff_create(dim, L, J[r], T[r], seed[r]) computes: same start lattice, same site draws, same bond
 * variables, same update index (the index is shared by the chains of a batch and advances by n_updates per run).
 * Layouts are replica-major: E[r], M[r]; cluster_sizes[r * n_updates + k]; spins[r * N + i]; series likewise.
 * Ownership, pointer kinds (host or device), error codes and blocking behaviour are those of the single-chain calls. */
typedef struct wolff_batch_ctx *wolff_batch;

/* J, T, seed: host arrays of R values.  1 <= R <= 2^20; the device must hold R * 5 N bytes. */
WOLFF_API wolff_batch wolff_batch_create(int dim, int L, int R, const double *J, const double *T, const uint64_t *seed);
WOLFF_API int wolff_batch_run(wolff_batch b, uint64_t n_updates, void *cuda_stream);
/* E[R], M[R] of the current lattices (whole-lattice sums); cluster_sizes[R * n_updates] of the most recent run. */
WOLFF_API int wolff_batch_observables(wolff_batch b, int64_t *E, int64_t *M, uint32_t *cluster_sizes);
WOLFF_API int wolff_batch_get_spins(wolff_batch b, int8_t *dst);           /* R * N bytes */
WOLFF_API int wolff_batch_set_spins(wolff_batch b, const int8_t *src);     /* R * N bytes, each +1 or -1 */
WOLFF_API int wolff_batch_get_state(wolff_batch b, uint64_t *update_index, uint64_t *thresholds /* R values */);
WOLFF_API int wolff_batch_set_update_index(wolff_batch b, uint64_t update_index);
/* Keys: "measure" 0 | 1 (E and M after every update of every chain, inside the kernel: see wolff_get_series);
 * "threads" threads per CTA: 0 = auto (256 for few chains, 64 for many), 32, 64, 128, 256;
 * "queue_cap" entries of a CTA's shared-memory copy of the frontier (wider frontiers are read from the member list);
 * "resident" where a chain's lattice lives while a CTA works on it: 1 = the int8 lattice in global memory (L2 / HBM);
 *   2 = bit-packed in the CTA's shared memory, one bit per spin (N <= about 1.8 million: 2D L = 1024 is 128 KiB) plus, in
 *   a measured run, one mark bit per spin (then N <= about 900,000; a run that does not fit returns WOLFF_EINVAL),
 *   packed from / unpacked to the int8 lattice around the chain's turn;
 *   3 = bit-packed in the distributed shared memory of one thread-block cluster per chain (N <= 2^24: 2D L = 4096 and
 *   3D L = 256 are 2 MiB = 16 CTAs): every chain is one launch of the cluster-resident kernel of wolff_run, the launches
 *   spread over the library's own streams (behind the caller's stream, which continues behind them), so that as many
 *   chains run side by side as clusters fit the chip (7 of 16 CTAs on a B200); in-kernel measurement when L is a multiple
 *   of 32 (else a measured run returns WOLFF_EINVAL); at most 2^30 updates per call;
 *   0 = auto: 2 when a plane is at most 32 KiB (several chains per SM stay in flight), else 1.  Never changes a result.
 * "watchdog_ms" ("resident" = 3): an update that takes longer aborts its chain's launch (default 20000).
 * A chain whose kernel aborted (watchdog; an out-of-bounds index in a checked build) is reported like a single chain's:
 * EVERY synchronising batch call (observables, get/set_spins, get_series, get/reset_moments, get_stats) looks at the
 * chains' error words after it has waited, returns WOLFF_EINTERNAL naming the first such chain, and the batch stays
 * failed (its lattices, logs and moments are then unfinished). */
WOLFF_API int wolff_batch_set_option(wolff_batch b, const char *key, int64_t value);
/* E and M after every update of the most recent (measured) run: R * n_updates values each. */
WOLFF_API int wolff_batch_get_series(wolff_batch b, int64_t *E_series, int64_t *M_series);
/* moments: R * 10 words (layout of wolff_get_moments); binder: R doubles (Eq. 3).  Host pointers. */
WOLFF_API int wolff_batch_get_moments(wolff_batch b, uint64_t *moments, double *binder);
WOLFF_API int wolff_batch_reset_moments(wolff_batch b);
/* Counters of the most recent run (host pointer, 4 values): updates, flipped spins, BFS levels, claim attempts,
 * summed over the chains. */
WOLFF_API int wolff_batch_get_stats(wolff_batch b, uint64_t *stats);
WOLFF_API int wolff_batch_destroy(wolff_batch b);

/* ------------------------------------------------------------------------------------------------------------------
 * E and M without any allocation, for callers that cannot let a library allocate on the device.
 *
 * Everything above works on a handle, and making a handle calls cudaMalloc.  Some host programs cannot afford that: a
 * simulation that gave the whole card to its own arena at start-up (cudaMalloc then finds nothing); a service that
 * must stay inside a fixed memory budget once it is initialised; a program with a latency-critical loop on other
 * streams of the device, which cudaMalloc / cudaFree stall while they run.  For them this one call computes, from a
 * lattice that lives in THEIR device memory, the same two integers wolff_observables returns: E = - sum over bonds
 * s_i s_j (each bond once, units of J, periodic; Eq. 2) and M = sum s_i ("measurement of energy and
 * magnetization").  It calls no cudaMalloc, cudaFree or other allocating routine, and makes no staging
 * copies.
 *
 *   spins_dev   the lattice: N = L^dim bytes, +1 / -1, x fastest, in memory of the CURRENT device (or managed memory);
 *               16-byte aligned when L is a multiple of 16.  Read only; the bytes are not validated.
 *   dim, L      2 or 3; L >= 2; N <= WOLFF_NOALLOC_MAX_SITES (2^28: 2D up to L = 16384, 3D up to L = 645) -- larger
 *               lattices are refused with WOLFF_EINVAL, because the scratch memory is fixed in size
 *   E_dev, M_dev  one int64 each, in memory of the current device, managed memory or pinned host memory; either may be
 *               NULL.  Caller-owned, written by the kernel.
 *   cuda_stream a cudaStream_t passed as void* (NULL = the legacy default stream).  The call enqueues a 256-byte
 *               memset and one kernel there and returns without waiting: the results are in E_dev / M_dev once the
 *               stream has reached that point.
 *
 * Scratch memory: the partial sums of the reduction (one 16-byte slot per 16,384 sites) and a ticket live in a
 * file-scope __device__ array of 256.25 KiB inside the library image; every GPU on which the library is loaded holds
 * that much from load until the process exits.  All calls of a process share it, and it keeps what the last call left:
 * the ticket is cleared on the stream in front of every launch, the slots are overwritten before they are read.  Two
 * calls whose kernels can OVERLAP on the GPU (different streams without an ordering between them, or several host
 * threads) race on it and give wrong sums; calls on one stream, or ordered by events, are fine.
 * The FIRST call on each device looks the array's device address up (cudaGetSymbolAddress, with that device current)
 * and keeps it; make that first call before any stream capture begins on the thread.
 * Errors: WOLFF_EINVAL (dim, L, size beyond the limit, NULL / misaligned / host / other-device pointers),
 * WOLFF_ECUDA (the lookup, the memset or the launch failed); the text is in wolff_last_error(). */
#define WOLFF_NOALLOC_MAX_SITES (1u << 28)
WOLFF_API int wolff_energy_magnetisation_noalloc(const int8_t *spins_dev, int dim, int L, int64_t *E_dev, int64_t *M_dev,
                                                 void *cuda_stream);

/* Reason for the last failure on this thread (static storage, never NULL).  Not part of the method: the error
 * behaviour of the boundary ("Conventions" above). */
WOLFF_API const char *wolff_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* WOLFF_B200_H */
