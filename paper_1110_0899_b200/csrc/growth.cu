// growth.cu -- the persistent cluster-growth kernel.
//
// One launch performs n_updates Wolff single-cluster updates (steps i-v), each
// grown wave-front parallel (step iii'): every spin added in the previous level
// is expanded by one thread.  What differs from the paper's GTX-285 design:
//   - bond variables come from a counter-based Philox keyed on (seed, update, edge), so the
//     cluster is a well-defined connected component and any traversal order gives the same bits;
//   - "join the cluster" is one atomic that flips the spin (no flag word, and no
//     per-direction barrier): 2*dim barriers per level become one;
//   - the level loop runs in one of three tiers, chosen per level by the frontier width n:
//       one CTA      (n <= up)        shared-memory queues, __syncthreads only;
//       one cluster  (n <= cl_up)     the R CTAs of thread-block cluster 0, each with its own
//                                     shared-memory queue; counts are exchanged through distributed
//                                     shared memory and the level ends in the hardware cluster barrier;
//       whole grid   (n >  cl_up)     every CTA, over the global cluster list (the ic/in list of
//                                     PAPER.md:50), one atomic grid barrier per level (the role of the
//                                     paper's quasi-block synchronisation);
//   - the update loop itself is inside the kernel ("(v) Go to (i)").
// Why tiers: a level is a chain of dependent latencies (queue read -> L2 gather -> L2 atomic ->
// append -> barrier).  One SM sustains only ~0.5 scattered L2 requests per clock, so a frontier of a
// few hundred sites already takes microseconds on one CTA; sixteen SMs of a cluster take it in one
// pass, and their barrier costs ~0.2 us instead of the ~1.8 us of a grid-wide one.
#include "expand.cuh"
#include "internal.h"

namespace wolff {

namespace {

constexpr int kMaxClusterCtas = 16;

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ unsigned long long pack_bar(unsigned int gen, unsigned int phase, unsigned int hi)
{
    return ((unsigned long long)(gen & 0xFFFFFFu) << 40) | ((unsigned long long)(phase & 0xFFu) << 32) |
           (unsigned long long)hi;
}
__device__ __forceinline__ unsigned int bar_gen(unsigned long long w) { return (unsigned int)(w >> 40); }
__device__ __forceinline__ unsigned int bar_phase(unsigned long long w) { return (unsigned int)(w >> 32) & 0xFFu; }
__device__ __forceinline__ unsigned int bar_hi(unsigned long long w) { return (unsigned int)w; }

// ---------------------------------------------------------------- thread-block cluster primitives
__device__ __forceinline__ unsigned int cluster_ctarank()
{
    unsigned int r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned int cluster_nctarank()
{
    unsigned int r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned int cluster_id_x()
{
    unsigned int r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
// Hardware cluster barrier; release/acquire at cluster scope orders shared-memory (local and
// distributed) and global accesses of all threads of the cluster across it.
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// address of the same shared-memory location in CTA `rank` of this cluster
__device__ __forceinline__ uint32_t map_to_rank(uint32_t saddr, unsigned int rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ uint32_t ld_dsmem_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_dsmem_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// Wait until the barrier word carries generation `want`.  `bounded` waits (inside a grid phase,
// where every CTA is actively running) give up after ~2^24 polls and raise the error flag;
// parked CTAs wait without bound but leave when somebody else raised the flag.
__device__ __noinline__ unsigned long long wait_generation(Control *ctl, unsigned int want, bool bounded)
{
    unsigned int polls = 0;
    unsigned int ns = 32;
    for (;;) {
        const unsigned long long w = ld_acquire_u64(&ctl->bar);
        if (bar_gen(w) == (want & 0xFFFFFFu)) return w;
        ++polls;
        if ((polls & 0x3FFu) == 0u) {
            if (ld_relaxed_u32(&ctl->error) != 0u) return pack_bar(want, kPhaseAbort, 0u);
            if (bounded && polls > (1u << 24)) {
                st_relaxed_u32(&ctl->error, 1u);
                return pack_bar(want, kPhaseAbort, 0u);
            }
        }
        if (!bounded) {
            __nanosleep(ns);
            if (ns < 640) ns += ns >> 1;
        }
    }
}

// Command block, written by the master CTA into every CTA of cluster 0 (through distributed shared
// memory) right before the cluster barrier that wakes the helpers.
struct Command {
    unsigned int op;           // kCmdCluster / kCmdExit
    unsigned int par;          // queue buffer / count row that holds the frontier at entry
    int s0;                    // seed spin of the current update
    unsigned int u_lo, u_hi;   // update index
    unsigned int n;            // entries the master holds in its buffer `par`
    unsigned int size0;        // members of the cluster so far (measured runs: the member log clist[0, size0) ends with those n)
};

// Per-CTA shared state.
struct SharedState {
    // cluster mode: cnt[par][q] = entries CTA q of the cluster holds for the level of parity par;
    // every CTA writes its own count into the table of every CTA of the cluster before the barrier
    unsigned int cnt[2][kMaxClusterCtas];
    unsigned int acnt[2];      // cluster mode: own append counters (one per queue buffer)
    unsigned int lcnt[3];      // one-CTA mode: rotating level counters
    Command cmd;
    unsigned long long word;   // broadcast: grid barrier word
    unsigned long long post_acc;   // measured runs: boundary-bond sum of the post-pass (two's complement)
};

enum CommandOp : unsigned int { kCmdCluster = 1, kCmdExit = 2 };

// Registers every CTA carries through the launch.
struct Counters {
    unsigned int gen = 0;                 // grid barrier generation (the host zeroes the control block per launch)
    unsigned int attempts = 0;
    unsigned long long levels_grid = 0, levels_cluster = 0, levels_rebalanced = 0;
    uint32_t widest = 0;
#ifdef WOLFF_PROFILE
    long long prof[4] = {0, 0, 0, 0};   // cycles of a cluster level: head, expansion, CTA barrier + count exchange, cluster barrier
#endif
};

// Grid-wide level loop over the global cluster list (A2-A6, grid mode).  Called by every CTA with
// identical (lo, hi, gen); returns with the window/phase decided by the last CTA to arrive.
template <int DIM, bool POW2, bool SPEC>
__device__ __forceinline__ unsigned int grid_levels(const GrowthParams &p, SharedState &sh, int s0, uint32_t u_lo,
                                                    uint32_t u_hi, uint32_t &lo, uint32_t &hi, Counters &c)
{
    constexpr int T = kGrowthThreads;
    const unsigned int tid = threadIdx.x;
    const unsigned int G = gridDim.x, b = blockIdx.x;
    Control *ctl = p.ctl;
    for (;;) {
        const uint32_t n = hi - lo;
        if (n > c.widest) c.widest = n;
        ++c.levels_grid;
        // contiguous, warp-granular share of the frontier window for this CTA
        const uint32_t per = (((n + G - 1u) / G) + 31u) & ~31u;
        const uint64_t begin64 = (uint64_t)b * per;
        if (begin64 < n) {   // CTA-uniform
            const uint32_t begin = (uint32_t)begin64;
            const uint32_t end = (n - begin < per) ? n : begin + per;
            for (uint32_t pass = begin; pass < end; pass += T) {
                const uint32_t idx = pass + tid;
                const bool valid = idx < end;
                const uint32_t site = valid ? __ldcg(p.clist + lo + idx) : 0u;
                // winners go straight to the global list: one atomic on the tail per warp
                expand_sites<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, valid, site, p.clist, &ctl->tail, p.geo.N, c.attempts);
            }
        }
        // every thread's list writes happen-before thread 0's release (bar.sync, then atom.acq_rel)
        __syncthreads();
        // A6: grid barrier; the last CTA to arrive decides what the next level is
        if (tid == 0) {
            unsigned long long w;
            const unsigned int old = atom_add_acq_rel_u32(&ctl->arrive, 1u);
            if (old == G - 1u) {
                const unsigned int t = ld_relaxed_u32(&ctl->tail);
                const unsigned int width = t - hi;
                const unsigned int phase = (width == 0u) ? kPhaseDone : (width <= p.grid_down ? kPhaseToCluster : kPhaseGrid);
                st_relaxed_u32(&ctl->arrive, 0u);
                w = pack_bar(c.gen + 1u, phase, t);
                st_release_u64(&ctl->bar, w);
            } else {
                w = wait_generation(ctl, c.gen + 1u, true);
            }
            sh.word = w;
        }
        __syncthreads();
        const unsigned long long w = sh.word;
        ++c.gen;
        lo = hi;
        hi = bar_hi(w);
        const unsigned int phase = bar_phase(w);
        if (phase != kPhaseGrid) return phase;
    }
}

enum Outcome : unsigned int { kOutDone = 0, kOutToCta = 1, kOutAbort = 2 };

// Cluster-mode level loop (A2-A6), run by all R CTAs of cluster 0 in lock step.  At entry the
// frontier is what the count row sh.cnt[par][*] says: CTA q holds cnt[par][q] entries in its queue
// buffer `par`.  A level is processed either LOCALLY (every CTA expands its own queue; no remote
// reads) or, when the counts have drifted apart, REBALANCED (the concatenation of all queues is cut
// into R equal contiguous shares; a share's entries are read through distributed shared memory).
// Either way winners go to the CTA's own next queue, the CTA's count is stored into every peer's
// table, and the hardware cluster barrier ends the level.  Frontiers wider than cl_up (or than the
// queues can hold) leave for a grid phase and come back when they narrow to grid_down.
// Returns kOutDone (frontier empty), kOutToCta (frontier <= down: the master CTA has gathered it
// into its buffer 0, sh.lcnt[0] holds the count) or kOutAbort.  `added` accumulates the spins added.
template <int DIM, bool POW2, bool SPEC>
__device__ __forceinline__ unsigned int cluster_levels(const GrowthParams &p, SharedState &sh, uint32_t *q0, uint32_t *q1,
                                                       unsigned int R, unsigned int r, int s0, uint32_t u_lo, uint32_t u_hi,
                                                       unsigned int par, uint32_t size0, unsigned long long &added, Counters &c)
{
    constexpr int T = kGrowthThreads;
    const unsigned int tid = threadIdx.x;
    Control *ctl = p.ctl;
    const uint32_t sh_cnt = smem_addr(&sh.cnt[0][0]);
    const uint32_t sh_q0 = smem_addr(q0), sh_q1 = smem_addr(q1);
    bool first = true;
    for (;;) {
#ifdef WOLFF_PROFILE
        const long long pt0 = clock64();
#endif
        // ---- counts of this level (local shared memory; the peers stored them before the barrier)
        unsigned int cq[kMaxClusterCtas];
        unsigned int n = 0, maxq = 0, mine = 0, before = 0;
#pragma unroll
        for (int q = 0; q < kMaxClusterCtas; ++q) {
            cq[q] = ((unsigned int)q < R) ? sh.cnt[par][q] : 0u;
            before += ((unsigned int)q < r) ? cq[q] : 0u;
            mine = ((unsigned int)q == r) ? cq[q] : mine;
            n += cq[q];
            maxq = cq[q] > maxq ? cq[q] : maxq;
        }
        uint32_t *const cur = par ? q1 : q0;
        uint32_t *const nxt = par ? q0 : q1;
        if (!first) {
            added += n;
            // measured runs: the member log (clist) takes this level's sites; whoever hands a frontier to this loop
            // has logged it already
            if (p.measure) {
                const uint32_t base = size0 + (uint32_t)(added - n) + before;
                for (unsigned int e = tid; e < mine; e += T)
                    if (WOLFF_CHECK(&ctl->error, base + e < p.geo.N, 22)) p.clist[base + e] = cur[e];
            }
        }
        first = false;
        if (n == 0u) return kOutDone;
        if (n > c.widest) c.widest = n;
        const uint32_t sh_cur = par ? sh_q1 : sh_q0;

        if (n <= p.down) {
            // ---- back to one CTA: the master gathers every queue into its buffer 0
            if (r != 0u) return kOutToCta;       // helpers go back to sleep; their queues stay untouched
            uint32_t *const dst = q0;
            // with par == 0 the master's own entries already sit at the front of q0
            unsigned int at = (par == 0u) ? mine : 0u;
            for (unsigned int q = (par == 0u) ? 1u : 0u; q < R; ++q) {
                const unsigned int have = sh.cnt[par][q];
                const uint32_t base = map_to_rank(sh_cur, q);
                for (unsigned int e = tid; e < have; e += T) dst[at + e] = ld_dsmem_u32(base + 4u * e);
                at += have;
            }
            if (tid == 0) { sh.lcnt[0] = n; sh.lcnt[1] = 0u; }
            __syncthreads();
            return kOutToCta;
        }

        const uint32_t per = (((n + R - 1u) / R) + 31u) & ~31u;     // rebalanced share, warp-granular
        const bool fits_local = maxq * (2u * DIM) <= p.qcap;
        const bool fits_shared = per * (2u * DIM) <= p.qcap;
        if (n > p.cl_up || !fits_shared) {
            // ---- grid phase over a window of the global list: [0, n), filled from the queues now -- or, in a measured
            // run, the end of the member log, where this frontier already sits: [S - n, S), S = members so far
            const uint32_t S = size0 + (uint32_t)added;
            const uint32_t lo0 = p.measure ? S - n : 0u, hi0 = p.measure ? S : n;
            if (!p.measure)
                for (unsigned int e = tid; e < mine; e += T) p.clist[before + e] = cur[e];
            if (r == 0u && tid == 0) {
                st_relaxed_u32(&ctl->tail, hi0);
                st_relaxed_u32(&ctl->lo, lo0);
                st_relaxed_u32(reinterpret_cast<unsigned int *>(&ctl->s0), (unsigned int)s0);
                ctl->u = ((unsigned long long)u_hi << 32) | u_lo;
            }
            __threadfence();
            cluster_sync();
            if (r == 0u && tid == 0) st_release_u64(&ctl->bar, pack_bar(c.gen + 1u, kPhaseGrid, hi0));
            ++c.gen;
            uint32_t lo = lo0, hi = hi0;
            const unsigned int out = grid_levels<DIM, POW2, SPEC>(p, sh, s0, u_lo, u_hi, lo, hi, c);
            added += (unsigned long long)(hi - hi0);
            if (out == kPhaseAbort) return kOutAbort;
            if (out == kPhaseDone) return kOutDone;
            // ---- frontier narrowed: window [lo, hi) goes back into the cluster's queues, equal shares
            const unsigned int m = hi - lo;
            const unsigned int share = (m + R - 1u) / R;
            const unsigned int b0 = r * share < m ? r * share : m;
            const unsigned int b1 = b0 + share < m ? b0 + share : m;
            for (unsigned int e = b0 + tid; e < b1; e += T) q0[e - b0] = __ldcg(p.clist + lo + e);
            if (tid < R) {
                const unsigned int a0 = tid * share < m ? tid * share : m;
                const unsigned int a1 = a0 + share < m ? a0 + share : m;
                sh.cnt[0][tid] = a1 - a0;
            }
            if (tid == 0) { sh.acnt[0] = 0u; sh.acnt[1] = 0u; }
            __syncthreads();
            par = 0u;
            first = true;        // these entries were counted by the grid phase
            continue;
        }

        // ---- one cluster level
        ++c.levels_cluster;
        const bool local = fits_local && maxq <= (2u * per > p.bal_min ? 2u * per : p.bal_min);
        unsigned int *const dst_count = &sh.acnt[par ^ 1u];
#ifdef WOLFF_PROFILE
        const long long pt1 = clock64();
#endif
        if (local) {
            for (unsigned int pass = 0; pass < mine; pass += T) {
                const unsigned int idx = pass + tid;
                const bool valid = idx < mine;
                const uint32_t site = valid ? cur[idx] : 0u;
                expand_sites<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, valid, site, nxt, dst_count, p.qcap, c.attempts);
            }
        } else {
            ++c.levels_rebalanced;
            const unsigned int begin = r * per < n ? r * per : n;
            const unsigned int end = begin + per < n ? begin + per : n;
            for (unsigned int pass = begin; pass < end; pass += T) {
                const unsigned int idx = pass + tid;
                const bool valid = idx < end;
                uint32_t site = 0u;
                if (valid) {
                    unsigned int owner = 0, off = idx;
#pragma unroll
                    for (int q = 0; q < kMaxClusterCtas - 1; ++q) {
                        const bool beyond = ((unsigned int)q == owner) && off >= cq[q];
                        off -= beyond ? cq[q] : 0u;
                        owner += beyond ? 1u : 0u;
                    }
                    site = (owner == r) ? cur[off] : ld_dsmem_u32(map_to_rank(sh_cur, owner) + 4u * off);
                }
                expand_sites<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, valid, site, nxt, dst_count, p.qcap, c.attempts);
            }
        }
#ifdef WOLFF_PROFILE
        const long long pt2 = clock64();
#endif
        __syncthreads();                           // all appends of this CTA are done
        if (tid < R) st_dsmem_u32(map_to_rank(sh_cnt + 4u * ((par ^ 1u) * kMaxClusterCtas + r), tid), *dst_count);
        if (tid == 32) sh.acnt[par] = 0u;          // the buffer this level read becomes the next append target
#ifdef WOLFF_PROFILE
        const long long pt3 = clock64();
#endif
        cluster_sync();                            // A6: level barrier of the cluster
#ifdef WOLFF_PROFILE
        c.prof[0] += pt1 - pt0; c.prof[1] += pt2 - pt1; c.prof[2] += pt3 - pt2; c.prof[3] += clock64() - pt3;
#endif
        par ^= 1u;
    }
}

// Store the command block into CTA `target` of the cluster (called by the master, one lane per target).
__device__ __forceinline__ void send_command(SharedState &sh, unsigned int target, unsigned int op, unsigned int par, int s0,
                                             uint32_t u_lo, uint32_t u_hi, unsigned int n, unsigned int size0)
{
    const uint32_t cb = map_to_rank(smem_addr(&sh.cmd), target);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, op), op);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, par), par);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, s0), (unsigned int)s0);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, u_lo), u_lo);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, u_hi), u_hi);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, n), n);
    st_dsmem_u32(cb + (uint32_t)offsetof(Command, size0), size0);
}

// Entry into a cluster phase, run by every CTA of cluster 0 after the barrier that delivered the
// command: build the count row (only the master holds entries) and clear the append counters.
__device__ __forceinline__ void begin_cluster_phase(SharedState &sh, unsigned int par, unsigned int n)
{
    const unsigned int tid = threadIdx.x;
    if (tid < kMaxClusterCtas) sh.cnt[par][tid] = (tid == 0u) ? n : 0u;
    if (tid == 32) { sh.acnt[0] = 0u; sh.acnt[1] = 0u; }
    __syncthreads();
}

template <int DIM, bool POW2, bool SPEC>
__global__ void __launch_bounds__(kGrowthThreads, 1) growth_kernel(const GrowthParams p)
{
    constexpr int T = kGrowthThreads;
    extern __shared__ __align__(16) uint32_t smem_q[];   // two queue buffers of p.qcap entries
    __shared__ SharedState sh;
    uint32_t *const q0 = smem_q;
    uint32_t *const q1 = smem_q + p.qcap;
    const unsigned int tid = threadIdx.x;
    const unsigned int R = cluster_nctarank(), r = cluster_ctarank();
    const bool in_cluster0 = cluster_id_x() == 0u;
    Control *ctl = p.ctl;
    Counters c;
    // sticky error flag: an earlier launch of this handle was aborted and the host has not yet looked
    if (ld_relaxed_u32(&ctl->error) != 0u) return;

    if (!in_cluster0) {
        // ---------------------------------------------------------------- worker CTAs: grid phases only
        for (;;) {
            if (tid == 0) sh.word = wait_generation(ctl, c.gen + 1u, false);
            __syncthreads();
            const unsigned long long w = sh.word;
            __syncthreads();
            ++c.gen;
            if (bar_phase(w) != kPhaseGrid) break;   // exit or abort
            uint32_t lo = ld_relaxed_u32(&ctl->lo), hi = bar_hi(w);
            const int s0 = (int)ld_relaxed_u32(reinterpret_cast<unsigned int *>(&ctl->s0));
            const unsigned long long u = __ldcg(&ctl->u);
            const unsigned int out = grid_levels<DIM, POW2, SPEC>(p, sh, s0, (uint32_t)u, (uint32_t)(u >> 32), lo, hi, c);
            if (out == kPhaseAbort) break;
        }
        if (c.attempts) atomicAdd(&ctl->stats[7], (unsigned long long)c.attempts);
        return;
    }

    if (r != 0u) {
        // ---------------------------------------------------------------- helper CTAs of cluster 0
        // Asleep in the hardware cluster barrier until the master arrives with a command.
        for (;;) {
            cluster_sync();
            if (sh.cmd.op != kCmdCluster) break;
            const unsigned int par = sh.cmd.par;
            const int s0 = sh.cmd.s0;
            const uint32_t u_lo = sh.cmd.u_lo, u_hi = sh.cmd.u_hi;
            begin_cluster_phase(sh, par, sh.cmd.n);
            unsigned long long added = 0;
            const unsigned int out = cluster_levels<DIM, POW2, SPEC>(p, sh, q0, q1, R, r, s0, u_lo, u_hi, par, sh.cmd.size0, added, c);
            if (out == kOutAbort) break;
        }
        if (c.attempts) atomicAdd(&ctl->stats[7], (unsigned long long)c.attempts);
        return;
    }

    // -------------------------------------------------------------------- master CTA: the update loop
    unsigned long long flipped = 0, levels_cta = 0, to_cluster = 0;
    bool aborted = false;
    // measured runs (thread 0): running E and M, from the whole-lattice reduction the host queued before this launch
    long long runE = 0, runM = 0;
    Moments mom;
    if (p.measure && tid == 0) { runE = ctl->E; runM = ctl->M; mom.load(ctl->moments); }
    for (unsigned long long k = 0; k < p.n_updates && !aborted; ++k) {
        const unsigned long long u = p.u0 + k;
        const uint32_t u_lo = (uint32_t)u, u_hi = (uint32_t)(u >> 32);
        unsigned long long t_start = 0;
        // A1: seed draw (reading R8) and initial flip
        if (tid == 0) {
            t_start = globaltimer_ns();
            const uint4 x = philox4x32_10(0u, kDomainSite, u_lo, u_hi, p.key0, p.key1);
            const unsigned long long rr = (unsigned long long)x.x | ((unsigned long long)x.y << 32);
            const uint32_t i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
            const int s = load_spin_l2(p.spins, i0);
            claim_with_bits(p.spins, i0, s, p.claim_bits);
            if (p.measure) p.clist[0] = i0;
            q0[0] = i0;
            sh.lcnt[0] = 1u;
            sh.lcnt[1] = 0u;
            sh.cmd.s0 = s;
        }
        __syncthreads();
        const int s0 = sh.cmd.s0;
        unsigned long long size = 1;
        unsigned int lvl = 0;        // level counter modulo 3 (counter slot)
        uint32_t *cur = q0, *nxt = q1;
        for (;;) {
            const unsigned int n = sh.lcnt[lvl];
            if (n == 0u) break;
            if (n > c.widest) c.widest = n;
            if (n > p.up) {
                // ---- the frontier outgrew one CTA: wake the cluster
                ++to_cluster;
                const unsigned int par = (cur == q1) ? 1u : 0u;
                __syncthreads();                                      // everybody has read lcnt/cmd of this level
                if (tid < R) send_command(sh, tid, kCmdCluster, par, s0, u_lo, u_hi, n, (unsigned int)size);
                cluster_sync();
                begin_cluster_phase(sh, par, n);
                unsigned long long added = 0;
                const unsigned int out = cluster_levels<DIM, POW2, SPEC>(p, sh, q0, q1, R, 0u, s0, u_lo, u_hi, par, (uint32_t)size, added, c);
                size += added;
                if (out == kOutAbort) { aborted = true; break; }
                if (out == kOutDone) break;
                lvl = 0; cur = q0; nxt = q1;                          // kOutToCta: frontier gathered into q0, lcnt[0] set
                continue;
            }
            // ---- one-CTA level: shared-memory queues, __syncthreads only
            ++levels_cta;
            const unsigned int lvl1 = (lvl == 2u) ? 0u : lvl + 1u;
            const unsigned int lvl2 = (lvl1 == 2u) ? 0u : lvl1 + 1u;
            if (tid == 0) sh.lcnt[lvl2] = 0u;
            for (unsigned int pass = 0; pass < n; pass += T) {
                const unsigned int idx = pass + tid;
                const bool valid = idx < n;
                const uint32_t site = valid ? cur[idx] : 0u;
                expand_sites<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, valid, site, nxt, &sh.lcnt[lvl1], p.qcap, c.attempts);
            }
            __syncthreads();
            const unsigned int n1 = sh.lcnt[lvl1];
            if (p.measure)                                            // member log of a measured run
                for (unsigned int e = tid; e < n1; e += T)
                    if (WOLFF_CHECK(&ctl->error, (uint32_t)size + e < p.geo.N, 21)) p.clist[(uint32_t)size + e] = nxt[e];
            size += n1;
            lvl = lvl1;
            uint32_t *t = cur; cur = nxt; nxt = t;
        }
        if (p.measure && !aborted) {
            // ---- post-pass of a measured update: dE from the cluster's boundary bonds (every member still carries its
            // mark), then the marks go: members get their plain value -s0.  M changes by -2 s0 |C|.
            if (tid == 0) sh.post_acc = 0ull;
            __syncthreads();
            int part = boundary_partial<DIM, POW2>(p.geo, p.spins, p.clist, s0, (uint32_t)size, tid, (uint32_t)T);
            part = __reduce_add_sync(kFullMask, part);
            if ((tid & 31u) == 0u && part != 0) atomicAdd(&sh.post_acc, (unsigned long long)(long long)part);
            __syncthreads();
            const int8_t plain = (int8_t)(-s0);
            for (uint32_t e = tid; e < (uint32_t)size; e += T) p.spins[__ldcg(p.clist + e)] = plain;
            if (tid == 0) {
                runE += 2ll * (long long)sh.post_acc;
                runM -= 2ll * (long long)s0 * (long long)size;
                p.E_log[k] = runE;
                p.M_log[k] = runM;
                mom.add(runE, runM);
            }
        }
        // A7: epilogue
        if (tid == 0) {
            p.sizes[k] = (uint32_t)size;
            const unsigned long long dt = globaltimer_ns() - t_start;
            p.ns_log[k] = dt > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)dt;
        }
        flipped += size;
        __syncthreads();
    }
    if (p.measure && tid == 0) { ctl->E = runE; ctl->M = runM; mom.store(ctl->moments); }
    if (!aborted) {
        if (tid == 0) st_release_u64(&ctl->bar, pack_bar(c.gen + 1u, kPhaseExit, 0u));   // workers leave
        if (tid < R) send_command(sh, tid, kCmdExit, 0u, 0, 0u, 0u, 0u, 0u);                 // helpers leave
        cluster_sync();
    }
    if (tid == 0) {
        ctl->stats[0] = p.n_updates;
        ctl->stats[1] = flipped;
        ctl->stats[2] = levels_cta;
        ctl->stats[3] = c.levels_cluster;
        ctl->stats[4] = c.levels_grid;
        ctl->stats[5] = to_cluster;
        ctl->stats[6] = c.levels_rebalanced;
        ctl->stats[8] = c.widest;
#ifdef WOLFF_PROFILE
        for (int k = 0; k < 4; ++k) ctl->stats[10 + k] = (unsigned long long)c.prof[k];
#endif
    }
    if (c.attempts) atomicAdd(&ctl->stats[7], (unsigned long long)c.attempts);
}

template <int DIM, bool POW2, bool SPEC>
cudaError_t prepare_one(const GrowthLaunch &l, int *max_clusters)
{
    const void *fn = reinterpret_cast<const void *>(&growth_kernel<DIM, POW2, SPEC>);
    cudaError_t e = allow_max_dynamic_smem(fn);
    if (e != cudaSuccess) return e;
    if (l.cluster_ctas > 8) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    if (max_clusters) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned int)l.cluster_ctas);
        cfg.blockDim = dim3(kGrowthThreads);
        cfg.dynamicSmemBytes = l.smem_bytes;
        cudaLaunchAttribute attr;
        attr.id = cudaLaunchAttributeClusterDimension;
        attr.val.clusterDim.x = (unsigned int)l.cluster_ctas;
        attr.val.clusterDim.y = 1;
        attr.val.clusterDim.z = 1;
        cfg.attrs = &attr;
        cfg.numAttrs = 1;
        e = cudaOccupancyMaxActiveClusters(max_clusters, growth_kernel<DIM, POW2, SPEC>, &cfg);
    }
    return e;
}

template <int DIM, bool POW2, bool SPEC>
cudaError_t launch_one(const GrowthParams &p, const GrowthLaunch &l, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned int)l.grid_ctas);
    cfg.blockDim = dim3(kGrowthThreads);
    cfg.dynamicSmemBytes = l.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attrs[2];
    attrs[0].id = cudaLaunchAttributeClusterDimension;
    attrs[0].val.clusterDim.x = (unsigned int)l.cluster_ctas;
    attrs[0].val.clusterDim.y = 1;
    attrs[0].val.clusterDim.z = 1;
    attrs[1].id = cudaLaunchAttributeCooperative;     // all CTAs co-resident: the grid barrier needs it
    attrs[1].val.cooperative = 1;
    cfg.attrs = attrs;
    cfg.numAttrs = l.cooperative ? 2 : 1;
    // per-process kernel attributes may have been changed by another handle since this one derived its shape
    const cudaError_t ea = prepare_one<DIM, POW2, SPEC>(l, nullptr);
    if (ea != cudaSuccess) return ea;
    return cudaLaunchKernelEx(&cfg, growth_kernel<DIM, POW2, SPEC>, p);
}

}  // namespace

#define WOLFF_GROWTH_DISPATCH(CALL)                                                     \
    do {                                                                               \
        if (dim == 2) {                                                                \
            if (pow2) return l.spec ? CALL(2, true, true) : CALL(2, true, false);      \
            return l.spec ? CALL(2, false, true) : CALL(2, false, false);              \
        }                                                                              \
        if (pow2) return l.spec ? CALL(3, true, true) : CALL(3, true, false);          \
        return l.spec ? CALL(3, false, true) : CALL(3, false, false);                  \
    } while (0)

cudaError_t launch_growth(const GrowthParams &p, int dim, const GrowthLaunch &l, cudaStream_t stream)
{
    const bool pow2 = p.geo.pow2 != 0u;
#define WOLFF_CALL(D, P, S) launch_one<D, P, S>(p, l, stream)
    WOLFF_GROWTH_DISPATCH(WOLFF_CALL);
#undef WOLFF_CALL
}

cudaError_t growth_max_clusters(int dim, bool pow2, const GrowthLaunch &l, int *max_clusters)
{
#define WOLFF_CALL(D, P, S) prepare_one<D, P, S>(l, max_clusters)
    WOLFF_GROWTH_DISPATCH(WOLFF_CALL);
#undef WOLFF_CALL
}

}  // namespace wolff
