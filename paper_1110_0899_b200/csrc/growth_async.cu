// growth_async.cu -- the barrier-free cluster-growth kernel (8(f) row 2).
//
// Same computation as growth.cu: n_updates Wolff single-cluster updates (steps i-v),
// every newly added spin expanded by one thread (step iii').  What is different is
// row A6, the hand-over of newly added spins to the threads that expand them.  The paper synchronises
// all blocks after every direction of every pass and names that wait as its
// bottleneck; growth.cu still has one barrier per BFS level.  Because a bond variable
// here is a function of (seed, update, bond), the cluster is the connected component of the seed site
// whatever the order of expansion, so no level structure is needed at all:
//
//   - the lattice is cut into tiles of 2^tile_log sites per side; tile (tx,ty,tz) belongs to CTA
//     (tx + A*ty + B*tz) mod G, and a site is always expanded by the CTA that owns its tile;
//   - a warp that claims neighbours inside the tile keeps up to 32 of them and expands them itself in
//     its next pass (no queue, no barrier: the dependent chain of one hop is Philox -> L2 atomic ->
//     ballot); what does not fit goes to the CTA's shared-memory ring, which idle warps of the CTA drain;
//   - a claimed site of another tile goes to the owner's INBOX, a segment of one global array with room
//     for every site the owner owns, so a push never waits (one L2 atomicAdd + one store); a service
//     warp per CTA moves arrivals into the ring;
//   - termination: CTA c publishes gdone[c] = "inbox entries whose whole local progeny is processed"
//     whenever its ring runs dry; a monitor warp reads all gdone[], then all gtail[] (entries ever
//     pushed); equal sums mean nothing is queued, in flight or being expanded anywhere.
//
// A small frontier is spatially compact, hence in one or a few tiles: the chain stays inside one SM.
// A wide frontier is spread over many tiles, hence over many SMs: L2 request throughput scales.
// Small clusters never leave CTA 0: it grows the first levels alone with __syncthreads (one-CTA tier,
// as in growth.cu) and only publishes a phase to the other CTAs when the frontier outgrows `up`.
#include "expand.cuh"
#include "internal.h"

namespace wolff {
namespace {

constexpr uint32_t kEmpty = 0xFFFFFFFFu;
constexpr int kT = kGrowthThreads;
constexpr int kWarps = kT / 32;
constexpr int kStage = 32 * 6;              // winners one warp can produce in one pass (2*dim per lane)
constexpr unsigned int kInboxPoll = 8;      // inbox slots the service warp looks at per pass

enum Op : unsigned int { kOpNone = 0, kOpGo = 1, kOpFin = 2, kOpExit = 3, kOpAbort = 4 };

__device__ __forceinline__ unsigned long long pack_state(unsigned int seq, unsigned int op, int s0)
{
    return ((unsigned long long)seq << 32) | (s0 < 0 ? 0x100ull : 0ull) | (unsigned long long)op;
}
__device__ __forceinline__ unsigned int state_seq(unsigned long long w) { return (unsigned int)(w >> 32); }
__device__ __forceinline__ unsigned int state_op(unsigned long long w) { return (unsigned int)w & 0xFFu; }
__device__ __forceinline__ int state_s0(unsigned long long w) { return (w & 0x100ull) ? -1 : 1; }

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

__device__ __forceinline__ unsigned int ld_vol(const unsigned int *p) { return *reinterpret_cast<const volatile unsigned int *>(p); }
__device__ __forceinline__ void st_vol(unsigned int *p, unsigned int v) { *reinterpret_cast<volatile unsigned int *>(p) = v; }
__device__ __forceinline__ unsigned long long ld_vol64(const unsigned long long *p)
{
    return *reinterpret_cast<const volatile unsigned long long *>(p);
}
__device__ __forceinline__ void st_vol64(unsigned long long *p, unsigned long long v)
{
    *reinterpret_cast<volatile unsigned long long *>(p) = v;
}
__device__ __forceinline__ void st_relaxed_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Per-CTA shared state.
struct AShared {
    // ring: entries [head, tail) wait for a consumer; `retired` counts ring entries whose warp ran dry
    unsigned int head, tail, retired;
    unsigned int added;                 // spins claimed by this CTA's warps, not yet flushed to ctl->added
    unsigned long long ihead;           // inbox entries moved into the ring (written by the service warp only)
    unsigned long long last_pub;        // largest ihead published to gdone[]
    unsigned int stop;                  // the phase is over
    int s0;                             // seed spin of the running update
    uint32_t u_lo, u_hi;                // its index
    unsigned int seq;                   // 2g: the running phase
    unsigned int lcnt[3];               // one-CTA tier: rotating level counters
    unsigned long long word;            // broadcast slot
    unsigned long long size_acc;
};

struct Tally {
    unsigned int attempts = 0;          // claim atomics (per lane)
    unsigned int inbox_pushes = 0;      // sites handed to another CTA or spilled to the own inbox (per lane)
    unsigned int ring_pushes = 0;       // sites handed to the ring (per lane)
    unsigned int passes = 0;            // warp passes (lane 0)
};

template <int DIM, bool POW2>
__device__ __forceinline__ unsigned int owner_of(const AsyncParams &ap, uint32_t j, unsigned int G)
{
    uint32_t x, y, z;
    site_coords<DIM, POW2>(ap.g.geo, j, x, y, z);
    uint32_t t = (x >> ap.tile_log) + ap.hashA * (y >> ap.tile_log);
    if (DIM == 3) t += ap.hashB * (z >> ap.tile_log);
    return t % G;
}

// Store entry `pos` (a running count) of CTA o's inbox.  The slot is empty: within one update at most
// cap(o) sites are ever pushed to o, and every earlier entry was taken before its update ended.
__device__ __forceinline__ void inbox_store(const AsyncParams &ap, unsigned int o, unsigned long long pos, uint32_t v)
{
    const uint32_t off = __ldg(ap.seg + o);
    const uint32_t cap = __ldg(ap.seg + o + 1) - off;
    st_relaxed_u32(ap.inbox + off + (uint32_t)(pos % cap), v);
}

// Reserve n consecutive ring entries; false when the ring cannot take them (entries [head, head+cap) only).
__device__ __forceinline__ bool ring_reserve(AShared &sh, uint32_t cap, unsigned int n, unsigned int &base)
{
    unsigned int t = ld_vol(&sh.tail);
    for (;;) {
        const unsigned int h = ld_vol(&sh.head);
        if (t + n - h > cap) return false;
        const unsigned int seen = atomicCAS(&sh.tail, t, t + n);
        if (seen == t) { base = t; return true; }
        t = seen;
    }
}

// Fill a reserved ring slot.  The previous lap's entry of this slot has been ACQUIRED (head moved past
// it) but may not have been read yet; in that case the exchange hands it back, its reader takes our
// value instead, and we re-install the old one as soon as the slot is empty again.
__device__ __forceinline__ void ring_put(uint32_t *slot, uint32_t v)
{
    const uint32_t old = atomicExch(slot, v);
    if (old != kEmpty) {
        while (atomicCAS(slot, kEmpty, old) != kEmpty) { }
    }
}

__device__ __forceinline__ void raise_abort(Control *ctl, unsigned int code)
{
    st_relaxed_u32(&ctl->error, code);
    st_release_u64(&ctl->state, pack_state(0xFFFFFFFFu, kOpAbort, 1));
}

// ------------------------------------------------------------------------------------------ consumer warp
// Expands sites owned by this CTA until the phase is over.
template <int DIM, bool POW2, bool SPEC>
__device__ __forceinline__ void consumer_warp(const AsyncParams &ap, AShared &sh, uint32_t *ring, uint32_t *stage,
                                              unsigned int c, unsigned int G, Tally &tl)
{
    const GrowthParams &p = ap.g;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int bit = 1u << lane, lt = bit - 1u;
    const uint32_t rmask = ap.ring_cap - 1u;
    const int s0 = sh.s0;
    const uint32_t u_lo = sh.u_lo, u_hi = sh.u_hi;
    const uint32_t tag = ((sh.seq >> 1) & 1u) << 31;      // phase parity carried by inbox entries
    const uint32_t tmask = (1u << ap.tile_log) - 1u;
    const uint32_t Lm1 = p.geo.L - 1u;
    uint32_t site = 0;
    bool have = false;
    unsigned int acq = 0;        // ring entries acquired since the last retire (warp-uniform)
    unsigned int mywon = 0;      // spins this lane claimed since the last retire

    for (;;) {
        if (!__any_sync(kFullMask, have)) {
            if (acq) {
                // ---- the warp ran dry: retire what it took from the ring, then test the CTA for quiescence
                const unsigned int w = __reduce_add_sync(kFullMask, mywon);
                if (lane == 0) {
                    if (w) atomicAdd(&sh.added, w);
                    __threadfence_block();
                    atomicAdd(&sh.retired, acq);
                    __threadfence_block();
                    const unsigned long long I = ld_vol64(&sh.ihead);
                    const unsigned int r = ld_vol(&sh.retired);
                    const unsigned int t = ld_vol(&sh.tail);
                    if (r == t && I > ld_vol64(&sh.last_pub)) {
                        // every ring entry ever pushed here is retired: inbox entries < I are done for good
                        const unsigned int a = atomicExch(&sh.added, 0u);
                        if (a) atomicAdd(&p.ctl->added, (unsigned long long)a);
                        __threadfence();
                        atomicMax(&ap.gdone[c], I);
                        atomicMax(&sh.last_pub, I);
                    }
                }
                acq = 0;
                mywon = 0;
            }
            // ---- take up to 32 entries from the ring
            unsigned int k = 0, h = 0;
            if (lane == 0) {
                for (;;) {
                    const unsigned int t = ld_vol(&sh.tail);
                    h = ld_vol(&sh.head);
                    if (t != h) {
                        k = t - h < 32u ? t - h : 32u;
                        if (atomicCAS(&sh.head, h, h + k) == h) break;
                        k = 0;
                        continue;
                    }
                    if (ld_vol(&sh.stop)) break;
                }
            }
            k = __shfl_sync(kFullMask, k, 0);
            h = __shfl_sync(kFullMask, h, 0);
            if (k == 0) break;                                   // phase over
            if (lane < k) {
                uint32_t *slot = ring + ((h + lane) & rmask);
                unsigned int spins = 0;
                do {
                    site = atomicExch(slot, kEmpty);             // the producer reserved it; its store is on the way
                    if (site == kEmpty && ++spins > (1u << 26)) { raise_abort(p.ctl, 4u); site = 0u; }
                } while (site == kEmpty);
                have = true;
            }
            acq += k;
        }

        // ---- A2-A4 for up to 32 sites
        uint32_t nbr[2 * DIM];
        unsigned int won;
        uint32_t x, y, z;
        claim_neighbours<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, have, site, nbr, won, x, y, z, tl.attempts);
        mywon += __popc(won);
        if (lane == 0) ++tl.passes;

        // which winners lie in another tile?
        unsigned int cross = 0;
        if (won) {
            cross |= (((x & tmask) == tmask) || x == Lm1) ? 1u : 0u;
            cross |= ((x & tmask) == 0u) ? 2u : 0u;
            cross |= (((y & tmask) == tmask) || y == Lm1) ? 4u : 0u;
            cross |= ((y & tmask) == 0u) ? 8u : 0u;
            if (DIM == 3) {
                cross |= (((z & tmask) == tmask) || z == Lm1) ? 16u : 0u;
                cross |= ((z & tmask) == 0u) ? 32u : 0u;
            }
        }
        const unsigned int wl = won & ~cross, wr = won & cross;

        // ---- A5, inside the tile: compact the winners; the first 32 are this warp's next pass
        unsigned int total = 0;
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) {
            const bool mine = (wl >> k) & 1u;
            const unsigned int b = __ballot_sync(kFullMask, mine);
            if (mine) stage[total + __popc(b & lt)] = nbr[k];
            total += __popc(b);
        }
        const bool any_remote = __any_sync(kFullMask, wr != 0u);
        __syncwarp();
        have = lane < total;
        if (have) site = stage[lane];
        if (total > 32u) {
            // the rest goes to the ring (or, if the ring is full, to the own inbox, which cannot be)
            const unsigned int ex = total - 32u;
            unsigned int base = 0, ok = 0;
            if (lane == 0) ok = ring_reserve(sh, ap.ring_cap, ex, base) ? 1u : 0u;
            ok = __shfl_sync(kFullMask, ok, 0);
            base = __shfl_sync(kFullMask, base, 0);
            if (ok) {
                for (unsigned int j = lane; j < ex; j += 32u) { ring_put(ring + ((base + j) & rmask), stage[32u + j]); ++tl.ring_pushes; }
            } else {
                unsigned long long pos = 0;
                if (lane == 0) pos = atomicAdd(&ap.gtail[c], (unsigned long long)ex);
                pos = __shfl_sync(kFullMask, pos, 0);
                for (unsigned int j = lane; j < ex; j += 32u) { inbox_store(ap, c, pos + j, stage[32u + j] | tag); ++tl.inbox_pushes; }
            }
        }
        // ---- A5, across a tile edge (rare): one push per winner
        if (any_remote) {
#pragma unroll
            for (int k = 0; k < 2 * DIM; ++k) {
                if ((wr >> k) & 1u) {
                    const uint32_t j = nbr[k];
                    const unsigned int o = owner_of<DIM, POW2>(ap, j, G);
                    unsigned int base;
                    if (o == c && ring_reserve(sh, ap.ring_cap, 1u, base)) {
                        ring_put(ring + (base & rmask), j);
                        ++tl.ring_pushes;
                    } else {
                        const unsigned long long pos = atomicAdd(&ap.gtail[o], 1ull);
                        inbox_store(ap, o, pos, j | tag);
                        ++tl.inbox_pushes;
                    }
                }
            }
        }
        __syncwarp();      // stage[] is rewritten in the next pass
    }
}

// ------------------------------------------------------------------------------------------ service warp
// Moves arrivals from the CTA's inbox into its ring and watches the phase word.
__device__ __forceinline__ void service_warp(const AsyncParams &ap, AShared &sh, uint32_t *ring, unsigned int c)
{
    const unsigned int lane = threadIdx.x & 31u;
    Control *ctl = ap.g.ctl;
    const uint32_t rmask = ap.ring_cap - 1u;
    const uint32_t off = __ldg(ap.seg + c);
    const uint32_t cap = __ldg(ap.seg + c + 1) - off;
    const unsigned int seq = sh.seq;
    const uint32_t par = (seq >> 1) & 1u;
    unsigned int passes = 0;
    for (;;) {
        unsigned long long st = 0;
        if (lane == 0) st = ld_relaxed_u64(&ctl->state);
        const unsigned long long ih = ld_vol64(&sh.ihead);
        uint32_t *slot = nullptr;
        uint32_t v = kEmpty;
        if (lane < kInboxPoll && lane < cap) {
            slot = ap.inbox + off + (uint32_t)((ih + lane) % cap);
            v = ld_relaxed_u32(slot);
        }
        const bool ok = (v != kEmpty) && ((v >> 31) == par);
        const unsigned int b = __ballot_sync(kFullMask, ok);
        const unsigned int k = (unsigned int)__ffs((int)~b) - 1u;   // arrivals in order: the contiguous prefix
        st = __shfl_sync(kFullMask, st, 0);
        if (state_seq(st) != seq) break;                  // the phase is over (or the launch is aborted)
        if (k != 0u) {
            uint32_t item = 0;
            if (lane < k) item = atomicExch(slot, kEmpty) & 0x7FFFFFFFu;
            unsigned int base = 0, good = 1;
            if (lane == 0) {
                unsigned int tries = 0;
                while (!ring_reserve(sh, ap.ring_cap, k, base)) {   // consumers drain the ring without waiting for us
                    if ((++tries & 0xFFFu) == 0u && ld_relaxed_u32(&ctl->error) != 0u) { good = 0; break; }
                }
            }
            good = __shfl_sync(kFullMask, good, 0);
            if (!good) break;
            base = __shfl_sync(kFullMask, base, 0);
            if (lane < k) ring_put(ring + ((base + lane) & rmask), item);
            __threadfence_block();                        // the ring push is visible before ihead moves
            __syncwarp();
            if (lane == 0) st_vol64(&sh.ihead, ih + k);
            __syncwarp();
            continue;
        }
        if ((++passes & 0x3FFu) == 0u && ld_relaxed_u32(&ctl->error) != 0u) break;
    }
    __syncwarp();
    if (lane == 0) st_vol(&sh.stop, 1u);
}

// ------------------------------------------------------------------------------------------ monitor warp
// CTA 0 only.  Termination: read every gdone[], then every gtail[]; both only grow, gdone never
// overtakes gtail, and a site is pushed (gtail) before the entry that caused it is done (gdone), so
// equal sums mean that at the moment between the two passes nothing was queued or being expanded.
__device__ __forceinline__ void monitor_warp(const AsyncParams &ap, AShared &sh, unsigned int G)
{
    const unsigned int lane = threadIdx.x & 31u;
    Control *ctl = ap.g.ctl;
    const unsigned int seq = sh.seq;
    const unsigned long long t0 = globaltimer_ns();
    unsigned int passes = 0;
    bool aborted = false;
    for (;;) {
        unsigned long long d = 0, t = 0;
        for (unsigned int cc = lane; cc < G; cc += 32u) d += ld_relaxed_u64(ap.gdone + cc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) d += __shfl_xor_sync(kFullMask, d, o);
        // the second pass is issued only after the first has returned (its addresses depend on it)
        const unsigned long long *gt = ap.gtail + ((unsigned int)d & ap.zero);
        for (unsigned int cc = lane; cc < G; cc += 32u) t += ld_relaxed_u64(gt + cc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(kFullMask, t, o);
        if (d == t) break;
        if ((++passes & 0xFFu) == 0u) {
            unsigned int bad = 0;
            if (lane == 0) {
                if (ld_relaxed_u32(&ctl->error) != 0u) bad = 1;
                else if (globaltimer_ns() - t0 > ap.watchdog_ns) { raise_abort(ctl, 3u); bad = 1; }
            }
            if (__shfl_sync(kFullMask, bad, 0)) { aborted = true; break; }
        }
    }
    if (!aborted) {
        fence_acq_rel_gpu();
        if (lane == 0) st_release_u64(&ctl->state, pack_state(seq + 1u, kOpFin, 1));
    }
}

template <int DIM, bool POW2, bool SPEC>
__device__ __forceinline__ void run_phase(const AsyncParams &ap, AShared &sh, uint32_t *ring, uint32_t *stage_all,
                                          unsigned int c, unsigned int G, Tally &tl)
{
    const unsigned int warp = threadIdx.x >> 5;
    if (warp == 0u) service_warp(ap, sh, ring, c);
    else if (c == 0u && warp == 1u) monitor_warp(ap, sh, G);
    else consumer_warp<DIM, POW2, SPEC>(ap, sh, ring, stage_all + warp * kStage, c, G, tl);
    __syncthreads();
}

template <int DIM, bool POW2, bool SPEC>
__global__ void __launch_bounds__(kT, 1) growth_async_kernel(const AsyncParams ap)
{
    extern __shared__ __align__(16) uint32_t smem_a[];
    __shared__ AShared sh;
    uint32_t *const ring = smem_a;
    uint32_t *const stage_all = ring + ap.ring_cap;
    uint32_t *const q0 = stage_all + kWarps * kStage;
    uint32_t *const q1 = q0 + ap.lvl_cap;
    const GrowthParams &p = ap.g;
    const unsigned int tid = threadIdx.x;
    const unsigned int c = blockIdx.x, G = gridDim.x;
    Control *ctl = p.ctl;
    Tally tl;

    for (unsigned int i = tid; i < ap.ring_cap; i += kT) ring[i] = kEmpty;
    if (tid == 0) {
        sh.head = sh.tail = sh.retired = sh.added = 0u;
        sh.ihead = 0ull;
        sh.last_pub = 0ull;
        sh.stop = 0u;
        sh.size_acc = 0ull;
    }
    __syncthreads();

    if (c != 0u) {
        // ------------------------------------------------------------------ helper CTAs: phases only
        unsigned int acked = 0;       // phases this CTA has reported as over
        unsigned int last_run = 0;    // seq of the last phase this CTA took part in
        for (;;) {
            if (tid == 0) {
                unsigned int ns = 20;
                unsigned long long w;
                for (;;) {
                    w = ld_relaxed_u64(&ctl->state);
                    const unsigned int s = state_seq(w), op = state_op(w);
                    if (op == kOpExit || op == kOpAbort) break;
                    // phase g is over once seq >= 2g+1; CTA 0 reuses a phase parity only after everybody said so
                    const unsigned int f = s ? (s - 1u) >> 1 : 0u;
                    if (f > acked) { atomicAdd(&ctl->acks, (unsigned long long)(f - acked)); acked = f; }
                    if (op == kOpGo && s > last_run) break;
                    __nanosleep(ns);
                    if (ns < 320u) ns += ns >> 1;
                }
                fence_acq_rel_gpu();
                sh.word = w;
                if (state_op(w) == kOpGo) {
                    const unsigned long long u = ld_relaxed_u64(&ctl->u);
                    sh.s0 = state_s0(w);
                    sh.u_lo = (uint32_t)u;
                    sh.u_hi = (uint32_t)(u >> 32);
                    sh.seq = state_seq(w);
                    sh.stop = 0u;
                }
            }
            __syncthreads();
            const unsigned long long w = sh.word;
            if (state_op(w) != kOpGo) break;
            last_run = state_seq(w);
            run_phase<DIM, POW2, SPEC>(ap, sh, ring, stage_all, c, G, tl);
        }
    } else {
        // ------------------------------------------------------------------ CTA 0: the update loop
        unsigned long long flipped = 0, levels_cta = 0, phases = 0;
        uint32_t widest = 0;
        bool aborted = false;
        for (unsigned long long k = 0; k < p.n_updates && !aborted; ++k) {
            const unsigned long long u = p.u0 + k;
            const uint32_t u_lo = (uint32_t)u, u_hi = (uint32_t)(u >> 32);
            // A1: seed draw (reading R8) and initial flip
            if (tid == 0) {
                const uint4 xr = philox4x32_10(0u, kDomainSite, u_lo, u_hi, p.key0, p.key1);
                const unsigned long long rr = (unsigned long long)xr.x | ((unsigned long long)xr.y << 32);
                const uint32_t i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
                const int s = load_spin_l2(p.spins, i0);
                claim_and_flip(p.spins, i0, s);
                q0[0] = i0;
                sh.lcnt[0] = 1u;
                sh.lcnt[1] = 0u;
                sh.s0 = s;
            }
            __syncthreads();
            const int s0 = sh.s0;
            unsigned long long size = 1;
            unsigned int lvl = 0;
            uint32_t *cur = q0, *nxt = q1;
            for (;;) {
                const unsigned int n = sh.lcnt[lvl];
                if (n == 0u) break;
                if (n > widest) widest = n;
                if (n > p.up) {
                    // ---- the frontier outgrew one CTA: hand it to its owners and run a barrier-free phase
                    ++phases;
                    const unsigned int seq = (unsigned int)(2ull * phases);
                    const uint32_t tag = (uint32_t)(phases & 1ull) << 31;
                    if (tid == 0 && phases >= 2ull) {
                        // every helper must have seen the end of the previous phase before entries of a new one appear
                        const unsigned long long need = (unsigned long long)(G - 1u) * (phases - 1ull);
                        unsigned int polls = 0;
                        while (ld_relaxed_u64(&ctl->acks) < need) {
                            if ((++polls & 0xFFFFu) == 0u) {
                                if (ld_relaxed_u32(&ctl->error) != 0u) break;
                                if (polls > (1u << 28)) { raise_abort(ctl, 5u); break; }
                            }
                        }
                    }
                    __syncthreads();
                    for (unsigned int e = tid; e < n; e += kT) {
                        const uint32_t j = cur[e];
                        const unsigned int o = owner_of<DIM, POW2>(ap, j, G);
                        const unsigned long long pos = atomicAdd(&ap.gtail[o], 1ull);
                        inbox_store(ap, o, pos, j | tag);
                        ++tl.inbox_pushes;
                    }
                    __syncthreads();
                    if (tid == 0) {
                        sh.u_lo = u_lo;
                        sh.u_hi = u_hi;
                        sh.seq = seq;
                        sh.stop = 0u;
                        st_relaxed_u64(&ctl->u, u);
                        __threadfence();
                        st_release_u64(&ctl->state, pack_state(seq, kOpGo, s0));
                    }
                    __syncthreads();
                    run_phase<DIM, POW2, SPEC>(ap, sh, ring, stage_all, 0u, G, tl);
                    if (tid == 0) {
                        fence_acq_rel_gpu();
                        sh.size_acc = atomicExch(&ctl->added, 0ull);
                        sh.word = ld_relaxed_u64(&ctl->state);
                    }
                    __syncthreads();
                    size += sh.size_acc;
                    if (state_op(sh.word) == kOpAbort) aborted = true;
                    __syncthreads();
                    break;
                }
                // ---- one-CTA level: shared-memory queues, __syncthreads only
                ++levels_cta;
                const unsigned int lvl1 = (lvl == 2u) ? 0u : lvl + 1u;
                const unsigned int lvl2 = (lvl1 == 2u) ? 0u : lvl1 + 1u;
                if (tid == 0) sh.lcnt[lvl2] = 0u;
                for (unsigned int pass = 0; pass < n; pass += kT) {
                    const unsigned int idx = pass + tid;
                    const bool valid = idx < n;
                    const uint32_t site = valid ? cur[idx] : 0u;
                    expand_sites<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, valid, site, nxt, &sh.lcnt[lvl1], tl.attempts);
                }
                __syncthreads();
                size += sh.lcnt[lvl1];
                lvl = lvl1;
                uint32_t *t = cur; cur = nxt; nxt = t;
            }
            // A7: epilogue
            if (tid == 0) p.sizes[k] = (uint32_t)size;
            flipped += size;
            __syncthreads();
        }
        if (tid == 0) {
            if (!aborted) st_release_u64(&ctl->state, pack_state((unsigned int)(2ull * phases + 2ull), kOpExit, 1));
            ctl->stats[0] = p.n_updates;
            ctl->stats[1] = flipped;
            ctl->stats[2] = levels_cta;
            ctl->stats[8] = widest;
            ctl->stats[10] = phases;
        }
    }
    // tallies
    const unsigned int a = __reduce_add_sync(kFullMask, tl.attempts);
    const unsigned int ib = __reduce_add_sync(kFullMask, tl.inbox_pushes);
    const unsigned int rp = __reduce_add_sync(kFullMask, tl.ring_pushes);
    if ((tid & 31u) == 0u) {
        if (a) atomicAdd(&ctl->stats[7], (unsigned long long)a);
        if (ib) atomicAdd(&ctl->stats[11], (unsigned long long)ib);
        if (rp) atomicAdd(&ctl->stats[12], (unsigned long long)rp);
        if (tl.passes) atomicAdd(&ctl->stats[13], (unsigned long long)tl.passes);
    }
}

template <int DIM, bool POW2, bool SPEC>
cudaError_t launch_one(const AsyncParams &ap, int ctas, size_t smem_bytes, cudaStream_t stream)
{
    void *args[] = { const_cast<AsyncParams *>(&ap) };
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(&growth_async_kernel<DIM, POW2, SPEC>), dim3((unsigned int)ctas),
                                       dim3(kT), args, smem_bytes, stream);
}

template <int DIM, bool POW2, bool SPEC>
cudaError_t prepare_one(size_t smem_bytes, int *ctas_per_sm)
{
    const void *fn = reinterpret_cast<const void *>(&growth_async_kernel<DIM, POW2, SPEC>);
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, growth_async_kernel<DIM, POW2, SPEC>, kT, smem_bytes);
}

}  // namespace

#define WOLFF_ASYNC_DISPATCH(CALL)                                                   \
    do {                                                                             \
        if (dim == 2) {                                                              \
            if (pow2) return spec ? CALL(2, true, true) : CALL(2, true, false);      \
            return spec ? CALL(2, false, true) : CALL(2, false, false);              \
        }                                                                            \
        if (pow2) return spec ? CALL(3, true, true) : CALL(3, true, false);          \
        return spec ? CALL(3, false, true) : CALL(3, false, false);                  \
    } while (0)

cudaError_t async_prepare(int dim, bool pow2, bool spec, size_t smem_bytes, int *ctas_per_sm)
{
#define WOLFF_CALL(D, P, S) prepare_one<D, P, S>(smem_bytes, ctas_per_sm)
    WOLFF_ASYNC_DISPATCH(WOLFF_CALL);
#undef WOLFF_CALL
}

cudaError_t launch_growth_async(const AsyncParams &ap, int dim, bool spec, int ctas, size_t smem_bytes, cudaStream_t stream)
{
    const bool pow2 = ap.g.geo.pow2 != 0u;
#define WOLFF_CALL(D, P, S) launch_one<D, P, S>(ap, ctas, smem_bytes, stream)
    WOLFF_ASYNC_DISPATCH(WOLFF_CALL);
#undef WOLFF_CALL
}

size_t async_smem_bytes(uint32_t ring_cap, uint32_t lvl_cap)
{
    return ((size_t)ring_cap + (size_t)kWarps * kStage + 2u * (size_t)lvl_cap) * sizeof(uint32_t);
}

}  // namespace wolff
