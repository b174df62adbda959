// growth_tiles.cu -- the shared-memory-resident, barrier-free cluster-growth kernel
// (8(f) rows 2 and 4 folded into the hot path).
//
// Same computation as growth.cu: n_updates Wolff single-cluster updates (steps i-v),
// every newly added spin expanded by one thread (step iii').  The paper names two costs
// (PAPER.md:187): the wait of all blocks at every synchronisation, and the latency of the uncoalesced
// global-memory update that marks a spin as a member.  growth.cu still pays both once per BFS level
// (one barrier, one L2 atomic round trip).  This kernel pays neither on the critical path:
//
//   - for the length of one launch the int8 lattice LIVES IN SHARED MEMORY.  It is cut into tiles of
//     B^dim sites; tile t belongs to CTA (t*A mod ntiles) mod G, one CTA per SM, so every BASELINE
//     lattice (<= 16 MiB) fits the 148 x 227 KiB of the chip.  Claim-and-flip (A4) is the same single
//     idempotent atomic as in growth.cu, but on shared memory: the dependent chain of one hop is
//     LDS gather || Philox -> ATOMS -> ballot, a few hundred cycles instead of two L2 round trips;
//   - a site is always expanded by the CTA that owns its tile.  A warp that claims neighbours keeps up to
//     32 of them in registers and expands them in its next pass; the rest goes to a shared-memory ring that
//     the other warps of the CTA drain (overflow: a per-CTA global spill list);
//   - an active bond that leaves the CTA's territory becomes a MESSAGE "claim site j" in the owner's inbox
//     (global memory, one L2 atomicAdd for the slot + one 8-byte store); the owner's receiver warp polls its
//     inbox, makes the claim on its own shared memory and feeds its ring.  Bond variables are a function of
//     (seed, update, bond), so the cluster is the connected component of the seed
//     site whatever the order of expansion: no BFS levels, no barrier (A6 becomes a work hand-over);
//   - termination of an update: every CTA publishes gdone[c] = "inbox messages consumed, with their whole
//     local progeny expanded" whenever it runs dry; a monitor warp in CTA 0 reads every gdone[], then every
//     gtail[] (messages ever pushed).  Both only grow, a message is counted in gtail before anything it
//     causes can be counted in gdone, so equal sums mean: at the instant between the two passes nothing was
//     queued, in flight or being expanded anywhere.  The monitor then logs the size (A7) and sends the seed
//     message of the next update (A1) to the owner of the seed site.
//
// The global lattice stays the authoritative copy between launches: tiles are loaded in the prologue and
// written back in the epilogue (N bytes each way per launch, amortised over n_updates).
#include "expand.cuh"
#include "internal.h"

namespace wolff {
namespace {

constexpr uint32_t kEmpty = 0xFFFFFFFFu;
constexpr int kT = kTileThreads;
constexpr int kWarps = kT / 32;
constexpr int kStage = 32;                         // winners one warp can produce in one pass (one per lane)

// message = [kind:2 | lap:1 | k:29] [site:31 | s0<0:1]
enum Kind : unsigned int { kKindNone = 0, kKindClaim = 1, kKindSeed = 2, kKindExit = 3 };
constexpr unsigned int kMaxK = (1u << 29);

__device__ __forceinline__ unsigned long long pack_msg(unsigned int kind, unsigned int lap, unsigned int k, uint32_t site, int s0)
{
    const unsigned int hi = (kind << 30) | ((lap & 1u) << 29) | (k & (kMaxK - 1u));
    const unsigned int lo = (site << 1) | (s0 < 0 ? 1u : 0u);
    return ((unsigned long long)hi << 32) | (unsigned long long)lo;
}

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

// Branch-free forms for the dependent chain of a worker pass (predicated instructions instead of divergent regions).
__device__ __forceinline__ uint32_t selp_u32(uint32_t a, uint32_t b, bool pick_a)
{
    uint32_t r;
    asm("{\n .reg .pred p;\n setp.ne.u32 p, %3, 0;\n selp.u32 %0, %1, %2, p;\n}" : "=r"(r) : "r"(a), "r"(b), "r"((unsigned int)pick_a));
    return r;
}
// Claim on shared memory: OR (s0 = +1) or AND (s0 = -1) on the word at shared address saddr, when `go`; returns the old word.
__device__ __forceinline__ unsigned int atoms_claim(uint32_t saddr, unsigned int mask_or, bool go_or, bool go_and)
{
    unsigned int old = 0;
    asm volatile("{\n .reg .pred p, q;\n .reg .b32 m;\n setp.ne.u32 p, %3, 0;\n setp.ne.u32 q, %4, 0;\n not.b32 m, %2;\n"
                 " @p atom.shared.or.b32 %0, [%1], %2;\n @q atom.shared.and.b32 %0, [%1], m;\n}"
                 : "+r"(old) : "r"(saddr), "r"(mask_or), "r"((unsigned int)go_or), "r"((unsigned int)go_and) : "memory");
    return old;
}
__device__ __forceinline__ unsigned long long atomg_inc_if(unsigned long long *p, bool go)
{
    unsigned long long old = 0;
    asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %2, 0;\n @p atom.global.add.u64 %0, [%1], 1;\n}"
                 : "+l"(old) : "l"(p), "r"((unsigned int)go) : "memory");
    return old;
}

// Per-CTA shared state.
struct alignas(16) TShared {
    unsigned int head, tail;            // ring: entries [head, tail) wait for a worker warp (one aligned 64-bit word)
    unsigned int pending;               // sites claimed by this CTA and not yet expanded (+ receiver tokens)
    unsigned int claimed;               // spins claimed since the last publish
    unsigned int stop;                  // leave: exit message seen, or the launch is aborted
    unsigned int pub_lock;              // publishers of this CTA take turns
    int s0;                             // seed spin of the running update
    uint32_t u_lo, u_hi;                // its index
    unsigned long long ihead;           // inbox messages consumed (written by the receiver warp only)
    unsigned long long spill_head, spill_tail;   // running positions in the CTA's global spill list (kept across launches)
};

struct Tally {
    unsigned int attempts = 0;          // claim atomics on shared memory (per lane)
    unsigned int messages = 0;          // messages pushed (per lane)
    unsigned int ring_pushes = 0;       // sites handed to the ring (per lane)
    unsigned int spills = 0;            // sites spilled to global memory (per lane)
    unsigned int passes = 0;            // warp passes (lane 0)
#ifdef WOLFF_PROFILE
    unsigned long long cyc_pass = 0;    // cycles inside passes (lane 0)
    unsigned long long lanes = 0;       // sites expanded (lane 0)
    unsigned long long cyc1 = 0, n1 = 0, cyc1r = 0, cyc2 = 0, cyc3 = 0, cyc23c = 0, n23c = 0;
#endif
};

// ------------------------------------------------------------------------------------------ geometry of the tiling
// Site i = x + L*y (+ L*L*z), L a power of two.  Tile coordinates (x >> b, ...), tile index t = tx + ntx*ty (+ ...),
// p = (t * A) mod ntiles (A odd: a bijection), owner = p mod G, slot = p div G.  Inside a tile sites are
// row-major again: w = (x & m) + B*(y & m) (+ B*B*(z & m)); shared-memory byte address = slot*B^dim + w.
template <int DIM>
struct Tiling {
    uint32_t b, m, nt_log, nt_mask, ntiles_mask, A, G, logL, Lmask;
    unsigned long long magic;

    __device__ __forceinline__ explicit Tiling(const TileParams &tp)
        : b(tp.tile_log), m((1u << tp.tile_log) - 1u), nt_log(tp.g.geo.logL - tp.tile_log),
          nt_mask((1u << (tp.g.geo.logL - tp.tile_log)) - 1u), ntiles_mask(tp.ntiles - 1u), A(tp.permA), G(tp.G),
          logL(tp.g.geo.logL), Lmask(tp.g.geo.L - 1u), magic(tp.magicG) {}

    __device__ __forceinline__ void coords(uint32_t i, uint32_t &x, uint32_t &y, uint32_t &z) const
    {
        x = i & Lmask;
        y = (i >> logL) & Lmask;
        z = (DIM == 3) ? (i >> (2u * logL)) : 0u;
    }
    __device__ __forceinline__ uint32_t tile_of(uint32_t x, uint32_t y, uint32_t z) const
    {
        uint32_t t = (x >> b) | ((y >> b) << nt_log);
        if (DIM == 3) t |= (z >> b) << (2u * nt_log);
        return t;
    }
    __device__ __forceinline__ uint32_t within(uint32_t x, uint32_t y, uint32_t z) const
    {
        uint32_t w = (x & m) | ((y & m) << b);
        if (DIM == 3) w |= (z & m) << (2u * b);
        return w;
    }
    // p -> (owner, slot); magic = ceil(2^40 / G), exact for p < 2^24 (checked by the host)
    __device__ __forceinline__ void place(uint32_t t, uint32_t &owner, uint32_t &slot) const
    {
        const uint32_t p = (t * A) & ntiles_mask;
        slot = (uint32_t)(((unsigned long long)p * magic) >> 40);
        owner = p - slot * G;
    }
};

// ------------------------------------------------------------------------------------------ queues
// Reserve n consecutive ring entries; false when the ring cannot take them.
__device__ __forceinline__ bool ring_reserve(TShared &sh, uint32_t cap, unsigned int n, unsigned int &base)
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
// Fill a reserved ring slot.  The previous lap's entry of this slot has been acquired (head moved past it) but
// may not have been taken yet: wait for the slot to be empty (its taker never waits for us).
__device__ __forceinline__ void ring_put(uint32_t *slot, uint32_t v)
{
    while (atomicCAS(slot, kEmpty, v) != kEmpty) { }
}

// Spill list of CTA c: entry = (site << 1) | tag, tag = ((pos / cap) + 1) & 1, so an entry left from the lap
// before (or the zero the list starts with) never looks valid and nothing has to be cleared.
__device__ __forceinline__ uint32_t spill_tag(unsigned long long pos, uint32_t cap_log) { return (uint32_t)((pos >> cap_log) + 1ull) & 1u; }

// Hand n sites (stage[0..n), warp-collective) to the other warps of the CTA: the ring, or the spill list when
// the ring is full.  The caller has already counted them in sh.pending.
__device__ __forceinline__ void hand_over(const TileParams &tp, TShared &sh, uint32_t *ring, const uint32_t *items, unsigned int n,
                                          unsigned int c, Tally &tl)
{
    const unsigned int lane = threadIdx.x & 31u;
    const uint32_t rmask = tp.ring_cap - 1u;
    unsigned int base = 0, ok = 0;
    if (lane == 0) ok = ring_reserve(sh, tp.ring_cap, n, base) ? 1u : 0u;
    ok = __shfl_sync(kFullMask, ok, 0);
    base = __shfl_sync(kFullMask, base, 0);
    if (ok) {
        for (unsigned int j = lane; j < n; j += 32u) { ring_put(ring + ((base + j) & rmask), items[j]); ++tl.ring_pushes; }
    } else {
        unsigned long long sbase = 0;
        if (lane == 0) sbase = atomicAdd(&sh.spill_tail, (unsigned long long)n);
        sbase = __shfl_sync(kFullMask, sbase, 0);
        uint32_t *const seg = tp.spill + ((size_t)c << tp.spill_log);
        const uint32_t smask = (1u << tp.spill_log) - 1u;
        for (unsigned int j = lane; j < n; j += 32u) {
            const unsigned long long pos = sbase + (unsigned long long)j;
            st_relaxed_u32(seg + ((uint32_t)pos & smask), (items[j] << 1) | spill_tag(pos, tp.spill_log));
            ++tl.spills;
        }
    }
}

// Called by the lane whose atomic brought sh.pending to zero: the CTA has (for the moment) nothing queued and
// nothing being expanded.  ihead is read BEFORE pending is looked at again, and the receiver raises pending before
// it moves ihead, so pending == 0 here means every message below I is done with all its local progeny.  Publishers
// of one CTA take turns (pub_lock): the claims of an earlier one reach `added` before a later one moves gdone.
__device__ __forceinline__ void publish(const TileParams &tp, TShared &sh, unsigned int c)
{
    while (atomicCAS(&sh.pub_lock, 0u, 1u) != 0u) { }
    const unsigned long long I = ld_vol64(&sh.ihead);
    __threadfence_block();
    if (ld_vol(&sh.pending) == 0u) {
        const unsigned int a = atomicExch(&sh.claimed, 0u);
        if (a) atomicAdd(tp.added, (unsigned long long)a);
        __threadfence();
        atomicMax(tp.gdone + c, I);
        __threadfence();
    }
    atomicExch(&sh.pub_lock, 0u);
}

__device__ __forceinline__ void raise_abort(Control *ctl, unsigned int code) { st_relaxed_u32(&ctl->error, code); }

// ------------------------------------------------------------------------------------------ worker warp
// Expands sites owned by this CTA until the launch is over (A2-A5 on shared memory).
//
// One LANE PER BOND: a warp holds up to S = 32 / (2*DIM) sites per pass (8 in 2D, 5 in 3D) and lane (q, k) tests the
// bond from site q to its neighbour k (k = 2d: +d, k = 2d + 1: -d).  The frontier inside one CTA is a handful of
// sites wide, so lanes are cheap and the dependent instruction chain of a pass is what an update waits for: per lane
// one neighbour address, one Philox block (the bond owner's), one LDS, one ATOMS, one ballot for the whole warp.
template <int DIM>
__device__ __forceinline__ void worker_warp(const TileParams &tp, TShared &sh, int8_t *lat, uint32_t *ring, uint32_t *stage,
                                            unsigned int c, Tally &tl)
{
    constexpr unsigned int ND = 2u * DIM, S = 32u / ND;
    const GrowthParams &p = tp.g;
    const Tiling<DIM> tg(tp);
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int bit = 1u << lane, lt = bit - 1u;
    const unsigned int q = lane / ND, k = lane - q * ND, d = k >> 1, sgn = k & 1u;
    const bool alive = q < S;
    const uint32_t sh_d = d * tg.logL, fmask = tg.Lmask << sh_d, delta = sgn ? 0xFFFFFFFFu : 1u;
    const uint32_t rmask = tp.ring_cap - 1u;
    const uint32_t tile_sites_log = DIM * tp.tile_log;
    const uint32_t in_mask = tp.in_cap - 1u;
    const uint32_t lat_s = (uint32_t)__cvta_generic_to_shared(lat);
    uint32_t site = 0;
    unsigned int nsites = 0;     // sites held by the warp (warp-uniform); lanes of group q < nsites work
    int s0 = 1;
    unsigned int s0_byte = 1u;
    uint32_t u_lo = 0, u_hi = 0, krel = 0;
    unsigned int mywon = 0;      // spins this lane claimed since the warp last ran dry

    for (;;) {
        if (nsites == 0u) {
            // ---- take up to S sites from the ring, else from the spill list
            unsigned int n = 0, h = 0, from_spill = 0;
            unsigned long long sh_pos = 0;
            if (lane == 0) {
                unsigned int idle = 0;
                for (;;) {
                    // one 64-bit load: a consistent (head, tail) pair; the three loads of an idle poll are independent
                    const unsigned long long ht = ld_vol64(reinterpret_cast<const unsigned long long *>(&sh.head));
                    sh_pos = ld_vol64(&sh.spill_head);
                    const unsigned long long st = ld_vol64(&sh.spill_tail);
                    const unsigned int stop = ld_vol(&sh.stop);
                    h = (unsigned int)ht;
                    const unsigned int t = (unsigned int)(ht >> 32);
                    if (t != h) {
                        n = t - h < S ? t - h : S;
                        if (atomicCAS(&sh.head, h, h + n) == h) break;
                        n = 0;
                        continue;
                    }
                    if (st != sh_pos) {
                        n = st - sh_pos < (unsigned long long)S ? (unsigned int)(st - sh_pos) : S;
                        if (atomicCAS(&sh.spill_head, sh_pos, sh_pos + n) == sh_pos) { from_spill = 1; break; }
                        n = 0;
                        continue;
                    }
                    if (stop) break;
                    // idle warps share the SM's load/store pipe with the working ones: back off (the warps of a CTA are
                    // staggered by their idle counts, so one of them polls every few tens of nanoseconds)
                    ++idle;
                    if (idle > 2u) __nanosleep(idle < 8u ? 64u : (idle < 16u ? 256u : tp.idle_ns));
                }
            }
            n = __shfl_sync(kFullMask, n, 0);
            h = __shfl_sync(kFullMask, h, 0);
            from_spill = __shfl_sync(kFullMask, from_spill, 0);
            sh_pos = __shfl_sync(kFullMask, sh_pos, 0);
            if (n == 0u) break;                                  // launch over
            uint32_t ent = 0;
            if (lane < n) {
                unsigned int spins = 0;
                if (!from_spill) {
                    uint32_t *slot = ring + ((h + lane) & rmask);
                    do {
                        ent = atomicExch(slot, kEmpty);          // the producer reserved it; its store is on the way
                        if (ent == kEmpty && ++spins > (1u << 26)) { raise_abort(p.ctl, 4u); ent = 0u; }
                    } while (ent == kEmpty);
                } else {
                    const unsigned long long pos = sh_pos + (unsigned long long)lane;
                    const uint32_t *slot = tp.spill + ((size_t)c << tp.spill_log) + ((uint32_t)pos & ((1u << tp.spill_log) - 1u));
                    const uint32_t tag = spill_tag(pos, tp.spill_log);
                    uint32_t v;
                    do {
                        v = ld_relaxed_u32(slot);
                        if ((v & 1u) != tag && ++spins > (1u << 24)) { raise_abort(p.ctl, 5u); v = tag; }
                    } while ((v & 1u) != tag);
                    ent = v >> 1;
                }
            }
            site = __shfl_sync(kFullMask, ent, q);
            nsites = n;
            // the update these sites belong to (written by the receiver before it fed the ring)
            s0 = *reinterpret_cast<volatile int *>(&sh.s0);
            s0_byte = (unsigned int)s0 & 0xFFu;
            u_lo = ld_vol(&sh.u_lo);
            u_hi = ld_vol(&sh.u_hi);
            krel = (uint32_t)((((unsigned long long)u_hi << 32) | u_lo) - p.u0);
        }
#ifdef WOLFF_PROFILE
        const long long tp0 = clock64();
#endif
        const unsigned int expanded = nsites;
        const bool have = alive && q < nsites;

        // ---- A2: this lane's neighbour; is it in this CTA's shared memory, and where
        const uint32_t nid = (site & ~fmask) | ((((site >> sh_d) + delta) & tg.Lmask) << sh_d);
        uint32_t nx, ny, nz, own, slot;
        tg.coords(nid, nx, ny, nz);
        tg.place(tg.tile_of(nx, ny, nz), own, slot);
        const uint32_t addr = (slot << tile_sites_log) + tg.within(nx, ny, nz);
        const bool local = own == c;
        const unsigned int shift = (addr & 3u) * 8u;
        // gather (LDS), in flight while the Philox rounds execute
        const uint32_t saddr = lat_s + (addr & ~3u);
        unsigned int spw = 0;
        if (have && local) asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(spw) : "r"(saddr));
        // ---- A3: the bond to the +d neighbour is owned by this site, the bond to the -d neighbour by that neighbour
        const uint4 blk = philox4x32_10(sgn ? nid : site, kDomainBond, u_lo, u_hi, p.key0, p.key1);
        const uint32_t r = selp_u32(blk.x, selp_u32(blk.y, blk.z, d == 1u), d == 0u);
        const bool active = have && (r < tp.thr32 || tp.thr_all != 0u);
        const bool cand_l = active && local && (((spw >> shift) & 0xFFu) == s0_byte);
        const bool cand_r = active && !local;

        // ---- A4 across the territory border: a message to the owner (slot by one L2 atomic, then one 8-byte store)
        const unsigned long long pos = atomg_inc_if(tp.gtail + own, cand_r);
        // ---- A4 inside the territory: the same idempotent atomic as claim_and_flip(), on shared memory
        const unsigned int old = atoms_claim(saddr, 0xFEu << shift, cand_l && s0 > 0, cand_l && s0 < 0);
        const bool won = cand_l && (((old >> shift) & 0xFFu) == s0_byte);
        tl.attempts += cand_l ? 1u : 0u;
        mywon += won ? 1u : 0u;
        if (lane == 0) ++tl.passes;
#ifdef WOLFF_PROFILE
        const long long tp1 = clock64();
        const bool anyr = __any_sync(kFullMask, cand_r);
        if (anyr) tl.cyc1r += (unsigned long long)(tp1 - tp0); else { tl.cyc1 += (unsigned long long)(tp1 - tp0); ++tl.n1; }
#endif

        // ---- A5: compact the winners; the first S are this warp's next pass
        const unsigned int wb = __ballot_sync(kFullMask, won);
        const unsigned int total = __popc(wb);
        if (won) stage[__popc(wb & lt)] = nid;
        // messages leave before this pass is accounted for
        if (cand_r) {
            const unsigned int lap = (unsigned int)(pos >> tp.in_log) & 1u;
            st_relaxed_u64(tp.inbox + ((size_t)own << tp.in_log) + ((uint32_t)pos & in_mask), pack_msg(kKindClaim, lap, krel, nid, s0));
            ++tl.messages;
        }
        __syncwarp();
#ifdef WOLFF_PROFILE
        const long long tp2 = clock64();
        tl.cyc2 += (unsigned long long)(tp2 - tp1);
#endif
        // ---- accounting: the new sites are counted before any of them can be seen by another warp
        if (total == 0u) {
            // the warp runs dry: its claims become visible to the publisher before its sites stop being pending
            const unsigned int w = __reduce_add_sync(kFullMask, mywon);
            mywon = 0;
            if (lane == 0) {
                if (w) atomicAdd(&sh.claimed, w);
                __threadfence_block();
                const unsigned int before = atomicSub(&sh.pending, expanded);
                if (before == expanded) publish(tp, sh, c);
            }
        } else if (total != expanded) {
            if (lane == 0) atomicAdd(&sh.pending, total - expanded);
        }
        nsites = total < S ? total : S;
        if (alive && q < nsites) site = stage[q];
        if (total > S) hand_over(tp, sh, ring, stage + S, total - S, c, tl);
        __syncwarp();      // stage[] is rewritten in the next pass
#ifdef WOLFF_PROFILE
        const long long tp3 = clock64();
        tl.cyc_pass += (unsigned long long)(tp3 - tp0);
        tl.cyc3 += (unsigned long long)(tp3 - tp2);
        if (total != 0u && total <= S && !anyr) { tl.cyc23c += (unsigned long long)(tp3 - tp1); ++tl.n23c; }
        tl.lanes += expanded;
#endif
    }
}

// ------------------------------------------------------------------------------------------ receiver warp
// Polls the CTA's inbox; makes the claims other CTAs (and the monitor: the seed site, A1) ask for, on its own
// shared memory; feeds the ring.
template <int DIM>
__device__ __forceinline__ void receiver_warp(const TileParams &tp, TShared &sh, int8_t *lat, uint32_t *ring, uint32_t *stage,
                                              unsigned int c, Tally &tl)
{
    const GrowthParams &p = tp.g;
    const Tiling<DIM> tg(tp);
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int bit = 1u << lane, lt = bit - 1u;
    const uint32_t in_mask = tp.in_cap - 1u;
    const uint32_t tile_sites_log = DIM * tp.tile_log;
    const unsigned long long *const box = tp.inbox + ((size_t)c << tp.in_log);
    unsigned long long ih = ld_vol64(&sh.ihead);
    unsigned int polls = 0;
    for (;;) {
        const unsigned long long pos = ih + (unsigned long long)lane;
        const unsigned long long v = ld_relaxed_u64(box + ((uint32_t)pos & in_mask));
        const unsigned int hi = (unsigned int)(v >> 32), lo = (unsigned int)v;
        const unsigned int kind = hi >> 30;
        const bool ok = kind != kKindNone && ((hi >> 29) & 1u) == ((unsigned int)(pos >> tp.in_log) & 1u);
        const unsigned int b = __ballot_sync(kFullMask, ok);
        const unsigned int k = (b == kFullMask) ? 32u : (unsigned int)__ffs((int)~b) - 1u;   // arrivals in order: the contiguous prefix
        if (k == 0u) {
            if ((++polls & 0xFFu) == 0u && ld_relaxed_u32(&p.ctl->error) != 0u) break;
            continue;
        }
        const bool mine = lane < k;
        if (__any_sync(kFullMask, mine && kind == kKindExit)) {
            // sent by the monitor after the last update is complete: nothing is queued anywhere
            ih += (unsigned long long)k;
            if (lane == 0) { st_vol64(&sh.ihead, ih); atomicMax(tp.gdone + c, ih); }
            break;
        }
        const uint32_t site = lo >> 1;
        int s0 = (lo & 1u) ? -1 : 1;
        bool win = false;
        if (mine) {
            uint32_t x, y, z, own, slot;
            tg.coords(site, x, y, z);
            tg.place(tg.tile_of(x, y, z), own, slot);
            const uint32_t addr = (slot << tile_sites_log) + tg.within(x, y, z);
            if (kind == kKindSeed) s0 = (int)*reinterpret_cast<volatile signed char *>(lat + addr);   // A1: the seed spin
            win = claim_and_flip(lat, addr, s0);
            ++tl.attempts;
        }
        const unsigned int wb = __ballot_sync(kFullMask, win);
        const unsigned int w = __popc(wb);
        const int s0u = __shfl_sync(kFullMask, s0, 0);
        const unsigned int krel = __shfl_sync(kFullMask, hi & (kMaxK - 1u), 0);
        ih += (unsigned long long)k;
        if (lane == 0) {
            const unsigned long long u = p.u0 + (unsigned long long)krel;
            *reinterpret_cast<volatile int *>(&sh.s0) = s0u;
            st_vol(&sh.u_lo, (uint32_t)u);
            st_vol(&sh.u_hi, (uint32_t)(u >> 32));
            atomicAdd(&sh.pending, w + 1u);            // the winners, and a token that keeps the CTA busy until they are queued
            if (w) atomicAdd(&sh.claimed, w);
            __threadfence_block();
            st_vol64(&sh.ihead, ih);                   // after pending: see publish()
            __threadfence_block();
        }
        if (win) stage[__popc(wb & lt)] = site;
        __syncwarp();
        if (w) hand_over(tp, sh, ring, stage, w, c, tl);
        __syncwarp();
        if (lane == 0) {
            const unsigned int before = atomicSub(&sh.pending, 1u);
            if (before == 1u) publish(tp, sh, c);
        }
    }
    __syncwarp();
    if (lane == 0) { __threadfence_block(); st_vol(&sh.stop, 1u); }
}

// ------------------------------------------------------------------------------------------ monitor warp
// CTA 0 only: the update loop ("(v) Go to (i)").  Sends the seed message of update u (A1, reading R8),
// waits for the update to terminate (see the header), logs its size (A7).
template <int DIM>
__device__ __forceinline__ void monitor_warp(const TileParams &tp, Tally &tl)
{
    const GrowthParams &p = tp.g;
    const Tiling<DIM> tg(tp);
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int G = tp.G;
    const uint32_t in_mask = tp.in_cap - 1u;
    Control *ctl = p.ctl;
    unsigned long long prev = ld_relaxed_u64(tp.added);
    unsigned long long flipped = 0, polls_total = 0;
    bool aborted = false;
    for (unsigned long long k = 0; k < p.n_updates && !aborted; ++k) {
        if (lane == 0) {
            const unsigned long long u = p.u0 + k;
            const uint4 xr = philox4x32_10(0u, kDomainSite, (uint32_t)u, (uint32_t)(u >> 32), p.key0, p.key1);
            const unsigned long long rr = (unsigned long long)xr.x | ((unsigned long long)xr.y << 32);
            const uint32_t i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
            uint32_t x, y, z, own, slot;
            tg.coords(i0, x, y, z);
            tg.place(tg.tile_of(x, y, z), own, slot);
            const unsigned long long pos = atomicAdd(tp.gtail + own, 1ull);
            st_relaxed_u64(tp.inbox + ((size_t)own << tp.in_log) + ((uint32_t)pos & in_mask),
                           pack_msg(kKindSeed, (unsigned int)(pos >> tp.in_log) & 1u, (unsigned int)k, i0, 1));
            ++tl.messages;
        }
        const unsigned long long t0 = globaltimer_ns();
        unsigned int passes = 0;
        for (;;) {
            unsigned long long d = 0, t = 0;
            for (unsigned int cc = lane; cc < G; cc += 32u) d += ld_relaxed_u64(tp.gdone + cc);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) d += __shfl_xor_sync(kFullMask, d, o);
            fence_acq_rel_gpu();      // every gtail (and `added`) is read after every gdone
            for (unsigned int cc = lane; cc < G; cc += 32u) t += ld_relaxed_u64(tp.gtail + cc);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(kFullMask, t, o);
            ++passes;
            if (d == t) break;
            if ((passes & 0xFFu) == 0u) {
                unsigned int bad = 0;
                if (lane == 0) {
                    if (ld_relaxed_u32(&ctl->error) != 0u) bad = 1;
                    else if (globaltimer_ns() - t0 > tp.watchdog_ns) { raise_abort(ctl, 3u); bad = 1; }
                }
                if (__shfl_sync(kFullMask, bad, 0)) { aborted = true; break; }
            }
        }
        polls_total += passes;
        if (!aborted && lane == 0) {
            const unsigned long long a = ld_relaxed_u64(tp.added);
            p.sizes[k] = (uint32_t)(a - prev);      // A7
            flipped += a - prev;
            prev = a;
        }
    }
    // everybody leaves (also after an abort: receivers poll the error flag, but an exit message is quicker)
    for (unsigned int cc = lane; cc < G; cc += 32u) {
        const unsigned long long pos = atomicAdd(tp.gtail + cc, 1ull);
        st_relaxed_u64(tp.inbox + ((size_t)cc << tp.in_log) + ((uint32_t)pos & in_mask),
                       pack_msg(kKindExit, (unsigned int)(pos >> tp.in_log) & 1u, 0u, 0u, 1));
    }
    if (lane == 0) {
        ctl->stats[0] += p.n_updates;
        ctl->stats[1] += flipped;
#ifndef WOLFF_PROFILE
        ctl->stats[9] += polls_total;
#endif
    }
}

// ------------------------------------------------------------------------------------------ the kernel
// Copy the tiles of CTA c between the global lattice and shared memory, one 32-bit word (4 sites along x) at a time.
template <int DIM, bool LOAD>
__device__ __forceinline__ void copy_tiles(const TileParams &tp, int8_t *lat, unsigned int c)
{
    const uint32_t b = tp.tile_log, m = (1u << b) - 1u;
    const uint32_t nt_log = tp.g.geo.logL - b, nt_mask = (1u << nt_log) - 1u;
    const uint32_t ts_log = DIM * b;
    const uint32_t words_per_tile = 1u << (ts_log - 2u);
    const uint32_t logL = tp.g.geo.logL;
    unsigned int *const glob = reinterpret_cast<unsigned int *>(tp.g.spins);
    unsigned int *const loc = reinterpret_cast<unsigned int *>(lat);
    for (uint32_t slot = 0; slot < tp.slots; ++slot) {
        const uint32_t pidx = slot * tp.G + c;
        if (pidx >= tp.ntiles) break;
        const uint32_t t = (pidx * tp.permAinv) & (tp.ntiles - 1u);
        const uint32_t ox = (t & nt_mask) << b;
        const uint32_t oy = ((t >> nt_log) & nt_mask) << b;
        const uint32_t oz = (DIM == 3) ? ((t >> (2u * nt_log)) << b) : 0u;
        for (uint32_t w4 = threadIdx.x; w4 < words_per_tile; w4 += kT) {
            const uint32_t w = w4 << 2;
            const uint32_t wx = w & m, wy = (w >> b) & m, wz = (DIM == 3) ? (w >> (2u * b)) : 0u;
            uint32_t gi = (ox + wx) + ((oy + wy) << logL);
            if (DIM == 3) gi += (oz + wz) << (2u * logL);
            if (LOAD) loc[(slot << (ts_log - 2u)) + w4] = __ldcg(glob + (gi >> 2));
            else glob[gi >> 2] = loc[(slot << (ts_log - 2u)) + w4];
        }
    }
}

template <int DIM>
__global__ void __launch_bounds__(kT, 1) growth_tiles_kernel(const TileParams tp)
{
    extern __shared__ __align__(16) unsigned char smem_t[];
    __shared__ TShared sh;
    const uint32_t lat_bytes = tp.slots << (DIM * tp.tile_log);
    int8_t *const lat = reinterpret_cast<int8_t *>(smem_t);
    uint32_t *const ring = reinterpret_cast<uint32_t *>(smem_t + lat_bytes);
    uint32_t *const stage_all = ring + tp.ring_cap;
    const unsigned int tid = threadIdx.x, warp = tid >> 5;
    const unsigned int c = blockIdx.x;
    Tally tl;

    for (unsigned int i = tid; i < tp.ring_cap; i += kT) ring[i] = kEmpty;
    if (tid == 0) {
        sh.head = sh.tail = 0u;
        sh.pending = sh.claimed = 0u;
        sh.stop = 0u;
        sh.pub_lock = 0u;
        sh.s0 = 1;
        sh.u_lo = sh.u_hi = 0u;
        sh.ihead = ld_relaxed_u64(tp.gdone + c);          // everything ever sent to this CTA was consumed by the last launch
        sh.spill_head = sh.spill_tail = ld_relaxed_u64(tp.gspill + c);
    }
    copy_tiles<DIM, true>(tp, lat, c);
    __syncthreads();

    if (warp == 0u) receiver_warp<DIM>(tp, sh, lat, ring, stage_all, c, tl);
    else if (warp == 1u && c == 0u) monitor_warp<DIM>(tp, tl);
    else worker_warp<DIM>(tp, sh, lat, ring, stage_all + warp * kStage, c, tl);
    __syncthreads();

    copy_tiles<DIM, false>(tp, lat, c);
    if (tid == 0) tp.gspill[c] = ld_vol64(&sh.spill_tail);
    // tallies
    Control *ctl = tp.g.ctl;
    const unsigned int a = __reduce_add_sync(kFullMask, tl.attempts);
    const unsigned int ms = __reduce_add_sync(kFullMask, tl.messages);
    const unsigned int rp = __reduce_add_sync(kFullMask, tl.ring_pushes);
    const unsigned int sp = __reduce_add_sync(kFullMask, tl.spills);
    if ((tid & 31u) == 0u) {
        if (a) atomicAdd(&ctl->stats[7], (unsigned long long)a);
        if (ms) atomicAdd(&ctl->stats[11], (unsigned long long)ms);
        if (rp) atomicAdd(&ctl->stats[12], (unsigned long long)rp);
        if (tl.passes) atomicAdd(&ctl->stats[13], (unsigned long long)tl.passes);
        if (sp) atomicAdd(&ctl->stats[14], (unsigned long long)sp);
#ifdef WOLFF_PROFILE
        if (tl.cyc_pass) atomicAdd(&ctl->stats[15], tl.cyc_pass);
        if (tl.lanes) atomicAdd(&ctl->stats[10], tl.lanes);
        if (tl.cyc1) atomicAdd(&ctl->stats[2], tl.cyc1);
        if (tl.n1) atomicAdd(&ctl->stats[3], tl.n1);
        if (tl.cyc1r) atomicAdd(&ctl->stats[4], tl.cyc1r);
        if (tl.cyc2) atomicAdd(&ctl->stats[5], tl.cyc2);
        if (tl.cyc3) atomicAdd(&ctl->stats[6], tl.cyc3);
        if (tl.cyc23c) atomicAdd(&ctl->stats[8], tl.cyc23c);
        if (tl.n23c) atomicAdd(&ctl->stats[9], tl.n23c);
#endif
    }
}

template <int DIM>
cudaError_t launch_one(const TileParams &tp, size_t smem_bytes, cudaStream_t stream)
{
    void *args[] = { const_cast<TileParams *>(&tp) };
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(&growth_tiles_kernel<DIM>), dim3(tp.G), dim3(kT), args,
                                       smem_bytes, stream);
}

template <int DIM>
cudaError_t prepare_one(size_t smem_bytes, int *ctas_per_sm)
{
    const void *fn = reinterpret_cast<const void *>(&growth_tiles_kernel<DIM>);
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, growth_tiles_kernel<DIM>, kT, smem_bytes);
}

}  // namespace

size_t tiles_smem_bytes(int dim, uint32_t tile_log, uint32_t slots, uint32_t ring_cap)
{
    return ((size_t)slots << ((uint32_t)dim * tile_log)) + ((size_t)ring_cap + (size_t)kWarps * kStage) * sizeof(uint32_t);
}

cudaError_t tiles_prepare(int dim, size_t smem_bytes, int *ctas_per_sm)
{
    return dim == 2 ? prepare_one<2>(smem_bytes, ctas_per_sm) : prepare_one<3>(smem_bytes, ctas_per_sm);
}

cudaError_t launch_growth_tiles(const TileParams &tp, int dim, size_t smem_bytes, cudaStream_t stream)
{
    return dim == 2 ? launch_one<2>(tp, smem_bytes, stream) : launch_one<3>(tp, smem_bytes, stream);
}

}  // namespace wolff
