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
//     idempotent atomic as in growth.cu, but on shared memory;
//   - inside a CTA a site is its LOCAL ADDRESS a = slot * B^dim + (within-tile index): a neighbour in the
//     same tile is a +- stride, a neighbour across a tile border comes from a small per-slot table
//     (owner CTA, slot) built in the prologue.  Global site ids are only rebuilt where a Philox counter
//     needs one;
//   - ONE LANE PER BOND: a warp holds up to 32 / (2 dim) sites per pass and lane (q, k) tests the bond
//     from site q to its neighbour k.  The frontier inside one CTA is a handful of sites wide, so lanes
//     are cheap; what an update waits for is the dependent instruction chain of a pass;
//   - BOND TABLES: the bond variables of update v are a pure function of (seed, v, bond) -- they do not
//     depend on the spins -- so warps with nothing to expand evaluate Philox4x32-10 for the tiles of
//     their CTA AHEAD of time (update v, then v + 1, double-buffered bit planes in shared memory, one
//     bit per bond).  A worker then reads one bit instead of running ten Philox rounds on its critical
//     path; where a tile's table is not ready (or the bond belongs to a site of another CTA) the lane
//     evaluates the same Philox block inline.  Both give the same bit, so the result cannot depend on
//     which one ran;
//   - a warp that claims neighbours keeps up to S of them in registers for its next pass; the rest goes
//     to a shared-memory ring that the other warps of the CTA drain (overflow: a per-CTA global spill list);
//     one idle warp per CTA holds the "watch" and polls the ring without backing off;
//   - an active bond that leaves the CTA's territory becomes a MESSAGE "claim the site at your local
//     address a" in the owner's inbox (global memory, one L2 atomicAdd for the slot + one 8-byte
//     store); the owner's receiver warp polls its inbox, makes the claim on its own shared memory and
//     feeds its ring.  Bond variables are a function of (seed, update, bond), so
//     the cluster is the connected component of the seed site whatever the order of expansion: no BFS
//     levels, no barrier (A6 becomes a work hand-over);
//   - termination of an update: every CTA publishes gdone[c] = "inbox messages consumed, with their whole
//     local progeny expanded" whenever it runs dry; a monitor warp in CTA 0 reads every gdone[], then every
//     gtail[] (messages ever pushed; 32-bit running counters, sums compared modulo 2^32 -- what is in flight is far
//     below 2^32).  Both only grow, a message is counted in gtail before anything it
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

#ifndef WOLFF_WIDE
#define WOLFF_WIDE 1
#endif

constexpr unsigned int kWide = WOLFF_WIDE;         // sites per lane group and pass: a warp holds up to kWide * 32 / (2 dim) sites
constexpr uint32_t kEmpty = 0xFFFFFFFFu;
constexpr int kT = kTileThreads;
constexpr int kWarps = kT / 32;
constexpr int kStage = 64 * WOLFF_WIDE;            // two buffers of 32 * kWide winners per warp (kWide winners per lane and pass)
constexpr uint32_t kBusy = 0x80000000u;            // bond-table state: a warp is filling this tile

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
// Shared-memory atomics by ONE lane of a warp, as plain PTX: nvcc would otherwise wrap them in warp aggregation
// (a vote, a reduction, a prefix scan) that costs more than the atomic.
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned int lds_u32(uint32_t saddr)
{
    unsigned int v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ unsigned int lds_u8(uint32_t saddr)
{
    unsigned int v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ uint4 lds_v4(uint32_t saddr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32(uint32_t saddr, unsigned int v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory");
}
__device__ __forceinline__ void red_shared_add(uint32_t saddr, unsigned int v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned int atom_shared_add(uint32_t saddr, unsigned int v)
{
    unsigned int old;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v) : "memory");
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
    unsigned int krel;                  // ... relative to the first update of the launch
    unsigned int fill_on;               // idle warps fill bond tables (adaptive: off when updates are too short to pay for it)
    unsigned int watcher;               // 1 while some idle worker warp holds the watch (polls the ring without backing off)
    unsigned int ready_tag[2];          // k + 1 when EVERY tile of the CTA has its bits of update k in buffer k & 1
    unsigned int meas_req;              // k + 1 once the monitor has asked for the measurement after update k (in-kernel measurement)
    unsigned int meas_un, meas_ng;      // ... this CTA's sums of one evaluation: unequal forward bonds, negative spins (a CTA
                                        // holds fewer than 2^18 spins: 32 bits, i.e. native shared-memory reductions)
    unsigned long long ihead;           // inbox messages consumed (written by the receiver warp only)
    unsigned long long spill_head, spill_tail;   // running positions in the CTA's global spill list (kept across launches)
};

struct Tally {
    unsigned int attempts = 0;          // claim atomics on shared memory (per lane)
    unsigned int messages = 0;          // messages pushed (per lane)
    unsigned int passes = 0;            // warp passes (lane 0)
    unsigned int inline_passes = 0;     // ... of which at least one lane ran Philox inline (lane 0)
    unsigned int chunks = 0;            // bond-table chunks filled: 32 sites each (lane 0)
    unsigned int ring_pushes = 0;       // sites handed to other warps through the ring (lane 0)
    unsigned int spills = 0;            // ... through the global spill list (lane 0)
#ifdef WOLFF_PROFILE
    unsigned long long cyc_pass = 0;    // cycles inside passes (lane 0)
    unsigned long long lanes = 0;       // sites expanded (lane 0)
#endif
};

// ------------------------------------------------------------------------------------------ geometry of the tiling
// Site i = x + L*y (+ L*L*z), L a power of two.  Tile coordinates (x >> b, ...), tile index t = tx + ntx*ty (+ ...),
// p = (t * A) mod ntiles (A odd: a bijection), owner = p mod G, slot = p div G.  Inside a tile sites are
// row-major again: w = (x & m) + B*(y & m) (+ B*B*(z & m)); local address a = slot * B^dim + w.
template <int DIM>
struct Tiling {
    uint32_t b, m, nt_log, nt_mask, ntiles_mask, A, G, logL, Lmask, ts_log, ts_mask;
    unsigned long long magic;

    __device__ __forceinline__ explicit Tiling(const TileParams &tp)
        : b(tp.tile_log), m((1u << tp.tile_log) - 1u), nt_log(tp.g.geo.logL - tp.tile_log),
          nt_mask((1u << (tp.g.geo.logL - tp.tile_log)) - 1u), ntiles_mask(tp.ntiles - 1u), A(tp.permA), G(tp.G),
          logL(tp.g.geo.logL), Lmask(tp.g.geo.L - 1u), ts_log(DIM * tp.tile_log), ts_mask((1u << (DIM * tp.tile_log)) - 1u),
          magic(tp.magicG) {}

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
    // global site id of a within-tile index, relative to the tile's origin
    __device__ __forceinline__ uint32_t spread(uint32_t w) const
    {
        uint32_t g = (w & m) | (((w >> b) & m) << logL);
        if (DIM == 3) g |= (w >> (2u * b)) << (2u * logL);
        return g;
    }
    // (owner CTA, local address there) of global site i
    __device__ __forceinline__ void locate(uint32_t i, uint32_t &owner, uint32_t &addr) const
    {
        uint32_t x, y, z, slot;
        coords(i, x, y, z);
        place(tile_of(x, y, z), owner, slot);
        addr = (slot << ts_log) | within(x, y, z);
    }
};

// Shared-memory layout of one CTA (offsets follow tiles_smem_bytes()).
struct Layout {
    int8_t *lat;           // slots * B^dim spins
    uint32_t *bond;        // [buf 2][d DIM][slot][B^dim / 32] bond bits (only when tp.tables): bit w of (d, slot) = bond (site w, d)
    uint32_t *halo;        // [buf 2][d DIM][slot][fw] bits of the bonds that enter the tile through its low-d face: bit i of
                           // (d, slot) = bond (n, d), n the -d neighbour (another tile's site) of face site i
    uint32_t *state;       // [buf 2][slot]: k + 1 when the tile's bits of update k (relative to the launch) are complete
    uint32_t *nbrtab;      // [slot][2 DIM]: (owner << 16) | slot of the neighbouring tile
    uint32_t *origin;      // [slot]: global id of the tile's first site
    uint32_t *ring;        // ring_cap entries
    uint32_t *stage;       // kWarps * kStage
    uint32_t wpt;          // bond words per tile and plane
    uint32_t plane;        // bond words per plane (slots * wpt)
    uint32_t fw;           // halo words per tile and direction: max(1, B^(dim-1) / 32)
    uint32_t myslots;      // slots this CTA really owns

    template <int DIM>
    static __device__ __forceinline__ Layout make(const TileParams &tp, unsigned char *base, unsigned int c)
    {
        Layout l;
        l.init<DIM>(tp, base, c);
        return l;
    }
    template <int DIM>
    __device__ __forceinline__ void init(const TileParams &tp, unsigned char *base, unsigned int c)
    {
        const uint32_t ts_log = DIM * tp.tile_log;
        const uint32_t lat_bytes = ((tp.slots << ts_log) + 15u) & ~15u;
        lat = reinterpret_cast<int8_t *>(base);
        uint32_t *q = reinterpret_cast<uint32_t *>(base + lat_bytes);
        wpt = tp.tables ? (1u << (ts_log - 5u)) : 0u;
        plane = tp.slots * wpt;
        bond = q;   q += tp.nbuf * DIM * plane;
        const uint32_t face_log = (DIM - 1) * tp.tile_log;
        fw = tp.tables ? (face_log > 5u ? 1u << (face_log - 5u) : 1u) : 0u;
        halo = q;   q += tp.nbuf * DIM * tp.slots * fw;
        state = q;  q += 2u * tp.slots;
        nbrtab = q; q += 2u * DIM * tp.slots;
        origin = q; q += tp.slots;
        ring = q;   q += tp.ring_cap;
        stage = q;
        myslots = c < tp.ntiles ? (tp.ntiles - c + tp.G - 1u) / tp.G : 0u;
    }
};

template <typename T>
__device__ __forceinline__ T vol(const T *p) { return *reinterpret_cast<const volatile T *>(p); }

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

// Hand n sites (items[0..n), warp-collective) to the other warps of the CTA: the ring, or the spill list when
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
    WOLFF_JITTER_POINT(11);          // reserved, not yet filled
    if (ok) {
        for (unsigned int j = lane; j < n; j += 32u) ring_put(ring + ((base + j) & rmask), items[j]);
        if (lane == 0) tl.ring_pushes += n;
    } else {
        unsigned long long sbase = 0;
        if (lane == 0) sbase = atomicAdd(&sh.spill_tail, (unsigned long long)n);
        sbase = __shfl_sync(kFullMask, sbase, 0);
        uint32_t *const seg = tp.spill + ((size_t)c << tp.spill_log);
        const uint32_t smask = (1u << tp.spill_log) - 1u;
        WOLFF_CHECK(&tp.g.ctl->error, sbase + n - ld_vol64(&sh.spill_head) <= (1ull << tp.spill_log), 3);
        for (unsigned int j = lane; j < n; j += 32u) {
            const unsigned long long pos = sbase + (unsigned long long)j;
            st_relaxed_u32(seg + ((uint32_t)pos & smask), (items[j] << 1) | spill_tag(pos, tp.spill_log));
        }
        if (lane == 0) tl.spills += n;
    }
}

// Called by the lane whose atomic brought sh.pending to zero: the CTA has (for the moment) nothing queued and
// nothing being expanded.  ihead is read BEFORE pending is looked at again, and the receiver raises pending before
// it moves ihead, so pending == 0 here means every message below I is done with all its local progeny.  Publishers
// of one CTA take turns (pub_lock): the claims of an earlier one reach `added` before a later one moves gdone.
__device__ __noinline__ void publish(const TileParams &tp, TShared &sh, unsigned int c)
{
    while (atomicCAS(&sh.pub_lock, 0u, 1u) != 0u) { }
    const unsigned long long I = ld_vol64(&sh.ihead);
    __threadfence_block();
    WOLFF_JITTER_POINT(12);          // between the look at ihead and the look at pending
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

// Back-pressure of the inboxes.  Slot pos of CTA `own` may be written once its receiver has taken message
// pos - in_cap out of it: pos - gihead[own] < in_cap (32-bit running counters; gihead only grows, so a value read
// earlier is a safe lower bound).  Rare: the sender has usually read a recent gihead next to its slot atomic.  The
// receiver never waits for a sender (it only claims, and feeds its ring or spill list), so this wait always ends.
__device__ __noinline__ void wait_inbox(const TileParams &tp, uint32_t own, unsigned int pos)
{
    if (!tp.bp) return;            // worst-case inboxes: nothing can overflow
    unsigned int polls = 0;
    while (pos - ld_relaxed_u32(tp.gihead + own) >= tp.in_cap) {
        if ((++polls & 0x3FFu) == 0u && ld_relaxed_u32(&tp.g.ctl->error) != 0u) return;     // the launch is being aborted
        __nanosleep(64);
    }
}

// ------------------------------------------------------------------------------------------ bond tables
// State a warp keeps about the tile it is filling (warp-uniform registers).
struct Filler {
    unsigned int active = 0, buf = 0, slot = 0, chunk = 0, v = 0;
};

// True when every tile of this CTA has its complete bond table of the update with tag `tag` (warp-collective).
__device__ __forceinline__ bool tables_ready(const TileParams &tp, const Layout &ly, unsigned int buf, unsigned int tag)
{
    const unsigned int lane = threadIdx.x & 31u;
    bool ok = true;
    for (unsigned int base = 0; base < ly.myslots; base += 32u) {
        const unsigned int sl = base + lane;
        if (sl < ly.myslots && vol(ly.state + buf * tp.slots + sl) != tag) ok = false;
    }
    return __all_sync(kFullMask, ok);
}

// One step of table filling by an idle warp (warp-collective): claim a tile that has no bits for the running update
// or the next one, or evaluate 32 more sites of the claimed tile.  Returns false when there is nothing to do.
// A tile is written by the one warp that holds its kBusy claim, so a warp that is called away to expand sites simply
// continues later; a claim that has become useless (the update is over) is dropped.
template <int DIM>
__device__ __forceinline__ bool fill_step(const TileParams &tp, TShared &sh, const Layout &ly, const Tiling<DIM> &tg, Filler &f, Tally &tl)
{
    const GrowthParams &p = tp.g;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int cur = ld_vol(&sh.krel);
    if (!f.active) {
        if (ld_vol(&sh.fill_on) == 0u) return false;
        for (unsigned int t = 0; t < tp.nbuf; ++t) {
            const unsigned int v = cur + t;
            if ((unsigned long long)v >= p.n_updates) break;
            const unsigned int buf = v & (tp.nbuf - 1u), tag = v + 1u;
            for (unsigned int base = 0; base < ly.myslots; base += 32u) {
                const unsigned int sl = base + lane;
                const unsigned int st = sl < ly.myslots ? vol(ly.state + buf * tp.slots + sl) : tag;
                const unsigned int cand = __ballot_sync(kFullMask, st != tag && (st & kBusy) == 0u);
                if (cand == 0u) continue;
                const unsigned int pick = (unsigned int)__ffs((int)cand) - 1u;
                const unsigned int seen = __shfl_sync(kFullMask, st, pick);
                unsigned int ok = 0;
                if (lane == 0) ok = atomicCAS(ly.state + buf * tp.slots + base + pick, seen, kBusy | tag) == seen ? 1u : 0u;
                ok = __shfl_sync(kFullMask, ok, 0);
                if (ok) { f.active = 1u; f.buf = buf; f.slot = base + pick; f.chunk = 0u; f.v = v; }
                return true;       // claimed, or lost the race: either way something is going on
            }
        }
        return false;
    }
    if (f.v < cur || f.v >= cur + tp.nbuf) {   // the update these bits were for is over
        if (lane == 0) st_vol(ly.state + f.buf * tp.slots + f.slot, 0u);
        f.active = 0u;
        return true;
    }
    const unsigned long long u = p.u0 + (unsigned long long)f.v;
    const bool all = tp.thr_all != 0u;
    if (f.chunk < ly.wpt) {
        // 32 sites of the tile: all their forward bonds
        const uint32_t w = f.chunk * 32u + lane;
        const uint32_t gid = vol(ly.origin + f.slot) + tg.spread(w);
        const uint4 blk = philox4x32_10(gid, kDomainBond, (uint32_t)u, (uint32_t)(u >> 32), p.key0, p.key1);
        const unsigned int b0 = __ballot_sync(kFullMask, all || blk.x < tp.thr32);
        const unsigned int b1 = __ballot_sync(kFullMask, all || blk.y < tp.thr32);
        const unsigned int b2 = DIM == 3 ? __ballot_sync(kFullMask, all || blk.z < tp.thr32) : 0u;
        if (lane < (unsigned int)DIM && WOLFF_CHECK(&p.ctl->error, f.buf < tp.nbuf && f.slot < ly.myslots && f.chunk < ly.wpt, 4))
            ly.bond[(f.buf * DIM + lane) * ly.plane + f.slot * ly.wpt + f.chunk] = lane == 0u ? b0 : (lane == 1u ? b1 : b2);
    } else {
        // 32 sites of the low-d face: the bond each of them has with its -d neighbour (owned by that neighbour)
        const uint32_t j = f.chunk - ly.wpt, d = j / ly.fw, i = (j - d * ly.fw) * 32u + lane;
        const uint32_t db = d * tg.b, sh_d = d * tg.logL;
        const uint32_t w = (i & ((1u << db) - 1u)) | ((i >> db) << (db + tg.b));          // face site: coordinate d = 0
        const bool valid = i < (1u << ((DIM - 1) * tg.b));
        const uint32_t gs = vol(ly.origin + f.slot) + tg.spread(valid ? w : 0u);
        const uint32_t gn = (gs & ~(tg.Lmask << sh_d)) | ((((gs >> sh_d) - 1u) & tg.Lmask) << sh_d);
        const uint4 blk = philox4x32_10(gn, kDomainBond, (uint32_t)u, (uint32_t)(u >> 32), p.key0, p.key1);
        const uint32_t r = d == 0u ? blk.x : (d == 1u ? blk.y : blk.z);
        const unsigned int bb = __ballot_sync(kFullMask, valid && (all || r < tp.thr32));
        if (lane == 0 && WOLFF_CHECK(&p.ctl->error, f.buf < tp.nbuf && d < (uint32_t)DIM && f.slot < ly.myslots && j - d * ly.fw < ly.fw, 5))
            ly.halo[((f.buf * DIM + d) * tp.slots + f.slot) * ly.fw + (j - d * ly.fw)] = bb;
    }
    if (lane == 0) ++tl.chunks;
    if (++f.chunk == ly.wpt + DIM * ly.fw) {
        __syncwarp();
        if (lane == 0) { __threadfence_block(); st_vol(ly.state + f.buf * tp.slots + f.slot, f.v + 1u); }
        f.active = 0u;
        __syncwarp();
        if (tables_ready(tp, ly, f.buf, f.v + 1u) && lane == 0) st_vol(&sh.ready_tag[f.buf], f.v + 1u);
    }
    return true;
}

// ------------------------------------------------------------------------------------------ in-kernel measurement
// "+ measurement": E and M of the whole lattice after an update, evaluated where the lattice
// is -- in the CTAs' shared memory -- without leaving the persistent kernel.  The forward bonds (+d) of a tile's
// high-d face end in the low-d face of the next tile, which lives in another CTA: every CTA first copies the low
// faces of its tiles to global memory (tp.faces), all CTAs meet at an arrival counter, then every CTA sums its own
// tiles (16 sites per load; sign-bit XOR + popc as in measure.cu) and adds its two counts to the control block.
// Called by every warp of the CTA but the monitor, between two updates (nothing is queued or in flight).
__device__ __forceinline__ void bar_sync_named(unsigned int id, unsigned int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// Sign bits of up to eight words in ONE population count: the sign bits sit at bits 7, 15, 23, 31 of a word, so word j
// shifted right by j lands on bits 7-j of every byte.  (POPC runs at a quarter of the ALU rate: with one per word the
// sums below were bound by it.)
__device__ __forceinline__ unsigned int merge4(unsigned int a, unsigned int b, unsigned int c, unsigned int d)
{
    return (a & 0x80808080u) | ((b & 0x80808080u) >> 1) | ((c & 0x80808080u) >> 2) | ((d & 0x80808080u) >> 3);
}
__device__ __forceinline__ unsigned int merge4(const uint4 &v) { return merge4(v.x, v.y, v.z, v.w); }
__device__ __forceinline__ uint4 xor4(const uint4 &a, const uint4 &b) { return make_uint4(a.x ^ b.x, a.y ^ b.y, a.z ^ b.z, a.w ^ b.w); }

template <int DIM>
__device__ __noinline__ void measure_phase(const TileParams &tp, TShared &sh, uint32_t lat_s, uint32_t nbr_s, uint32_t myslots, unsigned int c,
                                          unsigned int ptid, unsigned int P, unsigned int krel)
{
    // lat_s: the tiles, nbr_s: the table of neighbouring tiles (shared-window addresses)
    constexpr unsigned int ND = 2u * DIM;
    const Tiling<DIM> tg(tp);
    Control *ctl = tp.g.ctl;
    const uint32_t b = tg.b, B = 1u << b, m = tg.m;
    const uint32_t f_log = (DIM - 1) * b, F = 1u << f_log;            // sites of one face
    const unsigned char *const faces = reinterpret_cast<const unsigned char *>(tp.faces);
    unsigned char *const faces_out = reinterpret_cast<unsigned char *>(tp.faces);
#ifdef WOLFF_PROFILE
    const bool prof = ptid == 0u && c == 1u;
    unsigned long long pt[6] = {0, 0, 0, 0, 0, 0};
    if (prof) pt[0] = globaltimer_ns();
#endif
    // ---- 1. the low faces of my tiles -> global memory.  x = 0 (a byte every B in the tile): one site per lane, so that
    // a warp's loads spread over the banks; y = 0 / z = 0 (runs of B consecutive bytes): four sites per lane.
    for (uint32_t idx = ptid; idx < (myslots << f_log); idx += P) {
        const uint32_t slot = idx >> f_log, f = idx & (F - 1u);
        faces_out[(size_t)((slot * tp.G + c) * DIM) * F + f] = (unsigned char)lds_u8(lat_s + (slot << tg.ts_log) + (f << b));
    }
    {
        unsigned int *const fout = reinterpret_cast<unsigned int *>(tp.faces);
        const uint32_t f4_log = f_log - 2u;                           // log2 of the words of one face (B >= 4)
        const uint32_t nwords = (myslots * (DIM - 1)) << f4_log;
        for (uint32_t idx = ptid; idx < nwords; idx += P) {
            const uint32_t sd = idx >> f4_log, slot = sd / (DIM - 1), d = 1u + (sd - slot * (DIM - 1)), f0 = (idx & ((1u << f4_log) - 1u)) << 2;
            const uint32_t low = (1u << (d * b)) - 1u;                // f = x | z << b (y = 0)  or  x | y << b (z = 0)
            fout[(((slot * tp.G + c) * DIM + d) << f4_log) + (f0 >> 2)] =
                lds_u32(lat_s + (slot << tg.ts_log) + ((f0 & low) | ((f0 >> (d * b)) << ((d + 1u) * b))));
        }
    }
    __threadfence();
#ifdef WOLFF_PROFILE
    if (prof) pt[1] = globaltimer_ns();
#endif
    bar_sync_named(1u, P);
#ifdef WOLFF_PROFILE
    if (prof) pt[2] = globaltimer_ns();
#endif
    // (summing the bonds inside the tiles before this wait instead of after it changes nothing: measured)
    if (ptid == 0u) {
        atomicAdd(&ctl->meas_arrive_a, 1u);
        const unsigned int target = (krel + 1u) * tp.G;
        unsigned int polls = 0;
        while (ld_acquire_u32(&ctl->meas_arrive_a) != target)
            if ((++polls & 0xFFu) == 0u && ld_relaxed_u32(&ctl->error) != 0u) break;
    }
    bar_sync_named(1u, P);
#ifdef WOLFF_PROFILE
    if (prof) pt[3] = globaltimer_ns();
#endif
    // ---- 2. my tiles: negative spins and unequal forward bonds
    unsigned int un = 0, ng = 0;
    auto face_of = [&](uint32_t slot, uint32_t d) -> const unsigned char * {
        const uint32_t nt = lds_u32(nbr_s + (slot * ND + 2u * d) * 4u);       // (owner << 16) | slot of the +d neighbouring tile
        return faces + (size_t)(((nt & 0xFFFFu) * tp.G + (nt >> 16)) * DIM + d) * F;
    };
    if (b >= 4u) {
        // (a) the bonds inside my tiles: shared memory only, 16 sites per load
        const uint32_t cpt_log = tg.ts_log - 4u, total = myslots << cpt_log;
        // spins are +1 / -1 bytes, so a signed 8-bit dot product of two words IS the sum of four bond products s_i s_j
        // (and against 0x01010101 the sum of four spins): one IDP4A per word and direction instead of mask, shift, merge
        // and population count.  #unequal = (#bonds - sum of products) / 2, #negative = (#spins - sum of spins) / 2.
        int dps = 0, sps = 0;
        unsigned int nch = 0;
        auto chunk = [&](uint32_t ch) {
            const uint32_t slot = ch >> cpt_log, w0 = (ch & ((1u << cpt_log) - 1u)) << 4;
            const uint32_t x0 = w0 & m, y = (w0 >> b) & m, z = DIM == 3 ? (w0 >> (2u * b)) : 0u;
            const uint32_t at = lat_s + (slot << tg.ts_log) + w0;
            const uint4 a = lds_v4(at);
            // forward rows: inside the tile, else the row itself (a product of a spin with itself counts as an equal
            // pair, i.e. nothing unequal; the bond is counted in (b))
            const uint4 by = lds_v4(y + 1u < B ? at + B : at);
            const uint4 bz = DIM == 3 ? lds_v4(z + 1u < B ? at + (B << b) : at) : a;
            // +x: the 16 sites shifted by one byte; the 17th is the next site of the row -- or, at the end of the row, a
            // copy of the 16th, so that the bond across the tile border counts nothing here
            const uint32_t nb = x0 + 16u < B ? lds_u8(at + 16u) : (a.w >> 24);
            sps = __dp4a((int)a.x, 0x01010101, sps); sps = __dp4a((int)a.y, 0x01010101, sps);
            sps = __dp4a((int)a.z, 0x01010101, sps); sps = __dp4a((int)a.w, 0x01010101, sps);
            dps = __dp4a((int)a.x, (int)__funnelshift_r(a.x, a.y, 8), dps); dps = __dp4a((int)a.y, (int)__funnelshift_r(a.y, a.z, 8), dps);
            dps = __dp4a((int)a.z, (int)__funnelshift_r(a.z, a.w, 8), dps); dps = __dp4a((int)a.w, (int)__funnelshift_r(a.w, nb, 8), dps);
            dps = __dp4a((int)a.x, (int)by.x, dps); dps = __dp4a((int)a.y, (int)by.y, dps);
            dps = __dp4a((int)a.z, (int)by.z, dps); dps = __dp4a((int)a.w, (int)by.w, dps);
            if (DIM == 3) {
                dps = __dp4a((int)a.x, (int)bz.x, dps); dps = __dp4a((int)a.y, (int)bz.y, dps);
                dps = __dp4a((int)a.z, (int)bz.z, dps); dps = __dp4a((int)a.w, (int)bz.w, dps);
            }
            ++nch;
        };
        uint32_t ch = ptid;
        for (; ch + P < total; ch += 2u * P) { chunk(ch); chunk(ch + P); }
        if (ch < total) chunk(ch);
        un += (unsigned int)(((int)(nch * 16u * (unsigned int)DIM) - dps) >> 1);
        ng += (unsigned int)(((int)(nch * 16u) - sps) >> 1);
        // (b1) the bonds across the +x border of a tile: my site x = B - 1 against the next tile's x = 0 (global memory),
        // one site per lane, eight global loads in flight per lane (a trip costs one L2 round trip, not eight)
        constexpr uint32_t kSites = 8;
        const uint32_t nsites = myslots << f_log;
        for (uint32_t i0 = ptid; i0 < nsites; i0 += P * kSites) {
            unsigned int theirs[kSites], mine[kSites];
#pragma unroll
            for (uint32_t j = 0; j < kSites; ++j) {
                const uint32_t idx = i0 + j * P, ii = idx < nsites ? idx : 0u, slot = ii >> f_log, f = ii & (F - 1u);
                theirs[j] = __ldcg(face_of(slot, 0u) + f);
                mine[j] = lds_u8(lat_s + (slot << tg.ts_log) + (f << b) + m);
            }
#pragma unroll
            for (uint32_t j = 0; j < kSites; ++j)
                if (i0 + j * P < nsites) un += ((mine[j] ^ theirs[j]) >> 7) & 1u;
        }
        // (b2) across the +y / +z borders: 16 sites per load on both sides, four tasks per trip, their global loads first
        const uint32_t g_log = f_log - 4u;                            // log2 of the 16-site groups of one face
        const uint32_t tasks = (myslots * (DIM - 1)) << g_log;
        constexpr uint32_t kTasks = 4;
        for (uint32_t t0 = ptid; t0 < tasks; t0 += P * kTasks) {
            uint4 theirs[kTasks], mine[kTasks];
            bool on[kTasks];
#pragma unroll
            for (uint32_t j = 0; j < kTasks; ++j) {
                const uint32_t t = t0 + j * P;
                on[j] = t < tasks;
                const uint32_t tt = on[j] ? t : 0u, sd = tt >> g_log, slot = sd / (DIM - 1), d = 1u + (sd - slot * (DIM - 1));
                const uint32_t f0 = (tt & ((1u << g_log) - 1u)) << 4, low = (1u << (d * b)) - 1u;
                theirs[j] = __ldcg(reinterpret_cast<const uint4 *>(face_of(slot, d) + f0));
                mine[j] = lds_v4(lat_s + (slot << tg.ts_log) + ((f0 & low) | ((f0 >> (d * b)) << ((d + 1u) * b)) | (m << (d * b))));   // coordinate d = B - 1
            }
#pragma unroll
            for (uint32_t j = 0; j < kTasks; ++j)
                if (on[j]) un += (unsigned int)((16 - __dp4a((int)mine[j].x, (int)theirs[j].x, __dp4a((int)mine[j].y, (int)theirs[j].y,
                                                     __dp4a((int)mine[j].z, (int)theirs[j].z, __dp4a((int)mine[j].w, (int)theirs[j].w, 0))))) >> 1);
        }
    } else {
        // tiles narrower than a 16-byte load (test configurations): one site at a time
        const uint32_t total = myslots << tg.ts_log;
        for (uint32_t idx = ptid; idx < total; idx += P) {
            const uint32_t slot = idx >> tg.ts_log, w = idx & tg.ts_mask;
            const uint32_t s0b = lds_u8(lat_s + idx);
            ng += s0b >> 7;
#pragma unroll
            for (uint32_t d = 0; d < (uint32_t)DIM; ++d) {
                const uint32_t low = (1u << (d * b)) - 1u;
                uint32_t nbv;
                if (((w >> (d * b)) & m) != m) nbv = lds_u8(lat_s + idx + (1u << (d * b)));
                else nbv = __ldcg(face_of(slot, d) + ((w & low) | ((w >> ((d + 1u) * b)) << (d * b))));
                un += ((s0b ^ nbv) >> 7) & 1u;
            }
        }
    }
    un = __reduce_add_sync(kFullMask, un);
    ng = __reduce_add_sync(kFullMask, ng);
    if ((threadIdx.x & 31u) == 0u) {
        if (un) red_shared_add(smem_addr(&sh.meas_un), un);
        if (ng) red_shared_add(smem_addr(&sh.meas_ng), ng);
    }
#ifdef WOLFF_PROFILE
    if (prof) pt[4] = globaltimer_ns();
#endif
    bar_sync_named(1u, P);
#ifdef WOLFF_PROFILE
    if (prof) {
        pt[5] = globaltimer_ns();
        // [2] faces  [3] wait for the CTA's warps  [4] wait for all CTAs  [5] sums  [6] wait for the CTA's warps again
        for (int i = 0; i < 5; ++i) atomicAdd(&ctl->stats[2 + i], pt[i + 1] - pt[i]);
    }
#endif
    if (ptid == 0u) {
        const unsigned long long tun = ld_vol(&sh.meas_un), tng = ld_vol(&sh.meas_ng);
        st_vol(&sh.meas_un, 0u);
        st_vol(&sh.meas_ng, 0u);
        if (tun) atomicAdd(&ctl->meas_unequal, tun);
        if (tng) atomicAdd(&ctl->meas_negative, tng);
        __threadfence();
        atomicAdd(&ctl->meas_arrive_b, 1u);
    }
}

// ------------------------------------------------------------------------------------------ worker warp
// Expands sites owned by this CTA until the launch is over (A2-A5 on shared memory), one lane per bond: a warp
// holds up to S = 32 / (2*DIM) sites per pass (8 in 2D, 5 in 3D) and lane (q, k) tests the bond from site q to its
// neighbour k (k = 2d: +d, k = 2d + 1: -d).  Per lane and pass: one neighbour address, one bond bit (table, else one
// Philox block), one LDS of the neighbour's spin, one ATOMS; per warp one ballot and one hand-over of the winners
// through its private stage.  An update waits for the dependent chain of these passes (one per BFS level the CTA
// takes part in), so the loop is written for instruction count, not for lane utilisation.
//
// Accounting (sh.pending): a warp that took n sites from the ring holds n units until it runs dry, whatever its
// private frontier does in between; only the sites it hands to other warps are added.
struct WorkerState {
    uint32_t a[kWide] = {};      // local addresses of this lane's sites
    unsigned int nsites = 0;     // sites held by the warp (warp-uniform); lanes of group q < nsites work
    unsigned int units = 0;      // what the warp owes sh.pending when it runs dry
    int s0 = 1;
    uint32_t u_lo = 0, u_hi = 0, krel = 0;
    unsigned int mywon = 0;      // spins this lane claimed since the warp last ran dry
    unsigned int sbuf = 0;       // which half of stage[] the next pass writes
};

// Passes until the warp holds no site (READY) or for at most 32 passes (!READY: the caller looks again whether the
// tables have become complete).  POS: the seed spin s0 of the running update is +1 (claim = OR), else -1 (AND).
// READY: every tile of this CTA has its bond table of this update, so no state is checked and no Philox runs here.
// BP: the inboxes are smaller than what one update can send (knob "inbox_log"), so a sender checks the capacity
// before it stores a message (wait_inbox).  With worst-case inboxes (the default) the check does not exist: measured
// on B200 the check costs 15 % (C3) / 40 % (C5a) of the throughput -- one more L2 load in flight per message and a
// call in the pass -- while the size of the inboxes (2^12 against 2^16 entries per CTA at C5a) makes no difference.
template <int DIM, bool POS, bool READY, bool BP>
__device__ __forceinline__ void run_passes(const TileParams &tp, TShared &sh, const Layout &ly, const Tiling<DIM> &tg, uint32_t *stage,
                                           unsigned int c, WorkerState &ws, Tally &tl)
{
    constexpr unsigned int ND = 2u * DIM, S = 32u / ND, W = kWide;
    const GrowthParams &p = tp.g;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int lt = (1u << lane) - 1u;
    const unsigned int q = lane / ND, k = lane - q * ND, d = k >> 1, sgn = k & 1u;
    const uint32_t db = d * tg.b, lowmask = (1u << db) - 1u;
    const uint32_t edge = sgn ? 0u : tg.m;                                   // within-tile coordinate at which the neighbour is in the next tile
    const uint32_t step_in = sgn ? 0u - (1u << db) : (1u << db);             // a -> neighbour in the same tile
    const uint32_t step_out = sgn ? (tg.m << db) : 0u - (tg.m << db);        // w -> within-tile index in the neighbouring tile
    const uint32_t sh_d = d * tg.logL, fmask = tg.Lmask << sh_d, delta = sgn ? 0xFFFFFFFFu : 1u;
    const uint32_t in_mask = tp.in_cap - 1u;
    // shared-window addresses: every shared-memory access of the loop is a plain ld/st/atom.shared on one of these
    const uint32_t lat_s = smem_addr(ly.lat), pend_s = smem_addr(&sh.pending), claimed_s = smem_addr(&sh.claimed);
    const uint32_t nbr_s = smem_addr(ly.nbrtab + k), origin_s = smem_addr(ly.origin), stage_s = smem_addr(stage);
    const bool tables = tp.tables != 0u;
    const uint32_t krel = ws.krel, u_lo = ws.u_lo, u_hi = ws.u_hi;
    const uint32_t bond_s = smem_addr(ly.bond + ((krel & (tp.nbuf - 1u)) * DIM + d) * ly.plane);    // plane (buffer of krel, d)
    const uint32_t halo_s = smem_addr(ly.halo + ((krel & (tp.nbuf - 1u)) * DIM + d) * tp.slots * ly.fw);
    const uint32_t state_s = smem_addr(ly.state + (krel & (tp.nbuf - 1u)) * tp.slots);
    const uint32_t fw4 = ly.fw * 4u;
    const uint32_t tag = krel + 1u;
    const unsigned int s0w = POS ? 0x01010101u : 0xFFFFFFFFu;                // the seed spin in every byte
    const uint32_t cself = c << 16;
    uint32_t a[W];
#pragma unroll
    for (unsigned int j = 0; j < W; ++j) a[j] = ws.a[j];
    unsigned int nsites = ws.nsites, mywon = ws.mywon, sbuf = ws.sbuf;
    unsigned int msg_pos[W];           // messages whose inbox slots are on their way back from L2
    unsigned int msg_seen[W];          // ... and what the owner's receiver had consumed at about that time (back-pressure)
    uint32_t msg_own[W], msg_na[W];
    bool msg_valid[W];
#pragma unroll
    for (unsigned int j = 0; j < W; ++j) { msg_pos[j] = msg_seen[j] = 0; msg_own[j] = msg_na[j] = 0; msg_valid[j] = false; }
    unsigned int budget = 32u;

    auto send = [&](unsigned int j) {
        WOLFF_JITTER_POINT(13);      // slot counted in gtail, message not yet stored
        if (BP && msg_pos[j] - msg_seen[j] >= tp.in_cap) wait_inbox(tp, msg_own[j], msg_pos[j]);
        st_relaxed_u64(tp.inbox + ((size_t)msg_own[j] << tp.in_log) + (msg_pos[j] & in_mask),
                       pack_msg(kKindClaim, (msg_pos[j] >> tp.in_log) & 1u, krel, msg_na[j], POS ? 1 : -1));
        msg_valid[j] = false;
    };

    // one pass; 0: go on, 1: the warp ran dry, 2: back to the caller (!READY only).  Lane (q, k) works on the sites
    // q, q + S, ... (W of them): W independent dependent-chains side by side, so a pass over W*S sites takes little
    // longer than a pass over S.
    auto pass = [&]() -> int {
#ifdef WOLFF_PROFILE
        const long long tp0 = clock64();
        tl.lanes += nsites;
#endif
        bool have[W], local[W], bit[W];
        uint32_t w[W], slot[W], na[W], own[W], bi[W];
        unsigned int st[W], bw[W], spw[W], bytemask[W], old[W];
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) {
            have[j] = q < S && q + j * S < nsites;       // lanes 30, 31 in 3D (q = S) never hold a site
            // ---- A2: this lane's neighbour: same tile (a +- stride) or across a tile border (table of neighbouring tiles)
            w[j] = a[j] & tg.ts_mask;
            slot[j] = a[j] >> tg.ts_log;
            const bool inside = ((w[j] >> db) & tg.m) != edge;
            uint32_t nt = cself;
            if (!inside) nt = lds_u32(nbr_s + slot[j] * (ND * 4u));   // lanes without a site hold a stale (valid) address: their loads are harmless
            na[j] = inside ? a[j] + step_in : (((nt & 0xFFFFu) << tg.ts_log) | (w[j] + step_out));
            own[j] = nt >> 16;
            local[j] = own[j] == c;
            // ---- A3, table.  The bond to the +d neighbour is owned by this site (bit a of plane d); the bond to the -d
            // neighbour is owned by that neighbour: bit na of plane d when it is in the same tile, else the halo bit of
            // this site's place on the tile's low-d face.
            const bool use_halo = sgn != 0u && !inside;
            const uint32_t fidx = (w[j] & lowmask) | ((w[j] >> (db + tg.b)) << db);
            bi[j] = use_halo ? fidx : (sgn ? na[j] : a[j]);
            const uint32_t baddr = (use_halo ? halo_s + slot[j] * fw4 : bond_s) + ((bi[j] >> 5) << 2);
            st[j] = tag; bw[j] = 0; spw[j] = 0;
            if (READY) {
                bw[j] = lds_u32(baddr);
            } else if (tables) {
                st[j] = lds_u32(state_s + slot[j] * 4u);                              // state first: see fill_step()
                bw[j] = lds_u32(baddr);
            }
            if (have[j] && !WOLFF_CHECK(&p.ctl->error, local[j] ? na[j] < (ly.myslots << tg.ts_log) : own[j] < tp.G, 1)) { have[j] = false; local[j] = true; na[j] = 0u; }
            if (local[j]) spw[j] = lds_u32(lat_s + (na[j] & ~3u));                    // gather
            bytemask[j] = 0xFFu << ((na[j] & 3u) * 8u);
        }
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) bit[j] = have[j] && (bw[j] & (1u << (bi[j] & 31u))) != 0u;
        if (!READY) {
            // ---- A3, inline: the same Philox block the table would hold
            bool need_inline[W];
            bool any = false;
#pragma unroll
            for (unsigned int j = 0; j < W; ++j) {
                const bool tabled = tables && st[j] == tag;
                bit[j] = bit[j] && tabled;
                need_inline[j] = have[j] && !tabled;
                any = any || need_inline[j];
            }
            if (__any_sync(kFullMask, any)) {
#pragma unroll
                for (unsigned int j = 0; j < W; ++j) {
                    if (need_inline[j]) {
                        const uint32_t gs = lds_u32(origin_s + slot[j] * 4u) + tg.spread(w[j]);
                        const uint32_t gn = (gs & ~fmask) | ((((gs >> sh_d) + delta) & tg.Lmask) << sh_d);
                        const uint4 blk = philox4x32_10(sgn ? gn : gs, kDomainBond, u_lo, u_hi, p.key0, p.key1);
                        const uint32_t r = selp_u32(blk.x, selp_u32(blk.y, blk.z, d == 1u), d == 0u);
                        bit[j] = r < tp.thr32 || tp.thr_all != 0u;
                    }
                }
                if (lane == 0) ++tl.inline_passes;
            }
        }
        bool cand_r[W];
        bool any_r = false;
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) {
            const bool cand_l = bit[j] && local[j] && ((spw[j] ^ s0w) & bytemask[j]) == 0u;
            cand_r[j] = bit[j] && !local[j];
            any_r = any_r || cand_r[j] || msg_valid[j];
            // ---- A4 inside the territory: the same idempotent atomic as claim_and_flip(), on shared memory
            old[j] = ~s0w;
            if (POS) asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %3, 0;\n @p atom.shared.or.b32 %0, [%1], %2;\n}"
                                  : "+r"(old[j]) : "r"(lat_s + (na[j] & ~3u)), "r"(0xFEFEFEFEu & bytemask[j]), "r"((unsigned int)cand_l) : "memory");
            else     asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %3, 0;\n @p atom.shared.and.b32 %0, [%1], %2;\n}"
                                  : "+r"(old[j]) : "r"(lat_s + (na[j] & ~3u)), "r"(~(0xFEFEFEFEu & bytemask[j])), "r"((unsigned int)cand_l) : "memory");
            tl.attempts += cand_l ? 1u : 0u;
        }
        // ---- A4 across the territory border: a message to the owner (slot by one L2 atomic, then one 8-byte store).
        // The store waits for the atomic's round trip, so it is issued one pass later (or when the warp runs dry):
        // the slot is counted in gtail -- the atomic has returned -- before the pass that caused it stops being pending.
        if (__any_sync(kFullMask, any_r)) {
#pragma unroll
            for (unsigned int j = 0; j < W; ++j) {
                if (msg_valid[j]) send(j);
                // the atomic writes the loop-carried register itself (an in-out operand, 32 bits: a 64-bit result needs an
                // aligned register pair, which ptxas then copies out of -- and a copy waits for the L2 round trip here)
                if (BP)
                    asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %3, 0;\n @p atom.global.add.u32 %0, [%2], 1;\n"
                                 " @p ld.relaxed.gpu.global.u32 %1, [%4];\n}"
                                 : "+r"(msg_pos[j]), "+r"(msg_seen[j]) : "l"(tp.gtail + own[j]), "r"((unsigned int)cand_r[j]), "l"(tp.gihead + own[j])
                                 : "memory");
                else
                    asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %2, 0;\n @p atom.global.add.u32 %0, [%1], 1;\n}"
                                 : "+r"(msg_pos[j]) : "l"(tp.gtail + own[j]), "r"((unsigned int)cand_r[j]) : "memory");
                if (cand_r[j]) {
                    msg_own[j] = own[j];
                    msg_na[j] = na[j];
                    msg_valid[j] = true;
                    ++tl.messages;
                }
            }
        }
        bool won[W];
        unsigned int wb[W];
        unsigned int total = 0;
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) {
            won[j] = ((old[j] ^ s0w) & bytemask[j]) == 0u;
            mywon += won[j] ? 1u : 0u;
        }
#ifdef WOLFF_PROFILE
        if (lane == 0) ++tl.passes;
#endif
        // ---- A5: compact the winners; the first W*S are this warp's next pass, the rest goes to the ring
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) { wb[j] = __ballot_sync(kFullMask, won[j]); total += __popc(wb[j]); }
        if (total == 0u) return 1;                               // the warp runs dry
        uint32_t *const st_out = stage + sbuf;
        const uint32_t out_s = stage_s + sbuf * 4u;
        const unsigned int sbuf_prev = sbuf; (void)sbuf_prev;
        sbuf ^= 32u * W;
        unsigned int before = 0;
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) {
            if (won[j] && WOLFF_CHECK(&p.ctl->error, sbuf_prev + before + __popc(wb[j] & lt) < (unsigned int)kStage, 8))
                sts_u32(out_s + (before + __popc(wb[j] & lt)) * 4u, na[j]);
            before += __popc(wb[j]);
        }
        __syncwarp();
        nsites = total < W * S ? total : W * S;
#pragma unroll
        for (unsigned int j = 0; j < W; ++j)
            if (q < S && q + j * S < nsites) a[j] = lds_u32(out_s + (q + j * S) * 4u);
        if (total > W * S) {
            if (lane == 0) red_shared_add(pend_s, total - W * S);    // counted before another warp can see them
            hand_over(tp, sh, ly.ring, st_out + W * S, total - W * S, c, tl);
        }
#ifdef WOLFF_PROFILE
        tl.cyc_pass += (unsigned long long)(clock64() - tp0);
#endif
        if (!READY && --budget == 0u) {
            // back to the caller: have the tables become complete?  (messages in flight leave first)
#pragma unroll
            for (unsigned int j = 0; j < W; ++j) if (msg_valid[j]) send(j);
            ws.nsites = nsites; ws.mywon = mywon; ws.sbuf = sbuf;
#pragma unroll
            for (unsigned int j = 0; j < W; ++j) ws.a[j] = a[j];
            return 2;
        }
        return 0;
    };
    // two passes per trip: the loop-back (and the YIELD ptxas puts at the head of such loops) costs about 50 cycles
    int status;
    for (;;) {
        status = pass();
        if (status != 0) break;
        status = pass();
        if (status != 0) break;
    }
    if (status == 2) return;
    // ---- dry: the messages leave, the claims become visible to the publisher, then the warp's units stop being pending
#pragma unroll
    for (unsigned int j = 0; j < W; ++j) if (msg_valid[j]) send(j);
    const unsigned int wsum = __reduce_add_sync(kFullMask, mywon);
    WOLFF_JITTER_POINT(14);          // messages sent, units not yet handed back
    if (lane == 0) {
        if (wsum) red_shared_add(claimed_s, wsum);
        __threadfence_block();
        const unsigned int before = atom_shared_add(pend_s, 0u - ws.units);
        if (before == ws.units) publish(tp, sh, c);
    }
    ws.nsites = 0u; ws.mywon = 0u; ws.sbuf = sbuf;
}

template <int DIM>
__device__ __forceinline__ void worker_warp(const TileParams &tp, TShared &sh, const Layout &ly, uint32_t *stage, unsigned int c, Tally &tl)
{
    constexpr unsigned int ND = 2u * DIM, S = 32u / ND, W = kWide;
    const GrowthParams &p = tp.g;
    const Tiling<DIM> tg(tp);
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int q = lane / ND;
    const uint32_t rmask = tp.ring_cap - 1u;
    const bool tables = tp.tables != 0u;
    bool watcher = false;        // this warp holds the CTA's watch: it polls the ring without sleeping or filling
    WorkerState ws;
    unsigned int idle = 0;
    Filler fl;
    // in-kernel measurement: every warp of the CTA but the monitor takes part
    const unsigned int warp = threadIdx.x >> 5;
    const unsigned int P = c == 0u ? kT - 32u : kT, ptid = c == 0u ? (warp - 1u) * 32u + lane : threadIdx.x;
    unsigned int meas_done = 0;

    for (;;) {
        // ---- take up to S sites from the ring, else from the spill list; with neither, fill bond tables or sleep
        unsigned int n = 0, h = 0, from_spill = 0, stop = 0, mreq = 0;
        unsigned long long sh_pos = 0;
        if (lane == 0) {
            // one 64-bit load: a consistent (head, tail) pair; the loads of a poll are independent
            const unsigned long long ht = ld_vol64(reinterpret_cast<const unsigned long long *>(&sh.head));
            sh_pos = ld_vol64(&sh.spill_head);
            const unsigned long long st = ld_vol64(&sh.spill_tail);
            stop = ld_vol(&sh.stop);
            mreq = ld_vol(&sh.meas_req);
            h = (unsigned int)ht;
            const unsigned int t = (unsigned int)(ht >> 32);
            if (t != h) {
                n = t - h < W * S ? t - h : W * S;
                if (atomicCAS(&sh.head, h, h + n) != h) { n = 0; stop = 0; }
            } else if (st != sh_pos) {
                n = st - sh_pos < (unsigned long long)(W * S) ? (unsigned int)(st - sh_pos) : W * S;
                if (atomicCAS(&sh.spill_head, sh_pos, sh_pos + n) == sh_pos) from_spill = 1; else { n = 0; stop = 0; }
            }
        }
        n = __shfl_sync(kFullMask, n, 0);
        if (n == 0u) {
            mreq = __shfl_sync(kFullMask, mreq, 0);
            if (mreq != meas_done) {                                   // the update is over everywhere: measure (see measure_phase)
                measure_phase<DIM>(tp, sh, smem_addr(ly.lat), smem_addr(ly.nbrtab), ly.myslots, c, ptid, P, mreq - 1u);
                meas_done = mreq;
                continue;
            }
            if (__shfl_sync(kFullMask, stop, 0)) break;                // launch over
            // one idle warp per CTA holds the watch: it does nothing but poll the ring, so what the receiver (or a warp
            // with more winners than it can keep) hands over starts at once; the watch passes on when its holder finds work
            if (!watcher) {
                unsigned int got = 0;
                if (lane == 0) got = atomicCAS(&sh.watcher, 0u, 1u) == 0u ? 1u : 0u;
                watcher = __shfl_sync(kFullMask, got, 0) != 0u;
            }
            if (watcher) continue;
            if (tables && fill_step<DIM>(tp, sh, ly, tg, fl, tl)) { idle = 0; continue; }
            // idle warps share the SM's issue slots and load/store pipe with the working ones: back off
            ++idle;
            if (idle > 2u) __nanosleep(idle < 8u ? 64u : (idle < 16u ? 256u : tp.idle_ns));
            continue;
        }
        idle = 0;
        WOLFF_JITTER_POINT(15);      // entries acquired (head moved), not yet taken out of their slots
        if (watcher) { watcher = false; if (lane == 0) st_vol(&sh.watcher, 0u); }
        h = __shfl_sync(kFullMask, h, 0);
        from_spill = __shfl_sync(kFullMask, from_spill, 0);
        sh_pos = __shfl_sync(kFullMask, sh_pos, 0);
        uint32_t ent = 0;
        if (lane < n) {
            unsigned int spins = 0;
            if (!from_spill) {
                uint32_t *slot = ly.ring + ((h + lane) & rmask);
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
#pragma unroll
        for (unsigned int j = 0; j < W; ++j) ws.a[j] = __shfl_sync(kFullMask, ent, (q + j * S) & 31u);
        ws.nsites = n;
        ws.units = n;
        // the update these sites belong to (written by the receiver before it fed the ring)
        ws.s0 = *reinterpret_cast<volatile int *>(&sh.s0);
        ws.u_lo = ld_vol(&sh.u_lo);
        ws.u_hi = ld_vol(&sh.u_hi);
        ws.krel = ld_vol(&sh.krel);
        while (ws.nsites != 0u) {
            const bool ready = tables && ld_vol(&sh.ready_tag[ws.krel & (tp.nbuf - 1u)]) == ws.krel + 1u;
            if (tp.bp) {
                if (ws.s0 > 0) {
                    if (ready) run_passes<DIM, true, true, true>(tp, sh, ly, tg, stage, c, ws, tl);
                    else run_passes<DIM, true, false, true>(tp, sh, ly, tg, stage, c, ws, tl);
                } else {
                    if (ready) run_passes<DIM, false, true, true>(tp, sh, ly, tg, stage, c, ws, tl);
                    else run_passes<DIM, false, false, true>(tp, sh, ly, tg, stage, c, ws, tl);
                }
            } else if (ws.s0 > 0) {
                if (ready) run_passes<DIM, true, true, false>(tp, sh, ly, tg, stage, c, ws, tl);
                else run_passes<DIM, true, false, false>(tp, sh, ly, tg, stage, c, ws, tl);
            } else {
                if (ready) run_passes<DIM, false, true, false>(tp, sh, ly, tg, stage, c, ws, tl);
                else run_passes<DIM, false, false, false>(tp, sh, ly, tg, stage, c, ws, tl);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ receiver warp
// Polls the CTA's inbox; makes the claims other CTAs (and the monitor: the seed site, A1) ask for, on its own
// shared memory; feeds the ring.  A message names the site by its local address in THIS CTA.
template <int DIM>
__device__ __forceinline__ void receiver_warp(const TileParams &tp, TShared &sh, const Layout &ly, uint32_t *stage, unsigned int c, Tally &tl)
{
    const GrowthParams &p = tp.g;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int lt = (1u << lane) - 1u;
    const uint32_t in_mask = tp.in_cap - 1u;
    const unsigned long long *const box = tp.inbox + ((size_t)c << tp.in_log);
    unsigned long long ih = ld_vol64(&sh.ihead);
    unsigned int polls = 0;
    // adaptive table filling: mean time per update between two updates this CTA hears of
    unsigned long long last_t = globaltimer_ns();
    unsigned int last_k = 0;
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
        const unsigned int ctlb = __ballot_sync(kFullMask, mine && kind == kKindExit);
        if (ctlb != 0u) {
            // sent by the monitor when an update is complete and nothing is queued anywhere: leave (site field 0),
            // or take part in the measurement after update krel (site field 1)
            const unsigned int src = (unsigned int)__ffs((int)ctlb) - 1u;
            const unsigned int what = __shfl_sync(kFullMask, lo >> 1, src), krel_m = __shfl_sync(kFullMask, hi & (kMaxK - 1u), src);
            ih += (unsigned long long)k;
            if (lane == 0) { st_vol64(&sh.ihead, ih); st_relaxed_u32(tp.gihead + c, (unsigned int)ih); atomicMax(tp.gdone + c, ih); }
            if (what == 1u) {
                if (lane == 0) { __threadfence_block(); st_vol(&sh.meas_req, krel_m + 1u); }
                __syncwarp();
                measure_phase<DIM>(tp, sh, smem_addr(ly.lat), smem_addr(ly.nbrtab), ly.myslots, c, lane, c == 0u ? kT - 32u : kT, krel_m);
                continue;
            }
            break;
        }
        const uint32_t addr = lo >> 1;
        int s0 = (lo & 1u) ? -1 : 1;
        bool win = false;
        if (mine && WOLFF_CHECK(&p.ctl->error, addr < (ly.myslots << (DIM * tp.tile_log)) && (unsigned long long)(hi & (kMaxK - 1u)) < p.n_updates, 2)) {
            if (kind == kKindSeed) s0 = (int)vol(reinterpret_cast<const signed char *>(ly.lat) + addr);   // A1: the seed spin
            win = claim_and_flip(ly.lat, addr, s0);
            ++tl.attempts;
        }
        const unsigned int wb = __ballot_sync(kFullMask, win);
        const unsigned int w = __popc(wb);
        const int s0u = __shfl_sync(kFullMask, s0, 0);
        const unsigned int krel = __shfl_sync(kFullMask, hi & (kMaxK - 1u), 0);
        ih += (unsigned long long)k;
        if (lane == 0) {
            st_relaxed_u32(tp.gihead + c, (unsigned int)ih);     // these slots may be written again (back-pressure)
            const unsigned long long u = p.u0 + (unsigned long long)krel;
            *reinterpret_cast<volatile int *>(&sh.s0) = s0u;
            st_vol(&sh.u_lo, (uint32_t)u);
            st_vol(&sh.u_hi, (uint32_t)(u >> 32));
            st_vol(&sh.krel, krel);
            atomicAdd(&sh.pending, w + 1u);            // the winners, and a token that keeps the CTA busy until they are queued
            if (w) atomicAdd(&sh.claimed, w);
            __threadfence_block();
            WOLFF_JITTER_POINT(16);                    // pending raised, ihead not yet moved
            st_vol64(&sh.ihead, ih);                   // after pending: see publish()
            __threadfence_block();
        }
        if (win) stage[__popc(wb & lt)] = addr;
        WOLFF_JITTER_POINT(17);
        __syncwarp();
        if (w) hand_over(tp, sh, ly.ring, stage, w, c, tl);
        __syncwarp();
        if (lane == 0) {
            const unsigned int before = atomicSub(&sh.pending, 1u);
            if (before == 1u) publish(tp, sh, c);
            if (tp.fill_mode == 1u && krel != last_k) {
                const unsigned long long now = globaltimer_ns();
                st_vol(&sh.fill_on, now - last_t > (unsigned long long)(krel - last_k) * tp.fill_min_ns ? 1u : 0u);
                last_t = now;
                last_k = krel;
            }
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
    Moments mom;
    long long lastE = 0, lastM = 0;
    if (p.measure && lane == 0) mom.load(ctl->moments);
    for (unsigned long long k = 0; k < p.n_updates && !aborted; ++k) {
        if (lane == 0) {
            const unsigned long long u = p.u0 + k;
            const uint4 xr = philox4x32_10(0u, kDomainSite, (uint32_t)u, (uint32_t)(u >> 32), p.key0, p.key1);
            const unsigned long long rr = (unsigned long long)xr.x | ((unsigned long long)xr.y << 32);
            const uint32_t i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
            uint32_t own, addr;
            tg.locate(i0, own, addr);
            WOLFF_CHECK(&ctl->error, i0 < p.geo.N && own < G && addr < (tp.slots << (DIM * tp.tile_log)), 7);
            const unsigned int pos = atomicAdd(tp.gtail + own, 1u);
            wait_inbox(tp, own, pos);
            st_relaxed_u64(tp.inbox + ((size_t)own << tp.in_log) + (pos & in_mask),
                           pack_msg(kKindSeed, (pos >> tp.in_log) & 1u, (unsigned int)k, addr, 1));
            ++tl.messages;
        }
        const unsigned long long t0 = globaltimer_ns();
        unsigned int passes = 0;
        for (;;) {
            // sums modulo 2^32: gtail[] are 32-bit running counters, and what is in flight is far below 2^32 messages
            unsigned int d = 0, t = 0;
            for (unsigned int cc = lane; cc < G; cc += 32u) d += (unsigned int)ld_relaxed_u64(tp.gdone + cc);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) d += __shfl_xor_sync(kFullMask, d, o);
            fence_acq_rel_gpu();      // every gtail (and `added`) is read after every gdone
            WOLFF_JITTER_POINT(18);
            for (unsigned int cc = lane; cc < G; cc += 32u) t += ld_relaxed_u32(tp.gtail + cc);
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
            const unsigned long long dt = globaltimer_ns() - t0;
            p.ns_log[k] = dt > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)dt;
            flipped += a - prev;
            prev = a;
        }
        if (p.measure && !aborted) {
#ifdef WOLFF_PROFILE
            const unsigned long long tm0 = globaltimer_ns();
#endif
            // "+ measurement": every CTA evaluates its tiles (measure_phase); the request travels like the exit message
            for (unsigned int base = 0; base < G; base += 256u) {
                unsigned int pos[8];
#pragma unroll
                for (unsigned int i = 0; i < 8u; ++i) {
                    const unsigned int cc = base + i * 32u + lane;
                    pos[i] = cc < G ? atomicAdd(tp.gtail + cc, 1u) : 0u;
                }
#pragma unroll
                for (unsigned int i = 0; i < 8u; ++i) {
                    const unsigned int cc = base + i * 32u + lane;
                    if (cc < G) {
                        wait_inbox(tp, cc, pos[i]);
                        st_relaxed_u64(tp.inbox + ((size_t)cc << tp.in_log) + (pos[i] & in_mask),
                                       pack_msg(kKindExit, (pos[i] >> tp.in_log) & 1u, (unsigned int)k, 1u, 1));
                    }
                }
            }
            unsigned int bad = 0;
            if (lane == 0) {
                const unsigned int target = ((unsigned int)k + 1u) * G;
                unsigned int polls = 0;
                while (ld_acquire_u32(&ctl->meas_arrive_b) != target) {
                    if ((++polls & 0xFFu) == 0u) {
                        if (ld_relaxed_u32(&ctl->error) != 0u) { bad = 1; break; }
                        if (globaltimer_ns() - t0 > tp.watchdog_ns) { raise_abort(ctl, 6u); bad = 1; break; }
                    }
                }
                if (!bad) {
                    const unsigned long long un = atomicExch(&ctl->meas_unequal, 0ull), ng = atomicExch(&ctl->meas_negative, 0ull);
                    lastE = 2ll * (long long)un - (long long)DIM * (long long)p.geo.N;
                    lastM = (long long)p.geo.N - 2ll * (long long)ng;
                    p.E_log[k] = lastE;
                    p.M_log[k] = lastM;
                    mom.add(lastE, lastM);
                }
            }
            if (__shfl_sync(kFullMask, bad, 0)) aborted = true;
#ifdef WOLFF_PROFILE
            if (lane == 0) atomicAdd(&ctl->stats[8], globaltimer_ns() - tm0);     // the monitor's view of one measurement
#endif
        }
    }
    if (p.measure && lane == 0 && !aborted && p.n_updates > 0) { ctl->E = lastE; ctl->M = lastM; mom.store(ctl->moments); }
    // everybody leaves (also after an abort: receivers poll the error flag, but an exit message is quicker).  Eight slot
    // atomics per lane are in flight before the first message is stored.
    for (unsigned int base = 0; base < G; base += 256u) {
        unsigned int pos[8];
#pragma unroll
        for (unsigned int i = 0; i < 8u; ++i) {
            const unsigned int cc = base + i * 32u + lane;
            pos[i] = cc < G ? atomicAdd(tp.gtail + cc, 1u) : 0u;
        }
#pragma unroll
        for (unsigned int i = 0; i < 8u; ++i) {
            const unsigned int cc = base + i * 32u + lane;
            if (cc < G) {
                wait_inbox(tp, cc, pos[i]);
                st_relaxed_u64(tp.inbox + ((size_t)cc << tp.in_log) + (pos[i] & in_mask), pack_msg(kKindExit, (pos[i] >> tp.in_log) & 1u, 0u, 0u, 1));
            }
        }
    }
    if (lane == 0) {
        ctl->stats[0] += p.n_updates;
        ctl->stats[1] += flipped;
        ctl->stats[9] += polls_total;
    }
}

// ------------------------------------------------------------------------------------------ the kernel
// Copy the tiles of CTA c between the global lattice and shared memory, one 32-bit word (4 sites along x) at a time.
template <int DIM, bool LOAD, typename V>
__device__ __forceinline__ void copy_tiles_vec(const TileParams &tp, const Layout &ly)
{
    // V = uint4 (16 sites along x) when a tile row holds at least 16 sites, else unsigned int (4 sites).  The local
    // lattice is linear in (slot, within-tile index); U loads are in flight per thread before the first store.
    constexpr uint32_t VB = sizeof(V), U = 4;
    const Tiling<DIM> tg(tp);
    const uint32_t total = (ly.myslots << tg.ts_log) / VB;           // vectors this CTA owns
    V *const loc = reinterpret_cast<V *>(ly.lat);
    for (uint32_t base = threadIdx.x; base < total; base += kT * U) {
        V v[U];
        V *gp[U];
#pragma unroll
        for (uint32_t u = 0; u < U; ++u) {
            const uint32_t idx = base + u * kT;
            const uint32_t a = (idx < total ? idx : 0u) * VB;
            const uint32_t gi = ly.origin[a >> tg.ts_log] + tg.spread(a & tg.ts_mask);
            gp[u] = reinterpret_cast<V *>(tp.g.spins + gi);
            WOLFF_CHECK(&tp.g.ctl->error, idx >= total || (size_t)gi + VB <= (((size_t)tp.g.geo.N + 15u) & ~(size_t)15u), 6);
            if (idx < total) v[u] = LOAD ? __ldcg(gp[u]) : loc[idx];
        }
#pragma unroll
        for (uint32_t u = 0; u < U; ++u) {
            const uint32_t idx = base + u * kT;
            if (idx < total) { if (LOAD) loc[idx] = v[u]; else *gp[u] = v[u]; }
        }
    }
}

// Copy the tiles of CTA c between the global lattice and shared memory (after build_tables(): uses origin[]).
template <int DIM, bool LOAD>
__device__ __forceinline__ void copy_tiles(const TileParams &tp, const Layout &ly)
{
    if (tp.tile_log >= 4u) copy_tiles_vec<DIM, LOAD, uint4>(tp, ly);
    else copy_tiles_vec<DIM, LOAD, unsigned int>(tp, ly);
}

// Per-slot tables of CTA c: origin of the tile, and (owner, slot) of its 2*DIM neighbouring tiles.
template <int DIM>
__device__ __forceinline__ void build_tables(const TileParams &tp, const Layout &ly, unsigned int c)
{
    constexpr unsigned int ND = 2u * DIM;
    const Tiling<DIM> tg(tp);
    for (uint32_t i = threadIdx.x; i < tp.slots * ND; i += kT) {
        const uint32_t slot = i / ND, k = i - slot * ND, d = k >> 1;
        const uint32_t pidx = slot * tp.G + c;
        uint32_t entry = c << 16;
        if (pidx < tp.ntiles) {
            const uint32_t t = (pidx * tp.permAinv) & tg.ntiles_mask;
            const uint32_t tc = (t >> (d * tg.nt_log)) & tg.nt_mask;
            const uint32_t tn = (t & ~(tg.nt_mask << (d * tg.nt_log))) | ((((k & 1u) ? tc - 1u : tc + 1u) & tg.nt_mask) << (d * tg.nt_log));
            uint32_t own, ns;
            tg.place(tn, own, ns);
            entry = (own << 16) | ns;
            if (k == 0u) {
                uint32_t o = (t & tg.nt_mask) << tg.b;
                o |= (((t >> tg.nt_log) & tg.nt_mask) << tg.b) << tg.logL;
                if (DIM == 3) o |= ((t >> (2u * tg.nt_log)) << tg.b) << (2u * tg.logL);
                ly.origin[slot] = o;
            }
        } else if (k == 0u) {
            ly.origin[slot] = 0u;
        }
        ly.nbrtab[i] = entry;
    }
    for (uint32_t i = threadIdx.x; i < 2u * tp.slots; i += kT) ly.state[i] = 0u;
}

template <int DIM>
__global__ void __launch_bounds__(kT, 1) growth_tiles_kernel(const __grid_constant__ TileParams tp)
{
    extern __shared__ __align__(16) unsigned char smem_t[];
    __shared__ TShared sh;
    const unsigned int tid = threadIdx.x, warp = tid >> 5;
    const unsigned int c = blockIdx.x;
    const Layout ly = Layout::make<DIM>(tp, smem_t, c);
    Tally tl;
    // the error flag is sticky: an earlier launch of this handle was aborted and the host has not yet looked (the
    // queues are not in a state to continue from; the host marks the handle failed at its next synchronising call)
    if (ld_relaxed_u32(&tp.g.ctl->error) != 0u) return;

    for (unsigned int i = tid; i < tp.ring_cap; i += kT) ly.ring[i] = kEmpty;
    if (tid == 0) {
        sh.head = sh.tail = 0u;
        sh.pending = sh.claimed = 0u;
        sh.stop = 0u;
        sh.pub_lock = 0u;
        sh.s0 = 1;
        sh.u_lo = sh.u_hi = 0u;
        sh.krel = 0u;
        sh.ready_tag[0] = sh.ready_tag[1] = 0u;
        sh.watcher = 0u;
        sh.meas_req = 0u;
        sh.meas_un = sh.meas_ng = 0u;
        sh.fill_on = tp.fill_mode == 0u ? 0u : (tp.fill_mode == 2u ? 1u : tp.gfill[c]);
        sh.ihead = ld_relaxed_u64(tp.gdone + c);          // everything ever sent to this CTA was consumed by the last launch
        sh.spill_head = sh.spill_tail = ld_relaxed_u64(tp.gspill + c);
    }
#ifdef WOLFF_PROFILE
    const unsigned long long tk0 = globaltimer_ns();
#endif
    build_tables<DIM>(tp, ly, c);
    __syncthreads();
    copy_tiles<DIM, true>(tp, ly);
    __syncthreads();
#ifdef WOLFF_PROFILE
    const unsigned long long tk1 = globaltimer_ns();
#endif

    if (warp == 0u) receiver_warp<DIM>(tp, sh, ly, ly.stage, c, tl);
    else if (warp == 1u && c == 0u) monitor_warp<DIM>(tp, tl);
    else worker_warp<DIM>(tp, sh, ly, ly.stage + warp * kStage, c, tl);
    __syncthreads();

#ifdef WOLFF_PROFILE
    const unsigned long long tk2 = globaltimer_ns();
#endif
    copy_tiles<DIM, false>(tp, ly);
#ifdef WOLFF_PROFILE
    __syncthreads();
    if (tid == 0 && c == 0 && !tp.g.measure) {     // (a measured profiling run uses these slots for the measurement's phases)
        tp.g.ctl->stats[4] = tk1 - tk0; tp.g.ctl->stats[5] = tk2 - tk1; tp.g.ctl->stats[6] = globaltimer_ns() - tk2;
    }
#endif
    if (tid == 0) {
        tp.gspill[c] = ld_vol64(&sh.spill_tail);
        tp.gfill[c] = ld_vol(&sh.fill_on);
    }
    // tallies
    Control *ctl = tp.g.ctl;
    const unsigned int a = __reduce_add_sync(kFullMask, tl.attempts);
    const unsigned int ms = __reduce_add_sync(kFullMask, tl.messages);
    if ((tid & 31u) == 0u) {
        if (a) atomicAdd(&ctl->stats[7], (unsigned long long)a);
        if (tl.inline_passes) atomicAdd(&ctl->stats[10], (unsigned long long)tl.inline_passes);
        if (ms) atomicAdd(&ctl->stats[11], (unsigned long long)ms);
        if (tl.passes) atomicAdd(&ctl->stats[13], (unsigned long long)tl.passes);
        if (tl.chunks) atomicAdd(&ctl->stats[15], (unsigned long long)tl.chunks);
        if (tl.ring_pushes) atomicAdd(&ctl->stats[12], (unsigned long long)tl.ring_pushes);
        if (tl.spills) atomicAdd(&ctl->stats[14], (unsigned long long)tl.spills);
#ifdef WOLFF_PROFILE
        if (tl.cyc_pass && !tp.g.measure) atomicAdd(&ctl->stats[2], tl.cyc_pass);
        if (tl.lanes && !tp.g.measure) atomicAdd(&ctl->stats[3], tl.lanes);
#endif
    }
}

template <int DIM>
cudaError_t launch_one(const TileParams &tp, size_t smem_bytes, cudaStream_t stream)
{
    // the attribute belongs to the kernel function, i.e. to the process: only ever raised to the device's maximum (internal.h)
    const void *fn = reinterpret_cast<const void *>(&growth_tiles_kernel<DIM>);
    const cudaError_t ea = allow_max_dynamic_smem(fn);
    if (ea != cudaSuccess) return ea;
    void *args[] = { const_cast<TileParams *>(&tp) };
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(&growth_tiles_kernel<DIM>), dim3(tp.G), dim3(kT), args,
                                       smem_bytes, stream);
}

template <int DIM>
cudaError_t prepare_one(size_t smem_bytes, int *ctas_per_sm)
{
    const void *fn = reinterpret_cast<const void *>(&growth_tiles_kernel<DIM>);
    cudaError_t e = allow_max_dynamic_smem(fn);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, growth_tiles_kernel<DIM>, kT, smem_bytes);
}

}  // namespace

size_t tiles_smem_bytes(int dim, uint32_t tile_log, uint32_t slots, uint32_t ring_cap, uint32_t nbuf)
{
    const uint32_t ts_log = (uint32_t)dim * tile_log;
    size_t bytes = (((size_t)slots << ts_log) + 15u) & ~(size_t)15u;                       // lattice
    size_t words = 0;
    if (nbuf) {
        const uint32_t face_log = (uint32_t)(dim - 1) * tile_log;
        words += (size_t)nbuf * dim * slots * ((size_t)1 << (ts_log - 5u));                  // bond planes
        words += (size_t)nbuf * dim * slots * (face_log > 5u ? (size_t)1 << (face_log - 5u) : 1u);   // halo planes
    }
    words += 2u * (size_t)slots + 2u * (size_t)dim * slots + slots;                         // state, nbrtab, origin
    words += (size_t)ring_cap + (size_t)kWarps * kStage;                                    // ring, stage
    return bytes + words * sizeof(uint32_t);
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
