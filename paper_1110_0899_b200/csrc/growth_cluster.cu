// growth_cluster.cu -- the cluster-resident, bit-packed, barrier-free growth kernel
// (8(f) row 4 as written: "1 bit/spin ... 2D L=4096 and 3D L=256 = 2 MiB fit a 16-CTA
// cluster's distributed shared memory").
//
// Same computation as growth.cu and growth_tiles.cu: n_updates Wolff single-cluster updates (steps
// i-v), every newly added spin expanded in parallel (step iii').  growth_tiles.cu keeps the int8
// lattice in the shared memory of all 148 SMs, and a claim that crosses into another CTA's tiles travels through L2
// (an atomic for the inbox slot, a store, the receiver's poll: 1.5-3 us per hop, which is what bounds it in 3D where
// 16^3 tiles make 0.16 such hops per spin).  Here the lattice is ONE BIT PER SPIN (the sign), so every BASELINE
// lattice (<= 2^24 spins = 2 MiB) fits the distributed shared memory of ONE thread-block cluster of 16 CTAs (any L: the
// coordinates of a site come from shifts when L is a power of two, from two multiplications otherwise), and
//
//   - claim-and-flip (A4) is ONE atomic on the 32-bit word holding the neighbour's bit, wherever that word lives:
//     atom.shared::cluster.or / .and on the own CTA's window (about 40 ns as a dependent operation) or on a peer's
//     (about 140 ns; an L2 atomic is 270 ns: profiles/r2_dsmem_latency.md).  The atomic is idempotent on a spin that
//     is not parallel to the seed spin, so it is issued for every active bond without looking at the neighbour first
//     (no gather on the critical path: A2 is the atomic's own read), and its returned bit says whether this lane
//     claimed the site.  There are no tiles, no inboxes, no messages and no receiver: ANY warp may expand ANY site;
//   - one lane per bond, as in growth_tiles.cu: a warp holds up to S = 32 / (2 dim) sites per pass, lane (q, k) tests
//     the bond from site q to its neighbour k: one Philox4x32-10 block (A3, inline: bond tables for 2 MiB of spins do
//     not fit beside them), one atomic, then ballot/popc compaction of the winners (A5);
//   - the first S winners of a pass stay in the warp; the rest goes to the CTA's shared-memory ring, drained by the
//     other warps of the CTA -- and, when those are busy, by the idle warps of the OTHER CTAs of the cluster: one idle
//     warp per CTA (the watch) reads the (head, tail) words of all peers in one round of remote loads and takes sites
//     out of a peer's ring with remote atomics (A6 is work stealing; there are no levels and no barrier).  Overflow
//     of a ring goes to one global-memory spill list shared by the cluster;
//   - termination (A7): ONE 64-bit word in CTA 0's shared memory holds [claimed : 32 | pending : 32].  pending counts
//     units of outstanding work: a warp that takes n sites holds n units until it runs dry; sites handed to a ring
//     are added BEFORE they become visible (an atomic with return, so the addition has been performed).  When a warp
//     runs dry one remote reduction subtracts its units and adds the spins it claimed, so the monitor warp (CTA 0)
//     that reads pending == 0 reads the complete cluster size in the same word;
//   - the monitor warp draws the seed site (A1), flips its bit and EXPANDS IT ITSELF, as a worker would; its own unit and
//     claims never touch the shared word, and only when a site is about to leave its hands does it publish the update's
//     index and seed spin to every CTA.  A cluster of a handful of spins (the literal random start of the BASELINE configs,
//     T above T_c) is complete after its few passes, without a hand-over, a poll or a remote word besides the spins'.
//
// The int8 lattice in global memory stays the authoritative copy between launches: every CTA packs its slab of the
// lattice in the prologue and unpacks it in the epilogue (N bytes each way per launch, by 16 SMs).
//
// "measure" = 1 (L a multiple of 32): E and M after EVERY update inside the kernel, by population counts over the bit
// lattice (measure_slab), logged and accumulated as in the other kernels.
#include <cooperative_groups.h>

#include "expand.cuh"
#include "internal.h"

namespace cg = cooperative_groups;

namespace wolff {
namespace {

constexpr int kCT = kClusterThreads;
constexpr int kCWarps = kCT / 32;
constexpr uint32_t kEmpty = 0xFFFFFFFFu;
constexpr int kCStage = 64;                        // two buffers of 32 winners per warp

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared::cluster address of the same variable in the CTA of rank r (the own rank gives the own window)
__device__ __forceinline__ uint32_t mapa(uint32_t a, uint32_t r)
{
    uint32_t o;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(o) : "r"(a), "r"(r));
    return o;
}
// Every word that a peer CTA may touch is accessed with shared::cluster operations by everybody, the own CTA included.
__device__ __forceinline__ uint32_t cl_ld_u32(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.volatile.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long cl_ld_u64(uint32_t a)
{
    unsigned long long v;
    asm volatile("ld.volatile.shared::cluster.u64 %0, [%1];" : "=l"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void cl_st_u32(uint32_t a, uint32_t v) { asm volatile("st.volatile.shared::cluster.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ uint32_t cl_atom_xor(uint32_t a, uint32_t v)
{
    uint32_t o;
    asm volatile("atom.shared::cluster.xor.b32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory");
    return o;
}
__device__ __forceinline__ uint32_t cl_atom_exch(uint32_t a, uint32_t v)
{
    uint32_t o;
    asm volatile("atom.shared::cluster.exch.b32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory");
    return o;
}
__device__ __forceinline__ uint32_t cl_atom_cas(uint32_t a, uint32_t cmp, uint32_t v)
{
    uint32_t o;
    asm volatile("atom.shared::cluster.cas.b32 %0, [%1], %2, %3;" : "=r"(o) : "r"(a), "r"(cmp), "r"(v) : "memory");
    return o;
}
__device__ __forceinline__ unsigned long long cl_atom_add64(uint32_t a, unsigned long long v)
{
    unsigned long long o;
    asm volatile("atom.shared::cluster.add.u64 %0, [%1], %2;" : "=l"(o) : "r"(a), "l"(v) : "memory");
    return o;
}
__device__ __forceinline__ void cl_red_add64(uint32_t a, unsigned long long v) { asm volatile("red.shared::cluster.add.u64 [%0], %1;" ::"r"(a), "l"(v) : "memory"); }
__device__ __forceinline__ unsigned int lds_u32(uint32_t saddr)
{
    unsigned int v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32(uint32_t saddr, unsigned int v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }
__device__ __forceinline__ void st_relaxed_u32_g(unsigned int *p, unsigned int v) { asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }
__device__ __forceinline__ void raise_abort(Control *ctl, unsigned int code) { st_relaxed_u32(&ctl->error, code); }

// Per-CTA shared state (the same layout in every CTA of the cluster: peers address it through mapa).
struct alignas(16) CShared {
    unsigned int head, tail;            // ring: entries [head, tail) wait for a warp (one aligned 64-bit word)
    unsigned long long pc;              // CTA 0 only: [spins claimed since the launch began : 32 | pending units : 32]
    unsigned int upd;                   // (krel << 1) | (seed spin is -1) of the running update, written by the monitor
    unsigned int stop;                  // the launch is over (or aborted)
    unsigned int watcher;               // 1 while some idle warp of this CTA holds the watch
    unsigned int meas_req;              // k + 1 once the monitor has asked for the measurement after update k ("measure" = 1)
    // in-kernel measurement: this CTA's sums of one evaluation and the warps that have added theirs
    unsigned int meas_un, meas_ng, meas_warps, pad;
    // CTA 0 only: the cluster's sums of one evaluation, [CTAs arrived : 13 | negative spins : 25 | unequal bonds : 26]
    unsigned long long meas_acc;
};

struct CTally {
    unsigned int attempts = 0;          // claim atomics (per lane)
    unsigned int steals = 0;            // sites taken out of a peer's ring (lane 0)
    unsigned int ring_pushes = 0;       // sites handed over through the own ring (lane 0)
    unsigned int spills = 0;            // ... through the global spill list (lane 0)
    unsigned int passes = 0;            // warp passes (lane 0)
#ifdef WOLFF_PROFILE
    unsigned long long cyc_pass = 0, cyc_hand = 0, cyc_take = 0, sites = 0;   // lane 0
    unsigned int hands = 0, takes = 0;
#endif
};

__device__ __forceinline__ uint32_t spill_tag(unsigned long long pos, uint32_t cap_log) { return (uint32_t)((pos >> cap_log) + 1ull) & 1u; }

// Four spin bytes (0x01 / 0xFF) -> four sign bits (byte k -> bit k), and back.
__device__ __forceinline__ uint32_t pack4(uint32_t bytes) { return ((bytes & 0x80808080u) * 0x00204081u) >> 28; }
__device__ __forceinline__ uint32_t unpack4(uint32_t nibble) { return 0x01010101u | (((nibble * 0x00204081u) & 0x01010101u) * 0xFEu); }
__device__ __forceinline__ uint32_t pack16(const uint4 &v) { return pack4(v.x) | (pack4(v.y) << 4) | (pack4(v.z) << 8) | (pack4(v.w) << 12); }
__device__ __forceinline__ uint4 unpack16(uint32_t b) { return make_uint4(unpack4(b & 15u), unpack4((b >> 4) & 15u), unpack4((b >> 8) & 15u), unpack4((b >> 12) & 15u)); }

// Hand n sites (items[0..n), warp-collective) to the other warps: the own ring, or the cluster's spill list when the
// ring is full.  The caller has already added them to the pending count.
__device__ __forceinline__ void hand_over(const ClusterParams &cp, uint32_t head_c, uint32_t ring_c, const uint32_t *items, unsigned int n, CTally &tl)
{
    const unsigned int lane = threadIdx.x & 31u;
    const uint32_t rmask = cp.ring_cap - 1u;
    unsigned int base = 0, ok = 0;
    if (lane == 0) {
        // reserve n consecutive entries, unless the ring cannot take them
        unsigned int t = cl_ld_u32(head_c + 4u);
        for (;;) {
            const unsigned int h = cl_ld_u32(head_c);
            if (t + n - h > cp.ring_cap) break;
            const unsigned int seen = cl_atom_cas(head_c + 4u, t, t + n);
            if (seen == t) { base = t; ok = 1u; break; }
            t = seen;
        }
    }
    ok = __shfl_sync(kFullMask, ok, 0);
    base = __shfl_sync(kFullMask, base, 0);
    WOLFF_JITTER_POINT(1);           // reserved, not yet filled
    if (ok) {
        // the entry of the lap before has been acquired (head moved past it) but may not have been taken yet
        for (unsigned int j = lane; j < n; j += 32u) {
            const uint32_t slot = ring_c + (((base + j) & rmask) << 2);
            while (cl_atom_cas(slot, kEmpty, items[j]) != kEmpty) { }
        }
        if (lane == 0) tl.ring_pushes += n;
    } else {
        unsigned long long sbase = 0;
        if (lane == 0) sbase = atomicAdd(cp.spill_ctr, (unsigned long long)n);
        sbase = __shfl_sync(kFullMask, sbase, 0);
        const uint32_t smask = (1u << cp.spill_log) - 1u;
        WOLFF_JITTER_POINT(2);
        for (unsigned int j = lane; j < n; j += 32u) {
            const unsigned long long pos = sbase + (unsigned long long)j;
            st_relaxed_u32_g(cp.spill + ((uint32_t)pos & smask), (items[j] << 1) | spill_tag(pos, cp.spill_log));
        }
        if (lane == 0) tl.spills += n;
    }
}

// ------------------------------------------------------------------------------------------ in-kernel measurement
// "+ measurement": E and M of the whole lattice after an update, evaluated where the lattice is
// -- one bit per spin in the cluster's shared memory -- without leaving the kernel: 32 spins per word, so
//   #negative = popc(word),  #unequal bonds in direction d = popc(word ^ word of the +d neighbours)
// (+x: the word shifted by one bit, its last bit from the next word of the row; +y, +z: the word L/32 or L^2/32 words
// further on, wrapping; a word of another CTA's slab is read through its shared::cluster address).  Needs L to be a
// multiple of 32 (the host checks).  Called by every warp of the cluster but the monitor, between two updates; the CTA's
// last warp sends the CTA's sums and its arrival to CTA 0 in ONE remote reduction.
template <int DIM, bool POW2>
__device__ __noinline__ void measure_slab(const ClusterParams &cp, CShared &sh, uint32_t bits_s, unsigned int rank, unsigned int ptid, unsigned int P)
{
    const Geometry &g = cp.g.geo;
    const uint32_t W = g.L >> 5, wmask = cp.wpc - 1u;
    const uint32_t plane = g.L * W;                                   // words of one z-plane (of the lattice in 2D)
    auto ldw = [&](uint32_t gw) { return cl_ld_u32(mapa(bits_s + ((gw & wmask) << 2), gw >> cp.wpc_log)); };
    unsigned int un = 0, ng = 0;
    for (uint32_t w = ptid; w < cp.wpc; w += P) {
        const uint32_t gw = rank * cp.wpc + w;
        if (gw >= cp.words) break;
        const uint32_t word = lds_u32(bits_s + (w << 2));
        uint32_t row, xw, y, z;                                       // row = y + L z
        if (POW2) {
            row = gw >> (g.logL - 5u); xw = gw & (W - 1u);
            z = DIM == 3 ? row >> g.logL : 0u; y = row & (g.L - 1u);
        } else {
            row = gw / W; xw = gw - row * W;
            z = DIM == 3 ? row / g.L : 0u; y = row - z * g.L;
        }
        const uint32_t wx = ldw(xw + 1u == W ? gw + 1u - W : gw + 1u);
        const uint32_t wy = ldw(y + 1u == g.L ? gw + W - plane : gw + W);
        ng += __popc(word);
        un += __popc(word ^ ((word >> 1) | (wx << 31))) + __popc(word ^ wy);
        if (DIM == 3) un += __popc(word ^ ldw(z + 1u == g.L ? gw + plane - cp.words : gw + plane));
    }
    un = __reduce_add_sync(kFullMask, un);
    ng = __reduce_add_sync(kFullMask, ng);
    if ((threadIdx.x & 31u) == 0u) {
        if (un) atomicAdd(&sh.meas_un, un);
        if (ng) atomicAdd(&sh.meas_ng, ng);
        __threadfence_block();
        if (atomicAdd(&sh.meas_warps, 1u) == P / 32u - 1u) {
            // the last warp of this CTA: every other warp's sums are in (its fence preceded its count)
            __threadfence_block();
            const unsigned long long tun = *reinterpret_cast<volatile unsigned int *>(&sh.meas_un);
            const unsigned long long tng = *reinterpret_cast<volatile unsigned int *>(&sh.meas_ng);
            *reinterpret_cast<volatile unsigned int *>(&sh.meas_un) = 0u;
            *reinterpret_cast<volatile unsigned int *>(&sh.meas_ng) = 0u;
            *reinterpret_cast<volatile unsigned int *>(&sh.meas_warps) = 0u;
            __threadfence_block();
            cl_red_add64(mapa(smem_addr(&sh.meas_acc), 0u), tun | (tng << 26) | (1ull << 51));
        }
    }
}

struct CWorker {
    uint32_t a = 0;              // this lane's site (global id)
    unsigned int nsites = 0;     // sites held by the warp (warp-uniform); lanes of group q < nsites work
    unsigned int units = 0;      // what the warp owes the pending count when it runs dry
    unsigned int mywon = 0;      // spins this lane claimed since the warp last ran dry
    unsigned int sbuf = 0;       // which half of stage[] the next pass writes
    // the monitor warp only (it expands the seed site itself): what it publishes to every CTA before the first site of
    // the update leaves its hands, and whether that has happened
    uint32_t upd_s = 0, upd_v = 0;
    bool handed = false;
};

// Passes until the warp holds no site.  POS: the seed spin of the running update is +1 (its bit is 0; claim = OR).
// MONITOR: the caller is the monitor warp, which starts every update by expanding the seed site itself -- a cluster of
// a few spins (the literal random start of the BASELINE configs, T well above T_c) is then complete without a single
// hand-over, a poll or a remote word besides the spins'.  Its own unit of work and the spins it claims are not part of
// the cluster's pending / claimed word; before the first site of the update leaves its hands it writes the update's
// index and seed spin into every CTA and reads them back (the load returns only after the store has been performed
// there), so every warp that later takes a site of this update finds them.
// POW2: L is a power of two (coordinates by shifts and masks); else by two multiplications with ceil(2^40 / divisor), exact
// for sites below 2^24 and divisors up to 2^16 (the host checks both).
template <int DIM, bool POS, bool MONITOR, bool POW2>
__device__ __forceinline__ void run_passes(const ClusterParams &cp, uint32_t bits_s, uint32_t pc_c, uint32_t head_c, uint32_t ring_c, uint32_t *stage,
                                           uint32_t u_lo, uint32_t u_hi, CWorker &ws, CTally &tl)
{
    constexpr unsigned int ND = 2u * DIM, S = 32u / ND;
    const GrowthParams &p = cp.g;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int lt = (1u << lane) - 1u;
    const unsigned int q = lane / ND, k = lane - q * ND, d = k >> 1, sgn = k & 1u;
    const uint32_t Lmask = p.geo.L - 1u;
    const uint32_t sh_d = d * p.geo.logL, fmask = Lmask << sh_d, delta = sgn ? 0xFFFFFFFFu : 1u;
    // any L: this lane's stride L^d, its magic, and the steps to the neighbour inside the lattice / across the wrap
    const uint32_t stride = d == 0u ? 1u : (d == 1u ? p.geo.L : p.geo.LL);
    const unsigned long long magic_s = d == 0u ? (1ull << 40) : (d == 1u ? cp.magicL : cp.magicLL);
    const uint32_t edge_c = sgn ? 0u : Lmask;                                        // coordinate at which the neighbour wraps
    const uint32_t step_in = sgn ? 0u - stride : stride, step_wrap = sgn ? Lmask * stride : 0u - Lmask * stride;
    const uint32_t wmask = cp.wpc - 1u;
    const uint32_t stage_s = smem_addr(stage);
    uint32_t a = ws.a;
    unsigned int nsites = ws.nsites, mywon = ws.mywon, sbuf = ws.sbuf;

    for (;;) {
#ifdef WOLFF_PROFILE
        const long long tp0 = clock64();
        tl.sites += nsites;
#endif
        const bool have = q < S && q < nsites;               // lanes 30, 31 in 3D (q = S) never hold a site
        // ---- this lane's neighbour (periodic) and the owner of the bond between them (reading R6)
        uint32_t n;
        if (POW2) {
            n = (a & ~fmask) | ((((a >> sh_d) + delta) & Lmask) << sh_d);
        } else {
            const uint32_t q1 = (uint32_t)(((unsigned long long)a * magic_s) >> 40);                         // a div L^d
            const uint32_t c = q1 - (uint32_t)(((unsigned long long)q1 * cp.magicL) >> 40) * p.geo.L;         // ... mod L
            n = a + (c == edge_c ? step_wrap : step_in);
        }
        // ---- A3: the bond variable, one Philox block per lane (word d of the block of the bond's owner)
        const uint4 blk = philox4x32_10(sgn ? n : a, kDomainBond, u_lo, u_hi, p.key0, p.key1);
        const uint32_t r = d == 0u ? blk.x : (d == 1u ? blk.y : blk.z);
        const bool bit = have && (r < cp.thr32 || cp.thr_all != 0u);
        // ---- A2 + A4: one atomic on the word holding the neighbour's sign bit, in whichever CTA holds it
        const uint32_t wi = n >> 5, m = 1u << (n & 31u);
        const uint32_t addr = mapa(bits_s + ((wi & wmask) << 2), wi >> cp.wpc_log);
        uint32_t old = POS ? 0xFFFFFFFFu : 0u;               // reads as "not claimed by me"
        if (POS) asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %3, 0;\n @p atom.shared::cluster.or.b32 %0, [%1], %2;\n}"
                              : "+r"(old) : "r"(addr), "r"(m), "r"((unsigned int)bit) : "memory");
        else     asm volatile("{\n .reg .pred p;\n setp.ne.u32 p, %3, 0;\n @p atom.shared::cluster.and.b32 %0, [%1], %2;\n}"
                              : "+r"(old) : "r"(addr), "r"(~m), "r"((unsigned int)bit) : "memory");
        tl.attempts += bit ? 1u : 0u;
        const bool won = POS ? (old & m) == 0u : (old & m) != 0u;
        mywon += won ? 1u : 0u;
        if (lane == 0) ++tl.passes;
        // ---- A5: compact the winners; the first S are this warp's next pass, the rest goes to the ring
        const unsigned int wb = __ballot_sync(kFullMask, won);
        const unsigned int total = __popc(wb);
#ifdef WOLFF_PROFILE
        if (total == 0u) tl.cyc_pass += (unsigned long long)(clock64() - tp0);
#endif
        if (total == 0u) break;                                  // the warp runs dry
        uint32_t *const st_out = stage + sbuf;
        const uint32_t out_s = stage_s + sbuf * 4u;
        sbuf ^= 32u;
        if (won && WOLFF_CHECK(&p.ctl->error, n < p.geo.N && (wi >> cp.wpc_log) < cp.nC && __popc(wb & lt) < 32, 32)) sts_u32(out_s + __popc(wb & lt) * 4u, n);
        __syncwarp();
        nsites = total < S ? total : S;
        if (q < S && q < nsites) a = lds_u32(out_s + q * 4u);
#ifdef WOLFF_PROFILE
        const long long th0 = clock64();
#endif
        if (total > S) {
            if (MONITOR && !ws.handed) {
                if (lane < cp.nC) {
                    const uint32_t ua = mapa(ws.upd_s, lane);
                    cl_st_u32(ua, ws.upd_v);
                    unsigned int polls = 0;
                    while (cl_ld_u32(ua) != ws.upd_v) if (++polls > (1u << 20)) { raise_abort(p.ctl, 7u); break; }
                }
                ws.handed = true;
                __syncwarp();
            }
            // counted (the atomic has returned: the addition has been performed) before another warp can see them
            if (lane == 0) (void)cl_atom_add64(pc_c, (unsigned long long)(total - S));
            WOLFF_JITTER_POINT(3);
            __syncwarp();
            hand_over(cp, head_c, ring_c, st_out + S, total - S, tl);
#ifdef WOLFF_PROFILE
            tl.cyc_hand += (unsigned long long)(clock64() - th0);
            ++tl.hands;
#endif
        }
#ifdef WOLFF_PROFILE
        tl.cyc_pass += (unsigned long long)(th0 - tp0);
#endif
    }
    // ---- dry: one reduction hands back the warp's units and adds the spins it claimed
    const unsigned int wsum = __reduce_add_sync(kFullMask, mywon);
    WOLFF_JITTER_POINT(4);           // claims made, units not yet handed back
    if (!MONITOR && lane == 0) cl_red_add64(pc_c, ((unsigned long long)wsum << 32) - (unsigned long long)ws.units);
    ws.nsites = 0u; ws.mywon = MONITOR ? wsum : 0u; ws.sbuf = sbuf; ws.a = a;
}

template <int DIM, bool POW2>
__device__ __forceinline__ void worker_warp(const ClusterParams &cp, CShared &sh, uint32_t bits_s, uint32_t ring_s, uint32_t *stage, unsigned int rank,
                                            CTally &tl)
{
    constexpr unsigned int ND = 2u * DIM, S = 32u / ND;
    const GrowthParams &p = cp.g;
    const unsigned int lane = threadIdx.x & 31u;
    const unsigned int q = lane / ND;
    const uint32_t rmask = cp.ring_cap - 1u;
    const uint32_t head_s = smem_addr(&sh.head);
    const uint32_t head_c = mapa(head_s, rank), ring_c = mapa(ring_s, rank), pc_c = mapa(smem_addr(&sh.pc), 0u);
    const uint32_t smask = (1u << cp.spill_log) - 1u;
    bool watcher = false;
    unsigned int idle = 0, meas_done = 0;
    // in-kernel measurement: every warp of the cluster but the monitor takes part
    const unsigned int P = rank == 0u ? kCT - 32u : kCT, ptid = rank == 0u ? threadIdx.x - 32u : threadIdx.x;
    CWorker ws;

    for (;;) {
        // ---- take up to S sites: the own ring; as the CTA's watch also a peer's ring or the spill list
        unsigned int n = 0, h = 0, stop = 0, mreq = 0, src = rank;      // src: rank whose ring the sites come from, 32 = the spill list
        unsigned long long sp_pos = 0;
        if (lane == 0) {
            const unsigned long long ht = cl_ld_u64(head_c);
            stop = *reinterpret_cast<volatile unsigned int *>(&sh.stop);
            mreq = *reinterpret_cast<volatile unsigned int *>(&sh.meas_req);
            h = (unsigned int)ht;
            const unsigned int t = (unsigned int)(ht >> 32);
            if (t != h) {
                n = t - h < S ? t - h : S;
                if (cl_atom_cas(head_c, h, h + n) != h) { n = 0; stop = 0; }
            }
        }
        n = __shfl_sync(kFullMask, n, 0);
        if (n == 0u) {
            mreq = __shfl_sync(kFullMask, mreq, 0);
            if (mreq != meas_done) {                               // the update is over everywhere: measure (measure_slab)
                measure_slab<DIM, POW2>(cp, sh, bits_s, rank, ptid, P);
                meas_done = mreq;
                continue;
            }
            if (__shfl_sync(kFullMask, stop, 0)) break;            // launch over
            if (!watcher) {
                unsigned int got = 0;
                if (lane == 0) got = atomicCAS(&sh.watcher, 0u, 1u) == 0u ? 1u : 0u;
                watcher = __shfl_sync(kFullMask, got, 0) != 0u;
            }
            if (!watcher) {
                // idle warps share the SM's issue slots and load/store pipe with the working ones: back off
                ++idle;
                if (idle > 2u) __nanosleep(idle < 8u ? 64u : (idle < 16u ? 256u : cp.idle_ns));
                continue;
            }
            // ---- the watch: one round of remote loads shows every peer's ring (lanes 0..nC-1) and the spill list (lane 31)
            unsigned int backlog = 0, vh = 0;
            if (lane < cp.nC && lane != rank) {
                const unsigned long long ht = cl_ld_u64(mapa(head_s, lane));
                vh = (unsigned int)ht;
                backlog = (unsigned int)(ht >> 32) - vh;
            } else if (lane == 31u) {
                // the head first: the tail read afterwards is at least the head seen (both only grow)
                const unsigned long long shd = ld_relaxed_u64(cp.spill_ctr + 1);
                const unsigned long long st = ld_relaxed_u64(cp.spill_ctr);
                sp_pos = shd;
                backlog = st - shd > 0xFFFFFFFFull ? 0xFFFFFFFFu : (unsigned int)(st - shd);
            }
            WOLFF_JITTER_POINT(6);   // the peers' rings as they were a while ago
            const unsigned int cand = __ballot_sync(kFullMask, backlog != 0u);
            if (cand == 0u) continue;
            // the first candidate after the own rank, cyclically: thieves spread over the victims
            const unsigned int rot = (rank + 1u) & 31u;
            const unsigned int rc = rot ? ((cand >> rot) | (cand << (32u - rot))) : cand;
            const unsigned int pick = ((unsigned int)__ffs((int)rc) - 1u + rot) & 31u;
            const unsigned int vb = __shfl_sync(kFullMask, backlog, pick);
            vh = __shfl_sync(kFullMask, vh, pick);
            sp_pos = __shfl_sync(kFullMask, sp_pos, 31);
            unsigned int got = 0;
            if (lane == 0) {
                got = vb < S ? vb : S;
                if (pick == 31u) {
                    if (atomicCAS(cp.spill_ctr + 1, sp_pos, sp_pos + got) != sp_pos) got = 0;
                } else if (cl_atom_cas(mapa(head_s, pick), vh, vh + got) != vh) got = 0;
            }
            n = __shfl_sync(kFullMask, got, 0);
            if (n == 0u) continue;
            src = pick == 31u ? 32u : pick;
            h = vh;
            if (lane == 0 && src != 32u) tl.steals += n;
        } else {
            h = __shfl_sync(kFullMask, h, 0);
        }
        idle = 0;
        WOLFF_JITTER_POINT(5);       // entries acquired (head moved), not yet taken out of their slots
#ifdef WOLFF_PROFILE
        const long long tt0 = clock64();
#endif
        if (watcher) { watcher = false; if (lane == 0) *reinterpret_cast<volatile unsigned int *>(&sh.watcher) = 0u; }
        uint32_t ent = 0;
        if (lane < n) {
            unsigned int spins = 0;
            if (src != 32u) {
                const uint32_t slot = mapa(ring_s, src) + (((h + lane) & rmask) << 2);
                do {
                    ent = cl_atom_exch(slot, kEmpty);          // the producer reserved it; its store is on the way
                    if (ent == kEmpty && ++spins > (1u << 24)) { raise_abort(p.ctl, 4u); ent = 0u; }
                } while (ent == kEmpty);
            } else {
                const unsigned long long pos = sp_pos + (unsigned long long)lane;
                const uint32_t *slot = cp.spill + ((uint32_t)pos & smask);
                const uint32_t tag = spill_tag(pos, cp.spill_log);
                uint32_t v;
                do {
                    v = ld_relaxed_u32(slot);
                    if ((v & 1u) != tag && ++spins > (1u << 24)) { raise_abort(p.ctl, 5u); v = tag; }
                } while ((v & 1u) != tag);
                ent = v >> 1;
            }
            if (!WOLFF_CHECK(&p.ctl->error, ent < p.geo.N, 30)) ent = 0u;
        }
        ws.a = __shfl_sync(kFullMask, ent, q & 31u);
        ws.nsites = n;
        ws.units = n;
        WOLFF_JITTER_POINT(8);
        // the update these sites belong to: written into every CTA (and read back) by the monitor before the first site
        // of the update left its hands
        const unsigned int upd = *reinterpret_cast<volatile unsigned int *>(&sh.upd);
        const unsigned long long u = p.u0 + (unsigned long long)(upd >> 1);
#ifdef WOLFF_PROFILE
        tl.cyc_take += (unsigned long long)(clock64() - tt0);
        ++tl.takes;
#endif
        if (upd & 1u) run_passes<DIM, false, false, POW2>(cp, bits_s, pc_c, head_c, ring_c, stage, (uint32_t)u, (uint32_t)(u >> 32), ws, tl);
        else          run_passes<DIM, true, false, POW2>(cp, bits_s, pc_c, head_c, ring_c, stage, (uint32_t)u, (uint32_t)(u >> 32), ws, tl);
    }
}

// CTA 0 only: the update loop ("(v) Go to (i)").  Draws the seed site of update u (A1, reading R8), flips
// it, expands it (run_passes<MONITOR>); when sites have left its hands it waits for the pending count to return to zero;
// logs the size (A7).
template <int DIM, bool POW2>
__device__ __forceinline__ void monitor_warp(const ClusterParams &cp, CShared &sh, uint32_t bits_s, uint32_t ring_s, uint32_t *stage, CTally &tl)
{
    constexpr unsigned int ND = 2u * DIM;
    const GrowthParams &p = cp.g;
    const unsigned int lane = threadIdx.x & 31u;
    Control *ctl = p.ctl;
    const uint32_t head_s = smem_addr(&sh.head), stop_s = smem_addr(&sh.stop);
    const uint32_t pc_c = mapa(smem_addr(&sh.pc), 0u), head_c = mapa(head_s, 0u), ring_c = mapa(ring_s, 0u);
    const uint32_t wmask = cp.wpc - 1u;
    unsigned int prev_claimed = 0;
    unsigned long long flipped = 0, polls_total = 0;
    bool aborted = false;
    Moments mom;
    long long lastE = 0, lastM = 0;
    if (p.measure && lane == 0) mom.load(ctl->moments);
    const uint32_t mreq_s = smem_addr(&sh.meas_req), macc_c = mapa(smem_addr(&sh.meas_acc), 0u);
    CWorker ws;
    ws.upd_s = smem_addr(&sh.upd);
    for (unsigned long long k = 0; k < p.n_updates && !aborted; ++k) {
        const unsigned long long t0 = globaltimer_ns();
        const unsigned long long u = p.u0 + k;
        unsigned int s0neg = 0;
        uint32_t i0 = 0;
        if (lane == 0) {
            const uint4 xr = philox4x32_10(0u, kDomainSite, (uint32_t)u, (uint32_t)(u >> 32), p.key0, p.key1);
            const unsigned long long rr = (unsigned long long)xr.x | ((unsigned long long)xr.y << 32);
            i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
            const uint32_t wi = i0 >> 5, m = 1u << (i0 & 31u);
            (void)WOLFF_CHECK(&ctl->error, i0 < p.geo.N && (wi >> cp.wpc_log) < cp.nC, 31);
            // A1: nothing else runs between two updates, so the seed's flip is a plain exchange of its bit
            s0neg = (cl_atom_xor(mapa(bits_s + ((wi & wmask) << 2), wi >> cp.wpc_log), m) & m) ? 1u : 0u;
        }
        s0neg = __shfl_sync(kFullMask, s0neg, 0);
        i0 = __shfl_sync(kFullMask, i0, 0);
        WOLFF_JITTER_POINT(7);
        ws.a = lane < ND ? i0 : 0u;          // the lanes of site 0
        ws.nsites = 1u;
        ws.units = 0u;
        ws.mywon = 0u;
        ws.upd_v = ((unsigned int)k << 1) | s0neg;
        ws.handed = false;
        if (s0neg) run_passes<DIM, false, true, POW2>(cp, bits_s, pc_c, head_c, ring_c, stage, (uint32_t)u, (uint32_t)(u >> 32), ws, tl);
        else       run_passes<DIM, true, true, POW2>(cp, bits_s, pc_c, head_c, ring_c, stage, (uint32_t)u, (uint32_t)(u >> 32), ws, tl);
        unsigned int size = 1u + ws.mywon;     // the seed and what this warp claimed itself
        if (ws.handed) {
            // sites have left this warp's hands: the update is complete when nothing is pending anywhere
            unsigned int polls = 0;
            unsigned long long pcv = 0;
            for (;;) {
                if (lane == 0) pcv = cl_ld_u64(pc_c);
                pcv = __shfl_sync(kFullMask, pcv, 0);
                ++polls;
                if ((unsigned int)pcv == 0u) break;
                if ((polls & 0x3FFu) == 0u) {
                    unsigned int bad = 0;
                    if (lane == 0) {
                        if (ld_relaxed_u32(&ctl->error) != 0u) bad = 1;
                        else if (globaltimer_ns() - t0 > cp.watchdog_ns) { raise_abort(ctl, 3u); bad = 1; }
                    }
                    if (__shfl_sync(kFullMask, bad, 0)) { aborted = true; break; }
                }
            }
            polls_total += polls;
            const unsigned int claimed = (unsigned int)(pcv >> 32);
            size += claimed - prev_claimed;       // modulo 2^32: a cluster has at most 2^31 spins
            prev_claimed = claimed;
        }
        if (!aborted && lane == 0) {
            p.sizes[k] = size;                    // A7
            flipped += size;
            const unsigned long long dt = globaltimer_ns() - t0;
            p.ns_log[k] = dt > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)dt;
        }
        if (p.measure && !aborted) {
            // "+ measurement": every CTA evaluates its slab (measure_slab); the sums and the arrivals come back in one word
            if (lane < cp.nC) cl_st_u32(mapa(mreq_s, lane), (unsigned int)k + 1u);
            unsigned int bad = 0;
            if (lane == 0) {
                unsigned long long acc;
                unsigned int polls = 0;
                while (((acc = cl_ld_u64(macc_c)) >> 51) != (unsigned long long)cp.nC) {
                    if ((++polls & 0x3FFu) == 0u) {
                        if (ld_relaxed_u32(&ctl->error) != 0u) { bad = 1; break; }
                        if (globaltimer_ns() - t0 > cp.watchdog_ns) { raise_abort(ctl, 6u); bad = 1; break; }
                    }
                }
                if (!bad) {
                    *reinterpret_cast<volatile unsigned long long *>(&sh.meas_acc) = 0ull;     // every CTA has arrived: nobody adds until the next request
                    const long long un = (long long)(acc & ((1ull << 26) - 1ull)), ng = (long long)((acc >> 26) & ((1ull << 25) - 1ull));
                    lastE = 2ll * un - (long long)DIM * (long long)p.geo.N;
                    lastM = (long long)p.geo.N - 2ll * ng;
                    p.E_log[k] = lastE;
                    p.M_log[k] = lastM;
                    mom.add(lastE, lastM);
                }
            }
            if (__shfl_sync(kFullMask, bad, 0)) aborted = true;
        }
    }
    if (p.measure && lane == 0 && !aborted && p.n_updates > 0) { ctl->E = lastE; ctl->M = lastM; mom.store(ctl->moments); }
    // everybody leaves
    if (lane < cp.nC) cl_st_u32(mapa(stop_s, lane), 1u);
    if (lane == 0) {
        ctl->stats[0] += p.n_updates;
        ctl->stats[1] += flipped;
        ctl->stats[9] += polls_total;
    }
}

template <int DIM, bool POW2>
__global__ void __launch_bounds__(kCT, 1) growth_cluster_kernel(const __grid_constant__ ClusterParams cp)
{
    extern __shared__ __align__(16) unsigned char smem_c[];
    __shared__ CShared sh;
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned int tid = threadIdx.x, warp = tid >> 5;
    const unsigned int rank = cluster.block_rank();
    const GrowthParams &p = cp.g;
    uint32_t *const bits = reinterpret_cast<uint32_t *>(smem_c);
    uint32_t *const ring = bits + cp.wpc;
    uint32_t *const stage = ring + cp.ring_cap;
    CTally tl;
    // the error flag is sticky: an earlier launch of this handle was aborted and the host has not yet looked
    const bool dead = ld_relaxed_u32(&p.ctl->error) != 0u;

    for (unsigned int i = tid; i < cp.ring_cap; i += kCT) ring[i] = kEmpty;
    if (tid == 0) {
        sh.head = sh.tail = 0u;
        sh.pc = 0ull;
        sh.upd = 0u;
        sh.stop = dead ? 1u : 0u;
        sh.watcher = 0u;
        sh.meas_req = 0u;
        sh.meas_un = sh.meas_ng = sh.meas_warps = 0u;
        sh.meas_acc = 0ull;
    }
    // ---- prologue: my slab of the lattice, one bit per spin (bit = 1: spin -1); word w of the lattice = sites 32 w ..
    // (the last word of the lattice may be partial and the last CTAs may hold fewer words than wpc, or none)
    const uint4 *const src = reinterpret_cast<const uint4 *>(p.spins);
    {
        // four words (eight 16-byte loads) in flight per thread: the slab is a megabyte per SM, and what the copy waits for
        // is the latency of L2 / HBM, not their bandwidth
        constexpr uint32_t U = 4;
        for (uint32_t w0 = tid; w0 < cp.wpc; w0 += kCT * U) {
            uint4 lo[U], hi[U];
            bool full[U];
#pragma unroll
            for (uint32_t u = 0; u < U; ++u) {
                const uint32_t w = w0 + u * kCT, gw = rank * cp.wpc + w;
                full[u] = w < cp.wpc && gw < cp.words && gw * 32u + 32u <= p.geo.N;
                if (full[u]) { lo[u] = __ldcg(src + 2u * (size_t)gw); hi[u] = __ldcg(src + 2u * (size_t)gw + 1u); }
            }
#pragma unroll
            for (uint32_t u = 0; u < U; ++u) {
                const uint32_t w = w0 + u * kCT, gw = rank * cp.wpc + w, first = gw * 32u;
                if (w >= cp.wpc) continue;
                uint32_t v = 0u;
                if (full[u]) v = pack16(lo[u]) | (pack16(hi[u]) << 16);
                else if (gw < cp.words) for (uint32_t i = first; i < p.geo.N; ++i) v |= (p.spins[i] < 0 ? 1u : 0u) << (i - first);
                bits[w] = v;
            }
        }
    }
    cluster.sync();                  // every CTA's shared memory is initialised before a peer touches it

    if (!dead) {
        if (warp == 0u && rank == 0u) monitor_warp<DIM, POW2>(cp, sh, smem_addr(bits), smem_addr(ring), stage, tl);
        else worker_warp<DIM, POW2>(cp, sh, smem_addr(bits), smem_addr(ring), stage + warp * kCStage, rank, tl);
    }
    cluster.sync();                  // no peer touches this CTA's shared memory any more

    // ---- epilogue: my slab back to the int8 lattice
    if (!dead) {
        uint4 *const dst = reinterpret_cast<uint4 *>(p.spins);
        for (uint32_t w = tid; w < cp.wpc; w += kCT) {
            const uint32_t gw = rank * cp.wpc + w, first = gw * 32u;
            if (gw >= cp.words) continue;
            const uint32_t b = bits[w];
            if (first + 32u <= p.geo.N) {
                dst[2u * (size_t)gw] = unpack16(b & 0xFFFFu);
                dst[2u * (size_t)gw + 1u] = unpack16(b >> 16);
            } else {
                for (uint32_t i = first; i < p.geo.N; ++i) p.spins[i] = ((b >> (i - first)) & 1u) ? (int8_t)-1 : (int8_t)1;
            }
        }
    }
    Control *ctl = p.ctl;
    const unsigned int a = __reduce_add_sync(kFullMask, tl.attempts);
    if ((tid & 31u) == 0u) {
        if (a) atomicAdd(&ctl->stats[7], (unsigned long long)a);
        if (tl.steals) atomicAdd(&ctl->stats[11], (unsigned long long)tl.steals);
        if (tl.ring_pushes) atomicAdd(&ctl->stats[12], (unsigned long long)tl.ring_pushes);
        if (tl.passes) atomicAdd(&ctl->stats[13], (unsigned long long)tl.passes);
        if (tl.spills) atomicAdd(&ctl->stats[14], (unsigned long long)tl.spills);
#ifdef WOLFF_PROFILE
        // [2] cycles in passes  [3] sites expanded  [4] cycles in hand-overs  [10] hand-overs  [6] cycles from a take to the
        // first pass  [8] takes  [15] passes of CTA 0's warps
        atomicAdd(&ctl->stats[2], tl.cyc_pass); atomicAdd(&ctl->stats[3], tl.sites); atomicAdd(&ctl->stats[4], tl.cyc_hand);
        atomicAdd(&ctl->stats[10], (unsigned long long)tl.hands); atomicAdd(&ctl->stats[6], tl.cyc_take); atomicAdd(&ctl->stats[8], (unsigned long long)tl.takes);
        if (rank == 0u) atomicAdd(&ctl->stats[15], (unsigned long long)tl.passes);
#endif
    }
}

template <int DIM, bool POW2>
cudaError_t set_attributes(size_t smem_bytes, int nC)
{
    const void *fn = reinterpret_cast<const void *>(&growth_cluster_kernel<DIM, POW2>);
    (void)smem_bytes;
    cudaError_t e = allow_max_dynamic_smem(fn);
    if (e != cudaSuccess) return e;
    if (nC > 8) e = cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    return e;
}

template <int DIM, bool POW2>
cudaError_t launch_one(const ClusterParams &cp, size_t smem_bytes, cudaStream_t stream, int *max_clusters)
{
    // per-process kernel attributes: another live handle may have changed them since this one made its plan
    cudaError_t e = set_attributes<DIM, POW2>(smem_bytes, (int)cp.nC);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(cp.nC);
    cfg.blockDim = dim3(kCT);
    cfg.dynamicSmemBytes = smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = cp.nC;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    if (max_clusters) return cudaOccupancyMaxActiveClusters(max_clusters, growth_cluster_kernel<DIM, POW2>, &cfg);
    return cudaLaunchKernelEx(&cfg, growth_cluster_kernel<DIM, POW2>, cp);
}

}  // namespace

size_t cluster_smem_bytes(uint32_t wpc, uint32_t ring_cap)
{
    return ((size_t)wpc + (size_t)ring_cap + (size_t)kCWarps * kCStage) * sizeof(uint32_t);
}

namespace {
cudaError_t dispatch(const ClusterParams &cp, int dim, bool pow2, size_t smem_bytes, cudaStream_t stream, int *max_clusters)
{
    if (dim == 2) return pow2 ? launch_one<2, true>(cp, smem_bytes, stream, max_clusters) : launch_one<2, false>(cp, smem_bytes, stream, max_clusters);
    return pow2 ? launch_one<3, true>(cp, smem_bytes, stream, max_clusters) : launch_one<3, false>(cp, smem_bytes, stream, max_clusters);
}
}  // namespace

// The launch shape for a lattice: the largest cluster (at most max_ctas CTAs) whose CTAs each hold a power-of-two number
// of 32-bit words of the bit lattice, the ring and the stages in their shared memory.  false: the lattice does not fit
// one cluster (more than 2^24 spins), or no such cluster can be resident.
bool cluster_plan(int dim, const Geometry &geo, int max_ctas, uint32_t ring_cap, size_t smem_optin, ClusterParams *cp, size_t *smem_bytes,
                  int *max_clusters)
{
    // sites are carried in 24 bits and divided by L and L^2 with 40-bit reciprocals: N <= 2^24, L^2 <= 2^16 in 3D
    const uint64_t N = geo.N;
    if (N > (1ull << 24) || (dim == 3 && (uint64_t)geo.L * geo.L > (1ull << 16))) return false;
    const uint64_t words = (N + 31) / 32;
    uint32_t nC = 16;
    while (nC > 1 && (nC > (uint32_t)max_ctas || nC > words)) nC >>= 1;
    uint32_t wpc = 1;
    while ((uint64_t)wpc * nC < words) wpc <<= 1;
    const size_t smem = cluster_smem_bytes(wpc, ring_cap);
    if (smem + 1024 > smem_optin) return false;
    int clusters = 0;
    const cudaError_t e = cluster_prepare(dim, geo.pow2 != 0u, nC, smem, &clusters);
    if (e != cudaSuccess || clusters < 1) { cudaGetLastError(); return false; }
    *cp = ClusterParams{};
    cp->nC = nC;
    cp->wpc = wpc;
    cp->wpc_log = 0;
    while ((1u << cp->wpc_log) < wpc) ++cp->wpc_log;
    cp->words = (uint32_t)words;
    cp->magicL = ((1ull << 40) + (uint64_t)geo.L - 1) / (uint64_t)geo.L;
    cp->magicLL = ((1ull << 40) + (uint64_t)geo.LL - 1) / (uint64_t)geo.LL;
    cp->ring_cap = ring_cap;
    cp->spill_log = 0;
    while ((1ull << cp->spill_log) < N) ++cp->spill_log;
    *smem_bytes = smem;
    if (max_clusters) *max_clusters = clusters;
    return true;
}

cudaError_t cluster_prepare(int dim, bool pow2, uint32_t nC, size_t smem_bytes, int *max_clusters)
{
    ClusterParams cp{};
    cp.nC = nC;
    return dispatch(cp, dim, pow2, smem_bytes, nullptr, max_clusters);
}

cudaError_t launch_growth_cluster(const ClusterParams &cp, int dim, size_t smem_bytes, cudaStream_t stream)
{
    return dispatch(cp, dim, cp.g.geo.pow2 != 0u, smem_bytes, stream, nullptr);
}

}  // namespace wolff
