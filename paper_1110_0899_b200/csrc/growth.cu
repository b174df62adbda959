// growth.cu -- the persistent cluster-growth kernel.
//
// One launch performs n_updates Wolff single-cluster updates (steps i-v), each
// grown wave-front parallel (step iii'): every spin added in the previous level
// is expanded by one thread.  What differs from the paper's GTX-285 design:
//   - bond variables come from a counter-based Philox keyed on (seed, update, edge), so the
//     cluster is a well-defined connected component and any traversal order gives the same bits;
//   - "join the cluster" is one atomic that flips the spin (no flag word, and no
//     per-direction barrier): 2*dim barriers per level become one;
//   - small frontiers are grown by ONE CTA out of shared-memory queues with __syncthreads only;
//     when the frontier outgrows `up`, the level loop becomes grid-wide over the global cluster
//     list (the ic/in list of PAPER.md:50) with one atomic barrier per level, and drops back when
//     the frontier narrows to `down`;
//   - the update loop itself is inside the kernel ("(v) Go to (i)").
#include "internal.h"

namespace wolff {

namespace {

constexpr unsigned int kFullMask = 0xFFFFFFFFu;

__device__ __forceinline__ unsigned long long pack_bar(unsigned int gen, unsigned int phase, unsigned int hi)
{
    return ((unsigned long long)(gen & 0xFFFFFFu) << 40) | ((unsigned long long)(phase & 0xFFu) << 32) |
           (unsigned long long)hi;
}
__device__ __forceinline__ unsigned int bar_gen(unsigned long long w) { return (unsigned int)(w >> 40); }
__device__ __forceinline__ unsigned int bar_phase(unsigned long long w) { return (unsigned int)(w >> 32) & 0xFFu; }
__device__ __forceinline__ unsigned int bar_hi(unsigned long long w) { return (unsigned int)w; }

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

// Expand one frontier site per lane (A2-A5): gather the 2*DIM neighbour spins, decide the bonds,
// claim-and-flip, and append the winners to dst[] with ONE atomic per warp on *dst_count
// (ballot/popc aggregation).  dst/dst_count are the shared-memory queue in one-CTA mode and the
// global cluster list and its tail in grid mode.  Must be called by all 32 lanes of a warp.
template <int DIM, bool POW2>
__device__ __forceinline__ void expand_sites(const GrowthParams &p, int s0, uint32_t u_lo, uint32_t u_hi,
                                             bool valid, uint32_t i, uint32_t *dst, unsigned int *dst_count,
                                             unsigned int &attempts)
{
    uint32_t nbr[2 * DIM];
    bool cand[2 * DIM];
    unsigned int old[2 * DIM];
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) { nbr[k] = 0u; cand[k] = false; old[k] = 0u; }

    if (valid) {
        neighbours<DIM, POW2>(p.geo, i, nbr);
        // A2: neighbour spins (L2 loads; in flight while the Philox rounds below execute)
        int sp[2 * DIM];
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) sp[k] = load_spin_l2(p.spins, nbr[k]);
        // A3: bond variables.  The bond to the +d neighbour is owned by this site (word d of the
        // site's block); the bond to the -d neighbour is owned by that neighbour (word d of ITS block).
        const uint4 fwd = philox4x32_10(i, kDomainBond, u_lo, u_hi, p.key0, p.key1);
        uint32_t bondword[2 * DIM];
#pragma unroll
        for (int d = 0; d < DIM; ++d) {
            bondword[2 * d] = word_of(fwd, d);
            const uint4 bwd = philox4x32_10(nbr[2 * d + 1], kDomainBond, u_lo, u_hi, p.key0, p.key1);
            bondword[2 * d + 1] = word_of(bwd, d);
        }
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) cand[k] = (sp[k] == s0) && ((unsigned long long)bondword[k] < p.thr);
    }

    // A4: claim-and-flip the same-sign neighbours behind active bonds.  All atomics of a lane are
    // issued before any result is looked at, so their L2 round trips overlap.
    unsigned int *const words = reinterpret_cast<unsigned int *>(p.spins);
    if (s0 > 0) {   // uniform for the whole update
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k)
            if (cand[k]) old[k] = atomicOr(words + (nbr[k] >> 2), 0xFEu << ((nbr[k] & 3u) * 8u));
    } else {
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k)
            if (cand[k]) old[k] = atomicAnd(words + (nbr[k] >> 2), ~(0xFEu << ((nbr[k] & 3u) * 8u)));
    }
    const unsigned int s0_byte = (unsigned int)s0 & 0xFFu;
    unsigned int ballots[2 * DIM];
    unsigned int total = 0;
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) {
        const bool won = cand[k] && (((old[k] >> ((nbr[k] & 3u) * 8u)) & 0xFFu) == s0_byte);
        attempts += cand[k] ? 1u : 0u;
        ballots[k] = __ballot_sync(kFullMask, won);
        total += __popc(ballots[k]);
    }

    // A5: warp-aggregated append
    if (total != 0u) {   // warp-uniform
        const unsigned int lane = threadIdx.x & 31u;
        unsigned int base = 0;
        if (lane == 0u) base = atomicAdd(dst_count, total);
        base = __shfl_sync(kFullMask, base, 0);
        const unsigned int bit = 1u << lane;
        const unsigned int lt = bit - 1u;
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) {
            if (ballots[k] & bit) dst[base + __popc(ballots[k] & lt)] = nbr[k];
            base += __popc(ballots[k]);
        }
    }
}

struct SharedState {
    unsigned int cnt[3];       // rotating level counters of the one-CTA queues
    int s0;                    // broadcast: seed spin of the current update
    unsigned long long word;   // broadcast: barrier word
};

// Grid-wide level loop over the global cluster list (A2-A6, grid mode).  Called by every CTA with
// identical (lo, hi, gen); returns with the window/phase decided by the last CTA to arrive.
template <int DIM, bool POW2>
__device__ __forceinline__ unsigned int grid_levels(const GrowthParams &p, SharedState &sh,
                                                    int s0, unsigned long long u, uint32_t &lo, uint32_t &hi,
                                                    unsigned int &gen, unsigned int &attempts,
                                                    unsigned long long &levels, uint32_t &widest)
{
    constexpr int T = kGrowthThreads;
    const unsigned int tid = threadIdx.x;
    const unsigned int G = gridDim.x, b = blockIdx.x;
    const uint32_t u_lo = (uint32_t)u, u_hi = (uint32_t)(u >> 32);
    Control *ctl = p.ctl;
    for (;;) {
        const uint32_t n = hi - lo;
        if (n > widest) widest = n;
        ++levels;
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
                expand_sites<DIM, POW2>(p, s0, u_lo, u_hi, valid, site, p.clist, &ctl->tail, attempts);
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
                const unsigned int phase = (width == 0u) ? kPhaseDone : (width <= p.down ? kPhaseToCta : kPhaseGrid);
                st_relaxed_u32(&ctl->arrive, 0u);
                w = pack_bar(gen + 1u, phase, t);
                st_release_u64(&ctl->bar, w);
            } else {
                w = wait_generation(ctl, gen + 1u, true);
            }
            sh.word = w;
        }
        __syncthreads();
        const unsigned long long w = sh.word;
        ++gen;
        lo = hi;
        hi = bar_hi(w);
        const unsigned int phase = bar_phase(w);
        if (phase != kPhaseGrid) return phase;
    }
}

template <int DIM, bool POW2>
__global__ void __launch_bounds__(kGrowthThreads, 1) growth_kernel(const GrowthParams p)
{
    constexpr int T = kGrowthThreads;
    extern __shared__ __align__(16) uint32_t smem_q[];   // two queue buffers of p.qcap entries
    __shared__ SharedState sh;
    uint32_t *const q0 = smem_q;
    uint32_t *const q1 = smem_q + p.qcap;
    const unsigned int tid = threadIdx.x;
    Control *ctl = p.ctl;
    unsigned int gen = 0;          // the host zeroes the control block before every launch
    unsigned int attempts = 0;
    unsigned long long levels_grid = 0;
    uint32_t widest = 0;

    if (blockIdx.x != 0) {
        // ---------------------------------------------------------------- worker CTAs
        for (;;) {
            if (tid == 0) sh.word = wait_generation(ctl, gen + 1u, false);
            __syncthreads();
            const unsigned long long w = sh.word;
            __syncthreads();
            ++gen;
            const unsigned int phase = bar_phase(w);
            if (phase != kPhaseGrid) break;   // exit or abort
            uint32_t lo = ld_relaxed_u32(&ctl->lo);
            uint32_t hi = bar_hi(w);
            const int s0 = (int)ld_relaxed_u32(reinterpret_cast<unsigned int *>(&ctl->s0));
            const unsigned long long u = __ldcg(&ctl->u);
            const unsigned int out = grid_levels<DIM, POW2>(p, sh, s0, u, lo, hi, gen, attempts, levels_grid, widest);
            if (out == kPhaseAbort) break;
        }
        if (attempts) atomicAdd(&ctl->stats[6], (unsigned long long)attempts);
        return;
    }

    // -------------------------------------------------------------------- CTA 0: the update loop
    unsigned long long flipped = 0, levels_cta = 0, ups = 0, downs = 0;
    bool aborted = false;
    for (unsigned long long k = 0; k < p.n_updates && !aborted; ++k) {
        const unsigned long long u = p.u0 + k;
        const uint32_t u_lo = (uint32_t)u, u_hi = (uint32_t)(u >> 32);
        // A1: seed draw (reading R8) and initial flip
        if (tid == 0) {
            const uint4 x = philox4x32_10(0u, kDomainSite, u_lo, u_hi, p.key0, p.key1);
            const unsigned long long r = (unsigned long long)x.x | ((unsigned long long)x.y << 32);
            const uint32_t i0 = (uint32_t)__umul64hi(r, (unsigned long long)p.geo.N);
            const int s = load_spin_l2(p.spins, i0);
            claim_and_flip(p.spins, i0, s);
            q0[0] = i0;
            sh.cnt[0] = 1u;
            sh.cnt[1] = 0u;
            sh.s0 = s;
        }
        __syncthreads();
        const int s0 = sh.s0;
        unsigned long long size = 1;
        unsigned int lvl = 0;        // level counter modulo 3 (counter slot)
        uint32_t *cur = q0, *nxt = q1;
        for (;;) {
            const unsigned int n = sh.cnt[lvl];
            if (n == 0u) break;
            if (n > widest) widest = n;
            if (n > p.up) {
                // ---- spill: the frontier becomes the window [0, n) of the global list, all CTAs join
                for (unsigned int e = tid; e < n; e += T) p.clist[e] = cur[e];
                if (tid == 0) {
                    st_relaxed_u32(&ctl->tail, n);
                    st_relaxed_u32(&ctl->lo, 0u);
                    st_relaxed_u32(reinterpret_cast<unsigned int *>(&ctl->s0), (unsigned int)s0);
                    ctl->u = u;
                }
                __threadfence();
                __syncthreads();
                if (tid == 0) st_release_u64(&ctl->bar, pack_bar(gen + 1u, kPhaseGrid, n));
                ++gen;
                ++ups;
                uint32_t lo = 0u, hi = n;
                const unsigned int out = grid_levels<DIM, POW2>(p, sh, s0, u, lo, hi, gen, attempts, levels_grid, widest);
                size += (unsigned long long)(hi - n);
                if (out == kPhaseAbort) { aborted = true; break; }
                if (out == kPhaseDone) break;
                // ---- back to one CTA: reload the window into the shared-memory queue
                ++downs;
                const unsigned int m = hi - lo;
                for (unsigned int e = tid; e < m; e += T) q0[e] = __ldcg(p.clist + lo + e);
                if (tid == 0) { sh.cnt[0] = m; sh.cnt[1] = 0u; }
                __syncthreads();
                lvl = 0; cur = q0; nxt = q1;
                continue;
            }
            // ---- one-CTA level: shared-memory queues, __syncthreads only
            ++levels_cta;
            const unsigned int lvl1 = (lvl == 2u) ? 0u : lvl + 1u;
            const unsigned int lvl2 = (lvl1 == 2u) ? 0u : lvl1 + 1u;
            if (tid == 0) sh.cnt[lvl2] = 0u;
            for (unsigned int pass = 0; pass < n; pass += T) {
                const unsigned int idx = pass + tid;
                const bool valid = idx < n;
                const uint32_t site = valid ? cur[idx] : 0u;
                expand_sites<DIM, POW2>(p, s0, u_lo, u_hi, valid, site, nxt, &sh.cnt[lvl1], attempts);
            }
            __syncthreads();
            size += sh.cnt[lvl1];
            lvl = lvl1;
            uint32_t *t = cur; cur = nxt; nxt = t;
        }
        // A7: epilogue
        if (tid == 0) p.sizes[k] = (uint32_t)size;
        flipped += size;
        __syncthreads();
    }
    if (tid == 0) {
        if (!aborted) st_release_u64(&ctl->bar, pack_bar(gen + 1u, kPhaseExit, 0u));
        ctl->stats[0] = p.n_updates;
        ctl->stats[1] = flipped;
        ctl->stats[2] = levels_cta;
        ctl->stats[3] = levels_grid;
        ctl->stats[4] = ups;
        ctl->stats[5] = downs;
        ctl->stats[7] = widest;
    }
    if (attempts) atomicAdd(&ctl->stats[6], (unsigned long long)attempts);
}

template <int DIM, bool POW2>
cudaError_t launch_one(const GrowthParams &p, int grid_ctas, size_t smem_bytes, cudaStream_t stream)
{
    void *args[] = { const_cast<GrowthParams *>(&p) };
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(&growth_kernel<DIM, POW2>), dim3(grid_ctas),
                                       dim3(kGrowthThreads), args, smem_bytes, stream);
}

template <int DIM, bool POW2>
cudaError_t prepare_one(size_t smem_bytes, int *ctas_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void *>(&growth_kernel<DIM, POW2>),
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    if (ctas_per_sm)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, growth_kernel<DIM, POW2>, kGrowthThreads, smem_bytes);
    return e;
}

}  // namespace

cudaError_t launch_growth(const GrowthParams &p, int dim, int grid_ctas, size_t smem_bytes, cudaStream_t stream)
{
    const bool pow2 = p.geo.pow2 != 0u;
    if (dim == 2) return pow2 ? launch_one<2, true>(p, grid_ctas, smem_bytes, stream) : launch_one<2, false>(p, grid_ctas, smem_bytes, stream);
    return pow2 ? launch_one<3, true>(p, grid_ctas, smem_bytes, stream) : launch_one<3, false>(p, grid_ctas, smem_bytes, stream);
}

cudaError_t growth_max_ctas(int dim, bool pow2, size_t smem_bytes, int *ctas_per_sm)
{
    if (dim == 2) return pow2 ? prepare_one<2, true>(smem_bytes, ctas_per_sm) : prepare_one<2, false>(smem_bytes, ctas_per_sm);
    return pow2 ? prepare_one<3, true>(smem_bytes, ctas_per_sm) : prepare_one<3, false>(smem_bytes, ctas_per_sm);
}

cudaError_t growth_prepare(int dim, bool pow2, size_t smem_bytes) { return growth_max_ctas(dim, pow2, smem_bytes, nullptr); }

}  // namespace wolff
