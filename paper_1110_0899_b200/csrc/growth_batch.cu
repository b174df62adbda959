// growth_batch.cu -- R independent chains in ONE persistent launch, one CTA per chain.
//
// The paper's results are sweeps: the Binder ratio and the timings over temperatures and lattice sizes
// (Figs. 1-2), i.e. many independent Wolff chains.  One chain at T_c keeps a handful of frontier
// sites per CTA busy and, in the small-cluster regime (high T, or the literal random start of the BASELINE configs),
// a single SM; replicas are what turns the chip into throughput.  Here every chain (its own T, J and seed; dim and L
// shared) is grown by one CTA at a time, level-synchronously with __syncthreads only (the one-CTA tier of growth.cu:
// PAPER.md:84-98 step iii', one thread per wave-front spin), the update loop inside the kernel.  CTAs
// take chains from a counter, so a launch holds as many chains in flight as CTAs are resident (8-16 per SM).
//
// Per chain: int8 lattice in global memory (L2 / HBM; claim-and-flip is the same single idempotent atomic as in
// growth.cu); the member list of the running cluster (uint32 x N, the ic/in list of PAPER.md:50) doubles as the
// frontier queue -- level l is the window [lo, hi) of the list -- with a copy of the window in shared memory while
// it fits.  Bond variables: Philox4x32-10 keyed on (seed of the chain, update, edge), so chain r computes exactly what
// a single chain created with (dim, L, J[r], T[r], seed[r]) computes.
//
// Bit-packed, shared-memory-resident variant ("1 bit/spin: 2D L=1024 = 128 KiB fits one SM's shared
// memory"; knob "resident"): for the length of a chain's turn its lattice lives in the CTA's shared memory as one bit per
// spin (the sign), packed from the int8 lattice in a prologue and unpacked in an epilogue.  Gather and claim then are
// ld.shared / atom.shared on a 32-bit word (claim = atom.or / atom.and of one bit, the same idempotent single atomic),
// and a second bit plane carries the membership marks of a measured run.
//
// In-kernel measurement ("measure" = 1) as in growth.cu: members of the running cluster carry a mark (bit 1 of the
// byte), dE = 2 * sum over the cluster's boundary bonds, dM = -2 s0 |C|, running from a whole-lattice evaluation
// the host queues before the launch.
#include "expand.cuh"
#include "internal.h"

namespace wolff {
namespace {

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned int lds_u32(uint32_t saddr)
{
    unsigned int v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ unsigned int atoms_or(uint32_t saddr, unsigned int v)
{
    unsigned int old;
    asm volatile("atom.shared.or.b32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ unsigned int atoms_and(uint32_t saddr, unsigned int v)
{
    unsigned int old;
    asm volatile("atom.shared.and.b32 %0, [%1], %2;" : "=r"(old) : "r"(saddr), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ void reds_or(uint32_t saddr, unsigned int v) { asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }
__device__ __forceinline__ void reds_and(uint32_t saddr, unsigned int v) { asm volatile("red.shared.and.b32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }

// Four spin bytes (0x01 / 0xFF) -> four sign bits (byte k -> bit k), and back.
__device__ __forceinline__ uint32_t pack4(uint32_t bytes) { return ((bytes & 0x80808080u) * 0x00204081u) >> 28; }
__device__ __forceinline__ uint32_t unpack4(uint32_t nibble) { return 0x01010101u | (((nibble * 0x00204081u) & 0x01010101u) * 0xFEu); }

// A2-A4 on the bit-packed lattice (one site per lane; the counterpart of claim_neighbours() in expand.cuh).  sign_s: the
// sign plane (bit = 1: spin -1), mark_s: the plane of membership marks of the running cluster (0: not a measured run);
// both shared-window addresses.  s0neg: the seed spin is -1.
template <int DIM, bool POW2>
__device__ __forceinline__ void claim_neighbours_bits(const GrowthParams &p, uint32_t sign_s, uint32_t mark_s, unsigned int s0neg, uint32_t u_lo,
                                                      uint32_t u_hi, bool valid, uint32_t i, uint32_t (&nbr)[2 * DIM], unsigned int &won,
                                                      unsigned int &attempts)
{
    bool cand[2 * DIM];
    unsigned int old[2 * DIM];
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) { nbr[k] = 0u; cand[k] = false; old[k] = 0u; }
    won = 0u;
    if (valid) {
        uint32_t x, y, z;
        site_coords<DIM, POW2>(p.geo, i, x, y, z);
        neighbours_at<DIM>(p.geo, i, x, y, z, nbr);
        unsigned int sp[2 * DIM];
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) sp[k] = (lds_u32(sign_s + ((nbr[k] >> 5) << 2)) >> (nbr[k] & 31u)) & 1u;
        uint32_t ctr0[1 + DIM];
        uint4 blk[1 + DIM];
        ctr0[0] = i;
#pragma unroll
        for (int d = 0; d < DIM; ++d) ctr0[1 + d] = nbr[2 * d + 1];
        philox4x32_10_multi<1 + DIM>(ctr0, kDomainBond, u_lo, u_hi, p.key0, p.key1, blk);
#pragma unroll
        for (int d = 0; d < DIM; ++d) {
            cand[2 * d] = (unsigned long long)word_of(blk[0], d) < p.thr && sp[2 * d] == s0neg;
            cand[2 * d + 1] = (unsigned long long)word_of(blk[1 + d], d) < p.thr && sp[2 * d + 1] == s0neg;
        }
    }
    // A4: one atomic on the word that holds the neighbour's bit: set it (+1 -> -1) or clear it (-1 -> +1)
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) {
        if (cand[k]) {
            const uint32_t a = sign_s + ((nbr[k] >> 5) << 2), bit = 1u << (nbr[k] & 31u);
            old[k] = s0neg ? atoms_and(a, ~bit) : atoms_or(a, bit);
        }
    }
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) {
        const bool w = cand[k] && ((old[k] >> (nbr[k] & 31u)) & 1u) == s0neg;
        attempts += cand[k] ? 1u : 0u;
        won |= w ? (1u << k) : 0u;
        if (w && mark_s) reds_or(mark_s + ((nbr[k] >> 5) << 2), 1u << (nbr[k] & 31u));
    }
}

// Post-pass of a measured update on the bit-packed lattice (boundary_partial() of expand.cuh): members carry a mark.
template <int DIM, bool POW2>
__device__ __forceinline__ int boundary_partial_bits(const Geometry &geo, uint32_t sign_s, uint32_t mark_s, const uint32_t *list, unsigned int s0neg,
                                                     uint32_t size, uint32_t first, uint32_t step)
{
    int acc = 0;
    for (uint32_t e = first; e < size; e += step) {
        const uint32_t i = __ldcg(list + e);
        uint32_t x, y, z, nbr[2 * DIM];
        site_coords<DIM, POW2>(geo, i, x, y, z);
        neighbours_at<DIM>(geo, i, x, y, z, nbr);
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) {
            const uint32_t wo = (nbr[k] >> 5) << 2, sh = nbr[k] & 31u;
            const unsigned int marked = (lds_u32(mark_s + wo) >> sh) & 1u, neg = (lds_u32(sign_s + wo) >> sh) & 1u;
            if (!marked) acc += (neg == s0neg) ? 1 : -1;
        }
    }
    return acc;
}

struct BatchShared {
    unsigned int cnt[3];       // rotating level counters (entries appended to the list by the running level)
    unsigned int chain;        // the chain this CTA works on
    int s0;
    unsigned long long post_acc;
};

template <int DIM, bool POW2, bool BITS>
__global__ void __launch_bounds__(kBatchMaxThreads) growth_batch_kernel(const BatchParams bp)
{
    extern __shared__ __align__(16) uint32_t smem_bq[];          // two frontier buffers of bp.qcap entries [+ the bit planes]
    // BITS: the sign plane and (measured runs) the mark plane behind the frontier buffers
    const uint32_t nwords = (bp.geo.N + 31u) >> 5;
    uint32_t *const sign_w = smem_bq + 2u * bp.qcap;
    const uint32_t sign_s = smem_addr(sign_w), mark_s = (BITS && bp.measure) ? sign_s + nwords * 4u : 0u;
    __shared__ BatchShared sh;
    const unsigned int tid = threadIdx.x, T = blockDim.x, lane = tid & 31u;
    const unsigned int lt = (1u << lane) - 1u;
    unsigned long long t_updates = 0, t_flipped = 0, t_levels = 0;
    unsigned int attempts = 0;

    for (;;) {
        __syncthreads();
        if (tid == 0) sh.chain = atomicAdd(bp.next, 1u);
        __syncthreads();
        const unsigned int r = sh.chain;
        if (r >= bp.R) break;

        // ---- this chain as a single-chain problem
        GrowthParams p{};
        p.spins = bp.spins + (size_t)r * bp.lattice_stride;
        p.clist = bp.lists + (size_t)r * bp.geo.N;
        p.geo = bp.geo;
        p.key0 = bp.keys[r].x; p.key1 = bp.keys[r].y;
        p.thr = bp.thr[r];
        p.measure = bp.measure;
        p.claim_bits = bp.measure ? 0xFCu : 0xFEu;
        uint32_t *const sizes = bp.sizes + (size_t)r * bp.n_updates;
        long long runE = 0, runM = 0;
        Moments mom;
        if (bp.measure && tid == 0) { runE = bp.EM[2 * r]; runM = bp.EM[2 * r + 1]; mom.load(bp.moments + 10 * (size_t)r); }
        if (BITS) {
            // prologue: the chain's int8 lattice -> one bit per spin in shared memory (32 sites per word)
            const uint32_t full = bp.geo.N >> 5;
            for (uint32_t w = tid; w < nwords; w += T) {
                uint32_t word = 0;
                if (w < full) {
                    const uint4 lo4 = __ldcg(reinterpret_cast<const uint4 *>(p.spins + 32u * w));
                    const uint4 hi4 = __ldcg(reinterpret_cast<const uint4 *>(p.spins + 32u * w + 16u));
                    word = pack4(lo4.x) | (pack4(lo4.y) << 4) | (pack4(lo4.z) << 8) | (pack4(lo4.w) << 12) |
                           (pack4(hi4.x) << 16) | (pack4(hi4.y) << 20) | (pack4(hi4.z) << 24) | (pack4(hi4.w) << 28);
                } else {
                    for (uint32_t j = 32u * w; j < bp.geo.N; ++j) word |= (p.spins[j] < 0 ? 1u : 0u) << (j & 31u);
                }
                sign_w[w] = word;
                if (bp.measure) sign_w[nwords + w] = 0u;
            }
            __syncthreads();
        }

        for (unsigned long long k = 0; k < bp.n_updates; ++k) {
            const unsigned long long u = bp.u0 + k;
            const uint32_t u_lo = (uint32_t)u, u_hi = (uint32_t)(u >> 32);
            // A1: seed draw (reading R8) and initial flip
            if (tid == 0) {
                const uint4 x = philox4x32_10(0u, kDomainSite, u_lo, u_hi, p.key0, p.key1);
                const unsigned long long rr = (unsigned long long)x.x | ((unsigned long long)x.y << 32);
                const uint32_t i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
                int s;
                if (BITS) {
                    const uint32_t a = sign_s + ((i0 >> 5) << 2), bit = 1u << (i0 & 31u);
                    const unsigned int neg = (lds_u32(a) >> (i0 & 31u)) & 1u;
                    s = neg ? -1 : 1;
                    if (neg) atoms_and(a, ~bit); else atoms_or(a, bit);
                    if (mark_s) reds_or(mark_s + ((i0 >> 5) << 2), bit);
                } else {
                    s = load_spin_l2(p.spins, i0);
                    claim_with_bits(p.spins, i0, s, p.claim_bits);
                }
                p.clist[0] = i0;
                smem_bq[0] = i0;
                sh.cnt[0] = 0u; sh.cnt[1] = 0u;
                sh.s0 = s;
            }
            __syncthreads();
            const int s0 = sh.s0;
            uint32_t lo = 0u, hi = 1u;          // the frontier is list[lo, hi)
            unsigned int lvl = 0, par = 0;      // counter slot of the running level; frontier buffer
            bool in_smem = true;
            while (hi != lo) {
                const uint32_t n = hi - lo;
                const unsigned int lvl1 = lvl == 2u ? 0u : lvl + 1u;
                if (tid == 0) sh.cnt[lvl1] = 0u;                       // the counter of the level after this one
                const uint32_t *const cur = smem_bq + par * bp.qcap;
                uint32_t *const nxt = smem_bq + (par ^ 1u) * bp.qcap;
                for (uint32_t pass = 0; pass < n; pass += T) {
                    const uint32_t idx = pass + tid;
                    const bool valid = idx < n;
                    const uint32_t site = valid ? (in_smem ? cur[idx] : __ldcg(p.clist + lo + idx)) : 0u;
                    uint32_t nbr[2 * DIM], x, y, z;
                    unsigned int won;
                    if (BITS) claim_neighbours_bits<DIM, POW2>(p, sign_s, mark_s, s0 < 0 ? 1u : 0u, u_lo, u_hi, valid, site, nbr, won, attempts);
                    else claim_neighbours<DIM, POW2, false>(p, s0, u_lo, u_hi, valid, site, nbr, won, x, y, z, attempts);
                    // A5: winners -> the list (always) and the shared-memory copy of the next window (while it fits)
                    unsigned int ballots[2 * DIM], total = 0;
#pragma unroll
                    for (int q = 0; q < 2 * DIM; ++q) { ballots[q] = __ballot_sync(kFullMask, (won >> q) & 1u); total += __popc(ballots[q]); }
                    if (total != 0u) {
                        unsigned int base = 0;
                        if (lane == 0u) base = atomicAdd(&sh.cnt[lvl], total);
                        base = __shfl_sync(kFullMask, base, 0);
#pragma unroll
                        for (int q = 0; q < 2 * DIM; ++q) {
                            if (ballots[q] & (1u << lane)) {
                                const unsigned int pos = base + __popc(ballots[q] & lt);
                                if (WOLFF_CHECK(reinterpret_cast<unsigned int *>(bp.stats + 7), hi + pos < bp.geo.N && nbr[q] < bp.geo.N, 40))
                                    p.clist[hi + pos] = nbr[q];
                                if (pos < bp.qcap) nxt[pos] = nbr[q];
                            }
                            base += __popc(ballots[q]);
                        }
                    }
                }
                __syncthreads();                                       // A6: the level is complete
                const unsigned int added = sh.cnt[lvl];
                lo = hi; hi += added;
                in_smem = added <= bp.qcap;
                par ^= 1u;
                lvl = lvl1;
                ++t_levels;
            }
            const uint32_t size = hi;
            if (bp.measure) {
                // post-pass: dE from the cluster's boundary bonds while every member still carries its mark, then the
                // members get their plain value (see growth.cu)
                if (tid == 0) sh.post_acc = 0ull;
                __syncthreads();
                int part = BITS ? boundary_partial_bits<DIM, POW2>(p.geo, sign_s, mark_s, p.clist, s0 < 0 ? 1u : 0u, size, tid, T)
                                : boundary_partial<DIM, POW2>(p.geo, p.spins, p.clist, s0, size, tid, T);
                part = __reduce_add_sync(kFullMask, part);
                if (lane == 0u && part != 0) atomicAdd(&sh.post_acc, (unsigned long long)(long long)part);
                __syncthreads();
                if (BITS) {
                    for (uint32_t e = tid; e < size; e += T) {
                        const uint32_t i = __ldcg(p.clist + e);
                        reds_and(mark_s + ((i >> 5) << 2), ~(1u << (i & 31u)));
                    }
                } else {
                    const int8_t plain = (int8_t)(-s0);
                    for (uint32_t e = tid; e < size; e += T) p.spins[__ldcg(p.clist + e)] = plain;
                }
                if (tid == 0) {
                    runE += 2ll * (long long)sh.post_acc;
                    runM -= 2ll * (long long)s0 * (long long)size;
                    bp.E_log[(size_t)r * bp.n_updates + k] = runE;
                    bp.M_log[(size_t)r * bp.n_updates + k] = runM;
                    mom.add(runE, runM);
                }
            }
            if (tid == 0) sizes[k] = size;                             // A7
            t_flipped += size;
            ++t_updates;
            __syncthreads();
        }
        if (bp.measure && tid == 0) { bp.EM[2 * r] = runE; bp.EM[2 * r + 1] = runM; mom.store(bp.moments + 10 * (size_t)r); }
        if (BITS) {
            // epilogue: the bits -> the chain's int8 lattice
            const uint32_t full = bp.geo.N >> 5;
            for (uint32_t w = tid; w < nwords; w += T) {
                const uint32_t word = sign_w[w];
                if (w < full) {
                    uint4 lo4, hi4;
                    lo4.x = unpack4(word & 15u); lo4.y = unpack4((word >> 4) & 15u); lo4.z = unpack4((word >> 8) & 15u); lo4.w = unpack4((word >> 12) & 15u);
                    hi4.x = unpack4((word >> 16) & 15u); hi4.y = unpack4((word >> 20) & 15u); hi4.z = unpack4((word >> 24) & 15u); hi4.w = unpack4(word >> 28);
                    *reinterpret_cast<uint4 *>(p.spins + 32u * w) = lo4;
                    *reinterpret_cast<uint4 *>(p.spins + 32u * w + 16u) = hi4;
                } else {
                    for (uint32_t j = 32u * w; j < bp.geo.N; ++j) p.spins[j] = ((word >> (j & 31u)) & 1u) ? (int8_t)-1 : (int8_t)1;
                }
            }
        }
    }
    attempts = __reduce_add_sync(kFullMask, attempts);
    if (lane == 0u && attempts) atomicAdd(&bp.stats[3], (unsigned long long)attempts);
    if (tid == 0) {
        atomicAdd(&bp.stats[0], t_updates);
        atomicAdd(&bp.stats[1], t_flipped);
        atomicAdd(&bp.stats[2], t_levels);
    }
}

// E and M of every chain (the A8 reduction, one CTA per chain and slice): into EM[2r], EM[2r+1] by atomics on zeroed words.
template <int DIM>
__global__ void __launch_bounds__(256) batch_energy_kernel(const int8_t *spins, size_t stride, Geometry g, uint32_t R, uint32_t slices,
                                                           unsigned long long *acc)
{
    const uint32_t r = blockIdx.x / slices, sl = blockIdx.x - r * slices;
    if (r >= R) return;
    const int8_t *s = spins + (size_t)r * stride;
    unsigned long long unequal = 0, negative = 0;
    const uint32_t per = (g.N + slices - 1u) / slices, begin = sl * per, end = begin + per < g.N ? begin + per : g.N;
    for (uint32_t i = begin + threadIdx.x; i < end; i += blockDim.x) {
        uint32_t nbr[2 * DIM];
        if (g.pow2) neighbours<DIM, true>(g, i, nbr); else neighbours<DIM, false>(g, i, nbr);
        const int v = s[i];
        negative += (v < 0);
#pragma unroll
        for (int d = 0; d < DIM; ++d) unequal += ((s[nbr[2 * d]] < 0) != (v < 0));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unequal += __shfl_xor_sync(0xFFFFFFFFu, unequal, o);
        negative += __shfl_xor_sync(0xFFFFFFFFu, negative, o);
    }
    if ((threadIdx.x & 31u) == 0u) {
        if (unequal) atomicAdd(acc + 2 * (size_t)r, unequal);
        if (negative) atomicAdd(acc + 2 * (size_t)r + 1, negative);
    }
}

// The same for L a multiple of 16: sixteen sites per load (the loop of energy_magnetisation_vec16 in measure.cu), the chain
// in blockIdx.y.
template <int DIM>
__global__ void __launch_bounds__(256) batch_energy_vec16_kernel(const int8_t *spins, size_t stride, Geometry g, unsigned long long *acc)
{
    const uint32_t r = blockIdx.y;
    const int8_t *s = spins + (size_t)r * stride;
    const uint32_t chunks = g.N / 16u, chunks_per_row = g.L / 16u;
    unsigned long long unequal = 0, negative = 0;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < chunks; c += gridDim.x * blockDim.x) {
        const uint32_t i = c * 16u, row = c / chunks_per_row, cx = c - row * chunks_per_row;
        const uint32_t y = (DIM == 3) ? row % g.L : row;
        const uint4 a = *reinterpret_cast<const uint4 *>(s + i);
        const uint32_t inext = (cx + 1u == chunks_per_row) ? i + 16u - g.L : i + 16u;
        const uint32_t nb = (uint32_t)(uint8_t)s[inext];
        const uint32_t iy = (y + 1u == g.L) ? i - (g.LL - g.L) : i + g.L;
        const uint4 by = *reinterpret_cast<const uint4 *>(s + iy);
        uint32_t un = __popc((a.x ^ __funnelshift_r(a.x, a.y, 8)) & 0x80808080u) + __popc((a.y ^ __funnelshift_r(a.y, a.z, 8)) & 0x80808080u) +
                      __popc((a.z ^ __funnelshift_r(a.z, a.w, 8)) & 0x80808080u) + __popc((a.w ^ __funnelshift_r(a.w, nb, 8)) & 0x80808080u);
        un += __popc((a.x ^ by.x) & 0x80808080u) + __popc((a.y ^ by.y) & 0x80808080u) + __popc((a.z ^ by.z) & 0x80808080u) + __popc((a.w ^ by.w) & 0x80808080u);
        if (DIM == 3) {
            const uint32_t z = row / g.L;
            const uint32_t iz = (z + 1u == g.L) ? i - (g.N - g.LL) : i + g.LL;
            const uint4 bz = *reinterpret_cast<const uint4 *>(s + iz);
            un += __popc((a.x ^ bz.x) & 0x80808080u) + __popc((a.y ^ bz.y) & 0x80808080u) + __popc((a.z ^ bz.z) & 0x80808080u) + __popc((a.w ^ bz.w) & 0x80808080u);
        }
        unequal += un;
        negative += __popc(a.x & 0x80808080u) + __popc(a.y & 0x80808080u) + __popc(a.z & 0x80808080u) + __popc(a.w & 0x80808080u);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unequal += __shfl_xor_sync(0xFFFFFFFFu, unequal, o);
        negative += __shfl_xor_sync(0xFFFFFFFFu, negative, o);
    }
    if ((threadIdx.x & 31u) == 0u) {
        if (unequal) atomicAdd(acc + 2 * (size_t)r, unequal);
        if (negative) atomicAdd(acc + 2 * (size_t)r + 1, negative);
    }
}

// acc (unequal, negative) -> (E, M) per chain
__global__ void batch_finish_energy_kernel(unsigned long long *acc, long long *EM, uint32_t R, uint32_t N, int dim)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    EM[2 * r] = 2ll * (long long)acc[2 * r] - (long long)dim * (long long)N;
    EM[2 * r + 1] = (long long)N - 2ll * (long long)acc[2 * r + 1];
}

template <int DIM, bool POW2, bool BITS>
cudaError_t launch_one(const BatchParams &bp, int grid, int threads, size_t smem, cudaStream_t stream)
{
    // per-process kernel attribute: only ever raised to the device's maximum (internal.h)
    const cudaError_t e = allow_max_dynamic_smem(reinterpret_cast<const void *>(&growth_batch_kernel<DIM, POW2, BITS>));
    if (e != cudaSuccess) return e;
    growth_batch_kernel<DIM, POW2, BITS><<<grid, threads, smem, stream>>>(bp);
    return cudaGetLastError();
}

template <int DIM, bool POW2, bool BITS>
cudaError_t occupancy_one(int threads, size_t smem, int *per_sm)
{
    const cudaError_t e = allow_max_dynamic_smem(reinterpret_cast<const void *>(&growth_batch_kernel<DIM, POW2, BITS>));
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, growth_batch_kernel<DIM, POW2, BITS>, threads, smem);
}

}  // namespace

size_t batch_smem_bytes(uint32_t N, uint32_t qcap, bool bits, bool measure)
{
    size_t words = 2ull * qcap;
    if (bits) words += (size_t)((N + 31u) >> 5) * (measure ? 2u : 1u);
    return words * sizeof(uint32_t);
}

#define WOLFF_BATCH_DISPATCH(CALL)                                                   \
    do {                                                                            \
        if (dim == 2) {                                                             \
            if (pow2) return bits ? CALL(2, true, true) : CALL(2, true, false);     \
            return bits ? CALL(2, false, true) : CALL(2, false, false);             \
        }                                                                           \
        if (pow2) return bits ? CALL(3, true, true) : CALL(3, true, false);         \
        return bits ? CALL(3, false, true) : CALL(3, false, false);                 \
    } while (0)

cudaError_t launch_growth_batch(const BatchParams &bp, int dim, bool bits, int grid, int threads, cudaStream_t stream)
{
    const size_t smem = batch_smem_bytes(bp.geo.N, bp.qcap, bits, bp.measure != 0u);
    const bool pow2 = bp.geo.pow2 != 0u;
#define WOLFF_CALL(D, P, B) launch_one<D, P, B>(bp, grid, threads, smem, stream)
    WOLFF_BATCH_DISPATCH(WOLFF_CALL);
#undef WOLFF_CALL
}

cudaError_t batch_ctas_per_sm(int dim, bool pow2, bool bits, int threads, size_t smem, int *per_sm)
{
#define WOLFF_CALL(D, P, B) occupancy_one<D, P, B>(threads, smem, per_sm)
    WOLFF_BATCH_DISPATCH(WOLFF_CALL);
#undef WOLFF_CALL
}

cudaError_t launch_batch_energy(const int8_t *spins, size_t stride, const Geometry &geo, int dim, uint32_t R, unsigned long long *acc,
                                long long *EM, int num_sms, cudaStream_t stream)
{
    cudaError_t e = cudaMemsetAsync(acc, 0, 2 * (size_t)R * sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return e;
    if (geo.L % 16u == 0u && R <= 65535u) {
        // enough CTAs per chain to fill the chip whatever R is, at most one per 256 chunks
        uint32_t per_chain = (uint32_t)((8u * (uint32_t)num_sms + R - 1u) / R);
        const uint32_t most = (geo.N / 16u + 255u) / 256u;
        if (per_chain > most) per_chain = most;
        if (per_chain < 1u) per_chain = 1u;
        if (dim == 2) batch_energy_vec16_kernel<2><<<dim3(per_chain, R), 256, 0, stream>>>(spins, stride, geo, acc);
        else          batch_energy_vec16_kernel<3><<<dim3(per_chain, R), 256, 0, stream>>>(spins, stride, geo, acc);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        batch_finish_energy_kernel<<<(R + 127u) / 128u, 128, 0, stream>>>(acc, EM, R, geo.N, dim);
        return cudaGetLastError();
    }
    // enough CTAs to fill the chip whatever R is
    uint32_t slices = (uint32_t)((8u * (uint32_t)num_sms + R - 1u) / R);
    const uint32_t max_slices = (geo.N + 255u) / 256u;
    if (slices > max_slices) slices = max_slices;
    if (slices < 1u) slices = 1u;
    if (dim == 2) batch_energy_kernel<2><<<R * slices, 256, 0, stream>>>(spins, stride, geo, R, slices, acc);
    else          batch_energy_kernel<3><<<R * slices, 256, 0, stream>>>(spins, stride, geo, R, slices, acc);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    batch_finish_energy_kernel<<<(R + 127u) / 128u, 128, 0, stream>>>(acc, EM, R, geo.N, dim);
    return cudaGetLastError();
}

}  // namespace wolff
