// expand.cuh -- expansion of one cluster site per lane for the level-synchronous
// kernel (growth.cu).  growth_tiles.cu includes it for kFullMask only: its pass is written per bond, not per site.
//
// PAPER.md:45-46 (steps ii/iii): every neighbour of a newly added spin that is parallel to the seed
// spin and not yet a member joins with probability p = 1 - exp(-2J/T).  Here the random number of a
// bond is a function of (seed, update, bond) (readings R6, R10), and "join" is one atomic that flips
// the spin (reading R3), so the order in which sites are expanded cannot show in the result.
#pragma once
#include "internal.h"

namespace wolff {

constexpr unsigned int kFullMask = 0xFFFFFFFFu;

// A2-A4 for one site per lane.  On return nbr[] holds the 2*DIM neighbour ids, bit k of `won` is set
// when THIS lane flipped nbr[k] from s0 to -s0 (so nbr[k] is a new member of the cluster), and
// (x, y, z) are the site's coordinates.  Lanes with valid == false do nothing and return won = 0.
//
// SPEC == false: gather the neighbour spins first (A2, ld.global.cg, in flight while the Philox rounds
//   execute) and issue the claim atomic only for same-sign neighbours behind active bonds.
// SPEC == true: no gather.  The claim atomic is idempotent on a spin that is not s0 (OR 0xFE on 0xFF,
//   AND 0x01.. on 0x01 change nothing) and returns the old byte, so it is issued for every active bond
//   and the returned byte says whether the neighbour was parallel: the dependent chain of one hop
//   loses the L2 load (about 2*dim*p atomics per site instead of about 1.1, on an idle atomic unit).
template <int DIM, bool POW2, bool SPEC>
__device__ __forceinline__ void claim_neighbours(const GrowthParams &p, int s0, uint32_t u_lo, uint32_t u_hi, bool valid,
                                                 uint32_t i, uint32_t (&nbr)[2 * DIM], unsigned int &won, uint32_t &x,
                                                 uint32_t &y, uint32_t &z, unsigned int &attempts)
{
    bool cand[2 * DIM];
    unsigned int old[2 * DIM];
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) { nbr[k] = 0u; cand[k] = false; old[k] = 0u; }
    x = y = z = 0u;
    won = 0u;

    if (valid) {
        site_coords<DIM, POW2>(p.geo, i, x, y, z);
        neighbours_at<DIM>(p.geo, i, x, y, z, nbr);
        int sp[2 * DIM];
        if (!SPEC) {
#pragma unroll
            for (int k = 0; k < 2 * DIM; ++k) sp[k] = load_spin_l2(p.spins, nbr[k]);
        }
        // A3: the bond to the +d neighbour is owned by this site (word d of the site's block); the bond
        // to the -d neighbour is owned by that neighbour (word d of ITS block).  The 1 + DIM blocks are
        // independent chains and run with their rounds interleaved.
        uint32_t ctr0[1 + DIM];
        uint4 blk[1 + DIM];
        ctr0[0] = i;
#pragma unroll
        for (int d = 0; d < DIM; ++d) ctr0[1 + d] = nbr[2 * d + 1];
        philox4x32_10_multi<1 + DIM>(ctr0, kDomainBond, u_lo, u_hi, p.key0, p.key1, blk);
#pragma unroll
        for (int d = 0; d < DIM; ++d) {
            cand[2 * d] = (unsigned long long)word_of(blk[0], d) < p.thr;
            cand[2 * d + 1] = (unsigned long long)word_of(blk[1 + d], d) < p.thr;
            if (!SPEC) {
                cand[2 * d] = cand[2 * d] && (sp[2 * d] == s0);
                cand[2 * d + 1] = cand[2 * d + 1] && (sp[2 * d + 1] == s0);
            }
        }
    }

    // A4: all atomics of a lane are issued before any result is looked at, so their L2 round trips overlap.
    unsigned int *const words = reinterpret_cast<unsigned int *>(p.spins);
    if (s0 > 0) {   // uniform for the whole update
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k)
            if (cand[k]) old[k] = atomicOr(words + (nbr[k] >> 2), p.claim_bits << ((nbr[k] & 3u) * 8u));
    } else {
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k)
            if (cand[k]) old[k] = atomicAnd(words + (nbr[k] >> 2), ~(p.claim_bits << ((nbr[k] & 3u) * 8u)));
    }
    const unsigned int s0_byte = (unsigned int)s0 & 0xFFu;
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) {
        const bool w = cand[k] && (((old[k] >> ((nbr[k] & 3u) * 8u)) & 0xFFu) == s0_byte);
        attempts += cand[k] ? 1u : 0u;
        won |= w ? (1u << k) : 0u;
    }
}

// Post-pass of a measured update (in-kernel measurement, growth.cu / growth_batch.cu): this thread's share of
//   sum over members i, over the 2*DIM bonds (i, j) with j NOT a member, of (+1 if s_j == s0 else -1)
// for the members list[first], list[first + step], ... below `size`.  Flipping the cluster changes exactly the
// bonds between a member and a non-member, from -s0*s_j to +s0*s_j, so dE = 2 * (that sum) in units of J.  Called
// after the cluster is complete and before the marks are removed: members read 0xFD / 0x03 (claim_with_bits).
template <int DIM, bool POW2>
__device__ __forceinline__ int boundary_partial(const Geometry &geo, const int8_t *spins, const uint32_t *list, int s0,
                                                uint32_t size, uint32_t first, uint32_t step)
{
    int acc = 0;
    const unsigned int want_negative = s0 < 0 ? 1u : 0u;
    for (uint32_t e = first; e < size; e += step) {
        const uint32_t i = __ldcg(list + e);
        uint32_t x, y, z, nbr[2 * DIM];
        site_coords<DIM, POW2>(geo, i, x, y, z);
        neighbours_at<DIM>(geo, i, x, y, z, nbr);
        unsigned int b[2 * DIM];
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) b[k] = (unsigned int)__ldcg(reinterpret_cast<const unsigned char *>(spins) + nbr[k]);
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k)
            if (!is_marked_member(b[k])) acc += ((b[k] >> 7) == want_negative) ? 1 : -1;
    }
    return acc;
}

// A2-A5 for one site per lane: claim_neighbours, then append the winners to dst[] with ONE atomic per
// warp on *dst_count (ballot/popc aggregation).  Must be called by all 32 lanes of a warp.
template <int DIM, bool POW2, bool SPEC>
__device__ __forceinline__ void expand_sites(const GrowthParams &p, int s0, uint32_t u_lo, uint32_t u_hi, bool valid,
                                             uint32_t i, uint32_t *dst, unsigned int *dst_count, uint32_t dst_cap, unsigned int &attempts)
{
    (void)dst_cap;       // entries dst[] can hold: looked at by checked builds only
    uint32_t nbr[2 * DIM];
    unsigned int won;
    uint32_t x, y, z;
    claim_neighbours<DIM, POW2, SPEC>(p, s0, u_lo, u_hi, valid, i, nbr, won, x, y, z, attempts);
    unsigned int ballots[2 * DIM];
    unsigned int total = 0;
#pragma unroll
    for (int k = 0; k < 2 * DIM; ++k) {
        ballots[k] = __ballot_sync(kFullMask, (won >> k) & 1u);
        total += __popc(ballots[k]);
    }
    if (total != 0u) {   // warp-uniform
        const unsigned int lane = threadIdx.x & 31u;
        unsigned int base = 0;
        if (lane == 0u) base = atomicAdd(dst_count, total);
        base = __shfl_sync(kFullMask, base, 0);
        const unsigned int bit = 1u << lane;
        const unsigned int lt = bit - 1u;
#pragma unroll
        for (int k = 0; k < 2 * DIM; ++k) {
            if ((ballots[k] & bit) && WOLFF_CHECK(&p.ctl->error, base + __popc(ballots[k] & lt) < dst_cap && nbr[k] < p.geo.N, 20))
                dst[base + __popc(ballots[k] & lt)] = nbr[k];
            base += __popc(ballots[k]);
        }
    }
}

}  // namespace wolff
