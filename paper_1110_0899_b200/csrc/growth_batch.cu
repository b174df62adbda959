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
// In-kernel measurement ("measure" = 1) as in growth.cu: members of the running cluster carry a mark (bit 1 of the
// byte), dE = 2 * sum over the cluster's boundary bonds, dM = -2 s0 |C|, running from a whole-lattice evaluation
// the host queues before the launch.
#include "expand.cuh"
#include "internal.h"

namespace wolff {
namespace {

struct BatchShared {
    unsigned int cnt[3];       // rotating level counters (entries appended to the list by the running level)
    unsigned int chain;        // the chain this CTA works on
    int s0;
    unsigned long long post_acc;
};

template <int DIM, bool POW2>
__global__ void __launch_bounds__(kBatchMaxThreads) growth_batch_kernel(const BatchParams bp)
{
    extern __shared__ __align__(16) uint32_t smem_bq[];          // two frontier buffers of bp.qcap entries
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

        for (unsigned long long k = 0; k < bp.n_updates; ++k) {
            const unsigned long long u = bp.u0 + k;
            const uint32_t u_lo = (uint32_t)u, u_hi = (uint32_t)(u >> 32);
            // A1: seed draw (reading R8) and initial flip
            if (tid == 0) {
                const uint4 x = philox4x32_10(0u, kDomainSite, u_lo, u_hi, p.key0, p.key1);
                const unsigned long long rr = (unsigned long long)x.x | ((unsigned long long)x.y << 32);
                const uint32_t i0 = (uint32_t)__umul64hi(rr, (unsigned long long)p.geo.N);
                const int s = load_spin_l2(p.spins, i0);
                claim_with_bits(p.spins, i0, s, p.claim_bits);
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
                    claim_neighbours<DIM, POW2, false>(p, s0, u_lo, u_hi, valid, site, nbr, won, x, y, z, attempts);
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
                int part = boundary_partial<DIM, POW2>(p.geo, p.spins, p.clist, s0, size, tid, T);
                part = __reduce_add_sync(kFullMask, part);
                if (lane == 0u && part != 0) atomicAdd(&sh.post_acc, (unsigned long long)(long long)part);
                __syncthreads();
                const int8_t plain = (int8_t)(-s0);
                for (uint32_t e = tid; e < size; e += T) p.spins[__ldcg(p.clist + e)] = plain;
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

// acc (unequal, negative) -> (E, M) per chain
__global__ void batch_finish_energy_kernel(unsigned long long *acc, long long *EM, uint32_t R, uint32_t N, int dim)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    EM[2 * r] = 2ll * (long long)acc[2 * r] - (long long)dim * (long long)N;
    EM[2 * r + 1] = (long long)N - 2ll * (long long)acc[2 * r + 1];
}

template <int DIM, bool POW2>
cudaError_t launch_one(const BatchParams &bp, int grid, int threads, size_t smem, cudaStream_t stream)
{
    growth_batch_kernel<DIM, POW2><<<grid, threads, smem, stream>>>(bp);
    return cudaGetLastError();
}

template <int DIM, bool POW2>
cudaError_t occupancy_one(int threads, size_t smem, int *per_sm)
{
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, growth_batch_kernel<DIM, POW2>, threads, smem);
}

}  // namespace

cudaError_t launch_growth_batch(const BatchParams &bp, int dim, int grid, int threads, cudaStream_t stream)
{
    const size_t smem = 2ull * bp.qcap * sizeof(uint32_t);
    const bool pow2 = bp.geo.pow2 != 0u;
    if (dim == 2) return pow2 ? launch_one<2, true>(bp, grid, threads, smem, stream) : launch_one<2, false>(bp, grid, threads, smem, stream);
    return pow2 ? launch_one<3, true>(bp, grid, threads, smem, stream) : launch_one<3, false>(bp, grid, threads, smem, stream);
}

cudaError_t batch_ctas_per_sm(int dim, bool pow2, int threads, uint32_t qcap, int *per_sm)
{
    const size_t smem = 2ull * qcap * sizeof(uint32_t);
    if (dim == 2) return pow2 ? occupancy_one<2, true>(threads, smem, per_sm) : occupancy_one<2, false>(threads, smem, per_sm);
    return pow2 ? occupancy_one<3, true>(threads, smem, per_sm) : occupancy_one<3, false>(threads, smem, per_sm);
}

cudaError_t launch_batch_energy(const int8_t *spins, size_t stride, const Geometry &geo, int dim, uint32_t R, unsigned long long *acc,
                                long long *EM, int num_sms, cudaStream_t stream)
{
    cudaError_t e = cudaMemsetAsync(acc, 0, 2 * (size_t)R * sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return e;
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
