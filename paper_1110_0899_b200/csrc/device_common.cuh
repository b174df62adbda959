// device_common.cuh -- device-side building blocks shared by the kernels of libwolff_b200.
//
// Nothing here is shared with oracle/: the oracle has its own plain-C statement of the same
// definitions (readings R5-R11).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace wolff {

// ---------------------------------------------------------------- checked builds
// -DWOLFF_CHECKED: every index the growth kernels compute for a queue, a list, a tile or a bit plane is compared with
// its bound before it is used; a violation stores 1000 + code into the error word (the handle then reports
// WOLFF_EINTERNAL with that code) and the access is skipped.  compute-sanitizer is closed on the pool this library was
// developed on, so this is the memory check that can be run there (profiles/ holds the summary of such a run); the
// release build contains none of it.
#ifdef WOLFF_CHECKED
__device__ __forceinline__ bool wolff_check_failed(void *errword, unsigned int code)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(errword), "r"(1000u + code) : "memory");
    return false;
}
#define WOLFF_CHECK(errword, cond, code) ((cond) ? true : wolff::wolff_check_failed((void *)(errword), (unsigned int)(code)))
#else
#define WOLFF_CHECK(errword, cond, code) (true)
#endif

// ---------------------------------------------------------------- schedule-perturbing builds
// -DWOLFF_JITTER: the lock-free protocols of the growth kernels (ring reserve / put / take, inbox slot / message,
// pending counts and publishing, work stealing, termination) are correct for every interleaving of their steps, not
// only for the ones the hardware usually produces.  This build makes unusual interleavings common: at every marked
// point between two steps of a protocol a thread sleeps, one time in four, for a pseudo-random 0-2 microseconds
// (thousands of cycles: longer than any of the protocol's round trips).  With compute-sanitizer's racecheck closed on
// the development pool, running the parity cases on this build is the race test that can be run there
// (tests/test_gpu_checked.py, profiles/r2_checked_build.md); the release build contains none of it.
#ifdef WOLFF_JITTER
__device__ __forceinline__ void wolff_jitter(unsigned int id)
{
    unsigned int t;
    asm volatile("mov.u32 %0, %%clock;" : "=r"(t));
    unsigned int h = t ^ (id * 0x9E3779B9u) ^ (threadIdx.x * 0x85EBCA6Bu) ^ (blockIdx.x * 0xC2B2AE35u);
    h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12;
    if ((h & 3u) == 0u) __nanosleep(h >> 21);
}
#define WOLFF_JITTER_POINT(id) wolff::wolff_jitter((unsigned int)(id))
#else
#define WOLFF_JITTER_POINT(id) ((void)0)
#endif

// ---------------------------------------------------------------- Philox4x32-10 (reading R11)
// Salmon et al., SC'11.  One round maps (c0,c1,c2,c3) to
// (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)); the key is bumped by the Weyl
// constants between rounds.  Written as two 32x32->64 multiplies per round (IMAD.WIDE.U32).
constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

// Domain tags (bits 31:30 of counter word 1) keep the three streams disjoint (reading R10).
constexpr uint32_t kDomainBond = 0u << 30;
constexpr uint32_t kDomainSite = 1u << 30;
constexpr uint32_t kDomainInit = 2u << 30;

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// K independent blocks with the rounds interleaved: the ten rounds of one block form a dependent
// chain (IMAD.WIDE -> LOP3 -> IMAD.WIDE ...), so running K chains side by side costs about the
// latency of one.  All blocks share counter words 1..3 and the key; only word 0 differs.
template <int K>
__device__ __forceinline__ void philox4x32_10_multi(const uint32_t (&ctr0)[K], uint32_t c1_, uint32_t c2_, uint32_t c3_,
                                                    uint32_t k0, uint32_t k1, uint4 (&out)[K])
{
    uint32_t c0[K], c1[K], c2[K], c3[K];
#pragma unroll
    for (int j = 0; j < K; ++j) { c0[j] = ctr0[j]; c1[j] = c1_; c2[j] = c2_; c3[j] = c3_; }
#pragma unroll
    for (int round = 0; round < 10; ++round) {
#pragma unroll
        for (int j = 0; j < K; ++j) {
            const uint64_t p0 = (uint64_t)kPhiloxM0 * (uint64_t)c0[j];
            const uint64_t p1 = (uint64_t)kPhiloxM1 * (uint64_t)c2[j];
            const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1[j] ^ k0;
            const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3[j] ^ k1;
            c1[j] = (uint32_t)p1;
            c3[j] = (uint32_t)p0;
            c0[j] = n0;
            c2[j] = n2;
        }
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
#pragma unroll
    for (int j = 0; j < K; ++j) out[j] = make_uint4(c0[j], c1[j], c2[j], c3[j]);
}

__device__ __forceinline__ uint32_t word_of(const uint4 &v, int d)
{
    return d == 0 ? v.x : (d == 1 ? v.y : (d == 2 ? v.z : v.w));
}

// ---------------------------------------------------------------- lattice geometry (reading R5)
// Site id i = x + L*y (+ L*L*z).  nbr[2d] is the +d neighbour, nbr[2d+1] the -d neighbour,
// coordinates wrap periodically.
struct Geometry {
    uint32_t L;      // linear size
    uint32_t N;      // L^dim   (N <= 2^31)
    uint32_t LL;     // L*L
    uint32_t logL;   // log2 L when L is a power of two, else 0
    uint32_t pow2;   // 1 when L is a power of two
};

// Coordinates of site i (reading R5).
template <int DIM, bool POW2>
__device__ __forceinline__ void site_coords(const Geometry &g, uint32_t i, uint32_t &x, uint32_t &y, uint32_t &z)
{
    z = 0;
    if (POW2) {
        const uint32_t mask = g.L - 1u;
        x = i & mask;
        y = (i >> g.logL) & mask;
        if (DIM == 3) z = i >> (2u * g.logL);
    } else {
        x = i % g.L;
        const uint32_t t = i / g.L;
        y = t % g.L;
        if (DIM == 3) z = t / g.L;
    }
}

// nbr[2d] = +d neighbour, nbr[2d+1] = -d neighbour of site i at (x, y, z), periodic.
template <int DIM>
__device__ __forceinline__ void neighbours_at(const Geometry &g, uint32_t i, uint32_t x, uint32_t y, uint32_t z,
                                              uint32_t (&nbr)[2 * DIM])
{
    const uint32_t Lm1 = g.L - 1u;
    nbr[0] = (x == Lm1) ? i - Lm1 : i + 1u;
    nbr[1] = (x == 0u) ? i + Lm1 : i - 1u;
    const uint32_t ywrap = g.LL - g.L;                 // L*(L-1)
    nbr[2] = (y == Lm1) ? i - ywrap : i + g.L;
    nbr[3] = (y == 0u) ? i + ywrap : i - g.L;
    if (DIM == 3) {
        const uint32_t zwrap = g.N - g.LL;             // L*L*(L-1)
        nbr[4] = (z == Lm1) ? i - zwrap : i + g.LL;
        nbr[5] = (z == 0u) ? i + zwrap : i - g.LL;
    }
}

template <int DIM, bool POW2>
__device__ __forceinline__ void neighbours(const Geometry &g, uint32_t i, uint32_t (&nbr)[2 * DIM])
{
    uint32_t x, y, z;
    site_coords<DIM, POW2>(g, i, x, y, z);
    neighbours_at<DIM>(g, i, x, y, z, nbr);
}

// ---------------------------------------------------------------- spins
// int8 storage, +1 = 0x01, -1 = 0xFF.  All lattice reads in the growth kernel bypass L1
// (ld.global.cg): the kernel is persistent across updates, and an L1 line cached during an
// earlier update could show a spin with its old sign.
__device__ __forceinline__ int load_spin_l2(const int8_t *spins, uint32_t i)
{
    return (int)__ldcg(reinterpret_cast<const signed char *>(spins) + i);
}

// Claim-and-flip: one atomic on the 32-bit word containing byte j that
// sets the byte to -s0 and returns whether THIS thread changed it from s0.  CUDA has no 8-bit
// CAS; with +1 = 0x01 and -1 = 0xFF the transition s0 -> -s0 is an idempotent bit operation
// (OR 0xFE for +1 -> -1, AND 0x01 for -1 -> +1), so a single atom.or / atom.and has exactly
// the semantics of CAS(s0 -> -s0) and never needs a retry when a sibling byte changes.
__device__ __forceinline__ bool claim_and_flip(int8_t *spins, uint32_t j, int s0)
{
    unsigned int *word = reinterpret_cast<unsigned int *>(spins) + (j >> 2);
    const unsigned int shift = (j & 3u) * 8u;
    unsigned int old;
    if (s0 > 0) old = atomicOr(word, 0xFEu << shift);
    else        old = atomicAnd(word, ~(0xFEu << shift));
    return ((old >> shift) & 0xFFu) == ((unsigned int)s0 & 0xFFu);
}

// Claim with an explicit bit pattern (in-kernel measurement, growth.cu / growth_batch.cu): claim_bits = 0xFE is
// claim_and_flip(); claim_bits = 0xFC leaves bit 1 as it was, so a spin claimed in the RUNNING update reads 0xFD
// (was +1, now -1) or 0x03 (was -1, now +1): its sign (bit 7) is already the new one, and bit 1 != bit 7 marks it as
// a member of the running cluster -- the role of the flag the paper packs into the spin word -- until
// the update's post-pass has counted the cluster's boundary bonds and stored the plain value.
__device__ __forceinline__ bool claim_with_bits(int8_t *spins, uint32_t j, int s0, unsigned int claim_bits)
{
    unsigned int *word = reinterpret_cast<unsigned int *>(spins) + (j >> 2);
    const unsigned int shift = (j & 3u) * 8u;
    unsigned int old;
    if (s0 > 0) old = atomicOr(word, claim_bits << shift);
    else        old = atomicAnd(word, ~(claim_bits << shift));
    return ((old >> shift) & 0xFFu) == ((unsigned int)s0 & 0xFFu);
}
__device__ __forceinline__ bool is_marked_member(unsigned int byte) { return (((byte >> 1) ^ (byte >> 7)) & 1u) != 0u; }

// ---------------------------------------------------------------- measurement (Eq. 3)
// Accumulated sums of the measured series, ten 64-bit words (layout of wolff_get_moments):
// [0] n  [1] sum E  [2] sum |M|  [3..4] sum E^2  [5..6] sum M^2  [7..8] sum M^4 (low, high)  [9] reserved.
// M^4 reaches 2^96 at N = 2^24, so the even moments are exact 128-bit integers.
struct Moments {
    unsigned long long n = 0, sum_absM = 0;
    long long sum_E = 0;
    unsigned __int128 sum_E2 = 0, sum_M2 = 0, sum_M4 = 0;

    __device__ __forceinline__ void load(const unsigned long long *w)
    {
        n = w[0]; sum_E = (long long)w[1]; sum_absM = w[2];
        sum_E2 = ((unsigned __int128)w[4] << 64) | w[3];
        sum_M2 = ((unsigned __int128)w[6] << 64) | w[5];
        sum_M4 = ((unsigned __int128)w[8] << 64) | w[7];
    }
    __device__ __forceinline__ void store(unsigned long long *w) const
    {
        w[0] = n; w[1] = (unsigned long long)sum_E; w[2] = sum_absM;
        w[3] = (unsigned long long)sum_E2; w[4] = (unsigned long long)(sum_E2 >> 64);
        w[5] = (unsigned long long)sum_M2; w[6] = (unsigned long long)(sum_M2 >> 64);
        w[7] = (unsigned long long)sum_M4; w[8] = (unsigned long long)(sum_M4 >> 64);
        w[9] = 0ull;
    }
    __device__ __forceinline__ void add(long long E, long long M)
    {
        const unsigned long long aM = (unsigned long long)(M < 0 ? -M : M), aE = (unsigned long long)(E < 0 ? -E : E);
        const unsigned __int128 m2 = (unsigned __int128)aM * aM;
        n += 1ull;
        sum_E += E;
        sum_absM += aM;
        sum_E2 += (unsigned __int128)aE * aE;
        sum_M2 += m2;
        sum_M4 += m2 * m2;
    }
};

// ---------------------------------------------------------------- inter-CTA synchronisation words
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned int atom_add_acq_rel_u32(unsigned int *p, unsigned int v)
{
    unsigned int old;
    asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int *p)
{
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_u32(unsigned int *p, unsigned int v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

}  // namespace wolff
