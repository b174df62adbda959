// measure.cu -- whole-lattice kernels: start lattice, validation, and the E/M reduction (A8).
//
// E/M: "measurement of energy and magnetization" (Eq. 2 at PAPER.md:38).  In units
// of J, E = -sum_i sum_{d<dim} s_i s_{nbr(i,d,+)} and M = sum_i s_i (reading R13).  With +1 = 0x01
// and -1 = 0xFF the sign is bit 7 of the byte, so for 16 sites held in four 32-bit words
//   #negative  = popc(word & 0x80808080)
//   #unequal_d = popc((word ^ word_shifted_to_the_+d_neighbour) & 0x80808080)
// and E = 2 * #unequal - dim*N, M = N - 2 * #negative.  Integer only; bandwidth-bound: N bytes
// read once from HBM (forward rows/planes are re-read through L2).
#include "internal.h"

namespace wolff {

namespace {

constexpr int kThreads = 256;
constexpr uint32_t kSignMask = 0x80808080u;

// ---------------------------------------------------------------- start lattice (reading R9)
// Site i takes bit (i mod 128) of Philox(key = seed, ctr = (i div 128, INIT, 0, 0)): bit (i mod 32)
// of word ((i div 32) mod 4); 1 -> +1, 0 -> -1.  One thread writes 16 sites (one 16-byte store).
__device__ __forceinline__ uint32_t expand4(uint32_t bits4)
{
    // bits4: 4 low bits -> 4 bytes, bit set -> 0x01 (+1), clear -> 0xFF (-1)
    uint32_t w = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) w |= (((bits4 >> k) & 1u) ? 0x01u : 0xFFu) << (8 * k);
    return w;
}

__global__ void __launch_bounds__(kThreads) init_lattice_kernel(int8_t *spins, uint32_t N, uint32_t key0, uint32_t key1)
{
    const uint32_t chunks = (N + 15u) / 16u;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < chunks; c += gridDim.x * blockDim.x) {
        const uint32_t i = c * 16u;                 // first site of the chunk (N <= 2^31: no overflow)
        const uint4 x = philox4x32_10(i >> 7, kDomainInit, 0u, 0u, key0, key1);
        const uint32_t word = word_of(x, (int)((i >> 5) & 3u));
        const uint32_t bits = (word >> (i & 31u)) & 0xFFFFu;
        if (i + 16u <= N) {
            uint4 out;
            out.x = expand4(bits);
            out.y = expand4(bits >> 4);
            out.z = expand4(bits >> 8);
            out.w = expand4(bits >> 12);
            *reinterpret_cast<uint4 *>(spins + i) = out;
        } else {
            for (uint32_t k = 0; i + k < N; ++k) spins[i + k] = ((bits >> k) & 1u) ? (int8_t)1 : (int8_t)-1;
        }
    }
}

// ---------------------------------------------------------------- set_spins validation
__global__ void __launch_bounds__(kThreads) validate_kernel(const int8_t *spins, uint32_t N, Control *ctl)
{
    bool bad = false;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        const int8_t s = spins[i];
        bad |= (s != 1 && s != -1);
    }
    if (__any_sync(0xFFFFFFFFu, bad) && (threadIdx.x & 31) == 0) atomicOr(&ctl->invalid, 1u);
}

// ---------------------------------------------------------------- E / M reduction
__device__ __forceinline__ void block_accumulate(unsigned long long unequal, unsigned long long negative, Control *ctl,
                                                 uint32_t N, int dim)
{
    __shared__ unsigned long long s_un[kThreads / 32], s_ng[kThreads / 32];
    __shared__ bool last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unequal += __shfl_xor_sync(0xFFFFFFFFu, unequal, o);
        negative += __shfl_xor_sync(0xFFFFFFFFu, negative, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s_un[warp] = unequal; s_ng[warp] = negative; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long un = 0, ng = 0;
        for (int w = 0; w < kThreads / 32; ++w) { un += s_un[w]; ng += s_ng[w]; }
        if (un) atomicAdd(&ctl->acc_unequal, un);
        if (ng) atomicAdd(&ctl->acc_negative, ng);
        __threadfence();
        const unsigned int t = atomicAdd(&ctl->ticket, 1u);
        last = (t == gridDim.x - 1u);
        if (last) {
            // every other CTA's contribution is visible: its fence preceded its ticket
            __threadfence();
            const unsigned long long tun = atomicAdd(&ctl->acc_unequal, 0ull);
            const unsigned long long tng = atomicAdd(&ctl->acc_negative, 0ull);
            ctl->E = 2ll * (long long)tun - (long long)dim * (long long)N;
            ctl->M = (long long)N - 2ll * (long long)tng;
            ctl->acc_unequal = 0ull;
            ctl->acc_negative = 0ull;
            ctl->ticket = 0u;
        }
    }
}

// Vector path: L is a multiple of 16, so a 16-byte chunk never straddles a row.
template <int DIM>
__global__ void __launch_bounds__(kThreads) energy_magnetisation_vec16(const int8_t *__restrict__ spins, Geometry g, Control *ctl)
{
    const uint32_t chunks = g.N / 16u;
    const uint32_t chunks_per_row = g.L / 16u;
    unsigned long long unequal = 0, negative = 0;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < chunks; c += gridDim.x * blockDim.x) {
        const uint32_t i = c * 16u;
        const uint32_t row = c / chunks_per_row;          // y + L*z
        const uint32_t cx = c - row * chunks_per_row;     // chunk index along x
        const uint32_t y = (DIM == 3) ? row % g.L : row;
        const uint4 a = *reinterpret_cast<const uint4 *>(spins + i);
        // +x: the 16 sites shifted by one byte; the 17th byte is the first site of the next chunk (wrapping)
        const uint32_t inext = (cx + 1u == chunks_per_row) ? i + 16u - g.L : i + 16u;
        const uint32_t nb = (uint32_t)(uint8_t)spins[inext];
        uint32_t acc = 0, neg = 0;
        acc += __popc((a.x ^ __funnelshift_r(a.x, a.y, 8)) & kSignMask);
        acc += __popc((a.y ^ __funnelshift_r(a.y, a.z, 8)) & kSignMask);
        acc += __popc((a.z ^ __funnelshift_r(a.z, a.w, 8)) & kSignMask);
        acc += __popc((a.w ^ __funnelshift_r(a.w, nb, 8)) & kSignMask);
        neg += __popc(a.x & kSignMask) + __popc(a.y & kSignMask) + __popc(a.z & kSignMask) + __popc(a.w & kSignMask);
        // +y
        const uint32_t iy = (y + 1u == g.L) ? i - (g.LL - g.L) : i + g.L;
        const uint4 by = *reinterpret_cast<const uint4 *>(spins + iy);
        acc += __popc((a.x ^ by.x) & kSignMask) + __popc((a.y ^ by.y) & kSignMask) +
               __popc((a.z ^ by.z) & kSignMask) + __popc((a.w ^ by.w) & kSignMask);
        if (DIM == 3) {
            const uint32_t z = row / g.L;
            const uint32_t iz = (z + 1u == g.L) ? i - (g.N - g.LL) : i + g.LL;
            const uint4 bz = *reinterpret_cast<const uint4 *>(spins + iz);
            acc += __popc((a.x ^ bz.x) & kSignMask) + __popc((a.y ^ bz.y) & kSignMask) +
                   __popc((a.z ^ bz.z) & kSignMask) + __popc((a.w ^ bz.w) & kSignMask);
        }
        unequal += acc;
        negative += neg;
    }
    block_accumulate(unequal, negative, ctl, g.N, DIM);
}

// Generic path: any L >= 2, one site per thread iteration.
template <int DIM>
__global__ void __launch_bounds__(kThreads) energy_magnetisation_scalar(const int8_t *__restrict__ spins, Geometry g, Control *ctl)
{
    unsigned long long unequal = 0, negative = 0;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < g.N; i += gridDim.x * blockDim.x) {
        uint32_t nbr[2 * DIM];
        neighbours<DIM, false>(g, i, nbr);
        const int s = spins[i];
        negative += (s < 0);
#pragma unroll
        for (int d = 0; d < DIM; ++d) unequal += (spins[nbr[2 * d]] != s);
    }
    block_accumulate(unequal, negative, ctl, g.N, DIM);
}

inline int grid_for(uint64_t items, int num_sms, int per_sm)
{
    uint64_t blocks = (items + kThreads - 1) / kThreads;
    const uint64_t cap = (uint64_t)num_sms * (uint64_t)per_sm;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    return (int)blocks;
}

}  // namespace

cudaError_t launch_init_lattice(int8_t *spins, uint32_t N, uint64_t seed, cudaStream_t stream)
{
    const int grid = grid_for((N + 15u) / 16u, 148, 8);
    init_lattice_kernel<<<grid, kThreads, 0, stream>>>(spins, N, (uint32_t)seed, (uint32_t)(seed >> 32));
    return cudaGetLastError();
}

cudaError_t launch_validate(const int8_t *spins, uint32_t N, Control *ctl, cudaStream_t stream)
{
    const int grid = grid_for(N, 148, 8);
    validate_kernel<<<grid, kThreads, 0, stream>>>(spins, N, ctl);
    return cudaGetLastError();
}

cudaError_t launch_energy_magnetisation(const int8_t *spins, const Geometry &geo, int dim, Control *ctl, int num_sms,
                                        cudaStream_t stream)
{
    if (geo.L % 16u == 0u) {
        // one wave: every SM holds up to 8 CTAs of 256 threads
        const int grid = grid_for(geo.N / 16u, num_sms, 8);
        if (dim == 2) energy_magnetisation_vec16<2><<<grid, kThreads, 0, stream>>>(spins, geo, ctl);
        else          energy_magnetisation_vec16<3><<<grid, kThreads, 0, stream>>>(spins, geo, ctl);
    } else {
        const int grid = grid_for(geo.N, num_sms, 8);
        if (dim == 2) energy_magnetisation_scalar<2><<<grid, kThreads, 0, stream>>>(spins, geo, ctl);
        else          energy_magnetisation_scalar<3><<<grid, kThreads, 0, stream>>>(spins, geo, ctl);
    }
    return cudaGetLastError();
}

}  // namespace wolff
