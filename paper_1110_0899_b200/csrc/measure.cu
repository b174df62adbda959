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
// A word of four spins is valid when every byte is 0x01 or 0xFF: with s = the four sign bits, the only valid word
// is 0x01010101 | s * 0xFE.  16 bytes per load (the staging buffer is 16-byte aligned and padded), bytes beyond N
// are not looked at.
__device__ __forceinline__ bool word_valid(uint32_t w)
{
    const uint32_t s = (w >> 7) & 0x01010101u;
    return w == (0x01010101u | (s * 0xFEu));
}

__global__ void __launch_bounds__(kThreads) validate_kernel(const int8_t *spins, size_t N, unsigned int *invalid)
{
    bool bad = false;
    const size_t chunks = N / 16u;
    const uint4 *const v = reinterpret_cast<const uint4 *>(spins);
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < chunks; c += (size_t)gridDim.x * blockDim.x) {
        const uint4 a = v[c];
        bad |= !(word_valid(a.x) && word_valid(a.y) && word_valid(a.z) && word_valid(a.w));
    }
    if (blockIdx.x == 0 && threadIdx.x < (N & 15u)) {            // ragged tail, at most 15 bytes
        const int8_t b = spins[chunks * 16u + threadIdx.x];
        bad |= (b != 1 && b != -1);
    }
    if (__any_sync(0xFFFFFFFFu, bad) && (threadIdx.x & 31) == 0) atomicOr(invalid, 1u);
}

// ---------------------------------------------------------------- E / M reduction
__device__ __forceinline__ void block_accumulate(unsigned long long unequal, unsigned long long negative, Control *ctl,
                                                 uint32_t N, int dim, long long *E_dst, long long *M_dst)
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
        // one atomic per CTA on one word: #unequal (at most dim * N < 2^33) in the low 33 bits, #negative (at most N <= 2^31)
        // above them.  Hundreds of CTAs finish within a microsecond of each other and their atomics on one address are
        // served one after the other, so every atomic saved is time off the kernel's tail.
        atomicAdd(&ctl->acc_unequal, un | (ng << 33));
        __threadfence();
        const unsigned int t = atomicAdd(&ctl->ticket, 1u);
        last = (t == gridDim.x - 1u);
        if (last) {
            // every other CTA's contribution is visible: its fence preceded its ticket
            __threadfence();
            const unsigned long long packed = atomicAdd(&ctl->acc_unequal, 0ull);
            const unsigned long long tun = packed & ((1ull << 33) - 1ull), tng = packed >> 33;
            const long long Ev = 2ll * (long long)tun - (long long)dim * (long long)N;
            const long long Mv = (long long)N - 2ll * (long long)tng;
            ctl->E = Ev;
            ctl->M = Mv;
            if (E_dst) *E_dst = Ev;          // the caller's device words: no bounce through the host
            if (M_dst) *M_dst = Mv;
            ctl->acc_unequal = 0ull;
            ctl->ticket = 0u;
        }
    }
}

// Vector path: L is a multiple of 16, so a 16-byte chunk never straddles a row.  A thread takes kU chunks per
// iteration and issues all their loads (the chunk, its +y and +z neighbours, the byte that follows it) before it
// uses any: the kernel is a few microseconds long, so what it needs is bytes in flight.
constexpr int kU = 4;

// Sign bits of four words in one word: they sit at bits 7, 15, 23, 31, so word j shifted right by j lands on bit 7 - j of
// every byte; two such merges (the second shifted by 4) give eight words per population count (POPC runs at a quarter
// of the ALU rate).
__device__ __forceinline__ uint32_t merge4(uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    return (a & kSignMask) | ((b & kSignMask) >> 1) | ((c & kSignMask) >> 2) | ((d & kSignMask) >> 3);
}

// POW2: L is a power of two (>= 16), so the chunk's row and its position in the row are a shift and a mask instead of two
// integer divisions per chunk and a third for z (profiles/r3_a8.md: at 1 GiB the divisions made the kernel issue-bound,
// sm throughput 68 %, DRAM 35 %).
template <int DIM, bool POW2>
__global__ void __launch_bounds__(kThreads) energy_magnetisation_vec16(const int8_t *__restrict__ spins, Geometry g, Control *ctl,
                                                                       long long *E_dst, long long *M_dst)
{
    const uint32_t chunks = g.N / 16u;
    const uint32_t chunks_per_row = g.L / 16u;
    const uint32_t row_shift = POW2 ? g.logL - 4u : 0u;
    const uint32_t stride = gridDim.x * blockDim.x;
    unsigned long long unequal = 0, negative = 0;
    for (uint32_t c0 = blockIdx.x * blockDim.x + threadIdx.x; c0 < chunks; c0 += stride * kU) {
        uint4 a[kU], by[kU], bz[kU];
        uint32_t nb[kU];
        bool on[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const uint32_t c = c0 + (uint32_t)u * stride;
            on[u] = c < chunks;
            const uint32_t cc = on[u] ? c : 0u;
            const uint32_t i = cc * 16u;
            const uint32_t row = POW2 ? cc >> row_shift : cc / chunks_per_row;      // y + L*z
            const uint32_t cx = cc - row * chunks_per_row;     // chunk index along x
            const uint32_t y = (DIM == 3) ? (POW2 ? row & (g.L - 1u) : row % g.L) : row;
            a[u] = *reinterpret_cast<const uint4 *>(spins + i);
            // +x: the 16 sites shifted by one byte; the 17th byte is the first site of the next chunk (wrapping)
            const uint32_t inext = (cx + 1u == chunks_per_row) ? i + 16u - g.L : i + 16u;
            nb[u] = (uint32_t)(uint8_t)spins[inext];
            const uint32_t iy = (y + 1u == g.L) ? i - (g.LL - g.L) : i + g.L;
            by[u] = *reinterpret_cast<const uint4 *>(spins + iy);
            if (DIM == 3) {
                const uint32_t z = POW2 ? row >> g.logL : row / g.L;
                const uint32_t iz = (z + 1u == g.L) ? i - (g.N - g.LL) : i + g.LL;
                bz[u] = *reinterpret_cast<const uint4 *>(spins + iz);
            }
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const uint32_t neg = __popc(merge4(a[u].x, a[u].y, a[u].z, a[u].w));
            const uint32_t bx = merge4(a[u].x ^ __funnelshift_r(a[u].x, a[u].y, 8), a[u].y ^ __funnelshift_r(a[u].y, a[u].z, 8),
                                       a[u].z ^ __funnelshift_r(a[u].z, a[u].w, 8), a[u].w ^ __funnelshift_r(a[u].w, nb[u], 8));
            const uint32_t byb = merge4(a[u].x ^ by[u].x, a[u].y ^ by[u].y, a[u].z ^ by[u].z, a[u].w ^ by[u].w);
            uint32_t acc = __popc(bx | (byb >> 4));
            if (DIM == 3) acc += __popc(merge4(a[u].x ^ bz[u].x, a[u].y ^ bz[u].y, a[u].z ^ bz[u].z, a[u].w ^ bz[u].w));
            if (on[u]) { unequal += acc; negative += neg; }
        }
    }
    block_accumulate(unequal, negative, ctl, g.N, DIM, E_dst, M_dst);
}

// Generic path: any L >= 2, one site per thread iteration.
template <int DIM>
__global__ void __launch_bounds__(kThreads) energy_magnetisation_scalar(const int8_t *__restrict__ spins, Geometry g, Control *ctl,
                                                                        long long *E_dst, long long *M_dst)
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
    block_accumulate(unequal, negative, ctl, g.N, DIM, E_dst, M_dst);
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

cudaError_t launch_init_lattice(int8_t *spins, uint32_t N, uint64_t seed, int num_sms, cudaStream_t stream)
{
    const int grid = grid_for((N + 15u) / 16u, num_sms, 8);
    init_lattice_kernel<<<grid, kThreads, 0, stream>>>(spins, N, (uint32_t)seed, (uint32_t)(seed >> 32));
    return cudaGetLastError();
}

#ifdef WOLFF_CHECKED
__global__ void check_selftest_kernel(Control *ctl) { WOLFF_CHECK(&ctl->error, ctl == nullptr, 99); }
cudaError_t launch_check_selftest(Control *ctl, cudaStream_t stream)
{
    check_selftest_kernel<<<1, 1, 0, stream>>>(ctl);
    return cudaGetLastError();
}
#endif

cudaError_t launch_validate(const int8_t *spins, uint32_t N, Control *ctl, int num_sms, cudaStream_t stream)
{
    return launch_validate_word(spins, (size_t)N, &ctl->invalid, num_sms, stream);
}

cudaError_t launch_validate_word(const int8_t *spins, size_t n_bytes, unsigned int *invalid, int num_sms, cudaStream_t stream)
{
    const int grid = grid_for((n_bytes + 15u) / 16u, num_sms, 8);
    validate_kernel<<<grid, kThreads, 0, stream>>>(spins, n_bytes, invalid);
    return cudaGetLastError();
}

cudaError_t launch_energy_magnetisation(const int8_t *spins, const Geometry &geo, int dim, Control *ctl,
                                        long long *E_dst, long long *M_dst, int num_sms, cudaStream_t stream)
{
    if (geo.L % 16u == 0u) {
        // kU chunks in flight per thread, a few CTAs per SM (every CTA ends with two atomics on the same two words)
        // (measured on B200, 16 MiB, cold L2, ncu: 12.7 / 9.7 / 11.1 us with 2 / 4 / 8 CTAs per SM)
        // lattices far beyond L2 (64 MiB and more) run long enough that the tail no longer matters and more loads in flight do:
        // 8 CTAs per SM there (profiles/r3_a8.md)
        const int grid = grid_for((geo.N / 16u + kU - 1) / kU, num_sms, geo.N >= (1u << 26) ? 8 : 4);
        if (geo.pow2) {
            if (dim == 2) energy_magnetisation_vec16<2, true><<<grid, kThreads, 0, stream>>>(spins, geo, ctl, E_dst, M_dst);
            else          energy_magnetisation_vec16<3, true><<<grid, kThreads, 0, stream>>>(spins, geo, ctl, E_dst, M_dst);
        } else {
            if (dim == 2) energy_magnetisation_vec16<2, false><<<grid, kThreads, 0, stream>>>(spins, geo, ctl, E_dst, M_dst);
            else          energy_magnetisation_vec16<3, false><<<grid, kThreads, 0, stream>>>(spins, geo, ctl, E_dst, M_dst);
        }
    } else {
        const int grid = grid_for(geo.N, num_sms, 8);
        if (dim == 2) energy_magnetisation_scalar<2><<<grid, kThreads, 0, stream>>>(spins, geo, ctl, E_dst, M_dst);
        else          energy_magnetisation_scalar<3><<<grid, kThreads, 0, stream>>>(spins, geo, ctl, E_dst, M_dst);
    }
    return cudaGetLastError();
}

}  // namespace wolff
