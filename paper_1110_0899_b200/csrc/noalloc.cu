// noalloc.cu -- wolff_energy_magnetisation_noalloc: E and M of a lattice the CALLER already holds on the device, for
// callers that cannot let this library allocate device memory.
//
// Who that is.  Every other entry point works on a handle, and wolff_create / wolff_batch_create call cudaMalloc (the
// library's own copy of the lattice, the cluster list, the control block).  Three kinds of host program cannot go that
// way: one that handed the whole card to its own arena at start-up, so that cudaMalloc has nothing left to find; one
// that runs under a fixed memory budget and must not grow once it is initialised; and one with a latency-critical loop
// on other streams of the same device, which cudaMalloc and cudaFree stall while they run.  Such a program still wants
// the measurement of PAPER.md:126 ("measurement of energy and magnetization"; Eq. 2) on a lattice that
// sits in ITS memory.  This file gives it one call that allocates nothing: the lattice and the two result words are the
// caller's, and the reduction's scratch memory (one partial sum per CTA and a ticket) is the file-scope array below,
// which is part of the library image: every GPU that loads the library holds its 256.25 KiB until the process exits.
//
// What it computes is what wolff_observables computes (measure.cu, reading R13): in units of J,
//   E = - sum_i sum_{d < dim} s_i s_{i + e_d}     (periodic; equals 2 * #unequal forward bonds - dim * N)
//   M =   sum_i s_i                               (equals N - 2 * #negative spins)
// as exact integers.  The kernels here are a variant of the A8 reduction with a FIXED amount of lattice per CTA
// (kSitesPerCta), so that the number of partial sums, and with it the scratch, is bounded by the lattice size: that is
// where the size limit WOLFF_NOALLOC_MAX_SITES comes from.  Each CTA stores its two partial counts into its own slot
// (no same-address atomics), takes a ticket, and the CTA that draws the last ticket adds the slots up and writes E, M.
//
// The scratch array is shared by every call in the process and keeps what the last call left in it.  The slots need no
// clearing (every slot a launch reads was written by that launch); the ticket must start at zero and is cleared on the
// caller's stream in front of every launch.  Two calls whose kernels overlap on the GPU (different streams, no
// ordering between them) would mix their slots and tickets: such calls race, and the caller must order them.
#include <cstdarg>
#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/wolff.h"

namespace wolff {
void set_error_v(const char *fmt, va_list ap);      // api.cu: the thread-local text behind wolff_last_error()
}

namespace {

constexpr int kThreads = 256;
constexpr uint32_t kSitesPerCta = 16384u;                                  // 16 KiB of lattice per CTA
constexpr uint32_t kMaxCtas = WOLFF_NOALLOC_MAX_SITES / kSitesPerCta;      // 16,384 slots
constexpr uint32_t kHeaderWords = 32u;                                     // 256 bytes: the ticket, alone in its lines
constexpr uint32_t kSignMask = 0x80808080u;
static_assert(WOLFF_NOALLOC_MAX_SITES % kSitesPerCta == 0u, "whole CTAs");
static_assert(3ull * WOLFF_NOALLOC_MAX_SITES < (1ull << 32), "bond counts of the largest lattice stay far inside 64 bits");

// The scratch memory: [0] ticket (low 32 bits used), [kHeaderWords + 2 b] #unequal forward bonds of CTA b,
// [kHeaderWords + 2 b + 1] #negative spins of CTA b.  In HOST code this name is only a stand-in for the symbol, not a
// device address; the address a kernel can use comes from cudaGetSymbolAddress (scratch_of_current_device below).
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kHeaderWords + 2u * kMaxCtas];

void set_error(const char *fmt, ...) __attribute__((format(printf, 1, 2)));
void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    wolff::set_error_v(fmt, ap);
    va_end(ap);
}

// ---------------------------------------------------------------- device side
// Partial sums of the CTA -> its slot; the last CTA to finish adds all slots and writes the results.
__device__ __forceinline__ void finish(uint32_t unequal, uint32_t negative, unsigned long long *scratch, uint32_t N, int dim,
                                       long long *E_dst, long long *M_dst)
{
    __shared__ unsigned long long s_un[kThreads / 32], s_ng[kThreads / 32];
    __shared__ bool s_last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unequal += __shfl_xor_sync(0xFFFFFFFFu, unequal, o);
        negative += __shfl_xor_sync(0xFFFFFFFFu, negative, o);
    }
    if (lane == 0) { s_un[warp] = unequal; s_ng[warp] = negative; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long un = 0, ng = 0;
        for (int w = 0; w < kThreads / 32; ++w) { un += s_un[w]; ng += s_ng[w]; }
        unsigned long long *slot = scratch + kHeaderWords + 2u * blockIdx.x;
        __stcg(reinterpret_cast<ulonglong2 *>(slot), make_ulonglong2(un, ng));
        __threadfence();                                     // the slot is visible before the ticket is
        const unsigned int t = atomicAdd(reinterpret_cast<unsigned int *>(scratch), 1u);
        s_last = (t == gridDim.x - 1u);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();                                         // every other CTA's fence came before its ticket
    unsigned long long un = 0, ng = 0;
    for (uint32_t b = threadIdx.x; b < gridDim.x; b += kThreads) {
        const ulonglong2 v = __ldcg(reinterpret_cast<const ulonglong2 *>(scratch + kHeaderWords + 2u * b));
        un += v.x;
        ng += v.y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        un += __shfl_xor_sync(0xFFFFFFFFu, un, o);
        ng += __shfl_xor_sync(0xFFFFFFFFu, ng, o);
    }
    if (lane == 0) { s_un[warp] = un; s_ng[warp] = ng; }     // thread 0 read the old values before the barrier above
    __syncthreads();
    if (threadIdx.x == 0) {
        un = 0; ng = 0;
        for (int w = 0; w < kThreads / 32; ++w) { un += s_un[w]; ng += s_ng[w]; }
        if (E_dst) *E_dst = 2ll * (long long)un - (long long)dim * (long long)N;
        if (M_dst) *M_dst = (long long)N - 2ll * (long long)ng;
    }
}

// sign bits (bit 7 of every byte: +1 = 0x01, -1 = 0xFF) of four words gathered into one word
__device__ __forceinline__ uint32_t merge4(uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    return (a & kSignMask) | ((b & kSignMask) >> 1) | ((c & kSignMask) >> 2) | ((d & kSignMask) >> 3);
}

// L a multiple of 16: a 16-byte chunk never straddles a row.  CTA b takes chunks [1024 b, 1024 (b + 1)), thread t the
// chunks 1024 b + t + 256 u, u = 0..3, all loads issued before any is used.
// POW2: L = 2^logL (the host says so): rows and positions by shifts and masks instead of integer divisions.
template <int DIM, bool POW2>
__global__ void __launch_bounds__(kThreads) noalloc_em_vec16(const int8_t *__restrict__ spins, uint32_t L, uint32_t logL, uint32_t N,
                                                             unsigned long long *scratch, long long *E_dst, long long *M_dst)
{
    constexpr int kU = (int)(kSitesPerCta / 16u) / kThreads;     // 4
    const uint32_t chunks = N / 16u, chunks_per_row = L / 16u, LL = L * L;
    const uint32_t row_shift = POW2 ? logL - 4u : 0u;
    const uint32_t first = blockIdx.x * (kSitesPerCta / 16u) + threadIdx.x;
    uint4 a[kU], by[kU], bz[kU];
    uint32_t nb[kU];
    bool on[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
        const uint32_t c = first + (uint32_t)u * kThreads;
        on[u] = c < chunks;
        const uint32_t cc = on[u] ? c : 0u;
        const uint32_t i = cc * 16u;
        const uint32_t row = POW2 ? cc >> row_shift : cc / chunks_per_row;       // y + L z
        const uint32_t cx = cc - row * chunks_per_row;
        const uint32_t y = (DIM == 3) ? (POW2 ? row & (L - 1u) : row % L) : row;
        a[u] = *reinterpret_cast<const uint4 *>(spins + i);
        // +x: the sixteen sites one byte on; the seventeenth is the first site of the next chunk, or of the row (wrap)
        nb[u] = (uint32_t)(uint8_t)spins[(cx + 1u == chunks_per_row) ? i + 16u - L : i + 16u];
        by[u] = *reinterpret_cast<const uint4 *>(spins + ((y + 1u == L) ? i - (LL - L) : i + L));
        if (DIM == 3) {
            const uint32_t z = POW2 ? row >> logL : row / L;
            bz[u] = *reinterpret_cast<const uint4 *>(spins + ((z + 1u == L) ? i - (N - LL) : i + LL));
        }
    }
    uint32_t unequal = 0, negative = 0;
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
    finish(unequal, negative, scratch, N, DIM, E_dst, M_dst);
}

// Any L >= 2: CTA b takes sites [16384 b, 16384 (b + 1)), one site per thread and step.
template <int DIM>
__global__ void __launch_bounds__(kThreads) noalloc_em_scalar(const int8_t *__restrict__ spins, uint32_t L, uint32_t N,
                                                              unsigned long long *scratch, long long *E_dst, long long *M_dst)
{
    const uint32_t LL = L * L;
    const uint32_t begin = blockIdx.x * kSitesPerCta;
    const uint32_t end = (N - begin < kSitesPerCta) ? N : begin + kSitesPerCta;
    uint32_t unequal = 0, negative = 0;
    for (uint32_t i = begin + threadIdx.x; i < end; i += kThreads) {
        const uint32_t x = i % L, t = i / L;
        const uint32_t y = (DIM == 3) ? t % L : t;
        const int s = spins[i];
        negative += (s < 0);
        unequal += (spins[(x + 1u == L) ? i + 1u - L : i + 1u] != s);
        unequal += (spins[(y + 1u == L) ? i - (LL - L) : i + L] != s);
        if (DIM == 3) {
            const uint32_t z = t / L;
            unequal += (spins[(z + 1u == L) ? i - (N - LL) : i + LL] != s);
        }
    }
    finish(unequal, negative, scratch, N, DIM, E_dst, M_dst);
}

// ---------------------------------------------------------------- host side
// Device address of g_noalloc_scratch on each device, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_lookup_mutex;
unsigned long long *g_scratch_addr[kMaxDevices] = {};

int scratch_of_current_device(unsigned long long **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        set_error("no usable CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
        return WOLFF_ECUDA;
    }
    if (dev < 0 || dev >= kMaxDevices) { set_error("device ordinal %d is beyond the %d this entry point keeps track of", dev, kMaxDevices); return WOLFF_EINVAL; }
    std::lock_guard<std::mutex> lock(g_lookup_mutex);
    if (!g_scratch_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            set_error("cudaGetSymbolAddress(scratch) on device %d: %s", dev, cudaGetErrorString(e));
            return WOLFF_ECUDA;
        }
        g_scratch_addr[dev] = static_cast<unsigned long long *>(p);
    }
    *out = g_scratch_addr[dev];
    return WOLFF_OK;
}

// The address a kernel on the CURRENT device can use for p, or null when there is none.
void *device_view(const void *p, bool writable, const char *name, int dev, int *rc)
{
    cudaPointerAttributes at{};
    const cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        set_error("%s: cudaPointerGetAttributes: %s", name, cudaGetErrorString(e));
        *rc = WOLFF_ECUDA;
        return nullptr;
    }
    const bool on_device = (at.type == cudaMemoryTypeDevice && at.device == dev) || at.type == cudaMemoryTypeManaged;
    const bool pinned = writable && at.type == cudaMemoryTypeHost && at.devicePointer != nullptr;
    if (!on_device && !pinned) {
        set_error("%s must be memory of the current device (%d)%s; this entry point makes no staging copy, because it allocates nothing",
                  name, dev, writable ? ", managed memory or pinned host memory" : " or managed memory");
        *rc = WOLFF_EINVAL;
        return nullptr;
    }
    return at.devicePointer;
}

}  // namespace

extern "C" int wolff_energy_magnetisation_noalloc(const int8_t *spins_dev, int dim, int L, int64_t *E_dev, int64_t *M_dev,
                                                  void *cuda_stream)
{
    if (dim != 2 && dim != 3) { set_error("dim must be 2 or 3 (got %d)", dim); return WOLFF_EINVAL; }
    if (L < 2) { set_error("L must be >= 2 (got %d)", L); return WOLFF_EINVAL; }
    unsigned long long N = 1;
    for (int d = 0; d < dim; ++d) {
        N *= (unsigned long long)L;
        if (N > (unsigned long long)WOLFF_NOALLOC_MAX_SITES) {
            set_error("a lattice of L = %d in %d dimensions has more than WOLFF_NOALLOC_MAX_SITES = %u sites: the scratch array of "
                      "wolff_energy_magnetisation_noalloc is fixed in size (one slot per %u sites); use wolff_create, wolff_set_spins "
                      "and wolff_observables for larger lattices", L, dim, (unsigned)WOLFF_NOALLOC_MAX_SITES, (unsigned)kSitesPerCta);
            return WOLFF_EINVAL;
        }
    }
    if (!spins_dev) { set_error("spins_dev is NULL"); return WOLFF_EINVAL; }
    if ((L % 16 == 0) && (reinterpret_cast<uintptr_t>(spins_dev) & 15u)) {
        set_error("spins_dev must be 16-byte aligned when L is a multiple of 16 (the lattice is read 16 sites per load)");
        return WOLFF_EINVAL;
    }
    if (!E_dev && !M_dev) return WOLFF_OK;

    unsigned long long *scratch = nullptr;
    int rc = scratch_of_current_device(&scratch);      // the first call on a device looks the address up
    if (rc != WOLFF_OK) return rc;
    int dev = 0;
    (void)cudaGetDevice(&dev);
    const int8_t *spins = static_cast<const int8_t *>(device_view(spins_dev, false, "spins_dev", dev, &rc));
    if (!spins) return rc;
    long long *E_dst = nullptr, *M_dst = nullptr;
    if (E_dev) { E_dst = static_cast<long long *>(device_view(E_dev, true, "E_dev", dev, &rc)); if (!E_dst) return rc; }
    if (M_dev) { M_dst = static_cast<long long *>(device_view(M_dev, true, "M_dev", dev, &rc)); if (!M_dst) return rc; }

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    // the ticket starts at zero, whatever an earlier call (or one that was cut short) left there
    cudaError_t e = cudaMemsetAsync(scratch, 0, kHeaderWords * sizeof(unsigned long long), stream);
    if (e != cudaSuccess) { set_error("clearing the ticket: %s", cudaGetErrorString(e)); return WOLFF_ECUDA; }
    const uint32_t n = (uint32_t)N, l = (uint32_t)L;
    const unsigned int grid = (unsigned int)((N + kSitesPerCta - 1u) / kSitesPerCta);       // <= kMaxCtas: one slot each
    if (L % 16 == 0) {
        uint32_t logL = 0;
        while ((1u << logL) < l) ++logL;
        if ((1u << logL) == l) {
            if (dim == 2) noalloc_em_vec16<2, true><<<grid, kThreads, 0, stream>>>(spins, l, logL, n, scratch, E_dst, M_dst);
            else          noalloc_em_vec16<3, true><<<grid, kThreads, 0, stream>>>(spins, l, logL, n, scratch, E_dst, M_dst);
        } else {
            if (dim == 2) noalloc_em_vec16<2, false><<<grid, kThreads, 0, stream>>>(spins, l, 0u, n, scratch, E_dst, M_dst);
            else          noalloc_em_vec16<3, false><<<grid, kThreads, 0, stream>>>(spins, l, 0u, n, scratch, E_dst, M_dst);
        }
    } else {
        if (dim == 2) noalloc_em_scalar<2><<<grid, kThreads, 0, stream>>>(spins, l, n, scratch, E_dst, M_dst);
        else          noalloc_em_scalar<3><<<grid, kThreads, 0, stream>>>(spins, l, n, scratch, E_dst, M_dst);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("launch of the E/M reduction: %s", cudaGetErrorString(e)); return WOLFF_ECUDA; }
    return WOLFF_OK;
}
