// microbench.cu -- dependent-latency microbenchmarks that define the LATENCY roofline of the growth
// kernel ("Microbenchmarks to ship with the bench").  One BFS level of the growth
// kernel is a chain  queue read -> neighbour gather (L2 load) -> claim (L2 atomic) -> append ->
// barrier;  these kernels time each link in isolation on the same device, same access kinds
// (ld.global.cg on an L2-resident 16 MiB buffer, atom.or with return, bar.sync at 512 threads, and
// the library's own atomic grid barrier at the persistent kernel's launch shape).
#include <cstdio>

#include "../../include/wolff.h"
#include "internal.h"

namespace wolff {
namespace {

__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// out[0] = ns per dependent ld.global.cg (one lane), out[1] = ns per dependent scattered warp load
// (32 lanes, 32 distinct lines), out[2] = ns per dependent atom.or with return (one lane),
// out[3] = ns per dependent scattered warp atomic, out[4] = ns per __syncthreads (512 threads),
// out[5] = ns for three back-to-back Philox4x32-10 blocks (one warp)
__global__ void __launch_bounds__(512, 1) latency_kernel(unsigned int *buf, uint32_t mask, int iters, double *out)
{
    const unsigned int tid = threadIdx.x;
    __shared__ unsigned int sink;
    if (tid == 0) sink = 0;
    __syncthreads();
    // warm the buffer into L2
    for (uint32_t i = tid; i <= mask; i += blockDim.x) buf[i] = 0u;
    __syncthreads();

    if (tid == 0) {
        uint32_t idx = 12345u & mask;
        unsigned long long t0 = globaltimer_ns();
        for (int k = 0; k < iters; ++k) {
            const unsigned int v = __ldcg(buf + idx);
            idx = (idx * 1664525u + 1013904223u + v) & mask;
        }
        unsigned long long t1 = globaltimer_ns();
        out[0] = (double)(t1 - t0) / iters;
        atomicAdd(&sink, idx);
        idx = 777u & mask;
        t0 = globaltimer_ns();
        for (int k = 0; k < iters; ++k) {
            const unsigned int v = atomicOr(buf + idx, 0u);
            idx = (idx * 1664525u + 1013904223u + v) & mask;
        }
        t1 = globaltimer_ns();
        out[2] = (double)(t1 - t0) / iters;
        atomicAdd(&sink, idx);
    }
    __syncthreads();
    if (tid < 32) {
        uint32_t idx = (tid * 2654435761u) & mask;
        unsigned long long t0 = globaltimer_ns();
        for (int k = 0; k < iters; ++k) {
            const unsigned int v = __ldcg(buf + idx);
            idx = (idx * 1664525u + 1013904223u + v + tid) & mask;
        }
        unsigned long long t1 = globaltimer_ns();
        if (tid == 0) out[1] = (double)(t1 - t0) / iters;
        atomicAdd(&sink, idx);
        t0 = globaltimer_ns();
        for (int k = 0; k < iters; ++k) {
            const unsigned int v = atomicOr(buf + idx, 0u);
            idx = (idx * 1664525u + 1013904223u + v + tid) & mask;
        }
        t1 = globaltimer_ns();
        if (tid == 0) out[3] = (double)(t1 - t0) / iters;
        atomicAdd(&sink, idx);
        // Philox: three dependent-free blocks per iteration, chained through the counter
        uint32_t c = tid;
        t0 = globaltimer_ns();
        for (int k = 0; k < iters; ++k) {
            const uint4 a = philox4x32_10(c, 0u, 1u, 2u, 3u, 4u);
            const uint4 b = philox4x32_10(c + 1u, 0u, 1u, 2u, 3u, 4u);
            const uint4 d = philox4x32_10(c + 2u, 0u, 1u, 2u, 3u, 4u);
            c = a.x ^ b.y ^ d.z;
        }
        t1 = globaltimer_ns();
        if (tid == 0) out[5] = (double)(t1 - t0) / iters;
        atomicAdd(&sink, c);
    }
    __syncthreads();
    unsigned long long t0 = globaltimer_ns();
    for (int k = 0; k < iters; ++k) __syncthreads();
    unsigned long long t1 = globaltimer_ns();
    if (tid == 0) out[4] = (double)(t1 - t0) / iters;
    if (tid == 0 && sink == 0xFFFFFFFFu) out[0] = -1.0;   // keep the chains alive
}

// The library's grid barrier (same instructions as growth.cu's level barrier) at the persistent
// kernel's launch shape: out[6] = ns per barrier.
__global__ void __launch_bounds__(kGrowthThreads, 1) grid_barrier_kernel(Control *ctl, int iters, double *out)
{
    const unsigned int G = gridDim.x;
    __shared__ unsigned int sh_gen;
    unsigned int gen = 0;
    unsigned long long t0 = 0;
    if (threadIdx.x == 0 && blockIdx.x == 0) t0 = globaltimer_ns();
    for (int k = 0; k < iters; ++k) {
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned int old = atom_add_acq_rel_u32(&ctl->arrive, 1u);
            if (old == G - 1u) {
                st_relaxed_u32(&ctl->arrive, 0u);
                st_release_u64(&ctl->bar, (unsigned long long)(gen + 1u));
            } else {
                unsigned int polls = 0;
                while (ld_acquire_u64(&ctl->bar) != (unsigned long long)(gen + 1u))
                    if (++polls > (1u << 24)) break;
            }
            sh_gen = gen + 1u;
        }
        __syncthreads();
        gen = sh_gen;
    }
    if (threadIdx.x == 0 && blockIdx.x == 0) out[6] = (double)(globaltimer_ns() - t0) / iters;
}

// out[7] = ns per pass of the minimal dependent chain of the shared-memory-resident kernel (growth_tiles.cu), one warp
// alone on an SM: site address -> ld.shared of the neighbour's spin word and of a bond word -> compare ->
// atom.shared (claim) -> compare -> ballot, popc -> st.shared (stage) -> __syncwarp -> ld.shared (next site).
// Every lane wins every pass (fresh bytes; the seed spin flips sign after each sweep of the 64 KiB region), so
// this is the floor of one pass: no Philox, no messages, no queue.
__global__ void __launch_bounds__(32, 1) smem_pass_kernel(int iters, double *out)
{
    extern __shared__ __align__(16) unsigned int dyn[];
    constexpr unsigned int kBytes = 64u << 10, kStep = 132u, kSweep = (kBytes - 128u) / kStep;
    unsigned int *const lat = dyn;                         // kBytes of spins, 0x01 = +1, 0xFF = -1
    unsigned int *const bond = dyn + kBytes / 4u;          // one bit per site
    unsigned int *const stage = bond + kBytes / 32u;
    const unsigned int lane = threadIdx.x, lt = (1u << lane) - 1u;
    for (unsigned int i = lane; i < kBytes / 4u; i += 32u) lat[i] = 0x01010101u;
    for (unsigned int i = lane; i < kBytes / 32u; i += 32u) bond[i] = 0xFFFFFFFFu;
    __syncwarp();
    unsigned int a = lane * 4u, won_total = 0;
    const unsigned long long t0 = globaltimer_ns();
    for (int k = 0; k < iters; ++k) {
        const unsigned int step = (unsigned int)k % kSweep;
        const bool pos = (((unsigned int)k / kSweep) & 1u) == 0u;
        const unsigned int s0w = pos ? 0x01010101u : 0xFFFFFFFFu;
        const unsigned int na = step == 0u ? lane * 4u + (a & 3u) : a + kStep;      // depends on the staged site
        const unsigned int spw = *reinterpret_cast<volatile unsigned int *>(lat + (na >> 2));
        const unsigned int bw = *reinterpret_cast<volatile unsigned int *>(bond + (na >> 5));
        const unsigned int bytemask = 0xFFu << ((na & 3u) * 8u);
        const bool cand = ((bw >> (na & 31u)) & 1u) != 0u && ((spw ^ s0w) & bytemask) == 0u;
        unsigned int old = ~s0w;
        if (cand) old = pos ? atomicOr(lat + (na >> 2), 0xFEFEFEFEu & bytemask) : atomicAnd(lat + (na >> 2), ~(0xFEFEFEFEu & bytemask));
        const bool won = ((old ^ s0w) & bytemask) == 0u;
        const unsigned int wb = __ballot_sync(0xFFFFFFFFu, won);
        if (won) *reinterpret_cast<volatile unsigned int *>(stage + __popc(wb & lt)) = na;
        __syncwarp();
        won_total += __popc(wb);
        a = *reinterpret_cast<volatile unsigned int *>(stage + ((lane + 1u) & 31u));
    }
    const unsigned long long t1 = globaltimer_ns();
    if (lane == 0) { out[7] = (double)(t1 - t0) / iters; out[8] = (double)won_total / (32.0 * iters); }
}

// out[9..12]: the links of the cluster-resident kernel (growth_cluster.cu) between two CTAs of one thread-block
// cluster: out[9] = ns per dependent ld.shared::cluster on the PEER's shared memory (one lane), out[10] = ns per dependent
// atom.shared::cluster.or with return on the peer (one lane), out[11] = the same with 32 lanes on 32 scattered words,
// out[12] = ns one way for a word stored into the peer's shared memory to be seen by a warp polling there (half of a
// ping-pong round trip).
__device__ __forceinline__ uint32_t mb_smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t mb_mapa(uint32_t a, uint32_t r)
{
    uint32_t o;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(o) : "r"(a), "r"(r));
    return o;
}
__device__ __forceinline__ uint32_t mb_cl_ld(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.volatile.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void mb_cl_st(uint32_t a, uint32_t v) { asm volatile("st.volatile.shared::cluster.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ uint32_t mb_cl_or(uint32_t a, uint32_t v)
{
    uint32_t o;
    asm volatile("atom.shared::cluster.or.b32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory");
    return o;
}
__device__ __forceinline__ void mb_cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t mb_cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(32, 1) dsmem_kernel(int iters, double *out)
{
    extern __shared__ __align__(16) unsigned int dyn[];
    constexpr unsigned int kWords = 8192;             // 32 KiB of the peer's shared memory
    __shared__ unsigned int flag;
    const unsigned int lane = threadIdx.x, rank = mb_cluster_rank();
    for (unsigned int i = lane; i < kWords; i += 32u) dyn[i] = 0u;
    if (lane == 0) flag = 0u;
    mb_cluster_sync();
    const uint32_t mask = kWords - 1u;
    if (rank == 0u) {
        const uint32_t peer = mb_mapa(mb_smem_addr(dyn), 1u);
        if (lane == 0) {
            uint32_t idx = 12345u & mask;
            unsigned long long t0 = globaltimer_ns();
            for (int k = 0; k < iters; ++k) { const uint32_t v = mb_cl_ld(peer + idx * 4u); idx = (idx * 1664525u + 1013904223u + v) & mask; }
            unsigned long long t1 = globaltimer_ns();
            out[9] = (double)(t1 - t0) / iters;
            t0 = globaltimer_ns();
            for (int k = 0; k < iters; ++k) { const uint32_t v = mb_cl_or(peer + idx * 4u, 0u); idx = (idx * 1664525u + 1013904223u + v) & mask; }
            t1 = globaltimer_ns();
            out[10] = (double)(t1 - t0) / iters + (idx == 0xFFFFFFFFu ? 1.0 : 0.0);
        }
        __syncwarp();
        uint32_t idx = (lane * 2654435761u) & mask;
        const unsigned long long t0 = globaltimer_ns();
        for (int k = 0; k < iters; ++k) { const uint32_t v = mb_cl_or(peer + idx * 4u, 0u); idx = (idx * 1664525u + 1013904223u + v + lane) & mask; }
        const unsigned long long t1 = globaltimer_ns();
        if (lane == 0) out[11] = (double)(t1 - t0) / iters + (idx == 0xFFFFFFFFu ? 1.0 : 0.0);
    }
    mb_cluster_sync();
    if (lane == 0) {
        const uint32_t mine = mb_smem_addr(&flag), theirs = mb_mapa(mine, rank ^ 1u);
        if (rank == 0u) {
            const unsigned long long t0 = globaltimer_ns();
            for (int k = 1; k <= iters; ++k) {
                mb_cl_st(theirs, (uint32_t)k);
                while (mb_cl_ld(mine) != (uint32_t)k) { }
            }
            out[12] = (double)(globaltimer_ns() - t0) / (2.0 * iters);
        } else {
            for (int k = 1; k <= iters; ++k) {
                while (mb_cl_ld(mine) != (uint32_t)k) { }
                mb_cl_st(theirs, (uint32_t)k);
            }
        }
    }
    mb_cluster_sync();
}

}  // namespace
}  // namespace wolff

using namespace wolff;

extern "C" WOLFF_API int wolff_microbench(double *out_host, int n_out)
{
    if (!out_host || n_out < WOLFF_NMICRO) return WOLFF_EINVAL;
    const uint32_t words = 4u << 20;   // 16 MiB, the size of the largest BASELINE lattice
    unsigned int *buf = nullptr;
    double *out = nullptr;
    Control *ctl = nullptr;
    cudaDeviceProp prop{};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return WOLFF_ECUDA;
    if (cudaMalloc(&buf, (size_t)words * 4) != cudaSuccess || cudaMalloc(&out, sizeof(double) * WOLFF_NMICRO) != cudaSuccess ||
        cudaMalloc(&ctl, sizeof(Control)) != cudaSuccess) {
        cudaFree(buf); cudaFree(out); cudaFree(ctl);
        return WOLFF_ENOMEM;
    }
    cudaMemset(out, 0, sizeof(double) * WOLFF_NMICRO);
    cudaMemset(ctl, 0, sizeof(Control));
    int rc = WOLFF_OK;
    const int iters = 2000;
    latency_kernel<<<1, 512>>>(buf, words - 1u, iters, out);
    int grid = prop.multiProcessorCount;
    void *args[] = { &ctl, const_cast<int *>(&iters), &out };
    cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(&grid_barrier_kernel), dim3(grid),
                                                dim3(kGrowthThreads), args, 0, nullptr);
    if (e == cudaSuccess) {
        const size_t smem = (64u << 10) + (64u << 10) / 8u + 32u * sizeof(unsigned int);
        e = cudaFuncSetAttribute(smem_pass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) smem_pass_kernel<<<1, 32, smem>>>(4 * 496, out);
    }
    if (e == cudaSuccess) {
        dsmem_kernel<<<2, 32, 8192 * sizeof(unsigned int)>>>(iters, out);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(out_host, out, sizeof(double) * WOLFF_NMICRO, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) rc = WOLFF_ECUDA;
    cudaFree(buf); cudaFree(out); cudaFree(ctl);
    return rc;
}
