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
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(out_host, out, sizeof(double) * WOLFF_NMICRO, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) rc = WOLFF_ECUDA;
    cudaFree(buf); cudaFree(out); cudaFree(ctl);
    return rc;
}
