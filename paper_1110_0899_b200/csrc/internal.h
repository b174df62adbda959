// internal.h -- host/device shared declarations of libwolff_b200 (not part of the public ABI).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "device_common.cuh"

namespace wolff {

// Phases carried in the barrier word (bits 39:32).
enum Phase : unsigned int {
    kPhaseGrid = 1,    // next level is grid-wide
    kPhaseToCluster = 2,   // frontier narrowed: cluster 0 continues from the window [lo, hi)
    kPhaseDone = 3,    // the frontier is empty: the update's cluster is complete
    kPhaseExit = 4,    // all updates of this launch are done
    kPhaseAbort = 5    // watchdog fired
};

// Global-memory control block of one handle.  Every hot word sits in its own 128-byte line.
// The words before acc_unequal are zeroed at every launch of a growth kernel.
struct alignas(128) Control {
    // [gen:24 | phase:8 | hi:32]; polled by every CTA, written by the last arriver / by CTA 0.
    alignas(128) unsigned long long bar;
    alignas(128) unsigned int arrive;          // grid barrier arrival counter
    alignas(128) unsigned int tail;            // append cursor of the cluster list
    // descriptor of a grid phase / of a barrier-free phase, written by CTA 0 before it releases the others
    alignas(128) unsigned int lo;
    int s0;
    unsigned long long u;
    // barrier-free kernel: [seq:32 | .. | s0<0:1 | op:8]; seq = 2g when phase g starts, 2g+1 when it is over
    alignas(128) unsigned long long state;
    alignas(128) unsigned long long added;     // barrier-free kernel: spins claimed in the running phase
    alignas(128) unsigned long long acks;      // barrier-free kernel: phase ends seen, summed over helper CTAs
    alignas(128) unsigned int error;           // nonzero: a barrier / phase timed out
    unsigned int pad4;
    unsigned long long stats[16];              // see WOLFF_NSTATS in wolff.h
    // E/M reduction scratch
    alignas(128) unsigned long long acc_unequal;
    unsigned long long acc_negative;
    unsigned int ticket;
    unsigned int invalid;         // set_spins validation
    long long E;
    long long M;
};

struct GrowthParams {
    int8_t *spins;
    uint32_t *clist;        // cluster list, N entries
    uint32_t *sizes;        // per-update cluster sizes of this launch
    Control *ctl;
    Geometry geo;
    uint32_t key0, key1;    // Philox key = seed
    unsigned long long thr; // bond threshold in [0, 2^32]
    unsigned long long u0;  // first update index of this launch
    unsigned long long n_updates;
    uint32_t up;            // leave one-CTA mode (wake the cluster) when the frontier is wider than this
    uint32_t down;          // return to one-CTA mode when the frontier is at most this wide
    uint32_t cl_up;         // leave cluster mode (grid phase) when the frontier is wider than this
    uint32_t grid_down;     // return from a grid phase to cluster mode when the frontier is at most this wide
    uint32_t bal_min;       // cluster mode: a CTA holding more than max(bal_min, 2 x fair share) triggers rebalancing
    uint32_t qcap;          // entries per shared-memory queue buffer
};

// Barrier-free kernel (growth_async.cu): the lattice is cut into tiles of 2^tile_log sites per side, tile
// (tx, ty, tz) belongs to CTA (tx + hashA*ty + hashB*tz) mod G, and a claimed site is expanded by the CTA that
// owns its tile.  Sites that cross into another CTA's tile travel through that CTA's inbox, a segment of one
// global array sized by the number of sites the CTA owns (a site is handed over at most once per update).
struct AsyncParams {
    GrowthParams g;
    uint32_t *inbox;                 // N entries, every one kEmpty between phases
    const uint32_t *seg;             // [G + 1] first inbox entry of each CTA
    unsigned long long *gtail;       // [G] entries pushed into CTA c's inbox since the launch began
    unsigned long long *gdone;       // [G] of those, how many are completely processed (with all local descendants)
    uint32_t tile_log;
    uint32_t hashA, hashB;
    uint32_t ring_cap;               // entries of the shared-memory ring (power of two)
    uint32_t lvl_cap;                // entries per one-CTA level buffer
    uint32_t zero;                   // always 0: makes the second pass of the termination check depend on the first
    unsigned long long watchdog_ns;  // a phase longer than this aborts the launch
};

// Launch shape of the persistent kernel.
struct GrowthLaunch {
    int grid_ctas;          // total CTAs, a multiple of cluster_ctas
    int cluster_ctas;       // CTAs per thread-block cluster (1, 2, 4, 8 or 16)
    size_t smem_bytes;      // dynamic shared memory per CTA (the two queue buffers)
    bool cooperative;       // launch with the cooperative attribute (co-residency guaranteed by the driver)
    bool spec;              // speculative claims: no neighbour gather, one atomic per active bond (expand.cuh)
};

constexpr int kGrowthThreads = 512;

// launchers (defined next to their kernels)
cudaError_t launch_growth(const GrowthParams &p, int dim, const GrowthLaunch &l, cudaStream_t stream);
// sets the kernel's attributes for this launch shape and reports how many clusters can be co-resident
cudaError_t growth_max_clusters(int dim, bool pow2, const GrowthLaunch &l, int *max_clusters);
// barrier-free kernel: sets attributes, reports co-resident CTAs per SM; launches `ctas` CTAs cooperatively
cudaError_t async_prepare(int dim, bool pow2, bool spec, size_t smem_bytes, int *ctas_per_sm);
cudaError_t launch_growth_async(const AsyncParams &p, int dim, bool spec, int ctas, size_t smem_bytes, cudaStream_t stream);
cudaError_t launch_init_lattice(int8_t *spins, uint32_t N, uint64_t seed, cudaStream_t stream);
cudaError_t launch_validate(const int8_t *spins, uint32_t N, Control *ctl, cudaStream_t stream);
cudaError_t launch_energy_magnetisation(const int8_t *spins, const Geometry &geo, int dim, Control *ctl,
                                        int num_sms, cudaStream_t stream);

}  // namespace wolff
