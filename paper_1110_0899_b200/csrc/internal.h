// internal.h -- host/device shared declarations of libwolff_b200 (not part of the public ABI).
#pragma once
#include <cstddef>
#include <cstdint>
#include <mutex>
#include <utility>
#include <vector>
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
// The words before `error` are zeroed at every launch of a growth kernel (kControlClearBytes); what follows is
// never cleared by a launch: the error flag is STICKY (a kernel that finds it set leaves at once; the host reads it
// at its next synchronising call and marks the handle failed), and the measurement state runs on across launches.
struct alignas(128) Control {
    // [gen:24 | phase:8 | hi:32]; polled by every CTA, written by the last arriver / by CTA 0.
    alignas(128) unsigned long long bar;
    alignas(128) unsigned int arrive;          // grid barrier arrival counter
    alignas(128) unsigned int tail;            // append cursor of the cluster list
    // descriptor of a grid phase, written by CTA 0 before it releases the others
    alignas(128) unsigned int lo;
    int s0;
    unsigned long long u;
    alignas(128) unsigned long long stats[16]; // see WOLFF_NSTATS in wolff.h
    // in-kernel measurement of the shared-memory-resident kernel: arrival counters (modulo 2^32: G per measured
    // update) and the sums of one whole-lattice evaluation
    alignas(128) unsigned int meas_arrive_a;   // CTAs whose tile faces of the finished update are in global memory
    alignas(128) unsigned int meas_arrive_b;   // CTAs whose partial sums are in meas_unequal / meas_negative
    alignas(128) unsigned long long meas_unequal;
    unsigned long long meas_negative;
    // ---------------------------------------------------------------- not cleared by a launch
    alignas(128) unsigned int error;           // nonzero: a barrier / an update timed out (sticky)
    unsigned int invalid;                      // set_spins validation
    unsigned int ticket;                       // E/M reduction: CTAs done
    unsigned int pad0;
    unsigned long long acc_unequal;            // E/M reduction scratch: #unequal bonds | #negative spins << 33
    unsigned long long acc_negative;           // (unused)
    long long E;                               // result of the last reduction; with in-kernel measurement: the
    long long M;                               // running values after the last measured update
    unsigned long long moments[10];            // in-kernel measurement: accumulated sums (layout: wolff_get_moments)
};
constexpr size_t kControlClearBytes = offsetof(Control, error);

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
    // in-kernel measurement (wolff_set_option "measure"): E and M after every update, accumulated moments
    uint32_t measure;       // 1: on
    uint32_t claim_bits;    // 0xFE, or 0xFC when measuring in the level-synchronous kernel (membership mark, device_common.cuh)
    long long *E_log;       // per-update E, M of this launch (n_updates entries each) when measure
    long long *M_log;
    uint32_t *ns_log;       // per-update duration in nanoseconds (always written; saturates at 2^32 - 1)
};

// Shared-memory-resident barrier-free kernel (growth_tiles.cu).  The lattice (L a power of two) is cut into tiles of
// 2^tile_log sites per side; tile t belongs to CTA ((t * permA) mod ntiles) mod G and sits in that CTA's shared
// memory for the length of the launch.  A claim that crosses into another CTA's territory travels as a 64-bit
// message through that CTA's inbox (global memory).  All counters below run on across launches (nothing is reset).
struct TileParams {
    GrowthParams g;
    unsigned long long *inbox;       // G segments of in_cap messages; slot validity by lap parity, never cleared
    unsigned int *gtail;             // [G] messages ever pushed into CTA c's inbox, modulo 2^32 (its low bits are the inbox slot)
    unsigned long long *gdone;       // [G] of those, how many are consumed with their whole local progeny expanded
    unsigned long long *gspill;      // [G] running position of CTA c's spill list
    unsigned int *gihead;            // [G] messages CTA c's receiver has taken out of its inbox, modulo 2^32: a sender may write
                                     // slot pos only while pos - gihead[c] < in_cap (back-pressure)
    unsigned long long *added;       // spins ever claimed (sum over CTAs, published with gdone)
    uint32_t *spill;                 // G segments of 2^spill_log entries: overflow of the shared-memory ring
    unsigned long long magicG;       // ceil(2^40 / G)
    uint32_t tile_log;
    uint32_t ntiles;                 // (L >> tile_log)^dim, a power of two
    uint32_t permA, permAinv;        // odd multiplier and its inverse mod ntiles
    uint32_t G;                      // CTAs (one per SM, all co-resident)
    uint32_t slots;                  // tiles per CTA (upper bound)
    uint32_t in_log, in_cap;         // inbox entries per CTA (a power of two, at least 32)
    uint32_t bp;                     // 1: in_cap is below what one update can send a CTA: senders check the capacity (back-pressure)
    uint32_t spill_log;              // spill entries per CTA (at least the sites the CTA owns)
    uint32_t ring_cap;               // entries of the shared-memory ring (power of two)
    unsigned long long watchdog_ns;  // an update longer than this aborts the launch
    uint32_t tables;                 // 1: bond tables (nbuf buffers of dim bit planes per tile) are part of the shared-memory layout
    uint32_t nbuf;                   // 2: the tables of the running update and the next one; 1: the running update only (0 without tables)
    uint32_t fill_mode;              // idle warps fill bond tables: 0 never, 1 when updates are long enough to pay for it, 2 always
    unsigned long long fill_min_ns;  // fill_mode 1: mean time per update above which tables are filled
    uint32_t *gfill;                 // [G] fill_on of CTA c at the end of the last launch
    uint32_t thr32, thr_all;         // low word of the bond threshold; thr_all = 1 when thr = 2^32 (every bond active)
    uint32_t idle_ns;                // longest sleep of an idle worker warp between two polls of the ring
    // in-kernel measurement: the low faces of every tile (the sites with coordinate d = 0 inside the tile), written by
    // the tile's owner after each measured update and read by the owner of the tile next to it in direction -d:
    // faces[((slot * G + owner) * dim + d) * B^(dim-1) + f], one byte per site
    int8_t *faces;
};

// Cluster-resident bit-packed kernel (growth_cluster.cu).  The lattice (any L, N <= 2^24) is held as one bit per spin in
// the distributed shared memory of ONE thread-block cluster of nC CTAs: word w (sites 32 w .. 32 w + 31) lives in CTA
// w / wpc (the last word may be partial, the last CTAs may hold fewer words, or none).  The spill list and its two counters run on across launches (nothing is reset).
struct ClusterParams {
    GrowthParams g;
    uint32_t nC;                     // CTAs of the cluster (1, 2, 4, 8 or 16)
    uint32_t wpc, wpc_log;           // 32-bit words of the bit lattice per CTA (a power of two)
    uint32_t words;                  // words of the whole lattice: ceil(N / 32)
    unsigned long long magicL, magicLL;   // ceil(2^40 / L), ceil(2^40 / L^2): a div L for a < 2^24 when L is not a power of two
    uint32_t ring_cap;               // entries of a CTA's shared-memory ring (power of two)
    uint32_t *spill;                 // 2^spill_log entries (>= N): overflow of the rings, shared by the cluster
    uint32_t spill_log;
    unsigned long long *spill_ctr;   // [0] entries ever pushed, [1] entries ever taken
    unsigned long long watchdog_ns;  // an update longer than this aborts the launch
    uint32_t thr32, thr_all;         // low word of the bond threshold; thr_all = 1 when thr = 2^32 (every bond active)
    uint32_t idle_ns;                // longest sleep of an idle warp between two polls of its ring
};

// R independent chains in one launch, one CTA per chain at a time (growth_batch.cu).
struct BatchParams {
    int8_t *spins;                   // R lattices, lattice_stride bytes apart
    uint32_t *lists;                 // R member lists of N entries (the list of the running cluster; its tail is the frontier)
    uint32_t *sizes;                 // [R][n_updates] cluster sizes of this launch
    long long *E_log, *M_log;        // [R][n_updates] E, M after every update (measure)
    const uint2 *keys;               // [R] Philox key = seed of the chain
    const unsigned long long *thr;   // [R] bond threshold of the chain
    long long *EM;                   // [R][2] E, M of every chain: the last whole-lattice evaluation / the running values
    unsigned long long *moments;     // [R][10] accumulated sums (layout: wolff_get_moments)
    unsigned long long *stats;       // [4] updates, flipped spins, levels, claim attempts of this launch
    unsigned int *next;              // the next chain to be taken by a CTA (zeroed per launch)
    Geometry geo;
    size_t lattice_stride;
    unsigned long long u0;           // first update index of this launch (shared by all chains)
    unsigned long long n_updates;
    uint32_t R;
    uint32_t measure;
    uint32_t qcap;                   // entries per shared-memory frontier buffer
};
constexpr int kBatchMaxThreads = 256;

// Launch shape of the persistent kernel.
struct GrowthLaunch {
    int grid_ctas;          // total CTAs, a multiple of cluster_ctas
    int cluster_ctas;       // CTAs per thread-block cluster (1, 2, 4, 8 or 16)
    size_t smem_bytes;      // dynamic shared memory per CTA (the two queue buffers)
    bool cooperative;       // launch with the cooperative attribute (co-residency guaranteed by the driver)
    bool spec;              // speculative claims: no neighbour gather, one atomic per active bond (expand.cuh)
};

constexpr int kGrowthThreads = 512;
constexpr int kTileThreads = 384;
constexpr int kClusterThreads = 512;

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel function (per device), not to a handle.  If every
// handle set it to its own need, two host threads driving handles of different L could interleave set(A), set(B smaller),
// launch(A) and A's launch would be refused.  So the library only ever sets ONE value per kernel: the most the device
// allows it (the opt-in maximum minus the kernel's static shared memory).  Setting it again, from any thread, changes
// nothing, and every handle's launch fits under it; occupancy follows the shared memory a launch asks for, not this cap.
inline cudaError_t allow_max_dynamic_smem(const void *fn)
{
    static std::mutex mu;
    static std::vector<std::pair<const void *, int>> done;      // (kernel, device) pairs already raised: a launch pays one lookup
    int dev = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    {
        std::lock_guard<std::mutex> lock(mu);
        for (const auto &d : done)
            if (d.first == fn && d.second == dev) return cudaSuccess;
    }
    e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    cudaFuncAttributes fa{};
    e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    done.emplace_back(fn, dev);
    return cudaSuccess;
}

// launchers (defined next to their kernels)
cudaError_t launch_growth(const GrowthParams &p, int dim, const GrowthLaunch &l, cudaStream_t stream);
// sets the kernel's attributes for this launch shape and reports how many clusters can be co-resident
cudaError_t growth_max_clusters(int dim, bool pow2, const GrowthLaunch &l, int *max_clusters);
// shared-memory-resident kernel: shared memory needed, attributes + co-resident CTAs per SM, cooperative launch of tp.G CTAs
size_t tiles_smem_bytes(int dim, uint32_t tile_log, uint32_t slots, uint32_t ring_cap, uint32_t nbuf);
cudaError_t tiles_prepare(int dim, size_t smem_bytes, int *ctas_per_sm);
cudaError_t launch_growth_tiles(const TileParams &tp, int dim, size_t smem_bytes, cudaStream_t stream);
// cluster-resident kernel: shared memory needed, attributes + co-resident clusters, launch of one cluster of cp.nC CTAs
size_t cluster_smem_bytes(uint32_t wpc, uint32_t ring_cap);
cudaError_t cluster_prepare(int dim, bool pow2, uint32_t nC, size_t smem_bytes, int *max_clusters);
// fills nC, wpc, wpc_log, words, magicL, magicLL, ring_cap, spill_log of *cp; false when the lattice does not fit one cluster
bool cluster_plan(int dim, const Geometry &geo, int max_ctas, uint32_t ring_cap, size_t smem_optin, ClusterParams *cp, size_t *smem_bytes,
                  int *max_clusters);
cudaError_t launch_growth_cluster(const ClusterParams &cp, int dim, size_t smem_bytes, cudaStream_t stream);
// batch of chains: CTAs of `threads` threads, `grid` of them; co-resident CTAs per SM; E, M of every chain into EM
// bits: the bit-packed shared-memory-resident variant; its shared memory: the frontier buffers + N/8 bytes per plane
size_t batch_smem_bytes(uint32_t N, uint32_t qcap, bool bits, bool measure);
cudaError_t launch_growth_batch(const BatchParams &bp, int dim, bool bits, int grid, int threads, cudaStream_t stream);
cudaError_t batch_ctas_per_sm(int dim, bool pow2, bool bits, int threads, size_t smem, int *per_sm);
cudaError_t launch_batch_energy(const int8_t *spins, size_t stride, const Geometry &geo, int dim, uint32_t R, unsigned long long *acc,
                                long long *EM, int num_sms, cudaStream_t stream);
#ifdef WOLFF_CHECKED
cudaError_t launch_check_selftest(Control *ctl, cudaStream_t stream);      // one failing WOLFF_CHECK (code 99)
#endif
cudaError_t launch_init_lattice(int8_t *spins, uint32_t N, uint64_t seed, int num_sms, cudaStream_t stream);
cudaError_t launch_validate(const int8_t *spins, uint32_t N, Control *ctl, int num_sms, cudaStream_t stream);
// n_bytes spins (16-byte aligned buffer) are all +1 / -1, else *invalid |= 1
cudaError_t launch_validate_word(const int8_t *spins, size_t n_bytes, unsigned int *invalid, int num_sms, cudaStream_t stream);
// E and M of the lattice into ctl->E, ctl->M and, when not null, into the DEVICE words E_dst, M_dst
cudaError_t launch_energy_magnetisation(const int8_t *spins, const Geometry &geo, int dim, Control *ctl,
                                        long long *E_dst, long long *M_dst, int num_sms, cudaStream_t stream);

}  // namespace wolff
