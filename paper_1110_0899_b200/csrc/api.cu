// api.cu -- the extern "C" boundary declared in include/wolff.h (host side only).
#include <cmath>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <new>

#include "../../include/wolff.h"
#include "internal.h"

using namespace wolff;

namespace {

thread_local char g_error[512] = "";

void set_error(const char *fmt, ...) __attribute__((format(printf, 1, 2)));
void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_error, sizeof(g_error), fmt, ap);
    va_end(ap);
}

}  // namespace

namespace wolff {
void set_error_v(const char *fmt, va_list ap) { vsnprintf(g_error, sizeof(g_error), fmt, ap); }
uint64_t bond_threshold(double J, double T);
}

struct wolff_ctx {
    int dim = 0, L = 0;
    double J = 0, T = 0;
    uint64_t seed = 0;
    uint64_t N = 0;
    uint64_t thr = 0;
    uint64_t u = 0;                 // next update index
    int device = 0;
    int num_sms = 0;
    Geometry geo{};
    int8_t *spins = nullptr;
    uint32_t *clist = nullptr;
    uint32_t *sizes = nullptr;
    uint32_t *ns_log = nullptr;     // per-update duration of the most recent run
    long long *E_log = nullptr;     // per-update E, M of the most recent run ("measure" = 1)
    long long *M_log = nullptr;
    uint64_t sizes_cap = 0;         // entries allocated in the size and duration logs
    uint64_t em_cap = 0;            // entries allocated in E_log and M_log (allocated by the first measured run)
    uint64_t meas_count = 0;        // samples in the moment accumulators (host-side count, for the overflow bound)
    int measure = 0;                // in-kernel measurement after every update
    bool last_measured = false;     // the most recent run was a measured one
    bool em_valid = false;          // the control block holds E and M of the current lattice
    uint64_t last_n = 0;            // updates in the most recent wolff_run
    Control *ctl = nullptr;
    cudaStream_t last_stream = nullptr;
    bool cuda_failed = false;
    bool ran = false;
    // knobs
    int mode = 0;
    uint32_t qcap = 0;
    uint32_t up = 0, down = 0;      // one CTA <-> cluster
    uint32_t cl_up = 0, grid_down = 0;   // cluster <-> grid
    uint32_t bal_min = 0;
    int grid_ctas = 0;              // requested total CTAs, 0 = as many clusters as fit
    int cluster_ctas = 0;           // CTAs per cluster
    int cooperative = 1;
    int spec = 0;                   // speculative claims (no neighbour gather)
    // launch shape derived from the knobs (recomputed when shape_dirty)
    bool shape_dirty = true;
    int max_clusters = 0;           // co-resident limit for this cluster size
    size_t smem_bytes = 0;
    // shared-memory-resident kernel (growth_tiles.cu): knobs, plan, and the device state that goes with the plan
    int tile_log_opt = 0;           // 0 = auto
    int tile_ctas_opt = 0;          // 0 = one CTA per SM
    uint32_t ring_cap = 2048;
    int inbox_log_opt = 0;          // 0 = auto: what one update can send at most (no capacity checks)
    int fill_mode = 1;              // bond tables: 0 off, 1 adaptive, 2 always
    uint64_t fill_min_us = 30;
    int fill_bufs = 0;              // 0 = two buffers when they fit, else one; 1 = one
    uint64_t watchdog_ms = 20000;
    uint32_t idle_ns = 1000;
    size_t smem_optin = 0;          // shared memory one CTA may use
    bool plan_dirty = true;
    bool plan_ok = false;
    TileParams tp{};
    size_t tile_smem = 0;
    unsigned long long *tile_inbox = nullptr;
    unsigned long long *tile_ctr = nullptr;     // gtail[G], gdone[G], gspill[G], added
    uint32_t *tile_spill = nullptr;
    uint32_t *tile_fill = nullptr;
    int8_t *tile_faces = nullptr;   // in-kernel measurement: the low faces of every tile
    // cluster-resident bit-packed kernel (growth_cluster.cu): plan and the device state that goes with it
    int resident_ctas = 16;         // largest cluster the plan may use
    bool cl_dirty = true;
    bool cl_ok = false;
    ClusterParams cp{};
    size_t cl_smem = 0;
    uint32_t *cl_spill = nullptr;
    unsigned long long *cl_spill_ctr = nullptr;
    // kernel choice in mode 0: mean cluster size of the last finished run (read when the caller next synchronises)
    uint64_t small_cluster = 32768; // below this mean size mode 0 leaves the kernel of all SMs for the cluster-resident one; 0 = never
                                    // (set by wolff_create: 8192 in 2D, 32768 in 3D)
    bool have_mean = false;
    bool run_since_set = false;     // a run has been queued since the lattice was last loaded: its counters describe this lattice
    double mean_cluster = 0.0;
};

namespace {

int fail_cuda(wolff_ctx *h, cudaError_t e, const char *what)
{
    set_error("%s: %s", what, cudaGetErrorString(e));
    if (h) h->cuda_failed = true;
    return WOLFF_ECUDA;
}

#define CHECK_CUDA(h, call, what)                                   \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return fail_cuda((h), e_, (what));   \
    } while (0)

// Makes the handle's device current for the length of one API call and puts the caller's device back afterwards
// (work the caller issues next on this thread must not land on another GPU).
class DeviceScope {
public:
    explicit DeviceScope(const wolff_ctx *h)
    {
        if (!h) return;
        if (cudaGetDevice(&prev_) != cudaSuccess) { cudaGetLastError(); prev_ = -1; }
        if (prev_ != h->device) { cudaSetDevice(h->device); switched_ = true; }
    }
    ~DeviceScope() { if (switched_ && prev_ >= 0) cudaSetDevice(prev_); }
    DeviceScope(const DeviceScope &) = delete;
    DeviceScope &operator=(const DeviceScope &) = delete;
private:
    int prev_ = -1;
    bool switched_ = false;
};

int check_handle(wolff_ctx *h)
{
    if (!h) { set_error("null handle"); return WOLFF_EINVAL; }
    if (h->cuda_failed) { set_error("handle is in a failed CUDA state"); return WOLFF_ECUDA; }
    return WOLFF_OK;
}

}  // namespace

// Reading R7: p = -expm1(-2J/T) in IEEE double, thr = floor(p * 2^32) in [0, 2^32].
uint64_t wolff::bond_threshold(double J, double T)
{
    const double p = -std::expm1(-2.0 * J / T);
    if (!(p > 0.0)) return 0;
    const double scaled = std::floor(std::ldexp(p, 32));
    if (scaled >= 4294967296.0) return 4294967296ull;
    return (uint64_t)scaled;
}

namespace {

uint32_t cta_capacity(const wolff_ctx *h) { return h->qcap / (2u * (uint32_t)h->dim); }   // next level must fit one buffer
uint32_t cluster_capacity(const wolff_ctx *h) { return (uint32_t)h->cluster_ctas * (cta_capacity(h) & ~31u); }

void effective_thresholds(const wolff_ctx *h, GrowthParams *p)
{
    const uint32_t up_max = cta_capacity(h), cl_max = cluster_capacity(h);
    p->bal_min = h->bal_min;
    if (h->mode == 1) { p->up = p->down = p->cl_up = p->grid_down = 0; return; }      // every level grid-wide
    uint32_t up = h->up < up_max ? h->up : up_max;
    uint32_t down = h->down < up ? h->down : up;
    uint32_t cl_up = h->cl_up < cl_max ? h->cl_up : cl_max;
    if (h->mode == 2) { up = up_max; down = up_max; }                                 // one CTA whenever it fits
    if (h->mode == 3) { up = 0; down = 0; cl_up = cl_max; }                           // the cluster whenever it fits
    p->up = up; p->down = down; p->cl_up = cl_up;
    p->grid_down = h->grid_down < cl_up ? h->grid_down : cl_up;
}

// (Re)derive the launch shape from the knobs: kernel attributes and the co-resident cluster limit.
int refresh_shape(wolff_ctx *h)
{
    if (!h->shape_dirty) return WOLFF_OK;
    GrowthLaunch l{h->cluster_ctas, h->cluster_ctas, h->smem_bytes, h->cooperative != 0, h->spec != 0};
    int clusters = 0;
    cudaError_t e = growth_max_clusters(h->dim, h->geo.pow2 != 0, l, &clusters);
    if (e != cudaSuccess || clusters < 1) {
        cudaGetLastError();
        set_error("growth kernel cannot be made resident with clusters of %d CTAs: %s", h->cluster_ctas,
                  e != cudaSuccess ? cudaGetErrorString(e) : "no cluster fits");
        return WOLFF_EINVAL;
    }
    h->max_clusters = clusters;
    h->shape_dirty = false;
    return WOLFF_OK;
}

void free_tile_state(wolff_ctx *h)
{
    cudaFree(h->tile_inbox); h->tile_inbox = nullptr;
    cudaFree(h->tile_ctr); h->tile_ctr = nullptr;
    cudaFree(h->tile_spill); h->tile_spill = nullptr;
    cudaFree(h->tile_fill); h->tile_fill = nullptr;
    cudaFree(h->tile_faces); h->tile_faces = nullptr;
}

uint32_t ceil_log2(uint64_t v) { uint32_t l = 0; while ((1ull << l) < v) ++l; return l; }

void free_cluster_state(wolff_ctx *h)
{
    cudaFree(h->cl_spill); h->cl_spill = nullptr;
    cudaFree(h->cl_spill_ctr); h->cl_spill_ctr = nullptr;
}

// (Re)derive the launch shape of growth_cluster.cu: the largest cluster (at most "cluster_ctas" CTAs) whose CTAs each
// hold a power-of-two number of 32-bit words of the bit lattice, the ring and the stages in their shared memory.
// cl_ok == false (the lattice does not fit one cluster: more than 2^24 spins) is not an error.
int refresh_cluster_plan(wolff_ctx *h, cudaStream_t stream)
{
    if (!h->cl_dirty) return WOLFF_OK;
    if (h->ran) CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    free_cluster_state(h);
    h->cl_ok = false;
    h->cl_dirty = false;
    ClusterParams &cp = h->cp;
    size_t smem = 0;
    if (!cluster_plan(h->dim, h->geo, h->resident_ctas, h->ring_cap, h->smem_optin, &cp, &smem, nullptr)) return WOLFF_OK;
    cp.watchdog_ns = h->watchdog_ms * 1000000ull;
    cp.thr32 = (uint32_t)h->thr;
    cp.thr_all = (h->thr >> 32) != 0 ? 1u : 0u;
    cp.idle_ns = h->idle_ns;
    h->cl_smem = smem;
    const size_t spill_bytes = ((size_t)1 << cp.spill_log) * sizeof(uint32_t);
    if (cudaMalloc(&h->cl_spill, spill_bytes) != cudaSuccess || cudaMalloc(&h->cl_spill_ctr, 2 * sizeof(unsigned long long)) != cudaSuccess) {
        cudaGetLastError();
        free_cluster_state(h);
        return WOLFF_OK;
    }
    CHECK_CUDA(h, cudaMemsetAsync(h->cl_spill, 0, spill_bytes, stream), "clear spill list");
    CHECK_CUDA(h, cudaMemsetAsync(h->cl_spill_ctr, 0, 2 * sizeof(unsigned long long), stream), "clear spill counters");
    cp.spill = h->cl_spill;
    cp.spill_ctr = h->cl_spill_ctr;
    h->cl_ok = true;
    return WOLFF_OK;
}

// (Re)derive the tiling of growth_tiles.cu from the knobs and allocate its inboxes, spill lists and counters.
// plan_ok == false (L not a power of two, L < 4, or the lattice does not fit the chip's shared memory) is not an
// error: wolff_run then uses the level-synchronous kernel of growth.cu.
int refresh_plan(wolff_ctx *h, cudaStream_t stream)
{
    if (!h->plan_dirty) return WOLFF_OK;
    if (h->ran) CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    free_tile_state(h);
    h->plan_ok = false;
    h->plan_dirty = false;
    if (!h->geo.pow2 || h->L < 4) return WOLFF_OK;
    const uint32_t dim = (uint32_t)h->dim, logL = h->geo.logL;
    uint32_t b = h->tile_log_opt > 0 ? (uint32_t)h->tile_log_opt : (dim == 2 ? 6u : 4u);
    if (b > logL) b = logL;
    const uint64_t ntiles = 1ull << (dim * (logL - b));
    if (ntiles > (1ull << 24)) return WOLFF_OK;
    uint32_t G = (uint32_t)h->num_sms;
    if (h->tile_ctas_opt > 0 && (uint32_t)h->tile_ctas_opt < G) G = (uint32_t)h->tile_ctas_opt;
    if (ntiles < G) G = (uint32_t)ntiles;
    const uint32_t slots = (uint32_t)((ntiles + G - 1) / G);
    if (slots > 0xFFFFu || G > 0xFFFFu) return WOLFF_OK;
    // bond tables (growth_tiles.cu) when they fit beside the lattice; a tile must hold at least one 32-bit word of bonds
    uint32_t nbuf = (h->fill_mode != 0 && dim * b >= 5u) ? (h->fill_bufs == 1 ? 1u : 2u) : 0u;
    size_t smem = tiles_smem_bytes(h->dim, b, slots, h->ring_cap, nbuf);
    while (nbuf > 0 && smem + 256 > h->smem_optin) { --nbuf; smem = tiles_smem_bytes(h->dim, b, slots, h->ring_cap, nbuf); }
    if (smem + 256 > h->smem_optin) return WOLFF_OK;
    const bool tables = nbuf != 0;
    int per_sm = 0;
    cudaError_t e = tiles_prepare(h->dim, smem, &per_sm);
    if (e != cudaSuccess || per_sm < 1) { cudaGetLastError(); return WOLFF_OK; }

    TileParams &tp = h->tp;
    tp = TileParams{};
    tp.tile_log = b;
    tp.ntiles = (uint32_t)ntiles;
    tp.permA = (0x9E3779B1u & (uint32_t)(ntiles - 1)) | 1u;
    uint32_t inv = tp.permA;                      // Newton iteration for the inverse of an odd number mod 2^32
    for (int it = 0; it < 5; ++it) inv *= 2u - tp.permA * inv;
    tp.permAinv = inv & (uint32_t)(ntiles - 1);
    tp.G = G;
    tp.magicG = ((1ull << 40) + G - 1) / G;
    tp.slots = slots;
    // Inbox of a CTA: by default what one update can send it at most (every bond across the surface of its tiles once,
    // the seed, the control messages), so nothing can overflow and senders check nothing.  Knob "inbox_log": a smaller
    // inbox; senders then check the capacity before each store and wait for the receiver, which never waits for anybody
    // (the check costs throughput; the size of the inboxes does not: growth_tiles.cu, run_passes).
    const uint64_t surface = (uint64_t)slots * 2ull * dim * (1ull << ((dim - 1) * b));
    tp.in_log = ceil_log2(surface + 4);
    if (tp.in_log < 5u) tp.in_log = 5u;              // the receiver looks at 32 slots at a time
    tp.bp = 0u;
    if (h->inbox_log_opt > 0 && (uint32_t)h->inbox_log_opt < tp.in_log) { tp.in_log = (uint32_t)h->inbox_log_opt; tp.bp = 1u; }
    tp.in_cap = 1u << tp.in_log;
    tp.spill_log = ceil_log2((uint64_t)slots << (dim * b));
    tp.ring_cap = h->ring_cap;
    tp.watchdog_ns = h->watchdog_ms * 1000000ull;
    tp.idle_ns = h->idle_ns;
    tp.tables = tables ? 1u : 0u;
    tp.nbuf = nbuf;
    tp.fill_mode = tables ? (uint32_t)h->fill_mode : 0u;
    tp.fill_min_ns = h->fill_min_us * 1000ull;
    tp.thr32 = (uint32_t)h->thr;
    tp.thr_all = (h->thr >> 32) != 0 ? 1u : 0u;
    h->tile_smem = smem;

    const size_t inbox_bytes = ((size_t)G << tp.in_log) * sizeof(unsigned long long);
    const size_t ctr_bytes = (4 * (size_t)G + 1) * sizeof(unsigned long long);
    const size_t spill_bytes = ((size_t)G << tp.spill_log) * sizeof(uint32_t);
    // one byte per site of the dim low faces of every tile (indexed by slot * G + owner: slots * G tiles at most)
    const size_t faces_bytes = (size_t)slots * G * dim * ((size_t)1 << ((dim - 1) * b)) + 16;
    if (cudaMalloc(&h->tile_inbox, inbox_bytes) != cudaSuccess || cudaMalloc(&h->tile_ctr, ctr_bytes) != cudaSuccess ||
        cudaMalloc(&h->tile_spill, spill_bytes) != cudaSuccess || cudaMalloc(&h->tile_fill, (size_t)G * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&h->tile_faces, faces_bytes) != cudaSuccess) {
        cudaGetLastError();
        free_tile_state(h);
        return WOLFF_OK;      // not enough memory for the tiled kernel's queues: the level-synchronous kernel needs none
    }
    // cleared on the stream the kernel is about to be launched on: nothing else on the device has to wait
    CHECK_CUDA(h, cudaMemsetAsync(h->tile_inbox, 0, inbox_bytes, stream), "clear inboxes");
    CHECK_CUDA(h, cudaMemsetAsync(h->tile_ctr, 0, ctr_bytes, stream), "clear counters");
    CHECK_CUDA(h, cudaMemsetAsync(h->tile_spill, 0, spill_bytes, stream), "clear spill lists");
    CHECK_CUDA(h, cudaMemsetAsync(h->tile_fill, 0, (size_t)G * sizeof(uint32_t), stream), "clear fill flags");
    tp.inbox = h->tile_inbox;
    tp.gtail = reinterpret_cast<unsigned int *>(h->tile_ctr);      // G 32-bit counters in the first G 64-bit words
    tp.gdone = h->tile_ctr + G;
    tp.gspill = h->tile_ctr + 2 * (size_t)G;
    tp.gihead = reinterpret_cast<unsigned int *>(h->tile_ctr + 3 * (size_t)G);   // G 32-bit words
    tp.added = h->tile_ctr + 4 * (size_t)G;
    tp.spill = h->tile_spill;
    tp.gfill = h->tile_fill;
    tp.faces = h->tile_faces;
    h->plan_ok = true;
    return WOLFF_OK;
}

// What the host needs from the control block after a run, read in one copy.
int read_control(wolff_ctx *h, Control *host, cudaStream_t s)
{
    CHECK_CUDA(h, cudaMemcpyAsync(host, h->ctl, sizeof(Control), cudaMemcpyDeviceToHost, s), "read control block");
    CHECK_CUDA(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    return WOLFF_OK;
}

// After a synchronise: the sticky device error flag and the counters of the last run.
int digest_control(wolff_ctx *h, const Control &c)
{
    if (!h->ran) return WOLFF_OK;
    if (c.error != 0) {
        if (c.error >= 1000u) set_error("checked build: index out of bounds in a growth kernel (code %u)", c.error - 1000u);
        else set_error("device watchdog: an update or a grid barrier did not complete (error flag %u)", c.error);
        h->cuda_failed = true;
        return WOLFF_EINTERNAL;
    }
    if (c.stats[0] > 0 && h->run_since_set) { h->have_mean = true; h->mean_cluster = (double)c.stats[1] / (double)c.stats[0]; }
    return WOLFF_OK;
}

int sync_and_check(wolff_ctx *h)
{
    if (!h->ran) {
        CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
        return WOLFF_OK;
    }
    Control c;
    const int rc = read_control(h, &c, h->last_stream);
    return rc ? rc : digest_control(h, c);
}

}  // namespace

extern "C" {

const char *wolff_last_error(void) { return g_error; }

wolff_handle wolff_create(int dim, int L, double J, double T, uint64_t seed)
{
    if (dim != 2 && dim != 3) { set_error("dim must be 2 or 3 (got %d)", dim); return nullptr; }
    if (L < 2) { set_error("L must be >= 2 (got %d)", L); return nullptr; }
    if (!(J >= 0.0) || !std::isfinite(J)) { set_error("J must be finite and >= 0"); return nullptr; }
    if (!(T > 0.0) || !std::isfinite(T)) { set_error("T must be finite and > 0"); return nullptr; }
    uint64_t N = 1;
    for (int k = 0; k < dim; ++k) {
        N *= (uint64_t)L;
        if (N > (1ull << 31)) { set_error("N = L^dim exceeds 2^31"); return nullptr; }
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        set_error("no usable CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
        return nullptr;
    }
    wolff_ctx *h = new (std::nothrow) wolff_ctx();
    if (!h) { set_error("out of host memory"); return nullptr; }
    h->dim = dim; h->L = L; h->J = J; h->T = T; h->seed = seed; h->N = N;
    h->thr = bond_threshold(J, T);
    h->small_cluster = dim == 2 ? 8192 : 32768;     // measured crossover of the two barrier-free kernels
    h->geo.L = (uint32_t)L;
    h->geo.N = (uint32_t)N;
    h->geo.LL = (uint32_t)((uint64_t)L * (uint64_t)L);
    h->geo.pow2 = ((L & (L - 1)) == 0) ? 1u : 0u;
    h->geo.logL = 0;
    if (h->geo.pow2) while ((1u << h->geo.logL) < (uint32_t)L) ++h->geo.logL;

    cudaDeviceProp prop{};
    bool ok = cudaGetDevice(&h->device) == cudaSuccess && cudaGetDeviceProperties(&prop, h->device) == cudaSuccess;
    if (!ok) { set_error("cudaGetDeviceProperties failed"); delete h; return nullptr; }
    if (!prop.cooperativeLaunch) { set_error("device lacks cooperative launch"); delete h; return nullptr; }
    h->num_sms = prop.multiProcessorCount;
    h->smem_optin = prop.sharedMemPerBlockOptin;

    h->qcap = 16384;                      // entries per queue buffer: 2 x 64 KiB of shared memory per CTA
    h->smem_bytes = 2ull * h->qcap * sizeof(uint32_t);
    h->cluster_ctas = 16;
    h->up = 64; h->down = 24;
    h->cl_up = 32768; h->grid_down = 8192;
    h->bal_min = 64;
    if (refresh_shape(h) != WOLFF_OK) {
        // clusters of 16 need the non-portable size; fall back to the portable maximum
        h->cluster_ctas = 8;
        h->shape_dirty = true;
        if (refresh_shape(h) != WOLFF_OK) { delete h; return nullptr; }
    }

    // N spins padded to a multiple of 16 bytes; N list entries; control block
    const size_t lattice_bytes = (size_t)((N + 15ull) & ~15ull);
    if (cudaMalloc(&h->spins, lattice_bytes) != cudaSuccess || cudaMalloc(&h->clist, (size_t)N * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&h->ctl, sizeof(Control)) != cudaSuccess) {
        set_error("device allocation failed for N = %llu", (unsigned long long)N);
        wolff_destroy(h);
        return nullptr;
    }
    e = cudaMemset(h->ctl, 0, sizeof(Control));
    if (e == cudaSuccess) e = cudaMemset(h->spins, 0, lattice_bytes);
    if (e == cudaSuccess) e = launch_init_lattice(h->spins, h->geo.N, seed, h->num_sms, nullptr);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        set_error("lattice initialisation failed: %s", cudaGetErrorString(e));
        wolff_destroy(h);
        return nullptr;
    }
    return h;
}

int wolff_destroy(wolff_handle h)
{
    if (!h) return WOLFF_OK;
    DeviceScope scope(h);
    if (h->last_stream || h->ran) cudaStreamSynchronize(h->last_stream);
    cudaFree(h->spins);
    cudaFree(h->clist);
    cudaFree(h->sizes);
    cudaFree(h->ns_log);
    cudaFree(h->E_log);
    cudaFree(h->M_log);
    cudaFree(h->ctl);
    free_tile_state(h);
    free_cluster_state(h);
    delete h;
    return WOLFF_OK;
}

int wolff_run(wolff_handle h, uint64_t n_updates, void *cuda_stream)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (n_updates == 0) return WOLFF_OK;
    if (n_updates > (1ull << 32)) { set_error("n_updates too large for one call (max 2^32)"); return WOLFF_EINVAL; }
    if (h->ran && stream != h->last_stream) {
        // the size log and control block are about to be reused: finish the previous run first
        CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    }
    if (h->measure) {
        // the 128-bit accumulators are exact while samples * N^4 < 2^128 (sum M^4 is the largest; |M| <= N): any number of
        // samples up to N = 2^16, 2^32 at N = 2^24, 2^16 at N = 2^28, 16 at N = 2^31.  Beyond that they would wrap without
        // a trace (the oracle's wrap the same way, so no parity test could see it): refuse instead.
        const unsigned __int128 n2 = (unsigned __int128)h->N * h->N, n4 = n2 * n2;       // <= 2^124
        const unsigned __int128 limit = ~(unsigned __int128)0 / n4;
        if ((unsigned __int128)h->meas_count + n_updates > limit) {
            set_error("measured run refused: %llu + %llu samples of M^4 <= N^4 (N = %llu) would overflow the 128-bit moment "
                      "accumulators; call wolff_reset_moments first (or run with \"measure\" = 0)",
                      (unsigned long long)h->meas_count, (unsigned long long)n_updates, (unsigned long long)h->N);
            return WOLFF_EINVAL;
        }
    }
    if (n_updates > h->sizes_cap) {
        if (h->ran) CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
        uint64_t cap = h->sizes_cap ? h->sizes_cap : 1024;
        while (cap < n_updates) cap *= 2;
        uint32_t *fresh = nullptr, *fresh_ns = nullptr;
        if (cudaMalloc(&fresh, (size_t)cap * sizeof(uint32_t)) != cudaSuccess || cudaMalloc(&fresh_ns, (size_t)cap * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(fresh); cudaFree(fresh_ns);
            set_error("cannot allocate the per-update logs for %llu updates", (unsigned long long)n_updates);
            return WOLFF_ENOMEM;
        }
        cudaFree(h->sizes); cudaFree(h->ns_log);
        h->sizes = fresh; h->ns_log = fresh_ns;
        h->sizes_cap = cap;
    }
    if (h->measure && n_updates > h->em_cap) {
        // E and M after every update: 16 bytes per update, allocated only once a measured run asks for them
        if (h->ran) CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
        const uint64_t cap = h->sizes_cap;
        long long *fresh_E = nullptr, *fresh_M = nullptr;
        if (cudaMalloc(&fresh_E, (size_t)cap * sizeof(long long)) != cudaSuccess || cudaMalloc(&fresh_M, (size_t)cap * sizeof(long long)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(fresh_E); cudaFree(fresh_M);
            set_error("cannot allocate the per-update E / M logs for %llu updates", (unsigned long long)n_updates);
            return WOLFF_ENOMEM;
        }
        cudaFree(h->E_log); cudaFree(h->M_log);
        h->E_log = fresh_E; h->M_log = fresh_M;
        h->em_cap = cap;
    }
    GrowthParams p{};
    p.spins = h->spins; p.clist = h->clist; p.sizes = h->sizes; p.ctl = h->ctl; p.geo = h->geo;
    p.key0 = (uint32_t)h->seed; p.key1 = (uint32_t)(h->seed >> 32);
    p.thr = h->thr; p.u0 = h->u; p.n_updates = n_updates; p.qcap = h->qcap;
    p.measure = h->measure ? 1u : 0u;
    p.claim_bits = 0xFEu;
    p.E_log = h->E_log; p.M_log = h->M_log; p.ns_log = h->ns_log;
    // control words of the growth kernels start from zero at every launch (generation 0, no stats); the error flag
    // is not among them: it is sticky until the host has read it
    CHECK_CUDA(h, cudaMemsetAsync(h->ctl, 0, kControlClearBytes, stream), "cudaMemsetAsync(control)");
    if (h->mode == 0) {
        rc = refresh_plan(h, stream);
        if (rc) return rc;
    }
    // kernel choice in mode 0, by the mean cluster of the last finished run: below "small_cluster" spins the
    // cluster-resident kernel (its update costs what its few passes cost: no cooperative grid, no messages, no poll over
    // 148 CTAs), above it the shared-memory-resident kernel of all SMs; measured runs on clusters of a handful of spins go
    // to the level-synchronous kernel
    const bool small = h->small_cluster > 0 && h->have_mean && h->mean_cluster < (double)h->small_cluster;
    const bool tiny = small && h->mean_cluster < 16.0;
    bool clustered = false;
    // (a lattice the kernel of all SMs does not apply to -- L not a power of two -- runs here whatever its clusters)
    // (it measures inside the kernel when L is a multiple of 32; below 16 spins per cluster a measured run is cheaper on
    // the level-synchronous kernel, whose measurement costs what the cluster costs, not what the lattice costs)
    const bool cl_measures = h->L % 32 == 0;
    // (a launch of this kernel packs and unpacks the lattice with 16 SMs: 9 us + 50 us per 2^24 spins, against 11 us for a
    // launch of the level-synchronous kernel and 32 us for the kernel of all SMs.  A call of a few updates on a large
    // lattice -- the host loop run(1) + observables -- is therefore left to those two: fewer than N / 2^20 updates)
    const bool brief = n_updates < (h->N >> 20) && (tiny || h->plan_ok);
    if ((h->mode == 5 || (h->mode == 0 && (small || !h->plan_ok) && !(h->measure && tiny) && !brief)) && (!h->measure || cl_measures)) {
        rc = refresh_cluster_plan(h, stream);
        if (rc) return rc;
        clustered = h->cl_ok;
    }
    if (clustered) {
        // the monitor publishes the update index relative to the launch in 31 bits
        const uint64_t chunk = 1ull << 30;
        for (uint64_t done = 0; done < n_updates && clustered; done += chunk) {
            ClusterParams cp = h->cp;
            cp.g = p;
            cp.g.u0 = h->u + done;
            cp.g.n_updates = n_updates - done < chunk ? n_updates - done : chunk;
            cp.g.sizes = h->sizes + done;
            cp.g.ns_log = h->ns_log + done;
            cp.g.E_log = h->measure ? h->E_log + done : nullptr;
            cp.g.M_log = h->measure ? h->M_log + done : nullptr;
            if (h->measure && cp.idle_ns > 200u) cp.idle_ns = 200u;     // every warp of the cluster is waited for after each update
            const cudaError_t e = launch_growth_cluster(cp, h->dim, h->cl_smem, stream);
            if (e == cudaErrorLaunchOutOfResources || e == cudaErrorInvalidConfiguration || e == cudaErrorCooperativeLaunchTooLarge) {
                cudaGetLastError();       // the SMs of one GPC cannot be had right now: not a fault of the handle
                if (done == 0) { clustered = false; break; }
            }
            CHECK_CUDA(h, e, "launch cluster-resident growth kernel");
        }
    }
    if (h->mode == 5 && !clustered) {
        rc = refresh_plan(h, stream);
        if (rc) return rc;
    }
    bool tiled = !clustered && (h->mode == 0 || h->mode == 5) && h->plan_ok && !tiny;      // (tiny: the level-synchronous kernel)
    if (tiled) {
        // shared-memory-resident kernel; a message carries the update index relative to the launch in 29 bits
        const uint64_t chunk = (1ull << 29) - 1;
        for (uint64_t done = 0; done < n_updates && tiled; done += chunk) {
            TileParams tp = h->tp;
            tp.g = p;
            tp.g.u0 = h->u + done;
            tp.g.n_updates = n_updates - done < chunk ? n_updates - done : chunk;
            tp.g.sizes = h->sizes + done;
            tp.g.ns_log = h->ns_log + done;
            tp.g.E_log = h->measure ? h->E_log + done : nullptr;
            tp.g.M_log = h->measure ? h->M_log + done : nullptr;
            if (h->measure && tp.idle_ns > 200u) tp.idle_ns = 200u;     // every warp of every CTA is waited for after each update
            if (done != 0)        // the measurement's arrival counters count from zero in every launch
                CHECK_CUDA(h, cudaMemsetAsync(&h->ctl->meas_arrive_a, 0, offsetof(Control, error) - offsetof(Control, meas_arrive_a), stream),
                           "cudaMemsetAsync(measurement counters)");
            const cudaError_t e = launch_growth_tiles(tp, h->dim, h->tile_smem, stream);
            if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources || e == cudaErrorInvalidConfiguration) {
                // the SMs cannot all be had right now (another context holds some): not a fault of the handle.
                // Nothing has run when the first launch is refused, so the level-synchronous kernel takes the call.
                cudaGetLastError();
                if (done == 0) { tiled = false; break; }
            }
            CHECK_CUDA(h, e, "launch tiled growth kernel");
        }
    }
    if (!tiled && !clustered) {
        if (h->measure) {
            // the level-synchronous kernel keeps running E and M: it starts from a whole-lattice evaluation (into the
            // control block) and marks the members of the running cluster in the spin bytes (claim_with_bits)
            p.claim_bits = 0xFCu;
            if (!h->em_valid)
                CHECK_CUDA(h, launch_energy_magnetisation(h->spins, h->geo, h->dim, h->ctl, nullptr, nullptr, h->num_sms, stream),
                           "launch E/M reduction");
        }
        effective_thresholds(h, &p);
        rc = refresh_shape(h);
        if (rc) return rc;
        int clusters = h->grid_ctas > 0 ? h->grid_ctas / h->cluster_ctas : h->max_clusters;
        if (clusters > h->max_clusters) clusters = h->max_clusters;
        if (clusters < 1) clusters = 1;
        const GrowthLaunch shape{clusters * h->cluster_ctas, h->cluster_ctas, h->smem_bytes, h->cooperative != 0, h->spec != 0};
        CHECK_CUDA(h, launch_growth(p, h->dim, shape, stream), "launch growth kernel");
    }
    h->u += n_updates;
    h->last_n = n_updates;
    h->last_measured = h->measure != 0;
    if (h->measure) h->meas_count += n_updates;
    h->em_valid = h->measure != 0;      // a measured run leaves E and M of the final lattice in the control block
    h->last_stream = stream;
    h->ran = true;
    h->run_since_set = true;
    return WOLFF_OK;
}

int wolff_observables(wolff_handle h, int64_t *E, int64_t *M, uint32_t *cluster_sizes)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    cudaStream_t s = h->last_stream;
    // Everything is queued behind the last run on its stream.  E and M: a destination in device memory is written by
    // the reduction kernel itself (its last CTA); a host destination is filled from the ONE small device-to-host copy
    // that also brings the error flag and the run's counters.  One synchronise ends the call.
    long long *dev_dst[2] = {nullptr, nullptr};
    int64_t *const dst[2] = {E, M};
    for (int k = 0; k < 2; ++k) {
        if (!dst[k]) continue;
        cudaPointerAttributes attr{};
        const cudaError_t e = cudaPointerGetAttributes(&attr, dst[k]);
        if (e != cudaSuccess) cudaGetLastError();
        if (e == cudaSuccess && (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged))
            dev_dst[k] = reinterpret_cast<long long *>(dst[k]);
    }
    if (E || M) {
        CHECK_CUDA(h, launch_energy_magnetisation(h->spins, h->geo, h->dim, h->ctl, dev_dst[0], dev_dst[1], h->num_sms, s),
                   "launch E/M reduction");
        h->em_valid = true;
    }
    if (cluster_sizes && h->last_n > 0)
        CHECK_CUDA(h, cudaMemcpyAsync(cluster_sizes, h->sizes, (size_t)h->last_n * sizeof(uint32_t), cudaMemcpyDefault, s),
                   "copy cluster sizes");
    Control c;
    rc = read_control(h, &c, s);
    if (rc) return rc;
    rc = digest_control(h, c);
    if (rc) return rc;
    for (int k = 0; k < 2; ++k)
        if (dst[k] && !dev_dst[k]) *dst[k] = (int64_t)(k == 0 ? c.E : c.M);
    return WOLFF_OK;
}

int wolff_get_spins(wolff_handle h, int8_t *dst)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    if (!dst) { set_error("dst is NULL"); return WOLFF_EINVAL; }
    rc = sync_and_check(h);
    if (rc) return rc;
    CHECK_CUDA(h, cudaMemcpyAsync(dst, h->spins, (size_t)h->N, cudaMemcpyDefault, h->last_stream), "copy lattice out");
    CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    return WOLFF_OK;
}

int wolff_set_spins(wolff_handle h, const int8_t *src)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    if (!src) { set_error("src is NULL"); return WOLFF_EINVAL; }
    rc = sync_and_check(h);
    if (rc) return rc;
    cudaStream_t s = h->last_stream;
    // stage in the cluster list (N * 4 bytes, idle between runs), validate there, then commit
    int8_t *staging = reinterpret_cast<int8_t *>(h->clist);
    CHECK_CUDA(h, cudaMemcpyAsync(staging, src, (size_t)h->N, cudaMemcpyDefault, s), "copy lattice in");
    CHECK_CUDA(h, cudaMemsetAsync(&h->ctl->invalid, 0, sizeof(unsigned int), s), "reset validation flag");
    CHECK_CUDA(h, launch_validate(staging, h->geo.N, h->ctl, h->num_sms, s), "launch validation");
    unsigned int invalid = 0;
    CHECK_CUDA(h, cudaMemcpyAsync(&invalid, &h->ctl->invalid, sizeof(invalid), cudaMemcpyDeviceToHost, s), "read validation flag");
    CHECK_CUDA(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    if (invalid) { set_error("set_spins: every byte must be +1 or -1"); return WOLFF_EINVAL; }
    CHECK_CUDA(h, cudaMemcpyAsync(h->spins, staging, (size_t)h->N, cudaMemcpyDeviceToDevice, s), "commit lattice");
    h->em_valid = false;
    h->have_mean = false;           // a new lattice: nothing is known about its clusters
    h->run_since_set = false;
    CHECK_CUDA(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    return WOLFF_OK;
}

int wolff_get_state(wolff_handle h, uint64_t *update_index, uint64_t *threshold)
{
    if (!h) { set_error("null handle"); return WOLFF_EINVAL; }
    if (update_index) *update_index = h->u;
    if (threshold) *threshold = h->thr;
    return WOLFF_OK;
}

int wolff_set_update_index(wolff_handle h, uint64_t update_index)
{
    if (!h) { set_error("null handle"); return WOLFF_EINVAL; }
    h->u = update_index;
    return WOLFF_OK;
}

int wolff_set_option(wolff_handle h, const char *key, int64_t value)
{
    if (!h || !key) { set_error("null handle or key"); return WOLFF_EINVAL; }
    DeviceScope scope(h);
    const uint32_t up_max = cta_capacity(h);
    if (!strcmp(key, "mode")) {
        if (value < 0 || value > 5) { set_error("mode must be 0, 1, 2, 3, 4 or 5"); return WOLFF_EINVAL; }
        h->mode = (int)value;
    } else if (!strcmp(key, "tile_log")) {
        if (value != 0 && (value < 2 || value > 12)) { set_error("tile_log must be 0 (auto) or in [2, 12]"); return WOLFF_EINVAL; }
        h->tile_log_opt = (int)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "tile_ctas")) {
        if (value < 0 || value > 1 << 16) { set_error("tile_ctas must be in [0, 65536]"); return WOLFF_EINVAL; }
        h->tile_ctas_opt = (int)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "watchdog_ms")) {
        if (value < 1 || value > 3600000) { set_error("watchdog_ms must be in [1, 3600000]"); return WOLFF_EINVAL; }
        h->watchdog_ms = (uint64_t)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "small_cluster")) {
        if (value < 0 || value > (int64_t)0x7FFFFFFF) { set_error("small_cluster must be in [0, 2^31)"); return WOLFF_EINVAL; }
        h->small_cluster = (uint64_t)value;
    } else if (!strcmp(key, "fill")) {
        if (value < 0 || value > 2) { set_error("fill must be 0 (never), 1 (adaptive) or 2 (always)"); return WOLFF_EINVAL; }
        h->fill_mode = (int)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "fill_bufs")) {
        if (value < 0 || value > 2) { set_error("fill_bufs must be 0 (auto), 1 or 2"); return WOLFF_EINVAL; }
        h->fill_bufs = (int)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "fill_min_us")) {
        if (value < 0 || value > 1000000) { set_error("fill_min_us must be in [0, 1000000]"); return WOLFF_EINVAL; }
        h->fill_min_us = (uint64_t)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "idle_ns")) {
        if (value < 0 || value > 1000000) { set_error("idle_ns must be in [0, 1000000]"); return WOLFF_EINVAL; }
        h->idle_ns = (uint32_t)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "ring_cap")) {
        if (value < 32 || value > 32768 || (value & (value - 1)) != 0) { set_error("ring_cap must be a power of two in [32, 32768]"); return WOLFF_EINVAL; }
        h->ring_cap = (uint32_t)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "measure")) {
        if (value != 0 && value != 1) { set_error("measure must be 0 or 1"); return WOLFF_EINVAL; }
        h->measure = (int)value;
    } else if (!strcmp(key, "inbox_log")) {
        if (value != 0 && (value < 5 || value > 24)) { set_error("inbox_log must be 0 (auto) or in [5, 24]"); return WOLFF_EINVAL; }
        h->inbox_log_opt = (int)value;
        h->plan_dirty = h->cl_dirty = true;
    } else if (!strcmp(key, "up_threshold")) {
        if (value < 0 || value > (int64_t)up_max) { set_error("up_threshold must be in [0, %u]", up_max); return WOLFF_EINVAL; }
        h->up = (uint32_t)value;
    } else if (!strcmp(key, "down_threshold")) {
        if (value < 0 || value > (int64_t)up_max) { set_error("down_threshold must be in [0, %u]", up_max); return WOLFF_EINVAL; }
        h->down = (uint32_t)value;
    } else if (!strcmp(key, "cluster_up_threshold")) {
        if (value < 0 || value > (int64_t)0x7FFFFFFF) { set_error("cluster_up_threshold must be in [0, 2^31)"); return WOLFF_EINVAL; }
        h->cl_up = (uint32_t)value;
    } else if (!strcmp(key, "grid_down_threshold")) {
        if (value < 0 || value > (int64_t)0x7FFFFFFF) { set_error("grid_down_threshold must be in [0, 2^31)"); return WOLFF_EINVAL; }
        h->grid_down = (uint32_t)value;
    } else if (!strcmp(key, "balance_min")) {
        if (value < 0 || value > (int64_t)0x7FFFFFFF) { set_error("balance_min must be in [0, 2^31)"); return WOLFF_EINVAL; }
        h->bal_min = (uint32_t)value;
    } else if (!strcmp(key, "grid_ctas")) {
        if (value < 0 || value > 1 << 20) { set_error("grid_ctas must be in [0, 2^20]"); return WOLFF_EINVAL; }
        h->grid_ctas = (int)value;
    } else if (!strcmp(key, "cluster_ctas")) {
        if (value != 1 && value != 2 && value != 4 && value != 8 && value != 16) {
            set_error("cluster_ctas must be 1, 2, 4, 8 or 16");
            return WOLFF_EINVAL;
        }
        const int before = h->cluster_ctas;
        h->cluster_ctas = (int)value;
        h->shape_dirty = true;
        if (refresh_shape(h) != WOLFF_OK) {
            h->cluster_ctas = before;
            h->shape_dirty = true;
            return WOLFF_EINVAL;
        }
    } else if (!strcmp(key, "resident_ctas")) {
        if (value != 1 && value != 2 && value != 4 && value != 8 && value != 16) {
            set_error("resident_ctas must be 1, 2, 4, 8 or 16");
            return WOLFF_EINVAL;
        }
        h->resident_ctas = (int)value;
        h->cl_dirty = true;
    } else if (!strcmp(key, "speculative")) {
        if (value != 0 && value != 1) { set_error("speculative must be 0 or 1"); return WOLFF_EINVAL; }
        h->spec = (int)value;
        h->shape_dirty = true;
        if (refresh_shape(h) != WOLFF_OK) return WOLFF_EINVAL;
    } else if (!strcmp(key, "cooperative")) {
        if (value != 0 && value != 1) { set_error("cooperative must be 0 or 1"); return WOLFF_EINVAL; }
        h->cooperative = (int)value;
#ifdef WOLFF_CHECKED
    } else if (!strcmp(key, "check_selftest")) {
        // checked builds only: one failing WOLFF_CHECK on the handle's control block, so that a test can see that the checks
        // are compiled in and that a violation reaches the caller (WOLFF_EINTERNAL at the next synchronising call)
        h->ran = true;
        CHECK_CUDA(h, launch_check_selftest(h->ctl, h->last_stream), "launch check self-test");
#endif
    } else {
        set_error("unknown option '%s'", key);
        return WOLFF_EINVAL;
    }
    return WOLFF_OK;
}

int wolff_get_series(wolff_handle h, int64_t *E_series, int64_t *M_series, uint32_t *update_ns)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    if ((E_series || M_series) && h->ran && !h->last_measured) {
        set_error("the most recent wolff_run was not a measured one (wolff_set_option \"measure\" = 1)");
        return WOLFF_EINVAL;
    }
    cudaStream_t s = h->last_stream;
    const size_t n = h->ran ? (size_t)h->last_n : 0;
    if (n) {
        if (E_series) CHECK_CUDA(h, cudaMemcpyAsync(E_series, h->E_log, n * sizeof(int64_t), cudaMemcpyDefault, s), "copy E series");
        if (M_series) CHECK_CUDA(h, cudaMemcpyAsync(M_series, h->M_log, n * sizeof(int64_t), cudaMemcpyDefault, s), "copy M series");
        if (update_ns) CHECK_CUDA(h, cudaMemcpyAsync(update_ns, h->ns_log, n * sizeof(uint32_t), cudaMemcpyDefault, s), "copy update times");
    }
    return sync_and_check(h);
}

int wolff_get_moments(wolff_handle h, uint64_t *moments, double *binder)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    Control c;
    rc = read_control(h, &c, h->last_stream);
    if (rc) return rc;
    rc = digest_control(h, c);
    if (rc) return rc;
    if (moments) memcpy(moments, c.moments, sizeof(c.moments));
    if (binder) {
        // Eq. 3: U = 1 - <M^4> / (3 <M^2>^2) = 1 - n S4 / (3 S2^2)
        const long double two64 = 18446744073709551616.0L;
        const long double n = (long double)c.moments[0];
        const long double s2 = (long double)c.moments[6] * two64 + (long double)c.moments[5];
        const long double s4 = (long double)c.moments[8] * two64 + (long double)c.moments[7];
        *binder = (c.moments[0] == 0 || s2 == 0.0L) ? std::nan("") : (double)(1.0L - (n * s4) / (3.0L * s2 * s2));
    }
    return WOLFF_OK;
}

int wolff_reset_moments(wolff_handle h)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    rc = sync_and_check(h);
    if (rc) return rc;
    CHECK_CUDA(h, cudaMemsetAsync(h->ctl->moments, 0, sizeof(h->ctl->moments), h->last_stream), "clear moments");
    CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    h->meas_count = 0;
    return WOLFF_OK;
}

int wolff_get_stats(wolff_handle h, uint64_t *stats)
{
    int rc = check_handle(h);
    DeviceScope scope(h);
    if (rc) return rc;
    if (!stats) { set_error("stats is NULL"); return WOLFF_EINVAL; }
    if (!h->ran) { memset(stats, 0, WOLFF_NSTATS * sizeof(uint64_t)); return WOLFF_OK; }
    Control c;
    rc = read_control(h, &c, h->last_stream);
    if (rc) return rc;
    rc = digest_control(h, c);
    if (rc) return rc;
    static_assert(sizeof(c.stats) == WOLFF_NSTATS * sizeof(uint64_t), "stats layout");
    memcpy(stats, c.stats, sizeof(c.stats));
    return WOLFF_OK;
}

}  // extern "C"
