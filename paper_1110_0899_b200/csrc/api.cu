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
    uint64_t sizes_cap = 0;         // entries allocated
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
    // kernel choice in mode 0: mean cluster size of the last finished run (read when the caller next synchronises)
    uint64_t small_cluster = 16;    // below this mean size the level-synchronous kernel runs (its fixed cost per update is lower); 0 = never
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

int check_handle(wolff_ctx *h)
{
    if (!h) { set_error("null handle"); return WOLFF_EINVAL; }
    if (h->cuda_failed) { set_error("handle is in a failed CUDA state"); return WOLFF_ECUDA; }
    cudaError_t e = cudaSetDevice(h->device);
    if (e != cudaSuccess) return fail_cuda(h, e, "cudaSetDevice");
    return WOLFF_OK;
}

// Reading R7: p = -expm1(-2J/T) in IEEE double, thr = floor(p * 2^32) in [0, 2^32].
uint64_t bond_threshold(double J, double T)
{
    const double p = -std::expm1(-2.0 * J / T);
    if (!(p > 0.0)) return 0;
    const double scaled = std::floor(std::ldexp(p, 32));
    if (scaled >= 4294967296.0) return 4294967296ull;
    return (uint64_t)scaled;
}

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
}

uint32_t ceil_log2(uint64_t v) { uint32_t l = 0; while ((1ull << l) < v) ++l; return l; }

// (Re)derive the tiling of growth_tiles.cu from the knobs and allocate its inboxes, spill lists and counters.
// plan_ok == false (L not a power of two, L < 4, or the lattice does not fit the chip's shared memory) is not an
// error: wolff_run then uses the level-synchronous kernel of growth.cu.
int refresh_plan(wolff_ctx *h)
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
    // messages one update can send to one CTA: every bond across the surface of its tiles once, the seed, the exit
    const uint64_t surface = (uint64_t)slots * 2ull * dim * (1ull << ((dim - 1) * b));
    tp.in_log = ceil_log2(surface + 4);
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
    const size_t ctr_bytes = (3 * (size_t)G + 1) * sizeof(unsigned long long);
    const size_t spill_bytes = ((size_t)G << tp.spill_log) * sizeof(uint32_t);
    if (cudaMalloc(&h->tile_inbox, inbox_bytes) != cudaSuccess || cudaMalloc(&h->tile_ctr, ctr_bytes) != cudaSuccess ||
        cudaMalloc(&h->tile_spill, spill_bytes) != cudaSuccess || cudaMalloc(&h->tile_fill, (size_t)G * sizeof(uint32_t)) != cudaSuccess) {
        cudaGetLastError();
        free_tile_state(h);
        return WOLFF_OK;      // not enough memory for the tiled kernel's queues: the level-synchronous kernel needs none
    }
    CHECK_CUDA(h, cudaMemset(h->tile_inbox, 0, inbox_bytes), "clear inboxes");
    CHECK_CUDA(h, cudaMemset(h->tile_ctr, 0, ctr_bytes), "clear counters");
    CHECK_CUDA(h, cudaMemset(h->tile_spill, 0, spill_bytes), "clear spill lists");
    CHECK_CUDA(h, cudaMemset(h->tile_fill, 0, (size_t)G * sizeof(uint32_t)), "clear fill flags");
    // The memsets above run on the legacy default stream; the kernel that uses these buffers may be launched on a
    // non-blocking stream, which does not wait for it: finish them here (a plan is made once per knob change).
    CHECK_CUDA(h, cudaDeviceSynchronize(), "cudaDeviceSynchronize");
    tp.inbox = h->tile_inbox;
    tp.gtail = reinterpret_cast<unsigned int *>(h->tile_ctr);      // G 32-bit counters in the first G 64-bit words
    tp.gdone = h->tile_ctr + G;
    tp.gspill = h->tile_ctr + 2 * (size_t)G;
    tp.added = h->tile_ctr + 3 * (size_t)G;
    tp.spill = h->tile_spill;
    tp.gfill = h->tile_fill;
    h->plan_ok = true;
    return WOLFF_OK;
}

int sync_and_check(wolff_ctx *h)
{
    CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    if (h->ran) {
        // error flag and the first two counters (updates, flipped spins) of the last run: 8 + 16 bytes behind one another
        struct { unsigned int error, pad; unsigned long long updates, flipped; } head;
        static_assert(offsetof(Control, stats) == offsetof(Control, error) + 8, "Control layout");
        CHECK_CUDA(h, cudaMemcpy(&head, &h->ctl->error, sizeof(head), cudaMemcpyDeviceToHost), "read error flag");
        if (head.error != 0) {
            set_error("device watchdog: a grid barrier did not complete (error flag %u)", head.error);
            h->cuda_failed = true;
            return WOLFF_EINTERNAL;
        }
        if (head.updates > 0 && h->run_since_set) { h->have_mean = true; h->mean_cluster = (double)head.flipped / (double)head.updates; }
    }
    return WOLFF_OK;
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
    if (e == cudaSuccess) e = launch_init_lattice(h->spins, h->geo.N, seed, nullptr);
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
    cudaSetDevice(h->device);
    if (h->last_stream || h->ran) cudaStreamSynchronize(h->last_stream);
    cudaFree(h->spins);
    cudaFree(h->clist);
    cudaFree(h->sizes);
    cudaFree(h->ctl);
    free_tile_state(h);
    delete h;
    return WOLFF_OK;
}

int wolff_run(wolff_handle h, uint64_t n_updates, void *cuda_stream)
{
    int rc = check_handle(h);
    if (rc) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (n_updates == 0) return WOLFF_OK;
    if (n_updates > (1ull << 32)) { set_error("n_updates too large for one call (max 2^32)"); return WOLFF_EINVAL; }
    if (h->ran && stream != h->last_stream) {
        // the size log and control block are about to be reused: finish the previous run first
        CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
    }
    if (n_updates > h->sizes_cap) {
        if (h->ran) CHECK_CUDA(h, cudaStreamSynchronize(h->last_stream), "cudaStreamSynchronize");
        uint64_t cap = h->sizes_cap ? h->sizes_cap : 1024;
        while (cap < n_updates) cap *= 2;
        uint32_t *fresh = nullptr;
        if (cudaMalloc(&fresh, (size_t)cap * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            set_error("cannot allocate the cluster-size log for %llu updates", (unsigned long long)n_updates);
            return WOLFF_ENOMEM;
        }
        cudaFree(h->sizes);
        h->sizes = fresh;
        h->sizes_cap = cap;
    }
    GrowthParams p{};
    p.spins = h->spins; p.clist = h->clist; p.sizes = h->sizes; p.ctl = h->ctl; p.geo = h->geo;
    p.key0 = (uint32_t)h->seed; p.key1 = (uint32_t)(h->seed >> 32);
    p.thr = h->thr; p.u0 = h->u; p.n_updates = n_updates; p.qcap = h->qcap;
    // control words of the growth kernels start from zero at every launch (generation 0, no error, no stats)
    CHECK_CUDA(h, cudaMemsetAsync(h->ctl, 0, offsetof(Control, acc_unequal), stream), "cudaMemsetAsync(control)");
    if (h->mode == 0) {
        rc = refresh_plan(h);
        if (rc) return rc;
    }
    const bool small = h->small_cluster > 0 && h->have_mean && h->mean_cluster < (double)h->small_cluster;
    if (h->mode == 0 && h->plan_ok && !small) {
        // shared-memory-resident kernel; a message carries the update index relative to the launch in 29 bits
        const uint64_t chunk = (1ull << 29) - 1;
        for (uint64_t done = 0; done < n_updates; done += chunk) {
            TileParams tp = h->tp;
            tp.g = p;
            tp.g.u0 = h->u + done;
            tp.g.n_updates = n_updates - done < chunk ? n_updates - done : chunk;
            tp.g.sizes = h->sizes + done;
            CHECK_CUDA(h, launch_growth_tiles(tp, h->dim, h->tile_smem, stream), "launch tiled growth kernel");
        }
    } else {
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
    h->last_stream = stream;
    h->ran = true;
    h->run_since_set = true;
    return WOLFF_OK;
}

int wolff_observables(wolff_handle h, int64_t *E, int64_t *M, uint32_t *cluster_sizes)
{
    int rc = check_handle(h);
    if (rc) return rc;
    cudaStream_t s = h->last_stream;
    // Everything is queued behind the last run on its stream; ONE small device-to-host copy then brings the error
    // flag, the run's first counters and E, M (they sit within 296 bytes of the control block), and one
    // synchronise ends the call.
    if (E || M) CHECK_CUDA(h, launch_energy_magnetisation(h->spins, h->geo, h->dim, h->ctl, h->num_sms, s), "launch E/M reduction");
    if (cluster_sizes && h->last_n > 0)
        CHECK_CUDA(h, cudaMemcpyAsync(cluster_sizes, h->sizes, (size_t)h->last_n * sizeof(uint32_t), cudaMemcpyDefault, s),
                   "copy cluster sizes");
    constexpr size_t span = offsetof(Control, M) + sizeof(long long) - offsetof(Control, error);
    unsigned char head[span];
    CHECK_CUDA(h, cudaMemcpyAsync(head, &h->ctl->error, span, cudaMemcpyDeviceToHost, s), "read control block");
    CHECK_CUDA(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    unsigned int err = 0;
    unsigned long long updates = 0, flipped = 0;
    long long Ev = 0, Mv = 0;
    memcpy(&err, head, sizeof(err));
    memcpy(&updates, head + (offsetof(Control, stats) - offsetof(Control, error)), sizeof(updates));
    memcpy(&flipped, head + (offsetof(Control, stats) - offsetof(Control, error)) + 8, sizeof(flipped));
    memcpy(&Ev, head + (offsetof(Control, E) - offsetof(Control, error)), sizeof(Ev));
    memcpy(&Mv, head + (offsetof(Control, M) - offsetof(Control, error)), sizeof(Mv));
    if (h->ran) {
        if (err != 0) {
            set_error("device watchdog: an update or a grid barrier did not complete (error flag %u)", err);
            h->cuda_failed = true;
            return WOLFF_EINTERNAL;
        }
        if (updates > 0 && h->run_since_set) { h->have_mean = true; h->mean_cluster = (double)flipped / (double)updates; }
    }
    // E and M go to host or device memory, whichever the caller passed
    int64_t *const dst[2] = {E, M};
    const long long val[2] = {Ev, Mv};
    const long long *const src[2] = {&h->ctl->E, &h->ctl->M};
    bool queued = false;
    for (int k = 0; k < 2; ++k) {
        if (!dst[k]) continue;
        cudaPointerAttributes attr{};
        const cudaError_t e = cudaPointerGetAttributes(&attr, dst[k]);
        if (e != cudaSuccess) cudaGetLastError();
        if (e == cudaSuccess && (attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged)) {
            CHECK_CUDA(h, cudaMemcpyAsync(dst[k], src[k], sizeof(int64_t), cudaMemcpyDeviceToDevice, s), "copy E/M");
            queued = true;
        } else {
            *dst[k] = (int64_t)val[k];
        }
    }
    if (queued) CHECK_CUDA(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    return WOLFF_OK;
}

int wolff_get_spins(wolff_handle h, int8_t *dst)
{
    int rc = check_handle(h);
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
    if (rc) return rc;
    if (!src) { set_error("src is NULL"); return WOLFF_EINVAL; }
    rc = sync_and_check(h);
    if (rc) return rc;
    cudaStream_t s = h->last_stream;
    // stage in the cluster list (N * 4 bytes, idle between runs), validate there, then commit
    int8_t *staging = reinterpret_cast<int8_t *>(h->clist);
    CHECK_CUDA(h, cudaMemcpyAsync(staging, src, (size_t)h->N, cudaMemcpyDefault, s), "copy lattice in");
    CHECK_CUDA(h, cudaMemsetAsync(&h->ctl->invalid, 0, sizeof(unsigned int), s), "reset validation flag");
    CHECK_CUDA(h, launch_validate(staging, h->geo.N, h->ctl, s), "launch validation");
    unsigned int invalid = 0;
    CHECK_CUDA(h, cudaMemcpyAsync(&invalid, &h->ctl->invalid, sizeof(invalid), cudaMemcpyDeviceToHost, s), "read validation flag");
    CHECK_CUDA(h, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    if (invalid) { set_error("set_spins: every byte must be +1 or -1"); return WOLFF_EINVAL; }
    CHECK_CUDA(h, cudaMemcpyAsync(h->spins, staging, (size_t)h->N, cudaMemcpyDeviceToDevice, s), "commit lattice");
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
    const uint32_t up_max = cta_capacity(h);
    if (!strcmp(key, "mode")) {
        if (value < 0 || value > 4) { set_error("mode must be 0, 1, 2, 3 or 4"); return WOLFF_EINVAL; }
        h->mode = (int)value;
    } else if (!strcmp(key, "tile_log")) {
        if (value != 0 && (value < 2 || value > 12)) { set_error("tile_log must be 0 (auto) or in [2, 12]"); return WOLFF_EINVAL; }
        h->tile_log_opt = (int)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "tile_ctas")) {
        if (value < 0 || value > 1 << 16) { set_error("tile_ctas must be in [0, 65536]"); return WOLFF_EINVAL; }
        h->tile_ctas_opt = (int)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "watchdog_ms")) {
        if (value < 1 || value > 3600000) { set_error("watchdog_ms must be in [1, 3600000]"); return WOLFF_EINVAL; }
        h->watchdog_ms = (uint64_t)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "small_cluster")) {
        if (value < 0 || value > (int64_t)0x7FFFFFFF) { set_error("small_cluster must be in [0, 2^31)"); return WOLFF_EINVAL; }
        h->small_cluster = (uint64_t)value;
    } else if (!strcmp(key, "fill")) {
        if (value < 0 || value > 2) { set_error("fill must be 0 (never), 1 (adaptive) or 2 (always)"); return WOLFF_EINVAL; }
        h->fill_mode = (int)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "fill_bufs")) {
        if (value < 0 || value > 2) { set_error("fill_bufs must be 0 (auto), 1 or 2"); return WOLFF_EINVAL; }
        h->fill_bufs = (int)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "fill_min_us")) {
        if (value < 0 || value > 1000000) { set_error("fill_min_us must be in [0, 1000000]"); return WOLFF_EINVAL; }
        h->fill_min_us = (uint64_t)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "idle_ns")) {
        if (value < 0 || value > 1000000) { set_error("idle_ns must be in [0, 1000000]"); return WOLFF_EINVAL; }
        h->idle_ns = (uint32_t)value;
        h->plan_dirty = true;
    } else if (!strcmp(key, "ring_cap")) {
        if (value < 32 || value > 32768 || (value & (value - 1)) != 0) { set_error("ring_cap must be a power of two in [32, 32768]"); return WOLFF_EINVAL; }
        h->ring_cap = (uint32_t)value;
        h->plan_dirty = true;
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
        if (check_handle(h) != WOLFF_OK || refresh_shape(h) != WOLFF_OK) {
            h->cluster_ctas = before;
            h->shape_dirty = true;
            return WOLFF_EINVAL;
        }
    } else if (!strcmp(key, "speculative")) {
        if (value != 0 && value != 1) { set_error("speculative must be 0 or 1"); return WOLFF_EINVAL; }
        h->spec = (int)value;
        h->shape_dirty = true;
        if (check_handle(h) != WOLFF_OK || refresh_shape(h) != WOLFF_OK) return WOLFF_EINVAL;
    } else if (!strcmp(key, "cooperative")) {
        if (value != 0 && value != 1) { set_error("cooperative must be 0 or 1"); return WOLFF_EINVAL; }
        h->cooperative = (int)value;
    } else {
        set_error("unknown option '%s'", key);
        return WOLFF_EINVAL;
    }
    return WOLFF_OK;
}

int wolff_get_stats(wolff_handle h, uint64_t *stats)
{
    int rc = check_handle(h);
    if (rc) return rc;
    if (!stats) { set_error("stats is NULL"); return WOLFF_EINVAL; }
    rc = sync_and_check(h);
    if (rc) return rc;
    if (!h->ran) { memset(stats, 0, WOLFF_NSTATS * sizeof(uint64_t)); return WOLFF_OK; }
    CHECK_CUDA(h, cudaMemcpy(stats, h->ctl->stats, WOLFF_NSTATS * sizeof(uint64_t), cudaMemcpyDeviceToHost), "read stats");
    return WOLFF_OK;
}

}  // extern "C"
