// batch_api.cu -- the extern "C" boundary of the batch of chains declared in include/wolff.h (host side only).
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/wolff.h"
#include "internal.h"

using namespace wolff;

// defined in api.cu: the thread-local error string shared by the whole library, and reading R7
namespace wolff {
void set_error_v(const char *fmt, va_list ap);
uint64_t bond_threshold(double J, double T);
}

namespace {

void set_error(const char *fmt, ...) __attribute__((format(printf, 1, 2)));
void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    wolff::set_error_v(fmt, ap);
    va_end(ap);
}

}  // namespace

struct wolff_batch_ctx {
    int dim = 0, L = 0;
    uint32_t R = 0;
    uint64_t N = 0;
    size_t stride = 0;              // bytes between two lattices (N padded to 16)
    uint64_t u = 0;                 // next update index (shared by all chains)
    int device = 0, num_sms = 0;
    Geometry geo{};
    std::vector<uint64_t> thr, seed;
    int8_t *spins = nullptr;
    uint32_t *lists = nullptr;
    uint32_t *sizes = nullptr;
    long long *E_log = nullptr, *M_log = nullptr;
    uint64_t log_cap = 0;           // updates per chain the size log can hold
    uint64_t em_cap = 0;            // updates per chain E_log and M_log can hold (allocated by the first measured run)
    uint64_t meas_count = 0;        // samples per chain in the moment accumulators (host-side count, for the overflow bound)
    uint2 *keys = nullptr;
    unsigned long long *thr_dev = nullptr;
    long long *EM = nullptr;
    unsigned long long *moments = nullptr;
    unsigned long long *acc = nullptr;      // E/M reduction scratch, 2 per chain
    unsigned long long *stats = nullptr;    // 4 counters + the chain counter
    uint64_t last_n = 0;
    bool ran = false, last_measured = false, cuda_failed = false;
    bool em_valid = false;          // EM holds E and M of the current lattices (a measured run or an evaluation left them there)
    cudaStream_t last_stream = nullptr;
    int measure = 0, threads_opt = 0;
    int resident = 0;               // 0 auto, 1 int8 lattice in global memory, 2 bit-packed lattice in shared memory,
                                    // 3 one thread-block cluster per chain (growth_cluster.cu), chains side by side on streams
    size_t smem_optin = 0;
    uint32_t qcap = 1024;
    uint64_t watchdog_ms = 20000;   // resident = 3: an update that takes longer aborts its chain's launch
    // resident = 3: the launch shape of the cluster-resident kernel and, per chain, a control block, a spill list and its
    // two counters; the per-update durations the kernel records; the streams the chains' launches are spread over
    bool cl_ready = false;
    ClusterParams cl{};
    size_t cl_smem = 0;
    Control *cl_ctl = nullptr;
    uint32_t *cl_spill = nullptr;
    unsigned long long *cl_ctr = nullptr;
    uint32_t *cl_ns = nullptr;
    uint64_t cl_ns_cap = 0;
    std::vector<cudaStream_t> cl_streams;
    std::vector<cudaEvent_t> cl_events;     // one per stream, and the last one for the caller's stream
};

constexpr int kClusterStreams = 8;          // seven clusters of 16 CTAs are resident at a time on a B200

namespace {

class DeviceScope {
public:
    explicit DeviceScope(const wolff_batch_ctx *b)
    {
        if (!b) return;
        if (cudaGetDevice(&prev_) != cudaSuccess) { cudaGetLastError(); prev_ = -1; }
        if (prev_ != b->device) { cudaSetDevice(b->device); switched_ = true; }
    }
    ~DeviceScope() { if (switched_ && prev_ >= 0) cudaSetDevice(prev_); }
private:
    int prev_ = -1;
    bool switched_ = false;
};

int fail_cuda(wolff_batch_ctx *b, cudaError_t e, const char *what)
{
    set_error("%s: %s", what, cudaGetErrorString(e));
    if (b) b->cuda_failed = true;
    return WOLFF_ECUDA;
}

#define CHECK_CUDA(b, call, what)                                   \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return fail_cuda((b), e_, (what));   \
    } while (0)

int check(wolff_batch_ctx *b)
{
    if (!b) { set_error("null batch handle"); return WOLFF_EINVAL; }
    if (b->cuda_failed) { set_error("batch handle is in a failed CUDA state"); return WOLFF_ECUDA; }
    return WOLFF_OK;
}

// Every synchronising batch call ends here: wait for the stream, then look at what the kernels reported on the device.
// resident = 3: each chain's control block has a sticky error word (watchdog codes, 1000 + code in checked builds);
// the other kernels report through stats[7] (checked builds only).  An aborted chain has a half-grown cluster and
// unfinished logs, so the handle is marked failed, as a single chain's is (wolff.h: WOLFF_EINTERNAL).
int sync_and_check(wolff_batch_ctx *b)
{
    cudaStream_t s = b->last_stream;
    if (b->cl_ready && b->ran) {
        std::vector<unsigned int> err(b->R);
        CHECK_CUDA(b, cudaMemcpy2DAsync(err.data(), sizeof(unsigned int), &b->cl_ctl[0].error, sizeof(Control), sizeof(unsigned int), b->R,
                                        cudaMemcpyDeviceToHost, s), "read the chains' error words");
        CHECK_CUDA(b, cudaStreamSynchronize(s), "cudaStreamSynchronize");
        for (uint32_t r = 0; r < b->R; ++r) {
            if (err[r] == 0u) continue;
            if (err[r] >= 1000u) set_error("chain %u: checked build: index out of bounds in the cluster-resident kernel (code %u)", r, err[r] - 1000u);
            else set_error("chain %u: device watchdog: an update did not complete (error flag %u)", r, err[r]);
            b->cuda_failed = true;
            return WOLFF_EINTERNAL;
        }
        return WOLFF_OK;
    }
    unsigned long long flag = 0;
    CHECK_CUDA(b, cudaMemcpyAsync(&flag, b->stats + 7, sizeof(flag), cudaMemcpyDeviceToHost, s), "read the batch kernel's check word");
    CHECK_CUDA(b, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    if (flag != 0) {
        set_error("checked build: index out of bounds in the batch kernel (code %llu)", flag);
        b->cuda_failed = true;
        return WOLFF_EINTERNAL;
    }
    return WOLFF_OK;
}

void free_all(wolff_batch_ctx *b)
{
    cudaFree(b->cl_ctl); cudaFree(b->cl_spill); cudaFree(b->cl_ctr); cudaFree(b->cl_ns);
    for (cudaStream_t s : b->cl_streams) cudaStreamDestroy(s);
    for (cudaEvent_t e : b->cl_events) cudaEventDestroy(e);
    b->cl_streams.clear(); b->cl_events.clear();
    cudaFree(b->spins); cudaFree(b->lists); cudaFree(b->sizes); cudaFree(b->E_log); cudaFree(b->M_log);
    cudaFree(b->keys); cudaFree(b->thr_dev); cudaFree(b->EM); cudaFree(b->moments); cudaFree(b->acc); cudaFree(b->stats);
}

// Does this batch run on the bit-packed shared-memory-resident lattice?  "resident" 2: whenever the planes fit one CTA;
// auto: when they are small enough (32 KiB) that several chains per SM stay in flight.
bool use_bits(const wolff_batch_ctx *b)
{
    if (b->resident == 1) return false;
    const size_t planes = batch_smem_bytes(b->geo.N, 0, true, b->measure != 0);
    const size_t all = batch_smem_bytes(b->geo.N, b->qcap, true, b->measure != 0);
    if (all + 1024 > b->smem_optin) return false;
    return b->resident == 2 || planes <= (32u << 10);
}

// resident = 3: plan and per-chain state of the cluster-resident kernel (once per handle)
int prepare_clusters(wolff_batch_ctx *b)
{
    if (b->cl_ready) return WOLFF_OK;
    if (!cluster_plan(b->dim, b->geo, 16, 2048, b->smem_optin, &b->cl, &b->cl_smem, nullptr)) {
        set_error("resident = 3: a lattice of N = %llu spins does not fit one thread-block cluster (at most 2^24)", (unsigned long long)b->N);
        return WOLFF_EINVAL;
    }
    const size_t R = b->R, cap = (size_t)1 << b->cl.spill_log;
    if (cudaMalloc(&b->cl_ctl, R * sizeof(Control)) != cudaSuccess || cudaMalloc(&b->cl_spill, R * cap * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&b->cl_ctr, R * 2 * sizeof(unsigned long long)) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(b->cl_ctl); cudaFree(b->cl_spill); cudaFree(b->cl_ctr);
        b->cl_ctl = nullptr; b->cl_spill = nullptr; b->cl_ctr = nullptr;
        set_error("resident = 3: cannot allocate the spill lists of %u chains", b->R);
        return WOLFF_ENOMEM;
    }
    CHECK_CUDA(b, cudaMemset(b->cl_ctl, 0, R * sizeof(Control)), "clear control blocks");
    CHECK_CUDA(b, cudaMemset(b->cl_spill, 0, R * cap * sizeof(uint32_t)), "clear spill lists");
    CHECK_CUDA(b, cudaMemset(b->cl_ctr, 0, R * 2 * sizeof(unsigned long long)), "clear spill counters");
    const int ns = (int)(b->R < (uint32_t)kClusterStreams ? b->R : (uint32_t)kClusterStreams);
    for (int i = 0; i < ns; ++i) {
        cudaStream_t s = nullptr;
        CHECK_CUDA(b, cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking), "cudaStreamCreate");
        b->cl_streams.push_back(s);
    }
    for (int i = 0; i <= ns; ++i) {
        cudaEvent_t e = nullptr;
        CHECK_CUDA(b, cudaEventCreateWithFlags(&e, cudaEventDisableTiming), "cudaEventCreate");
        b->cl_events.push_back(e);
    }
    b->cl.watchdog_ns = b->watchdog_ms * 1000000ull;
    b->cl.idle_ns = 1000;
    b->cl_ready = true;
    return WOLFF_OK;
}

// resident = 3: every chain is one launch of the cluster-resident kernel (one cluster of up to 16 CTAs); the launches are
// spread over a few streams, so that as many chains run side by side as clusters fit the chip (7 of 16 CTAs on a B200).
// The streams start behind the caller's stream and the caller's stream continues behind them.
int run_clusters(wolff_batch_ctx *b, uint64_t n_updates, cudaStream_t stream)
{
    int rc = prepare_clusters(b);
    if (rc) return rc;
    if (n_updates > (1ull << 30)) { set_error("resident = 3: at most 2^30 updates per call"); return WOLFF_EINVAL; }
    if (n_updates > b->cl_ns_cap) {
        uint32_t *fresh = nullptr;
        if (cudaMalloc(&fresh, (size_t)b->R * (size_t)b->log_cap * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            set_error("cannot allocate the per-update durations for %u chains", b->R);
            return WOLFF_ENOMEM;
        }
        cudaFree(b->cl_ns);
        b->cl_ns = fresh;
        b->cl_ns_cap = b->log_cap;
    }
    // counters of the growth kernel start from zero at every launch; the error flags stay
    CHECK_CUDA(b, cudaMemset2DAsync(b->cl_ctl, sizeof(Control), 0, kControlClearBytes, b->R, stream), "clear control blocks");
    const bool measure = b->measure != 0;
    if (measure)      // the kernel accumulates into its control block: start from the batch's sums
        CHECK_CUDA(b, cudaMemcpy2DAsync(&b->cl_ctl[0].moments, sizeof(Control), b->moments, 10 * sizeof(unsigned long long),
                                        10 * sizeof(unsigned long long), b->R, cudaMemcpyDeviceToDevice, stream), "moments -> control blocks");
    const size_t ns = b->cl_streams.size(), cap = (size_t)1 << b->cl.spill_log;
    cudaEvent_t start = b->cl_events[ns];
    CHECK_CUDA(b, cudaEventRecord(start, stream), "cudaEventRecord");
    for (size_t i = 0; i < ns; ++i) CHECK_CUDA(b, cudaStreamWaitEvent(b->cl_streams[i], start, 0), "cudaStreamWaitEvent");
    for (uint32_t r = 0; r < b->R; ++r) {
        ClusterParams cp = b->cl;
        GrowthParams &g = cp.g;
        g.spins = b->spins + (size_t)r * b->stride;
        g.clist = nullptr;
        g.sizes = b->sizes + (size_t)r * (size_t)n_updates;
        g.ctl = b->cl_ctl + r;
        g.geo = b->geo;
        g.key0 = (uint32_t)b->seed[r]; g.key1 = (uint32_t)(b->seed[r] >> 32);
        g.thr = b->thr[r]; g.u0 = b->u; g.n_updates = n_updates;
        g.measure = measure ? 1u : 0u; g.claim_bits = 0xFEu;
        g.E_log = measure ? b->E_log + (size_t)r * (size_t)n_updates : nullptr;      // the logs exist once a measured run has asked for them
        g.M_log = measure ? b->M_log + (size_t)r * (size_t)n_updates : nullptr;
        g.ns_log = b->cl_ns + (size_t)r * (size_t)n_updates;
        if (measure) cp.idle_ns = 200;
        cp.thr32 = (uint32_t)b->thr[r];
        cp.thr_all = (b->thr[r] >> 32) != 0 ? 1u : 0u;
        cp.spill = b->cl_spill + (size_t)r * cap;
        cp.spill_ctr = b->cl_ctr + 2 * (size_t)r;
        CHECK_CUDA(b, launch_growth_cluster(cp, b->dim, b->cl_smem, b->cl_streams[r % ns]), "launch cluster-resident growth kernel");
    }
    for (size_t i = 0; i < ns; ++i) {
        CHECK_CUDA(b, cudaEventRecord(b->cl_events[i], b->cl_streams[i]), "cudaEventRecord");
        CHECK_CUDA(b, cudaStreamWaitEvent(stream, b->cl_events[i], 0), "cudaStreamWaitEvent");
    }
    if (measure) {
        CHECK_CUDA(b, cudaMemcpy2DAsync(b->moments, 10 * sizeof(unsigned long long), &b->cl_ctl[0].moments, sizeof(Control),
                                        10 * sizeof(unsigned long long), b->R, cudaMemcpyDeviceToDevice, stream), "control blocks -> moments");
        CHECK_CUDA(b, cudaMemcpy2DAsync(b->EM, 2 * sizeof(long long), &b->cl_ctl[0].E, sizeof(Control), 2 * sizeof(long long), b->R,
                                        cudaMemcpyDeviceToDevice, stream), "control blocks -> E, M");
    }
    return WOLFF_OK;
}

// threads per CTA and CTAs of a launch: every chain resident at once when the chip can hold them
void launch_shape(const wolff_batch_ctx *b, bool bits, int *threads, int *grid)
{
    int t = b->threads_opt;
    if (t == 0) {
        const uint32_t per_sm = (b->R + (uint32_t)b->num_sms - 1u) / (uint32_t)b->num_sms;     // chains per SM
        t = per_sm >= 8u ? 64 : (per_sm >= 3u ? 128 : 256);
    }
    int per_sm = 1;
    const size_t smem = batch_smem_bytes(b->geo.N, b->qcap, bits, b->measure != 0);
    if (batch_ctas_per_sm(b->dim, b->geo.pow2 != 0, bits, t, smem, &per_sm) != cudaSuccess || per_sm < 1) { cudaGetLastError(); per_sm = 1; }
    uint64_t g = (uint64_t)per_sm * (uint64_t)b->num_sms;
    if (g > b->R) g = b->R;
    *threads = t;
    *grid = (int)g;
}

}  // namespace

extern "C" {

wolff_batch wolff_batch_create(int dim, int L, int R, const double *J, const double *T, const uint64_t *seed)
{
    if (dim != 2 && dim != 3) { set_error("dim must be 2 or 3 (got %d)", dim); return nullptr; }
    if (L < 2) { set_error("L must be >= 2 (got %d)", L); return nullptr; }
    if (R < 1 || R > (1 << 20)) { set_error("R must be in [1, 2^20] (got %d)", R); return nullptr; }
    if (!J || !T || !seed) { set_error("J, T and seed must point to R values each"); return nullptr; }
    uint64_t N = 1;
    for (int k = 0; k < dim; ++k) {
        N *= (uint64_t)L;
        if (N > (1ull << 31)) { set_error("N = L^dim exceeds 2^31"); return nullptr; }
    }
    for (int r = 0; r < R; ++r) {
        if (!(J[r] >= 0.0) || !std::isfinite(J[r])) { set_error("J[%d] must be finite and >= 0", r); return nullptr; }
        if (!(T[r] > 0.0) || !std::isfinite(T[r])) { set_error("T[%d] must be finite and > 0", r); return nullptr; }
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        set_error("no usable CUDA device (%s); this library has no CPU fallback", cudaGetErrorString(e));
        return nullptr;
    }
    wolff_batch_ctx *b = new (std::nothrow) wolff_batch_ctx();
    if (!b) { set_error("out of host memory"); return nullptr; }
    b->dim = dim; b->L = L; b->R = (uint32_t)R; b->N = N;
    b->stride = (size_t)((N + 15ull) & ~15ull);
    b->geo.L = (uint32_t)L; b->geo.N = (uint32_t)N; b->geo.LL = (uint32_t)((uint64_t)L * (uint64_t)L);
    b->geo.pow2 = ((L & (L - 1)) == 0) ? 1u : 0u;
    b->geo.logL = 0;
    if (b->geo.pow2) while ((1u << b->geo.logL) < (uint32_t)L) ++b->geo.logL;
    cudaDeviceProp prop{};
    if (cudaGetDevice(&b->device) != cudaSuccess || cudaGetDeviceProperties(&prop, b->device) != cudaSuccess) {
        set_error("cudaGetDeviceProperties failed"); delete b; return nullptr;
    }
    b->num_sms = prop.multiProcessorCount;
    b->smem_optin = prop.sharedMemPerBlockOptin;
    std::vector<uint2> keys((size_t)R);
    b->thr.resize((size_t)R); b->seed.assign(seed, seed + R);
    for (int r = 0; r < R; ++r) {
        b->thr[(size_t)r] = bond_threshold(J[r], T[r]);
        keys[(size_t)r] = make_uint2((uint32_t)seed[r], (uint32_t)(seed[r] >> 32));
    }
    const size_t Rz = (size_t)R;
    bool ok = cudaMalloc(&b->spins, Rz * b->stride) == cudaSuccess && cudaMalloc(&b->lists, Rz * (size_t)N * sizeof(uint32_t)) == cudaSuccess &&
              cudaMalloc(&b->keys, Rz * sizeof(uint2)) == cudaSuccess && cudaMalloc(&b->thr_dev, Rz * sizeof(unsigned long long)) == cudaSuccess &&
              cudaMalloc(&b->EM, 2 * Rz * sizeof(long long)) == cudaSuccess && cudaMalloc(&b->moments, 10 * Rz * sizeof(unsigned long long)) == cudaSuccess &&
              cudaMalloc(&b->acc, 2 * Rz * sizeof(unsigned long long)) == cudaSuccess && cudaMalloc(&b->stats, 8 * sizeof(unsigned long long)) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        set_error("device allocation failed for %d chains of N = %llu", R, (unsigned long long)N);
        free_all(b); delete b;
        return nullptr;
    }
    static_assert(sizeof(unsigned long long) == sizeof(uint64_t), "threshold layout");
    e = cudaMemcpy(b->keys, keys.data(), Rz * sizeof(uint2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(b->thr_dev, b->thr.data(), Rz * sizeof(uint64_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(b->moments, 0, 10 * Rz * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(b->EM, 0, 2 * Rz * sizeof(long long));
    if (e == cudaSuccess) e = cudaMemset(b->stats, 0, 8 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(b->spins, 0, Rz * b->stride);
    // every chain starts from its own seed-derived random lattice (reading R9), as wolff_create does
    for (int r = 0; r < R && e == cudaSuccess; ++r)
        e = launch_init_lattice(b->spins + (size_t)r * b->stride, b->geo.N, seed[r], b->num_sms, nullptr);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        set_error("batch initialisation failed: %s", cudaGetErrorString(e));
        free_all(b); delete b;
        return nullptr;
    }
    return b;
}

int wolff_batch_destroy(wolff_batch b)
{
    if (!b) return WOLFF_OK;
    DeviceScope scope(b);
    if (b->ran) cudaStreamSynchronize(b->last_stream);
    free_all(b);
    delete b;
    return WOLFF_OK;
}

int wolff_batch_run(wolff_batch b, uint64_t n_updates, void *cuda_stream)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (n_updates == 0) return WOLFF_OK;
    if (n_updates > (1ull << 32)) { set_error("n_updates too large for one call (max 2^32)"); return WOLFF_EINVAL; }
    if (b->resident == 2 && batch_smem_bytes(b->geo.N, b->qcap, true, b->measure != 0) + 1024 > b->smem_optin) {
        set_error("resident = 2: the bit planes of N = %llu spins (%d of them%s) and the frontier buffers do not fit one CTA's shared memory",
                  (unsigned long long)b->N, b->measure ? 2 : 1, b->measure ? ": a measured run keeps a mark per spin" : "");
        return WOLFF_EINVAL;
    }
    if (b->ran && (stream != b->last_stream || n_updates > b->log_cap))
        CHECK_CUDA(b, cudaStreamSynchronize(b->last_stream), "cudaStreamSynchronize");
    if (b->measure) {
        // exact while samples * N^4 < 2^128 (see wolff_run): refuse what would wrap the accumulators silently
        const unsigned __int128 n2 = (unsigned __int128)b->N * b->N, n4 = n2 * n2;
        const unsigned __int128 limit = ~(unsigned __int128)0 / n4;
        if ((unsigned __int128)b->meas_count + n_updates > limit) {
            set_error("measured run refused: %llu + %llu samples of M^4 <= N^4 (N = %llu) would overflow the 128-bit moment "
                      "accumulators; call wolff_batch_reset_moments first", (unsigned long long)b->meas_count,
                      (unsigned long long)n_updates, (unsigned long long)b->N);
            return WOLFF_EINVAL;
        }
    }
    if (n_updates > b->log_cap) {
        uint64_t cap = b->log_cap ? b->log_cap : 1024;
        while (cap < n_updates) cap *= 2;
        uint32_t *fresh = nullptr;
        const size_t entries = (size_t)b->R * (size_t)cap;
        if (cudaMalloc(&fresh, entries * sizeof(uint32_t)) != cudaSuccess) {
            cudaGetLastError();
            set_error("cannot allocate the cluster-size log for %u chains x %llu updates", b->R, (unsigned long long)n_updates);
            return WOLFF_ENOMEM;
        }
        cudaFree(b->sizes);
        b->sizes = fresh;
        b->log_cap = cap;
    }
    if (b->measure && n_updates > b->em_cap) {
        // E and M after every update of every chain: 16 R bytes per update, allocated only once a measured run asks for them
        if (b->ran) CHECK_CUDA(b, cudaStreamSynchronize(b->last_stream), "cudaStreamSynchronize");
        long long *fresh_E = nullptr, *fresh_M = nullptr;
        const size_t entries = (size_t)b->R * (size_t)b->log_cap;
        if (cudaMalloc(&fresh_E, entries * sizeof(long long)) != cudaSuccess || cudaMalloc(&fresh_M, entries * sizeof(long long)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(fresh_E); cudaFree(fresh_M);
            set_error("cannot allocate the E / M logs for %u chains x %llu updates", b->R, (unsigned long long)n_updates);
            return WOLFF_ENOMEM;
        }
        cudaFree(b->E_log); cudaFree(b->M_log);
        b->E_log = fresh_E; b->M_log = fresh_M;
        b->em_cap = b->log_cap;
    }
    if (b->resident == 3) {
        if (b->measure && b->L % 32 != 0) {
            set_error("resident = 3 measures inside the kernel only when L is a multiple of 32 (L = %d): use resident 0, 1 or 2", b->L);
            return WOLFF_EINVAL;
        }
        rc = run_clusters(b, n_updates, stream);
        if (rc) return rc;
        b->u += n_updates;
        b->last_n = n_updates;
        b->last_measured = b->measure != 0;
        if (b->measure) b->meas_count += n_updates;
        b->em_valid = b->measure != 0;
        b->last_stream = stream;
        b->ran = true;
        return WOLFF_OK;
    }
    if (b->measure && !b->em_valid)      // running E and M start from a whole-lattice evaluation of every chain
        CHECK_CUDA(b, launch_batch_energy(b->spins, b->stride, b->geo, b->dim, b->R, b->acc, b->EM, b->num_sms, stream), "launch batch E/M reduction");
    CHECK_CUDA(b, cudaMemsetAsync(b->stats, 0, 8 * sizeof(unsigned long long), stream), "cudaMemsetAsync(stats)");
    BatchParams bp{};
    bp.spins = b->spins; bp.lists = b->lists; bp.sizes = b->sizes; bp.E_log = b->E_log; bp.M_log = b->M_log;
    bp.keys = b->keys; bp.thr = b->thr_dev; bp.EM = b->EM; bp.moments = b->moments; bp.stats = b->stats;
    bp.next = reinterpret_cast<unsigned int *>(b->stats + 4);
    bp.geo = b->geo; bp.lattice_stride = b->stride; bp.u0 = b->u; bp.n_updates = n_updates; bp.R = b->R;
    bp.measure = b->measure ? 1u : 0u; bp.qcap = b->qcap;
    int threads = 0, grid = 0;
    const bool bits = use_bits(b);
    launch_shape(b, bits, &threads, &grid);
    CHECK_CUDA(b, launch_growth_batch(bp, b->dim, bits, grid, threads, stream), "launch batch growth kernel");
    b->u += n_updates;
    b->last_n = n_updates;
    b->last_measured = b->measure != 0;
    if (b->measure) b->meas_count += n_updates;
    b->em_valid = b->measure != 0;       // a measured run leaves the running values in EM; an unmeasured one outdates them
    b->last_stream = stream;
    b->ran = true;
    return WOLFF_OK;
}

int wolff_batch_observables(wolff_batch b, int64_t *E, int64_t *M, uint32_t *cluster_sizes)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    cudaStream_t s = b->last_stream;
    const size_t R = b->R;
    if (E || M) {
        CHECK_CUDA(b, launch_batch_energy(b->spins, b->stride, b->geo, b->dim, b->R, b->acc, b->EM, b->num_sms, s), "launch batch E/M reduction");
        b->em_valid = true;
        // (E, M) pairs -> the caller's two arrays (host or device): strided copies
        if (E) CHECK_CUDA(b, cudaMemcpy2DAsync(E, sizeof(int64_t), b->EM, 2 * sizeof(long long), sizeof(int64_t), R, cudaMemcpyDefault, s), "copy E");
        if (M) CHECK_CUDA(b, cudaMemcpy2DAsync(M, sizeof(int64_t), b->EM + 1, 2 * sizeof(long long), sizeof(int64_t), R, cudaMemcpyDefault, s), "copy M");
    }
    if (cluster_sizes && b->ran && b->last_n > 0)
        CHECK_CUDA(b, cudaMemcpyAsync(cluster_sizes, b->sizes, R * (size_t)b->last_n * sizeof(uint32_t), cudaMemcpyDefault, s), "copy cluster sizes");
    return sync_and_check(b);
}

int wolff_batch_get_spins(wolff_batch b, int8_t *dst)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    if (!dst) { set_error("dst is NULL"); return WOLFF_EINVAL; }
    cudaStream_t s = b->last_stream;
    CHECK_CUDA(b, cudaMemcpy2DAsync(dst, (size_t)b->N, b->spins, b->stride, (size_t)b->N, b->R, cudaMemcpyDefault, s), "copy lattices out");
    return sync_and_check(b);
}

int wolff_batch_set_spins(wolff_batch b, const int8_t *src)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    if (!src) { set_error("src is NULL"); return WOLFF_EINVAL; }
    cudaStream_t s = b->last_stream;
    rc = sync_and_check(b);
    if (rc) return rc;
    // stage in the member lists (4 N bytes per chain, idle between runs), validate there, then commit
    int8_t *staging = reinterpret_cast<int8_t *>(b->lists);
    const size_t total = (size_t)b->R * (size_t)b->N;
    CHECK_CUDA(b, cudaMemcpyAsync(staging, src, total, cudaMemcpyDefault, s), "copy lattices in");
    unsigned int *invalid = reinterpret_cast<unsigned int *>(b->stats + 6);
    CHECK_CUDA(b, cudaMemsetAsync(invalid, 0, sizeof(unsigned int), s), "reset validation flag");
    CHECK_CUDA(b, launch_validate_word(staging, total, invalid, b->num_sms, s), "launch validation");
    unsigned int bad = 0;
    CHECK_CUDA(b, cudaMemcpyAsync(&bad, invalid, sizeof(bad), cudaMemcpyDeviceToHost, s), "read validation flag");
    CHECK_CUDA(b, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    if (bad) { set_error("batch set_spins: every byte must be +1 or -1"); return WOLFF_EINVAL; }
    b->em_valid = false;
    CHECK_CUDA(b, cudaMemcpy2DAsync(b->spins, b->stride, staging, (size_t)b->N, (size_t)b->N, b->R, cudaMemcpyDeviceToDevice, s), "commit lattices");
    CHECK_CUDA(b, cudaStreamSynchronize(s), "cudaStreamSynchronize");
    return WOLFF_OK;
}

int wolff_batch_get_state(wolff_batch b, uint64_t *update_index, uint64_t *thresholds)
{
    if (!b) { set_error("null batch handle"); return WOLFF_EINVAL; }
    if (update_index) *update_index = b->u;
    if (thresholds) memcpy(thresholds, b->thr.data(), (size_t)b->R * sizeof(uint64_t));
    return WOLFF_OK;
}

int wolff_batch_set_update_index(wolff_batch b, uint64_t update_index)
{
    if (!b) { set_error("null batch handle"); return WOLFF_EINVAL; }
    b->u = update_index;
    return WOLFF_OK;
}

int wolff_batch_set_option(wolff_batch b, const char *key, int64_t value)
{
    if (!b || !key) { set_error("null batch handle or key"); return WOLFF_EINVAL; }
    if (!strcmp(key, "measure")) {
        if (value != 0 && value != 1) { set_error("measure must be 0 or 1"); return WOLFF_EINVAL; }
        b->measure = (int)value;
    } else if (!strcmp(key, "threads")) {
        if (value != 0 && value != 32 && value != 64 && value != 128 && value != 256) { set_error("threads must be 0 (auto), 32, 64, 128 or 256"); return WOLFF_EINVAL; }
        b->threads_opt = (int)value;
    } else if (!strcmp(key, "resident")) {
        if (value < 0 || value > 3) {
            set_error("resident must be 0 (auto), 1 (int8 lattice in global memory), 2 (bit-packed in one CTA's shared memory) or 3 (bit-packed in one cluster's)");
            return WOLFF_EINVAL;
        }
        if (value == 3) {
            DeviceScope scope(b);
            const int rc3 = prepare_clusters(b);
            if (rc3) return rc3;
        }
        if (value == 2 && batch_smem_bytes(b->geo.N, b->qcap, true, false) + 1024 > b->smem_optin) {
            set_error("resident = 2: a bit plane of N = %llu spins does not fit one CTA's shared memory", (unsigned long long)b->N);
            return WOLFF_EINVAL;
        }
        b->resident = (int)value;
    } else if (!strcmp(key, "watchdog_ms")) {
        if (value < 1 || value > 3600000) { set_error("watchdog_ms must be in [1, 3600000]"); return WOLFF_EINVAL; }
        b->watchdog_ms = (uint64_t)value;
        b->cl.watchdog_ns = b->watchdog_ms * 1000000ull;
    } else if (!strcmp(key, "queue_cap")) {
        if (value < 8 || value > 16384) { set_error("queue_cap must be in [8, 16384]"); return WOLFF_EINVAL; }
        b->qcap = (uint32_t)value;
    } else {
        set_error("unknown batch option '%s'", key);
        return WOLFF_EINVAL;
    }
    return WOLFF_OK;
}

int wolff_batch_get_series(wolff_batch b, int64_t *E_series, int64_t *M_series)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    if (!b->ran || !b->last_measured) {
        set_error("the most recent wolff_batch_run was not a measured one (wolff_batch_set_option \"measure\" = 1)");
        return WOLFF_EINVAL;
    }
    cudaStream_t s = b->last_stream;
    const size_t bytes = (size_t)b->R * (size_t)b->last_n * sizeof(int64_t);
    if (E_series) CHECK_CUDA(b, cudaMemcpyAsync(E_series, b->E_log, bytes, cudaMemcpyDefault, s), "copy E series");
    if (M_series) CHECK_CUDA(b, cudaMemcpyAsync(M_series, b->M_log, bytes, cudaMemcpyDefault, s), "copy M series");
    return sync_and_check(b);
}

int wolff_batch_get_moments(wolff_batch b, uint64_t *moments, double *binder)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    std::vector<uint64_t> host(10 * (size_t)b->R);
    CHECK_CUDA(b, cudaMemcpyAsync(host.data(), b->moments, host.size() * sizeof(uint64_t), cudaMemcpyDeviceToHost, b->last_stream), "read moments");
    rc = sync_and_check(b);
    if (rc) return rc;
    if (moments) memcpy(moments, host.data(), host.size() * sizeof(uint64_t));
    if (binder) {
        const long double two64 = 18446744073709551616.0L;
        for (uint32_t r = 0; r < b->R; ++r) {
            const uint64_t *m = host.data() + 10 * (size_t)r;
            const long double n = (long double)m[0], s2 = (long double)m[6] * two64 + (long double)m[5], s4 = (long double)m[8] * two64 + (long double)m[7];
            binder[r] = (m[0] == 0 || s2 == 0.0L) ? std::nan("") : (double)(1.0L - (n * s4) / (3.0L * s2 * s2));
        }
    }
    return WOLFF_OK;
}

int wolff_batch_reset_moments(wolff_batch b)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    CHECK_CUDA(b, cudaMemsetAsync(b->moments, 0, 10 * (size_t)b->R * sizeof(unsigned long long), b->last_stream), "clear moments");
    b->meas_count = 0;
    return sync_and_check(b);
}

int wolff_batch_get_stats(wolff_batch b, uint64_t *stats)
{
    int rc = check(b);
    if (rc) return rc;
    DeviceScope scope(b);
    if (!stats) { set_error("stats is NULL"); return WOLFF_EINVAL; }
    uint64_t host[8];
    if (b->resident == 3 && b->cl_ready) {
        // one control block per chain: sum the counters, look at the error flags
        std::vector<Control> ctl(b->R);
        CHECK_CUDA(b, cudaMemcpyAsync(ctl.data(), b->cl_ctl, (size_t)b->R * sizeof(Control), cudaMemcpyDeviceToHost, b->last_stream), "read control blocks");
        CHECK_CUDA(b, cudaStreamSynchronize(b->last_stream), "cudaStreamSynchronize");
        memset(stats, 0, 4 * sizeof(uint64_t));
        for (uint32_t r = 0; r < b->R; ++r) {
            if (ctl[r].error != 0) {
                set_error("chain %u: %s (error flag %u)", r, ctl[r].error >= 1000u ? "checked build: index out of bounds" : "device watchdog", ctl[r].error);
                b->cuda_failed = true;
                return WOLFF_EINTERNAL;
            }
            stats[0] += ctl[r].stats[0]; stats[1] += ctl[r].stats[1]; stats[3] += ctl[r].stats[7];
        }
        return WOLFF_OK;
    }
    CHECK_CUDA(b, cudaMemcpyAsync(host, b->stats, sizeof(host), cudaMemcpyDeviceToHost, b->last_stream), "read stats");
    CHECK_CUDA(b, cudaStreamSynchronize(b->last_stream), "cudaStreamSynchronize");
    memcpy(stats, host, 4 * sizeof(uint64_t));
    if (host[7] != 0) {      // set by checked builds only (-DWOLFF_CHECKED): an index was out of its bounds
        set_error("checked build: index out of bounds in the batch kernel (code %llu)", (unsigned long long)host[7]);
        b->cuda_failed = true;
        return WOLFF_EINTERNAL;
    }
    return WOLFF_OK;
}

}  // extern "C"
