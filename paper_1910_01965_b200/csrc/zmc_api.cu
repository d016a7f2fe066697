// zmc_api.cu -- the C ABI of include/zmc.h: argument validation (H1), the batch scheduler (H2),
// kernel dispatch, and result streaming to host memory on a side stream (H8).
//
// PAPER.md:65 "we cut the parameter grid into several batches. Each batch is fed into one GPU
// device for evaluation"; PAPER.md:85, :132-140 report HToD, DToH and GPU evaluation time
// separately -- zmc_timing keeps that split.  There is no CPU fallback anywhere in this file.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "zmc_internal.h"
#include "zmc_params.h"
#include "zmc_rtc.h"

namespace zmc {
extern const KernelEntry kEntriesC12[];  extern const int kNumEntriesC12;
extern const KernelEntry kEntriesC3[];   extern const int kNumEntriesC3;
extern const KernelEntry kEntriesC45[];  extern const int kNumEntriesC45;
extern const KernelEntry kEntriesP6[];   extern const int kNumEntriesP6;
extern const KernelEntry kEntriesDiag[]; extern const int kNumEntriesDiag;
}  // namespace zmc

using namespace zmc;

namespace {

const zmc_integrand_info kFamilies[] = {
    {ZMC_FAM_C1_COS_XY, "c1_cos_xy", 1, 1, 1, 1, 0, 1},
    {ZMC_FAM_C2_SIN_XY2, "c2_sin_xy2", 2, 2, 2, 2, 0, 1},
    {ZMC_FAM_C3_OSCILLATORY, "c3_oscillatory", 1, ZMC_MAX_N, 3, 3, 1, 1},
    {ZMC_FAM_C4_GAUSS_PEAK, "c4_gauss_peak", 6, 6, 4, 4, 0, 1},
    {ZMC_FAM_C5_DAMPED_COS, "c5_damped_cos", 3, 3, 5, 5, 0, 1},
    {ZMC_FAM_P6_SIN_SUM, "p6_sin_sum", 1, ZMC_MAX_N, 1, ZMC_MAX_M, 0, 1},
    {ZMC_FAM_CONST_ONE, "const_one", 1, ZMC_MAX_N, 1, ZMC_MAX_M, 0, 1},
    {ZMC_FAM_PARAM_ECHO, "param_echo", 1, ZMC_MAX_N, 1, ZMC_MAX_M, 1, 1},
    {ZMC_FAM_LIN_Y, "lin_y", 1, ZMC_MAX_N, 1, ZMC_MAX_M, 1, 1},
    {ZMC_FAM_POLY, "poly", 1, ZMC_MAX_N, 1, ZMC_MAX_M, 0, 1},
};
const int kNumFamilies = sizeof(kFamilies) / sizeof(kFamilies[0]);

thread_local int tl_cuda_error = 0;

zmc_status cuda_fail(cudaError_t e) {
    tl_cuda_error = (int)e;
    cudaGetLastError();      // the runtime remembers a failed call until asked: left there, the NEXT kernel launch's error check would report it
    return (e == cudaErrorMemoryAllocation) ? ZMC_ERR_OUT_OF_MEMORY : ZMC_ERR_CUDA;
}
}  // namespace
namespace zmc {
void set_last_cuda_error(int e) { tl_cuda_error = e; }
int get_last_cuda_error() { return tl_cuda_error; }
}  // namespace zmc
namespace {
#define ZMC_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e__ = (call);                        \
        if (e__ != cudaSuccess) return cuda_fail(e__);   \
    } while (0)

// Built-in family or a registered user integrand (ids >= kFirstUserId); `storage` backs the latter's info.
const zmc_integrand_info* find_family(int id, zmc_integrand_info* storage) {
    for (int i = 0; i < kNumFamilies; ++i)
        if (kFamilies[i].id == id) return &kFamilies[i];
    if (const std::shared_ptr<const UserIntegrand> u = find_user_integrand(id)) {
        *storage = zmc_integrand_info{u->id, u->name.c_str(), u->N, u->N, u->M, u->M, u->n_consts, 0};
        return storage;
    }
    return nullptr;
}

struct Options {     // zmc_options with defaults applied
    int precision = ZMC_PREC_F64, out_dtype = ZMC_OUT_F64, out_location = ZMC_LOC_DEVICE;
    int schedule = ZMC_SCHED_AUTO, fast_math = ZMC_FAST_MATH_DEFAULT;
    uint64_t batch_points = 0, first_index = 0, count = 0;
    const double* consts = nullptr;
    int n_consts = 0;
    int flags = 0;
};

zmc_status read_options(const zmc_options* o, Options* out) {
    if (!o) return ZMC_OK;
    if (o->struct_size < sizeof(zmc_options)) return ZMC_ERR_INVALID_ARG;
    out->precision = o->precision;
    out->out_dtype = o->out_dtype;
    out->out_location = o->out_location;
    out->schedule = o->schedule;
    out->fast_math = o->fast_math;
    out->batch_points = o->batch_points;
    out->first_index = o->first_index;
    out->count = o->count;
    out->consts = o->consts;
    out->n_consts = o->n_consts;
    out->flags = o->flags;
    if (out->flags & ~(ZMC_OPT_EXPLICIT_COUNT | ZMC_OPT_FRESH_LISTS)) return ZMC_ERR_INVALID_ARG;
    if (out->precision != ZMC_PREC_F64 && out->precision != ZMC_PREC_F32E) return ZMC_ERR_INVALID_ARG;
    if (out->out_dtype != ZMC_OUT_F64 && out->out_dtype != ZMC_OUT_F32) return ZMC_ERR_INVALID_ARG;
    if (out->out_location != ZMC_LOC_DEVICE && out->out_location != ZMC_LOC_HOST) return ZMC_ERR_INVALID_ARG;
    if (out->schedule < ZMC_SCHED_AUTO || out->schedule > ZMC_SCHED_CTA) return ZMC_ERR_INVALID_ARG;
    if (out->fast_math < ZMC_FAST_MATH_DEFAULT || out->fast_math > ZMC_FAST_MATH_ON) return ZMC_ERR_INVALID_ARG;
    if (out->n_consts < 0 || out->n_consts > ZMC_MAX_CONSTS) return ZMC_ERR_INVALID_ARG;
    if (out->n_consts > 0 && !out->consts) return ZMC_ERR_INVALID_ARG;
    return ZMC_OK;
}

// All argument checks (reading Q18).  Nothing is enqueued and no output is touched on failure.
zmc_status validate(int id, int N, const double* bounds, int M, const zmc_param_list* lists, uint64_t n_samples,
                    const Options& o, uint64_t* G_out, uint64_t* first_out, uint64_t* count_out) {
    if (!bounds || !lists) return ZMC_ERR_INVALID_ARG;
    if (N < 1 || N > ZMC_MAX_N || M < 1 || M > ZMC_MAX_M) return ZMC_ERR_INVALID_ARG;
    if (n_samples < 2 || n_samples > 0xFFFFFFFFull) return ZMC_ERR_INVALID_ARG;
    if (n_samples * (uint64_t)N > (1ull << 34)) return ZMC_ERR_INVALID_ARG;   // block index stays 32-bit
    for (int k = 0; k < N; ++k) {
        const double a = bounds[2 * k], b = bounds[2 * k + 1];
        if (!std::isfinite(a) || !std::isfinite(b) || !(a < b)) return ZMC_ERR_INVALID_ARG;
    }
    uint64_t G = 1;
    for (int i = 0; i < M; ++i) {
        if (lists[i].count < 1 || !lists[i].values) return ZMC_ERR_INVALID_ARG;
        if (lists[i].count > 0x7FFFFFFFll) return ZMC_ERR_GRID_TOO_LARGE;
        for (int64_t j = 0; j < lists[i].count; ++j)
            if (!std::isfinite(lists[i].values[j])) return ZMC_ERR_INVALID_ARG;
        if ((uint64_t)lists[i].count > (1ull << 48) / G) return ZMC_ERR_GRID_TOO_LARGE;
        G *= (uint64_t)lists[i].count;
    }
    for (int c = 0; c < o.n_consts; ++c)
        if (!std::isfinite(o.consts[c])) return ZMC_ERR_INVALID_ARG;
    zmc_integrand_info user_info;
    const zmc_integrand_info* fam = find_family(id, &user_info);
    if (!fam) return ZMC_ERR_UNKNOWN_INTEGRAND;
    if (N < fam->N_min || N > fam->N_max || M < fam->M_min || M > fam->M_max || o.n_consts != fam->n_consts)
        return ZMC_ERR_SHAPE_MISMATCH;
    if (id == ZMC_FAM_PARAM_ECHO || id == ZMC_FAM_LIN_Y) {
        const double c = o.consts[0];
        const int lim = (id == ZMC_FAM_PARAM_ECHO) ? M : N;
        if (c < 0 || c >= lim || c != std::floor(c)) return ZMC_ERR_SHAPE_MISMATCH;
    }
    if (o.first_index > G) return ZMC_ERR_INVALID_ARG;
    // count == 0 means "to the end of the grid" unless ZMC_OPT_EXPLICIT_COUNT says it is meant literally (an empty shard)
    uint64_t count = (o.count || (o.flags & ZMC_OPT_EXPLICIT_COUNT)) ? o.count : G - o.first_index;
    if (count > G - o.first_index) return ZMC_ERR_INVALID_ARG;
    if (G_out) *G_out = G;
    if (first_out) *first_out = o.first_index;
    if (count_out) *count_out = count;
    return ZMC_OK;
}

// ---- per-device scratch: side stream, cached value lists, timing events, double-buffered result staging ----------
// Value lists are tiny (<= 16 KB for the BASELINE configs) and usually the same from call to call (a benchmark loop,
// the batches of zmc_scan_farm, a user re-scanning with another seed).  Each upload is kept in a small device-resident
// cache keyed by a hash of its content (and verified byte for byte against the pinned host copy), so a repeated call
// enqueues NO host-to-device copy at all: for a 10^3-point grid that copy and its bookkeeping cost more than the kernel.
constexpr int kRing = 8;
struct ListSlot {
    double* host = nullptr;      // pinned copy of what `dev` holds (or will hold once `uploaded` has fired)
    double* dev = nullptr;
    size_t cap = 0;              // entries
    size_t total = 0;            // entries in use
    uint64_t hash = 0;
    cudaEvent_t done = nullptr;      // last kernel that read `dev`
    cudaEvent_t uploaded = nullptr;  // the H2D copy into `dev`
    cudaStream_t last_stream = nullptr;
    bool multi_stream = false;   // read from more than one stream since the upload: `done` does not cover all readers
    bool upload_pending = false; // `uploaded` has not been seen complete yet
    bool used = false;
    bool captured = false;       // a CUDA graph holds `dev` in a kernel node (the call was issued during stream capture): the
                                 // slot is never evicted, overwritten or reallocated again until zmc_shutdown
    uint64_t last_use = 0;
};
struct DeviceScratch {
    bool init = false;
    int sm_count = 0;
    cudaStream_t side = nullptr;
    ListSlot ring[kRing];
    uint64_t use_counter = 0;
    std::vector<cudaEvent_t> timing_pool;    // timing events are created once and reused (creation costs microseconds)
    void* stage[2] = {nullptr, nullptr};     // result staging (mean, stderr[, n]), host-output mode
    size_t stage_cap = 0;                    // bytes each
    cudaEvent_t stage_free[2] = {nullptr, nullptr};   // last copy out of stage[i]
    bool stage_used[2] = {false, false};
    cudaEvent_t kernel_done[2] = {nullptr, nullptr};
    unsigned stage_rot = 0;                  // staging buffers alternate across batches AND across calls
};
constexpr int kMaxDevices = 64;
DeviceScratch g_scratch[kMaxDevices];
std::mutex g_dev_mutex[kMaxDevices];     // one per device: calls on different GPUs (zmc_scan_farm) do not serialise

void free_scratch(DeviceScratch& s) {
    for (int i = 0; i < kRing; ++i) {
        if (s.ring[i].host) cudaFreeHost(s.ring[i].host);
        if (s.ring[i].dev) cudaFree(s.ring[i].dev);
        if (s.ring[i].done) cudaEventDestroy(s.ring[i].done);
        if (s.ring[i].uploaded) cudaEventDestroy(s.ring[i].uploaded);
    }
    for (cudaEvent_t e : s.timing_pool) cudaEventDestroy(e);
    for (int i = 0; i < 2; ++i) {
        if (s.stage[i]) cudaFree(s.stage[i]);
        if (s.stage_free[i]) cudaEventDestroy(s.stage_free[i]);
        if (s.kernel_done[i]) cudaEventDestroy(s.kernel_done[i]);
    }
    if (s.side) cudaStreamDestroy(s.side);
    s = DeviceScratch();
}

zmc_status init_scratch(DeviceScratch& s, int dev) {
    ZMC_CUDA(cudaDeviceGetAttribute(&s.sm_count, cudaDevAttrMultiProcessorCount, dev));
    ZMC_CUDA(cudaStreamCreateWithFlags(&s.side, cudaStreamNonBlocking));
    for (int i = 0; i < kRing; ++i) {
        ZMC_CUDA(cudaEventCreateWithFlags(&s.ring[i].done, cudaEventDisableTiming));
        ZMC_CUDA(cudaEventCreateWithFlags(&s.ring[i].uploaded, cudaEventDisableTiming));
    }
    for (int i = 0; i < 2; ++i) {
        ZMC_CUDA(cudaEventCreateWithFlags(&s.stage_free[i], cudaEventDisableTiming));
        ZMC_CUDA(cudaEventCreateWithFlags(&s.kernel_done[i], cudaEventDisableTiming));
    }
    return ZMC_OK;
}

zmc_status get_scratch(int dev, DeviceScratch** out) {
    if (dev < 0 || dev >= kMaxDevices) return ZMC_ERR_CUDA;
    DeviceScratch& s = g_scratch[dev];
    if (!s.init) {
        const zmc_status st = init_scratch(s, dev);
        if (st != ZMC_OK) { free_scratch(s); return st; }     // nothing half-created is left behind
        s.init = true;
    }
    *out = &s;
    return ZMC_OK;
}

uint64_t hash_lists(int M, const zmc_param_list* lists) {       // FNV-1a style, one 64-bit word (a length or a value) at a time
    uint64_t h = 1469598103934665603ull;
    for (int i = 0; i < M; ++i) {
        h = (h ^ (uint64_t)lists[i].count) * 1099511628211ull;
        for (int64_t j = 0; j < lists[i].count; ++j) {
            uint64_t bits;
            std::memcpy(&bits, &lists[i].values[j], sizeof(bits));
            h = (h ^ bits) * 1099511628211ull;
            h ^= h >> 29;
        }
    }
    return h;
}

bool same_lists(const ListSlot& c, int M, const zmc_param_list* lists, const uint32_t* list_off, size_t total) {
    if (!c.used || c.total != total) return false;
    for (int l = 0; l < M; ++l)
        if (std::memcmp(c.host + list_off[l], lists[l].values, (size_t)lists[l].count * sizeof(double)) != 0) return false;
    return true;
}

// H1: the device copy of the concatenated lists -- a cache hit enqueues nothing, a miss uploads through the slot's
// pinned buffer on `stream`.  *h2d_bytes = bytes actually copied by this call.
zmc_status stage_lists(DeviceScratch* s, int M, const zmc_param_list* lists, const uint32_t* list_off, size_t total,
                       bool fresh, cudaStream_t stream, ListSlot** out, size_t* h2d_bytes, bool* capturing_out) {
    // A call issued while `stream` is being captured bakes the slot's device pointer into the graph's kernel nodes, and the
    // graph may be replayed at any later time: such a slot is marked `captured` and stays as it is until zmc_shutdown.
    // A captured call cannot upload (the copy and its allocations would become graph nodes reading the library's pinned
    // buffer at replay time), so its lists must already be cached -- otherwise it is refused before anything is enqueued.
    cudaStreamCaptureStatus cap_status = cudaStreamCaptureStatusNone;
    ZMC_CUDA(cudaStreamIsCapturing(stream, &cap_status));
    const bool capturing = cap_status != cudaStreamCaptureStatusNone;
    *capturing_out = capturing;
    if (capturing) fresh = false;
    ListSlot* hit = nullptr;
    uint64_t h = 0;
    if (!fresh) {
        // the usual case first -- the same lists as the last call: one memcmp against the most recently used slot
        ListSlot* mru = &s->ring[0];
        for (int i = 1; i < kRing; ++i)
            if (s->ring[i].last_use > mru->last_use) mru = &s->ring[i];
        if (same_lists(*mru, M, lists, list_off, total)) hit = mru;
    }
    if (!hit) {
        h = hash_lists(M, lists);
        for (int i = 0; i < kRing && !hit && !fresh; ++i)
            if (s->ring[i].hash == h && same_lists(s->ring[i], M, lists, list_off, total)) hit = &s->ring[i];
    }
    *h2d_bytes = 0;
    if (capturing) {
        int n_captured = 0;
        for (int i = 0; i < kRing; ++i) n_captured += s->ring[i].captured ? 1 : 0;
        // not cached, or the last slot ordinary calls could still use: refuse (cudaErrorStreamCaptureUnsupported)
        if (!hit || (!hit->captured && n_captured >= kRing - 1)) return cuda_fail(cudaErrorStreamCaptureUnsupported);
        hit->captured = true;
    }
    if (hit) {
        // Order this stream's kernels after the upload unless it is known to be behind them already.  The stream HANDLE is
        // not proof: a destroyed stream's handle is reused by the next one created (zmc_scan_farm does that on every call),
        // so the same-handle shortcut is taken only while the upload has visibly completed or the slot has never been
        // read from another handle since.  (No event query during capture: not permitted there.)
        bool ordered = hit->last_stream == stream && !hit->multi_stream;
        if (ordered && !capturing && hit->upload_pending) {
            if (cudaEventQuery(hit->uploaded) == cudaSuccess) hit->upload_pending = false;
            else { cudaGetLastError(); ordered = false; }
        }
        if (!ordered) {
            ZMC_CUDA(cudaStreamWaitEvent(stream, hit->uploaded, 0));
            if (hit->last_stream != stream) hit->multi_stream = true;
        }
    } else {
        hit = nullptr;                          // victim: a free slot if there is one, else the least recently used; never a captured one
        for (int i = 0; i < kRing; ++i) {
            ListSlot* c = &s->ring[i];
            if (c->captured) continue;
            if (!hit || (hit->used && (!c->used || c->last_use < hit->last_use))) hit = c;
        }
        if (!hit) return ZMC_ERR_OUT_OF_MEMORY;  // cannot happen: at most kRing - 1 slots are ever captured
        if (hit->used) {                        // evict: every kernel that reads the old content must have finished
            if (hit->multi_stream) ZMC_CUDA(cudaDeviceSynchronize());
            else ZMC_CUDA(cudaEventSynchronize(hit->done));
            // a scan that failed after its upload never recorded `done`: the copy out of `host` may still be in flight
            if (hit->upload_pending) ZMC_CUDA(cudaEventSynchronize(hit->uploaded));
        }
        hit->used = false;
        if (hit->cap < total) {
            if (hit->host) cudaFreeHost(hit->host);
            if (hit->dev) cudaFree(hit->dev);
            hit->host = nullptr; hit->dev = nullptr; hit->cap = 0;
            ZMC_CUDA(cudaMallocHost(&hit->host, total * sizeof(double)));
            ZMC_CUDA(cudaMalloc(&hit->dev, total * sizeof(double)));
            hit->cap = total;
        }
        for (int l = 0; l < M; ++l)
            std::memcpy(hit->host + list_off[l], lists[l].values, (size_t)lists[l].count * sizeof(double));
        ZMC_CUDA(cudaMemcpyAsync(hit->dev, hit->host, total * sizeof(double), cudaMemcpyHostToDevice, stream));
        ZMC_CUDA(cudaEventRecord(hit->uploaded, stream));
        hit->hash = h; hit->total = total; hit->multi_stream = false; hit->used = true; hit->upload_pending = true;
        *h2d_bytes = total * sizeof(double);
    }
    hit->last_stream = stream;
    hit->last_use = ++s->use_counter;
    *out = hit;
    return ZMC_OK;
}

const KernelEntry* find_kernel(int family, int N, int precision, int fast, int schedule) {
    const KernelEntry* tables[] = {kEntriesC12, kEntriesC3, kEntriesC45, kEntriesP6, kEntriesDiag};
    const int sizes[] = {kNumEntriesC12, kNumEntriesC3, kNumEntriesC45, kNumEntriesP6, kNumEntriesDiag};
    const KernelEntry* generic = nullptr;
    for (int t = 0; t < 5; ++t) {
        for (int i = 0; i < sizes[t]; ++i) {
            const KernelEntry& e = tables[t][i];
            if (e.family != family || e.precision != precision || e.schedule != schedule) continue;
            if (precision == ZMC_PREC_F32E && e.fast != fast && family < ZMC_FAM_CONST_ONE) continue;
            if (e.n_dim == N) return &e;
            if (e.n_dim == 0) generic = &e;
        }
    }
    return generic;
}

struct TimedSpan { cudaEvent_t a = nullptr, b = nullptr; };

}  // namespace

// --------------------------------------------------------------------------------------------------
extern "C" {

int zmc_integrand_count(void) { return kNumFamilies; }

zmc_status zmc_integrand_info_at(int index, zmc_integrand_info* info) {
    if (!info || index < 0 || index >= kNumFamilies) return ZMC_ERR_INVALID_ARG;
    *info = kFamilies[index];
    return ZMC_OK;
}

zmc_status zmc_integrand_info_by_id(int integrand_id, zmc_integrand_info* info) {
    if (!info) return ZMC_ERR_INVALID_ARG;
    zmc_integrand_info user_info;
    const zmc_integrand_info* f = find_family(integrand_id, &user_info);
    if (!f) return ZMC_ERR_UNKNOWN_INTEGRAND;
    *info = *f;
    return ZMC_OK;
}

const char* zmc_status_string(zmc_status s) {
    switch (s) {
        case ZMC_OK: return "ok";
        case ZMC_ERR_INVALID_ARG: return "invalid argument";
        case ZMC_ERR_UNKNOWN_INTEGRAND: return "unknown integrand id";
        case ZMC_ERR_SHAPE_MISMATCH: return "(N, M, n_consts) not accepted by this integrand family";
        case ZMC_ERR_GRID_TOO_LARGE: return "parameter grid too large";
        case ZMC_ERR_OUT_OF_MEMORY: return "out of memory";
        case ZMC_ERR_CUDA: return "CUDA error (see zmc_last_cuda_error)";
        case ZMC_ERR_COMPILE: return "user integrand did not compile (see zmc_last_compile_log)";
        case ZMC_ERR_NOALLOC_LIMIT: return "value lists exceed ZMC_NOALLOC_MAX_LIST_VALUES entries in total (zmc_scan_noalloc has a fixed buffer; use zmc_scan_ex)";
    }
    return "unknown status";
}

int zmc_last_cuda_error(void) { return tl_cuda_error; }

const char* zmc_version(void) { return "zmc_scan 0.1 (sm_100a)"; }

zmc_status zmc_validate(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                        uint64_t n_samples, const zmc_options* opt, uint64_t* grid_points) {
    Options o;
    zmc_status st = read_options(opt, &o);
    if (st != ZMC_OK) return st;
    return validate(integrand_id, N, bounds, M, lists, n_samples, o, grid_points, nullptr, nullptr);
}

// H6 schedule choice.  R = threads the device keeps resident: the fp64 kernels are launch-bounded to 3 CTAs of 256
// per SM, the fp32-evaluate ones to 4 (zmc_kernel.cuh); the SM count is the current device's (looked up once per device; 148, a
// B200's, while no device is visible).  THREAD needs >= 8 rounds of R (measured on cfg 2, 8.8 rounds: 2.8 % faster
// than WARP because rounds 1-2 of Philox run on the uniform datapath); WARP needs 2 rounds of R/32 resident warps
// (measured on B200 for the cfg 1-3 families with 2000-16000 points x 5000-50000 samples: below that the finer
// granularity of one CTA per point wins by up to 20 %, above it WARP by 5-15 % -- one shuffle tree instead of a tree,
// a barrier and a second tree per point); else CTA.  A point with few sample groups cannot feed 32 / 256 lanes, so
// small n falls back to fewer lanes.
static int current_sm_count() {     // of the CURRENT device, remembered per device; nothing is latched while no device answers
    static std::atomic<int> known[kMaxDevices];
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return 148; }
    if ((n = known[dev].load(std::memory_order_relaxed)) > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) { cudaGetLastError(); return 148; }
    known[dev].store(n, std::memory_order_relaxed);
    return n;
}

int zmc_pick_schedule_ex(uint64_t count, uint64_t n_samples, int N, int precision) {
    const uint64_t resident = (uint64_t)current_sm_count() * (precision == ZMC_PREC_F32E ? 1024ull : 768ull);
    const int g4 = (N % 4 == 0) ? 4 : (N % 2 == 0) ? 2 : 1;
    const uint64_t groups = n_samples / (uint64_t)(4 / g4) + 1;
    if (count >= 8 * resident || groups < 4 * 32) return ZMC_SCHED_THREAD;
    if (count >= 2 * (resident / 32) || groups < 4 * 256) return ZMC_SCHED_WARP;
    return ZMC_SCHED_CTA;
}

int zmc_pick_schedule(uint64_t count, uint64_t n_samples, int N) {
    return zmc_pick_schedule_ex(count, n_samples, N, ZMC_PREC_F64);
}

int64_t zmc_batch_range(uint64_t first_index, uint64_t count, uint64_t batch_points, int64_t b,
                        uint64_t* batch_first, uint64_t* batch_count) {
    if (batch_points == 0 || batch_points > count) batch_points = count;
    const int64_t nb = count ? (int64_t)((count + batch_points - 1) / batch_points) : 0;
    if (b >= 0 && b < nb) {
        const uint64_t f = first_index + (uint64_t)b * batch_points;
        const uint64_t c = ((uint64_t)b == (uint64_t)nb - 1) ? first_index + count - f : batch_points;
        if (batch_first) *batch_first = f;
        if (batch_count) *batch_count = c;
    }
    return nb;
}

void zmc_shutdown(void) {
    int cur = 0;
    const bool have = cudaGetDevice(&cur) == cudaSuccess;
    for (int d = 0; d < kMaxDevices; ++d) {
        std::lock_guard<std::mutex> lock(g_dev_mutex[d]);
        if (!g_scratch[d].init) continue;
        if (have) cudaSetDevice(d);
        free_scratch(g_scratch[d]);
    }
    if (have) cudaSetDevice(cur);
    unload_user_integrands();
}

zmc_status zmc_scan(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                    uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream) {
    return zmc_scan_ex(integrand_id, N, bounds, M, lists, n_samples, seed, out_mean, out_stderr, stream,
                       nullptr, nullptr);
}

}  // extern "C"

namespace zmc {

// The one scan routine behind zmc_scan_ex, zmc_scan_adaptive and the farm's feeder threads.
zmc_status scan_impl(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                     uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream_v,
                     const zmc_options* opt, zmc_timing* timing, const AdaptArgs* ad) {
    // ---- H1: validate -----------------------------------------------------------------------
    Options o;
    zmc_status st = read_options(opt, &o);
    if (st != ZMC_OK) return st;
    if (ad) {
        if (!ad->out_n) return ZMC_ERR_INVALID_ARG;
        if (n_samples < 256 || n_samples % 256 != 0) return ZMC_ERR_INVALID_ARG;           // lane ownership, see kernel
        if (ad->n_max < n_samples || ad->n_max % 8 != 0 || ad->n_max > 0xFFFFFFF8ull) return ZMC_ERR_INVALID_ARG;
        if (ad->n_max * (uint64_t)(N > 0 ? N : 1) > (1ull << 34)) return ZMC_ERR_INVALID_ARG;
        if (!(ad->target >= 0.0) || !std::isfinite(ad->target)) return ZMC_ERR_INVALID_ARG;
    }
    uint64_t G = 0, first = 0, count = 0;
    st = validate(integrand_id, N, bounds, M, lists, n_samples, o, &G, &first, &count);
    if (st != ZMC_OK) return st;
    if (!out_mean || !out_stderr) return ZMC_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    if (timing) std::memset(timing, 0, sizeof(*timing));

    const bool f32e = o.precision == ZMC_PREC_F32E;
    const int fast = f32e ? (o.fast_math == ZMC_FAST_MATH_OFF ? 0 : 1) : 0;
    const int schedule = ad ? (int)kSchedAdapt
                       : o.schedule == ZMC_SCHED_AUTO ? zmc_pick_schedule_ex(count, n_samples, N, o.precision) : o.schedule;
    const std::shared_ptr<const UserIntegrand> user = integrand_id >= kFirstUserId ? find_user_integrand(integrand_id) : nullptr;   // held for the whole call
    const KernelEntry* kern = user ? nullptr : find_kernel(integrand_id, N, o.precision, fast, schedule);
    if (!kern && !user) return ZMC_ERR_UNKNOWN_INTEGRAND;
    if (timing) { timing->schedule = ad ? (int)ZMC_SCHED_WARP : schedule; timing->host_out_pinned = -1; }
    if (count == 0) return ZMC_OK;

    int dev = 0;
    ZMC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return ZMC_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_dev_mutex[dev]);
    DeviceScratch* s = nullptr;
    st = get_scratch(dev, &s);
    if (st != ZMC_OK) return st;

    if (timing || o.out_location == ZMC_LOC_HOST) {     // these synchronise / copy on a side stream: not capturable, say so up front
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        ZMC_CUDA(cudaStreamIsCapturing(stream, &cs));
        if (cs != cudaStreamCaptureStatusNone) return cuda_fail(cudaErrorStreamCaptureUnsupported);
    }

    // ---- parameter block -----------------------------------------------------------------------
    ScanParams p;
    std::memset(&p, 0, sizeof(p));
    auto mirror = [f32e](double v) { return f32e ? (double)(float)v : v; };
    p.n = (uint32_t)n_samples;
    p.n_dim = (uint32_t)N;
    p.n_par = (uint32_t)M;
    p.out_f32 = o.out_dtype == ZMC_OUT_F32;
    p.volume = 1.0;
    for (int k = 0; k < N; ++k) {
        p.a[k] = mirror(bounds[2 * k]);
        p.width[k] = mirror(bounds[2 * k + 1] - bounds[2 * k]);
        p.volume *= p.width[k];
    }
    for (int c = 0; c < o.n_consts; ++c) p.consts[c] = mirror(o.consts[c]);
    {
        uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        for (int r = 0; r < 10; ++r) {
            p.rk[2 * r] = k0;
            p.rk[2 * r + 1] = k1;
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
    }
    size_t total = 0;
    for (int i = 0; i < M; ++i) {
        p.counts[i] = (uint32_t)lists[i].count;
        p.list_off[i] = (uint32_t)total;
        total += (size_t)lists[i].count;
    }
    if (total > 0xFFFFFFFFull) return ZMC_ERR_GRID_TOO_LARGE;
    p.lists_total = (uint32_t)total;
    // H3: reciprocals for the per-point digit extraction.  With s = max(2, ceil(log2 L)), P = 30 + s >= 32 and
    // m = floor(2^P / L) + 1 < 2^32:  m L - 2^P = e in (0, L], so r m / 2^P = r / L + r e / (L 2^P) and the second term is
    // below 1 / L for every r < 2^P / e, in particular for r < 2^30 (local indices of a launch): floor(r m / 2^P) = floor(r / L).
    for (int i = 0; i < M; ++i) {
        const uint64_t L = p.counts[i];
        int sh = 2;
        while ((1ull << sh) < L) ++sh;
        p.div_m[i] = L > 1 ? (uint32_t)((1ull << (30 + sh)) / L + 1) : 0u;
        p.div_s[i] = (uint32_t)(30 + sh - 32);
    }
    p.inv_n = 1.0 / (double)p.n;
    p.nn1 = (double)(p.n - 1) * (double)p.n;
    const size_t elem_eval = f32e ? 4 : 8;
    // shared-memory staging pays off when a CTA serves many points (THREAD schedule) and the lists fit
    const size_t smem_bytes = (schedule == ZMC_SCHED_THREAD && total * elem_eval <= 48 * 1024) ? total * elem_eval : 0;
    p.stage_smem = smem_bytes ? 1u : 0u;

    // timing events come from a per-device pool (created once, reused by every call)
    size_t pool_next = 0;
    auto new_tev = [s, &pool_next](cudaEvent_t* e) -> cudaError_t {
        if (pool_next == s->timing_pool.size()) {
            cudaEvent_t fresh = nullptr;
            const cudaError_t err = cudaEventCreate(&fresh);
            if (err != cudaSuccess) return err;
            s->timing_pool.push_back(fresh);
        }
        *e = s->timing_pool[pool_next++];
        return cudaSuccess;
    };

    // Timing events.  A one-batch scan into device memory whose lists are already cached is bracketed by two events
    // only (begin = kernel start, end = kernel end): on a 10^3-point grid every extra event is microseconds of a
    // 25-microsecond call.
    cudaEvent_t ev_begin = nullptr, ev_h2d = nullptr, ev_end = nullptr;
    if (timing) {
        ZMC_CUDA(new_tev(&ev_begin)); ZMC_CUDA(new_tev(&ev_end));
        ZMC_CUDA(cudaEventRecord(ev_begin, stream));
    }
    // ---- H1: the lists on the device (cached by content; a hit copies nothing) ----------------------------
    ListSlot* slot = nullptr;
    size_t h2d_bytes = 0;
    bool capturing = false;
    st = stage_lists(s, M, lists, p.list_off, total, (o.flags & ZMC_OPT_FRESH_LISTS) != 0, stream, &slot, &h2d_bytes, &capturing);
    if (st != ZMC_OK) return st;
    p.lists = slot->dev;
    if (timing && h2d_bytes) { ZMC_CUDA(new_tev(&ev_h2d)); ZMC_CUDA(cudaEventRecord(ev_h2d, stream)); }

    // ---- H2: batches ----------------------------------------------------------------------------------
    bool host_out = o.out_location == ZMC_LOC_HOST;
    const size_t elem_out = p.out_f32 ? 4 : 8;
    const int64_t n_batches = zmc_batch_range(first, count, o.batch_points, -1, nullptr, nullptr);
    uint64_t batch_max = (o.batch_points == 0 || o.batch_points > count) ? count : o.batch_points;
    // H8, small results: a one-batch scan whose results fit kDirectBytes and whose HOST buffers are page-locked and
    // mapped is written by the kernel itself, straight into host memory (posted writes over PCIe / C2C): no staging
    // buffer, no copy, no side stream.  For a 10^3-point grid the two copies and their events cost more than the kernel.
    constexpr size_t kDirectBytes = 1u << 20;
    bool direct = false;
    uint64_t direct_bytes = 0;
    uint32_t* direct_out_n = nullptr;
    if (host_out) {
        // Device alias of a page-locked, mapped host range, or NULL.  Both ends of the range are looked up: a buffer that
        // only STARTS in registered memory (a slice near the end of a cudaHostRegister'ed region, pageable memory behind
        // it) must take the staged path -- the kernel would fault on the part that is not mapped.
        auto mapped_alias = [](const void* host_ptr, size_t bytes) -> void* {
            cudaPointerAttributes first, last;
            if (bytes == 0 || cudaPointerGetAttributes(&first, host_ptr) != cudaSuccess || first.type != cudaMemoryTypeHost ||
                !first.devicePointer) return nullptr;
            if (cudaPointerGetAttributes(&last, static_cast<const char*>(host_ptr) + bytes - 1) != cudaSuccess ||
                last.type != cudaMemoryTypeHost || !last.devicePointer) return nullptr;
            if (static_cast<char*>(last.devicePointer) - static_cast<char*>(first.devicePointer) != (ptrdiff_t)(bytes - 1)) return nullptr;
            return first.devicePointer;
        };
        cudaPointerAttributes pa;
        const bool pinned = cudaPointerGetAttributes(&pa, out_mean) == cudaSuccess && pa.type == cudaMemoryTypeHost;
        cudaGetLastError();
        if (timing) timing->host_out_pinned = pinned ? 1 : 0;   // copies into pageable memory run synchronously on the host
        direct_bytes = count * (elem_out * 2 + (ad ? sizeof(uint32_t) : 0));
        if (pinned && n_batches == 1 && direct_bytes <= kDirectBytes) {
            void* d_mean = mapped_alias(out_mean, (size_t)count * elem_out);
            void* d_err = d_mean ? mapped_alias(out_stderr, (size_t)count * elem_out) : nullptr;
            direct_out_n = (d_err && ad) ? static_cast<uint32_t*>(mapped_alias(ad->out_n, (size_t)count * sizeof(uint32_t))) : nullptr;
            if (d_mean && d_err && (!ad || direct_out_n)) {
                direct = true;
                host_out = false;                                   // from here on: an ordinary one-batch scan into "device" pointers
                out_mean = d_mean;
                out_stderr = d_err;
                if (timing) timing->host_out_pinned = 2;            // 2 = pinned and written directly by the kernel
            }
        }
        cudaGetLastError();
    }
    if (host_out) {
        const size_t need = (size_t)batch_max * (elem_out * 2 + (ad ? sizeof(uint32_t) : 0));
        if (s->stage_cap < need) {
            for (int i = 0; i < 2; ++i) {          // wait for the copies still reading the old buffers, nothing else
                if (s->stage_used[i]) ZMC_CUDA(cudaEventSynchronize(s->stage_free[i]));
                if (s->stage[i]) cudaFree(s->stage[i]);
                s->stage[i] = nullptr;
            }
            s->stage_cap = 0; s->stage_used[0] = s->stage_used[1] = false;
            ZMC_CUDA(cudaMalloc(&s->stage[0], need));
            s->stage_cap = need;
        }
        if (!s->stage[1]) ZMC_CUDA(cudaMalloc(&s->stage[1], s->stage_cap));   // both: the buffers alternate across calls too
    }

    // One worker (thread / warp / CTA) per grid point, one CTA per `per_cta` points: the hardware CTA scheduler
    // balances the load.  A batch larger than kMaxLaunchPoints is cut into several launches so that local point
    // indices and the grid size stay 32-bit.
    const uint64_t per_cta = schedule == ZMC_SCHED_THREAD ? kThreads
                           : (schedule == ZMC_SCHED_WARP || schedule == kSchedAdapt) ? kThreads / 32 : 1;
    if (ad) {
        p.n_max = (uint32_t)ad->n_max; p.target = ad->target; p.out_n = ad->out_n;
        if (direct) p.out_n = direct_out_n;                     // the device alias of the caller's host array
    }
    constexpr uint64_t kMaxLaunchPoints = 1ull << 30;

    std::vector<TimedSpan> t_kernel, t_copy;
    int64_t launches = 0;
    uint64_t d2h_bytes = 0;
    for (int64_t b = 0; b < n_batches; ++b) {
        uint64_t bf = 0, bc = 0;
        zmc_batch_range(first, count, o.batch_points, b, &bf, &bc);
        void *dst_mean, *dst_err;
        uint64_t out_base;                     // flat index of element 0 of dst_mean / dst_err
        const int buf = host_out ? (int)(s->stage_rot++ & 1u) : 0;
        if (host_out) {
            if (s->stage_used[buf]) ZMC_CUDA(cudaStreamWaitEvent(stream, s->stage_free[buf], 0));
            dst_mean = s->stage[buf];
            dst_err = static_cast<char*>(s->stage[buf]) + (size_t)batch_max * elem_out;
            if (ad) p.out_n = reinterpret_cast<uint32_t*>(static_cast<char*>(s->stage[buf]) + (size_t)batch_max * elem_out * 2);
            out_base = bf;
        } else {
            dst_mean = out_mean;
            dst_err = out_stderr;
            out_base = first;
        }
        TimedSpan tk;
        const bool lean = timing && !host_out && n_batches == 1 && !ev_h2d;      // the call's two events are the kernel's
        if (lean) { tk.a = ev_begin; tk.b = ev_end; }
        else if (timing) { ZMC_CUDA(new_tev(&tk.a)); ZMC_CUDA(new_tev(&tk.b)); ZMC_CUDA(cudaEventRecord(tk.a, stream)); }
        for (uint64_t lf = bf, lc_done = 0; lf < bf + bc; lf += lc_done) {
            uint64_t lc = (bf + bc - lf < kMaxLaunchPoints) ? bf + bc - lf : kMaxLaunchPoints;
            const uint64_t to_wrap = (1ull << 32) - (lf & 0xFFFFFFFFull);   // the high word of t is launch-uniform
            if (lc > to_wrap) lc = to_wrap;
            p.first = lf;
            p.count = (uint32_t)lc;
            p.out_off = lf - out_base;
            {   // H3, 64-bit part: mixed-radix digits of the launch's first flat index
                uint64_t rest = lf;
                for (int i = M - 1; i >= 1; --i) { p.base_digits[i] = (uint32_t)(rest % p.counts[i]); rest /= p.counts[i]; }
                p.base_digits[0] = (uint32_t)rest;
            }
            const uint64_t grid = (lc + per_cta - 1) / per_cta;
            if (user) ZMC_CUDA(launch_user(*user, o.precision, schedule, p, dst_mean, dst_err, (int)grid, smem_bytes, stream));
            else ZMC_CUDA(kern->launch(p, dst_mean, dst_err, (int)grid, smem_bytes, stream));
            ++launches;
            lc_done = lc;
        }
        if (timing) { if (!lean) ZMC_CUDA(cudaEventRecord(tk.b, stream)); t_kernel.push_back(tk); }

        if (host_out) {   // H8: copy batch b on the side stream while batch b+1 computes
            ZMC_CUDA(cudaEventRecord(s->kernel_done[buf], stream));
            ZMC_CUDA(cudaStreamWaitEvent(s->side, s->kernel_done[buf], 0));
            TimedSpan tc;
            if (timing) { ZMC_CUDA(new_tev(&tc.a)); ZMC_CUDA(new_tev(&tc.b)); ZMC_CUDA(cudaEventRecord(tc.a, s->side)); }
            const size_t off = (size_t)(bf - first) * elem_out, bytes = (size_t)bc * elem_out;
            ZMC_CUDA(cudaMemcpyAsync(static_cast<char*>(out_mean) + off, dst_mean, bytes, cudaMemcpyDeviceToHost, s->side));
            ZMC_CUDA(cudaMemcpyAsync(static_cast<char*>(out_stderr) + off, dst_err, bytes, cudaMemcpyDeviceToHost, s->side));
            d2h_bytes += 2 * bytes;
            if (ad) {
                ZMC_CUDA(cudaMemcpyAsync(ad->out_n + (bf - first), p.out_n, (size_t)bc * sizeof(uint32_t), cudaMemcpyDeviceToHost, s->side));
                d2h_bytes += (size_t)bc * sizeof(uint32_t);
            }
            if (timing) { ZMC_CUDA(cudaEventRecord(tc.b, s->side)); t_copy.push_back(tc); }
            ZMC_CUDA(cudaEventRecord(s->stage_free[buf], s->side));
            s->stage_used[buf] = true;
        }
    }
    if (!capturing) ZMC_CUDA(cudaEventRecord(slot->done, stream));   // a captured slot is never evicted: nothing waits on `done`
    if (host_out) {   // join the side stream back into `stream`
        const int last = (int)((s->stage_rot - 1u) & 1u);
        ZMC_CUDA(cudaStreamWaitEvent(stream, s->stage_free[last], 0));
    }

    if (timing) {
        ZMC_CUDA(cudaEventRecord(ev_end, stream));
        ZMC_CUDA(cudaEventSynchronize(ev_end));
        float ms = 0.f;
        if (ev_h2d) { ZMC_CUDA(cudaEventElapsedTime(&ms, ev_begin, ev_h2d)); timing->h2d_ms = ms; }
        ZMC_CUDA(cudaEventElapsedTime(&ms, ev_begin, ev_end)); timing->wall_ms = ms;
        for (auto& k : t_kernel) { ZMC_CUDA(cudaEventElapsedTime(&ms, k.a, k.b)); timing->kernel_ms += ms; }
        for (auto& c : t_copy) { ZMC_CUDA(cudaEventElapsedTime(&ms, c.a, c.b)); timing->d2h_ms += ms; }
        const double exposed = timing->wall_ms - timing->h2d_ms - timing->kernel_ms;
        timing->exposed_d2h_ms = host_out ? (exposed > 0 ? exposed : 0.0) : 0.0;
        timing->n_batches = n_batches;
        timing->gpu_launches = launches;
        timing->d2h_bytes = direct ? direct_bytes : d2h_bytes;     // direct: written by the kernel, inside kernel_ms
        timing->h2d_bytes = h2d_bytes;
    }
    return ZMC_OK;
}

}  // namespace zmc

extern "C" {

zmc_status zmc_scan_ex(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                       uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream,
                       const zmc_options* opt, zmc_timing* timing) {
    return scan_impl(integrand_id, N, bounds, M, lists, n_samples, seed, out_mean, out_stderr, stream, opt, timing, nullptr);
}

zmc_status zmc_scan_adaptive(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                             uint64_t n_first, uint64_t n_max, double target_stderr, uint64_t seed, void* out_mean,
                             void* out_stderr, uint32_t* out_n, void* stream, const zmc_options* opt, zmc_timing* timing) {
    const AdaptArgs ad{n_max, target_stderr, out_n};
    return scan_impl(integrand_id, N, bounds, M, lists, n_first, seed, out_mean, out_stderr, stream, opt, timing, &ad);
}

}  // extern "C"
