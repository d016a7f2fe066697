// zmc_noalloc.cu -- zmc_scan_noalloc (include/zmc.h): the fixed-n scan for callers that must not allocate GPU memory.
//
// Who cannot allocate, and why.  cudaMalloc / cudaFree are not ordinary enqueues: they take a driver lock, may
// synchronise the whole device, and change the amount of free memory under the caller's feet.  That rules them out for
//   - a service that handed ALL device memory to its own pool at start-up (an inference server, a framework's caching
//     allocator): a library that quietly takes some more can push the owner into an out-of-memory error later;
//   - a caller inside a latency-critical loop (one scan per control / trigger / time step), where a device-wide
//     synchronisation in the middle of the loop stalls every other stream;
//   - a caller whose memory budget was signed off in advance (a fixed plan of buffers, nothing may appear that is not
//     in the plan).
// The ordinary path (zmc_scan_ex, zmc_api.cu) keeps a scratch copy of the concatenated value lists in device memory it
// allocates on demand (ListSlot::dev) -- the only global memory the scan kernel touches besides its outputs.  Here that
// scratch is a file-scope __device__ array of fixed size instead: part of the library image, present on every GPU that
// loads libzmc.so until the process exits, never allocated and never freed.
//
// Rules that follow from a shared static array (also stated in zmc.h):
//   - the lists of one call must fit ZMC_NOALLOC_MAX_LIST_VALUES doubles in total, else ZMC_ERR_NOALLOC_LIMIT;
//   - every call on a device uses the SAME array.  Calls that follow one another on one stream are ordered by the
//     stream; calls whose GPU work can overlap (different streams, or two host threads) race on it;
//   - the array keeps what the previous call left there.  Nothing in it has to start at zero: each call overwrites the
//     entries [0, total) its kernels read before they run, and reads nothing beyond them.
//
// The array's name below is, in HOST code, only a handle for the runtime -- not a device address.  The address the
// kernels need is asked for once per device with cudaGetSymbolAddress (that device current) and then passed in the
// parameter block like any other pointer.  Device code in this file (the staging kernel) names the array directly.
//
// This file adds an entry point next to the existing ones; it shares their kernels (the dispatch tables of the
// zmc_inst_*.cu units) and repeats, on purpose, the few lines of zmc_api.cu that fill the parameter block, so that the
// existing path is untouched.  tests/test_zz_no_alloc.py holds the two paths bit-identical.
#include <cmath>
#include <cstring>
#include <mutex>

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

// The scratch: the concatenated value lists of the call in progress (32 KiB per GPU, see the header of this file).
static __device__ __align__(256) double g_noalloc_lists[ZMC_NOALLOC_MAX_LIST_VALUES];

// H1 without a copy engine and without a staging buffer: the list values travel as KERNEL ARGUMENTS (copied by the
// launch itself, so the caller's host memory is free again when the call returns) and one small CTA writes them into
// the scratch array.  One chunk stays below the 4 KB every CUDA version accepts for kernel arguments.
constexpr uint32_t kChunkValues = 448;
struct StageChunk {
    uint32_t offset, count;          // g_noalloc_lists[offset + i] = v[i], i < count
    double v[kChunkValues];
};
static_assert(sizeof(StageChunk) <= 4096 - 64, "one chunk must fit the classic kernel-argument limit");

__global__ void __launch_bounds__(256)
zmc_noalloc_stage_kernel(const __grid_constant__ StageChunk c)
{
    for (uint32_t i = threadIdx.x; i < c.count; i += blockDim.x) g_noalloc_lists[c.offset + i] = c.v[i];
}

// Device address of g_noalloc_lists, per device (index = device ordinal).  Filled by the first call on that device.
constexpr int kMaxDevices = 64;
double* g_scratch_addr[kMaxDevices];
std::mutex g_setup_mutex;

zmc_status cuda_fail(cudaError_t e) {
    set_last_cuda_error((int)e);
    cudaGetLastError();      // do not leave the failed call in the runtime's last-error slot for the next launch to find
    return ZMC_ERR_CUDA;
}
#define ZMC_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e__ = (call);                        \
        if (e__ != cudaSuccess) return cuda_fail(e__);   \
    } while (0)

// Set-up, once per device, with that device current: turn the host-side handle into the device address.
zmc_status scratch_address(int dev, double** out) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        int cur = -1;
        ZMC_CUDA(cudaGetDevice(&cur));
        if (cur != dev) return ZMC_ERR_CUDA;             // the caller looked `dev` up a moment ago; it must still be current
        double* ptr = nullptr;
        ZMC_CUDA(cudaGetSymbolAddress((void**)&ptr, g_noalloc_lists));
        if (!ptr) return ZMC_ERR_CUDA;
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return ZMC_OK;
}

// the same lookup zmc_api.cu does over the instantiation units' tables
const KernelEntry* find_builtin_kernel(int family, int N, int precision, int fast, int schedule) {
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

}  // namespace

extern "C" zmc_status zmc_scan_noalloc(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                                       uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr,
                                       void* stream_v, const zmc_options* opt)
{
    // ---- argument checks: nothing is enqueued and no output is touched when one fails -------------------------
    if (integrand_id >= kFirstUserId) return ZMC_ERR_UNKNOWN_INTEGRAND;      // run-time compiled integrands load code: not here
    if (opt && opt->struct_size >= sizeof(zmc_options) && opt->out_location != ZMC_LOC_DEVICE)
        return ZMC_ERR_INVALID_ARG;                                          // host outputs need a staging buffer: not here
    uint64_t G = 0;
    zmc_status st = zmc_validate(integrand_id, N, bounds, M, lists, n_samples, opt, &G);   // exactly zmc_scan_ex's checks
    if (st != ZMC_OK) return st;
    if (!out_mean || !out_stderr) return ZMC_ERR_INVALID_ARG;
    uint64_t total = 0;
    for (int i = 0; i < M; ++i) total += (uint64_t)lists[i].count;
    if (total > ZMC_NOALLOC_MAX_LIST_VALUES) return ZMC_ERR_NOALLOC_LIMIT;

    const int precision = opt ? opt->precision : ZMC_PREC_F64;
    const bool f32e = precision == ZMC_PREC_F32E;
    const int fast = f32e ? ((opt && opt->fast_math == ZMC_FAST_MATH_OFF) ? 0 : 1) : 0;
    const uint64_t first = opt ? opt->first_index : 0;
    const uint64_t count = (opt && (opt->count || (opt->flags & ZMC_OPT_EXPLICIT_COUNT))) ? opt->count : G - first;
    const int schedule = (!opt || opt->schedule == ZMC_SCHED_AUTO) ? zmc_pick_schedule_ex(count, n_samples, N, precision)
                                                                   : opt->schedule;
    const KernelEntry* kern = find_builtin_kernel(integrand_id, N, precision, fast, schedule);
    if (!kern) return ZMC_ERR_UNKNOWN_INTEGRAND;
    if (count == 0) return ZMC_OK;

    int dev = 0;
    ZMC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return ZMC_ERR_CUDA;
    double* scratch = nullptr;
    st = scratch_address(dev, &scratch);
    if (st != ZMC_OK) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);

    // ---- parameter block: the same values, computed by the same operations, as scan_impl in zmc_api.cu --------------
    ScanParams p;
    std::memset(&p, 0, sizeof(p));
    auto mirror = [f32e](double v) { return f32e ? (double)(float)v : v; };
    p.n = (uint32_t)n_samples;
    p.n_dim = (uint32_t)N;
    p.n_par = (uint32_t)M;
    p.out_f32 = opt ? opt->out_dtype == ZMC_OUT_F32 : 0;
    p.volume = 1.0;
    for (int k = 0; k < N; ++k) {
        p.a[k] = mirror(bounds[2 * k]);
        p.width[k] = mirror(bounds[2 * k + 1] - bounds[2 * k]);
        p.volume *= p.width[k];
    }
    for (int c = 0; opt && c < opt->n_consts; ++c) p.consts[c] = mirror(opt->consts[c]);
    {
        uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        for (int r = 0; r < 10; ++r) {
            p.rk[2 * r] = k0;
            p.rk[2 * r + 1] = k1;
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
    }
    {
        uint32_t off = 0;
        for (int i = 0; i < M; ++i) {
            p.counts[i] = (uint32_t)lists[i].count;
            p.list_off[i] = off;
            off += (uint32_t)lists[i].count;
        }
    }
    p.lists_total = (uint32_t)total;
    for (int i = 0; i < M; ++i) {            // H3: round-up reciprocals (proof in zmc_api.cu)
        const uint64_t L = p.counts[i];
        int sh = 2;
        while ((1ull << sh) < L) ++sh;
        p.div_m[i] = L > 1 ? (uint32_t)((1ull << (30 + sh)) / L + 1) : 0u;
        p.div_s[i] = (uint32_t)(30 + sh - 32);
    }
    p.inv_n = 1.0 / (double)p.n;
    p.nn1 = (double)(p.n - 1) * (double)p.n;
    const size_t elem_eval = f32e ? 4 : 8;
    const size_t smem_bytes = (schedule == ZMC_SCHED_THREAD && total * elem_eval <= 48 * 1024) ? total * elem_eval : 0;
    p.stage_smem = smem_bytes ? 1u : 0u;
    p.lists = scratch;                       // the device address from cudaGetSymbolAddress, never the symbol itself

    // ---- H1: the lists into the scratch array, as kernel arguments, on `stream` ahead of the scan kernels -----------
    {
        StageChunk chunk;
        chunk.offset = 0;
        chunk.count = 0;
        auto flush = [&]() -> cudaError_t {
            if (chunk.count == 0) return cudaSuccess;
            zmc_noalloc_stage_kernel<<<1, 256, 0, stream>>>(chunk);
            chunk.offset += chunk.count;
            chunk.count = 0;
            return cudaGetLastError();
        };
        for (int l = 0; l < M; ++l) {
            for (int64_t j = 0; j < lists[l].count; ++j) {
                chunk.v[chunk.count++] = lists[l].values[j];
                if (chunk.count == kChunkValues) ZMC_CUDA(flush());
            }
        }
        ZMC_CUDA(flush());
    }

    // ---- the scan itself: one batch, cut into launches of at most 2^30 points that do not straddle a multiple of 2^32
    const uint64_t per_cta = schedule == ZMC_SCHED_THREAD ? kThreads : schedule == ZMC_SCHED_WARP ? kThreads / 32 : 1;
    constexpr uint64_t kMaxLaunchPoints = 1ull << 30;
    for (uint64_t lf = first, lc = 0; lf < first + count; lf += lc) {
        lc = (first + count - lf < kMaxLaunchPoints) ? first + count - lf : kMaxLaunchPoints;
        const uint64_t to_wrap = (1ull << 32) - (lf & 0xFFFFFFFFull);
        if (lc > to_wrap) lc = to_wrap;
        p.first = lf;
        p.count = (uint32_t)lc;
        p.out_off = lf - first;
        uint64_t rest = lf;                  // H3, 64-bit part: mixed-radix digits of the launch's first flat index
        for (int i = M - 1; i >= 1; --i) { p.base_digits[i] = (uint32_t)(rest % p.counts[i]); rest /= p.counts[i]; }
        p.base_digits[0] = (uint32_t)rest;
        const uint64_t grid = (lc + per_cta - 1) / per_cta;
        ZMC_CUDA(kern->launch(p, out_mean, out_stderr, (int)grid, smem_bytes, stream));
    }
    return ZMC_OK;
}
