// zmc_farm.cu -- NEXT-2 of SURVEY.md 8(f): the paper's title feature on one node.  PAPER.md:65 "we cut the parameter
// grid into several batches. Each batch is fed into one GPU device for evaluation"; PAPER.md:81 (Fig. 1) and Table 2
// (:132-140): batches are farmed out to whatever GPUs there are (its cluster mixes K40m, K80 and V100, so the
// assignment has to be dynamic).  Here: one host thread per device pulls batch indices from a shared atomic counter
// and scans each batch with zmc_scan_ex(first_index, count) straight into its slice of ONE host result array.
// No collective and no inter-device traffic: every random word is keyed by the global flat index, so the result is
// bit-identical to a single-device scan whatever the assignment turns out to be.
#include <atomic>
#include <chrono>
#include <cstring>
#include <thread>
#include <vector>

#include "zmc_internal.h"
#include "zmc_params.h"

namespace {

// n_samples is the fixed sample count, or (ad != nullptr) the first checkpoint of the adaptive scan
zmc_status farm_impl(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                     uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, const zmc::AdaptArgs* ad,
                     const int* devices, int n_devices, const zmc_options* opt, zmc_farm_timing* timing) {
    if (!devices || n_devices < 1 || n_devices > ZMC_MAX_FARM_DEVICES || !out_mean || !out_stderr) return ZMC_ERR_INVALID_ARG;
    zmc_options o;
    std::memset(&o, 0, sizeof(o));
    o.struct_size = sizeof(o);
    o.fast_math = ZMC_FAST_MATH_DEFAULT;
    if (opt) {
        if (opt->struct_size < sizeof(zmc_options)) return ZMC_ERR_INVALID_ARG;
        o = *opt;
    }
    o.out_location = ZMC_LOC_HOST;                 // several devices write one array: it has to live on the host
    uint64_t G = 0;
    zmc_status st = zmc_validate(integrand_id, N, bounds, M, lists, n_samples, &o, &G);
    if (st != ZMC_OK) return st;
    int n_visible = 0;
    if (cudaGetDeviceCount(&n_visible) != cudaSuccess || n_visible < 1) return ZMC_ERR_CUDA;
    for (int d = 0; d < n_devices; ++d)
        if (devices[d] < 0 || devices[d] >= n_visible) return ZMC_ERR_INVALID_ARG;

    const uint64_t first = o.first_index;
    const uint64_t count = (o.count || (o.flags & ZMC_OPT_EXPLICIT_COUNT)) ? o.count : G - first;
    if (timing) std::memset(timing, 0, sizeof(*timing));
    if (count == 0) return ZMC_OK;
    // AUTO is resolved once, from the whole range, so that every batch sums in the same order as a one-device scan
    if (o.schedule == ZMC_SCHED_AUTO) o.schedule = zmc_pick_schedule_ex(count, n_samples, N, o.precision);
    // default batch: ~8 batches per device so a slow device does not hold the tail (18 s vs 89 s per batch)
    uint64_t bp = o.batch_points ? o.batch_points : (count + 8ull * n_devices - 1) / (8ull * n_devices);
    if (bp > (1ull << 30)) bp = 1ull << 30;
    const int64_t n_batches = zmc_batch_range(first, count, bp, -1, nullptr, nullptr);
    const size_t elem = o.out_dtype == ZMC_OUT_F32 ? 4 : 8;

    std::atomic<int64_t> next{0};
    std::atomic<int> failed{ZMC_OK};
    std::atomic<int> cuda_error{0};              // a worker's cudaError_t, handed to the CALLER's zmc_last_cuda_error()
    auto fail_cuda = [&](cudaError_t e) { cuda_error = (int)e; failed = ZMC_ERR_CUDA; };
    std::vector<int64_t> done(n_devices, 0);
    std::vector<double> busy_ms(n_devices, 0.0);
    const auto t0 = std::chrono::steady_clock::now();

    auto worker = [&](int slot) {
        cudaError_t ce = cudaSetDevice(devices[slot]);
        if (ce != cudaSuccess) { fail_cuda(ce); return; }
        // At most two batches queued per device, on two alternating streams: every scan call ends by joining its result
        // copies back into its stream, so on ONE stream the kernel of batch b+1 would wait for the copy of batch b
        // (measured: 7 % on cfg 4); on the other stream it starts as soon as the SMs free up.
        cudaStream_t streams[2] = {nullptr, nullptr};
        cudaEvent_t inflight[2] = {nullptr, nullptr};
        auto release = [&] {
            for (int i = 0; i < 2; ++i) {
                if (inflight[i]) cudaEventDestroy(inflight[i]);
                if (streams[i]) cudaStreamDestroy(streams[i]);
            }
        };
        for (int i = 0; i < 2; ++i)
            if ((ce = cudaStreamCreateWithFlags(&streams[i], cudaStreamNonBlocking)) != cudaSuccess ||
                (ce = cudaEventCreateWithFlags(&inflight[i], cudaEventDisableTiming)) != cudaSuccess) {
                fail_cuda(ce);
                release();
                return;
            }
        bool used[2] = {false, false};
        const auto w0 = std::chrono::steady_clock::now();
        for (int64_t k = 0; failed == ZMC_OK; ++k) {
            const int e = (int)(k & 1);
            cudaStream_t stream = streams[e];
            if (used[e] && (ce = cudaEventSynchronize(inflight[e])) != cudaSuccess) { fail_cuda(ce); break; }
            const int64_t b = next.fetch_add(1);
            if (b >= n_batches) break;
            uint64_t bf = 0, bc = 0;
            zmc_batch_range(first, count, bp, b, &bf, &bc);
            zmc_options ob = o;
            ob.first_index = bf;
            ob.count = bc;
            ob.batch_points = 0;
            const size_t off = (size_t)(bf - first) * elem;
            zmc::AdaptArgs ab;
            if (ad) ab = zmc::AdaptArgs{ad->n_max, ad->target, ad->out_n + (bf - first)};
            // the value lists are uploaded once per device: every later batch hits the library's device-resident cache
            const zmc_status s = zmc::scan_impl(integrand_id, N, bounds, M, lists, n_samples, seed, static_cast<char*>(out_mean) + off,
                                                static_cast<char*>(out_stderr) + off, stream, &ob, nullptr, ad ? &ab : nullptr);
            if (s != ZMC_OK) { if (s == ZMC_ERR_CUDA || s == ZMC_ERR_OUT_OF_MEMORY) cuda_error = zmc::get_last_cuda_error(); failed = (int)s; break; }
            if ((ce = cudaEventRecord(inflight[e], stream)) != cudaSuccess) { fail_cuda(ce); break; }
            used[e] = true;
            ++done[slot];
        }
        for (int i = 0; i < 2; ++i)
            if ((ce = cudaStreamSynchronize(streams[i])) != cudaSuccess && failed == ZMC_OK) fail_cuda(ce);
        busy_ms[slot] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - w0).count();
        release();
    };

    int prev = 0;
    const bool have_prev = cudaGetDevice(&prev) == cudaSuccess;
    std::vector<std::thread> threads;
    for (int d = 0; d < n_devices; ++d) threads.emplace_back(worker, d);
    for (auto& t : threads) t.join();
    if (have_prev) cudaSetDevice(prev);

    if (timing) {
        timing->wall_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
        timing->n_batches = n_batches;
        timing->batch_points = bp;
        timing->n_devices = n_devices;
        for (int d = 0; d < n_devices; ++d) { timing->batches_done[d] = done[d]; timing->busy_ms[d] = busy_ms[d]; }
    }
    if (failed != ZMC_OK) zmc::set_last_cuda_error(cuda_error.load());
    return (zmc_status)failed.load();
}

}  // namespace

extern "C" {

zmc_status zmc_scan_farm(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                         uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, const int* devices,
                         int n_devices, const zmc_options* opt, zmc_farm_timing* timing) {
    return farm_impl(integrand_id, N, bounds, M, lists, n_samples, seed, out_mean, out_stderr, nullptr, devices, n_devices, opt, timing);
}

zmc_status zmc_scan_farm_adaptive(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                                  uint64_t n_first, uint64_t n_max, double target_stderr, uint64_t seed, void* out_mean,
                                  void* out_stderr, uint32_t* out_n, const int* devices, int n_devices,
                                  const zmc_options* opt, zmc_farm_timing* timing) {
    if (!out_n || n_first < 256 || n_first % 256 != 0 || n_max < n_first || n_max % 8 != 0 || n_max > 0xFFFFFFF8ull ||
        !(target_stderr >= 0.0))
        return ZMC_ERR_INVALID_ARG;              // the same checks zmc_scan_adaptive makes, before any thread starts
    const zmc::AdaptArgs ad{n_max, target_stderr, out_n};
    return farm_impl(integrand_id, N, bounds, M, lists, n_first, seed, out_mean, out_stderr, &ad, devices, n_devices, opt, timing);
}

}  // extern "C"
