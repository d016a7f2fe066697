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

#include "zmc_params.h"

extern "C" {

zmc_status zmc_scan_farm(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                         uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, const int* devices,
                         int n_devices, const zmc_options* opt, zmc_farm_timing* timing) {
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
    const uint64_t count = o.count ? o.count : G - first;
    if (timing) std::memset(timing, 0, sizeof(*timing));
    if (count == 0) return ZMC_OK;
    // AUTO is resolved once, from the whole range, so that every batch sums in the same order as a one-device scan
    if (o.schedule == ZMC_SCHED_AUTO) o.schedule = zmc_pick_schedule(count, n_samples, N);
    // default batch: ~8 batches per device so a slow device does not hold the tail (18 s vs 89 s per batch)
    uint64_t bp = o.batch_points ? o.batch_points : (count + 8ull * n_devices - 1) / (8ull * n_devices);
    if (bp > (1ull << 30)) bp = 1ull << 30;
    const int64_t n_batches = zmc_batch_range(first, count, bp, -1, nullptr, nullptr);
    const size_t elem = o.out_dtype == ZMC_OUT_F32 ? 4 : 8;

    std::atomic<int64_t> next{0};
    std::atomic<int> failed{ZMC_OK};
    std::vector<int64_t> done(n_devices, 0);
    std::vector<double> busy_ms(n_devices, 0.0);
    const auto t0 = std::chrono::steady_clock::now();

    auto worker = [&](int slot) {
        if (cudaSetDevice(devices[slot]) != cudaSuccess) { failed = ZMC_ERR_CUDA; return; }
        cudaStream_t stream = nullptr;
        if (cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking) != cudaSuccess) { failed = ZMC_ERR_CUDA; return; }
        cudaEvent_t inflight[2] = {nullptr, nullptr};          // at most two batches queued per device: the second one's
        cudaEventCreateWithFlags(&inflight[0], cudaEventDisableTiming);   // kernel overlaps the first one's D2H copy
        cudaEventCreateWithFlags(&inflight[1], cudaEventDisableTiming);
        bool used[2] = {false, false};
        const auto w0 = std::chrono::steady_clock::now();
        for (int64_t k = 0; failed == ZMC_OK; ++k) {
            const int e = (int)(k & 1);
            if (used[e] && cudaEventSynchronize(inflight[e]) != cudaSuccess) { failed = ZMC_ERR_CUDA; break; }
            const int64_t b = next.fetch_add(1);
            if (b >= n_batches) break;
            uint64_t bf = 0, bc = 0;
            zmc_batch_range(first, count, bp, b, &bf, &bc);
            zmc_options ob = o;
            ob.first_index = bf;
            ob.count = bc;
            ob.batch_points = 0;
            const size_t off = (size_t)(bf - first) * elem;
            const zmc_status s = zmc_scan_ex(integrand_id, N, bounds, M, lists, n_samples, seed, static_cast<char*>(out_mean) + off,
                                             static_cast<char*>(out_stderr) + off, stream, &ob, nullptr);
            if (s != ZMC_OK) { failed = (int)s; break; }
            cudaEventRecord(inflight[e], stream);
            used[e] = true;
            ++done[slot];
        }
        if (cudaStreamSynchronize(stream) != cudaSuccess && failed == ZMC_OK) failed = ZMC_ERR_CUDA;
        busy_ms[slot] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - w0).count();
        cudaEventDestroy(inflight[0]);
        cudaEventDestroy(inflight[1]);
        cudaStreamDestroy(stream);
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
    return (zmc_status)failed.load();
}

}  // extern "C"
