// zmc_params.h -- the kernel argument block (host fills it, kernels read it from the constant bank).
#pragma once
#include "zmc_compat.h"
#include "zmc.h"

namespace zmc {

struct ScanParams {
    uint64_t first;               // GLOBAL flat index (reading S3) of local point 0; [first, first+count) never
                                  // straddles a multiple of 2^32, so the high word of t is launch-uniform
    uint64_t out_off;             // element written = out_off + local point index
    uint32_t count;               // points of this launch (<= 2^30: local indices and the grid stay 32-bit)
    uint32_t base_digits[ZMC_MAX_M];    // mixed-radix digits of `first` (host-computed, 64-bit clean)
    const double* lists;          // device: the M value lists, concatenated
    uint32_t rk[20];              // Philox round keys: rk[2r] = k0 + r*W0, rk[2r+1] = k1 + r*W1
    uint32_t n;                   // samples per point
    uint32_t n_dim, n_par;        // N, M
    uint32_t lists_total;         // total list entries
    uint32_t stage_smem;          // 1: lists are staged in shared memory (else read through L1/L2)
    uint32_t out_f32;             // 1: outputs are float
    uint32_t counts[ZMC_MAX_M];   // list lengths L_i
    uint32_t list_off[ZMC_MAX_M]; // offset of list i in `lists`
    uint32_t div_m[ZMC_MAX_M];    // H3: floor(r / L_i) = umulhi(r, div_m[i]) >> div_s[i], exact for every r < 2^30 (host-computed
    uint32_t div_s[ZMC_MAX_M];    //     round-up reciprocal, see fill_divisors in zmc_api.cu); unused where L_i == 1
    double inv_n, nn1;            // H7: 1 / n and (n - 1) * n as doubles (the same IEEE operations the kernel would do per point)
    double a[ZMC_MAX_N], width[ZMC_MAX_N];   // box; in F32E mode already rounded to float (mirror, reading S5)
    double volume;                // prod_k width_k, k ascending
    // adaptive scan only (zmc_scan_adaptive, zmc_adapt_kernel): n is the first checkpoint
    double target;                // stop once stderr <= target ...
    uint32_t n_max;               // ... or n reaches n_max
    uint32_t* out_n;              // samples used per point (device), indexed like out_mean
    double consts[ZMC_MAX_CONSTS];
};

enum { kSchedThread = ZMC_SCHED_THREAD, kSchedWarp = ZMC_SCHED_WARP, kSchedCta = ZMC_SCHED_CTA,
       kSchedAdapt = 4 /* internal: the warp-per-point adaptive kernel */ };

constexpr int kThreads = 256;      // CTA size of every schedule

#ifndef __CUDACC_RTC__
// launcher signature shared by the dispatch table (zmc_api.cu) and the instantiation units
typedef cudaError_t (*LaunchFn)(const ScanParams& p, void* out_mean, void* out_stderr, int grid,
                                size_t smem_bytes, cudaStream_t stream);

struct KernelEntry {
    int family, n_dim /* 0 = any (runtime N) */, precision, fast, schedule;
    LaunchFn launch;
    const void* func;              // for occupancy queries / attributes
};
#endif  // !__CUDACC_RTC__

}  // namespace zmc
