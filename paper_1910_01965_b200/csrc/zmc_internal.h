// zmc_internal.h -- what zmc_api.cu shares with zmc_farm.cu (not part of the C ABI).
#pragma once
#include "zmc_params.h"

namespace zmc {

// adaptive scan (NEXT-4): n_samples is the first checkpoint; these are the other arguments of zmc_scan_adaptive.
// out_n follows out_mean's location (device pointer, or host pointer with ZMC_LOC_HOST).
struct AdaptArgs { uint64_t n_max; double target; uint32_t* out_n; };

zmc_status scan_impl(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                     uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream,
                     const zmc_options* opt, zmc_timing* timing, const AdaptArgs* ad);

// the calling thread's "last CUDA error" slot (zmc_last_cuda_error): a farm worker hands its error to the caller
void set_last_cuda_error(int e);
int get_last_cuda_error();

}  // namespace zmc
