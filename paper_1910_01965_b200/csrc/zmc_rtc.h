// zmc_rtc.h -- internal interface between zmc_api.cu and zmc_rtc.cu (user integrands compiled with NVRTC).
#pragma once
#include <string>
#include "zmc_params.h"

namespace zmc {

constexpr int kFirstUserId = 1000;

struct UserIntegrand {
    int id = 0;
    std::string name;
    int N = 0, M = 0, n_consts = 0, flags = 0;
    std::string body;
    unsigned long long hash = 0;          // of (body, N, M, n_consts, flags): re-registration returns the cached entry
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kern[2][4] = {};        // [precision][schedule - 1]; schedule 4 = the adaptive kernel
};

const UserIntegrand* find_user_integrand(int id);
cudaError_t launch_user(const UserIntegrand& u, int precision, int schedule, const ScanParams& p, void* out_mean,
                        void* out_stderr, int grid, size_t smem_bytes, cudaStream_t stream);
void unload_user_integrands();

}  // namespace zmc
