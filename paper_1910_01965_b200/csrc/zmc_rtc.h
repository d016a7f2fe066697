// zmc_rtc.h -- internal interface between zmc_api.cu and zmc_rtc.cu (user integrands compiled with NVRTC).
#pragma once
#include <atomic>
#include <memory>
#include <string>
#include "zmc_params.h"

namespace zmc {

constexpr int kFirstUserId = 1000;

struct UserIntegrand {
    int id = 0;
    std::string name;                     // the first registrant's (identical bodies share one entry)
    int N = 0, M = 0, n_consts = 0, flags = 0;
    std::string body;
    unsigned long long hash = 0;          // of (body, N, M, n_consts, flags): re-registration returns the cached entry
    int registrations = 1;                // zmc_register_integrand calls minus zmc_unregister_integrand calls (under the registry mutex)
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kern[2][4] = {};        // [precision][schedule - 1]; schedule 4 = the adaptive kernel
    mutable std::atomic<uint64_t> launched_on{0};   // bit d: a kernel of this integrand was launched on device d
    UserIntegrand() = default;
    UserIntegrand(const UserIntegrand&) = delete;
    ~UserIntegrand();                     // waits for the devices it was launched on, then unloads the code
};

// The entry is shared: the registry holds one reference, every scan in progress another, so the code stays loaded until the
// last of them lets go -- zmc_unregister_integrand during a scan only removes the id.
std::shared_ptr<const UserIntegrand> find_user_integrand(int id);
cudaError_t launch_user(const UserIntegrand& u, int precision, int schedule, const ScanParams& p, void* out_mean,
                        void* out_stderr, int grid, size_t smem_bytes, cudaStream_t stream);
void unload_user_integrands();

}  // namespace zmc
