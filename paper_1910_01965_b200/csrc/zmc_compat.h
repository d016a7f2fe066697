// zmc_compat.h -- the few standard names the kernel headers need, for both compilers that see them: nvcc (library
// build) and NVRTC (run-time compilation of user integrands, zmc_register_integrand; NVRTC has no host headers).
#pragma once
#ifdef __CUDACC_RTC__
typedef unsigned int uint32_t;
typedef int int32_t;
typedef unsigned long long uint64_t;
typedef long long int64_t;
namespace std {
template <class A, class B> struct is_same { static constexpr bool value = false; };
template <class A> struct is_same<A, A> { static constexpr bool value = true; };
}  // namespace std
#else
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#endif
