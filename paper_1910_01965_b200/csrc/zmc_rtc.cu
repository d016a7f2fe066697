// zmc_rtc.cu -- NEXT-3 of SURVEY.md 8(f): user-defined integrands.  PAPER.md:9 "users have a full flexibility to
// define their own integrands" (also :49, :162): the paper JIT-compiles a Python function with Numba; here the user
// hands over the body of a CUDA C++ device function, which NVRTC compiles into the SAME kernel template the
// built-in families use (decode, Philox, schedules, fp64 accumulation, store -- nothing is re-implemented), for
// sm_100a, at registration time.  libnvrtc is loaded with dlopen, so the library has no link-time dependency on it.
#include <dlfcn.h>
#include <nvrtc.h>

#include <cstdio>
#include <cstring>
#include <memory>
#include <mutex>
#include <string>
#include <vector>

#include "zmc_rtc.h"

namespace zmc {
namespace {

struct Header { const char* name; const char* text; };
const Header kHeaders[] = {
#include "zmc_rtc_headers.inc"
};
constexpr int kNumHeaders = sizeof(kHeaders) / sizeof(kHeaders[0]);

struct Nvrtc {
    void* handle = nullptr;
    decltype(&nvrtcCreateProgram) createProgram = nullptr;
    decltype(&nvrtcDestroyProgram) destroyProgram = nullptr;
    decltype(&nvrtcCompileProgram) compileProgram = nullptr;
    decltype(&nvrtcAddNameExpression) addNameExpression = nullptr;
    decltype(&nvrtcGetLoweredName) getLoweredName = nullptr;
    decltype(&nvrtcGetProgramLogSize) getProgramLogSize = nullptr;
    decltype(&nvrtcGetProgramLog) getProgramLog = nullptr;
    decltype(&nvrtcGetCUBINSize) getCUBINSize = nullptr;
    decltype(&nvrtcGetCUBIN) getCUBIN = nullptr;
    bool ok = false;
};

Nvrtc& nvrtc() {
    static Nvrtc n;
    static std::once_flag once;
    std::call_once(once, [] {
        for (const char* so : {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12"}) {
            n.handle = dlopen(so, RTLD_NOW | RTLD_LOCAL);
            if (n.handle) break;
        }
        if (!n.handle) return;
#define ZMC_SYM(field, sym) n.field = reinterpret_cast<decltype(n.field)>(dlsym(n.handle, #sym))
        ZMC_SYM(createProgram, nvrtcCreateProgram);
        ZMC_SYM(destroyProgram, nvrtcDestroyProgram);
        ZMC_SYM(compileProgram, nvrtcCompileProgram);
        ZMC_SYM(addNameExpression, nvrtcAddNameExpression);
        ZMC_SYM(getLoweredName, nvrtcGetLoweredName);
        ZMC_SYM(getProgramLogSize, nvrtcGetProgramLogSize);
        ZMC_SYM(getProgramLog, nvrtcGetProgramLog);
        ZMC_SYM(getCUBINSize, nvrtcGetCUBINSize);
        ZMC_SYM(getCUBIN, nvrtcGetCUBIN);
#undef ZMC_SYM
        n.ok = n.createProgram && n.destroyProgram && n.compileProgram && n.addNameExpression && n.getLoweredName &&
               n.getProgramLogSize && n.getProgramLog && n.getCUBINSize && n.getCUBIN;
    });
    return n;
}

std::mutex g_user_mutex;
std::vector<std::shared_ptr<UserIntegrand>> g_users;
int g_next_user_id = kFirstUserId;        // ids are never reused
thread_local std::string tl_compile_log;

// The translation unit NVRTC sees: the library's kernel template plus a family that evaluates the user's g.
// No folding of the affine sample map here (the user's g wants y itself): y_k = fma(u_k, width_k, a_k), reading S5.
std::string make_source(const char* body, int N, int M, int n_consts, int flags) {
    char head[256];
    std::snprintf(head, sizeof(head), "#define ZMC_USER_N %d\n#define ZMC_USER_M %d\n#define ZMC_USER_NC %d\n#define ZMC_USER_FAST %d\n",
                  N, M, n_consts, (flags & ZMC_USER_FAST_MATH) ? 1 : 0);
    std::string s = head;
    s += R"SRC(
#include "zmc_kernel.cuh"
namespace zmc {
// the library's own transcendentals, offered to the user's body (include/zmc.h, zmc_register_integrand)
__device__ __forceinline__ double zmc_sinpi(double z) { return sinpi_f64(z); }
__device__ __forceinline__ double zmc_cospi(double z) { return sinpi_f64(z + 0.5); }
__device__ __forceinline__ double zmc_sin(double v) { return sinpi_f64(v * kInvPi); }
__device__ __forceinline__ double zmc_cos(double v) { return sinpi_f64(::fma(v, kInvPi, 0.5)); }
__device__ __forceinline__ double zmc_exp(double v) { return ::exp(v); }
__device__ __forceinline__ double zmc_exp2(double v) { return ::exp2(v); }
#if ZMC_USER_FAST
__device__ __forceinline__ float zmc_sinpi(float z) { return Fn<float, true>::sin_phase(0.5f * z); }
__device__ __forceinline__ float zmc_cospi(float z) { return Fn<float, true>::sin_phase(fmaf(0.5f, z, 0.25f)); }
__device__ __forceinline__ float zmc_sin(float v) { return Fn<float, true>::sin_phase(v * 0.15915494309189535f); }
__device__ __forceinline__ float zmc_cos(float v) { return Fn<float, true>::sin_phase(fmaf(v, 0.15915494309189535f, 0.25f)); }
__device__ __forceinline__ float zmc_exp(float v) { return Fn<float, true>::exp2_neg(v * -1.4426950408889634f); }
__device__ __forceinline__ float zmc_exp2(float v) { return Fn<float, true>::exp2_neg(-v); }
#else
__device__ __forceinline__ float zmc_sinpi(float z) { return sinpif(z); }
__device__ __forceinline__ float zmc_cospi(float z) { return cospif(z); }
__device__ __forceinline__ float zmc_sin(float v) { return sinf(v); }
__device__ __forceinline__ float zmc_cos(float v) { return cosf(v); }
__device__ __forceinline__ float zmc_exp(float v) { return expf(v); }
__device__ __forceinline__ float zmc_exp2(float v) { return exp2f(v); }
#endif
template <typename R> struct FamUser {
    using real = R;
    static constexpr int kN = ZMC_USER_N <= 8 ? ZMC_USER_N : 0;     // compile-time N up to 8, else the runtime-N loop
    R a[ZMC_USER_N], wd[ZMC_USER_N], xs[ZMC_USER_M], cs[ZMC_USER_NC > 0 ? ZMC_USER_NC : 1];
    __device__ __forceinline__ void setup(const R* x, const ScanParams& p) {
#pragma unroll
        for (int k = 0; k < ZMC_USER_N; ++k) { a[k] = (R)p.a[k]; wd[k] = (R)p.width[k]; }
#pragma unroll
        for (int i = 0; i < ZMC_USER_M; ++i) xs[i] = x[i];
#pragma unroll
        for (int j = 0; j < ZMC_USER_NC; ++j) cs[j] = (R)p.consts[j];
    }
    // ---- the user's integrand g(y; x), PAPER.md:55-59 Eq. (1) ----
    __device__ __forceinline__ R g(const R* y, const R* x, const R* c) const {
)SRC";
    s += body;
    s += R"SRC(
    }
    __device__ __forceinline__ R eval(const uint32_t* w) const {
        R y[ZMC_USER_N];
#pragma unroll
        for (int k = 0; k < ZMC_USER_N; ++k) y[k] = Real<R>::fma(uniform<R>(w[k]), wd[k], a[k]);
        return g(y, xs, cs);
    }
    __device__ __forceinline__ R eval_shifted(const uint32_t* w, R K) const { return Real<R>::sub(eval(w), K); }      // never contracted into g's last multiply
};
}  // namespace zmc
)SRC";
    return s;
}

}  // namespace

std::shared_ptr<const UserIntegrand> find_user_integrand(int id) {
    std::lock_guard<std::mutex> lock(g_user_mutex);
    for (auto& u : g_users)
        if (u->id == id) return u;
    return nullptr;
}

// Runs when the last holder lets go (the registry after the last unregister / zmc_shutdown, or a scan that was in progress
// at that moment).  Kernels already enqueued may still be running: wait for every device that ever launched one before the
// code is unloaded.
UserIntegrand::~UserIntegrand() {
    if (!lib) return;
    const uint64_t mask = launched_on.load();
    int cur = 0;
    if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); return; }   // no runtime any more (process exit): nothing to unload
    for (int d = 0; d < 64; ++d)
        if (mask >> d & 1u) { if (cudaSetDevice(d) == cudaSuccess) cudaDeviceSynchronize(); }
    cudaSetDevice(cur);
    cudaLibraryUnload(lib);
    cudaGetLastError();
}

cudaError_t launch_user(const UserIntegrand& u, int precision, int schedule, const ScanParams& p, void* out_mean,
                        void* out_stderr, int grid, size_t smem_bytes, cudaStream_t stream) {
    cudaKernel_t k = u.kern[precision][schedule - 1];
    if (!k) return cudaErrorInvalidDeviceFunction;
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64) u.launched_on.fetch_or(1ull << dev);
    if (smem_bytes > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute((const void*)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
    }
    void* args[] = {const_cast<ScanParams*>(&p), &out_mean, &out_stderr};
    return cudaLaunchKernel((const void*)k, dim3((unsigned)grid), dim3(kThreads), args, smem_bytes, stream);
}

void unload_user_integrands() {
    std::lock_guard<std::mutex> lock(g_user_mutex);
    g_users.clear();                           // ids are valid until zmc_shutdown (include/zmc.h); they are never reused.
                                               // Each entry unloads its code when its last holder lets go (~UserIntegrand).
}

}  // namespace zmc

using namespace zmc;

extern "C" {

const char* zmc_last_compile_log(void) { return tl_compile_log.c_str(); }

static unsigned long long hash_integrand(const char* body, int N, int M, int n_consts, int flags) {
    unsigned long long h = 1469598103934665603ull;
    auto mix = [&h](const void* p, size_t n) {
        const unsigned char* b = static_cast<const unsigned char*>(p);
        for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
    };
    const int shape[4] = {N, M, n_consts, flags};
    mix(shape, sizeof(shape));
    mix(body, std::strlen(body));
    return h;
}

zmc_status zmc_register_integrand_ex(const char* name, const char* body, int N, int M, int n_consts, int flags,
                                     int* integrand_id) {
    tl_compile_log.clear();
    if (!name || !body || !integrand_id) return ZMC_ERR_INVALID_ARG;
    if (N < 1 || N > ZMC_MAX_N || M < 1 || M > ZMC_MAX_M || n_consts < 0 || n_consts > ZMC_MAX_CONSTS) return ZMC_ERR_INVALID_ARG;
    if (flags & ~ZMC_USER_FAST_MATH) return ZMC_ERR_INVALID_ARG;
    // the cache (SURVEY.md 8(f) NEXT-3 "cache by hash"): the same integrand registered again is the same id, no compile
    const unsigned long long h = hash_integrand(body, N, M, n_consts, flags);
    {
        std::lock_guard<std::mutex> lock(g_user_mutex);
        for (auto& u : g_users)
            if (u->hash == h && u->lib && u->N == N && u->M == M && u->n_consts == n_consts && u->flags == flags && u->body == body) {
                ++u->registrations;            // one more owner of this id: it takes as many unregister calls to drop it
                *integrand_id = u->id;
                return ZMC_OK;
            }
    }
    Nvrtc& rt = nvrtc();
    if (!rt.ok) {
        tl_compile_log = "libnvrtc.so.12 could not be loaded";
        return ZMC_ERR_COMPILE;
    }
    const std::string src = make_source(body, N, M, n_consts, flags);
    const char* names[kNumHeaders];
    const char* texts[kNumHeaders];
    for (int i = 0; i < kNumHeaders; ++i) { names[i] = kHeaders[i].name; texts[i] = kHeaders[i].text; }
    nvrtcProgram prog = nullptr;
    if (rt.createProgram(&prog, src.c_str(), "zmc_user_integrand.cu", kNumHeaders, texts, names) != NVRTC_SUCCESS) {
        tl_compile_log = "nvrtcCreateProgram failed";
        return ZMC_ERR_COMPILE;
    }
    struct Guard { Nvrtc& rt; nvrtcProgram* p; ~Guard() { rt.destroyProgram(p); } } guard{rt, &prog};
    static const char* kReal[2] = {"double", "float"};
    std::string expr[2][4];
    for (int pr = 0; pr < 2; ++pr)
        for (int sc = 0; sc < 4; ++sc) {
            expr[pr][sc] = sc < 3 ? std::string("zmc::zmc_scan_kernel<zmc::FamUser<") + kReal[pr] + ">, " + std::to_string(sc + 1) + ">"
                                  : std::string("zmc::zmc_adapt_kernel<zmc::FamUser<") + kReal[pr] + "> >";
            if (rt.addNameExpression(prog, expr[pr][sc].c_str()) != NVRTC_SUCCESS) {
                tl_compile_log = "nvrtcAddNameExpression failed";
                return ZMC_ERR_COMPILE;
            }
        }
    const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo", "-default-device", "--use_fast_math"};
    const nvrtcResult rc = rt.compileProgram(prog, (flags & ZMC_USER_FAST_MATH) ? 5 : 4, opts);
    size_t log_size = 0;
    if (rt.getProgramLogSize(prog, &log_size) == NVRTC_SUCCESS && log_size > 1) {
        tl_compile_log.resize(log_size);
        rt.getProgramLog(prog, &tl_compile_log[0]);
        while (!tl_compile_log.empty() && tl_compile_log.back() == '\0') tl_compile_log.pop_back();
    }
    if (rc != NVRTC_SUCCESS) return ZMC_ERR_COMPILE;
    size_t cubin_size = 0;
    if (rt.getCUBINSize(prog, &cubin_size) != NVRTC_SUCCESS || cubin_size == 0) return ZMC_ERR_COMPILE;
    std::vector<char> cubin(cubin_size);
    if (rt.getCUBIN(prog, cubin.data()) != NVRTC_SUCCESS) return ZMC_ERR_COMPILE;

    auto u = std::make_shared<UserIntegrand>();
    u->name = name; u->N = N; u->M = M; u->n_consts = n_consts; u->flags = flags; u->body = body; u->hash = h;
    cudaError_t e = cudaLibraryLoadData(&u->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e != cudaSuccess) { tl_compile_log += "\ncudaLibraryLoadData: "; tl_compile_log += cudaGetErrorString(e); return ZMC_ERR_CUDA; }
    for (int pr = 0; pr < 2; ++pr)
        for (int sc = 0; sc < 4; ++sc) {
            const char* lowered = nullptr;
            const bool named = rt.getLoweredName(prog, expr[pr][sc].c_str(), &lowered) == NVRTC_SUCCESS && lowered;
            e = named ? cudaLibraryGetKernel(&u->kern[pr][sc], u->lib, lowered) : cudaErrorInvalidDeviceFunction;
            if (e != cudaSuccess) return named ? ZMC_ERR_CUDA : ZMC_ERR_COMPILE;   // ~UserIntegrand releases the loaded code
        }
    std::lock_guard<std::mutex> lock(g_user_mutex);
    u->id = g_next_user_id++;
    *integrand_id = u->id;
    g_users.push_back(std::move(u));
    return ZMC_OK;
}

zmc_status zmc_register_integrand(const char* name, const char* body, int N, int M, int n_consts, int* integrand_id) {
    return zmc_register_integrand_ex(name, body, N, M, n_consts, 0, integrand_id);
}

zmc_status zmc_unregister_integrand(int integrand_id) {
    std::lock_guard<std::mutex> lock(g_user_mutex);
    for (size_t i = 0; i < g_users.size(); ++i)
        if (g_users[i]->id == integrand_id) {
            if (--g_users[i]->registrations > 0) return ZMC_OK;      // registered more than once: other owners keep the id
            std::shared_ptr<UserIntegrand> last = std::move(g_users[i]);
            g_users.erase(g_users.begin() + (long)i);
            return ZMC_OK;                     // `last` goes out of scope here: unloads now unless a scan still holds the entry
        }
    return ZMC_ERR_UNKNOWN_INTEGRAND;
}

}  // extern "C"
