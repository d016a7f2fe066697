// zmc_kernel.cuh -- the fused batch kernel of zmc_scan (sm_100a):
//   H3 decode -> H4 Philox sampler -> H5 integrand -> H6 fp64 accumulate + reduce -> H7 finalise + store
// for one contiguous range of flat grid indices (one batch).  One kernel template,
// three schedules (lanes per grid point): THREAD (1; the paper's mapping), WARP (32)
// and CTA (256) with __shfl_xor_sync trees -- the paper's one-thread-per-point scheme cannot fill
// the GPU for small grids and serialises large sample counts.
//
// Work split inside a point: samples are taken in block-aligned groups of S samples = NB whole
// Philox blocks (no random word is wasted, reading S3); lane l of L takes groups l, l+L, ...
// Every word is keyed by (seed, GLOBAL flat index t, word index), so results are independent of
// batching and grid size; the summation order (hence the last bits) depends on the schedule only.
//
// Accumulation (reading S6): values are shifted by K = g(sample 0 of the point), common to all
// lanes, and A = sum (g-K), B = sum (g-K)^2 are kept in fp64, so lanes combine by plain addition
// and  mean = V (K + A/n),  stderr = V sqrt((B - A^2/n) / ((n-1) n))  is free of cancellation.
#pragma once
#include "zmc_families.cuh"

// 1/n and (n-1)n: taken from the parameter block (computed on the host) or recomputed per point.  The values are the same
// IEEE results either way; what differs is the code ptxas generates AROUND them -- measured on B200: host values make the
// built-in cfg 2 kernel 1.2 % faster (17.72 -> 17.50 ms), but the NVRTC-compiled user kernel of the same integrand 3.5 %
// slower (19.13 -> 19.80 ms), so the run-time compiled kernels keep the per-point computation.
#ifndef ZMC_FINALISE_FROM_HOST
#ifdef __CUDACC_RTC__
#define ZMC_FINALISE_FROM_HOST 0
#else
#define ZMC_FINALISE_FROM_HOST 1
#endif
#endif

#ifndef ZMC_PIPELINE_F32
#define ZMC_PIPELINE_F32 0      // measured with the two-buffer loop too: cfg3 -0.2 %, cfg4 -1.4 %, cfg5 -0.5 %
#endif



namespace zmc {

constexpr int gcd4(int n) { return (n % 4 == 0) ? 4 : (n % 2 == 0) ? 2 : 1; }

// group shape for compile-time N: the smallest block-aligned group, doubled when it is a single block
template <int N> struct GroupShape {
    static constexpr int kMinS = 4 / gcd4(N), kMinNB = N / gcd4(N);
    static constexpr int kU = (kMinNB == 1) ? 2 : 1;
    static constexpr int S = kMinS * kU, NB = kMinNB * kU;
};
template <> struct GroupShape<0> {     // runtime N: 4 samples = N blocks
    static constexpr int S = 4, NB = ZMC_MAX_N;
};

template <typename R> struct Accum {
    double A = 0.0, B = 0.0;
    R K;
    __device__ __forceinline__ void add_shifted(R d_) {     // d_ = g - K, formed in the evaluation type
        const double d = (double)d_;                        // (fp32: exact when g ~ K by Sterbenz, else harmless)
        A += d;
        B = ::fma(d, d, B);
    }
};

// H3: mixed-radix decode.  digits(t) = digits(first) + digits(local) with carries: the 64-bit part was done on the
// host, the per-point part is 32-bit division only.  Writes the point's M parameter values (evaluation type) to x.
template <typename R>
__device__ __forceinline__ void decode_point(const ScanParams& p, uint32_t local, const R* __restrict__ slist, R (&x)[ZMC_MAX_M]) {
    const int M = (int)p.n_par;
    uint32_t rest = local, carry = 0;
#pragma unroll
    for (int i = ZMC_MAX_M - 1; i >= 1; --i) {
        if (i < M) {
            const uint32_t L = p.counts[i];
            // rest / L without a division: rest < 2^30 (a launch's local index), so the host's 32-bit round-up reciprocal is exact
            const uint32_t q = L == 1u ? rest : (__umulhi(rest, p.div_m[i]) >> p.div_s[i]);
            uint32_t d = p.base_digits[i] + (rest - q * L) + carry;
            carry = d >= L ? 1u : 0u;
            d -= carry ? L : 0u;
            rest = q;
            const uint32_t idx = p.list_off[i] + d;
            x[i] = p.stage_smem ? slist[idx] : (R)__ldg(p.lists + idx);
        } else {
            x[i] = (R)0;
        }
    }
    const uint32_t idx0 = p.list_off[0] + p.base_digits[0] + rest + carry;
    x[0] = p.stage_smem ? slist[idx0] : (R)__ldg(p.lists + idx0);
}

template <class Fam, int SCHED>
__global__ void __launch_bounds__(kThreads, std::is_same<typename Fam::real, double>::value ? 3 : 4)
zmc_scan_kernel(const __grid_constant__ ScanParams p, void* __restrict__ out_mean, void* __restrict__ out_stderr)
{
    using R = typename Fam::real;
    constexpr int kN = Fam::kN;
    using GS = GroupShape<kN>;
    constexpr int S = GS::S;
    const int N = kN ? kN : (int)p.n_dim;
    const int NB = kN ? GS::NB : N;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    R* slist = reinterpret_cast<R*>(smem_raw);
    __shared__ double red_a[kThreads / 32], red_b[kThreads / 32];

    // H1 (device side): stage the value lists in shared memory, rounded to the evaluation type
    if (p.stage_smem) {
        for (uint32_t i = threadIdx.x; i < p.lists_total; i += kThreads) slist[i] = (R)p.lists[i];
        __syncthreads();
    }

    // One grid point per worker (thread / warp / CTA); the grid has one CTA per kThreads / 8 / 1 points, so the
    // hardware CTA scheduler balances the load and refills every slot a finished CTA frees.
    const uint32_t lanes = SCHED == kSchedThread ? 1u : SCHED == kSchedWarp ? 32u : (uint32_t)kThreads;
    const uint32_t lane = SCHED == kSchedThread ? 0u : SCHED == kSchedWarp ? (threadIdx.x & 31u) : threadIdx.x;
    const uint32_t local = SCHED == kSchedThread ? blockIdx.x * kThreads + threadIdx.x
                         : SCHED == kSchedWarp   ? blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5)
                                                 : blockIdx.x;
    if (local >= p.count) return;                   // uniform per warp (WARP) / per CTA (CTA)
    const uint32_t t_lo = (uint32_t)p.first + local;      // no carry: a launch never straddles a multiple of 2^32

    R x[ZMC_MAX_M];
    decode_point<R>(p, local, slist, x);

    const uint32_t n = p.n;
    const uint32_t n_full = n / S;                 // full groups; the last group may be clipped
    const uint32_t rem = n - n_full * S;
#if ZMC_FINALISE_FROM_HOST
    const double inv_n = p.inv_n;                  // 1.0 / (double)n, divided once on the host (the same IEEE quotient)
#else
    const double inv_n = 1.0 / (double)n;
#endif

    Fam fam;
    fam.setup(x, p);
    PhiloxPoint px;
    px.init(t_lo, (uint32_t)(p.first >> 32), p.rk);

    uint32_t w[GS::NB * 4];
    Accum<R> acc;
    {   // shift K = g(sample 0): words 0..N-1
        const int nb0 = (N + 3) >> 2;
#pragma unroll
        for (int b = 0; b < (kN ? (kN + 3) / 4 : ZMC_MAX_N / 4); ++b)
            if (b < nb0) px.block((uint32_t)b, p.rk, *reinterpret_cast<uint32_t(*)[4]>(&w[4 * b]));
        acc.K = fam.eval(w);
    }

    // H4 + H5 + H6: the hot loop.  fp64 path: software-pipelined -- the Philox blocks of the NEXT group (integer
    // pipe) sit in the same basic block as the evaluation of the CURRENT one (FP64 pipe), so ptxas alternates the two
    // pipes instruction by instruction (measured +7 % on cfg2; the one group generated past the end is discarded).
    // fp32 path: FP32 and integer instructions share the dispatch port on sm_100 (profiles/), nothing to overlap.
    if constexpr (kN != 0 && (std::is_same<R, double>::value || ZMC_PIPELINE_F32)) {
        // two buffers, two groups per iteration: no register copies between "next" and "current"
        uint32_t wb[GS::NB * 4];
        const uint32_t step = lanes * (uint32_t)GS::NB;
        uint32_t j0 = lane * (uint32_t)GS::NB;
        if (lane < n_full) px.template blocks<GS::NB>(j0, p.rk, w);
        uint32_t g = lane;
        for (; g + lanes < n_full; g += 2u * lanes) {
            px.template blocks<GS::NB>(j0 + step, p.rk, wb);
#pragma unroll
            for (int s = 0; s < S; ++s) acc.add_shifted(fam.eval_shifted(&w[s * N], acc.K));
            j0 += 2u * step;
            px.template blocks<GS::NB>(j0, p.rk, w);
#pragma unroll
            for (int s = 0; s < S; ++s) acc.add_shifted(fam.eval_shifted(&wb[s * N], acc.K));
        }
        if (g < n_full) {
#pragma unroll
            for (int s = 0; s < S; ++s) acc.add_shifted(fam.eval_shifted(&w[s * N], acc.K));
        }
    } else {
        for (uint32_t g = lane; g < n_full; g += lanes) {
            const uint32_t j0 = g * (uint32_t)NB;
            if constexpr (kN != 0) {
                px.template blocks<GS::NB>(j0, p.rk, w);
            } else {
#pragma unroll
                for (int b = 0; b < GS::NB; ++b)
                    if (b < NB) px.block(j0 + b, p.rk, *reinterpret_cast<uint32_t(*)[4]>(&w[4 * b]));
            }
#pragma unroll
            for (int s = 0; s < S; ++s) acc.add_shifted(fam.eval_shifted(&w[s * N], acc.K));
        }
    }
    if (rem != 0 && (n_full % lanes) == lane) {        // clipped last group: warp-uniform trip count
        const uint32_t j0 = n_full * (uint32_t)NB;
#pragma unroll
        for (int b = 0; b < GS::NB; ++b)
            if (b < NB) px.block(j0 + b, p.rk, *reinterpret_cast<uint32_t(*)[4]>(&w[4 * b]));
#pragma unroll
        for (int s = 0; s < S - 1; ++s)
            if ((uint32_t)s < rem) acc.add_shifted(fam.eval_shifted(&w[s * N], acc.K));
    }

    // H6: combine lanes (plain sums: the shift K is common to all lanes of the point)
    double A = acc.A, B = acc.B;
    if (SCHED != kSchedThread) {
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
            A += __shfl_xor_sync(0xffffffffu, A, m);
            B += __shfl_xor_sync(0xffffffffu, B, m);
        }
    }
    if (SCHED == kSchedCta) {
        const int warp = threadIdx.x >> 5;
        if ((threadIdx.x & 31) == 0) { red_a[warp] = A; red_b[warp] = B; }
        __syncthreads();
        if (warp == 0) {
            A = (threadIdx.x < kThreads / 32) ? red_a[threadIdx.x] : 0.0;
            B = (threadIdx.x < kThreads / 32) ? red_b[threadIdx.x] : 0.0;
#pragma unroll
            for (int m = kThreads / 64; m >= 1; m >>= 1) {
                A += __shfl_xor_sync(0xffffffffu, A, m);
                B += __shfl_xor_sync(0xffffffffu, B, m);
            }
        }
    }

    // H7: finalise and store (coalesced across the warp in the THREAD schedule)
    if (lane == 0) {
        const double mean_g = (double)acc.K + A * inv_n;
        double m2 = ::fma(-A * inv_n, A, B);
        m2 = m2 > 0.0 ? m2 : 0.0;
        const double mean = p.volume * mean_g;
#if ZMC_FINALISE_FROM_HOST
        const double serr = p.volume * sqrt(m2 / p.nn1);          // nn1 = (double)(n - 1) * (double)n
#else
        const double serr = p.volume * sqrt(m2 / ((double)(n - 1) * (double)n));
#endif
        const uint64_t o = p.out_off + local;
        if (p.out_f32) {
            static_cast<float*>(out_mean)[o] = (float)mean;
            static_cast<float*>(out_stderr)[o] = (float)serr;
        } else {
            static_cast<double*>(out_mean)[o] = mean;
            static_cast<double*>(out_stderr)[o] = serr;
        }
    }
}

// NEXT-4: per-point adaptive sample count.  PAPER.md:116 leaves it to the user to "determine the
// number of sample points based on the desired accuracy ... increase this value"; here the kernel does it: one warp per
// grid point samples up to the checkpoints n_0 = p.n, 2 n_0, 4 n_0, ... (clipped to p.n_max) and stops at the first
// one where stderr <= p.target.  The stream is keyed by (seed, t, word index), so the estimate at a checkpoint uses
// exactly the first n words (prefix property) and -- n_0 being a multiple of 256, hence every checkpoint a multiple
// of 32 groups -- lane l owns groups l, l+32, ... exactly as in the fixed-n WARP schedule: the result is bit-identical
// to zmc_scan_ex(n_samples = n_used, schedule = WARP).
template <class Fam>
__global__ void __launch_bounds__(kThreads, std::is_same<typename Fam::real, double>::value ? 3 : 4)
zmc_adapt_kernel(const __grid_constant__ ScanParams p, void* __restrict__ out_mean, void* __restrict__ out_stderr)
{
    using R = typename Fam::real;
    constexpr int kN = Fam::kN;
    using GS = GroupShape<kN>;
    constexpr int S = GS::S;
    const int N = kN ? kN : (int)p.n_dim;
    const int NB = kN ? GS::NB : N;

    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t local = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    if (local >= p.count) return;                          // uniform per warp
    const uint32_t t_lo = (uint32_t)p.first + local;

    R x[ZMC_MAX_M];
    decode_point<R>(p, local, static_cast<const R*>(nullptr), x);      // stage_smem is 0 for this kernel

    Fam fam;
    fam.setup(x, p);
    PhiloxPoint px;
    px.init(t_lo, (uint32_t)(p.first >> 32), p.rk);

    uint32_t w[GS::NB * 4];
    Accum<R> acc;
    {
        const int nb0 = (N + 3) >> 2;
#pragma unroll
        for (int b = 0; b < (kN ? (kN + 3) / 4 : ZMC_MAX_N / 4); ++b)
            if (b < nb0) px.block((uint32_t)b, p.rk, *reinterpret_cast<uint32_t(*)[4]>(&w[4 * b]));
        acc.K = fam.eval(w);
    }

    uint32_t n_lo = 0, n_hi = p.n;                          // both multiples of S (validated on the host)
    double A, B, serr, inv_n;
    // fp64: software-pipelined like the fixed-n kernel -- w always holds the lane's NEXT group, generated in the same
    // basic block as the evaluation of the current one (the lane's groups l, l+32, ... run on across checkpoints, so the
    // look-ahead carries over; the one group generated past the last checkpoint is discarded).  Same order of sums.
    constexpr bool kPipelined = kN != 0 && std::is_same<R, double>::value;
    uint32_t g_next = lane;
    if constexpr (kPipelined) px.template blocks<GS::NB>(g_next * (uint32_t)GS::NB, p.rk, w);
    for (;;) {
        if constexpr (kPipelined) {
            for (; g_next < n_hi / S; g_next += 32u) {
                R d[S];
#pragma unroll
                for (int s = 0; s < S; ++s) d[s] = fam.eval_shifted(&w[s * N], acc.K);
                px.template blocks<GS::NB>((g_next + 32u) * (uint32_t)GS::NB, p.rk, w);
#pragma unroll
                for (int s = 0; s < S; ++s) acc.add_shifted(d[s]);
            }
        } else {
            for (uint32_t g = n_lo / S + lane; g < n_hi / S; g += 32u) {
                const uint32_t j0 = g * (uint32_t)NB;
                if constexpr (kN != 0) {
                    px.template blocks<GS::NB>(j0, p.rk, w);
                } else {
#pragma unroll
                    for (int b = 0; b < GS::NB; ++b)
                        if (b < NB) px.block(j0 + b, p.rk, *reinterpret_cast<uint32_t(*)[4]>(&w[4 * b]));
                }
#pragma unroll
                for (int s = 0; s < S; ++s) acc.add_shifted(fam.eval_shifted(&w[s * N], acc.K));
            }
        }
        A = acc.A; B = acc.B;                               // lane partials stay put; the tree works on copies
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
            A += __shfl_xor_sync(0xffffffffu, A, m);
            B += __shfl_xor_sync(0xffffffffu, B, m);
        }
        inv_n = 1.0 / (double)n_hi;                         // the same finalisation, operation for operation, as above
        double m2 = ::fma(-A * inv_n, A, B);
        m2 = m2 > 0.0 ? m2 : 0.0;
        serr = p.volume * sqrt(m2 / ((double)(n_hi - 1) * (double)n_hi));
        if (serr <= p.target || n_hi >= p.n_max) break;    // the same value in every lane: warp-uniform
        n_lo = n_hi;
        n_hi = (n_hi > p.n_max - n_hi) ? p.n_max : 2u * n_hi;
    }

    if (lane == 0) {
        const double mean = p.volume * ((double)acc.K + A * inv_n);
        const uint64_t o = p.out_off + local;
        if (p.out_f32) {
            static_cast<float*>(out_mean)[o] = (float)mean;
            static_cast<float*>(out_stderr)[o] = (float)serr;
        } else {
            static_cast<double*>(out_mean)[o] = mean;
            static_cast<double*>(out_stderr)[o] = serr;
        }
        p.out_n[o] = n_hi;
    }
}

#ifndef __CUDACC_RTC__
template <class Fam, int SCHED>
cudaError_t launch_scan(const ScanParams& p, void* out_mean, void* out_stderr, int grid, size_t smem_bytes,
                        cudaStream_t stream)
{
    auto kern = zmc_scan_kernel<Fam, SCHED>;
    if (smem_bytes > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, kThreads, smem_bytes, stream>>>(p, out_mean, out_stderr);
    return cudaGetLastError();
}

template <class Fam>
cudaError_t launch_adapt(const ScanParams& p, void* out_mean, void* out_stderr, int grid, size_t smem_bytes,
                         cudaStream_t stream)
{
    zmc_adapt_kernel<Fam><<<grid, kThreads, smem_bytes, stream>>>(p, out_mean, out_stderr);
    return cudaGetLastError();
}

// four table rows (the three schedules + the adaptive kernel) for one family type; the type goes last because it contains commas
#define ZMC_ENTRY(FAMILY_ID, NDIM, PREC, FAST, ...)                                                      \
    {FAMILY_ID, NDIM, PREC, FAST, kSchedThread, &launch_scan<__VA_ARGS__, kSchedThread>,                \
     (const void*)&zmc_scan_kernel<__VA_ARGS__, kSchedThread>},                                         \
    {FAMILY_ID, NDIM, PREC, FAST, kSchedWarp, &launch_scan<__VA_ARGS__, kSchedWarp>,                    \
     (const void*)&zmc_scan_kernel<__VA_ARGS__, kSchedWarp>},                                           \
    {FAMILY_ID, NDIM, PREC, FAST, kSchedCta, &launch_scan<__VA_ARGS__, kSchedCta>,                      \
     (const void*)&zmc_scan_kernel<__VA_ARGS__, kSchedCta>},                                            \
    {FAMILY_ID, NDIM, PREC, FAST, kSchedAdapt, &launch_adapt<__VA_ARGS__>,                              \
     (const void*)&zmc_adapt_kernel<__VA_ARGS__>}

// the three arithmetic variants of a family template F<R, ..., FAST>: fp64, fp32+MUFU, fp32 accurate
#define ZMC_ENTRY_FIXED(FAMILY_ID, NDIM, F)                                  \
    ZMC_ENTRY(FAMILY_ID, NDIM, ZMC_PREC_F64, 0, F<double, false>),           \
    ZMC_ENTRY(FAMILY_ID, NDIM, ZMC_PREC_F32E, 1, F<float, true>),            \
    ZMC_ENTRY(FAMILY_ID, NDIM, ZMC_PREC_F32E, 0, F<float, false>)
#define ZMC_ENTRY_NDIM(FAMILY_ID, NDIM, F)                                   \
    ZMC_ENTRY(FAMILY_ID, NDIM, ZMC_PREC_F64, 0, F<double, NDIM, false>),     \
    ZMC_ENTRY(FAMILY_ID, NDIM, ZMC_PREC_F32E, 1, F<float, NDIM, true>),      \
    ZMC_ENTRY(FAMILY_ID, NDIM, ZMC_PREC_F32E, 0, F<float, NDIM, false>)
#define ZMC_ENTRY_DIAG(FAMILY_ID, F)                                         \
    ZMC_ENTRY(FAMILY_ID, 0, ZMC_PREC_F64, 0, F<double>),                     \
    ZMC_ENTRY(FAMILY_ID, 0, ZMC_PREC_F32E, 0, F<float>)

#endif  // !__CUDACC_RTC__

}  // namespace zmc
