// bench_probe.cu -- bench_measure_pipes(): the roofline denominators of the zmc_scan hot loop, measured on the device the
// call runs on ("re-measure by micro-benchmark, these are the denominators").
// A MEASUREMENT TOOL of bench.py, not part of the product: built into its own libzmc_probe.so (bench_probe.py), declared in
// bench_probe.h; libzmc.so and include/zmc.h hold only the method's calls.  It shares no code with the library.
//
// The loop is ALU work -- a scalar integer hash (Philox: IMAD.WIDE + LOP3), a few FMAs and one transcendental per
// sample -- so its ceiling is how many warp-instructions of each class an SM sub-partition (SMSP) can dispatch per
// clock, and WHICH CLASSES OVERLAP.  Three kinds of measurement, all in SMSP-cycles per group of instructions per warp:
//   alone      one class, 8 independent chains per thread, 8 warps per SMSP: throughput, not latency
//   same warp  NA x class A then NB x class B in every warp; ptxas picks the static order (it interleaves the classes,
//              as it does in the real kernel): what a single instruction stream achieves
//   two warps  half of the warps run only A, the other half only B: the hardware scheduler interleaves the classes
//              (a warp-specialised producer/consumer split of the loop would behave like this)
// next to the two bounds that the per-class costs alone would give: `parallel` = max(A, B) if the classes were on
// independent pipes, `serial` = A + B if they share one.  The last rows replay cfg 2's instruction mix per Philox block
// (17 IMAD.WIDE+LOP3 pairs, 13 more integer ops, 32 FP64 ops): integer part alone, FP64 part alone, both in one warp,
// and split across warps.  bench.py prints the table in its JSON line ("pipe_rates").
#include <cstdio>
#include <cstring>

#include <cstdint>
#include <cuda_runtime.h>

#include "bench_probe.h"

namespace {

#define ZMC_PROBE_M0 0xD2511F53u

enum Op { LOP3, SHF, WL /* IMAD.WIDE.U32 + the LOP3 that eats both halves: a Philox half-round */, FFMA, DFMA, DADD, MUFU, F2F,
          IMADLO /* 32-bit product, low half only */, IMADHI, NONE };

struct Regs {
    uint32_t c0[8], c1[8], e[8];
    float f[8];
    double d[8];
};

__device__ __forceinline__ void init(Regs& r, uint32_t tid, uint32_t k) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        r.c0[i] = tid * 2654435761u + i * 40503u + k;
        r.c1[i] = r.c0[i] * 3u + 1u;
        r.e[i] = r.c0[i] ^ 0x5555u;
        r.f[i] = 1.0f + 1e-6f * (float)(tid + i);
        r.d[i] = 1.0 + 1e-9 * (double)(tid + i);
    }
}

__device__ __forceinline__ uint32_t fold(const Regs& r) {
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc ^= r.c0[i] ^ r.c1[i] ^ r.e[i] ^ __float_as_uint(r.f[i]) ^ (uint32_t)__double2loint(r.d[i]);
    return acc;
}

// one instruction of class OP on chain i (operands in registers / immediates, nothing foldable)
template <int OP> __device__ __forceinline__ void emit(Regs& r, int i, uint32_t k, float fk, float fc, double dk, double dc) {
    if (OP == LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0xE8;" : "+r"(r.e[i]) : "r"(r.e[(i + 1) & 7]), "r"(k));
    if (OP == SHF) asm volatile("shf.r.wrap.b32 %0, %0, %1, 9;" : "+r"(r.e[i]) : "r"(r.e[(i + 1) & 7]));
    if (OP == WL) {
        uint64_t p;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(r.c0[i]), "n"(ZMC_PROBE_M0));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r.c0[i]) : "r"((uint32_t)(p >> 32)), "r"((uint32_t)p), "r"(k));
    }
    if (OP == IMADLO) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r.c1[i]) : "n"(ZMC_PROBE_M0), "r"(r.c1[(i + 1) & 7]));
    if (OP == IMADHI) asm volatile("mad.hi.u32 %0, %0, %1, %2;" : "+r"(r.c1[i]) : "n"(ZMC_PROBE_M0), "r"(r.c1[(i + 1) & 7]));
    if (OP == FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(r.f[i]) : "f"(fk), "f"(fc));
    if (OP == DFMA) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(r.d[i]) : "d"(dk), "d"(dc));
    if (OP == DADD) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(r.d[i]) : "d"(dk));
    if (OP == MUFU) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(r.f[i]));
    if (OP == F2F) {
        double t;
        asm volatile("cvt.f64.f32 %0, %1;" : "=d"(t) : "f"(r.f[i]));
        r.d[i] = t;
        r.f[i] = __int_as_float(__double2hiint(t));
    }
}

template <int OP, int COUNT> __device__ __forceinline__ void burst(Regs& r, int u, uint32_t k, float fk, float fc, double dk, double dc) {
#pragma unroll
    for (int x = 0; x < COUNT; ++x) emit<OP>(r, (u + x) & 7, k, fk, fc, dk, dc);
}

// 8 groups of (NA x A, NB x B) per loop iteration.  SPLIT: warps 0-3 of the CTA run the A part only, warps 4-7 the B part only.
template <int A, int NA, int B, int NB, bool SPLIT>
__global__ void __launch_bounds__(256) probe_mix(uint32_t* out, int iters, uint32_t k, float fk, float fc, double dk, double dc) {
    Regs r;
    init(r, blockIdx.x * blockDim.x + threadIdx.x, k);
    const bool do_a = !SPLIT || (threadIdx.x & 128) == 0, do_b = !SPLIT || (threadIdx.x & 128) != 0;
    if (do_a && do_b) {
#pragma unroll 4
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) { burst<A, NA>(r, u, k, fk, fc, dk, dc); burst<B, NB>(r, u, k, fk, fc, dk, dc); }
    } else if (do_a) {
#pragma unroll 4
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) burst<A, NA>(r, u, k, fk, fc, dk, dc);
    } else {
#pragma unroll 4
        for (int it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) burst<B, NB>(r, u, k, fk, fc, dk, dc);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = fold(r);
}

// cfg 2's mix per Philox block: P x (IMAD.WIDE+LOP3), L x LOP3, D x DFMA.  PART: 0 both in every warp, 1 integer only,
// 2 FP64 only, 3 split (warps 0-3 integer, warps 4-7 FP64).
template <int P, int L, int D, int PART>
__global__ void __launch_bounds__(256) probe_block(uint32_t* out, int iters, uint32_t k, double dk, double dc) {
    Regs r;
    init(r, blockIdx.x * blockDim.x + threadIdx.x, k);
    const bool ints = PART == 0 || PART == 1 || (PART == 3 && (threadIdx.x & 128) == 0);
    const bool fp64 = PART == 0 || PART == 2 || (PART == 3 && (threadIdx.x & 128) != 0);
    if (ints && fp64) {
#pragma unroll 4
        for (int it = 0; it < iters; ++it) {
            burst<WL, P>(r, 0, k, 0.f, 0.f, dk, dc); burst<LOP3, L>(r, 0, k, 0.f, 0.f, dk, dc); burst<DFMA, D>(r, 0, k, 0.f, 0.f, dk, dc);
        }
    } else if (ints) {
#pragma unroll 4
        for (int it = 0; it < iters; ++it) { burst<WL, P>(r, 0, k, 0.f, 0.f, dk, dc); burst<LOP3, L>(r, 0, k, 0.f, 0.f, dk, dc); }
    } else {
#pragma unroll 4
        for (int it = 0; it < iters; ++it) burst<DFMA, D>(r, 0, k, 0.f, 0.f, dk, dc);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = fold(r);
}


// ------------------------------------------------------------------------------------------------------------------
// What a Philox4x32-10 block costs and WHY.  Three blocks in lock-step per thread, per-thread
// rounds 3-10 (16 multiplies + 18 three-input XORs per block, the library's own formulation; the block index is
// warp-uniform as in the THREAD schedule), in four variants:
//   kWide   the real thing: IMAD.WIDE.U32 gives both halves of each 32x32 product
//   kLowOnly  the same dataflow with the LOW halves only (IMAD.LO) -- NOT Philox, a control: shows that a 32-bit product
//             overlaps with the XORs and that it is the HIGH half of the product that costs
//   kHiF64  the real thing again, high halves from the FP64 pipe: with D = 2^52 + c held as a double,
//             fma.rz(D, M 2^-32, 2^52 - M 2^20) = 2^52 + floor(c M / 2^32) exactly, low halves by IMAD.LO (bit-identical output)
// plus EXTRA independent instructions of one class per block next to the real thing: the slope says what an instruction
// of that class costs inside the Philox stream (FFMA ~1, LOP3 ~2: they add, nothing hides).
enum PhiloxVariant { kWide, kLowOnly, kHiF64 };
#define ZMC_PROBE_M1 0xCD9E8D57u
struct ProbeKeys { uint32_t rk[20]; };

template <int VARIANT, int NB>
__device__ __forceinline__ void probe_philox_blocks(uint32_t e0, uint32_t e2, uint32_t c3i, uint32_t j0, const ProbeKeys& K, uint32_t* out) {
    if (VARIANT == kHiF64) {
        const double M0s = (double)ZMC_PROBE_M0 * 0x1p-32, M1s = (double)ZMC_PROBE_M1 * 0x1p-32;
        const double C0 = 0x1p52 - (double)ZMC_PROBE_M0 * 0x1p20, C1 = 0x1p52 - (double)ZMC_PROBE_M1 * 0x1p20;
        const unsigned long long kMagic = 0x4330000000000000ull;
        unsigned long long D0[NB], D2[NB];
        uint32_t c1[NB], c3[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const uint64_t p0 = (uint64_t)ZMC_PROBE_M0 * (j0 + (uint32_t)b);
            const uint64_t p1 = (uint64_t)ZMC_PROBE_M1 * ((uint32_t)(p0 >> 32) ^ K.rk[1]);
            D0[b] = kMagic | ((uint32_t)(p1 >> 32) ^ e0); c1[b] = (uint32_t)p1; D2[b] = kMagic | (e2 ^ (uint32_t)p0); c3[b] = c3i;
        }
#pragma unroll
        for (int r = 2; r < 10; ++r)
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                double h0, h2;
                asm("fma.rz.f64 %0, %1, %2, %3;" : "=d"(h0) : "d"(__longlong_as_double((long long)D0[b])), "d"(M0s), "d"(C0));
                asm("fma.rz.f64 %0, %1, %2, %3;" : "=d"(h2) : "d"(__longlong_as_double((long long)D2[b])), "d"(M1s), "d"(C1));
                const uint32_t lo0 = (uint32_t)D0[b] * ZMC_PROBE_M0, lo1 = (uint32_t)D2[b] * ZMC_PROBE_M1;
                D0[b] = (unsigned long long)__double_as_longlong(h2) ^ (unsigned long long)(c1[b] ^ K.rk[2 * r]);
                D2[b] = (unsigned long long)__double_as_longlong(h0) ^ (unsigned long long)(c3[b] ^ K.rk[2 * r + 1]);
                c1[b] = lo1; c3[b] = lo0;
            }
#pragma unroll
        for (int b = 0; b < NB; ++b) { out[4 * b] = (uint32_t)D0[b]; out[4 * b + 1] = c1[b]; out[4 * b + 2] = (uint32_t)D2[b]; out[4 * b + 3] = c3[b]; }
    } else {
        uint32_t c0[NB], c1[NB], c2[NB], c3[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const uint64_t p0 = (uint64_t)ZMC_PROBE_M0 * (j0 + (uint32_t)b);
            const uint64_t p1 = (uint64_t)ZMC_PROBE_M1 * ((uint32_t)(p0 >> 32) ^ K.rk[1]);
            c0[b] = (uint32_t)(p1 >> 32) ^ e0; c1[b] = (uint32_t)p1; c2[b] = e2 ^ (uint32_t)p0; c3[b] = c3i;
        }
#pragma unroll
        for (int r = 2; r < 10; ++r)
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                if (VARIANT == kWide) {
                    const uint64_t p0 = (uint64_t)ZMC_PROBE_M0 * c0[b], p1 = (uint64_t)ZMC_PROBE_M1 * c2[b];
                    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1[b] ^ K.rk[2 * r], n2 = (uint32_t)(p0 >> 32) ^ c3[b] ^ K.rk[2 * r + 1];
                    c1[b] = (uint32_t)p1; c3[b] = (uint32_t)p0; c0[b] = n0; c2[b] = n2;
                } else {
                    const uint32_t q0 = ZMC_PROBE_M0 * c0[b], q1 = ZMC_PROBE_M1 * c2[b];
                    const uint32_t n0 = q1 ^ c1[b] ^ K.rk[2 * r], n2 = q0 ^ c3[b] ^ K.rk[2 * r + 1];
                    c1[b] = q1; c3[b] = q0; c0[b] = n0; c2[b] = n2;
                }
            }
#pragma unroll
        for (int b = 0; b < NB; ++b) { out[4 * b] = c0[b]; out[4 * b + 1] = c1[b]; out[4 * b + 2] = c2[b]; out[4 * b + 3] = c3[b]; }
    }
}

template <int VARIANT, int EXTRA_OP, int EXTRA>
__global__ void __launch_bounds__(256, 4) probe_philox(uint32_t* out, int iters, uint32_t k, float fk, float fc, double dk, double dc,
                                                        const __grid_constant__ ProbeKeys K) {
    constexpr int NB = 3;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t e0 = tid * 2654435761u, e2 = tid * 40503u + 7u, c3i = tid ^ 0x55u;
    Regs r;
    init(r, tid, k);
    uint32_t acc = 0, w[4 * NB];
    for (int it = 0; it < iters; ++it) {
        probe_philox_blocks<VARIANT, NB>(e0, e2, c3i, (uint32_t)(it * NB), K, w);
        burst<EXTRA_OP, EXTRA * NB>(r, 0, k, fk, fc, dk, dc);
#pragma unroll
        for (int i = 0; i < 4 * NB; ++i) acc += w[i];          // consumer: one three-input add per two words (a sum: XOR would cancel
                                                                // the last round of the low-halves-only control)
    }
    out[tid] = acc ^ fold(r);
}

__global__ void probe_clock(long long* out) {
    const long long c0 = clock64();
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g0));
    do { asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g1)); } while (g1 - g0 < 5000000ull);     // 5 ms
    out[0] = clock64() - c0;
    out[1] = (long long)(g1 - g0);
}

const char* kName[] = {"LOP3", "SHF", "IMAD.WIDE+LOP3", "FFMA", "DFMA", "DADD", "MUFU.EX2", "F2F.F64.F32", "IMAD.LO", "IMAD.HI", ""};

struct Probe {
    cudaStream_t stream;
    uint32_t* out;
    int grid;                 // 4 CTAs of 256 per SM: 8 warps per SMSP
    double mhz;
    cudaEvent_t a, b;
    cudaError_t err = cudaSuccess;
    bench_pipe_report* rep;

    template <class K, class... Args> double time_ms(K kern, Args... args) {
        float best = 1e30f;
        for (int rep_i = 0; rep_i < 3 && err == cudaSuccess; ++rep_i) {       // first run warms up, best of the next two
            cudaEventRecord(a, stream);
            kern<<<grid, 256, 0, stream>>>(args...);
            cudaEventRecord(b, stream);
            err = cudaEventSynchronize(b);
            float ms = 0.f;
            if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, a, b);
            if (rep_i > 0 && ms < best) best = ms;
        }
        if (err == cudaSuccess) err = cudaGetLastError();
        return best;
    }
    // SMSP-cycles per group per warp: warps_per_smsp warps each run groups_per_warp groups
    double cycles(double ms, double groups_per_warp, double warps_per_smsp) const {
        return ms * 1e-3 * mhz * 1e6 / (groups_per_warp * warps_per_smsp);
    }
    void add(const char* name, double cyc, double parallel, double serial) {
        if (rep->n_rows >= BENCH_PIPE_MAX_ROWS) return;
        bench_pipe_row& row = rep->rows[rep->n_rows++];
        std::snprintf(row.name, sizeof(row.name), "%s", name);
        row.cycles = cyc; row.parallel = parallel; row.serial = serial;
    }
    static constexpr int kIters = 1500;
    template <int A> double alone() {
        // 4 per group, 8 groups, loop unrolled 4x: 128 instructions per trip, so the loop's own 3 cost < 3 %
        const double c = cycles(time_ms(probe_mix<A, 4, NONE, 0, false>, out, kIters, 12345u, 0.999f, 1e-3f, 0.999, 1e-3), 8.0 * kIters, 8.0) / 4.0;
        add(kName[A], c, c, c);
        return c;
    }
    template <int A, int NA, int B, int NB> void pair(double ca, double cb) {
        char name[64];
        const double par = NA * ca > NB * cb ? NA * ca : NB * cb, ser = NA * ca + NB * cb;
        std::snprintf(name, sizeof(name), "%dx%s + %dx%s, same warp", NA, kName[A], NB, kName[B]);
        add(name, cycles(time_ms(probe_mix<A, NA, B, NB, false>, out, kIters, 12345u, 0.999f, 1e-3f, 0.999, 1e-3), 8.0 * kIters, 8.0), par, ser);
        // split: 4 warps per SMSP run A, 4 run B; one "group" = NA x A in an A-warp plus NB x B in a B-warp
        std::snprintf(name, sizeof(name), "%dx%s | %dx%s, two warps", NA, kName[A], NB, kName[B]);
        add(name, cycles(time_ms(probe_mix<A, NA, B, NB, true>, out, kIters, 12345u, 0.999f, 1e-3f, 0.999, 1e-3), 8.0 * kIters, 4.0), par, ser);
    }
};

}  // namespace

extern "C" __attribute__((visibility("default"))) int bench_measure_pipes(bench_pipe_report* report, void* stream_v) {
    if (!report) return -1;
    std::memset(report, 0, sizeof(*report));
    Probe p;
    p.rep = report;
    p.stream = static_cast<cudaStream_t>(stream_v);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return (int)cudaGetLastError();
    p.grid = sms * 4;
    long long* clk = nullptr;
    if (cudaMalloc(&p.out, (size_t)p.grid * 256 * sizeof(uint32_t)) != cudaSuccess) return (int)cudaErrorMemoryAllocation;
    if (cudaMalloc(&clk, 2 * sizeof(long long)) != cudaSuccess) { cudaFree(p.out); return (int)cudaErrorMemoryAllocation; }
    cudaEventCreate(&p.a);
    cudaEventCreate(&p.b);
    p.mhz = 1.0;
    p.time_ms(probe_mix<FFMA, 4, NONE, 0, false>, p.out, Probe::kIters, 12345u, 0.999f, 1e-3f, 0.999, 1e-3);       // clocks up
    probe_clock<<<1, 1, 0, p.stream>>>(clk);
    long long h[2] = {0, 1};
    if (cudaMemcpyAsync(h, clk, sizeof(h), cudaMemcpyDeviceToHost, p.stream) != cudaSuccess || cudaStreamSynchronize(p.stream) != cudaSuccess)
        p.err = cudaErrorUnknown;
    p.mhz = (double)h[0] / (double)h[1] * 1e3;
    report->sm_mhz = p.mhz;
    report->sm_count = sms;

    const double lop = p.alone<LOP3>(), shf = p.alone<SHF>(), wl = p.alone<WL>(), ffma = p.alone<FFMA>();
    const double dfma = p.alone<DFMA>(), dadd = p.alone<DADD>(), mufu = p.alone<MUFU>(), f2f = p.alone<F2F>();
    const double imadlo = p.alone<IMADLO>();
    p.alone<IMADHI>();
    (void)shf; (void)dadd;
    p.pair<IMADLO, 1, LOP3, 1>(imadlo, lop);
    p.pair<LOP3, 1, DFMA, 1>(lop, dfma);
    p.pair<LOP3, 1, DADD, 1>(lop, dadd);
    p.pair<WL, 1, DFMA, 2>(wl, dfma);
    p.pair<WL, 1, LOP3, 2>(wl, lop);
    p.pair<LOP3, 1, FFMA, 2>(lop, ffma);
    p.pair<WL, 1, FFMA, 4>(wl, ffma);
    p.pair<LOP3, 4, MUFU, 1>(lop, mufu);
    p.pair<WL, 2, MUFU, 1>(wl, mufu);
    p.pair<FFMA, 8, MUFU, 1>(ffma, mufu);
    p.pair<LOP3, 4, F2F, 1>(lop, f2f);
    p.pair<DFMA, 4, F2F, 1>(dfma, f2f);
    {   // cfg 2's mix per Philox block (2 evaluations): 17 IMAD.WIDE+LOP3 pairs + 13 integer ops (uniform bits, sign) and 32 FP64 ops
        constexpr int P = 17, L = 13, D = 32;
        const int it = 4000;
        const double ci = p.cycles(p.time_ms(probe_block<P, L, D, 1>, p.out, it, 12345u, 0.999, 1e-3), it, 8.0);
        const double cd = p.cycles(p.time_ms(probe_block<P, L, D, 2>, p.out, it, 12345u, 0.999, 1e-3), it, 8.0);
        const double cm = p.cycles(p.time_ms(probe_block<P, L, D, 0>, p.out, it, 12345u, 0.999, 1e-3), it, 8.0);
        const double cs = p.cycles(p.time_ms(probe_block<P, L, D, 3>, p.out, it, 12345u, 0.999, 1e-3), it, 4.0);
        const double par = ci > cd ? ci : cd;
        p.add("cfg2 block: integer part alone (17 IMAD.WIDE+LOP3, 13 LOP3)", ci, ci, ci);
        p.add("cfg2 block: FP64 part alone (32 DFMA)", cd, cd, cd);
        p.add("cfg2 block: both, same warp (ptxas order)", cm, par, ci + cd);
        p.add("cfg2 block: integer warps | FP64 warps", cs, par, ci + cd);
    }

    {   // one Philox block inside the stream of the THREAD schedule (three blocks in lock-step, 8 warps per SMSP)
        ProbeKeys K;
        for (int r = 0; r < 10; ++r) { K.rk[2 * r] = 0xDEADBEEFu + r * 0x9E3779B9u; K.rk[2 * r + 1] = 0x12345678u + r * 0xBB67AE85u; }
        const int it = 1500;
        auto blk = [&](double ms) { return p.cycles(ms, 3.0 * it, 8.0); };
        const double alu = 18 * lop, all = 34 * lop;       // XORs alone | every integer instruction at the ALU rate
        const double base = blk(p.time_ms(probe_philox<kWide, NONE, 0>, p.out, it, 12345u, 0.999f, 1e-3f, 0.999, 1e-3, K));
        p.add("Philox block: 16 IMAD.WIDE + 18 LOP3 per thread + uniform rounds 1-2", base, alu, all);
        p.add("  + 8 independent FFMA per block", blk(p.time_ms(probe_philox<kWide, FFMA, 8>, p.out, it, 12345u, 0.999f, 1e-3f, 0.999, 1e-3, K)), base, base + 8 * ffma);
        p.add("  + 8 independent DFMA per block", blk(p.time_ms(probe_philox<kWide, DFMA, 8>, p.out, it, 12345u, 0.999f, 1e-3f, 0.999, 1e-3, K)), base, base + 8 * dfma);
        p.add("  + 8 independent LOP3 per block", blk(p.time_ms(probe_philox<kWide, LOP3, 8>, p.out, it, 12345u, 0.999f, 1e-3f, 0.999, 1e-3, K)), base, base + 8 * lop);
        p.add("  control: low halves only (16 IMAD.LO + 18 LOP3; NOT Philox)", blk(p.time_ms(probe_philox<kLowOnly, NONE, 0>, p.out, it, 12345u, 0.999f, 1e-3f, 0.999, 1e-3, K)), alu, 16 * imadlo + alu);
        p.add("  high halves by DFMA.RZ (FP64 pipe) + IMAD.LO: same output", blk(p.time_ms(probe_philox<kHiF64, NONE, 0>, p.out, it, 12345u, 0.999f, 1e-3f, 0.999, 1e-3, K)), alu, 16 * imadlo + alu + 16 * dfma);
    }
    cudaEventDestroy(p.a);
    cudaEventDestroy(p.b);
    cudaFree(p.out);
    cudaFree(clk);
    return (int)p.err;                     // 0 = cudaSuccess, else the first cudaError_t met
}
