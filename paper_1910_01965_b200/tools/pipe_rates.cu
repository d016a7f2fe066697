// pipe_rates.cu -- the roofline denominators of the zmc_scan hot loop, measured.
//
// The loop is ALU work, not a contraction and not HBM traffic, so its ceiling is how many warp-instructions
// of each kind an SM sub-partition (SMSP) can dispatch per clock.  This program measures, on the GPU it runs
// on, the dispatch cost in SMSP-cycles per warp-instruction of every instruction class the loop uses, alone
// and in the mixes that show which classes share a resource, plus the cost of one Philox4x32-10 block.
// All chains are independent (8 per thread, 64 warps/SM), so the numbers are throughput, not latency.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_rates pipe_rates.cu && ./pipe_rates
//   (or: python -m paper_1910_01965_b200.pipe_rates)
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#define M0 0xD2511F53u
#define M1 0xCD9E8D57u

enum Op { LOP3, SHF, WIDE_LOP3, FFMA, DFMA, DADD, MUFU, F2F, NONE };

// one instruction of class OP on chain i (all operands in registers / immediates; nothing foldable)
template <int OP> __device__ __forceinline__ void emit(uint32_t (&e)[8], float (&f)[8], double (&d)[8], int i, uint32_t k,
                                                        float fk, double dk) {
    if (OP == LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(e[i]) : "r"(k), "r"(e[(i + 1) & 7]));
    if (OP == SHF) asm volatile("shf.r.wrap.b32 %0, %0, %1, 9;" : "+r"(e[i]) : "r"(k));
    if (OP == WIDE_LOP3) {   // IMAD.WIDE.U32 with both halves consumed by one LOP3 (a Philox half-round)
        uint64_t p;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(e[i]), "n"(M0));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(e[i]) : "r"((uint32_t)p), "r"((uint32_t)(p >> 32)), "r"(k));
    }
    if (OP == FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(fk), "f"(1e-3f));
    if (OP == DFMA) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(dk), "d"(1e-3));
    if (OP == DADD) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(dk));
    if (OP == MUFU) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
    if (OP == F2F) { double t; asm volatile("cvt.f64.f32 %0, %1;" : "=d"(t) : "f"(f[i])); d[i] = t; f[i] = __int_as_float(__double2hiint(t)); }  // chained
}

// groups of NA x A followed by NB x B, 8 groups per loop iteration
template <int A, int NA, int B, int NB> __global__ void __launch_bounds__(256) mix(uint32_t* out, int iters, uint32_t k, float fk, double dk) {
    uint32_t e[8]; float f[8]; double d[8];
    for (int i = 0; i < 8; ++i) {
        e[i] = threadIdx.x * 2654435761u + i * 40503u + k;
        f[i] = 1.0f + 1e-6f * (threadIdx.x + i);
        d[i] = 1.0 + 1e-9 * (threadIdx.x + i);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int x = 0; x < NA; ++x) emit<A>(e, f, d, (u + x) & 7, k, fk, dk);
#pragma unroll
            for (int x = 0; x < NB; ++x) emit<B>(e, f, d, (u + x) & 7, k, fk, dk);
        }
    }
    uint32_t acc = 0;
    for (int i = 0; i < 8; ++i) acc ^= e[i] ^ __float_as_uint(f[i]) ^ (uint32_t)__double2loint(d[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// three-class groups, interleaved round-robin: P x (IMAD.WIDE+LOP3), L x LOP3, D x DFMA -- the instruction mix of the
// fp64 path (cfg 2 has 26 integer : 18 FP64 instructions per evaluation, i.e. P=1, L=1, D=2)
template <int P, int L, int D> __global__ void __launch_bounds__(256) mix3(uint32_t* out, int iters, uint32_t k, double dk) {
    uint32_t r[8], e[8]; double d[8];
    for (int i = 0; i < 8; ++i) {
        r[i] = threadIdx.x * 2654435761u + i * 40503u + k; e[i] = r[i] * 3u + 1u; d[i] = 1.0 + 1e-9 * (threadIdx.x + i);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            constexpr int T = (P > L ? P : L) > D ? (P > L ? P : L) : D;
#pragma unroll
            for (int x = 0; x < T; ++x) {
                if (x < P) {
                    uint64_t p;
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(r[(u + x) & 7]), "n"(M0));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r[(u + x) & 7]) : "r"((uint32_t)p), "r"((uint32_t)(p >> 32)), "r"(k));
                }
                if (x < D) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[(u + x) & 7]) : "d"(dk), "d"(1e-3));
                if (x < L) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(e[(u + x) & 7]) : "r"(k), "r"(e[(u + x + 1) & 7]));
            }
        }
    }
    uint32_t acc = 0;
    for (int i = 0; i < 8; ++i) acc ^= r[i] ^ e[i] ^ (uint32_t)__double2loint(d[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// Philox4x32-10 from its definition, counter (j, 0, t, 0): the compiler hoists what depends on t only
__global__ void __launch_bounds__(256) philox_only(uint32_t* out, int n_blocks, uint32_t k0, uint32_t k1) {
    uint32_t rk[20];
    for (int r = 0; r < 10; ++r) { rk[2 * r] = k0 + r * 0x9E3779B9u; rk[2 * r + 1] = k1 + r * 0xBB67AE85u; }
    const uint32_t t = blockIdx.x * 256 + threadIdx.x;
    uint32_t acc = 0;
    for (int j = 0; j < n_blocks; ++j) {
        uint32_t c0 = j, c1 = 0, c2 = t, c3 = 0;
#pragma unroll
        for (int r = 0; r < 10; ++r) {
            const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
            const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r], n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1];
            c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        }
        acc ^= c0 ^ c1; acc ^= c2 ^ c3;      // 2 LOP3 to keep all four words alive
    }
    out[t] = acc;
}

__global__ void clock_probe(long long* out) {
    long long c0 = clock64(); unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g0));
    do { asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g1)); } while (g1 - g0 < 20000000ull);   // 20 ms
    out[0] = clock64() - c0; out[1] = (long long)(g1 - g0);
}

static int g_sms = 0;
static double g_mhz = 0;
static const char* kName[] = {"LOP3", "SHF", "IMAD.WIDE+LOP3", "FFMA", "DFMA", "DADD", "MUFU.EX2", "F2F.F64.F32", ""};

template <int A, int NA, int B, int NB> void run_mix(uint32_t* out, bool quiet = false) {
    const int grid = g_sms * 8, iters = 2000;
    mix<A, NA, B, NB><<<grid, 256>>>(out, iters, 12345u, 0.999f, 0.999);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    cudaEventRecord(a);
    mix<A, NA, B, NB><<<grid, 256>>>(out, iters, 12345u, 0.999f, 0.999);
    cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    const double warp_groups_per_smsp = 8.0 * iters * (256 / 32) * 8 / 4.0;
    const double cyc = ms * 1e-3 * g_mhz * 1e6 / warp_groups_per_smsp;
    if (quiet) { cudaEventDestroy(a); cudaEventDestroy(b); return; }
    if (NB == 0) printf("%-16s alone                      : %6.2f SMSP-cycles per warp-instruction\n", kName[A], cyc / NA);
    else printf("%d x %-14s + %d x %-8s    : %6.2f SMSP-cycles per group  (if separate pipes: %s)\n", NA, kName[A], NB, kName[B], cyc,
                "max of the two, if shared: sum");
    cudaEventDestroy(a); cudaEventDestroy(b);
}

template <int P, int L, int D> void run_mix3(uint32_t* out) {
    const int grid = g_sms * 8, iters = 2000;
    mix3<P, L, D><<<grid, 256>>>(out, iters, 12345u, 0.999);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    cudaEventRecord(a); mix3<P, L, D><<<grid, 256>>>(out, iters, 12345u, 0.999); cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    const double warp_groups_per_smsp = 8.0 * iters * (256 / 32) * 8 / 4.0;
    printf("%d x (IMAD.WIDE+LOP3) + %d x LOP3 + %d x DFMA : %6.2f SMSP-cycles per group  (bound: integer %d, fp64 %d, issue %d)\n", P, L, D,
           ms * 1e-3 * g_mhz * 1e6 / warp_groups_per_smsp, 4 * P + 2 * L, 2 * D, 2 * P + L + D);
    cudaEventDestroy(a); cudaEventDestroy(b);
}

int main() {
    cudaDeviceProp prop; cudaGetDeviceProperties(&prop, 0); g_sms = prop.multiProcessorCount;
    uint32_t* out; cudaMalloc(&out, (size_t)g_sms * 8 * 256 * 4 * 4);
    long long* clk; cudaMalloc(&clk, 16);
    g_mhz = 1.0; run_mix<FFMA, 1, NONE, 0>(out, true);        // warm the clocks up
    clock_probe<<<1, 1>>>(clk); long long h[2]; cudaMemcpy(h, clk, 16, cudaMemcpyDeviceToHost);
    g_mhz = (double)h[0] / (double)h[1] * 1e3;
    printf("# %s, %d SMs, SM clock while measuring %.0f MHz\n", prop.name, g_sms, g_mhz);
    run_mix<LOP3, 1, NONE, 0>(out); run_mix<SHF, 1, NONE, 0>(out); run_mix<WIDE_LOP3, 1, NONE, 0>(out);
    run_mix<FFMA, 1, NONE, 0>(out); run_mix<DFMA, 1, NONE, 0>(out); run_mix<DADD, 1, NONE, 0>(out);
    run_mix<MUFU, 1, NONE, 0>(out); run_mix<F2F, 1, NONE, 0>(out);
    run_mix<WIDE_LOP3, 1, LOP3, 1>(out); run_mix<WIDE_LOP3, 1, LOP3, 2>(out); run_mix<WIDE_LOP3, 1, LOP3, 4>(out);
    run_mix<WIDE_LOP3, 1, FFMA, 2>(out); run_mix<WIDE_LOP3, 1, FFMA, 4>(out);
    run_mix<FFMA, 1, LOP3, 1>(out); run_mix<FFMA, 2, LOP3, 1>(out); run_mix<FFMA, 4, LOP3, 2>(out); run_mix<FFMA, 4, LOP3, 4>(out);
    run_mix<DFMA, 1, LOP3, 1>(out); run_mix<DFMA, 2, LOP3, 2>(out); run_mix<DFMA, 4, LOP3, 4>(out); run_mix<DFMA, 1, LOP3, 2>(out);
    run_mix<MUFU, 1, LOP3, 2>(out); run_mix<MUFU, 1, LOP3, 4>(out); run_mix<MUFU, 1, LOP3, 8>(out);
    run_mix<F2F, 1, LOP3, 2>(out); run_mix<F2F, 1, LOP3, 4>(out);
    run_mix3<1, 0, 1>(out); run_mix3<1, 0, 2>(out); run_mix3<1, 1, 2>(out); run_mix3<2, 3, 4>(out); run_mix3<0, 3, 2>(out);
    {
        const int grid = g_sms * 32, n_blocks = 4000;
        philox_only<<<grid, 256>>>(out, 16, 1u, 0u);
        cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
        cudaEventRecord(a); philox_only<<<grid, 256>>>(out, n_blocks, 1u, 0u); cudaEventRecord(b); cudaEventSynchronize(b);
        float ms; cudaEventElapsedTime(&ms, a, b);
        const double warp_blocks_per_smsp = (double)n_blocks * (256 / 32) * 32 / 4.0;
        const double cyc = ms * 1e-3 * g_mhz * 1e6 / warp_blocks_per_smsp;
        printf("Philox4x32-10 block (+2 LOP3)      : %6.2f SMSP-cycles per warp-block  -> %.3e blocks/s on this GPU\n", cyc,
               g_sms * 4 * 32 * g_mhz * 1e6 / cyc);
    }
    printf("status: %s\n", cudaGetErrorString(cudaDeviceSynchronize()));
    return 0;
}
