// zmc_math.cuh -- device arithmetic building blocks of the zmc_scan hot loop (sm_100a).
//
// H4 (sampler): Philox4x32-10 written from its definition (Salmon et al., SC'11; DESIGN.md
// reading Q1/S2) with the per-point part of the first two rounds hoisted, and the exact uniforms
// of reading S4 built by bit tricks (no I2F on the 16-lane XU pipe).
// H5 (integrand): a branch-free fp64 sin(pi z) (exact range reduction in units of pi, degree-15
// odd polynomial with immediate coefficients -- no table loads, no slow path) and thin wrappers
// over the MUFU transcendentals for the fp32 path.
#pragma once
#include "zmc_compat.h"

#ifndef ZMC_F64_UNIT_I2F
#define ZMC_F64_UNIT_I2F 0
#endif
#ifndef ZMC_F32_RINT_MAGIC
#define ZMC_F32_RINT_MAGIC 0
#endif

namespace zmc {

// ------------------------------------------------------------------------------------------
// Philox4x32-10.  Counter = (block j, 0, t lo, t hi), key = seed (stream layout S3).
// rk[2r], rk[2r+1] are the round keys k0 + r*0x9E3779B9, k1 + r*0xBB67AE85 (host-computed,
// read straight from the constant bank by LOP3).
// With t fixed per grid point, counter words 2,3 and word 1 (= 0) are loop invariants, so round
// 1 needs one multiply and round 2 one multiply: 18 IMAD.WIDE + 19 LOP3 per block instead of 20+20.
// ------------------------------------------------------------------------------------------
constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;

struct PhiloxPoint {
    uint32_t r1_c0, r1_c1;      // counter words 0,1 after round 1 (depend on t only)
    uint32_t r1_x;              // t_hi ^ rk[1]: folded into word 2 of round 1
    uint32_t r2_c3;             // counter word 3 after round 2 (t only)
    uint32_t r2_e0, r2_e2;      // invariants folded into words 0 and 2 of round 2

    // t_hi is passed separately: the host never lets a launch straddle a multiple of 2^32, so it is a launch-wide
    // constant and everything derived from it (and from a warp-uniform block index) stays on the uniform datapath.
    __device__ __forceinline__ void init(uint32_t t_lo, uint32_t t_hi, const uint32_t* __restrict__ rk) {
        const uint64_t p1 = (uint64_t)kPhiloxM1 * t_lo;           // round 1, multiply of word 2
        r1_c0 = (uint32_t)(p1 >> 32) ^ rk[0];                     // hi1 ^ c1(=0) ^ k0
        r1_c1 = (uint32_t)p1;                                     // lo1
        r1_x = t_hi ^ rk[1];
        const uint64_t p0 = (uint64_t)kPhiloxM0 * r1_c0;          // round 2, multiply of word 0
        r2_c3 = (uint32_t)p0;                                     // lo0
        r2_e2 = (uint32_t)(p0 >> 32) ^ rk[3];                     // hi0 ^ k1 (then ^ c3)
        r2_e0 = r1_c1 ^ rk[2];                                    // c1 ^ k0 (then ^ hi1)
    }

    // NBLK consecutive blocks j0 .. j0+NBLK-1 in lock-step (round by round), so that 2*NBLK independent
    // multiplies are in flight: the IMAD.WIDE (fmaheavy) pipe, not the dependent chain, sets the pace.
    template <int NBLK>
    __device__ __forceinline__ void blocks(uint32_t j0, const uint32_t* __restrict__ rk, uint32_t* __restrict__ out) const {
        uint32_t c0[NBLK], c1[NBLK], c2[NBLK], c3[NBLK];
#pragma unroll
        for (int b = 0; b < NBLK; ++b) {
            // round 1: only word 0 (= j) varies
            const uint64_t p0 = (uint64_t)kPhiloxM0 * (j0 + (uint32_t)b);
            const uint32_t t2 = (uint32_t)(p0 >> 32) ^ r1_x;
            // round 2: word 0 is invariant
            const uint64_t p1 = (uint64_t)kPhiloxM1 * t2;
            c0[b] = (uint32_t)(p1 >> 32) ^ r2_e0;
            c1[b] = (uint32_t)p1;
            c2[b] = r2_e2 ^ (uint32_t)p0;
            c3[b] = r2_c3;
        }
#pragma unroll
        for (int r = 2; r < 10; ++r) {
#pragma unroll
            for (int b = 0; b < NBLK; ++b) {
                const uint64_t p0 = (uint64_t)kPhiloxM0 * c0[b];
                const uint64_t p1 = (uint64_t)kPhiloxM1 * c2[b];
                const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1[b] ^ rk[2 * r];
                const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3[b] ^ rk[2 * r + 1];
                c1[b] = (uint32_t)p1;
                c3[b] = (uint32_t)p0;
                c0[b] = n0;
                c2[b] = n2;
            }
        }
#pragma unroll
        for (int b = 0; b < NBLK; ++b) {
            out[4 * b + 0] = c0[b]; out[4 * b + 1] = c1[b]; out[4 * b + 2] = c2[b]; out[4 * b + 3] = c3[b];
        }
    }

    __device__ __forceinline__ void block(uint32_t j, const uint32_t* __restrict__ rk, uint32_t (&out)[4]) const {
        blocks<1>(j, rk, out);
    }
};

// ------------------------------------------------------------------------------------------
// Uniforms (reading S4).  unit(w) is a value f, exact in the evaluation type, from which the lattice uniform is
// u = f * u_scale() - u_offset():
//   fp32: f = 1 + (w >> 9) * 2^-23 in [1,2), one funnel shift; u = f - (1 - 2^-24) = (2(w>>9)+1) 2^-24
//   fp64: f = 1 + w * 2^-32 in [1,2), a funnel shift and a shift; u = f - (1 - 2^-33) = (2w+1) 2^-33
//         (measured alternative, rejected: f = (2^52 + w) - 2^52 with one DADD costs two register moves per word
//          to pair the word with the 0x43300000 high half and is 5 % slower on cfg2)
// No I2F (16-lane XU pipe) anywhere.
// Families fold scale and offset into per-point constants, so the hot loop spends one FMA per dimension.
// ------------------------------------------------------------------------------------------
template <typename R> struct Real;

template <> struct Real<float> {
    static __device__ __forceinline__ float unit(uint32_t w) {
        return __uint_as_float(__funnelshift_r(w, 0x7Fu, 9));        // (w>>9) | 0x3F800000
    }
    static __device__ __forceinline__ double u_scale() { return 1.0; }
    static __device__ __forceinline__ double u_offset() { return 0x1.fffffep-1; }          // 1 - 2^-24
    static __device__ __forceinline__ float fma(float a, float b, float c) { return fmaf(a, b, c); }
    // a - b that the compiler may NOT contract with a multiply feeding a (g - K must round the same way in every kernel
    // a family is compiled into: the adaptive scan is bit-identical to the fixed-n scan)
    static __device__ __forceinline__ float sub(float a, float b) { return __fsub_rn(a, b); }
};

template <> struct Real<double> {
    static __device__ __forceinline__ double unit(uint32_t w) {
#if ZMC_F64_UNIT_I2F
        return (double)w;                                                               // I2F.F64.U32 (XU pipe)
    }
    static __device__ __forceinline__ double u_scale() { return 0x1p-32; }
    static __device__ __forceinline__ double u_offset() { return -0x1p-33; }
#else
        return __hiloint2double((int)__funnelshift_r(w, 0x3FFu, 12), (int)(w << 20));   // 1 + w*2^-32
    }
    static __device__ __forceinline__ double u_scale() { return 1.0; }
    static __device__ __forceinline__ double u_offset() { return 0x1.ffffffffp-1; }        // 1 - 2^-33
#endif
    static __device__ __forceinline__ double fma(double a, double b, double c) { return ::fma(a, b, c); }
    static __device__ __forceinline__ double sub(double a, double b) { return __dsub_rn(a, b); }
};

// exact lattice uniform u in (0,1) (diagnostic families; the hot families fold scale and offset)
template <typename R> __device__ __forceinline__ R uniform(uint32_t w) {
    return Real<R>::fma(Real<R>::unit(w), (R)Real<R>::u_scale(), (R)(-Real<R>::u_offset()));
}

// ------------------------------------------------------------------------------------------
// fp64 sin(pi z), any |z| < 2^51.  k = rint(z) by the magic-number add, r = z - k exact,
// sin(pi z) = (-1)^k sin(pi r), |r| <= 1/2; odd polynomial r*P7(r^2), max error 2.4e-16
// (Chebyshev-node fit of sin(pi sqrt(s))/sqrt(s) on [0,1/4]).
// ------------------------------------------------------------------------------------------
// sinpi_minus_f64(z, K) = sin(pi z) - K: the sign is applied to r BEFORE the polynomial and the shift K of the
// accumulator (reading S6) rides in the last FMA, so the whole thing is 12 fp64-pipe ops + 2 integer ops.
__device__ __forceinline__ double sinpi_minus_f64(double z, double K) {
    const double kMagic = 6755399441055744.0;                  // 1.5 * 2^52
    const double kf = z + kMagic;
    const double r0 = z - (kf - kMagic);
    // sign flip for odd k: xor bit 0 of k into the sign bit of r
    const double r = __hiloint2double(__double2hiint(r0) ^ (__double2loint(kf) << 31), __double2loint(r0));
    const double s = r0 * r0;
    double p = -0x1.62903d02bb153p-16;
    p = ::fma(p, s, 0x1.e89f6fe44fe7bp-12);
    p = ::fma(p, s, -0x1.e30631bdf732dp-8);
    p = ::fma(p, s, 0x1.5078327046959p-4);
    p = ::fma(p, s, -0x1.32d2cce1ea145p-1);
    p = ::fma(p, s, 0x1.466bc677522bdp+1);
    p = ::fma(p, s, -0x1.4abbce625bd83p+2);
    p = ::fma(p, s, 0x1.921fb54442d18p+1);                     // pi
    return ::fma(r, p, -K);
}
__device__ __forceinline__ double sinpi_f64(double z) { return sinpi_minus_f64(z, 0.0); }

// Transcendentals of the evaluation type.  FAST selects the MUFU forms for fp32 (north_star: "fast-math
// transcendentals only where the tolerance allows"); fp64 ignores it.  Trig families keep their phase in the unit
// kPhasePerRad * radians and call sin_phase():
//   fp64          : units of pi      -> sinpi_f64 (exact range reduction)
//   fp32 + MUFU   : turns (1/2pi)    -> r = ph - rint(ph) exactly, then sin.approx(2 pi r).  sin.approx scales its
//                   argument with a round-toward-zero FMUL; on an unreduced phase of up to 60 rad that bias
//                   (~ |ph| 2^-24 rad, same sign for every sample) exceeded the 1e-4 + 1e-6 tolerance at 0.01 % of
//                   cfg 5's grid points; on |2 pi r| <= pi it is 15x smaller and odd-symmetric, so it averages out
//   fp32 accurate : radians          -> sinf
template <typename R, bool FAST> struct Fn;

template <bool FAST> struct Fn<double, FAST> {
    static constexpr double kPhasePerRad = 0.31830988618379067154;       // 1/pi
    static constexpr double kQuarter = 0.5;                              // pi/2 in phase units
    static __device__ __forceinline__ double wrap(double c) { return c; }
    static __device__ __forceinline__ double sin_phase(double z) { return sinpi_f64(z); }
    static __device__ __forceinline__ double sin_phase_minus(double z, double K) { return sinpi_minus_f64(z, K); }
    static __device__ __forceinline__ double exp2_neg(double e) { return ::exp2(-e); }
};

template <> struct Fn<float, true> {
    static constexpr double kPhasePerRad = 0.15915494309189533577;       // 1/(2 pi)
    static constexpr double kQuarter = 0.25;
    static __device__ __forceinline__ double wrap(double c) { return c - rint(c); }
    static __device__ __forceinline__ float sin_phase(float t) {
#if ZMC_F32_RINT_MAGIC
        const float kf = t + 12582912.0f;                                // 1.5 * 2^23: rint(t) in the low mantissa bits
        const float r = t - (kf - 12582912.0f);                          // 3 FADD, exact for |t| < 2^22, no XU op
#else
        const float r = t - rintf(t);                                    // FRND (XU pipe) + FADD, exact
#endif
        return __sinf(r * 6.283185307179586f);                           // FMUL, then FMUL.RZ(1/2pi) + MUFU.SIN
    }
    static __device__ __forceinline__ float sin_phase_minus(float t, float K) { return sin_phase(t) - K; }
    static __device__ __forceinline__ float exp2_neg(float e) {            // 2^-e: one MUFU.EX2
        float r;
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(-e));
        return r;
    }
};

template <> struct Fn<float, false> {
    static constexpr double kPhasePerRad = 1.0;
    static constexpr double kQuarter = 1.5707963267948966;
    static __device__ __forceinline__ double wrap(double c) { return c - 6.283185307179586 * rint(c * 0.15915494309189533577); }
    static __device__ __forceinline__ float sin_phase(float a) { return sinf(a); }
    static __device__ __forceinline__ float sin_phase_minus(float a, float K) { return __fsub_rn(sinf(a), K); }
    static __device__ __forceinline__ float exp2_neg(float e) { return exp2f(-e); }
};

}  // namespace zmc
