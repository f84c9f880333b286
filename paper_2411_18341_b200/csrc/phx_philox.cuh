// phx_philox.cuh -- counter-based noise of the stochastic step (Eq. (22)).
// Philox4x32-10 (Salmon et al., SC'11) keyed by (seed, realisation) with counter (cell, step_lo, step_hi, 0)
// (BASELINE.json config 5; reading Q13).  Product code: shares nothing with oracle/.
#pragma once

#include "phx_common.cuh"

namespace phx {

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c.x, p1 = (uint64_t)0xCD9E8D57u * c.z;   // one IMAD.WIDE each
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

__device__ __forceinline__ uint4 noise_words(uint32_t seed, uint32_t realisation, uint64_t step, uint32_t cell) {
    return philox4x32_10(make_uint4(cell, (uint32_t)step, (uint32_t)(step >> 32), 0u), make_uint2(seed, realisation));
}

// Two words -> standard complex normal pair by Box-Muller.  u = ((w >> 9) + 0.5) 2^-23 is exact in fp32.
__device__ __forceinline__ float2 normal_pair(uint32_t w0, uint32_t w1, float) {
    const float u1 = ((float)(w0 >> 9) + 0.5f) * 1.1920928955078125e-07f;
    const float u2 = ((float)(w1 >> 9) + 0.5f) * 1.1920928955078125e-07f;
    const float rad = sqrtf(-2.0f * logf(u1));
    float s, c;
    sincospif(2.0f * u2, &s, &c);
    return make_float2(rad * c, rad * s);
}

__device__ __forceinline__ double2 normal_pair(uint32_t w0, uint32_t w1, double) {
    const double u1 = ((double)(w0 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double u2 = ((double)(w1 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double rad = sqrt(-2.0 * log(u1));
    double s, c;
    sincospi(2.0 * u2, &s, &c);
    return make_double2(rad * c, rad * s);
}

// The noise increment of one cell, Eq. (22): sqrt(var) (xi_1 + i xi_2) with var the variance per real component, as ONE
// square root: sqrt(-2 ln(u1) var) (cos, sin)(2 pi u2).
__device__ __forceinline__ float2 noise_increment(uint32_t w0, uint32_t w1, float var) {
    const float u1 = ((float)(w0 >> 9) + 0.5f) * 1.1920928955078125e-07f;
    const float u2 = ((float)(w1 >> 9) + 0.5f) * 1.1920928955078125e-07f;
    const float amp = sqrtf(-2.0f * logf(u1) * var);
    float s, c;
    sincospif(2.0f * u2, &s, &c);
    return make_float2(amp * c, amp * s);
}

// The same increment on the special-function unit (complex fp32, the fused kernels): lg2, sqrt, sin and cos are one MUFU
// instruction each instead of the 50 or so FP32 instructions of logf / sqrtf / sincospif, which sat on the FMA pipe that
// bounds those kernels.  -2 ln u1 = (-2 ln 2) lg2 u1; the angle is folded to [-pi, pi) exactly (u2 - 1/2 is exact), where
// sin.approx / cos.approx have an absolute error of about 2^-21: the increment is within 1e-6 of its magnitude of the
// full-precision one (measured field error at the 500-step gate of cfg5: DESIGN.md section 6).  PHX_FAST_NOISE=0 restores
// the full-precision map in every kernel.
#ifndef PHX_FAST_NOISE
#define PHX_FAST_NOISE 1
#endif
__device__ __forceinline__ float2 noise_increment_sfu(uint32_t w0, uint32_t w1, float var) {
#if PHX_FAST_NOISE
    const float u1 = ((float)(w0 >> 9) + 0.5f) * 1.1920928955078125e-07f;
    const float u2 = ((float)(w1 >> 9) + 0.5f) * 1.1920928955078125e-07f;
    float l2, amp, sn, cs;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(u1));                    // u1 >= 2^-24: never denormal
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(amp) : "f"(-1.3862943611198906f * l2 * var));
    const float th = 6.283185307179586f * (u2 - 0.5f);                          // angle - pi
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(sn) : "f"(th));
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cs) : "f"(th));
    return make_float2(-amp * cs, -amp * sn);                                   // cos(th + pi), sin(th + pi)
#else
    return noise_increment(w0, w1, var);
#endif
}
__device__ __forceinline__ double2 noise_increment_sfu(uint32_t w0, uint32_t w1, double var);

__device__ __forceinline__ double2 noise_increment(uint32_t w0, uint32_t w1, double var) {
    const double u1 = ((double)(w0 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double u2 = ((double)(w1 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double amp = sqrt(-2.0 * log(u1) * var);
    double s, c;
    sincospi(2.0 * u2, &s, &c);
    return make_double2(amp * c, amp * s);
}
__device__ __forceinline__ double2 noise_increment_sfu(uint32_t w0, uint32_t w1, double var) { return noise_increment(w0, w1, var); }

}  // namespace phx
