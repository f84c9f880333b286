// phx_philox.cuh -- counter-based noise of the stochastic step (Eq. (22)).
// Philox4x32-10 (Salmon et al., SC'11) keyed by (seed, realisation) with counter (cell, step_lo, step_hi, 0)
// (BASELINE.json config 5; reading Q13).  Product code: shares nothing with oracle/.
#pragma once

#include "phx_common.cuh"

namespace phx {

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
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

__device__ __forceinline__ double2 noise_increment(uint32_t w0, uint32_t w1, double var) {
    const double u1 = ((double)(w0 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double u2 = ((double)(w1 >> 9) + 0.5) * 1.1920928955078125e-07;
    const double amp = sqrt(-2.0 * log(u1) * var);
    double s, c;
    sincospi(2.0 * u2, &s, &c);
    return make_double2(amp * c, amp * s);
}

}  // namespace phx
