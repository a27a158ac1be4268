// ssp_philox.cuh -- the counter-based generator behind ssp_fill_noise and the seeded screen evolution (device code).
//
// Philox-4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11).  Block i of a stream has counter
// (i mod 2^32, i >> 32, stream mod 2^32, stream >> 32) and key (seed mod 2^32, seed >> 32); its words (x0, x1) make
// draw 2i and (x2, x3) draw 2i+1 by Box-Muller on 23-bit uniforms (ssp_noise.cu; Q3, Q29).
#pragma once

#include "ssp_internal.h"

namespace ssp {

__device__ __forceinline__ void philox_round(uint32_t (&c)[4], uint32_t k0, uint32_t k1)
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t h0 = __umulhi(M0, c[0]), l0 = M0 * c[0];
    const uint32_t h1 = __umulhi(M1, c[2]), l1 = M1 * c[2];
    c[0] = h1 ^ c[1] ^ k0;
    c[1] = l1;
    c[2] = h0 ^ c[3] ^ k1;
    c[3] = l0;
}

// sin / cos through the special-function unit (absolute error about 2^-21 on [-pi, pi]; the draw's error is that times
// r <= 5.8, below the fp32 rounding the screen generator adds afterwards); the logarithm stays the accurate one, because
// for u -> 1 the radius is sqrt of a small difference and an absolute error in ln u would be divided by r.
__device__ __forceinline__ float2 box_muller(uint32_t xr, uint32_t xa)
{
    const float u = ((float)(xr >> 9) + 0.5f) * 1.1920928955078125e-7f;          // 2^-23; k + 1/2 needs 24 bits: exact
    const float g = ((float)(xa >> 9) + 0.5f) * 2.384185791015625e-7f - 1.0f;    // 2 f - 1 in (-1, 1), exact
    float r;
    asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(-2.0f * logf(u)));
    // angle 2 pi f = pi g + pi:  cos(2 pi f) = -cos(pi g),  sin(2 pi f) = -sin(pi g)
    const float th = 3.14159265358979f * g;
    return make_float2(-r * __cosf(th), -r * __sinf(th));
}

// the four output words of block i of stream (s0, s1)
__device__ __forceinline__ void philox_block(const RoundKeys &keys, unsigned long long i, uint32_t s0, uint32_t s1,
                                             uint32_t (&c)[4])
{
    c[0] = (uint32_t)i; c[1] = (uint32_t)(i >> 32); c[2] = s0; c[3] = s1;
#pragma unroll
    for (int r = 0; r < 10; ++r) philox_round(c, keys.k[r][0], keys.k[r][1]);
}

} // namespace ssp
