// ssp_noise.cu -- device-side draws of the "unit-variance complex Gaussian" noise of the screen synthesis
// (PAPER.md:359 S16; Q3, Q29).  The paper draws it with its framework's generator on the GPU; here the noise
// arrays stay plain inputs of the screen calls and this kernel optionally fills them from (seed, stream).
//
// Generator: Philox-4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11).  Block i of a stream has counter
// (i mod 2^32, i >> 32, stream mod 2^32, stream >> 32) and key (seed mod 2^32, seed >> 32); its words (x0, x1) make
// draw 2i and (x2, x3) draw 2i+1 by Box-Muller on 23-bit uniforms (k + 1/2, k < 2^23, is exact in fp32):
//   u = ((x_even >> 9) + 1/2) 2^-23,  f = ((x_odd >> 9) + 1/2) 2^-23,  z = sqrt(-2 ln u) (cos 2 pi f + i sin 2 pi f).
// One thread makes one block = two complex64 draws = one 16-byte store; pure ALU + write stream (8 B per draw).
#include "ssp_internal.h"
#include "ssp_philox.cuh"

namespace ssp {

__global__ void __launch_bounds__(256) k_fill_noise(const RoundKeys keys, uint32_t s0, uint32_t s1,
                                                     unsigned long long first_block, unsigned long long n_draws,
                                                     float2 *__restrict__ out)
{
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;   // block within this call
    if (2 * j >= n_draws) return;
    uint32_t c[4];
    philox_block(keys, first_block + j, s0, s1, c);
    const float2 z0 = box_muller(c[0], c[1]), z1 = box_muller(c[2], c[3]);
    if (2 * j + 1 < n_draws) reinterpret_cast<float4 *>(out)[j] = make_float4(z0.x, z0.y, z1.x, z1.y);
    else out[2 * j] = z0;
}

// the generator's raw words (no Box-Muller): block first_block + j -> out[j] = (x0, x1, x2, x3); the block index wraps mod 2^64
__global__ void __launch_bounds__(256) k_philox_words(const RoundKeys keys, uint32_t s0, uint32_t s1,
                                                       unsigned long long first_block, unsigned long long n_blocks,
                                                       uint4 *__restrict__ out)
{
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_blocks) return;
    uint32_t c[4];
    philox_block(keys, first_block + j, s0, s1, c);
    out[j] = make_uint4(c[0], c[1], c[2], c[3]);
}

RoundKeys key_schedule(unsigned long long seed)
{
    RoundKeys keys;
    for (int r = 0; r < 10; ++r) {
        keys.k[r][0] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
        keys.k[r][1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
    }
    return keys;
}

int launch_fill_noise(ssp_ctx *ctx, unsigned long long seed, unsigned long long stream, unsigned long long first,
                      unsigned long long n, float2 *out)
{
    const unsigned long long blocks = (n + 1) / 2;
    const unsigned long long grid = (blocks + 255) / 256;
    if (grid > 0x7FFFFFFFull) return ctx->fail(SSP_EINVAL, "ssp_fill_noise: more than 2^40 draws in one call");
    const RoundKeys keys = key_schedule(seed);
    ctx->prof_begin("fill_noise", 8.0 * (double)n);
    k_fill_noise<<<(unsigned)grid, 256, 0, ctx->stream>>>(keys, (uint32_t)stream, (uint32_t)(stream >> 32), first / 2, n, out);
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

} // namespace ssp

extern "C" int ssp_fill_noise(ssp_ctx *ctx, unsigned long long seed, unsigned long long stream,
                              unsigned long long first, unsigned long long n, float *d_out)
{
    if (!ctx) return SSP_EINVAL;
    if (n == 0) return SSP_OK;
    if (!d_out || (first & 1ull) || (reinterpret_cast<uintptr_t>(d_out) & 15u))
        return ctx->fail(SSP_EINVAL, "ssp_fill_noise: null or misaligned output, or odd first draw");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    return ssp::launch_fill_noise(ctx, seed, stream, first, n, reinterpret_cast<float2 *>(d_out));
}

extern "C" int ssp_philox_words(ssp_ctx *ctx, unsigned long long seed, unsigned long long stream,
                                unsigned long long first_block, unsigned long long n_blocks, unsigned int *d_out)
{
    if (!ctx) return SSP_EINVAL;
    if (n_blocks == 0) return SSP_OK;
    if (!d_out || (reinterpret_cast<uintptr_t>(d_out) & 15u) || n_blocks > (1ull << 38))
        return ctx->fail(SSP_EINVAL, "ssp_philox_words: null or misaligned output, or more than 2^38 blocks");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const ssp::RoundKeys keys = ssp::key_schedule(seed);
    ssp::k_philox_words<<<(unsigned)((n_blocks + 255) / 256), 256, 0, ctx->stream>>>(
        keys, (uint32_t)stream, (uint32_t)(stream >> 32), first_block, n_blocks, reinterpret_cast<uint4 *>(d_out));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}
