// ssp_lines.cuh -- how lines of the field map onto CTAs, shared-memory exchange accessors,
// and the pointwise math applied between transforms.
#pragma once

#include "ssp_fft.cuh"

namespace ssp {

// ---- CTA shapes --------------------------------------------------------------------
template <int N>
struct RowCfg {
    static constexpr int T = PlanInfo<N>::T;
    static constexpr int THREADS = (T * N < 256) ? T * N : 256;
    static constexpr int LPB = THREADS / T;                        // lines (rows) per CTA
    static constexpr bool WARP_LOCAL = (T <= 32);                  // a line never spans two warps
    static constexpr size_t SMEM_X = (PlanInfo<N>::NSTAGE == 1) ? 0
        : sizeof(float2) * (size_t)LPB * PlanInfo<N>::LINE_ELEMS;       // exchange buffers
    static constexpr size_t SMEM_PHI = sizeof(float) * (size_t)LPB * N; // prefetched screen rows
    static constexpr size_t SMEM = SMEM_X + SMEM_PHI;
    static constexpr int MIN_BLOCKS = (THREADS * PlanInfo<N>::E >= 8192) ? 2 : 1;
};

template <int N>
struct ColCfg {
    static constexpr int T = PlanInfo<N>::T;
    // columns per CTA: 16 columns = 128-byte row segments while the tile fits one SM's
    // shared memory next to a second CTA; wider grids trade segment width for tile height.
    static constexpr int C = (N <= 8) ? 8 : (N <= 512 ? 16 : (N <= 2048 ? 8 : 4));
    static constexpr int THREADS = T * C;
    static constexpr size_t SMEM = (PlanInfo<N>::NSTAGE == 1) ? 0
        : sizeof(float2) * (size_t)C * PlanInfo<N>::LINE_ELEMS;
    static constexpr int MIN_BLOCKS = (THREADS <= 256) ? 2 : 1;
};

// ---- shared-memory exchange accessors -------------------------------------------------
template <bool WARP_LOCAL>
struct RowSmem {
    float2 *base; // this line's padded buffer
    __device__ __forceinline__ void st(int p, float2 x) { base[p] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p]; }
    __device__ __forceinline__ void sync()
    {
        if (WARP_LOCAL) __syncwarp(); else __syncthreads();
    }
};

template <int C>
struct ColSmem {
    float2 *base; // tile base + this thread's column
    __device__ __forceinline__ void st(int p, float2 x) { base[p * C] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p * C]; }
    __device__ __forceinline__ void sync() { __syncthreads(); }
};

// ---- asynchronous global -> shared copies (LDGSTS), 16 bytes each
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// ---- pointwise math -----------------------------------------------------------------
// sin/cos of a phase of any magnitude: Cody-Waite reduction by 2 pi, then the SFU.
__device__ __forceinline__ void sincos_reduced(float x, float *s, float *c)
{
    const float k = rintf(x * 0.15915494309189535f);
    float r = fmaf(-k, 6.2831854820251465f, x);          // 2 pi rounded to fp32
    r = fmaf(-k, -1.7484555e-7f, r);                     // 2 pi - fp32(2 pi)
    *s = __sinf(r);
    *c = __cosf(r);
}

// super-Gaussian window exp(-(q)^(h)), q = r^2/sigma^2 (q = 0 -> 1)
__device__ __forceinline__ float window_amp(float q, float h)
{
    return __expf(-__powf(q, h));
}

} // namespace ssp
