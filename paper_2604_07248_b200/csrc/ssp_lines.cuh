// ssp_lines.cuh -- how lines of the field map onto CTAs, shared-memory exchange accessors,
// and the pointwise math applied between transforms.
#pragma once

#include "ssp_fft.cuh"

namespace ssp {

// ---- CTA shapes --------------------------------------------------------------------
// WIDE: pad 2 per row of the exchange matrix (16-byte aligned rows) and 16-byte reads; taken where a warp's
// accesses stay conflict-free with it: the two-stage plans of N = 512 and 1024.
template <int N>
struct RowWide { static constexpr bool value = (N == 1024); };

// Row-kernel CTA size and resident CTAs per SM the register budget is sized for.  Default: 256
// threads, 512 resident threads at E = 32 and 1024 at E = 16.  N = 1024 (one warp per row, 32 points
// per thread) measured best on B200 with 168 registers: 3 CTAs of 4 rows.
template <int N>
struct RowTune {
    static constexpr int MAX_THREADS = 256;
    static constexpr int MIN_BLOCKS = (PlanInfo<N, 0>::E >= 32) ? 2 : 4;
};
template <>
struct RowTune<1024> {
    static constexpr int MAX_THREADS = 128;
    static constexpr int MIN_BLOCKS = 3;
};
#ifndef SSP_ROW512_TMEM
#define SSP_ROW512_TMEM 1
#endif
template <>
struct RowTune<2048> {
    static constexpr int MAX_THREADS = 64;
    static constexpr int MIN_BLOCKS = 6;
};
#if SSP_P4096_ROW64
template <>
struct RowTune<4096> {                                           // (64,64), 64 points per thread: two rows per CTA, 255 registers
    static constexpr int MAX_THREADS = 128;
    static constexpr int MIN_BLOCKS = 2;
};
#else
template <>
struct RowTune<4096> : RowTune<1024> {};
#endif

template <int N>
struct RowCfg {
    static constexpr int V = 0;                                   // plan variant
    static constexpr int T = PlanInfo<N, 0>::T;
    static constexpr int THREADS = (T * N < RowTune<N>::MAX_THREADS) ? T * N : RowTune<N>::MAX_THREADS;
    static constexpr int LPB = THREADS / T;                        // lines (rows) per CTA
    static constexpr bool WARP_LOCAL = (T <= 32);                  // a line never spans two warps
    static constexpr bool WIDE = RowWide<N>::value;
    static constexpr int LINE_ELEMS = WIDE ? PlanInfo<N, 0>::LINE_ELEMS2 : PlanInfo<N, 0>::LINE_ELEMS;
    static constexpr size_t SMEM_X = (PlanInfo<N, 0>::NSTAGE == 1) ? 0
        : sizeof(float2) * (size_t)LPB * LINE_ELEMS;                       // exchange buffers
    static constexpr size_t SMEM_PHI = sizeof(float) * (size_t)LPB * N; // prefetched screen rows
    static constexpr size_t SMEM = SMEM_X + SMEM_PHI;
    static constexpr int MIN_BLOCKS = (THREADS < RowTune<N>::MAX_THREADS) ? 1 : RowTune<N>::MIN_BLOCKS;
    // packed fp32 pairs in the split-step row kernel: measured 1024 +4 %, 2048 +2 %, 4096 +4 %; 512 (shuffle plan, one warp per row at 16 points per thread) -20 %
    static constexpr bool PACKED = (N >= 1024);
    // persistent common split-step kernel with the twiddles and hx per thread in tensor memory (+ 16 bytes for the TMEM slot)
#ifndef SSP_ROW1024_TMEM
#define SSP_ROW1024_TMEM 1
#endif
    // measured: 1024 +4 % (+1.3 % more with the next-row prefetch), 512 +12 % (3907 -> 4381 GB/s); 2048 as two rows per
    // 128-thread CTA -4 % and 4096 -10 % (both spill at 168 registers; 4096 with 255 registers at 2 or 3 CTAs/SM:
    // 3805 -> 3458 / 3427 GB/s; without the next-row prefetch, 168 registers: 3788 -> 3482), so those keep the
    // one-row-per-CTA kernels
    static constexpr bool TMEM = (N == 1024 && SSP_ROW1024_TMEM) || (N == 512 && SSP_ROW512_TMEM);
};

// Between the column kernel and the row kernel of a split step the field may stay re/im-swapped: the column
// kernel's inverse transform runs as forward code on swapped data and the row kernel's inverse transform wants
// exactly that, so neither swaps.  With scalar arithmetic the swap is register renaming and nothing is gained; with
// packed pairs it would cost two MOVs per element on each side.  Only the TMA column kernel writes this form.
template <int N>
struct MidSwapped {
    static constexpr bool value = RowCfg<N>::PACKED && PlanInfo<N, 0>::SYM && PlanInfo<N, 1>::SYM;
};

// The common split-step row kernel reads the window from a cached fp32 map instead of evaluating the super-Gaussian per
// pixel (5 FMA-pipe cycles and 3 SFU calls less per pixel, one coalesced 4-byte load more; the 4 MB map of 1024^2 stays in
// L2).  Measured: 1024 rows +2 % clock for clock; at 2048 the 16 MB map costs 4 % (4478 -> 4286 GB/s), so 1024 only.
template <int N>
struct WinMap { static constexpr bool value = RowCfg<N>::PACKED && N == 1024; };

// Statistics epilogue of the last row kernel: lanes of one row inside a warp form a group that writes one record;
// a field has N * T / W records.
template <int N>
struct StatsGroup {
    static constexpr int T = PlanInfo<N, 0>::T;
    static constexpr int W = T < 32 ? T : 32;
    static constexpr int RECORDS_PER_FIELD = N * (T / W);
};

template <int N, int V_ = 1>
struct ColCfg {
    static constexpr int V = V_;                                  // plan variant
    static constexpr int T = PlanInfo<N, V_>::T;
    // columns per CTA: 16 columns = 128-byte row segments while the tile fits one SM's
    // shared memory next to a second CTA; wider grids trade segment width for tile height.
    static constexpr int C = (N <= 8) ? 8 : (N <= 512 ? 16 : (N <= 2048 ? 8 : 4));
    static constexpr int THREADS = T * C;
    static constexpr size_t SMEM = (PlanInfo<N, V_>::NSTAGE == 1) ? 0
        : sizeof(float2) * (size_t)C * PlanInfo<N, V_>::LINE_ELEMS;
    static constexpr int MIN_BLOCKS = (THREADS <= 256 && PlanInfo<N, V_>::E <= 32) ? 2 : 1;   // 64 points per thread: 255 registers
};

// ---- shared-memory exchange accessors -------------------------------------------------
// T = threads per line.  A line inside one warp synchronises with __syncwarp; a line spanning
// several warps uses its own named barrier (id 1 + line-in-CTA), so lines never wait on each other.
template <int T, bool WIDE = false>
struct RowSmem {
    static constexpr int PAD = WIDE ? 2 : 1;
    static constexpr int LANE_STRIDE = 1;       // lanes per thread step of a line (ssp_fft.cuh: fft_logical_t)
    float2 *base; // this line's padded buffer
    int bar_id;
    __device__ __forceinline__ void ld2(int p, float2 &a, float2 &b) const
    {
        const float4 w = *reinterpret_cast<const float4 *>(base + p);
        a = make_float2(w.x, w.y);
        b = make_float2(w.z, w.w);
    }
    __device__ __forceinline__ void st(int p, float2 x) { base[p] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p]; }
    __device__ __forceinline__ void sync()
    {
        if constexpr (T <= 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(T) : "memory");
    }
};

// GT > 0: the CTA holds several tiles at once, each worked on by its own group of GT threads that synchronises on
// its own named barrier (bar_id) instead of the CTA-wide one.
template <int C, int GT = 0>
struct ColSmem {
    static constexpr int PAD = 1;
    static constexpr int LANE_STRIDE = C;       // lanes per thread step of a line (ssp_fft.cuh: fft_logical_t)
    float2 *base; // tile base + this thread's column
    int bar_id = 0;
    __device__ __forceinline__ void st(int p, float2 x) { base[p * C] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p * C]; }
    __device__ __forceinline__ void sync()
    {
        if constexpr (GT == 0) __syncthreads();
        else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(GT) : "memory");
    }
};

// ---- tensor-memory allocation (tcgen05.alloc / dealloc; one warp, address through shared memory) ----------------
__device__ __forceinline__ void tmem_alloc(unsigned *smem_slot, int cols_pow2)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(smem_slot)), "r"(cols_pow2) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned taddr, int cols_pow2)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols_pow2) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---- asynchronous global -> shared copies (LDGSTS), 16 bytes each
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;\n" ::"n"(PENDING) : "memory"); }

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

// the same reduction on two arguments at once (packed fp32 pairs; the SFU calls stay scalar)
__device__ __forceinline__ void sincos_reduced2(float2 x, float2 *s, float2 *c)
{
    const float2 kk = f2mul(x, make_float2(0.15915494309189535f, 0.15915494309189535f));
    const float2 nk = make_float2(-rintf(kk.x), -rintf(kk.y));
    float2 r = f2fma(nk, make_float2(6.2831854820251465f, 6.2831854820251465f), x);
    r = f2fma(nk, make_float2(-1.7484555e-7f, -1.7484555e-7f), r);
    *s = make_float2(__sinf(r.x), __sinf(r.y));
    *c = make_float2(__cosf(r.x), __cosf(r.y));
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2_approx(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// super-Gaussian window exp(-(q)^(h)), q = r^2/sigma^2: three SFU ops, no special-case fix-ups
// (q = 0: lg2 -> -inf, ex2 -> 0, exp(-0) = 1).
__device__ __forceinline__ float window_amp(float q, float h)
{
    return ex2_approx(-1.4426950408889634f * ex2_approx(h * lg2_approx(q)));
}

__device__ __forceinline__ float2 window_amp2(float2 q, float h)
{
    const float2 e = f2mul(make_float2(lg2_approx(q.x), lg2_approx(q.y)), make_float2(h, h));
    const float2 f = f2mul(make_float2(ex2_approx(e.x), ex2_approx(e.y)), make_float2(-1.4426950408889634f, -1.4426950408889634f));
    return make_float2(ex2_approx(f.x), ex2_approx(f.y));
}

} // namespace ssp
