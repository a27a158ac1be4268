// ssp_col_tma.cuh -- column pass of the split step with the tile moved by TMA (K5).
//
// A tile is C adjacent columns x N rows of one field.  Persistent CTAs walk the tiles with two
// shared-memory buffers each: while tile i is transformed (FFT_y -> * hy/N^2 -> IFFT_y, PAPER.md:37
// Eq.1) in buffer i&1, the TMA engine loads tile i+1 into the other buffer, and the result of tile
// i leaves through a TMA store from the buffer it was computed in.  No global load or store is
// issued by the threads, so the column kernel neither queues on the LSU nor exposes DRAM latency.
// The buffer is used three ways in turn: dense [row][C] tile written by TMA, padded exchange
// buffer of the in-register FFT (ssp_fft.cuh), dense result tile read by TMA.
#pragma once

#include <cuda.h>

#include "ssp_internal.h"
#include "ssp_lines.cuh"

namespace ssp {

// ---- mbarrier / bulk-tensor copy wrappers (PTX ISA: mbarrier, cp.async.bulk.tensor) ------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *tm, int x, int y, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(x), "r"(y), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap *tm, int x, int y, const void *src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(tm), "r"(x), "r"(y), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// ---- CTA shape ---------------------------------------------------------------------------------
// C columns per tile (TMA rows of 8 C bytes, at least 16), NBUF shared-memory buffers per CTA (2: persistent
// CTAs, the load of the next tile overlaps the transform; 1: one tile per CTA), resident CTAs per SM.
// NG = 2 (with NBUF = 3, one CTA per SM): two groups of T C threads work on two tiles at once, each on its own
// named barrier, and share three tile buffers -- tile n of the CTA goes to group n % 2 in buffer n % 3, and the load of
// tile n + 3 is issued into a buffer as soon as the store of tile n has read it.  A tall tile (N >= 2048: 64 KB) then
// always has its successor landed or in flight, which two independent one-buffer CTAs per SM cannot arrange.
template <int N>
struct ColTmaTune { static constexpr int C = 4, NBUF = 2, MIN_BLOCKS = 3, NG = 1; static constexpr bool ENABLED = false; };
template <> struct ColTmaTune<512> { static constexpr int C = 8, NBUF = 2, MIN_BLOCKS = 3, NG = 1; static constexpr bool ENABLED = true; };
#ifndef SSP_T1024_C
#define SSP_T1024_C 4
#define SSP_T1024_NBUF 2
#define SSP_T1024_MINB 3
#define SSP_T1024_NG 1
#endif
// 2048^2 (64 KB tiles of 4 columns), measured: one tile per CTA, 2 CTAs/SM 3749 GB/s; two groups on three buffers
// 2997 (200 KB of shared memory leave no L1 for the twiddle / hy reads), the same with those in tensor memory 4015
#ifndef SSP_T2048_C
#define SSP_T2048_C 4
#define SSP_T2048_NBUF 3
#define SSP_T2048_MINB 1
#define SSP_T2048_NG 2
#endif
#ifndef SSP_T4096_C
#define SSP_T4096_C 2
#define SSP_T4096_NBUF 1
#define SSP_T4096_MINB 2
#define SSP_T4096_NG 1
#endif
template <int C_, int NBUF_, int MINB_, int NG_> struct ColTmaTuneV { static constexpr int C = C_, NBUF = NBUF_, MIN_BLOCKS = MINB_, NG = NG_; static constexpr bool ENABLED = true; };
template <> struct ColTmaTune<1024> : ColTmaTuneV<SSP_T1024_C, SSP_T1024_NBUF, SSP_T1024_MINB, SSP_T1024_NG> {};
template <> struct ColTmaTune<2048> : ColTmaTuneV<SSP_T2048_C, SSP_T2048_NBUF, SSP_T2048_MINB, SSP_T2048_NG> {};
template <> struct ColTmaTune<4096> : ColTmaTuneV<SSP_T4096_C, SSP_T4096_NBUF, SSP_T4096_MINB, SSP_T4096_NG> {};

template <int N>
struct ColTmaCfg {
    static constexpr int T = PlanInfo<N, 1>::T;
    static constexpr int C = ColTmaTune<N>::C;
    static constexpr int NBUF = ColTmaTune<N>::NBUF;
    static constexpr int NG = ColTmaTune<N>::NG;                      // tiles in work at once (groups of GT threads)
    static constexpr int GT = T * C;
    static constexpr int THREADS = NG * GT;
    static_assert(NG == 1 || (NG == 2 && NBUF == 3 && GT % 32 == 0), "two groups rotate through three buffers");
    static constexpr int MIN_BLOCKS = ColTmaTune<N>::MIN_BLOCKS;
    static constexpr int BOX_ROWS = (N < 256) ? N : 256;              // TMA box dimensions are <= 256
    static constexpr int BOXES = N / BOX_ROWS;
    static constexpr int BUF_ELEMS = C * PlanInfo<N, 1>::LINE_ELEMS;  // float2 per buffer (padded exchange)
    static constexpr size_t SMEM = NBUF * sizeof(float2) * BUF_ELEMS + 64;   // + six mbarriers + the TMEM address slot
    static constexpr unsigned TILE_BYTES = (unsigned)(sizeof(float2) * C * N);
    // packed fp32 pairs: measured 2048 +3.6 %, 4096 +1.3 %; 1024 -1 % and 512 +1 % (within noise) stay scalar
#ifndef SSP_COL1024_PK
#define SSP_COL1024_PK 0
#endif
    static constexpr bool PACKED = (N >= 2048) || (N == 1024 && SSP_COL1024_PK);
    // first-stage twiddles and the hy table kept per thread in tensor memory (128 columns per CTA): persistent CTAs only
#ifndef SSP_COL1024_TMEM
#define SSP_COL1024_TMEM 1
#endif
// measured at 2048 / 4096 with ONE tile buffer (the persistent loop reloads it only after its own store has drained):
// 3735 -> 3375 GB/s and 3161 -> 2590 GB/s -- fresh CTAs overlap one tile's store with the next one's load better than
// the single-buffer loop does; 2048 runs two groups on three buffers (ColTmaTune) and keeps the cache, 4096 stays off
// (two groups there: 3164 -> 2464, with the cache 2499: 16-byte TMA rows are the limit, profiles/r02_tma_rows.md)
#ifndef SSP_COL2048_TMEM
#define SSP_COL2048_TMEM 1
#endif
#ifndef SSP_COL4096_TMEM
#define SSP_COL4096_TMEM 0
#endif
    static constexpr bool TMEM = ((N == 1024 && SSP_COL1024_TMEM) || (N == 2048 && SSP_COL2048_TMEM) || (N == 4096 && SSP_COL4096_TMEM)) &&
                                 PlanInfo<N, 1>::SYM && PlanInfo<N, 1>::E == PlanInfo<N, 1>::R1 && (THREADS % 128 == 0);
    // per thread: 2E words of twiddle pairs, then 2E words of hy; warps w and w + 4 take consecutive column blocks of 4E
    static constexpr int TM_HOFF = 2 * PlanInfo<N, 1>::E, TM_CW = 4 * PlanInfo<N, 1>::E;
    static constexpr int TM_NEED = (THREADS / 128) * TM_CW;
    static constexpr int TMEM_COLS = TM_NEED <= 128 ? 128 : (TM_NEED <= 256 ? 256 : 512);
    // persistent even with one buffer (the tile loop reloads the buffer after its store has drained) when TMEM is on
    static constexpr bool PERSIST = (NBUF >= 2) || TMEM;
};

// Screen generator (K1+K2): one tile per CTA, one buffer (noise -> exchange -> result) plus a second one only
// when a spectrum is read or kept (old spectrum -> new spectrum).
template <int N>
struct ScreenColTmaTune { static constexpr int C = 4, MIN_BLOCKS = 3; static constexpr bool ENABLED = false; };
template <> struct ScreenColTmaTune<512> { static constexpr int C = 8, MIN_BLOCKS = 3; static constexpr bool ENABLED = true; };
template <> struct ScreenColTmaTune<1024> { static constexpr int C = 4, MIN_BLOCKS = 3; static constexpr bool ENABLED = true; };

template <int N>
struct ScreenColTmaCfg {
    static constexpr int T = PlanInfo<N, 1>::T;
    static constexpr int C = ScreenColTmaTune<N>::C;
    static constexpr int THREADS = T * C;
    static constexpr int MIN_BLOCKS = ScreenColTmaTune<N>::MIN_BLOCKS;
    static constexpr int BOX_ROWS = (N < 256) ? N : 256;
    static constexpr int BOXES = N / BOX_ROWS;
    static constexpr int BUF_ELEMS = C * PlanInfo<N, 1>::LINE_ELEMS;
    static constexpr size_t HEAD = 128;                               // mbarrier, keeps the buffers 128-byte aligned
    static constexpr size_t smem(int nbuf) { return HEAD + (size_t)nbuf * sizeof(float2) * BUF_ELEMS; }
    static constexpr unsigned TILE_BYTES = (unsigned)(sizeof(float2) * C * N);
};

struct ColTmaArgs {
    const float2 *hy;            // [N] multiplier between the transforms (separable H), or
    const float2 *h2d;           // tile-major [N/C][N][C] multiplier H(ky,kx) when H2D (non-separable H)
    const float2 *tw;            // column-plan twiddles
    int ntiles;                  // B * N / C
};

// FFT_y -> * hy -> IFFT_y.  tm_in / tm_out describe the [B*N rows][2N floats] field buffers.
template <int N, bool H2D>
__global__ void __launch_bounds__(ColTmaCfg<N>::THREADS, ColTmaCfg<N>::MIN_BLOCKS)
k_col_tma(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_out, const ColTmaArgs a)
{
    using PI = PlanInfo<N, 1>;
    using CFG = ColTmaCfg<N>;
    constexpr int E = PI::E, C = CFG::C, R1 = PI::R1, RL = PI::RL;
    constexpr bool SYM = (R1 == RL), PK = CFG::PACKED;
    static_assert(SYM || !MidSwapped<N>::value, "the swapped hand-over needs the forward-only body");
    constexpr int GROUPS = N / C;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *sbuf = reinterpret_cast<float2 *>(smem_raw);
    unsigned long long *full = reinterpret_cast<unsigned long long *>(smem_raw + CFG::NBUF * sizeof(float2) * CFG::BUF_ELEMS);
    constexpr int NG = CFG::NG, GT = CFG::GT;
    const int tid = threadIdx.x, grp = tid / GT, ltid = tid % GT, c = ltid % C, t = fft_logical_t<N, 1, C>(ltid / C);
    auto group_sync = [&]() {                                     // the threads working on one tile
        if constexpr (NG == 1) __syncthreads();
        else asm volatile("bar.sync %0, %1;" ::"r"(1 + grp), "n"(GT) : "memory");
    };

    // bar: the mbarrier that announces this fill.  Two groups: fill k of a buffer uses the buffer's barrier k & 1, so
    // that a group waiting for fill k + 1 while the other group has not yet seen fill k complete never meets a barrier
    // whose previous phase has the parity it waits for.
    auto issue_load = [&](int tile, int buf, int bar) {
        const int b = tile / GROUPS, col0 = (tile % GROUPS) * C;
        mbar_expect_tx(&full[bar], CFG::TILE_BYTES);
#pragma unroll
        for (int j = 0; j < CFG::BOXES; ++j)
            tma_load_2d(sbuf + buf * CFG::BUF_ELEMS + j * CFG::BOX_ROWS * C, &tm_in, 2 * col0, b * N + j * CFG::BOX_ROWS,
                        &full[bar]);
    };
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < 6; ++i) mbar_init(&full[i], 1);
        fence_mbar_init();
        pdl_wait();                                               // (ssp_internal.h) the tiles are the previous kernel's output
        if ((int)blockIdx.x < a.ntiles) issue_load(blockIdx.x, 0, 0);
        if constexpr (NG == 2) {                                  // all three buffers start empty: fill 0 of buffers 1 and 2
            if ((int)(blockIdx.x + gridDim.x) < a.ntiles) issue_load(blockIdx.x + gridDim.x, 1, 2);
            if ((int)(blockIdx.x + 2 * gridDim.x) < a.ntiles) issue_load(blockIdx.x + 2 * gridDim.x, 2, 4);
        }
    }
    // Tensor memory as a per-thread constant cache: this thread's 16 twiddle pairs W_N^(t k) and the 32 hy values of
    // its points never change while the CTA walks its tiles, so they are read from the thread's own TMEM lane
    // (tcgen05.ld) instead of through the LSU data pipe, which this kernel saturates first.
    constexpr bool TM = CFG::TMEM;                                  // twiddles; the multiplier too when it is the 1-D table hy
    constexpr bool TMH = CFG::TMEM && !H2D;
    unsigned &tmem_slot = *reinterpret_cast<unsigned *>(full + 6);     // (a static __shared__ would shift the TMA buffers)
    unsigned taddr = 0;
    if constexpr (TM) {
        if (tid < 32) tmem_alloc(&tmem_slot, CFG::TMEM_COLS);
        tmem_fence_before_sync();
    }
    __syncthreads();
    if constexpr (TM) {
        tmem_fence_after_sync();
        taddr = tmem_slot + ((unsigned)(tid & 96) << 16) + (unsigned)(tid / 128) * CFG::TM_CW;   // lane quadrant w % 4, column block w / 4
        const float4 *tw4 = reinterpret_cast<const float4 *>(a.tw + PI::TW1) + t;
#pragma unroll
        for (int p = 0; p < R1 / 2; ++p) tmem_st4(taddr + 4 * p, __ldg(tw4 + p * (N / R1)));
        if constexpr (TMH) {
#pragma unroll
            for (int q = 0; q < RL; q += 2) {
                const float2 h0 = __ldg(a.hy + line_index<N, 1, RL>(t, 0, q)), h1 = __ldg(a.hy + line_index<N, 1, RL>(t, 0, q + 1));
                tmem_st4(taddr + CFG::TM_HOFF + 2 * q, make_float4(h0.x, h0.y, h1.x, h1.y));
            }
        }
        tmem_wait_st();
    }
    pdl_wait();                                                   // every thread: the H2D multiplier map may be the previous kernel's output

    // the CTA's n-th tile is blockIdx.x + n gridDim.x; with two groups, group grp takes n = grp, grp + 2, ..
    int it = (NG == 2) ? grp : 0;
    for (int tile = blockIdx.x + it * gridDim.x; tile < a.ntiles; tile += NG * gridDim.x, it += NG) {
        const int cur = (CFG::NBUF == 1) ? 0 : it % CFG::NBUF;    // NBUF == 1: one tile per CTA (grid = tiles)
        float2 *tile_s = sbuf + cur * CFG::BUF_ELEMS;
        ColSmem<C, NG == 1 ? 0 : GT> sm{tile_s + c, 1 + grp};
        const int fill = (CFG::NBUF == 1) ? it : it / CFG::NBUF;  // how often this buffer has been filled before
        const int bar = (NG == 2) ? 2 * cur + (fill & 1) : cur;
        mbar_wait(&full[bar], (NG == 2) ? ((fill >> 1) & 1) : (fill & 1));
        float2 v[E];
#pragma unroll
        for (int i = 0; i < E / R1; ++i)
#pragma unroll
            for (int q = 0; q < R1; ++q) v[i * R1 + q] = tile_s[line_index<N, 1, R1>(t, i, q) * C + c];
        group_sync();                                             // the tile is in registers: the buffer is free
        // multiplier of element (ky, this thread's column): hy[ky], or H(ky,kx) read through L1/L2
        const float2 *hcol = H2D ? a.h2d + (size_t)(tile % GROUPS) * N * C + c : a.hy;
        constexpr int HS = H2D ? C : 1;                           // stride of ky in the multiplier table
        if (CFG::NBUF == 2 && tid == 0 && tile + (int)gridDim.x < a.ntiles) {
            tma_store_wait_read();                                // the store of tile it-1 has released the other buffer
            issue_load(tile + gridDim.x, cur ^ 1, cur ^ 1);
        }
        if constexpr (SYM) {
            // pass 0: forward; * hy, leaving the product re/im-swapped; pass 1: forward on swapped data = inverse
#pragma unroll 1
            for (int pass = 0; pass < 2; ++pass) {
                if constexpr (TM) fft_line<N, 1, false, false, true, PK>(v, t, sm, TwTmem{a.tw, taddr});
                else fft_line<N, 1, false, false, true, PK>(v, t, sm, a.tw);
                if (pass == 0) {
                    if constexpr (TMH) {
#pragma unroll
                        for (int q = 0; q < RL; q += 4) {
                            float4 ha, hb;
                            tmem_ld8(taddr + CFG::TM_HOFF + 2 * q, ha, hb);
                            const float2 h[4] = {make_float2(ha.x, ha.y), make_float2(ha.z, ha.w), make_float2(hb.x, hb.y),
                                                 make_float2(hb.z, hb.w)};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const float2 x = v[q + e];
                                v[q + e] = make_float2(fmaf(x.x, h[e].y, x.y * h[e].x), fmaf(x.x, h[e].x, -x.y * h[e].y));
                            }
                        }
                    } else {
#pragma unroll
                    for (int i = 0; i < E / RL; ++i)
#pragma unroll
                        for (int q = 0; q < RL; ++q) {
                            const float2 h = __ldg(hcol + (size_t)line_index<N, 1, RL>(t, i, q) * HS), x = v[i * RL + q];
                            v[i * RL + q] = make_float2(fmaf(x.x, h.y, x.y * h.x), fmaf(x.x, h.x, -x.y * h.y));
                        }
                    }
                }
            }
#pragma unroll
            for (int i = 0; i < E / R1; ++i)
#pragma unroll
                for (int q = 0; q < R1; ++q) {
                    const float2 x = v[i * R1 + q];
                    tile_s[line_index<N, 1, R1>(t, i, q) * C + c] = MidSwapped<N>::value ? x : make_float2(x.y, x.x);
                }
        } else {
            fft_line<N, 1, false, false, true, PK>(v, t, sm, a.tw);   // strided by RL
#pragma unroll
            for (int i = 0; i < E / RL; ++i)
#pragma unroll
                for (int q = 0; q < RL; ++q)
                    v[i * RL + q] = cmul_c<false, PK>(v[i * RL + q], __ldg(hcol + (size_t)line_index<N, 1, RL>(t, i, q) * HS));
            fft_line<N, 1, true, true, true, PK>(v, t, sm, a.tw);     // inverse, reversed plan; strided by R1
#pragma unroll
            for (int i = 0; i < E / R1; ++i)
#pragma unroll
                for (int q = 0; q < R1; ++q) tile_s[line_index<N, 1, R1>(t, i, q) * C + c] = v[i * R1 + q];
        }
        fence_proxy_async();                                      // generic-proxy writes visible to the TMA store
        group_sync();
        if (ltid == 0) {
            const int b = tile / GROUPS, col0 = (tile % GROUPS) * C;
#pragma unroll
            for (int j = 0; j < CFG::BOXES; ++j)
                tma_store_2d(&tm_out, 2 * col0, b * N + j * CFG::BOX_ROWS, tile_s + j * CFG::BOX_ROWS * C);
            tma_store_commit();
            // one buffer, persistent / two groups on three buffers: reload this buffer once the store has read it
            constexpr int AHEAD = (NG == 2) ? CFG::NBUF : 1;
            if ((CFG::NBUF == 1 || NG == 2) && tile + AHEAD * (int)gridDim.x < a.ntiles) {
                tma_store_wait_read();
                issue_load(tile + AHEAD * gridDim.x, cur, (NG == 2) ? 2 * cur + ((fill + 1) & 1) : cur);
            }
        }
    }
    if (ltid == 0) tma_store_wait_read();
    if constexpr (TM) {
        tmem_fence_before_sync();
        __syncthreads();
        if (tid < 32) tmem_dealloc(tmem_slot, CFG::TMEM_COLS);
    }
}

// ---- wide tiles for the tallest grid ------------------------------------------------------------------------------
// The TMA engine moves about 0.5-0.7 tile ROWS per clock and SM whatever their width (profiles/r02_tma_rows.md): with
// the 16-byte rows of a two-column tile -- all that fits twice into shared memory at N = 4096 -- a plain TMA copy stops
// near 3 TB/s, and k_col_tma<4096> runs at that.  This kernel moves FOUR-column tiles (32-byte rows, 128 KB) and still
// overlaps every load with the transform: one persistent CTA per SM; the landing buffer L holds the tile only until it
// is in registers (64 points per thread), then takes the next tile's load at once; the transform's exchange runs in a
// separate buffer X of HALF a tile, which the two column pairs (warps 0-3: columns 0-1, warps 4-7: columns 2-3) use in
// turn -- pair g waits for the other pair's release before its first exchange write (fft_line's PRE hook) and releases
// X right after its last exchange read (HOOK), named barriers 3 / 4 counting arrivals -- and the result leaves through
// X as two half tiles of 2048 rows.  Twiddles and hy come from tensor memory (the 200 KB of buffers leave no L1).
#ifndef SSP_COL4096_WIDE
#define SSP_COL4096_WIDE 1
#endif
template <int N>
struct ColWideCfg {
    using PI = PlanInfo<N, 1>;
    static constexpr bool ENABLED = (N == 4096) && SSP_COL4096_WIDE;
    static constexpr int C = 4, CP = 2, NPAIR = C / CP;               // columns per tile / per pair
    static constexpr int T = PI::T, E = PI::E;
    static constexpr int GT = T * CP, THREADS = NPAIR * GT;           // 128 threads per pair, 256 per CTA
    static constexpr int BOX_ROWS = 256, BOXES = N / BOX_ROWS;
    static constexpr size_t L_BYTES = sizeof(float2) * (size_t)N * C;
    static constexpr int X_ELEMS = CP * PI::LINE_ELEMS;               // padded exchange of one pair >= half a dense tile
    static constexpr size_t SMEM = L_BYTES + sizeof(float2) * X_ELEMS + 64;
    static constexpr unsigned TILE_BYTES = (unsigned)L_BYTES;
    static constexpr bool PACKED = ColTmaCfg<N>::PACKED;
    static constexpr int TM_HOFF = 2 * E, TM_CW = 4 * E, TMEM_COLS = 512;
    static constexpr bool OK = PI::SYM && PI::NSTAGE == 2 && E == PI::R1 && N / PI::R1 == T && GT == 128 && NPAIR == 2 &&
                               (THREADS / 128) * TM_CW <= 512 && X_ELEMS >= (N / 2) * C && (sizeof(float2) * X_ELEMS) % 128 == 0;
};

template <int N, bool H2D>
__global__ void __launch_bounds__(ColWideCfg<N>::THREADS, 1)
k_col_tma_wide(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_out, const ColTmaArgs a)
{
    using PI = PlanInfo<N, 1>;
    using CFG = ColWideCfg<N>;
    static_assert(CFG::OK, "two-stage symmetric plan with one first-stage butterfly per thread, two pairs of 128 threads");
    constexpr int E = PI::E, T = PI::T, C = CFG::C, CP = CFG::CP, GT = CFG::GT;
    constexpr bool PK = CFG::PACKED;
    constexpr int GROUPS = N / C;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *L = reinterpret_cast<float2 *>(smem_raw);
    float2 *X = reinterpret_cast<float2 *>(smem_raw + CFG::L_BYTES);
    unsigned long long *full = reinterpret_cast<unsigned long long *>(smem_raw + CFG::L_BYTES + sizeof(float2) * CFG::X_ELEMS);
    unsigned &tmem_slot = *reinterpret_cast<unsigned *>(full + 1);
    const int tid = threadIdx.x, pair = tid / GT, ltid = tid % GT, cp = ltid % CP, t = ltid / CP, c = pair * CP + cp;

    auto issue_load = [&](int tile) {
        const int b = tile / GROUPS, col0 = (tile % GROUPS) * C;
        mbar_expect_tx(full, CFG::TILE_BYTES);
#pragma unroll
        for (int j = 0; j < CFG::BOXES; ++j) tma_load_2d(L + j * CFG::BOX_ROWS * C, &tm_in, 2 * col0, b * N + j * CFG::BOX_ROWS, full);
    };
    if (tid == 0) {
        mbar_init(full, 1);
        fence_mbar_init();
        pdl_wait();                                               // (ssp_internal.h) the tiles are the previous kernel's output
        if ((int)blockIdx.x < a.ntiles) issue_load(blockIdx.x);
    }
    if (tid < 32) tmem_alloc(&tmem_slot, CFG::TMEM_COLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    // per thread in its own TMEM lane: E twiddle pairs W_N^(t k), then (separable H) the E hy values of its points
    const unsigned taddr = tmem_slot + ((unsigned)(tid & 96) << 16) + (unsigned)(tid / 128) * CFG::TM_CW;
    {
        const float4 *tw4 = reinterpret_cast<const float4 *>(a.tw + PI::TW1) + t;
#pragma unroll
        for (int p = 0; p < E / 2; ++p) tmem_st4(taddr + 4 * p, __ldg(tw4 + p * (N / E)));
        if constexpr (!H2D) {
#pragma unroll
            for (int q = 0; q < E; q += 2) {
                const float2 h0 = __ldg(a.hy + line_index<N, 1, E>(t, 0, q)), h1 = __ldg(a.hy + line_index<N, 1, E>(t, 0, q + 1));
                tmem_st4(taddr + CFG::TM_HOFF + 2 * q, make_float4(h0.x, h0.y, h1.x, h1.y));
            }
        }
        tmem_wait_st();
    }
    // X hand-over between the pairs: barrier 3 = "pair 0 has read its exchange", 4 = "pair 1 has read its exchange"
    pdl_wait();                                                   // every thread: the H2D multiplier map may be the previous kernel's output
    auto release = [&]() { asm volatile("bar.arrive %0, %1;" ::"r"(3 + pair), "n"(2 * GT) : "memory"); };
    auto wait_other = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(4 - pair), "n"(2 * GT) : "memory"); };

    int it = 0;
    for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x, ++it) {
        mbar_wait(full, it & 1);
        float2 v[E];
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = L[line_index<N, 1, E>(t, 0, q) * C + c];
        if (tid == 0) tma_store_wait_read();                      // the previous tile's second half has left X meanwhile
        __syncthreads();                                          // the tile is in registers, X is free
        if (tid == 0 && tile + (int)gridDim.x < a.ntiles) issue_load(tile + gridDim.x);
        ColSmem<CP, GT> sm{X + cp, 1 + pair};
        const float2 *hcol = a.h2d + (size_t)(tile % GROUPS) * N * C + c;
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            // pass 0: forward, * hy leaving the product re/im-swapped; pass 1: forward on swapped data = inverse.
            // Turns on X: pair 0, pair 1, pair 0, pair 1; pair 0's first turn of a tile has nothing to wait for.
            auto pre = [&]() { if (pair == 1 || pass == 1) wait_other(); };
            fft_line<N, 1, false, false, false, PK>(v, t, sm, TwTmem{a.tw, taddr}, release, pre);
            if (pass == 0) {
                if constexpr (!H2D) {
#pragma unroll
                    for (int q = 0; q < E; q += 4) {
                        float4 ha, hb;
                        tmem_ld8(taddr + CFG::TM_HOFF + 2 * q, ha, hb);
                        const float2 h[4] = {make_float2(ha.x, ha.y), make_float2(ha.z, ha.w), make_float2(hb.x, hb.y), make_float2(hb.z, hb.w)};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float2 x = v[q + e];
                            v[q + e] = make_float2(fmaf(x.x, h[e].y, x.y * h[e].x), fmaf(x.x, h[e].x, -x.y * h[e].y));
                        }
                    }
                } else {
#pragma unroll
                    for (int q = 0; q < E; ++q) {
                        const float2 h = __ldg(hcol + (size_t)line_index<N, 1, E>(t, 0, q) * C), x = v[q];
                        v[q] = make_float2(fmaf(x.x, h.y, x.y * h.x), fmaf(x.x, h.x, -x.y * h.y));
                    }
                }
            }
        }
        if (pair == 0) wait_other();                              // pair 1's last turn: every arrival on 3 / 4 is now matched
        // the result leaves through X as two dense half tiles [N/2][C]
        const int b = tile / GROUPS, col0 = (tile % GROUPS) * C;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            __syncthreads();                                      // X is free: exchanges done / the first half's store has read it
#pragma unroll
            for (int q = 0; q < E / 2; ++q) {
                const float2 x = half ? v[q + E / 2] : v[q];
                X[line_index<N, 1, E>(t, 0, q) * C + c] = MidSwapped<N>::value ? x : make_float2(x.y, x.x);
            }
            fence_proxy_async();
            __syncthreads();
            if (tid == 0) {
#pragma unroll
                for (int j = 0; j < CFG::BOXES / 2; ++j)
                    tma_store_2d(&tm_out, 2 * col0, b * N + half * (N / 2) + j * CFG::BOX_ROWS, X + j * CFG::BOX_ROWS * C);
                tma_store_commit();
                if (half == 0) tma_store_wait_read();
            }
        }
    }
    if (tid == 0) tma_store_wait_read();
    tmem_fence_before_sync();
    __syncthreads();
    if (tid < 32) tmem_dealloc(tmem_slot, CFG::TMEM_COLS);
}

} // namespace ssp
