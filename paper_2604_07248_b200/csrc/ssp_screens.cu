// ssp_screens.cu -- phase-screen generator and AR evolver (K1-K3).
//
//   k_sh_prep    : subharmonic coefficients c_pab (+ AR recursion) and the analytic mean of phi_lo
//   k_screen_col : K1 spectral filter / AR prologue fused into K2, the inverse FFT along y
//   k_screen_row : K3 inverse FFT along x, real part, + subharmonics - mean
// (PAPER.md:359 S16; :57 Eq.2; :63 Eq.3; :80 Eq.5; :74 Eq.4.)
#include "ssp_internal.h"
#include "ssp_lines.cuh"
#include "ssp_col_tma.cuh"
#include "ssp_philox.cuh"

// unroll factor of the seeded kernel's draw loop (16 Philox blocks per thread), measured per config-3 frame: 1: 3.61 ms,
// 2: 3.43, 4: 3.37, 8: 4.18, 16 (full, draws kept in registers and swapped by shuffle): 4.60 -- the last two miss the
// instruction cache (ncu: no_instruction 1.7 stalled warps per issue)
#ifndef SSP_SEED_UNROLL
#define SSP_SEED_UNROLL 4
#endif
#define SSP_SEED_PRAGMA_(x) _Pragma(#x)
#define SSP_SEED_PRAGMA(x) SSP_SEED_PRAGMA_(x)

namespace ssp {

// sqrt of the frequency-dependent part of Phi^f at squared frequency f2 (cycles/m)^2.
// The scalar part (0.023 r0^-5/3, or the oceanic constants) and df are in the per-slab amplitude.
template <bool OCEAN>
__device__ __forceinline__ float psd_shape_sqrt_k(const ScreenFilter &f, float f2)
{
    if constexpr (OCEAN) {
        const float kap = f.two_pi * sqrtf(f2);
        const float ke = kap * f.eta;
        const float ke23 = exp2f(0.66666667f * __log2f(ke));
        const float delta = 8.284f * ke23 * ke23 + 12.978f * ke * ke;
        const float br = f.w * f.w * __expf(-1.863e-2f * delta) + __expf(-1.9e-4f * delta)
                         - 2.f * f.w * __expf(-9.41e-3f * delta);
        return exp2f(-1.8333334f * __log2f(kap)) * sqrtf(fmaxf((1.f + 2.35f * ke23) * br, 0.f));
    }
    // von Karman / Kolmogorov / power law: exp(-f2/(2 fm^2)) (f2 + f0^2)^(-pexp), pexp = 11/12 or alpha/4
    return exp2f(fmaf(-f.pexp, __log2f(f2 + f.f0sq), -f2 * f.inv_fm2_log2e));
}
__device__ __forceinline__ float psd_shape_sqrt(const ScreenFilter &f, float f2)
{
    return (f.kind == SSP_PSD_OCEAN_NIKISHOV) ? psd_shape_sqrt_k<true>(f, f2) : psd_shape_sqrt_k<false>(f, f2);
}

// SEEDED: the fresh noise is drawn here instead of loaded (see k_screen_col_tma below); the draws pass through the
// exchange buffer, which is idle until the transform.
template <int N, bool SEEDED = false>
__global__ void __launch_bounds__(ColCfg<N, 2>::THREADS, ColCfg<N, 2>::MIN_BLOCKS) k_screen_col(const ScreenColArgs a)
{
    using PI = PlanInfo<N, 2>;
    using CFG = ColCfg<N, 2>;
    constexpr int E = PI::E, T = PI::T, C = CFG::C, R1 = PI::R1, RL = PI::RL;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);
    const int tid = threadIdx.x;
    const int c = tid % C, t = fft_logical_t<N, 2, C>(tid / C);
    constexpr int GROUPS = N / C;
    const int scr = blockIdx.x / GROUPS, kx = (blockIdx.x % GROUPS) * C + c;
    ColSmem<C> sm{smem + c};
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)

    const float amp_s = __ldg(a.amp + (a.g0 + scr) % a.S);
    const float kxs = (float)((kx < N / 2) ? kx : kx - N);
    const float df2 = a.flt.df * a.flt.df;
    const size_t base = (size_t)scr * N * N + kx;
    const bool ar = a.old_spec != nullptr;
    float2 tx = make_float2(1.f, 0.f);
    if (ar && a.taux) tx = __ldg(a.taux + kx);

    float2 v[E];
    if constexpr (SEEDED) {
        static_assert(!SEEDED || (E == R1 && C % 2 == 0 && E % 2 == 0), "one first-stage butterfly per thread, column pairs in adjacent lanes");
        const unsigned long long e0 = a.first_draw + (unsigned long long)scr * N * N + (unsigned)(kx & ~1);
        const int odd = c & 1;
SSP_SEED_PRAGMA(unroll SSP_SEED_UNROLL)
        for (int q = 0; q < E; q += 2) {
            const int ky_m = line_index<N, 2, R1>(t, 0, q + odd);     // the row whose block this lane computes
            uint32_t w[4];
            philox_block(a.keys, (e0 + (unsigned long long)ky_m * N) >> 1, a.stream_lo, a.stream_hi, w);
            const float2 z0 = box_muller(w[0], w[1]), z1 = box_muller(w[2], w[3]);
            *reinterpret_cast<float4 *>(smem + ky_m * C + (c & ~1)) = make_float4(z0.x, z0.y, z1.x, z1.y);
        }
        __syncwarp();
#pragma unroll
        for (int q = 0; q < E; ++q) v[q] = smem[line_index<N, 2, R1>(t, 0, q) * C + c];
        __syncthreads();                                          // the exchange buffer is the transform's from here on
    } else {
    // all noise loads first (independent, in flight together), then filter in registers
#pragma unroll
    for (int i = 0; i < E / R1; ++i)
#pragma unroll
        for (int q = 0; q < R1; ++q) v[i * R1 + q] = __ldg(a.noise + base + (size_t)line_index<N, 2, R1>(t, i, q) * N);
    }
#pragma unroll
    for (int i = 0; i < E / R1; ++i)
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int ky = line_index<N, 2, R1>(t, i, q);
            const float kys = (float)((ky < N / 2) ? ky : ky - N);
            const float f2 = (kxs * kxs + kys * kys) * df2;
            const float amp = (kx == 0 && ky == 0) ? 0.f : amp_s * psd_shape_sqrt(a.flt, f2);
            v[i * R1 + q] = make_float2(v[i * R1 + q].x * amp, v[i * R1 + q].y * amp);
        }
    if (ar) { // C <- a tau C_old + sqrt(1-a^2) C_fresh, old spectrum loaded in batches of 8
        constexpr int G = (E < 8) ? E : 8;
#pragma unroll
        for (int e0 = 0; e0 < E; e0 += G) {
            float2 old[G];
#pragma unroll
            for (int e = 0; e < G; ++e)
                old[e] = a.old_spec[base + (size_t)line_index<N, 2, R1>(t, (e0 + e) / R1, (e0 + e) % R1) * N];
#pragma unroll
            for (int e = 0; e < G; ++e) {
                float2 o = old[e];
                if (a.taux) o = cmul(o, cmul(tx, __ldg(a.tauy + line_index<N, 2, R1>(t, (e0 + e) / R1, (e0 + e) % R1))));
                v[e0 + e] = make_float2(fmaf(a.ar_a, o.x, a.ar_g * v[e0 + e].x), fmaf(a.ar_a, o.y, a.ar_g * v[e0 + e].y));
            }
        }
    }
    if (a.spec_out) {
#pragma unroll
        for (int i = 0; i < E / R1; ++i)
#pragma unroll
            for (int q = 0; q < R1; ++q) a.spec_out[base + (size_t)line_index<N, 2, R1>(t, i, q) * N] = v[i * R1 + q];
    }
    fft_line<N, 2, false, true>(v, t, sm, a.tw); // unnormalised inverse along y
    float2 *dst = a.out + base;
#pragma unroll
    for (int i = 0; i < E / RL; ++i)
#pragma unroll
        for (int q = 0; q < RL; ++q) dst[(size_t)line_index<N, 2, RL>(t, i, q) * N] = v[i * RL + q];
}

// K1+K2 with the tiles moved by TMA: noise (and the old spectrum) arrive as C-column boxes in two
// shared-memory buffers, the new spectrum leaves from the buffer the old one came in, the column
// transform exchanges through the noise buffer and its result leaves from there.  Same arithmetic,
// element for element, as k_screen_col; no global load or store is issued by the threads.
// SEEDED: the fresh noise is not read but drawn here (ssp_philox.cuh: the generator and Box-Muller of ssp_fill_noise,
// draw index = first_draw + element index), so one of the kernel's four 8 B/px streams -- and the 8 B/px write of the
// separate noise fill -- disappears.  A Philox block makes the draws of two adjacent columns: the two lanes that own them
// (c, c ^ 1: adjacent lanes, same rows) each compute the blocks of every other row and hand the other half over through
// the (otherwise unused) noise buffer.
template <int N, bool OCEAN, bool AR, bool TILT, bool SEEDED = false>
__global__ void __launch_bounds__(ScreenColTmaCfg<N>::THREADS, ScreenColTmaCfg<N>::MIN_BLOCKS)
k_screen_col_tma(const __grid_constant__ CUtensorMap tm_noise, const __grid_constant__ CUtensorMap tm_spec,
                 const __grid_constant__ CUtensorMap tm_out, const ScreenColArgs a)
{
    using PI = PlanInfo<N, 1>;
    using CFG = ScreenColTmaCfg<N>;
    constexpr int E = PI::E, C = CFG::C, R1 = PI::R1;
    constexpr int GROUPS = N / C;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned long long *full = reinterpret_cast<unsigned long long *>(smem_raw);
    float2 *buf_x = reinterpret_cast<float2 *>(smem_raw + CFG::HEAD);     // noise -> exchange -> result
    float2 *buf_s = buf_x + CFG::BUF_ELEMS;                               // old -> new spectrum (present iff used)
    const int tid = threadIdx.x, c = tid % C, t = fft_logical_t<N, 1, C>(tid / C);
    const int scr = blockIdx.x / GROUPS, col0 = (blockIdx.x % GROUPS) * C, kx = col0 + c;
    constexpr bool ar = AR;
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)

    if (tid == 0) {
        mbar_init(full, 1);
        fence_mbar_init();
        if constexpr (ar || !SEEDED) mbar_expect_tx(full, (ar && !SEEDED) ? 2 * CFG::TILE_BYTES : CFG::TILE_BYTES);
        if constexpr (!SEEDED) {
#pragma unroll
            for (int j = 0; j < CFG::BOXES; ++j)
                tma_load_2d(buf_x + j * CFG::BOX_ROWS * C, &tm_noise, 2 * col0, scr * N + j * CFG::BOX_ROWS, full);
        }
        if (ar) {
#pragma unroll
            for (int j = 0; j < CFG::BOXES; ++j)
                tma_load_2d(buf_s + j * CFG::BOX_ROWS * C, &tm_spec, 2 * col0, scr * N + j * CFG::BOX_ROWS, full);
        }
    }
    const float amp_s = __ldg(a.amp + (a.g0 + scr) % a.S);
    const float kxs = (float)((kx < N / 2) ? kx : kx - N);
    const float df2 = a.flt.df * a.flt.df;
    float2 tx = make_float2(1.f, 0.f);
    if constexpr (TILT) tx = __ldg(a.taux + kx);
    __syncthreads();
    float2 v[E];
    if constexpr (SEEDED) {
        // the draws of this thread's points, made before the spectrum tile is waited for (they need no memory): written
        // into the noise buffer where the TMA load of the reading kernel would have put them, one 16-byte store per
        // block (two adjacent columns); the partner lane reads its half after a __syncwarp.  The loop stays rolled: fully
        // unrolled, the 16 blocks of ten rounds pushed the kernel past the instruction cache (ncu: no_instruction 1.7 per issue)
        static_assert(!SEEDED || (E == R1 && C % 2 == 0 && E % 2 == 0), "one first-stage butterfly per thread, column pairs in adjacent lanes");
        const unsigned long long e0 = a.first_draw + (unsigned long long)scr * N * N + (unsigned)(kx & ~1);
        const int odd = c & 1;
SSP_SEED_PRAGMA(unroll SSP_SEED_UNROLL)
        for (int q = 0; q < E; q += 2) {
            const int ky_m = line_index<N, 1, R1>(t, 0, q + odd);     // the row whose block this lane computes
            uint32_t w[4];
            philox_block(a.keys, (e0 + (unsigned long long)ky_m * N) >> 1, a.stream_lo, a.stream_hi, w);
            const float2 z0 = box_muller(w[0], w[1]), z1 = box_muller(w[2], w[3]);   // columns kx & ~1 and (kx & ~1) + 1
            *reinterpret_cast<float4 *>(buf_x + ky_m * C + (c & ~1)) = make_float4(z0.x, z0.y, z1.x, z1.y);
        }
        __syncwarp();
    }
    if constexpr (ar || !SEEDED) mbar_wait(full, 0);              // (seeded first synthesis: nothing is loaded)

#pragma unroll
    for (int i = 0; i < E / R1; ++i)
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int ky = line_index<N, 1, R1>(t, i, q);
            const float2 nz = buf_x[ky * C + c];
            const float kys = (float)((ky < N / 2) ? ky : ky - N);
            const float f2 = (kxs * kxs + kys * kys) * df2;
            const float amp = (kx == 0 && ky == 0) ? 0.f : amp_s * psd_shape_sqrt_k<OCEAN>(a.flt, f2);
            float2 x = make_float2(nz.x * amp, nz.y * amp);
            if constexpr (AR) { // C <- a tau C_old + sqrt(1-a^2) C_fresh
                float2 o = buf_s[ky * C + c];
                if constexpr (TILT) o = cmul(o, cmul(tx, __ldg(a.tauy + ky)));
                x = make_float2(fmaf(a.ar_a, o.x, a.ar_g * x.x), fmaf(a.ar_a, o.y, a.ar_g * x.y));
            }
            if (a.spec_out) buf_s[ky * C + c] = x;                        // same owner as the read above
            v[i * R1 + q] = x;
        }
    fence_proxy_async();
    __syncthreads();                                                      // tiles consumed, new spectrum complete
    if (tid == 0 && a.spec_out) {
#pragma unroll
        for (int j = 0; j < CFG::BOXES; ++j)
            tma_store_2d(&tm_spec, 2 * col0, scr * N + j * CFG::BOX_ROWS, buf_s + j * CFG::BOX_ROWS * C);
        tma_store_commit();
    }
    ColSmem<C> sm{buf_x + c};
    fft_line<N, 1, false, true, true>(v, t, sm, a.tw);                    // unnormalised inverse along y
    constexpr int RL = PI::RL;
#pragma unroll
    for (int i = 0; i < E / RL; ++i)
#pragma unroll
        for (int q = 0; q < RL; ++q) buf_x[line_index<N, 1, RL>(t, i, q) * C + c] = v[i * RL + q];
    fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < CFG::BOXES; ++j)
            tma_store_2d(&tm_out, 2 * col0, scr * N + j * CFG::BOX_ROWS, buf_x + j * CFG::BOX_ROWS * C);
        tma_store_commit();
        tma_store_wait_read();
    }
}

// PAIR: also write the imaginary part of the synthesis as a second screen (a.screens_im).
template <int N, bool PAIR>
__global__ void __launch_bounds__(RowCfg<N>::THREADS, RowCfg<N>::MIN_BLOCKS + (N == 1024 ? 1 : 0)) k_screen_row(const ScreenRowArgs a)
{
    using PI = PlanInfo<N, 0>;
    using CFG = RowCfg<N>;
    constexpr int E = PI::E, T = PI::T, R1 = PI::R1, RL = PI::RL;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);
    const int tid = threadIdx.x;
    const int lib = tid / T, t = fft_logical_t<N, 0, 1>(tid % T);
    const long long line = (long long)blockIdx.x * CFG::LPB + lib;
    const int scr = (int)(line / N), iy = (int)(line % N);
    RowSmem<T, CFG::WIDE> sm{smem + (size_t)lib * CFG::LINE_ELEMS, 1 + lib};
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)

    float2 v[E];
    const float2 *src = a.in + line * N;
#pragma unroll
    for (int i = 0; i < E / R1; ++i)
#pragma unroll
        for (int q = 0; q < R1; ++q) v[i * R1 + q] = src[line_index<N, 0, R1>(t, i, q)];
    fft_line<N, 0, false, true>(v, t, sm, a.tw); // unnormalised inverse along x; strided by RL

    // phi_lo(ix,iy) = sum_p Re( d_p0 conj(ex) + d_p1 + d_p2 ex ),  d_pb = c_p0b conj(ey) + c_p1b + c_p2b ey
    //              = sum_p [ (Re d_p0 + Re d_p2) cos_p(ix) + (Im d_p0 - Im d_p2) sin_p(ix) + Re d_p1 ]:
    // two FMAs per level and pixel; the ix-independent terms and the analytic mean go into one constant.
    // The imaginary part: Im( d_p0 conj(ex) + d_p1 + d_p2 ex ) = (Im d_p0 + Im d_p2) cos_p + (Re d_p2 - Re d_p0) sin_p + Im d_p1.
    float cst = 0.f, cst_im = 0.f;
    if (a.n_sh > 0) {
        cst = -__ldg(a.sh_mean + 2 * scr);
        if constexpr (PAIR) cst_im = -__ldg(a.sh_mean + 2 * scr + 1);
        for (int p = 0; p < a.n_sh; ++p) {
            const float2 *cf = a.sh_coef + ((size_t)scr * a.n_sh + p) * 9;
            const float2 ey = __ldg(a.ex + (size_t)p * N + iy);
            float2 d[3];
#pragma unroll
            for (int bb = 0; bb < 3; ++bb) {
                const float2 c0 = __ldg(cf + bb), c1 = __ldg(cf + 3 + bb), c2 = __ldg(cf + 6 + bb);
                const float2 lo = cmul_conj(c0, ey), hi = cmul(c2, ey);
                d[bb] = make_float2(lo.x + c1.x + hi.x, lo.y + c1.y + hi.y);
            }
            const float ca = d[0].x + d[2].x, sa = d[0].y - d[2].y;
            const float ci = d[0].y + d[2].y, si = d[2].x - d[0].x;
            cst += d[1].x;
            if constexpr (PAIR) cst_im += d[1].y;
            // ca cos(al + be) + sa sin(al + be) = cos(be) (ca cos al + sa sin al) + sin(be) (sa cos al - ca sin al): al from the
            // thread's own phasor ex[p][m], be = the warp-uniform phasor e2[p][q] (constant bank): still 2 FMAs per level
            // and pixel, but no per-pixel table read
            static_assert(RL <= 32, "e2 holds 32 phasors per level");
#pragma unroll
            for (int i = 0; i < E / RL; ++i) {
                const float2 e1 = __ldg(a.ex + (size_t)p * N + t + T * i);
                const float A = fmaf(ca, e1.x, sa * e1.y), Bq = fmaf(sa, e1.x, -ca * e1.y);
                const float Ai = fmaf(ci, e1.x, si * e1.y), Bi = fmaf(si, e1.x, -ci * e1.y);
#pragma unroll
                for (int q = 0; q < RL; ++q) {
                    const float2 e = a.e2[p][q];
                    v[i * RL + q].x = fmaf(A, e.x, fmaf(Bq, e.y, v[i * RL + q].x));
                    if constexpr (PAIR) v[i * RL + q].y = fmaf(Ai, e.x, fmaf(Bi, e.y, v[i * RL + q].y));
                }
            }
        }
    }
    float *dst = a.screens + line * N;
#pragma unroll
    for (int i = 0; i < E / RL; ++i)
#pragma unroll
        for (int q = 0; q < RL; ++q) dst[line_index<N, 0, RL>(t, i, q)] = v[i * RL + q].x + cst;
    if constexpr (PAIR) {
        float *dst_im = a.screens_im + line * N;
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q) dst_im[line_index<N, 0, RL>(t, i, q)] = v[i * RL + q].y + cst_im;
    }
}

// one block per screen, one thread per (p, a, b)
__global__ void __launch_bounds__(96) k_sh_prep(int S, int n_sh, const float2 *__restrict__ noise_sh,
                                                 const float *__restrict__ amp_sh, const float2 *__restrict__ tau_sh,
                                                 float ar_a, float ar_g, const float2 *old_coef, float2 *coef_out,
                                                 const float2 *__restrict__ mfac, float *__restrict__ mean_out)
{
    __shared__ float red[96], red_im[96];
    const int scr = blockIdx.x, i = threadIdx.x, s = scr % S;
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    float contrib = 0.f, contrib_im = 0.f;
    if (i < 9 * n_sh) {
        const size_t idx = (size_t)scr * n_sh * 9 + i;
        const float amp = __ldg(amp_sh + (size_t)s * n_sh * 9 + i); // 0 at the centre
        const float2 nz = noise_sh[idx];
        float2 cv = make_float2(nz.x * amp, nz.y * amp);
        if (old_coef) {
            float2 old = old_coef[idx];
            if (tau_sh) old = cmul(old, __ldg(tau_sh + i));
            cv = make_float2(fmaf(ar_a, old.x, ar_g * cv.x), fmaf(ar_a, old.y, ar_g * cv.y));
        }
        coef_out[idx] = cv;
        const float2 m = __ldg(mfac + i);
        contrib = cv.x * m.x - cv.y * m.y;                      // Re(c M): mean of the real-part screen's phi_lo
        contrib_im = cv.x * m.y + cv.y * m.x;                   // Im(c M): of the imaginary-part screen's
    }
    red[i] = contrib;
    red_im[i] = contrib_im;
    __syncthreads();
    if (i == 0) {
        float sum = 0.f, sum_im = 0.f;
        for (int k = 0; k < 9 * n_sh; ++k) { sum += red[k]; sum_im += red_im[k]; }
        mean_out[2 * scr] = sum;
        mean_out[2 * scr + 1] = sum_im;
    }
}

// ---- launchers ------------------------------------------------------------------------
template <int N>
static int launch_screen_col_n(ssp_ctx *ctx, const ScreenColArgs &a)
{
    using CFG = ColCfg<N, 2>;
    constexpr bool CAN_SEED = (N >= 2048);                        // the seeded instance is built for the tall grids only
    const bool seeded = !a.noise;
    if (seeded && !CAN_SEED) return ctx->fail(SSP_EUNSUPPORTED, "no seeded generator for N=%d", N);
    auto kern = (seeded && CAN_SEED) ? k_screen_col<N, CAN_SEED> : k_screen_col<N, false>;
    if (CFG::SMEM > 48 * 1024)
        SSP_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CFG::SMEM));
    const double bpp = (seeded ? 8.0 : 16.0) + (a.old_spec ? 8.0 : 0.0) + (a.spec_out ? 8.0 : 0.0);
    ctx->prof_begin(seeded ? "screen_col_seeded" : "screen_col", bpp * (double)a.nscr * N * N);
    SSP_CUDA(ctx, launch_pdl(kern, dim3(a.nscr * (N / CFG::C)), dim3(CFG::THREADS), CFG::SMEM, ctx->stream, pdl_enabled(), a));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

template <int N, bool OCEAN, bool AR, bool TILT, bool SEEDED = false>
static int launch_screen_col_tma_x(ssp_ctx *ctx, const ScreenColArgs &a)
{
    using CFG = ScreenColTmaCfg<N>;
    auto kern = k_screen_col_tma<N, OCEAN, AR, TILT, SEEDED>;
    const size_t smem = CFG::smem((a.old_spec || a.spec_out) ? 2 : 1);
    const size_t rows = (size_t)a.nscr * N;
    CUtensorMap tm_noise, tm_spec, tm_out;
    // (seeded: no noise array; the descriptor is not used by the kernel)
    if (int rc = make_tmap_c64(ctx, SEEDED ? (const void *)a.out : (const void *)a.noise, N, rows, CFG::C, CFG::BOX_ROWS, &tm_noise)) return rc;
    const void *spec = a.spec_out ? (const void *)a.spec_out : (const void *)a.old_spec;
    if (int rc = make_tmap_c64(ctx, spec ? spec : (const void *)a.noise, N, rows, CFG::C, CFG::BOX_ROWS, &tm_spec)) return rc;
    if (int rc = make_tmap_c64(ctx, a.out, N, rows, CFG::C, CFG::BOX_ROWS, &tm_out)) return rc;
    SSP_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CFG::smem(2)));
    const double bpp = (SEEDED ? 8.0 : 16.0) + (a.old_spec ? 8.0 : 0.0) + (a.spec_out ? 8.0 : 0.0);
    ctx->prof_begin(SEEDED ? "screen_col_seeded" : "screen_col", bpp * (double)a.nscr * N * N);
    SSP_CUDA(ctx, launch_pdl(kern, dim3(a.nscr * (N / CFG::C)), dim3(CFG::THREADS), smem, ctx->stream, pdl_enabled(), tm_noise, tm_spec, tm_out, a));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

template <int N>
static int launch_screen_col_tma_n(ssp_ctx *ctx, const ScreenColArgs &a)
{
    const bool ocean = a.flt.kind == SSP_PSD_OCEAN_NIKISHOV, ar = a.old_spec != nullptr, tilt = ar && a.taux;
    if (!a.noise) {                                               // seeded: the fresh noise is drawn in the kernel
        if (!ar) return ocean ? launch_screen_col_tma_x<N, true, false, false, true>(ctx, a) : launch_screen_col_tma_x<N, false, false, false, true>(ctx, a);
        if (ocean) return tilt ? launch_screen_col_tma_x<N, true, true, true, true>(ctx, a) : launch_screen_col_tma_x<N, true, true, false, true>(ctx, a);
        return tilt ? launch_screen_col_tma_x<N, false, true, true, true>(ctx, a) : launch_screen_col_tma_x<N, false, true, false, true>(ctx, a);
    }
    if (ocean) {
        if (!ar) return launch_screen_col_tma_x<N, true, false, false>(ctx, a);
        return tilt ? launch_screen_col_tma_x<N, true, true, true>(ctx, a) : launch_screen_col_tma_x<N, true, true, false>(ctx, a);
    }
    if (!ar) return launch_screen_col_tma_x<N, false, false, false>(ctx, a);
    return tilt ? launch_screen_col_tma_x<N, false, true, true>(ctx, a) : launch_screen_col_tma_x<N, false, true, false>(ctx, a);
}

template <int N>
static int launch_screen_row_n(ssp_ctx *ctx, const ScreenRowArgs &a)
{
    using CFG = RowCfg<N>;
    auto kern = a.screens_im ? k_screen_row<N, true> : k_screen_row<N, false>;
    // only the exchange buffers: no screen-row staging here, and what shared memory does not take stays L1
    // (the phasor and twiddle tables are read through it)
    constexpr size_t smem = CFG::SMEM_X;
    if (smem > 48 * 1024)
        SSP_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    ctx->prof_begin("screen_row", (a.screens_im ? 16.0 : 12.0) * (double)a.nscr * N * N);
    SSP_CUDA(ctx, launch_pdl(kern, dim3((unsigned)((long long)a.nscr * N / CFG::LPB)), dim3(CFG::THREADS), smem, ctx->stream, pdl_enabled(), a));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}


// the TMA generator runs the column plan (V = 1), the register-load one its own (V = 2); they differ at N >= 2048
bool screen_col_seeded_supported(int N) { return N >= 512; }

int screen_col_plan_variant(int N) { return (N == 512 || N == 1024) ? 1 : 2; }

int launch_screen_col(ssp_ctx *ctx, int N, const ScreenColArgs &a)
{
    // the TMA kernel keeps the stored spectrum in place: an old spectrum elsewhere takes the register-load kernel
    if (!a.old_spec || !a.spec_out || a.old_spec == a.spec_out) {
        if (N == 512) return launch_screen_col_tma_n<512>(ctx, a);
        if (N == 1024) return launch_screen_col_tma_n<1024>(ctx, a);
    }
    if (!a.noise && N < 2048)
        return ctx->fail(SSP_EUNSUPPORTED, "the seeded generator is built for N >= 512 (512 / 1024: spectrum kept in place)");
    SSP_DISPATCH_N(N, (launch_screen_col_n<NN>(ctx, a)));
}
int row_last_radix(int N)
{
    switch (N) {
    case 8: return PlanInfo<8, 0>::RL;
    case 16: return PlanInfo<16, 0>::RL;
    case 32: return PlanInfo<32, 0>::RL;
    case 64: return PlanInfo<64, 0>::RL;
    case 128: return PlanInfo<128, 0>::RL;
    case 256: return PlanInfo<256, 0>::RL;
    case 512: return PlanInfo<512, 0>::RL;
    case 1024: return PlanInfo<1024, 0>::RL;
    case 2048: return PlanInfo<2048, 0>::RL;
    case 4096: return PlanInfo<4096, 0>::RL;
    default: return 1;
    }
}

int launch_screen_row(ssp_ctx *ctx, int N, const ScreenRowArgs &a)
{
    SSP_DISPATCH_N(N, (launch_screen_row_n<NN>(ctx, a)));
}

int launch_sh_prep(ssp_ctx *ctx, int nscr, int S, int n_sh, const float2 *noise_sh, const float *amp_sh,
                   const float2 *tau_sh, float ar_a, float ar_g, const float2 *old_coef, float2 *coef_out,
                   const float2 *mfac, float *mean_out)
{
    SSP_CUDA(ctx, launch_pdl(k_sh_prep, dim3(nscr), dim3(96), 0, ctx->stream, pdl_enabled(), S, n_sh, noise_sh, amp_sh, tau_sh,
                             ar_a, ar_g, old_coef, coef_out, mfac, mean_out));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

} // namespace ssp
