// ssp_propagate.cu -- row and column kernels of the fused split step (K4-K7).
//
//   k_row<N,FIRST,SECOND>:  [IFFT_x] -> * exp(+-i phi) W [-> save plane / phase gradient]
//                           -> [FFT_x -> * hx(next step)]                  (Eq.1)
//   k_col<N,0>:             FFT_y -> * hy/N^2 -> IFFT_y   on a tile of C columns
//   k_col<N,1|2>:           single forward / unnormalised inverse column transform
//
// One split step = one k_col + one k_row launch = two HBM round trips of the field plus one
// fp32 read of the screen: 36 B/px.  H is separable for the Fresnel
// kernel, H = hx[kx] hy[ky], both 1-D tables built in double on the host.
#include "ssp_internal.h"
#include "ssp_lines.cuh"

namespace ssp {

template <int N, bool FIRST, bool SECOND>
__global__ void __launch_bounds__(RowCfg<N>::THREADS, RowCfg<N>::MIN_BLOCKS) k_row(const RowArgs a)
{
    using PI = PlanInfo<N, 0>;
    using CFG = RowCfg<N>;
    constexpr int E = PI::E, T = PI::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);

    const int tid = threadIdx.x;
    const int lib = tid / T, t = tid % T;
    const long long line = (long long)blockIdx.x * CFG::LPB + lib;
    const int b = (int)(line / N), iy = (int)(line % N);
    RowSmem<T> sm{smem + (size_t)lib * PI::LINE_ELEMS, 1 + lib};

    // the screen row is streamed from HBM: fetch it asynchronously now, use it after the first transform
    float *phis = reinterpret_cast<float *>(smem_raw + CFG::SMEM_X) + (size_t)lib * N;
    if (a.phi) {
        const float *g = a.phi + b * a.phi_batch_stride + (long long)iy * N;
#pragma unroll
        for (int i = 0; i < E / 4; ++i) cp_async16(phis + 4 * (t + T * i), g + 4 * (t + T * i));
        cp_async_commit();
    }

    float2 v[E];
    constexpr int RIN = FIRST ? PI::R1 : PI::RL;
    {
        const float2 *src = a.in + line * N;
#pragma unroll
        for (int i = 0; i < E / RIN; ++i)
#pragma unroll
            for (int q = 0; q < RIN; ++q) v[i * RIN + q] = src[line_index<N, 0, RIN>(t, i, q)];
    }
    if (a.pre) {
        const float2 pl = a.pre_line ? __ldg(a.pre_line + iy) : make_float2(1.f, 0.f);
#pragma unroll
        for (int i = 0; i < E / RIN; ++i)
#pragma unroll
            for (int q = 0; q < RIN; ++q)
                v[i * RIN + q] = cmul(v[i * RIN + q], cmul(pl, __ldg(a.pre + line_index<N, 0, RIN>(t, i, q))));
    }

    if constexpr (FIRST) fft_line<N, 0, false, true>(v, t, sm, a.tw); // inverse; now strided by RL

    // ---- pointwise stage in real space, layout strided by RL
    constexpr int RL = PI::RL;
    const bool pointwise = a.phi || a.win_on || a.grad || a.plane_out;
    if (pointwise) {
        if (a.phi) {
            cp_async_wait_all();
            sm.sync();
        }
        const long long pix0 = (long long)iy * N;
        const float yc = (float)(iy - N / 2);
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q) {
                const int ix = line_index<N, 0, RL>(t, i, q);
                float2 u = v[i * RL + q];
                if (a.grad) {
                    const float2 U = a.plane_in[b * a.plane_stride + pix0 + ix];
                    a.grad[b * a.grad_stride + pix0 + ix] = u.y * U.x - u.x * U.y; // Im(G conj(U))
                }
                float mr = 1.f, mi = 0.f;
                if (a.phi) {
                    sincos_reduced(phis[ix], &mi, &mr);
                    mi *= a.phase_sign;
                }
                if (a.win_on) {
                    const float xc = (float)(ix - N / 2);
                    const float amp = window_amp((xc * xc + yc * yc) * a.win_qs, a.win_half_order);
                    mr *= amp;
                    mi *= amp;
                }
                u = cmul(u, make_float2(mr, mi));
                if (a.plane_out) a.plane_out[b * a.plane_stride + pix0 + ix] = u;
                v[i * RL + q] = u;
            }
    }

    constexpr int ROUT = SECOND ? PI::R1 : PI::RL;
    if constexpr (SECOND) {
        if constexpr (FIRST) sm.sync();                  // the exchange buffer is reused
        fft_line<N, 0, true, false>(v, t, sm, a.tw);        // forward, reversed plan; strided by R1
    }
    float2 *dst = a.out + line * N;
    if (a.hx) {
#pragma unroll
        for (int i = 0; i < E / ROUT; ++i)
#pragma unroll
            for (int q = 0; q < ROUT; ++q) {
                const int k = line_index<N, 0, ROUT>(t, i, q);
                dst[k] = cmul(v[i * ROUT + q], __ldg(a.hx + k));
            }
    } else {
#pragma unroll
        for (int i = 0; i < E / ROUT; ++i)
#pragma unroll
            for (int q = 0; q < ROUT; ++q) dst[line_index<N, 0, ROUT>(t, i, q)] = v[i * ROUT + q];
    }
}

// MODE 0: FFT_y -> * hy -> IFFT_y.  MODE 1: FFT_y -> * hy.  MODE 2: unnormalised IFFT_y -> * hy.
template <int N, int MODE>
__global__ void __launch_bounds__(ColCfg<N>::THREADS, ColCfg<N>::MIN_BLOCKS) k_col(const ColArgs a)
{
    using PI = PlanInfo<N, 1>;
    using CFG = ColCfg<N>;
    constexpr int E = PI::E, T = PI::T, C = CFG::C;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);

    const int tid = threadIdx.x;
    const int c = tid % C, t = tid / C;
    constexpr int GROUPS = N / C;
    const int b = blockIdx.x / GROUPS, col = (blockIdx.x % GROUPS) * C + c;
    ColSmem<C> sm{smem + c};

    float2 v[E];
    constexpr int R1 = PI::R1, RL = PI::RL;
    const float2 *src = a.in + (size_t)b * N * N + col;
#pragma unroll
    for (int i = 0; i < E / R1; ++i)
#pragma unroll
        for (int q = 0; q < R1; ++q) v[i * R1 + q] = src[(size_t)line_index<N, 1, R1>(t, i, q) * N];

    fft_line<N, 1, false, MODE == 2>(v, t, sm, a.tw); // strided by RL
    if (a.hy) {
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q)
                v[i * RL + q] = cmul(v[i * RL + q], __ldg(a.hy + line_index<N, 1, RL>(t, i, q)));
    }
    float2 *dst = a.out + (size_t)b * N * N + col;
    if constexpr (MODE == 0) {
        sm.sync();
        fft_line<N, 1, true, true>(v, t, sm, a.tw);   // inverse, reversed plan; strided by R1
#pragma unroll
        for (int i = 0; i < E / R1; ++i)
#pragma unroll
            for (int q = 0; q < R1; ++q) dst[(size_t)line_index<N, 1, R1>(t, i, q) * N] = v[i * R1 + q];
    } else {
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q) dst[(size_t)line_index<N, 1, RL>(t, i, q) * N] = v[i * RL + q];
    }
}

// ---- launchers ------------------------------------------------------------------------
template <class K>
static int set_smem(ssp_ctx *ctx, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024)
        SSP_CUDA(ctx, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return SSP_OK;
}

template <int N, bool FIRST, bool SECOND>
static int launch_row_n(ssp_ctx *ctx, const RowArgs &a)
{
    using CFG = RowCfg<N>;
    if (a.n_lines % CFG::LPB) return ctx->fail(SSP_EINVAL, "row launch: %d lines not a multiple of %d", a.n_lines, CFG::LPB);
    auto kern = k_row<N, FIRST, SECOND>;
    if (int rc = set_smem(ctx, kern, CFG::SMEM)) return rc;
    // algorithmic bytes: field in + out, + the screen, + saved / read planes and the gradient
    const double bpp = 16.0 + (a.phi ? 4.0 : 0.0) + (a.plane_out ? 8.0 : 0.0) + (a.grad ? 12.0 : 0.0);
    ctx->prof_begin(FIRST ? (SECOND ? "row_ifft_pw_fft" : "row_ifft_pw") : "row_pw_fft", bpp * (double)a.n_lines * N);
    kern<<<a.n_lines / CFG::LPB, CFG::THREADS, CFG::SMEM, ctx->stream>>>(a);
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

template <int N>
static int launch_row_sel(ssp_ctx *ctx, bool first, bool second, const RowArgs &a)
{
    if (first && second) return launch_row_n<N, true, true>(ctx, a);
    if (first) return launch_row_n<N, true, false>(ctx, a);
    if (second) return launch_row_n<N, false, true>(ctx, a);
    return ctx->fail(SSP_EINVAL, "row launch with no transform");
}

template <int N, int MODE>
static int launch_col_n(ssp_ctx *ctx, const ColArgs &a)
{
    using CFG = ColCfg<N>;
    auto kern = k_col<N, MODE>;
    if (int rc = set_smem(ctx, kern, CFG::SMEM)) return rc;
    ctx->prof_begin(MODE == 0 ? "col_fft_h_ifft" : "col_single", 16.0 * (double)a.B * N * N);
    kern<<<a.B * (N / CFG::C), CFG::THREADS, CFG::SMEM, ctx->stream>>>(a);
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

#define SSP_DISPATCH_N(N_, EXPR)                                   \
    switch (N_) {                                                  \
    case 8: { constexpr int NN = 8; return EXPR; }                 \
    case 16: { constexpr int NN = 16; return EXPR; }               \
    case 32: { constexpr int NN = 32; return EXPR; }               \
    case 64: { constexpr int NN = 64; return EXPR; }               \
    case 128: { constexpr int NN = 128; return EXPR; }             \
    case 256: { constexpr int NN = 256; return EXPR; }             \
    case 512: { constexpr int NN = 512; return EXPR; }             \
    case 1024: { constexpr int NN = 1024; return EXPR; }           \
    case 2048: { constexpr int NN = 2048; return EXPR; }           \
    case 4096: { constexpr int NN = 4096; return EXPR; }           \
    default: return ctx->fail(SSP_EINVAL, "unsupported N=%d", N_); \
    }

int launch_row(ssp_ctx *ctx, int N, bool first, bool second, const RowArgs &a)
{
    SSP_DISPATCH_N(N, (launch_row_sel<NN>(ctx, first, second, a)));
}

int launch_col_prop(ssp_ctx *ctx, int N, const ColArgs &a)
{
    SSP_DISPATCH_N(N, (launch_col_n<NN, 0>(ctx, a)));
}

int launch_col_single(ssp_ctx *ctx, int N, bool inverse, const ColArgs &a)
{
    if (inverse) { SSP_DISPATCH_N(N, (launch_col_n<NN, 2>(ctx, a))); }
    SSP_DISPATCH_N(N, (launch_col_n<NN, 1>(ctx, a)));
}

} // namespace ssp
