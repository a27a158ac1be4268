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
#include "ssp_kernels.cuh"
#include "ssp_col_tma.cuh"

namespace ssp {

// ---- launchers ------------------------------------------------------------------------
template <class K>
static int set_smem(ssp_ctx *ctx, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024)
        SSP_CUDA(ctx, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return SSP_OK;
}

template <int N, bool FIRST, bool SECOND, bool GENERIC, bool FUSE = false>
static int launch_row_x(ssp_ctx *ctx, const RowArgs &a)
{
    using CFG = RowCfg<N>;
    if (a.n_lines % CFG::LPB) return ctx->fail(SSP_EINVAL, "row launch: %d lines not a multiple of %d", a.n_lines, CFG::LPB);
    auto kern = k_row<N, FIRST, SECOND, GENERIC, FUSE>;
    if (int rc = set_smem(ctx, kern, CFG::SMEM + 16)) return rc;
    // algorithmic bytes: field in + out, + the screen, + saved / read planes and the gradient
    const double bpp = 16.0 + (a.phi ? 4.0 : 0.0) + (FUSE ? 8.0 : 0.0) + (a.plane_out ? 8.0 : 0.0) + (a.grad ? 12.0 : 0.0);
    ctx->prof_begin(FUSE ? (SECOND ? "row_fused_screen_fft" : "row_fused_screen")
                         : (FIRST ? (SECOND ? "row_ifft_pw_fft" : "row_ifft_pw") : "row_pw_fft"), bpp * (double)a.n_lines * N);
    constexpr bool TM = CFG::TMEM && FIRST && SECOND && !GENERIC;           // persistent form (ssp_kernels.cuh)
    int grid = a.n_lines / CFG::LPB;
    if (TM) {
        const int resident = ctx->num_sms * CFG::MIN_BLOCKS;
        if (grid > resident) grid = resident;
    }
    SSP_CUDA(ctx, launch_pdl(kern, dim3(grid), dim3(CFG::THREADS), CFG::SMEM + (TM ? 16 : 0), ctx->stream, pdl_enabled(), a));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

// the common split step (screen and window present, nothing saved, no pre-multiply) has its own
// instantiation without run-time flag tests; everything else takes the generic one
template <int N, bool FIRST, bool SECOND>
static int launch_row_n(ssp_ctx *ctx, const RowArgs &a)
{
    constexpr bool MID = FIRST && MidSwapped<N>::value;
    if (a.in_swapped && !MID) return ctx->fail(SSP_EINVAL, "swapped row input for a kernel that does not take it");
    if (a.in_swapped && a.pre) return ctx->fail(SSP_EINVAL, "pre-multiply on a swapped row input");
    if (a.stats_acc && !(FIRST && !SECOND)) return ctx->fail(SSP_EINVAL, "statistics epilogue on a row kernel that is not the last");
    if (a.ycol) {                                                 // fused screen synthesis: the common 1024^2 kernels only
        if constexpr (N == 1024 && FIRST) {
            const bool ok = !a.phi && a.win_on && !a.grad && !a.plane_out && !a.pre && a.in_swapped &&
                            ((a.win_map != nullptr) == WinMap<N>::value);
            if (!ok) return ctx->fail(SSP_EUNSUPPORTED, "fused screen synthesis needs the common split step (window on, Fresnel H, nothing saved)");
            return launch_row_x<N, FIRST, SECOND, false, true>(ctx, a);
        } else return ctx->fail(SSP_EUNSUPPORTED, "fused screen synthesis is built for N = 1024");
    }
    const bool common = a.phi && a.win_on && !a.grad && !a.plane_out && !a.pre && (!MID || a.in_swapped) &&
                        ((a.win_map != nullptr) == WinMap<N>::value);
    if (common) return launch_row_x<N, FIRST, SECOND, false>(ctx, a);
    return launch_row_x<N, FIRST, SECOND, true>(ctx, a);
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
    SSP_CUDA(ctx, launch_pdl(kern, dim3(a.B * (N / CFG::C)), dim3(CFG::THREADS), CFG::SMEM, ctx->stream, pdl_enabled(), a));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}


int row_stats_records(int N)
{
    switch (N) {
    case 8: return StatsGroup<8>::RECORDS_PER_FIELD;
    case 16: return StatsGroup<16>::RECORDS_PER_FIELD;
    case 32: return StatsGroup<32>::RECORDS_PER_FIELD;
    case 64: return StatsGroup<64>::RECORDS_PER_FIELD;
    case 128: return StatsGroup<128>::RECORDS_PER_FIELD;
    case 256: return StatsGroup<256>::RECORDS_PER_FIELD;
    case 512: return StatsGroup<512>::RECORDS_PER_FIELD;
    case 1024: return StatsGroup<1024>::RECORDS_PER_FIELD;
    case 2048: return StatsGroup<2048>::RECORDS_PER_FIELD;
    case 4096: return StatsGroup<4096>::RECORDS_PER_FIELD;
    default: return 1;
    }
}

int launch_row(ssp_ctx *ctx, int N, bool first, bool second, const RowArgs &a)
{
    SSP_DISPATCH_N(N, (launch_row_sel<NN>(ctx, first, second, a)));
}

// TMA-fed persistent column kernel (ssp_col_tma.cuh)
template <int N, bool H2D>
static int launch_col_tma_x(ssp_ctx *ctx, const ColArgs &a)
{
    using CFG = ColTmaCfg<N>;
    auto kern = k_col_tma<N, H2D>;
    CUtensorMap tm_in, tm_out;
    if (int rc = make_tmap_c64(ctx, a.in, N, (size_t)a.B * N, CFG::C, CFG::BOX_ROWS, &tm_in)) return rc;
    if (int rc = make_tmap_c64(ctx, a.out, N, (size_t)a.B * N, CFG::C, CFG::BOX_ROWS, &tm_out)) return rc;
    if (int rc = set_smem(ctx, kern, CFG::SMEM)) return rc;
    const int ntiles = a.B * (N / CFG::C);
    const int resident = ctx->num_sms * CFG::MIN_BLOCKS;
    // two buffers: persistent CTAs walk the tiles; one buffer: one tile per CTA
    const int grid = (CFG::PERSIST && ntiles > resident) ? resident : ntiles;
    ColTmaArgs ta{a.hy, a.h2d, a.tw, ntiles};
    ctx->prof_begin("col_fft_h_ifft", 16.0 * (double)a.B * N * N);
    SSP_CUDA(ctx, launch_pdl(kern, dim3(grid), dim3(CFG::THREADS), CFG::SMEM, ctx->stream, pdl_enabled(), tm_in, tm_out, ta));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

// wide tiles, one persistent CTA per SM (ssp_col_tma.cuh: k_col_tma_wide)
template <int N, bool H2D>
static int launch_col_wide_x(ssp_ctx *ctx, const ColArgs &a)
{
    using CFG = ColWideCfg<N>;
    auto kern = k_col_tma_wide<N, H2D>;
    CUtensorMap tm_in, tm_out;
    if (int rc = make_tmap_c64(ctx, a.in, N, (size_t)a.B * N, CFG::C, CFG::BOX_ROWS, &tm_in)) return rc;
    if (int rc = make_tmap_c64(ctx, a.out, N, (size_t)a.B * N, CFG::C, CFG::BOX_ROWS, &tm_out)) return rc;
    if (int rc = set_smem(ctx, kern, CFG::SMEM)) return rc;
    const int ntiles = a.B * (N / CFG::C);
    const int grid = ntiles > ctx->num_sms ? ctx->num_sms : ntiles;
    ColTmaArgs ta{a.hy, a.h2d, a.tw, ntiles};
    ctx->prof_begin("col_fft_h_ifft", 16.0 * (double)a.B * N * N);
    SSP_CUDA(ctx, launch_pdl(kern, dim3(grid), dim3(CFG::THREADS), CFG::SMEM, ctx->stream, pdl_enabled(), tm_in, tm_out, ta));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

template <int N>
static int launch_col_tma_n(ssp_ctx *ctx, const ColArgs &a)
{
    if constexpr (ColWideCfg<N>::ENABLED) return a.h2d ? launch_col_wide_x<N, true>(ctx, a) : launch_col_wide_x<N, false>(ctx, a);
    else return a.h2d ? launch_col_tma_x<N, true>(ctx, a) : launch_col_tma_x<N, false>(ctx, a);
}

template <int N>
static constexpr int col_tile_width_n()
{
    return ColWideCfg<N>::ENABLED ? ColWideCfg<N>::C : (ColTmaTune<N>::ENABLED ? ColTmaCfg<N>::C : ColCfg<N>::C);
}

int col_tile_width(int N)
{
    switch (N) {
    case 8: return col_tile_width_n<8>();
    case 16: return col_tile_width_n<16>();
    case 32: return col_tile_width_n<32>();
    case 64: return col_tile_width_n<64>();
    case 128: return col_tile_width_n<128>();
    case 256: return col_tile_width_n<256>();
    case 512: return col_tile_width_n<512>();
    case 1024: return col_tile_width_n<1024>();
    case 2048: return col_tile_width_n<2048>();
    case 4096: return col_tile_width_n<4096>();
    default: return 1;
    }
}

// ---- cached window map (RowArgs::win_map) ------------------------------------------------------
__global__ void __launch_bounds__(256) k_window_map(int N, float qs, float half_order, float *__restrict__ out)
{
    const int iy = blockIdx.x;
    const float yc = (float)(iy - N / 2);
    const float y2 = yc * yc * qs;                                // the expressions of row_pointwise, term for term
    for (int ix = threadIdx.x; ix < N; ix += blockDim.x) {
        const float xc = (float)(ix - N / 2);
        out[(size_t)iy * N + ix] = window_amp(fmaf(xc * xc, qs, y2), half_order);
    }
}

template <int N>
static constexpr bool win_map_n() { return WinMap<N>::value; }

const float *window_map(ssp_ctx *ctx, int N, const RowArgs &r)
{
    bool use = false;
    switch (N) {
    case 1024: use = win_map_n<1024>(); break;
    default: break;
    }
    if (!use || !r.win_on) return nullptr;
    const auto key = std::make_tuple(N, r.win_qs, r.win_half_order);
    auto it = ctx->win_maps.find(key);
    if (it != ctx->win_maps.end()) return it->second;
    if (ctx->win_maps.size() >= 8) return nullptr;                // a caller cycling through windows: evaluate per pixel
    float *d = nullptr;
    if (cudaMalloc(&d, sizeof(float) * (size_t)N * N) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    k_window_map<<<N, 256, 0, ctx->stream>>>(N, r.win_qs, r.win_half_order, d);
    ctx->launches++;
    if (cudaGetLastError() != cudaSuccess) { cudaFree(d); return nullptr; }
    ctx->owned.push_back(d);
    ctx->win_maps[key] = d;
    return d;
}

template <int N>
static constexpr bool mid_swapped_n() { return ColTmaTune<N>::ENABLED && MidSwapped<N>::value; }
static_assert(!MidSwapped<8>::value && !MidSwapped<16>::value && !MidSwapped<32>::value && !MidSwapped<64>::value &&
              !MidSwapped<128>::value && !MidSwapped<256>::value && !MidSwapped<512>::value,
              "only the TMA column kernel hands the field over swapped");
static_assert(ColTmaTune<1024>::ENABLED && ColTmaTune<2048>::ENABLED && ColTmaTune<4096>::ENABLED, "see MidSwapped");

bool mid_swapped(int N)
{
    switch (N) {
    case 1024: return mid_swapped_n<1024>();
    case 2048: return mid_swapped_n<2048>();
    case 4096: return mid_swapped_n<4096>();
    default: return false;
    }
}

int launch_col_prop(ssp_ctx *ctx, int N, const ColArgs &a)
{
    if (!(a.hy || a.h2d) && mid_swapped(N)) return ctx->fail(SSP_EINVAL, "column pass without a multiplier");
    if (a.hy || a.h2d) {
        if (N == 512) return launch_col_tma_n<512>(ctx, a);
        if (N == 1024) return launch_col_tma_n<1024>(ctx, a);
        if (N == 2048) return launch_col_tma_n<2048>(ctx, a);
        if (N == 4096) return launch_col_tma_n<4096>(ctx, a);
    }
    SSP_DISPATCH_N(N, (launch_col_n<NN, 0>(ctx, a)));
}

int launch_col_single(ssp_ctx *ctx, int N, bool inverse, const ColArgs &a)
{
    if (inverse) { SSP_DISPATCH_N(N, (launch_col_n<NN, 2>(ctx, a))); }
    SSP_DISPATCH_N(N, (launch_col_n<NN, 1>(ctx, a)));
}

} // namespace ssp
