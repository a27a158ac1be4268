// ssp_internal.h -- context, table caches and kernel launchers shared by the .cu files.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <map>
#include <string>
#include <tuple>
#include <vector>

#include "../../include/ssp.h"

namespace ssp {

struct HKey {
    int N;
    double dx, lam_eff, dz;
    int conj;      // conj(H)
    int scaled;    // multiplied by 1/N^2
    bool operator<(const HKey &o) const
    {
        return std::tie(N, dx, lam_eff, dz, conj, scaled) <
               std::tie(o.N, o.dx, o.lam_eff, o.dz, o.conj, o.scaled);
    }
};

} // namespace ssp

struct ssp_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    long long launches = 0;
    int num_sms = 148;
    std::map<int, float2 *> twiddles;            // per (N, plan variant), device
    std::map<ssp::HKey, float2 *> htables;       // 1-D transfer-function tables, device [N]
    std::map<ssp::HKey, float2 *> h2d_tables;    // 2-D transfer functions [N][N] (angular spectrum), device
    size_t h2d_bytes = 0;
    std::map<int, float2 *> sign_tables;         // (-1)^k tables for the centred DFT
    std::map<std::tuple<int, float, float>, float *> win_maps; // window amplitude maps per (N, 1/sigma^2, order/2)
    void *scratch = nullptr;                     // small device scratch (stat accumulators, tables)
    size_t scratch_bytes = 0;
    std::vector<void *> owned;                   // misc device allocations freed at destroy
    void *encode_tiled = nullptr;                // cuTensorMapEncodeTiled, resolved through the runtime
    // TMA descriptors by (base pointer, columns, rows, box): a split step re-launches the column kernel on the same
    // buffers n_steps times, so the host-side encode runs once per buffer and shape; dropped at 256 entries
    std::map<std::tuple<const void *, size_t, size_t, int, int>, CUtensorMap> tmaps;
    // device lists of step descriptors of the on-chip path, by content: a repeated call re-uses its list without a copy
    // (so the call can be captured into a CUDA graph once it has run outside capture); dropped at 16 entries
    std::vector<std::pair<std::vector<unsigned char>, void *>> small_lists;
    // ssp_propagate_host: copy streams and events of the chunked host <-> device pipeline (created on first use)
    cudaStream_t copy_in = nullptr, copy_out = nullptr;
    std::vector<cudaEvent_t> pipe_events;

    // ---- optional per-launch timing with CUDA events on the context's stream (bench.py's roofline)
    struct ProfRec { const char *name; double bytes; int ev; };
    bool prof_on = false;
    std::vector<ProfRec> prof;
    std::vector<cudaEvent_t> prof_events;        // pool, two per record
    void prof_begin(const char *name, double alg_bytes)
    {
        if (!prof_on) return;
        const int ev = 2 * (int)prof.size();
        while ((int)prof_events.size() < ev + 2) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            prof_events.push_back(e);
        }
        prof.push_back(ProfRec{name, alg_bytes, ev});
        cudaEventRecord(prof_events[ev], stream);
    }
    void prof_end()
    {
        if (!prof_on || prof.empty()) return;
        cudaEventRecord(prof_events[prof.back().ev + 1], stream);
    }

    int fail(int code, const char *fmt, ...)
    {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        err = buf;
        return code;
    }
};

#define SSP_CUDA(ctx, call)                                                                  \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return (ctx)->fail(SSP_ECUDA, "%s failed: %s (%s:%d)", #call,                    \
                               cudaGetErrorString(e_), __FILE__, __LINE__);                  \
    } while (0)

// Run EXPR with `NN` bound to the compile-time grid size matching the run-time N_.
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

namespace ssp {

// ---- tables (ssp_tables.cu) ------------------------------------------------------
// V = 0: row-plan tables, V = 1: column-plan tables (ssp_fft.cuh)
int get_twiddles(ssp_ctx *ctx, int N, int V, const float2 **out);
int get_htable(ssp_ctx *ctx, const HKey &key, const float2 **out);
// Drops the 1-D table cache when it has grown past 4096 entries.  Called once at the entry of ssp_propagate /
// ssp_propagate_adjoint, never between the table look-ups of one call (their pointers stay valid until the launch).
int trim_htables(ssp_ctx *ctx);
// Angular-spectrum transfer function H(ky,kx)/N^2 as a complex64 map [N][N] (Eq.6, carrier removed,
// evanescent bins 0), evaluated once per (grid, lambda/n0, dz, conj) in double on the device and cached
// (8 N^2 bytes each, L2-resident at N <= 1024; the cache is dropped when it passes 1 GiB).
int get_h2d_table(ssp_ctx *ctx, const HKey &key, const float2 **out);
int get_sign_table(ssp_ctx *ctx, int N, const float2 **out);
int ensure_scratch(ssp_ctx *ctx, size_t bytes);

// ---- programmatic dependent launch (PDL) -----------------------------------------------------------------------
// The kernels of a frame follow one another on one stream, each reading what the previous one wrote.  Launched with
// programmatic stream serialization, a kernel is scheduled the moment the previous grid has finished instead of after the
// stream's full serialization step; pdl_wait() -- before the first access to anything an earlier kernel wrote and before
// the first write of anything it read -- then blocks until that grid's memory is visible.  Every kernel launched through
// launch_pdl() MUST call pdl_wait() on every path.  Measured (forward + adjoint, profiler off): 1024^2 B = 32 9.49 -> 9.36
// ms, 2048^2 3.50 -> 3.44, 256^2 B = 8 (launch-bound) 0.161 -> 0.119.  An EARLY trigger (griddepcontrol.launch_dependents
// at the top of each kernel, so that the next kernel's CTAs move in as this one's retire and run their prologue under its
// tail) measured much slower on the persistent kernels -- 1024^2 12.46 ms, 2048^2 3.81 --, a LATE one (at the start of a CTA's
// last tile) no better than none (1024^2 9.57 against 9.50 ms, 2048^2 3.87 against 3.52): no trigger is issued.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <class... KA, class... A>
static inline cudaError_t launch_pdl(void (*kern)(KA...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, A &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KA>(args)...);
}
#endif
bool pdl_enabled();            // off with SSP_NO_PDL in the environment (measurement switch)
// TMA descriptor of a row-major buffer of complex64: `cols` elements per row, `rows` rows, boxes of
// box_cols x box_rows elements (no swizzle).  Encoded on the host once per (buffer, shape, box) and cached in the context
// (the descriptor holds only the address and the geometry, so a caller who frees and re-allocates the same address with
// the same shape gets the same, still valid, descriptor).
int make_tmap_c64(ssp_ctx *ctx, const void *base, size_t cols, size_t rows, int box_cols, int box_rows,
                  CUtensorMap *out);
bool valid_N(int N);

// ---- row / column kernels (ssp_propagate.cu) ---------------------------------------
struct RowArgs {
    const float2 *in;
    float2 *out;
    int n_lines;                 // B * N
    // pointwise stage (applied in real space, between the two transforms)
    const float *phi;            // screen of this step for field 0, or null
    long long phi_batch_stride;  // elements between fields (0 = shared)
    float phase_sign;            // +1 forward, -1 adjoint
    int win_on;
    float win_qs;                // 1 / (sigma_frac N)^2
    float win_half_order;        // order / 2
    const float *win_map;        // [N][N] window amplitudes from the context cache (window_map()), or null: per pixel
    float2 *plane_out;           // optional: field after the pointwise stage, field b at + b*plane_stride
    long long plane_stride;      // elements (float2) between fields
    const float2 *plane_in;      // optional (adjoint gradient): forward plane
    float *grad;                 // optional: Im(G conj(U)), field b at + b*grad_stride
    long long grad_stride;
    // spectral post-multiply after the second transform
    const float2 *hx;            // [N] or null
    // generic pre-multiply on the input line index (centred DFT): [N] or null
    const float2 *pre;
    const float2 *pre_line;      // per-line factor pre_line[iy] multiplying the whole line, or null
    int in_swapped;              // the input holds (im, re) pairs: written by launch_col_prop when mid_swapped(N)
    const float2 *tw;
    // fused screen synthesis (k_row<.., FUSE>): column-transformed spectra [nscr][N][N] of the screen
    // generator instead of phi; the screen of field b is number scr0 + b * scr_stride
    const float2 *ycol;
    int scr0, scr_stride, n_sh;
    const float2 *sh_coef;       // [nscr][n_sh][3][3]
    const float *sh_mean;        // [nscr][2]
    const float2 *ex;            // [n_sh][N]
    // statistics epilogue of the LAST row kernel (first && !second): partial sums of the nine accumulators of
    // ssp_stats.cuh, stats_acc[field][row_stats_records(N)][ACC_N] (null: none); ROI = [roi_lo, roi_hi)^2
    double *stats_acc;
    int roi_lo, roi_hi;
};

struct ColArgs {
    const float2 *in;
    float2 *out;
    int B;
    const float2 *hy;            // [N] multiplier between / after the transforms, or null
    const float2 *h2d;           // multiplier H(ky,kx) used instead of hy (non-separable H), tile-major
                                 // [N/C][N][C] with C = col_tile_width(N), or null
    const float2 *tw;
};

// first: inverse FFT_x before the pointwise stage; second: forward FFT_x after it.
int launch_row(ssp_ctx *ctx, int N, bool first, bool second, const RowArgs &a);
// records of the nine statistics accumulators that the last row kernel writes per field (RowArgs::stats_acc)
int row_stats_records(int N);
// column pass of the propagator: FFT_y -> * hy -> IFFT_y, in place allowed.
int launch_col_prop(ssp_ctx *ctx, int N, const ColArgs &a);
// true when launch_col_prop leaves its output re/im-swapped for the row kernel that follows (RowArgs::in_swapped)
bool mid_swapped(int N);
// The window amplitudes W(ix,iy) of r's window as an fp32 [N][N] map cached in the context (built once by a kernel that
// evaluates the same expression as the row kernel: identical bits), for the grids whose common row kernel reads it
// (N = 1024); null otherwise or when it cannot be allocated -- the row kernel then evaluates W per pixel.
const float *window_map(ssp_ctx *ctx, int N, const RowArgs &r);
// single column transform (inverse != 0: unnormalised inverse) followed by * hy.
int launch_col_single(ssp_ctx *ctx, int N, bool inverse, const ColArgs &a);

// ---- on-chip path for small grids (ssp_small.cu) -----------------------------------------
struct SmallStep {               // one row pass, preceded (except op 0) by the column pass with hy
    const float *phi;            // screen of field 0 for this row pass, or null
    long long phi_batch_stride;
    float phase_sign;
    int first, second;           // inverse transform before / forward transform after the pointwise stage
    int win;                     // apply the window in this row pass
    const float2 *hx;            // multiplier after the forward transform, or null
    const float2 *hy;            // multiplier of the column pass before this row pass (op > 0)
};
struct SmallArgs {
    const float2 *in;
    float2 *out;
    ssp_stats *stats;            // optional: beam statistics of the output fields, finished inside the kernel (k_small)
    double *stats_acc;           // optional (k_cluster): one record of the nine accumulators per row, [B][N][ACC_N]
    int roi_lo, roi_hi;
    long long roi_n;
    double dx;
    int n_steps;                 // column passes; row passes = n_steps + 1
    int n_screens;               // bookkeeping (algorithmic bytes)
    const SmallStep *steps;      // device [n_steps + 1]
    int win_on;
    float win_qs, win_half_order;
    const float2 *tw_row, *tw_col;
};
bool small_path_available(int N);
int launch_small(ssp_ctx *ctx, int N, int B, const SmallArgs &a);
// the same with one field split over a cluster of 8 CTAs through distributed shared memory (ssp_cluster.cu)
bool cluster_path_available(int N, int B);
int launch_cluster(ssp_ctx *ctx, int N, int B, const SmallArgs &a);

// ---- screens (ssp_screens.cu) ------------------------------------------------------
struct ScreenFilter {
    int kind;
    float pexp;          // (f^2 + f0^2)^(-pexp): 11/12 atmospheric, alpha/4 power law
    float f0sq;          // von Karman: 1/L0^2 (0 for Kolmogorov)
    float inv_fm2_log2e; // von Karman: log2(e) / (2 fm^2)   (0 when l0 == 0)
    float df;            // 1/(N dx)
    // ocean
    float eta, w, two_pi;
};
struct NoiseSeed { unsigned long long seed, stream, first; };   // fresh noise drawn in the generator: draw index = first + element index
struct RoundKeys { uint32_t k[10][2]; };   // Philox key schedule (key + r * Weyl constants), computed once on the host
RoundKeys key_schedule(unsigned long long seed);
struct ScreenColArgs {
    const float2 *noise;      // [nscr][N][N]; null: drawn in the kernel (seeded), element e of this launch = draw first_draw + e
    RoundKeys keys;           // seeded: key schedule, stream words and the draw index of this launch's first element (even)
    uint32_t stream_lo, stream_hi;
    unsigned long long first_draw;
    const float2 *old_spec;   // AR: previous spectrum (may alias spec_out), or null
    float2 *spec_out;         // optional stored spectrum
    float2 *out;              // column-transformed intermediate [nscr][N][N]
    int nscr;
    int g0, S;                // first linear screen index (b*S+s) of this chunk, screens per stack
    const float *amp;         // per-slab amplitude factor [S] (device): sqrt of the PSD's scalar part * df
    ScreenFilter flt;
    float ar_a, ar_g;         // a, sqrt(1-a^2)
    const float2 *taux, *tauy; // AR tilt tables [N] or null
    const float2 *tw;
};
struct ScreenRowArgs {
    const float2 *in;         // [nscr][N][N]
    float *screens;           // [nscr][N][N]
    int nscr;
    int n_sh;
    const float2 *sh_coef;    // [nscr][n_sh][3][3]
    float *screens_im;        // optional [nscr][N][N]: the imaginary part of the synthesis as a second screen
    const float *sh_mean;     // [nscr][2]: analytic mean of phi_lo of the real-part and imaginary-part screens
    const float2 *ex;         // [n_sh][N] exp(i 2 pi df_p x)
    const float2 *tw;
    // exp(i 2 pi df_p q (N / RL) dx), q < RL (the row plan's last radix): pixel ix = q N/RL + m of a thread splits into
    // a per-thread phasor ex[p][m] and this warp-uniform one, read from the constant bank of the kernel arguments
    // instead of one table value per level and pixel through the LSU (the pipe this kernel saturates first)
    float2 e2[8][32];
};
int row_last_radix(int N);    // RL of the row plan at grid N
// argument checks of ssp_make_screens / ssp_evolve_screens (ssp_api_screens.cu), for callers that must validate
// before they queue anything (ssp_frame_host)
int check_screen_args(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, int B, int S, const double *cn2,
                      const double *dz, int n_sh, const void *noise, const void *noise_sh, const void *screens,
                      const void *ws, size_t ws_bytes);
// Fused screen synthesis: the AR step of ssp_evolve_screens up to and including the column pass; every
// screen's column-transformed spectrum goes to d_ycol (c64 [B][S][N][N]) and the row pass is left to the propagation's
// row kernels, which need the tables returned in `out` (they live in the caller's workspace).
struct FusedScreens {
    const float2 *ycol;
    const float2 *sh_coef;
    const float *sh_mean;
    const float2 *ex;
    int n_sh;
};
int evolve_to_ycol(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, int B, int S, const double *cn2,
                   const double *dz, int n_sh, double a, double vx, double vy, double T, const float *d_noise,
                   const float *d_noise_sh, float *d_spectrum, float *d_sh_coef, float *d_ycol, void *d_ws, size_t ws_bytes,
                   FusedScreens *out);
int launch_screen_col(ssp_ctx *ctx, int N, const ScreenColArgs &a);
bool screen_col_seeded_supported(int N);   // grids whose generator can draw the fresh noise itself (ScreenColArgs::noise == null)
int screen_col_plan_variant(int N);   // plan variant (ssp_fft.cuh) whose twiddles launch_screen_col expects in a.tw
int launch_screen_row(ssp_ctx *ctx, int N, const ScreenRowArgs &a);
// subharmonic coefficient update + analytic mean, one block per screen
int launch_sh_prep(ssp_ctx *ctx, int nscr, int S, int n_sh, const float2 *noise_sh,
                   const float *amp_sh /*[S][n_sh][9]*/, const float2 *tau_sh /*[n_sh][9] or null*/,
                   float ar_a, float ar_g, const float2 *old_coef, float2 *coef_out,
                   const float2 *mfac /*[n_sh][9] Mx*My*/, float *mean_out);

// ---- misc (ssp_misc.cu) ------------------------------------------------------------
int launch_stats(ssp_ctx *ctx, int N, double dx, int B, const float2 *field, double roi_frac,
                 ssp_stats *d_stats);
// ROI bounds of the statistics: [lo, hi)^2 with h = floor(roi_frac N / 2) pixels each side of N/2 (h = 0: the pixel N/2)
void stats_roi(int N, double roi_frac, int *lo, int *hi, long long *roi_n);
// per-field finaliser over bpf per-CTA partial records acc[b][k][ACC_N] (ssp_stats.cuh)
int launch_stats_final(ssp_ctx *ctx, int B, int bpf, double dx, long long roi_n, const double *acc, ssp_stats *d_stats);
int launch_welford(ssp_ctx *ctx, int N, int B, const float2 *field, float *mean, float *M2,
                   long long count0);
int launch_h2d_table(ssp_ctx *ctx, int N, int C, double dx, double lam_eff, double dz, int conj, float2 *out);
int col_tile_width(int N);     // columns per tile of the kernel launch_col_prop picks for N (layout of the H map)
int launch_adam(ssp_ctx *ctx, long long n, int B, const float *grad, float lr, float b1, float b2, float eps,
                float c1, float c2, float o1, float o2, float *m, float *v, float *theta);
int launch_aperture(ssp_ctx *ctx, int N, int B, long long r2max_px, const float2 *in, float2 *out);
int launch_phase_mul(ssp_ctx *ctx, int N, int B, const float *theta, float sign,
                     const float2 *in, float2 *out);
int launch_phase_grad(ssp_ctx *ctx, long long n, const float2 *g, const float2 *u, float *grad);
int launch_inner(ssp_ctx *ctx, int N, int B, const float2 *a, const float2 *b, double *out);
int launch_mae(ssp_ctx *ctx, int N, int B, const float2 *v, const float2 *t, double *loss, float2 *g);
int launch_lincomb(ssp_ctx *ctx, int N, int B, const float2 *coef /*dev [B][2] float2*/,
                   const float2 *a, const float2 *b, float2 *out);

} // namespace ssp
