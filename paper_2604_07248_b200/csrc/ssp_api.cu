// ssp_api.cu -- the extern "C" entry points declared in include/ssp.h (context, propagation,
// adjoint, statistics).  Argument checking and launch sequencing only: every step of the path
// runs in the kernels of ssp_propagate.cu / ssp_misc.cu.
#include <cmath>
#include <cstring>
#include <string>

#include "ssp_internal.h"

using namespace ssp;

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

extern "C" {

const char *ssp_version(void) { return "ssp 0.1 sm_100a"; }

int ssp_create(ssp_ctx **out, int device, void *cuda_stream)
{
    if (!out) return SSP_EINVAL;
    *out = nullptr;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0 || device < 0 || device >= n) return SSP_ECUDA;
    if (cudaSetDevice(device) != cudaSuccess) return SSP_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return SSP_ECUDA;
    if (prop.major != 10) return SSP_EUNSUPPORTED; // sm_100a cubins only
    ssp_ctx *ctx = new ssp_ctx();
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->num_sms = prop.multiProcessorCount;
    *out = ctx;
    return SSP_OK;
}

int ssp_destroy(ssp_ctx *ctx)
{
    if (!ctx) return SSP_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto &kv : ctx->twiddles) cudaFree(kv.second);
    for (auto &kv : ctx->htables) cudaFree(kv.second);
    for (auto &kv : ctx->h2d_tables) cudaFree(kv.second);
    for (auto &kv : ctx->sign_tables) cudaFree(kv.second);
    for (void *p : ctx->owned) cudaFree(p);
    for (cudaEvent_t e : ctx->prof_events) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->pipe_events) cudaEventDestroy(e);
    if (ctx->copy_in) cudaStreamDestroy(ctx->copy_in);
    if (ctx->copy_out) cudaStreamDestroy(ctx->copy_out);
    if (ctx->scratch) cudaFree(ctx->scratch);
    for (auto &e : ctx->small_lists) cudaFree(e.second);
    delete ctx;
    return SSP_OK;
}

const char *ssp_last_error(const ssp_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int ssp_profile_enable(ssp_ctx *ctx, int on)
{
    if (!ctx) return SSP_EINVAL;
    ctx->prof_on = (on != 0);
    ctx->prof.clear();
    return SSP_OK;
}

int ssp_profile_report(ssp_ctx *ctx, char *buf, size_t buf_bytes)
{
    if (!ctx || !buf || buf_bytes < 2) return SSP_EINVAL;
    SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    struct Agg { long long n = 0; double ms = 0, bytes = 0; };
    std::map<std::string, Agg> agg;
    for (const auto &r : ctx->prof) {
        float ms = 0.f;
        SSP_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->prof_events[r.ev], ctx->prof_events[r.ev + 1]));
        Agg &a = agg[r.name];
        a.n++; a.ms += ms; a.bytes += r.bytes;
    }
    ctx->prof.clear();
    size_t o = 0;
    buf[0] = 0;
    for (const auto &kv : agg) {
        int w = snprintf(buf + o, buf_bytes - o, "%s %lld %.6f %.0f\n", kv.first.c_str(), kv.second.n, kv.second.ms,
                         kv.second.bytes);
        if (w < 0 || (size_t)w >= buf_bytes - o) return ctx->fail(SSP_EINVAL, "profile report buffer too small");
        o += (size_t)w;
    }
    return SSP_OK;
}
long long ssp_launch_count(const ssp_ctx *ctx) { return ctx ? ctx->launches : 0; }

} // extern "C"

namespace {

struct PropGeom {
    int N, B, n_steps, S;
    double dx, lam_eff;
    const double *dz;
};

int check_prop(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind, int B, int n_steps,
               const double *dz, const float *d_screens, int S, const void *in, const void *out)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N)) return ctx->fail(SSP_EINVAL, "N=%d is not a power of two in [8, 4096]", grid.N);
    if (!(grid.dx > 0) || !(lambda > 0) || !(n0 > 0)) return ctx->fail(SSP_EINVAL, "dx, lambda and n0 must be > 0");
    if (h_kind != SSP_H_FRESNEL && h_kind != SSP_H_ANGULAR_SPECTRUM) return ctx->fail(SSP_EINVAL, "unknown h_kind %d", h_kind);
    if (B < 1 || n_steps < 1 || !dz) return ctx->fail(SSP_EINVAL, "B >= 1, n_steps >= 1 and dz are required");
    if (S < 0 || S > n_steps) return ctx->fail(SSP_EINVAL, "need 0 <= S <= n_steps (S=%d, n_steps=%d)", S, n_steps);
    if (S > 0 && !d_screens) return ctx->fail(SSP_EINVAL, "d_screens is null with S=%d", S);
    for (int j = 0; j < n_steps; ++j)
        if (!(dz[j] > 0)) return ctx->fail(SSP_EINVAL, "dz[%d] must be > 0", j);
    if (!in || !out) return ctx->fail(SSP_EINVAL, "field pointers are required");
    if (!aligned16(in) || !aligned16(out) || !aligned16(d_screens))
        return ctx->fail(SSP_EINVAL, "device pointers must be 16-byte aligned");
    return SSP_OK;
}

void fill_window(RowArgs &r, ssp_window win, int N)
{
    r.win_on = (win.order > 0 && win.sigma_frac > 0) ? 1 : 0;
    if (r.win_on) {
        const double s = win.sigma_frac * N;
        r.win_qs = (float)(1.0 / (s * s));
        r.win_half_order = (float)(0.5 * win.order);
    }
}

// On-chip path (ssp_small.cu): upload the step list and launch one kernel for the whole stack.
const size_t kSmallStepBytes = 16384;

struct SmallStats { ssp_stats *stats; int lo, hi; long long n; double dx; };

int run_small(ssp_ctx *ctx, int N, int B, const std::vector<SmallStep> &steps, int n_screens, const RowArgs &win,
              const float2 *in, float2 *out, const float2 *tw, const float2 *twc, const SmallStats *st = nullptr)
{
    const size_t nbytes = sizeof(SmallStep) * steps.size();
    if (nbytes > kSmallStepBytes) return ctx->fail(SSP_EINVAL, "too many steps for the on-chip path");
    void *d_steps = nullptr;
    for (auto &e : ctx->small_lists)
        if (e.first.size() == nbytes && memcmp(e.first.data(), steps.data(), nbytes) == 0) { d_steps = e.second; break; }
    if (!d_steps) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        SSP_CUDA(ctx, cudaStreamIsCapturing(ctx->stream, &cs));
        if (cs != cudaStreamCaptureStatusNone)
            return ctx->fail(SSP_EUNSUPPORTED, "stream capture: run this call once outside capture first (its step list is uploaded then)");
        if (ctx->small_lists.size() >= 16) {                      // kernels in flight may still read the old lists
            SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            for (auto &e : ctx->small_lists) cudaFree(e.second);
            ctx->small_lists.clear();
        }
        SSP_CUDA(ctx, cudaMalloc(&d_steps, nbytes));
        // pageable source: staged before cudaMemcpyAsync returns, so the vector may die afterwards
        const cudaError_t ce = cudaMemcpyAsync(d_steps, steps.data(), nbytes, cudaMemcpyHostToDevice, ctx->stream);
        if (ce != cudaSuccess) { cudaFree(d_steps); SSP_CUDA(ctx, ce); }
        const unsigned char *pb = reinterpret_cast<const unsigned char *>(steps.data());
        ctx->small_lists.emplace_back(std::vector<unsigned char>(pb, pb + nbytes), d_steps);
    }
    SmallArgs a{};
    a.in = in; a.out = out;
    a.n_steps = (int)steps.size() - 1;
    a.n_screens = n_screens;
    a.steps = reinterpret_cast<const SmallStep *>(d_steps);
    a.win_on = win.win_on; a.win_qs = win.win_qs; a.win_half_order = win.win_half_order;
    a.tw_row = tw; a.tw_col = twc;
    if (st && st->stats) { a.stats = st->stats; a.roi_lo = st->lo; a.roi_hi = st->hi; a.roi_n = st->n; a.dx = st->dx; }
    if (cluster_path_available(N, B)) {                           // one field over a cluster of 8 CTAs
        if (a.stats) {
            if (int rc = ensure_scratch(ctx, sizeof(double) * 9 * (size_t)B * N)) return rc;
            a.stats_acc = reinterpret_cast<double *>(ctx->scratch);
        }
        if (int rc = launch_cluster(ctx, N, B, a)) return rc;
        if (a.stats) return launch_stats_final(ctx, B, N, a.dx, a.roi_n, a.stats_acc, a.stats);
        return SSP_OK;
    }
    return launch_small(ctx, N, B, a);
}

// A *_host call that fails after copies have been queued must not return while DMA into the caller's host or
// device buffers is still in flight: wait for both copy streams and the context's stream, keep the first error.
int drain_pipeline(ssp_ctx *ctx, int rc)
{
    const std::string first = ctx->err;
    if (ctx->copy_in) cudaStreamSynchronize(ctx->copy_in);
    if (ctx->copy_out) cudaStreamSynchronize(ctx->copy_out);
    cudaStreamSynchronize(ctx->stream);
    cudaGetLastError();
    ctx->err = first;
    return rc;
}

bool small_ok(int N, int B, int h_kind, int n_steps, const void *planes)
{
    return (small_path_available(N) || cluster_path_available(N, B)) && h_kind == SSP_H_FRESNEL && !planes &&
           sizeof(SmallStep) * (size_t)(n_steps + 1) <= kSmallStepBytes;
}

} // namespace

extern "C" {

} // extern "C"

namespace {

// ssp_propagate, and (fused != null) the propagation half of ssp_evolve_propagate, in which the screen of step j is
// synthesised inside the row kernel from the column-transformed spectra instead of being read from d_screens.
int propagate_core(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                   int B, int n_steps, const double *dz,
                   const float *d_screens, long long screen_batch_stride, int S,
                   ssp_window win, const float *d_field_in, float *d_field_out,
                   float *d_planes, ssp_stats *d_stats, double roi_frac, const FusedScreens *fused)
{
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    if (int rc = trim_htables(ctx)) return rc;
    const int N = grid.N;
    const size_t px = (size_t)N * N;
    const double lam_eff = lambda / n0;
    const float2 *tw = nullptr, *twc = nullptr;          // row-plan and column-plan twiddles
    if (int rc = get_twiddles(ctx, N, 0, &tw)) return rc;
    if (int rc = get_twiddles(ctx, N, 1, &twc)) return rc;
    float2 *u = reinterpret_cast<float2 *>(d_field_out);
    // K8 rides on the last row pass (the output pixels are in registers there): ROI bounds decided here, in double
    int roi_lo = 0, roi_hi = 0;
    long long roi_n = 0;
    if (d_stats) stats_roi(N, roi_frac, &roi_lo, &roi_hi, &roi_n);

    if (!fused && small_ok(N, B, h_kind, n_steps, d_planes)) { // whole stack in one kernel, field resident in shared memory
        std::vector<SmallStep> ops(n_steps + 1);
        RowArgs w{};
        fill_window(w, win, N);
        for (int j = 0; j <= n_steps; ++j) {
            SmallStep &o = ops[j];
            o = SmallStep{};
            o.first = (j > 0); o.second = (j < n_steps); o.win = (j > 0);
            if (j >= 1 && j <= S) { o.phi = d_screens + (size_t)(j - 1) * px; o.phi_batch_stride = screen_batch_stride; o.phase_sign = 1.f; }
            if (j < n_steps) if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[j], 0, 0}, &o.hx)) return rc;
            if (j >= 1) if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[j - 1], 0, 1}, &o.hy)) return rc;
        }
        SmallStats st{d_stats, roi_lo, roi_hi, roi_n, grid.dx};
        return run_small(ctx, N, B, ops, S, w, reinterpret_cast<const float2 *>(d_field_in), u, tw, twc, &st);
    }
    const int bpf = row_stats_records(N);                     // records per field written by the last row kernel
    if (d_stats)
        if (int rc = ensure_scratch(ctx, sizeof(double) * 9 * (size_t)B * bpf)) return rc;
    // Fresnel: H = hx[kx] hy[ky], hx applied by the row kernels, hy by the column kernel.
    // Angular spectrum: H(ky,kx) is not separable; the column kernel applies the whole map, the rows none.
    const bool as = (h_kind == SSP_H_ANGULAR_SPECTRUM);
    // K4: FFT_x of the input, times hx of step 1
    const float2 *hx = nullptr;
    if (!as)
        if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[0], 0, 0}, &hx)) return rc;
    RowArgs r0{};
    r0.in = reinterpret_cast<const float2 *>(d_field_in);
    r0.out = u;
    r0.n_lines = B * N;
    r0.hx = hx;
    r0.tw = tw;
    if (int rc = launch_row(ctx, N, false, true, r0)) return rc;

    for (int j = 1; j <= n_steps; ++j) {
        // K5: FFT_y -> * hy_j / N^2 -> IFFT_y
        const float2 *hy = nullptr, *h2d = nullptr;
        if (as) { if (int rc = get_h2d_table(ctx, HKey{N, grid.dx, lam_eff, dz[j - 1], 0, 1}, &h2d)) return rc; }
        else if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[j - 1], 0, 1}, &hy)) return rc;
        ColArgs c{};
        c.in = u; c.out = u; c.B = B; c.hy = hy; c.h2d = h2d; c.tw = twc;
        if (int rc = launch_col_prop(ctx, N, c)) return rc;
        // K6: IFFT_x -> * exp(i phi_j) W -> [FFT_x -> * hx_{j+1}]
        RowArgs r{};
        r.in = u; r.out = u; r.n_lines = B * N; r.tw = tw;
        r.in_swapped = mid_swapped(N);
        if (j <= S && fused) {
            r.ycol = fused->ycol; r.scr0 = j - 1; r.scr_stride = S; r.n_sh = fused->n_sh;
            r.sh_coef = fused->sh_coef; r.sh_mean = fused->sh_mean; r.ex = fused->ex;
            r.phase_sign = 1.f;
        } else if (j <= S) {
            r.phi = d_screens + (size_t)(j - 1) * px;
            r.phi_batch_stride = screen_batch_stride;
            r.phase_sign = 1.f;
        }
        fill_window(r, win, N);
        r.win_map = window_map(ctx, N, r);
        if (d_planes) {
            r.plane_out = reinterpret_cast<float2 *>(d_planes) + (size_t)(j - 1) * px;
            r.plane_stride = (long long)n_steps * (long long)px;
        }
        const bool last = (j == n_steps);
        if (!last && !as) {
            if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[j], 0, 0}, &hx)) return rc;
            r.hx = hx;
        }
        if (last && d_stats) {
            r.stats_acc = reinterpret_cast<double *>(ctx->scratch);
            r.roi_lo = roi_lo; r.roi_hi = roi_hi;
        }
        if (int rc = launch_row(ctx, N, true, !last, r)) return rc;
    }
    if (d_stats)
        if (int rc = launch_stats_final(ctx, B, bpf, grid.dx, roi_n, reinterpret_cast<const double *>(ctx->scratch), d_stats)) return rc;
    return SSP_OK;
}

} // namespace

extern "C" {

int ssp_propagate(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                  int B, int n_steps, const double *dz,
                  const float *d_screens, long long screen_batch_stride, int S,
                  ssp_window win, const float *d_field_in, float *d_field_out,
                  float *d_planes, ssp_stats *d_stats, double roi_frac,
                  void *d_ws, size_t ws_bytes)
{
    (void)d_ws; (void)ws_bytes;
    if (int rc = check_prop(ctx, grid, lambda, n0, h_kind, B, n_steps, dz, d_screens, S, d_field_in, d_field_out))
        return rc;
    if (screen_batch_stride < 0 || (screen_batch_stride & 3))
        return ctx->fail(SSP_EINVAL, "screen_batch_stride must be >= 0 and a multiple of 4 elements");
    return propagate_core(ctx, grid, lambda, n0, h_kind, B, n_steps, dz, d_screens, screen_batch_stride, S, win, d_field_in,
                          d_field_out, d_planes, d_stats, roi_frac, nullptr);
}

int ssp_evolve_propagate(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, double n0,
                         int B, int S, const double *cn2, const double *dz, int n_sh,
                         double a, double vx, double vy, double T,
                         const float *d_fresh_noise, const float *d_fresh_noise_sh,
                         float *d_spectrum, float *d_sh_coef,
                         ssp_window win, const float *d_field_in, float *d_field_out,
                         ssp_stats *d_stats, double roi_frac, float *d_ycol, void *d_ws, size_t ws_bytes)
{
    if (!ctx) return SSP_EINVAL;
    if (grid.N != 1024) return ctx->fail(SSP_EUNSUPPORTED, "ssp_evolve_propagate is built for N = 1024 (use ssp_evolve_screens + ssp_propagate)");
    if (!(win.order > 0 && win.sigma_frac > 0)) return ctx->fail(SSP_EUNSUPPORTED, "ssp_evolve_propagate needs the absorbing window");
    if (!d_ycol || !aligned16(d_ycol)) return ctx->fail(SSP_EINVAL, "d_ycol (16-byte aligned) is required");
    // the propagation's argument checks first (d_ycol stands in for the screens: non-null, aligned), then the screens'
    if (int rc = check_prop(ctx, grid, lambda, n0, SSP_H_FRESNEL, B, S, dz, d_ycol, S, d_field_in, d_field_out)) return rc;
    FusedScreens fs{};
    if (int rc = evolve_to_ycol(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, a, vx, vy, T, d_fresh_noise, d_fresh_noise_sh,
                                d_spectrum, d_sh_coef, d_ycol, d_ws, ws_bytes, &fs))
        return rc;
    return propagate_core(ctx, grid, lambda, n0, SSP_H_FRESNEL, B, S, dz, nullptr, 0, S, win, d_field_in, d_field_out,
                          nullptr, d_stats, roi_frac, &fs);
}

int ssp_propagate_adjoint(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                          int B, int n_steps, const double *dz,
                          const float *d_screens, long long screen_batch_stride, int S,
                          ssp_window win, const float *d_g_out, float *d_g_in,
                          const float *d_planes, float *d_phase_grad,
                          void *d_ws, size_t ws_bytes)
{
    (void)d_ws; (void)ws_bytes;
    if (int rc = check_prop(ctx, grid, lambda, n0, h_kind, B, n_steps, dz, d_screens, S, d_g_out, d_g_in))
        return rc;
    if (screen_batch_stride < 0 || (screen_batch_stride & 3))
        return ctx->fail(SSP_EINVAL, "screen_batch_stride must be >= 0 and a multiple of 4 elements");
    if ((d_planes == nullptr) != (d_phase_grad == nullptr))
        return ctx->fail(SSP_EINVAL, "d_planes and d_phase_grad must both be given or both be null");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    if (int rc = trim_htables(ctx)) return rc;
    const int N = grid.N;
    const size_t px = (size_t)N * N;
    const double lam_eff = lambda / n0;
    const float2 *tw = nullptr, *twc = nullptr;          // row-plan and column-plan twiddles
    if (int rc = get_twiddles(ctx, N, 0, &tw)) return rc;
    if (int rc = get_twiddles(ctx, N, 1, &twc)) return rc;
    float2 *g = reinterpret_cast<float2 *>(d_g_in);

    if (small_ok(N, B, h_kind, n_steps, d_planes)) { // on-chip: op 0 = plane n_steps, then (column pass, plane j-1) for j = n_steps..1
        std::vector<SmallStep> ops(n_steps + 1);
        RowArgs w{};
        fill_window(w, win, N);
        for (int i = 0; i <= n_steps; ++i) {
            const int plane = n_steps - i;                       // the plane whose pointwise stage this row pass applies
            SmallStep &o = ops[i];
            o = SmallStep{};
            o.first = (i > 0); o.second = (plane >= 1); o.win = (plane >= 1);
            if (plane >= 1 && plane <= S) { o.phi = d_screens + (size_t)(plane - 1) * px; o.phi_batch_stride = screen_batch_stride; o.phase_sign = -1.f; }
            if (plane >= 1) if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[plane - 1], 1, 0}, &o.hx)) return rc;
            if (i >= 1) if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[plane], 1, 1}, &o.hy)) return rc;
        }
        return run_small(ctx, N, B, ops, S, w, reinterpret_cast<const float2 *>(d_g_out), g, tw, twc);
    }
    // pointwise stage of plane j: [grad_j] ; g <- W exp(-i phi_j) g
    auto plane_stage = [&](RowArgs &r, int j) {
        if (j <= S) {
            r.phi = d_screens + (size_t)(j - 1) * px;
            r.phi_batch_stride = screen_batch_stride;
            r.phase_sign = -1.f;
            if (d_phase_grad) {
                r.plane_in = reinterpret_cast<const float2 *>(d_planes) + (size_t)(j - 1) * px;
                r.plane_stride = (long long)n_steps * (long long)px;
                r.grad = d_phase_grad + (size_t)(j - 1) * px;
                r.grad_stride = (long long)S * (long long)px;
            }
        }
        fill_window(r, win, N);
        r.win_map = window_map(ctx, N, r);
    };

    const bool as = (h_kind == SSP_H_ANGULAR_SPECTRUM);
    const float2 *hx = nullptr;
    if (!as)
        if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[n_steps - 1], 1, 0}, &hx)) return rc;
    RowArgs r0{};
    r0.in = reinterpret_cast<const float2 *>(d_g_out);
    r0.out = g; r0.n_lines = B * N; r0.hx = hx; r0.tw = tw;
    plane_stage(r0, n_steps);
    if (int rc = launch_row(ctx, N, false, true, r0)) return rc;

    for (int j = n_steps; j >= 1; --j) {
        const float2 *hy = nullptr, *h2d = nullptr;
        if (as) { if (int rc = get_h2d_table(ctx, HKey{N, grid.dx, lam_eff, dz[j - 1], 1, 1}, &h2d)) return rc; }
        else if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[j - 1], 1, 1}, &hy)) return rc;
        ColArgs c{};
        c.in = g; c.out = g; c.B = B; c.hy = hy; c.h2d = h2d; c.tw = twc;
        if (int rc = launch_col_prop(ctx, N, c)) return rc;
        RowArgs r{};
        r.in = g; r.out = g; r.n_lines = B * N; r.tw = tw;
        r.in_swapped = mid_swapped(N);
        const bool last = (j == 1);
        if (!last) {
            plane_stage(r, j - 1);
            if (!as) {
                if (int rc = get_htable(ctx, HKey{N, grid.dx, lam_eff, dz[j - 2], 1, 0}, &hx)) return rc;
                r.hx = hx;
            }
        }
        if (int rc = launch_row(ctx, N, true, !last, r)) return rc;
    }
    return SSP_OK;
}

int ssp_beam_stats(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_field, double roi_frac,
                   ssp_stats *d_stats, float *d_mean, float *d_M2, long long *count)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || !(grid.dx > 0) || B < 1 || !d_field || !aligned16(d_field))
        return ctx->fail(SSP_EINVAL, "bad grid, batch or field pointer");
    const int n_opt = (d_mean != nullptr) + (d_M2 != nullptr) + (count != nullptr);
    if (n_opt != 0 && n_opt != 3) return ctx->fail(SSP_EINVAL, "d_mean, d_M2 and count go together");
    if (!d_stats && n_opt == 0) return ctx->fail(SSP_EINVAL, "nothing to compute");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const float2 *f = reinterpret_cast<const float2 *>(d_field);
    if (d_stats)
        if (int rc = launch_stats(ctx, grid.N, grid.dx, B, f, roi_frac, d_stats)) return rc;
    if (n_opt == 3) {
        if (*count < 0) return ctx->fail(SSP_EINVAL, "count must be >= 0");
        if (int rc = launch_welford(ctx, grid.N, B, f, d_mean, d_M2, *count)) return rc;
        *count += B;
    }
    return SSP_OK;
}

int ssp_propagate_host(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                       int B, int n_steps, const double *dz,
                       const float *h_screens, long long screen_batch_stride, int S,
                       ssp_window win, const float *h_field_in, float *h_field_out,
                       ssp_stats *h_stats, double roi_frac,
                       float *d_field, float *d_screens, ssp_stats *d_stats,
                       void *d_ws, size_t ws_bytes)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || S < 0) return ctx->fail(SSP_EINVAL, "bad grid, batch or S");
    if (!h_field_in || !h_field_out || !d_field) return ctx->fail(SSP_EINVAL, "field buffers are required");
    if (S > 0 && !d_screens) return ctx->fail(SSP_EINVAL, "d_screens is required");
    if (h_stats && !d_stats) return ctx->fail(SSP_EINVAL, "d_stats is required with h_stats");
    // everything the inner ssp_propagate calls would reject is rejected here, before the first copy is queued
    if (int rc = check_prop(ctx, grid, lambda, n0, h_kind, B, n_steps, dz, d_screens, S, d_field, d_field)) return rc;
    if (screen_batch_stride < 0 || (screen_batch_stride & 3))
        return ctx->fail(SSP_EINVAL, "screen_batch_stride must be >= 0 and a multiple of 4 elements");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t px = (size_t)grid.N * grid.N;
    const int rc_pipe = [&]() -> int {
    // Chunked pipeline over the batch: the host->device copy of chunk c+1 (copy_in stream) overlaps the
    // propagation of chunk c (context stream) and the device->host copy of chunk c-1 (copy_out stream).
    if (!ctx->copy_in) {
        SSP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_in, cudaStreamNonBlocking));
        SSP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_out, cudaStreamNonBlocking));
    }
    const int Bc = (B >= 8) ? B / 8 : 1;                        // fields per chunk
    const int n_chunks = (B + Bc - 1) / Bc;
    while ((int)ctx->pipe_events.size() < 2 * n_chunks + 2) {
        cudaEvent_t e;
        SSP_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->pipe_events.push_back(e);
    }
    cudaEvent_t ev_start = ctx->pipe_events[2 * n_chunks], ev_end = ctx->pipe_events[2 * n_chunks + 1];
    // earlier work on the context's stream may still use the device buffers
    SSP_CUDA(ctx, cudaEventRecord(ev_start, ctx->stream));
    SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_in, ev_start, 0));
    SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ev_start, 0));
    const bool shared = (screen_batch_stride == 0);
    const bool copy_screens = S > 0 && h_screens;               // NULL: the screens are already in d_screens
    if (copy_screens && shared)
        SSP_CUDA(ctx, cudaMemcpyAsync(d_screens, h_screens, sizeof(float) * (size_t)S * px, cudaMemcpyHostToDevice, ctx->copy_in));
    for (int c = 0; c < n_chunks; ++c) {
        const int b0 = c * Bc, nb = (B - b0 < Bc) ? B - b0 : Bc;
        cudaEvent_t ev_in = ctx->pipe_events[2 * c], ev_done = ctx->pipe_events[2 * c + 1];
        float *df = d_field + 2 * px * (size_t)b0;
        SSP_CUDA(ctx, cudaMemcpyAsync(df, h_field_in + 2 * px * (size_t)b0, sizeof(float) * 2 * px * nb, cudaMemcpyHostToDevice, ctx->copy_in));
        float *ds = d_screens;
        if (S > 0 && !shared) ds = d_screens + (size_t)b0 * (size_t)screen_batch_stride;
        if (copy_screens && !shared) {
            const size_t n_scr = (size_t)(nb - 1) * (size_t)screen_batch_stride + (size_t)S * px;
            SSP_CUDA(ctx, cudaMemcpyAsync(ds, h_screens + (size_t)b0 * (size_t)screen_batch_stride, sizeof(float) * n_scr,
                                          cudaMemcpyHostToDevice, ctx->copy_in));
        }
        SSP_CUDA(ctx, cudaEventRecord(ev_in, ctx->copy_in));
        SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ev_in, 0));
        if (int rc = ssp_propagate(ctx, grid, lambda, n0, h_kind, nb, n_steps, dz, ds, screen_batch_stride, S, win,
                                   df, df, nullptr, h_stats ? d_stats + b0 : nullptr, roi_frac, d_ws, ws_bytes))
            return rc;
        SSP_CUDA(ctx, cudaEventRecord(ev_done, ctx->stream));
        SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ev_done, 0));
        SSP_CUDA(ctx, cudaMemcpyAsync(h_field_out + 2 * px * (size_t)b0, df, sizeof(float) * 2 * px * nb, cudaMemcpyDeviceToHost, ctx->copy_out));
        if (h_stats)
            SSP_CUDA(ctx, cudaMemcpyAsync(h_stats + b0, d_stats + b0, sizeof(ssp_stats) * nb, cudaMemcpyDeviceToHost, ctx->copy_out));
    }
    SSP_CUDA(ctx, cudaEventRecord(ev_end, ctx->copy_out));
    SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ev_end, 0));
    SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SSP_OK;
    }();
    return rc_pipe ? drain_pipeline(ctx, rc_pipe) : SSP_OK;
}

int ssp_frame_chunk(int B) { return B >= 8 ? B / 8 : 1; }

int ssp_frame_host(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, double n0, int h_kind,
                   int B, int S, const double *cn2, const double *dz, int n_sh, const ssp_ar *ar,
                   ssp_window win, const float *h_field_in, float *h_field_out, ssp_stats *h_stats, double roi_frac,
                   float *d_field, float *d_spectrum, float *d_sh_coef, float *d_screens,
                   float *d_noise, float *d_noise_sh, ssp_stats *d_stats, void *d_ws, size_t ws_bytes,
                   float *h_adjoint_out, float *d_adjoint)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || S < 1 || !ar || !psd) return ctx->fail(SSP_EINVAL, "bad grid, batch, S or parameters");
    if (!h_field_in || !h_field_out || !d_field || !d_spectrum || !d_screens || !d_noise)
        return ctx->fail(SSP_EINVAL, "field, spectrum, screen and noise buffers are required");
    if (n_sh > 0 && (!d_sh_coef || !d_noise_sh)) return ctx->fail(SSP_EINVAL, "subharmonic buffers are required");
    if (h_stats && !d_stats) return ctx->fail(SSP_EINVAL, "d_stats is required with h_stats");
    if (h_adjoint_out && (!d_adjoint || !aligned16(d_adjoint)))
        return ctx->fail(SSP_EINVAL, "d_adjoint (16-byte aligned) is required with h_adjoint_out");
    // everything the inner calls would reject is rejected here, before the first copy is queued
    if (int rc = check_prop(ctx, grid, lambda, n0, h_kind, B, S, dz, d_screens, S, d_field, d_field)) return rc;
    if (int rc = check_screen_args(ctx, grid, psd, lambda, ssp_frame_chunk(B), S, cn2, dz, n_sh, d_noise, d_noise_sh,
                                   d_screens, d_ws, ws_bytes))
        return rc;
    if (!(ar->a >= 0.0 && ar->a <= 1.0)) return ctx->fail(SSP_EINVAL, "AR factor a must be in [0, 1]");
    if (!aligned16(d_spectrum) || !aligned16(d_sh_coef) || !aligned16(d_noise_sh))
        return ctx->fail(SSP_EINVAL, "device pointers must be 16-byte aligned");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t px = (size_t)grid.N * grid.N;
    if (!ctx->copy_in) {
        SSP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_in, cudaStreamNonBlocking));
        SSP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_out, cudaStreamNonBlocking));
    }
    const int rc_pipe = [&]() -> int {
    const int Bc = ssp_frame_chunk(B);
    const int n_chunks = (B + Bc - 1) / Bc;
    while ((int)ctx->pipe_events.size() < 2 * n_chunks + 2) {
        cudaEvent_t e;
        SSP_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->pipe_events.push_back(e);
    }
    cudaEvent_t ev_start = ctx->pipe_events[2 * n_chunks], ev_end = ctx->pipe_events[2 * n_chunks + 1];
    SSP_CUDA(ctx, cudaEventRecord(ev_start, ctx->stream));       // earlier work may still use the device buffers
    SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_in, ev_start, 0));
    SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ev_start, 0));
    // every field's upload is queued at once: it runs under the noise draws and the screen evolution of the first chunks
    for (int c = 0; c < n_chunks; ++c) {
        const int b0 = c * Bc, nb = (B - b0 < Bc) ? B - b0 : Bc;
        SSP_CUDA(ctx, cudaMemcpyAsync(d_field + 2 * px * (size_t)b0, h_field_in + 2 * px * (size_t)b0,
                                      sizeof(float) * 2 * px * nb, cudaMemcpyHostToDevice, ctx->copy_in));
        SSP_CUDA(ctx, cudaEventRecord(ctx->pipe_events[2 * c], ctx->copy_in));
    }
    const size_t sh_per_field = (size_t)S * (size_t)(n_sh > 0 ? n_sh : 0) * 9;
    if (n_sh > 0)
        if (int rc = ssp_fill_noise(ctx, ar->seed, 2 * ar->frame + 1, 0, (unsigned long long)B * sh_per_field, d_noise_sh)) return rc;
    // Screens evolve in uniform chunks (the noise scratch holds one chunk); the fields propagate in groups of chunks
    // that halve towards the end -- n/2, n/4, .., 1, 1 chunks -- so that the big groups run at full-batch efficiency
    // and only a small group's download is left uncovered at the end.
    int group_end = (n_chunks + 1) / 2, group_begin = 0;
    for (int c = 0; c < n_chunks; ++c) {
        const int b0 = c * Bc, nb = (B - b0 < Bc) ? B - b0 : Bc;
        const size_t off = (size_t)b0 * S * px;                   // in screens; complex arrays: 2 floats per element
        if (screen_col_seeded_supported(grid.N)) {
            // the generator draws the chunk's noise itself (same draws, bit for bit): no 8 B/px fill, no 8 B/px read
            if (int rc = ssp_evolve_screens_seeded(ctx, grid, psd, lambda, nb, S, cn2, dz, n_sh, ar->a, ar->vx, ar->vy, ar->T,
                                                   ar->seed, 2 * ar->frame, off,
                                                   n_sh > 0 ? d_noise_sh + 2 * (size_t)b0 * sh_per_field : nullptr, d_spectrum + 2 * off,
                                                   n_sh > 0 ? d_sh_coef + 2 * (size_t)b0 * sh_per_field : nullptr, d_screens + off,
                                                   d_ws, ws_bytes))
                return rc;
        } else {
            if (int rc = ssp_fill_noise(ctx, ar->seed, 2 * ar->frame, off, (unsigned long long)nb * S * px, d_noise)) return rc;
            if (int rc = ssp_evolve_screens(ctx, grid, psd, lambda, nb, S, cn2, dz, n_sh, ar->a, ar->vx, ar->vy, ar->T, d_noise,
                                            n_sh > 0 ? d_noise_sh + 2 * (size_t)b0 * sh_per_field : nullptr, d_spectrum + 2 * off,
                                            n_sh > 0 ? d_sh_coef + 2 * (size_t)b0 * sh_per_field : nullptr, d_screens + off,
                                            d_ws, ws_bytes))
                return rc;
        }
        if (c + 1 < group_end) continue;
        // fields of chunks group_begin .. c
        const int g0 = group_begin * Bc, gn = (b0 + nb) - g0;
        float *df = d_field + 2 * px * (size_t)g0;
        SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->pipe_events[2 * c], 0));   // copy_in is in order: chunk c done => all earlier done
        if (int rc = ssp_propagate(ctx, grid, lambda, n0, h_kind, gn, S, dz, d_screens + (size_t)g0 * S * px,
                                   (long long)S * (long long)px, S, win, df, df, nullptr, h_stats ? d_stats + g0 : nullptr,
                                   roi_frac, d_ws, ws_bytes))
            return rc;
        cudaEvent_t ev_done = ctx->pipe_events[2 * c + 1];
        SSP_CUDA(ctx, cudaEventRecord(ev_done, ctx->stream));
        SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ev_done, 0));
        SSP_CUDA(ctx, cudaMemcpyAsync(h_field_out + 2 * px * (size_t)g0, df, sizeof(float) * 2 * px * gn, cudaMemcpyDeviceToHost, ctx->copy_out));
        if (h_stats)
            SSP_CUDA(ctx, cudaMemcpyAsync(h_stats + g0, d_stats + g0, sizeof(ssp_stats) * gn, cudaMemcpyDeviceToHost, ctx->copy_out));
        if (h_adjoint_out) {
            // the received fields sent back through the same screens: A^H U_out (reads df while it is being downloaded)
            float *dg = d_adjoint + 2 * px * (size_t)g0;
            if (int rc = ssp_propagate_adjoint(ctx, grid, lambda, n0, h_kind, gn, S, dz, d_screens + (size_t)g0 * S * px,
                                               (long long)S * (long long)px, S, win, df, dg, nullptr, nullptr, d_ws, ws_bytes))
                return rc;
            SSP_CUDA(ctx, cudaEventRecord(ev_done, ctx->stream));   // re-recorded: the earlier wait has captured the first record
            SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_out, ev_done, 0));
            SSP_CUDA(ctx, cudaMemcpyAsync(h_adjoint_out + 2 * px * (size_t)g0, dg, sizeof(float) * 2 * px * gn, cudaMemcpyDeviceToHost, ctx->copy_out));
        }
        group_begin = c + 1;
        const int left = n_chunks - group_begin;
        group_end = group_begin + (left + 1) / 2;
    }
    SSP_CUDA(ctx, cudaEventRecord(ev_end, ctx->copy_out));
    SSP_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ev_end, 0));
    SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return SSP_OK;
    }();
    return rc_pipe ? drain_pipeline(ctx, rc_pipe) : SSP_OK;
}

} // extern "C"
