// ssp_api_screens.cu -- extern "C" entry points for screen generation / AR evolution and the
// mask-system helpers.  Host code here only derives per-slab scalars and small 1-D tables in
// double precision; the per-pixel work runs in ssp_screens.cu / ssp_propagate.cu / ssp_misc.cu.
#include <cmath>
#include <cstring>

#include "ssp_internal.h"

using namespace ssp;

namespace {

const double kPi = 3.14159265358979323846;
const int kMaxSh = 8;
const size_t kChunkBytes = (size_t)512 << 20; // intermediate (column-transformed) buffer budget

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct WsLayout {
    size_t tab_amp, tab_amp_sh, tab_mfac, tab_tau_sh, tab_ex, tab_taux, tab_tauy, tab_coef2;
    size_t sh_coef, sh_mean, inter, total;
    int chunk;
};

WsLayout ws_layout(int N, int B, int S)
{
    WsLayout L{};
    size_t o = 0;
    const size_t nscr = (size_t)B * (S > 0 ? S : 1);
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
    L.tab_amp = take(sizeof(float) * (S > 0 ? S : 1));
    L.tab_amp_sh = take(sizeof(float) * (S > 0 ? S : 1) * kMaxSh * 9);
    L.tab_mfac = take(sizeof(float2) * kMaxSh * 9);
    L.tab_tau_sh = take(sizeof(float2) * kMaxSh * 9);
    L.tab_ex = take(sizeof(float2) * kMaxSh * N);
    L.tab_taux = take(sizeof(float2) * N);
    L.tab_tauy = take(sizeof(float2) * N);
    L.tab_coef2 = take(sizeof(float2) * 2 * (size_t)B);   // ssp_lincomb scalars
    L.sh_coef = take(sizeof(float2) * nscr * kMaxSh * 9);
    L.sh_mean = take(sizeof(float) * 2 * nscr);
    const size_t per = sizeof(float2) * (size_t)N * N;
    size_t chunk = kChunkBytes / per;
    if (chunk < 1) chunk = 1;
    if (chunk > nscr) chunk = nscr;
    L.chunk = (int)chunk;
    L.inter = take(per * chunk);
    L.total = o;
    return L;
}

// Scalar (frequency-independent) part of sqrt(Phi^f) for one slab; the frequency-dependent
// part is evaluated per element on the device (ssp_screens.cu: psd_shape_sqrt).
double psd_scalar_sqrt(const ssp_psd *psd, double lambda, double cn2, double dz)
{
    const double k = 2.0 * kPi / lambda;
    if (psd->kind == SSP_PSD_OCEAN_NIKISHOV) {
        const double tp = 2.0 * kPi;
        return sqrt(tp * tp * tp * k * k * dz * 0.388e-8 * pow(psd->eps, -1.0 / 3.0) * psd->chi_T / (psd->w * psd->w));
    }
    if (psd->kind == SSP_PSD_POWER_LAW) { // (2 pi)^3 k^2 dz A (2 pi f)^-alpha: scalar part (PAPER.md:331 S12, :346 S14)
        const double tp = 2.0 * kPi;
        return sqrt(pow(tp, 3.0 - psd->alpha) * k * k * dz * psd->A);
    }
    const double r0 = pow(0.423 * k * k * cn2 * dz, -3.0 / 5.0); // PAPER.md:375 (S18)
    return sqrt(0.023) * pow(r0, -5.0 / 6.0);                     // PAPER.md:370 (S17)
}

// Frequency-dependent part of sqrt(Phi^f) in double (subharmonic coefficients: 8 per level).
double psd_shape_sqrt_host(const ssp_psd *psd, double f)
{
    if (!(f > 0)) return 0.0;
    if (psd->kind == SSP_PSD_OCEAN_NIKISHOV) {
        double eta = psd->eta > 0 ? psd->eta : pow(1e-18 / psd->eps, 0.25);
        const double kap = 2.0 * kPi * f, ke = kap * eta;
        const double delta = 8.284 * pow(ke, 4.0 / 3.0) + 12.978 * ke * ke;
        const double w = psd->w;
        const double br = w * w * exp(-1.863e-2 * delta) + exp(-1.9e-4 * delta) - 2.0 * w * exp(-9.41e-3 * delta);
        return sqrt(pow(kap, -11.0 / 3.0) * (1.0 + 2.35 * pow(ke, 2.0 / 3.0)) * (br > 0 ? br : 0));
    }
    double f0 = 0, inv_fm2 = 0;
    const bool pl = (psd->kind == SSP_PSD_POWER_LAW);
    if (psd->kind == SSP_PSD_VON_KARMAN || pl) {
        if (psd->L0 > 0) f0 = 1.0 / psd->L0;
        if (psd->l0 > 0) {
            const double kmc = psd->km_coeff > 0 ? psd->km_coeff : 2.0 * kPi;
            const double fm = kmc / (2.0 * kPi * psd->l0);
            inv_fm2 = 1.0 / (fm * fm);
        }
    }
    return exp(-0.5 * f * f * inv_fm2) * pow(f * f + f0 * f0, pl ? -0.25 * psd->alpha : -11.0 / 12.0);
}

int check_screens(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, int B, int S,
                  const double *cn2, const double *dz, int n_sh, const void *noise, const void *noise_sh,
                  const void *screens, const void *ws, size_t ws_bytes)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N)) return ctx->fail(SSP_EINVAL, "N=%d is not a power of two in [8, 4096]", grid.N);
    if (!(grid.dx > 0) || !(lambda > 0)) return ctx->fail(SSP_EINVAL, "dx and lambda must be > 0");
    if (!psd || B < 1 || S < 1 || !cn2 || !dz) return ctx->fail(SSP_EINVAL, "psd, B >= 1, S >= 1, cn2, dz are required");
    if (n_sh < 0 || n_sh > kMaxSh) return ctx->fail(SSP_EINVAL, "n_sh must be in [0, %d]", kMaxSh);
    if (psd->kind < 0 || psd->kind > SSP_PSD_POWER_LAW) return ctx->fail(SSP_EINVAL, "unknown PSD kind %d", psd->kind);
    if (psd->kind == SSP_PSD_POWER_LAW && (!(psd->alpha >= 3.0 && psd->alpha < 5.0) || !(psd->A >= 0)))
        return ctx->fail(SSP_EINVAL, "power-law PSD needs 3 <= alpha < 5 and A >= 0");
    if (psd->kind == SSP_PSD_VON_KARMAN && (!(psd->L0 > 0) || !(psd->l0 > 0)))
        return ctx->fail(SSP_EINVAL, "von Karman needs L0 > 0 and l0 > 0");
    if (psd->kind == SSP_PSD_OCEAN_NIKISHOV && (!(psd->eps > 0) || !(psd->chi_T > 0) || psd->w == 0))
        return ctx->fail(SSP_EINVAL, "ocean PSD needs eps > 0, chi_T > 0, w != 0");
    for (int s = 0; s < S; ++s) {
        if (!(dz[s] > 0)) return ctx->fail(SSP_EINVAL, "dz[%d] must be > 0", s);
        if (psd->kind <= SSP_PSD_VON_KARMAN && !(cn2[s] >= 0)) return ctx->fail(SSP_EINVAL, "cn2[%d] must be >= 0", s);
    }
    if (!noise || !screens) return ctx->fail(SSP_EINVAL, "noise and screens pointers are required");
    if (n_sh > 0 && !noise_sh) return ctx->fail(SSP_EINVAL, "noise_sh is required when n_sh > 0");
    if (!aligned16(noise) || !aligned16(screens) || !aligned16(ws))
        return ctx->fail(SSP_EINVAL, "device pointers must be 16-byte aligned");
    if (!ws || ws_bytes < ssp_workspace_bytes(grid, B, S))
        return ctx->fail(SSP_EWORKSPACE, "workspace of %zu bytes needed, %zu given", ssp_workspace_bytes(grid, B, S), ws_bytes);
    return SSP_OK;
}

// Shared body of make_screens (ar == false) and evolve_screens (ar == true).
int screens_impl(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, int B, int S,
                 const double *cn2, const double *dz, int n_sh, bool ar, double a, double vx, double vy, double T,
                 const float *d_noise, const float *d_noise_sh, float *d_spectrum, float *d_sh_coef,
                 float *d_screens, void *d_ws, float *d_screens_im = nullptr, float2 *ycol_out = nullptr,
                 ssp::FusedScreens *fused = nullptr, const ssp::NoiseSeed *seeded = nullptr)
{
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const int N = grid.N;
    const size_t px = (size_t)N * N;
    const double df = 1.0 / (N * grid.dx);
    const WsLayout L = ws_layout(N, B, S);
    char *ws = reinterpret_cast<char *>(d_ws);
    const float2 *tw = nullptr, *twc = nullptr;          // row-plan and screen-column-plan twiddles
    if (int rc = get_twiddles(ctx, N, 0, &tw)) return rc;
    if (int rc = get_twiddles(ctx, N, screen_col_plan_variant(N), &twc)) return rc;
    cudaStream_t st = ctx->stream;

    // ---- per-slab scalars and 1-D tables (double on the host, fp32 on the device)
    std::vector<float> amp(S), amp_sh((size_t)S * (n_sh > 0 ? n_sh : 1) * 9, 0.f);
    for (int s = 0; s < S; ++s) {
        const double sc = psd_scalar_sqrt(psd, lambda, cn2[s], dz[s]);
        amp[s] = (float)(sc * df);
        double dfp = df;
        for (int p = 0; p < n_sh; ++p) {
            dfp /= 3.0;
            for (int aa = 0; aa < 3; ++aa)
                for (int bb = 0; bb < 3; ++bb) {
                    if (aa == 1 && bb == 1) continue;
                    const double f = hypot((bb - 1) * dfp, (aa - 1) * dfp);
                    amp_sh[((size_t)s * n_sh + p) * 9 + aa * 3 + bb] = (float)(sc * psd_shape_sqrt_host(psd, f) * dfp);
                }
        }
    }
    SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_amp, amp.data(), sizeof(float) * S, cudaMemcpyHostToDevice, st));
    const float *d_amp = reinterpret_cast<const float *>(ws + L.tab_amp);

    const float2 *d_taux = nullptr, *d_tauy = nullptr;
    const bool tilt = ar && (vx != 0.0 || vy != 0.0) && T != 0.0;
    if (tilt) { // tau = exp(-i 2 pi T (fx vx + fy vy)) = taux[kx] tauy[ky]   (Eq.4; Q9)
        std::vector<float2> tx(N), ty(N);
        for (int k = 0; k < N; ++k) {
            const double f = (double)((k < N / 2) ? k : k - N) * df;
            const double ax = fmod(-2.0 * kPi * T * f * vx, 2.0 * kPi), ay = fmod(-2.0 * kPi * T * f * vy, 2.0 * kPi);
            tx[k] = make_float2((float)cos(ax), (float)sin(ax));
            ty[k] = make_float2((float)cos(ay), (float)sin(ay));
        }
        SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_taux, tx.data(), sizeof(float2) * N, cudaMemcpyHostToDevice, st));
        SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_tauy, ty.data(), sizeof(float2) * N, cudaMemcpyHostToDevice, st));
        d_taux = reinterpret_cast<const float2 *>(ws + L.tab_taux);
        d_tauy = reinterpret_cast<const float2 *>(ws + L.tab_tauy);
    }

    // ---- subharmonic coefficients and the analytic mean of phi_lo (P4)
    float2 *coef = d_sh_coef ? reinterpret_cast<float2 *>(d_sh_coef) : reinterpret_cast<float2 *>(ws + L.sh_coef);
    float *mean = reinterpret_cast<float *>(ws + L.sh_mean);
    const float2 *d_ex = reinterpret_cast<const float2 *>(ws + L.tab_ex);
    if (n_sh > 0) {
        std::vector<float2> mfac((size_t)n_sh * 9), tau_sh((size_t)n_sh * 9), ex((size_t)n_sh * N);
        double dfp = df;
        for (int p = 0; p < n_sh; ++p) {
            dfp /= 3.0;
            // M(+1) = (1/N) sum_i exp(i 2 pi dfp x_i);  M(-1) = conj, M(0) = 1
            double mr = 0, mi = 0;
            for (int i = 0; i < N; ++i) {
                const double ang = 2.0 * kPi * dfp * (double)(i - N / 2) * grid.dx;
                mr += cos(ang); mi += sin(ang);
                ex[(size_t)p * N + i] = make_float2((float)cos(ang), (float)sin(ang));
            }
            mr /= N; mi /= N;
            for (int aa = 0; aa < 3; ++aa)
                for (int bb = 0; bb < 3; ++bb) {
                    const double yr = (aa == 1) ? 1.0 : mr, yi = (aa == 1) ? 0.0 : (aa == 2 ? mi : -mi);
                    const double xr = (bb == 1) ? 1.0 : mr, xi = (bb == 1) ? 0.0 : (bb == 2 ? mi : -mi);
                    mfac[(size_t)p * 9 + aa * 3 + bb] = make_float2((float)(xr * yr - xi * yi), (float)(xr * yi + xi * yr));
                    const double ang = -2.0 * kPi * T * ((bb - 1) * dfp * vx + (aa - 1) * dfp * vy);
                    tau_sh[(size_t)p * 9 + aa * 3 + bb] = make_float2((float)cos(ang), (float)sin(ang));
                }
        }
        SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_amp_sh, amp_sh.data(), sizeof(float) * S * n_sh * 9, cudaMemcpyHostToDevice, st));
        SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_mfac, mfac.data(), sizeof(float2) * n_sh * 9, cudaMemcpyHostToDevice, st));
        SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_tau_sh, tau_sh.data(), sizeof(float2) * n_sh * 9, cudaMemcpyHostToDevice, st));
        SSP_CUDA(ctx, cudaMemcpyAsync(ws + L.tab_ex, ex.data(), sizeof(float2) * n_sh * N, cudaMemcpyHostToDevice, st));
        if (int rc = launch_sh_prep(ctx, B * S, S, n_sh, reinterpret_cast<const float2 *>(d_noise_sh),
                                    reinterpret_cast<const float *>(ws + L.tab_amp_sh),
                                    tilt ? reinterpret_cast<const float2 *>(ws + L.tab_tau_sh) : nullptr,
                                    (float)a, (float)sqrt(1.0 - a * a),
                                    ar ? reinterpret_cast<const float2 *>(d_sh_coef) : nullptr, coef,
                                    reinterpret_cast<const float2 *>(ws + L.tab_mfac), mean))
            return rc;
    }

    // ---- high-frequency part, chunk by chunk: K1+K2 (columns) then K3 (rows)
    ScreenFilter flt{};
    flt.kind = psd->kind;
    flt.df = (float)df;
    flt.two_pi = (float)(2.0 * kPi);
    flt.pexp = (psd->kind == SSP_PSD_POWER_LAW) ? (float)(0.25 * psd->alpha) : (float)(11.0 / 12.0);
    if (psd->kind == SSP_PSD_VON_KARMAN || psd->kind == SSP_PSD_POWER_LAW) {
        if (psd->L0 > 0) flt.f0sq = (float)(1.0 / (psd->L0 * psd->L0));
        if (psd->l0 > 0) {
            const double kmc = psd->km_coeff > 0 ? psd->km_coeff : 2.0 * kPi;
            const double fm = kmc / (2.0 * kPi * psd->l0);
            flt.inv_fm2_log2e = (float)(1.4426950408889634 / (2.0 * fm * fm));
        }
    } else if (psd->kind == SSP_PSD_OCEAN_NIKISHOV) {
        flt.eta = (float)(psd->eta > 0 ? psd->eta : pow(1e-18 / psd->eps, 0.25));
        flt.w = (float)psd->w;
    }
    // warp-uniform half of the subharmonic phasors (ScreenRowArgs::e2), in double like the other tables
    ScreenRowArgs rproto{};
    {
        const int RLr = row_last_radix(N);
        double dfp = df;
        for (int p = 0; p < n_sh; ++p) {
            dfp /= 3.0;
            for (int q = 0; q < RLr && q < 32; ++q) {
                const double ang = 2.0 * kPi * dfp * (double)q * (double)(N / RLr) * grid.dx;
                rproto.e2[p][q] = make_float2((float)cos(ang), (float)sin(ang));
            }
        }
    }
    float2 *inter = reinterpret_cast<float2 *>(ws + L.inter);
    const int nscr = B * S;
    for (int g0 = 0; g0 < nscr; g0 += L.chunk) {
        const int n = (nscr - g0 < L.chunk) ? nscr - g0 : L.chunk;
        ScreenColArgs c{};
        c.noise = seeded ? nullptr : reinterpret_cast<const float2 *>(d_noise) + (size_t)g0 * px;
        if (seeded) {                                             // the generator draws element e of the batch as draw first + e
            c.keys = key_schedule(seeded->seed);
            c.stream_lo = (uint32_t)seeded->stream; c.stream_hi = (uint32_t)(seeded->stream >> 32);
            c.first_draw = seeded->first + (unsigned long long)g0 * px;
        }
        c.old_spec = ar ? reinterpret_cast<const float2 *>(d_spectrum) + (size_t)g0 * px : nullptr;
        c.spec_out = d_spectrum ? reinterpret_cast<float2 *>(d_spectrum) + (size_t)g0 * px : nullptr;
        c.out = ycol_out ? ycol_out + (size_t)g0 * px : inter;   // fused synthesis: every screen's column-transformed spectrum is kept
        c.nscr = n; c.g0 = g0; c.S = S;
        c.amp = d_amp;
        c.flt = flt;
        c.ar_a = (float)a; c.ar_g = (float)sqrt(1.0 - a * a);
        c.taux = d_taux; c.tauy = d_tauy;
        c.tw = twc;
        if (int rc = launch_screen_col(ctx, N, c)) return rc;
        if (ycol_out) continue;                                   // K3 runs inside the propagation's row kernels
        ScreenRowArgs r = rproto;
        r.in = inter;
        r.screens = d_screens + (size_t)g0 * px;
        r.nscr = n; r.n_sh = n_sh;
        r.sh_coef = coef + (size_t)g0 * n_sh * 9;
        r.sh_mean = mean + 2 * (size_t)g0;
        r.screens_im = d_screens_im ? d_screens_im + (size_t)g0 * px : nullptr;
        r.ex = d_ex;
        r.tw = tw;
        if (int rc = launch_screen_row(ctx, N, r)) return rc;
    }
    if (fused) { fused->ycol = ycol_out; fused->sh_coef = coef; fused->sh_mean = mean; fused->ex = d_ex; fused->n_sh = n_sh; }
    return SSP_OK;
}

} // namespace

int ssp::evolve_to_ycol(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, int B, int S, const double *cn2,
                        const double *dz, int n_sh, double a, double vx, double vy, double T, const float *d_noise,
                        const float *d_noise_sh, float *d_spectrum, float *d_sh_coef, float *d_ycol, void *d_ws,
                        size_t ws_bytes, FusedScreens *out)
{
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_noise, d_noise_sh, d_ycol, d_ws, ws_bytes)) return rc;
    if (!(a >= 0.0 && a <= 1.0)) return ctx->fail(SSP_EINVAL, "a must be in [0, 1]");
    if (!d_spectrum || !aligned16(d_spectrum)) return ctx->fail(SSP_EINVAL, "d_spectrum (in-out) is required");
    if (n_sh > 0 && !d_sh_coef) return ctx->fail(SSP_EINVAL, "d_sh_coef (in-out) is required when n_sh > 0");
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, true, a, vx, vy, T, d_noise, d_noise_sh, d_spectrum,
                        d_sh_coef, nullptr, d_ws, nullptr, reinterpret_cast<float2 *>(d_ycol), out);
}

int ssp::check_screen_args(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, int B, int S, const double *cn2,
                           const double *dz, int n_sh, const void *noise, const void *noise_sh, const void *screens,
                           const void *ws, size_t ws_bytes)
{
    return check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, noise, noise_sh, screens, ws, ws_bytes);
}

extern "C" {

size_t ssp_workspace_bytes(ssp_grid grid, int B, int S)
{
    if (!valid_N(grid.N) || B < 1 || S < 0) return 0;
    return ws_layout(grid.N, B, S).total;
}

int ssp_make_screens(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                     int B, int S, const double *cn2, const double *dz, int n_sh,
                     const float *d_noise, const float *d_noise_sh,
                     float *d_spectrum, float *d_sh_coef, float *d_screens,
                     void *d_ws, size_t ws_bytes)
{
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_noise, d_noise_sh, d_screens, d_ws, ws_bytes))
        return rc;
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, false, 0.0, 0.0, 0.0, 0.0,
                        d_noise, d_noise_sh, d_spectrum, d_sh_coef, d_screens, d_ws);
}

int ssp_evolve_screens(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                       int B, int S, const double *cn2, const double *dz, int n_sh,
                       double a, double vx, double vy, double T,
                       const float *d_fresh_noise, const float *d_fresh_noise_sh,
                       float *d_spectrum, float *d_sh_coef, float *d_screens,
                       void *d_ws, size_t ws_bytes)
{
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_fresh_noise, d_fresh_noise_sh,
                               d_screens, d_ws, ws_bytes))
        return rc;
    if (!(a >= 0.0 && a <= 1.0)) return ctx->fail(SSP_EINVAL, "a must be in [0, 1]");
    if (!d_spectrum || !aligned16(d_spectrum)) return ctx->fail(SSP_EINVAL, "d_spectrum (in-out) is required");
    if (n_sh > 0 && !d_sh_coef) return ctx->fail(SSP_EINVAL, "d_sh_coef (in-out) is required when n_sh > 0");
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, true, a, vx, vy, T,
                        d_fresh_noise, d_fresh_noise_sh, d_spectrum, d_sh_coef, d_screens, d_ws);
}

int ssp_make_screens_seeded(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                            int B, int S, const double *cn2, const double *dz, int n_sh,
                            unsigned long long seed, unsigned long long stream, unsigned long long first,
                            const float *d_noise_sh, float *d_spectrum, float *d_sh_coef, float *d_screens,
                            void *d_ws, size_t ws_bytes)
{
    // (the screens pointer stands in for the absent noise array in the shared checks)
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_screens, d_noise_sh, d_screens, d_ws, ws_bytes))
        return rc;
    if (d_spectrum && !aligned16(d_spectrum)) return ctx->fail(SSP_EINVAL, "d_spectrum must be 16-byte aligned");
    if (first & 1ull) return ctx->fail(SSP_EINVAL, "the first draw index must be even");
    if (!screen_col_seeded_supported(grid.N))
        return ctx->fail(SSP_EUNSUPPORTED, "seeded synthesis is built for N >= 512 (use ssp_fill_noise + ssp_make_screens)");
    const ssp::NoiseSeed ns{seed, stream, first};
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, false, 0.0, 0.0, 0.0, 0.0, nullptr, d_noise_sh,
                        d_spectrum, d_sh_coef, d_screens, d_ws, nullptr, nullptr, nullptr, &ns);
}

int ssp_evolve_screens_seeded(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                              int B, int S, const double *cn2, const double *dz, int n_sh,
                              double a, double vx, double vy, double T,
                              unsigned long long seed, unsigned long long stream, unsigned long long first,
                              const float *d_fresh_noise_sh, float *d_spectrum, float *d_sh_coef, float *d_screens,
                              void *d_ws, size_t ws_bytes)
{
    // (the screens pointer stands in for the absent noise array in the shared checks)
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_screens, d_fresh_noise_sh, d_screens, d_ws, ws_bytes))
        return rc;
    if (!(a >= 0.0 && a <= 1.0)) return ctx->fail(SSP_EINVAL, "a must be in [0, 1]");
    if (!d_spectrum || !aligned16(d_spectrum)) return ctx->fail(SSP_EINVAL, "d_spectrum (in-out) is required");
    if (n_sh > 0 && !d_sh_coef) return ctx->fail(SSP_EINVAL, "d_sh_coef (in-out) is required when n_sh > 0");
    if (first & 1ull) return ctx->fail(SSP_EINVAL, "the first draw index must be even");
    if (!screen_col_seeded_supported(grid.N))
        return ctx->fail(SSP_EUNSUPPORTED, "seeded evolution is built for N >= 512 (use ssp_fill_noise + ssp_evolve_screens)");
    const ssp::NoiseSeed ns{seed, stream, first};
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, true, a, vx, vy, T, nullptr, d_fresh_noise_sh,
                        d_spectrum, d_sh_coef, d_screens, d_ws, nullptr, nullptr, nullptr, &ns);
}

int ssp_make_screens_pair(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                          int B, int S, const double *cn2, const double *dz, int n_sh,
                          const float *d_noise, const float *d_noise_sh,
                          float *d_spectrum, float *d_sh_coef, float *d_screens, float *d_screens_im,
                          void *d_ws, size_t ws_bytes)
{
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_noise, d_noise_sh, d_screens, d_ws, ws_bytes))
        return rc;
    if (!d_screens_im || !aligned16(d_screens_im)) return ctx->fail(SSP_EINVAL, "d_screens_im is required (16-byte aligned)");
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, false, 0.0, 0.0, 0.0, 0.0,
                        d_noise, d_noise_sh, d_spectrum, d_sh_coef, d_screens, d_ws, d_screens_im);
}

int ssp_evolve_screens_pair(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                            int B, int S, const double *cn2, const double *dz, int n_sh,
                            double a, double vx, double vy, double T,
                            const float *d_fresh_noise, const float *d_fresh_noise_sh,
                            float *d_spectrum, float *d_sh_coef, float *d_screens, float *d_screens_im,
                            void *d_ws, size_t ws_bytes)
{
    if (int rc = check_screens(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, d_fresh_noise, d_fresh_noise_sh,
                               d_screens, d_ws, ws_bytes))
        return rc;
    if (!(a >= 0.0 && a <= 1.0)) return ctx->fail(SSP_EINVAL, "a must be in [0, 1]");
    if (!d_spectrum || !aligned16(d_spectrum)) return ctx->fail(SSP_EINVAL, "d_spectrum (in-out) is required");
    if (n_sh > 0 && !d_sh_coef) return ctx->fail(SSP_EINVAL, "d_sh_coef (in-out) is required when n_sh > 0");
    if (!d_screens_im || !aligned16(d_screens_im)) return ctx->fail(SSP_EINVAL, "d_screens_im is required (16-byte aligned)");
    return screens_impl(ctx, grid, psd, lambda, B, S, cn2, dz, n_sh, true, a, vx, vy, T,
                        d_fresh_noise, d_fresh_noise_sh, d_spectrum, d_sh_coef, d_screens, d_ws, d_screens_im);
}

// ---- mask-system helpers -----------------------------------------------------------------

int ssp_phase_mul(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_theta, double sign,
                  const float *d_in, float *d_out)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || !d_theta || !d_in || !d_out) return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_phase_mul(ctx, grid.N, B, d_theta, (float)sign, reinterpret_cast<const float2 *>(d_in),
                            reinterpret_cast<float2 *>(d_out));
}

int ssp_dft2_centered(ssp_ctx *ctx, ssp_grid grid, int B, int inverse,
                      const float *d_in, float *d_out, void *d_ws, size_t ws_bytes)
{
    (void)d_ws; (void)ws_bytes;
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || !d_in || !d_out || !aligned16(d_in) || !aligned16(d_out))
        return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const int N = grid.N;
    const float2 *tw = nullptr, *twc = nullptr, *sg = nullptr;
    if (int rc = get_twiddles(ctx, N, 0, &tw)) return rc;
    if (int rc = get_twiddles(ctx, N, 1, &twc)) return rc;
    if (int rc = get_sign_table(ctx, N, &sg)) return rc;
    // F_c = (-1)^(kx+ky) FFT2( (-1)^(ix+iy) x ) / N; rows carry both input signs, each axis 1/sqrt(N)
    RowArgs r{};
    r.in = reinterpret_cast<const float2 *>(d_in);
    r.out = reinterpret_cast<float2 *>(d_out);
    r.n_lines = B * N;
    r.pre = sg; r.pre_line = sg; r.hx = sg + N; r.tw = tw;
    if (int rc = launch_row(ctx, N, inverse != 0, inverse == 0, r)) return rc;
    ColArgs c{};
    c.in = r.out; c.out = r.out; c.B = B; c.hy = sg + N; c.tw = twc;
    return launch_col_single(ctx, N, inverse != 0, c);
}

int ssp_adam_update(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_grad, double lr, double beta1,
                    double beta2, double eps, int t, float *d_m, float *d_v, float *d_theta)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || t < 1 || !d_grad || !d_m || !d_v || !d_theta || !(beta1 >= 0 && beta1 < 1) ||
        !(beta2 >= 0 && beta2 < 1) || !(eps > 0))
        return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const double c1 = 1.0 / (1.0 - pow(beta1, (double)t)), c2 = 1.0 / (1.0 - pow(beta2, (double)t));
    return launch_adam(ctx, (long long)grid.N * grid.N, B, d_grad, (float)lr, (float)beta1, (float)beta2, (float)eps,
                       (float)c1, (float)c2, (float)(1.0 - beta1), (float)(1.0 - beta2), d_m, d_v, d_theta);
}

int ssp_aperture(ssp_ctx *ctx, ssp_grid grid, int B, double radius, const float *d_in, float *d_out)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || !(grid.dx > 0) || B < 1 || !(radius >= 0) || !d_in || !d_out)
        return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    const double q = radius / grid.dx;
    return launch_aperture(ctx, grid.N, B, (long long)floor(q * q), reinterpret_cast<const float2 *>(d_in),
                           reinterpret_cast<float2 *>(d_out));
}

int ssp_phase_grad(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_g, const float *d_u, float *d_grad)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || !d_g || !d_u || !d_grad) return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_phase_grad(ctx, (long long)B * grid.N * grid.N, reinterpret_cast<const float2 *>(d_g),
                             reinterpret_cast<const float2 *>(d_u), d_grad);
}

int ssp_inner_products(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_a, const float *d_b, double *d_out)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || !d_a || !d_b || !d_out) return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_inner(ctx, grid.N, B, reinterpret_cast<const float2 *>(d_a), reinterpret_cast<const float2 *>(d_b), d_out);
}

int ssp_mae_loss(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_v, const float *d_t, double *d_loss, float *d_grad)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || !d_v || !d_t || !d_loss || !d_grad) return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_mae(ctx, grid.N, B, reinterpret_cast<const float2 *>(d_v), reinterpret_cast<const float2 *>(d_t), d_loss,
                      reinterpret_cast<float2 *>(d_grad));
}

int ssp_lincomb(ssp_ctx *ctx, ssp_grid grid, int B, const double *h_alpha, const float *d_a,
                const double *h_beta, const float *d_b, float *d_out)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || B < 1 || !h_alpha || !h_beta || !d_a || !d_b || !d_out)
        return ctx->fail(SSP_EINVAL, "bad arguments");
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    if (int rc = ensure_scratch(ctx, (size_t)65536 + sizeof(float2) * 2 * (size_t)B)) return rc;
    std::vector<float2> co(2 * (size_t)B);
    for (int b = 0; b < B; ++b) {
        co[2 * b] = make_float2((float)h_alpha[2 * b], (float)h_alpha[2 * b + 1]);
        co[2 * b + 1] = make_float2((float)h_beta[2 * b], (float)h_beta[2 * b + 1]);
    }
    // the coefficient slot sits past the statistics accumulators in the context scratch
    float2 *d_co = reinterpret_cast<float2 *>(reinterpret_cast<char *>(ctx->scratch) + 32768);
    if (sizeof(float2) * co.size() > ctx->scratch_bytes - 32768) return ctx->fail(SSP_EINVAL, "B too large");
    SSP_CUDA(ctx, cudaMemcpyAsync(d_co, co.data(), sizeof(float2) * co.size(), cudaMemcpyHostToDevice, ctx->stream));
    return launch_lincomb(ctx, grid.N, B, d_co, reinterpret_cast<const float2 *>(d_a),
                          reinterpret_cast<const float2 *>(d_b), reinterpret_cast<float2 *>(d_out));
}

} // extern "C"
