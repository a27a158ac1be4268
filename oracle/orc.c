/*
 * orc.c -- CPU ORACLE (test infrastructure only; see orc.h).
 *
 * Plain, slow, double-precision restatement of what the split-step phase-screen
 * path computes, written from /root/reference/PAPER.md.  Each function cites
 * the passage it follows.  No code is shared with the CUDA path.
 */
#include "orc.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------- */
/* P0: discrete Fourier transforms                                            */
/* ------------------------------------------------------------------------- */

/* The definition itself: X[k] = sum_n x[n] exp(sign * i 2 pi k n / N). */
int orc_dft1d_naive(double *a, int n, int sign)
{
    double *t = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    if (!t) return -1;
    for (int k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; ++j) {
            /* reduce k*j mod n in integers so the angle stays accurate */
            long long kj = ((long long)k * j) % n;
            double ang = sign * 2.0 * M_PI * (double)kj / (double)n;
            double c = cos(ang), s = sin(ang);
            sr += a[2 * j] * c - a[2 * j + 1] * s;
            si += a[2 * j] * s + a[2 * j + 1] * c;
        }
        t[2 * k] = sr;
        t[2 * k + 1] = si;
    }
    memcpy(a, t, sizeof(double) * 2 * (size_t)n);
    free(t);
    return 0;
}

/* Textbook iterative radix-2 decimation-in-time FFT (bit reversal, then log2 n
 * butterfly passes); every twiddle is evaluated directly with cos/sin. */
static int fft_radix2(double *a, int n, int sign)
{
    int lg = 0;
    while ((1 << lg) < n) ++lg;
    if ((1 << lg) != n) return -1;
    for (int i = 0; i < n; ++i) {
        int r = 0;
        for (int b = 0; b < lg; ++b)
            if (i & (1 << b)) r |= 1 << (lg - 1 - b);
        if (r > i) {
            double tr = a[2 * i], ti = a[2 * i + 1];
            a[2 * i] = a[2 * r];
            a[2 * i + 1] = a[2 * r + 1];
            a[2 * r] = tr;
            a[2 * r + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int j = 0; j < half; ++j) {
            double ang = sign * 2.0 * M_PI * (double)j / (double)len;
            double wr = cos(ang), wi = sin(ang);
            for (int base = 0; base < n; base += len) {
                int p = base + j, q = p + half;
                double xr = a[2 * q] * wr - a[2 * q + 1] * wi;
                double xi = a[2 * q] * wi + a[2 * q + 1] * wr;
                a[2 * q] = a[2 * p] - xr;
                a[2 * q + 1] = a[2 * p + 1] - xi;
                a[2 * p] += xr;
                a[2 * p + 1] += xi;
            }
        }
    }
    return 0;
}

int orc_fft1d(double *a, int n, int sign)
{
    if (n <= 32) return orc_dft1d_naive(a, n, sign);
    return fft_radix2(a, n, sign);
}

/* 2-D DFT = 1-D DFT of every row, then of every column (separability). */
int orc_fft2d(double *a, int N, int sign)
{
    double *col = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    if (!col) return -1;
    for (int iy = 0; iy < N; ++iy)
        if (orc_fft1d(a + 2 * (size_t)iy * N, N, sign)) { free(col); return -1; }
    for (int ix = 0; ix < N; ++ix) {
        for (int iy = 0; iy < N; ++iy) {
            col[2 * iy] = a[2 * ((size_t)iy * N + ix)];
            col[2 * iy + 1] = a[2 * ((size_t)iy * N + ix) + 1];
        }
        if (orc_fft1d(col, N, sign)) { free(col); return -1; }
        for (int iy = 0; iy < N; ++iy) {
            a[2 * ((size_t)iy * N + ix)] = col[2 * iy];
            a[2 * ((size_t)iy * N + ix) + 1] = col[2 * iy + 1];
        }
    }
    free(col);
    return 0;
}

/* O1: FFT-order frequency of bin k in cycles/m (negative Nyquist; Q22). */
static double freq_of(int k, int N, double dx)
{
    int ks = (k < N / 2) ? k : k - N;
    return (double)ks / ((double)N * dx);
}

/* ------------------------------------------------------------------------- */
/* O2: phase power spectral density in cycles/m                               */
/* ------------------------------------------------------------------------- */

/* PAPER.md:375 (S18) for a slab of constant Cn2 (Q16): integral = cn2*dz. */
double orc_r0(double lambda, double cn2, double dz)
{
    double k = 2.0 * M_PI / lambda;
    return pow(0.423 * k * k * cn2 * dz, -3.0 / 5.0);
}

/* Nikishov oceanic index spectrum Phi_n(kappa) [open literature; Q20,
 * constants unpinned by the paper]. */
static double nikishov_phi_n(const orc_psd_t *p, double kappa)
{
    double eta = p->eta;
    if (!(eta > 0.0)) eta = pow(1e-18 / p->eps, 0.25); /* nu = 1e-6 m^2/s */
    const double AT = 1.863e-2, AS = 1.9e-4, ATS = 9.41e-3;
    double ke = kappa * eta;
    double delta = 8.284 * pow(ke, 4.0 / 3.0) + 12.978 * ke * ke;
    double w = p->w;
    double bracket = w * w * exp(-AT * delta) + exp(-AS * delta) - 2.0 * w * exp(-ATS * delta);
    return 0.388e-8 * pow(p->eps, -1.0 / 3.0) * pow(kappa, -11.0 / 3.0) *
           (1.0 + 2.35 * pow(ke, 2.0 / 3.0)) * (p->chi_T / (w * w)) * bracket;
}

/* Phi^f(f; dz).  Atmosphere: PAPER.md:370 (S17) evaluated with f in cycles/m,
 * f0 = 1/L0, fm = kappa_m/(2 pi) (Q4, Q5); Kolmogorov = L0 -> inf, l0 -> 0
 * (Table S1; Q23).  Ocean: thin-screen projection
 * Phi_phi(kappa) = 2 pi k^2 dz Phi_n(kappa) (PAPER.md:346 S14 up to its
 * constant) converted to cycles/m: Phi^f(f) = (2 pi)^3 k^2 dz Phi_n(2 pi f).
 * Phi^f(0) := 0 (piston removed). */
double orc_psd_f(const orc_psd_t *psd, double lambda, double cn2, double dz, double f)
{
    if (!(f > 0.0)) return 0.0;
    if (psd->kind == ORC_PSD_KOLMOGOROV) {
        double r0 = orc_r0(lambda, cn2, dz);
        return 0.023 * pow(r0, -5.0 / 3.0) * pow(f, -11.0 / 3.0);
    }
    if (psd->kind == ORC_PSD_VON_KARMAN) {
        double r0 = orc_r0(lambda, cn2, dz);
        double kmc = (psd->km_coeff > 0.0) ? psd->km_coeff : 2.0 * M_PI;
        double f0 = 1.0 / psd->L0;
        double fm = kmc / (2.0 * M_PI * psd->l0);
        return 0.023 * pow(r0, -5.0 / 3.0) * exp(-(f * f) / (fm * fm)) /
               pow(f * f + f0 * f0, 11.0 / 6.0);
    }
    if (psd->kind == ORC_PSD_OCEAN_NIKISHOV) {
        double k = 2.0 * M_PI / lambda;
        double twopi = 2.0 * M_PI;
        return twopi * twopi * twopi * k * k * dz * nikishov_phi_n(psd, twopi * f);
    }
    if (psd->kind == ORC_PSD_POWER_LAW) {
        /* General power-law medium (PAPER.md:331 S12, Table S1): Phi_n(kappa) = A kappa^-alpha, with the
         * same optional outer / inner scale roll-offs as S17:
         *   Phi_n = A (kappa^2 + kappa0^2)^(-alpha/2) exp(-kappa^2/kappam^2),
         * kappa0 = 2 pi/L0 (L0 <= 0: none), kappam = km_coeff/l0 (l0 <= 0: none); projected like the ocean
         * spectrum: Phi^f(f) = (2 pi)^3 k^2 dz Phi_n(2 pi f) (PAPER.md:346 S14).  cn2 is not used. */
        double k = 2.0 * M_PI / lambda;
        double twopi = 2.0 * M_PI;
        double kap = twopi * f;
        double kap0 = (psd->L0 > 0.0) ? twopi / psd->L0 : 0.0;
        double phin = psd->A * pow(kap * kap + kap0 * kap0, -0.5 * psd->alpha);
        if (psd->l0 > 0.0) {
            double kmc = (psd->km_coeff > 0.0) ? psd->km_coeff : 2.0 * M_PI;
            double kapm = kmc / psd->l0;
            phin *= exp(-(kap * kap) / (kapm * kapm));
        }
        return twopi * twopi * twopi * k * k * dz * phin;
    }
    return 0.0;
}

/* ------------------------------------------------------------------------- */
/* O3-O4: screen synthesis                                                    */
/* ------------------------------------------------------------------------- */

/* index into sh_coef / noise_sh: [p][a][b], a <-> y multiplier a-1, b <-> x multiplier b-1 */
#define SH_IDX(p, a, b) ((((p) * 3) + (a)) * 3 + (b))

/* One screen from its stored spectrum and subharmonic coefficients.
 * phi_hi = Re sum_k C[ky,kx] exp(+i 2 pi (kx ix + ky iy)/N)   (PAPER.md:359 S16; Q3, Q6)
 * phi_lo = sum_p sum_{m,n} Re{ c exp(i 2 pi (n df_p x + m df_p y)) }  (Eq.2; Q7)
 * phi = phi_hi + (phi_lo - mean phi_lo)                          (PAPER.md:63 Eq.3, :362) */
/* part = 0: the real part of the synthesis (the screen, Q3); part = 1: its imaginary part, a second screen
 * with the same statistics drawn from the same noise (the part Q3 discards). */
static int synth_part(int N, double dx, int n_sh, const double *C, const double *shc,
                      double *phi, double *work, int part)
{
    size_t px = (size_t)N * N;
    memcpy(work, C, sizeof(double) * 2 * px);
    if (orc_fft2d(work, N, +1)) return -1;
    for (size_t i = 0; i < px; ++i) phi[i] = work[2 * i + part];
    if (n_sh > 0) {
        double df = 1.0 / ((double)N * dx);
        double *lo = (double *)calloc(px, sizeof(double));
        if (!lo) return -1;
        double dfp = df;
        for (int p = 0; p < n_sh; ++p) {
            dfp /= 3.0;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) {
                    if (a == 1 && b == 1) continue;
                    double cr = shc[2 * SH_IDX(p, a, b)], ci = shc[2 * SH_IDX(p, a, b) + 1];
                    double fy = (a - 1) * dfp, fx = (b - 1) * dfp;
                    for (int iy = 0; iy < N; ++iy) {
                        double y = (iy - N / 2) * dx;
                        for (int ix = 0; ix < N; ++ix) {
                            double x = (ix - N / 2) * dx;
                            double ang = 2.0 * M_PI * (fx * x + fy * y);
                            lo[(size_t)iy * N + ix] += part ? cr * sin(ang) + ci * cos(ang)
                                                            : cr * cos(ang) - ci * sin(ang);
                        }
                    }
                }
        }
        double mean = 0.0;
        for (size_t i = 0; i < px; ++i) mean += lo[i];
        mean /= (double)px;
        for (size_t i = 0; i < px; ++i) phi[i] += lo[i] - mean;
        free(lo);
    }
    return 0;
}

static int synth_one(int N, double dx, int n_sh, const double *C, const double *shc,
                     double *phi, double *work)
{
    return synth_part(N, dx, n_sh, C, shc, phi, work, 0);
}

int orc_synthesize_im(int N, double dx, int B, int S, int n_sh,
                      const double *spectrum, const double *sh_coef, double *screens)
{
    size_t px = (size_t)N * N;
    double *work = (double *)malloc(sizeof(double) * 2 * px);
    if (!work) return -1;
    for (int bs = 0; bs < B * S; ++bs) {
        const double *shc = (n_sh > 0) ? sh_coef + 2 * (size_t)bs * n_sh * 9 : NULL;
        if (synth_part(N, dx, n_sh, spectrum + 2 * (size_t)bs * px, shc,
                       screens + (size_t)bs * px, work, 1)) { free(work); return -1; }
    }
    free(work);
    return 0;
}

int orc_synthesize(int N, double dx, int B, int S, int n_sh,
                   const double *spectrum, const double *sh_coef, double *screens)
{
    size_t px = (size_t)N * N;
    double *work = (double *)malloc(sizeof(double) * 2 * px);
    if (!work) return -1;
    for (int bs = 0; bs < B * S; ++bs) {
        const double *shc = (n_sh > 0) ? sh_coef + 2 * (size_t)bs * n_sh * 9 : NULL;
        if (synth_one(N, dx, n_sh, spectrum + 2 * (size_t)bs * px, shc,
                      screens + (size_t)bs * px, work)) { free(work); return -1; }
    }
    free(work);
    return 0;
}

/* Filtered noise for one screen: C = (a + i b) sqrt(Phi^f(|f|)) df, C[0,0] = 0
 * (PAPER.md:359 S16); subharmonic level p uses df_p = df/3^p (Q7). */
static void filter_noise(int N, double dx, const orc_psd_t *psd, double lambda,
                         double cn2, double dz, int n_sh,
                         const float *noise, const float *noise_sh, double *C, double *shc)
{
    double df = 1.0 / ((double)N * dx);
    for (int ky = 0; ky < N; ++ky) {
        double fy = freq_of(ky, N, dx);
        for (int kx = 0; kx < N; ++kx) {
            double fx = freq_of(kx, N, dx);
            double amp = sqrt(orc_psd_f(psd, lambda, cn2, dz, hypot(fx, fy))) * df;
            size_t i = (size_t)ky * N + kx;
            C[2 * i] = (double)noise[2 * i] * amp;
            C[2 * i + 1] = (double)noise[2 * i + 1] * amp;
        }
    }
    double dfp = df;
    for (int p = 0; p < n_sh; ++p) {
        dfp /= 3.0;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                int i = SH_IDX(p, a, b);
                if (a == 1 && b == 1) { shc[2 * i] = shc[2 * i + 1] = 0.0; continue; }
                double amp = sqrt(orc_psd_f(psd, lambda, cn2, dz,
                                            hypot((b - 1) * dfp, (a - 1) * dfp))) * dfp;
                shc[2 * i] = (double)noise_sh[2 * i] * amp;
                shc[2 * i + 1] = (double)noise_sh[2 * i + 1] * amp;
            }
    }
}

int orc_make_screens(int N, double dx, const orc_psd_t *psd, double lambda, int B, int S,
                     const double *cn2, const double *dz, int n_sh,
                     const float *noise, const float *noise_sh,
                     double *spectrum, double *sh_coef, double *screens)
{
    size_t px = (size_t)N * N;
    double *C = (double *)malloc(sizeof(double) * 2 * px);
    double *work = (double *)malloc(sizeof(double) * 2 * px);
    double *shc = (double *)calloc((size_t)(n_sh > 0 ? n_sh : 1) * 18, sizeof(double));
    if (!C || !work || !shc) { free(C); free(work); free(shc); return -1; }
    int rc = 0;
    for (int b = 0; b < B && !rc; ++b)
        for (int s = 0; s < S && !rc; ++s) {
            size_t bs = (size_t)b * S + s;
            filter_noise(N, dx, psd, lambda, cn2[s], dz[s], n_sh, noise + 2 * bs * px,
                         (n_sh > 0) ? noise_sh + 2 * bs * n_sh * 9 : NULL, C, shc);
            if (spectrum) memcpy(spectrum + 2 * bs * px, C, sizeof(double) * 2 * px);
            if (sh_coef && n_sh > 0)
                memcpy(sh_coef + 2 * bs * n_sh * 9, shc, sizeof(double) * 18 * n_sh);
            rc = synth_one(N, dx, n_sh, C, shc, screens + bs * px, work);
        }
    free(C); free(work); free(shc);
    return rc;
}

/* ------------------------------------------------------------------------- */
/* O5: autoregressive evolution on the stored spectrum                        */
/* ------------------------------------------------------------------------- */

/* C <- a * tau * C + sqrt(1 - a^2) * C_fresh   (Eq.5),
 * tau = exp(-i 2 pi T (fx vx + fy vy))          (Eq.4 with its i; Q9),
 * the subharmonic coefficients follow the same recursion with tau at their
 * fractional frequency (Q8); then resynthesise (O3-O4). */
int orc_evolve_screens(int N, double dx, const orc_psd_t *psd, double lambda, int B, int S,
                       const double *cn2, const double *dz, int n_sh,
                       double a, double vx, double vy, double T,
                       const float *fresh, const float *fresh_sh,
                       double *spectrum, double *sh_coef, double *screens)
{
    if (a < 0.0 || a > 1.0) return -2;
    size_t px = (size_t)N * N;
    double *Cf = (double *)malloc(sizeof(double) * 2 * px);
    double *work = (double *)malloc(sizeof(double) * 2 * px);
    double *shf = (double *)calloc((size_t)(n_sh > 0 ? n_sh : 1) * 18, sizeof(double));
    if (!Cf || !work || !shf) { free(Cf); free(work); free(shf); return -1; }
    double g = sqrt(1.0 - a * a);
    double df = 1.0 / ((double)N * dx);
    int rc = 0;
    for (int b = 0; b < B && !rc; ++b)
        for (int s = 0; s < S && !rc; ++s) {
            size_t bs = (size_t)b * S + s;
            double *C = spectrum + 2 * bs * px;
            double *shc = (n_sh > 0) ? sh_coef + 2 * bs * n_sh * 9 : NULL;
            filter_noise(N, dx, psd, lambda, cn2[s], dz[s], n_sh, fresh + 2 * bs * px,
                         (n_sh > 0) ? fresh_sh + 2 * bs * n_sh * 9 : NULL, Cf, shf);
            for (int ky = 0; ky < N; ++ky) {
                double fy = freq_of(ky, N, dx);
                for (int kx = 0; kx < N; ++kx) {
                    double fx = freq_of(kx, N, dx);
                    double ang = -2.0 * M_PI * T * (fx * vx + fy * vy);
                    double tr = cos(ang), ti = sin(ang);
                    size_t i = (size_t)ky * N + kx;
                    double cr = C[2 * i], ci = C[2 * i + 1];
                    C[2 * i] = a * (tr * cr - ti * ci) + g * Cf[2 * i];
                    C[2 * i + 1] = a * (tr * ci + ti * cr) + g * Cf[2 * i + 1];
                }
            }
            double dfp = df;
            for (int p = 0; p < n_sh; ++p) {
                dfp /= 3.0;
                for (int aa = 0; aa < 3; ++aa)
                    for (int bb = 0; bb < 3; ++bb) {
                        int i = SH_IDX(p, aa, bb);
                        double ang = -2.0 * M_PI * T * ((bb - 1) * dfp * vx + (aa - 1) * dfp * vy);
                        double tr = cos(ang), ti = sin(ang);
                        double cr = shc[2 * i], ci = shc[2 * i + 1];
                        shc[2 * i] = a * (tr * cr - ti * ci) + g * shf[2 * i];
                        shc[2 * i + 1] = a * (tr * ci + ti * cr) + g * shf[2 * i + 1];
                    }
            }
            rc = synth_one(N, dx, n_sh, C, shc, screens + bs * px, work);
        }
    free(Cf); free(work); free(shf);
    return rc;
}

/* ------------------------------------------------------------------------- */
/* O6-O7: split-step propagation and its adjoint                              */
/* ------------------------------------------------------------------------- */

/* Transfer function of one diffraction step at bin (ky,kx).
 * Fresnel (north_star; named as the alternative at PAPER.md:39):
 *   H = exp(-i pi (lambda/n0) dz (fx^2 + fy^2))
 * Angular spectrum (Eq.6) with the unobservable carrier
 * exp(i dz n k0) removed (Q2):  H = exp(i dz (sqrt(km^2 - kappa^2) - km)),
 * km = 2 pi n0 / lambda, kappa = 2 pi |f|; evanescent bins (kappa > km) -> 0. */
static void transfer(int h_kind, double lambda, double n0, double dz, double fx, double fy,
                     double *hr, double *hi)
{
    double f2 = fx * fx + fy * fy;
    if (h_kind == ORC_H_FRESNEL) {
        double ang = -M_PI * (lambda / n0) * dz * f2;
        *hr = cos(ang);
        *hi = sin(ang);
    } else {
        double km = 2.0 * M_PI * n0 / lambda;
        double kap2 = 4.0 * M_PI * M_PI * f2;
        if (kap2 > km * km) { *hr = 0.0; *hi = 0.0; return; }
        /* sqrt(km^2-kap2) - km = -kap2 / (km + sqrt(km^2-kap2)) : same value, no cancellation */
        double ang = -dz * kap2 / (km + sqrt(km * km - kap2));
        *hr = cos(ang);
        *hi = sin(ang);
    }
}

/* Super-Gaussian absorbing window (not in the paper; north_star + Q12):
 *   W = exp(-((x^2 + y^2)/sigma^2)^(order/2)), sigma = sigma_frac * N * dx; order 0 -> 1. */
static double window_at(int order, double sigma_frac, int N, double dx, int iy, int ix)
{
    if (order <= 0) return 1.0;
    double x = (ix - N / 2) * dx, y = (iy - N / 2) * dx;
    double sig = sigma_frac * N * dx;
    return exp(-pow((x * x + y * y) / (sig * sig), 0.5 * order));
}

/* multiply spectrum by H (conj=0) or conj(H) (conj=1) */
static void apply_h(double *a, int N, double dx, int h_kind, double lambda, double n0,
                    double dz, int conj)
{
    for (int ky = 0; ky < N; ++ky) {
        double fy = freq_of(ky, N, dx);
        for (int kx = 0; kx < N; ++kx) {
            double fx = freq_of(kx, N, dx);
            double hr, hi;
            transfer(h_kind, lambda, n0, dz, fx, fy, &hr, &hi);
            if (conj) hi = -hi;
            size_t i = (size_t)ky * N + kx;
            double ur = a[2 * i], ui = a[2 * i + 1];
            a[2 * i] = ur * hr - ui * hi;
            a[2 * i + 1] = ur * hi + ui * hr;
        }
    }
}

/* U <- IDFT2( Hmul * DFT2(U) ) with the true inverse (1/N^2). */
static int diffract(double *u, int N, double dx, int h_kind, double lambda, double n0,
                    double dz, int conj)
{
    if (orc_fft2d(u, N, -1)) return -1;
    apply_h(u, N, dx, h_kind, lambda, n0, dz, conj);
    if (orc_fft2d(u, N, +1)) return -1;
    double inv = 1.0 / ((double)N * (double)N);
    for (size_t i = 0; i < 2 * (size_t)N * N; ++i) u[i] *= inv;
    return 0;
}

/* For j = 1..n_steps: U <- F^-1{F{U} H_j};  if j <= S: U <- U exp(i phi_j);  U <- U W
 * (Eq.1; step order Q11; window Q12).  planes[b][j-1] = U after step j. */
int orc_propagate(int N, double dx, double lambda, double n0, int B, int n_steps,
                  const double *dz, const double *screens, long long screen_batch_stride,
                  int S, int win_order, double win_sigma_frac, int h_kind,
                  const double *field_in, double *field_out, double *planes)
{
    size_t px = (size_t)N * N;
    if (S > n_steps) return -2;
    for (int b = 0; b < B; ++b) {
        double *u = field_out + 2 * (size_t)b * px;
        if (u != field_in + 2 * (size_t)b * px)
            memcpy(u, field_in + 2 * (size_t)b * px, sizeof(double) * 2 * px);
        for (int j = 1; j <= n_steps; ++j) {
            if (diffract(u, N, dx, h_kind, lambda, n0, dz[j - 1], 0)) return -1;
            const double *phi = (j <= S)
                ? screens + (size_t)b * (size_t)screen_batch_stride + (size_t)(j - 1) * px : NULL;
            for (int iy = 0; iy < N; ++iy)
                for (int ix = 0; ix < N; ++ix) {
                    size_t i = (size_t)iy * N + ix;
                    double ur = u[2 * i], ui = u[2 * i + 1];
                    if (phi) {
                        double c = cos(phi[i]), s = sin(phi[i]);
                        double tr = ur * c - ui * s;
                        ui = ur * s + ui * c;
                        ur = tr;
                    }
                    double w = window_at(win_order, win_sigma_frac, N, dx, iy, ix);
                    u[2 * i] = ur * w;
                    u[2 * i + 1] = ui * w;
                }
            if (planes)
                memcpy(planes + 2 * ((size_t)b * n_steps + (j - 1)) * px, u, sizeof(double) * 2 * px);
        }
    }
    return 0;
}

/* Adjoint (conjugate transpose) of orc_propagate (O7; north_star):
 * for j = n_steps..1:  [grad_j = Im(G_j conj(U_j))];  g <- W g;  if j <= S: g <- exp(-i phi_j) g;
 *                      g <- F^-1{ conj(H_j) F{g} }.
 * G_j is the adjoint field arriving at plane j (before the W exp(-i phi_j) multiply) and
 * U_j = planes[b][j-1] the forward field after step j.  Gradient convention
 * G = dl/dRe U + i dl/dIm U. */
int orc_propagate_adjoint(int N, double dx, double lambda, double n0, int B, int n_steps,
                          const double *dz, const double *screens, long long screen_batch_stride,
                          int S, int win_order, double win_sigma_frac, int h_kind,
                          const double *g_out, double *g_in,
                          const double *planes, double *phase_grad)
{
    size_t px = (size_t)N * N;
    if (S > n_steps) return -2;
    for (int b = 0; b < B; ++b) {
        double *g = g_in + 2 * (size_t)b * px;
        if (g != g_out + 2 * (size_t)b * px)
            memcpy(g, g_out + 2 * (size_t)b * px, sizeof(double) * 2 * px);
        for (int j = n_steps; j >= 1; --j) {
            const double *phi = (j <= S)
                ? screens + (size_t)b * (size_t)screen_batch_stride + (size_t)(j - 1) * px : NULL;
            if (planes && phase_grad && j <= S) {
                const double *u = planes + 2 * ((size_t)b * n_steps + (j - 1)) * px;
                double *gr = phase_grad + ((size_t)b * S + (j - 1)) * px;
                for (size_t i = 0; i < px; ++i)
                    gr[i] = g[2 * i + 1] * u[2 * i] - g[2 * i] * u[2 * i + 1];
            }
            for (int iy = 0; iy < N; ++iy)
                for (int ix = 0; ix < N; ++ix) {
                    size_t i = (size_t)iy * N + ix;
                    double w = window_at(win_order, win_sigma_frac, N, dx, iy, ix);
                    double gr = g[2 * i] * w, gi = g[2 * i + 1] * w;
                    if (phi) {
                        double c = cos(phi[i]), s = -sin(phi[i]);
                        double tr = gr * c - gi * s;
                        gi = gr * s + gi * c;
                        gr = tr;
                    }
                    g[2 * i] = gr;
                    g[2 * i + 1] = gi;
                }
            if (diffract(g, N, dx, h_kind, lambda, n0, dz[j - 1], 1)) return -1;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O8: per-realisation intensity statistics                                   */
/* ------------------------------------------------------------------------- */

/* I = |U|^2; P = sum I dx^2; centroid; central second moments; w2 = sqrt(2(sxx+syy))
 * (equals w for I ~ exp(-2 r^2/w^2), PAPER.md:402 S22); on-axis I; ROI sums for the
 * spatial scintillation index n sum I^2/(sum I)^2 - 1 (PAPER.md:423 S25).
 * ROI = [N/2-h, N/2+h)^2 with h = floor(roi_frac*N/2); h = 0 -> the single pixel N/2. */
int orc_beam_stats(int N, double dx, int B, const double *field, double roi_frac,
                   orc_stats_t *stats)
{
    size_t px = (size_t)N * N;
    int h = (int)floor(roi_frac * N / 2.0);
    int lo = N / 2 - h, hi = N / 2 + h;
    if (h <= 0) { lo = N / 2; hi = N / 2 + 1; }
    if (lo < 0) lo = 0;
    if (hi > N) hi = N;
    for (int b = 0; b < B; ++b) {
        const double *u = field + 2 * (size_t)b * px;
        double sI = 0, sx = 0, sy = 0;
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                size_t i = (size_t)iy * N + ix;
                double I = u[2 * i] * u[2 * i] + u[2 * i + 1] * u[2 * i + 1];
                sI += I;
                sx += (ix - N / 2) * dx * I;
                sy += (iy - N / 2) * dx * I;
            }
        orc_stats_t *st = stats + b;
        memset(st, 0, sizeof(*st));
        st->power = sI * dx * dx;
        double cx = (sI > 0) ? sx / sI : 0.0, cy = (sI > 0) ? sy / sI : 0.0;
        double sxx = 0, syy = 0, sxy = 0, rI = 0, rI2 = 0;
        long long rn = 0;
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                size_t i = (size_t)iy * N + ix;
                double I = u[2 * i] * u[2 * i] + u[2 * i + 1] * u[2 * i + 1];
                double x = (ix - N / 2) * dx - cx, y = (iy - N / 2) * dx - cy;
                sxx += x * x * I;
                syy += y * y * I;
                sxy += x * y * I;
                if (iy >= lo && iy < hi && ix >= lo && ix < hi) { rI += I; rI2 += I * I; ++rn; }
            }
        st->cx = cx;
        st->cy = cy;
        if (sI > 0) { st->sxx = sxx / sI; st->syy = syy / sI; st->sxy = sxy / sI; }
        st->w2 = sqrt(2.0 * (st->sxx + st->syy));
        size_t ic = (size_t)(N / 2) * N + N / 2;
        st->I_axis = u[2 * ic] * u[2 * ic] + u[2 * ic + 1] * u[2 * ic + 1];
        st->roi_sumI = rI;
        st->roi_sumI2 = rI2;
        st->roi_n = rn;
    }
    return 0;
}

/* Welford one-pass mean / M2 of the intensity per pixel across realisations
 * (PAPER.md:143): count += 1; d = I - mean; mean += d/count; M2 += d (I - mean). */
int orc_welford(int N, int B, const double *field, double *mean, double *M2, long long *count)
{
    size_t px = (size_t)N * N;
    for (int b = 0; b < B; ++b) {
        const double *u = field + 2 * (size_t)b * px;
        *count += 1;
        for (size_t i = 0; i < px; ++i) {
            double I = u[2 * i] * u[2 * i] + u[2 * i + 1] * u[2 * i + 1];
            double d = I - mean[i];
            mean[i] += d / (double)(*count);
            M2[i] += d * (I - mean[i]);
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O9 helpers: phase mask, centred unitary DFT, phase gradient                */
/* ------------------------------------------------------------------------- */

/* out = in * exp(i sign theta); theta is one [N][N] mask shared by the batch. */
int orc_phase_mul(int N, int B, const double *theta, double sign, const double *in, double *out)
{
    size_t px = (size_t)N * N;
    for (int b = 0; b < B; ++b)
        for (size_t i = 0; i < px; ++i) {
            double c = cos(theta[i]), s = sign * sin(theta[i]);
            double ur = in[2 * ((size_t)b * px + i)], ui = in[2 * ((size_t)b * px + i) + 1];
            out[2 * ((size_t)b * px + i)] = ur * c - ui * s;
            out[2 * ((size_t)b * px + i) + 1] = ur * s + ui * c;
        }
    return 0;
}

/* Lens as a DFT: centred unitary transform
 * F_c = fftshift o fft2 o ifftshift / N ; inverse: fftshift o ifft2 o ifftshift * N / N^2. */
int orc_dft2_centered(int N, int B, int inverse, const double *in, double *out)
{
    size_t px = (size_t)N * N;
    double *t = (double *)malloc(sizeof(double) * 2 * px);
    if (!t) return -1;
    int h = N / 2;
    for (int b = 0; b < B; ++b) {
        const double *src = in + 2 * (size_t)b * px;
        double *dst = out + 2 * (size_t)b * px;
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                size_t s = (size_t)((iy + h) % N) * N + (ix + h) % N; /* ifftshift */
                size_t d = (size_t)iy * N + ix;
                t[2 * d] = src[2 * s];
                t[2 * d + 1] = src[2 * s + 1];
            }
        if (orc_fft2d(t, N, inverse ? +1 : -1)) { free(t); return -1; }
        double sc = 1.0 / (double)N;
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                size_t s = (size_t)((iy + N - h) % N) * N + (ix + N - h) % N; /* fftshift */
                size_t d = (size_t)iy * N + ix;
                dst[2 * d] = t[2 * s] * sc;
                dst[2 * d + 1] = t[2 * s + 1] * sc;
            }
    }
    free(t);
    return 0;
}

/* grad = Im(g conj(u)) per pixel, summed over nothing (one map per batch entry). */
int orc_aperture(int N, int B, long long r2max_px, const double *in, double *out)
{
    for (int b = 0; b < B; ++b)
        for (int iy = 0; iy < N; ++iy)
            for (int ix = 0; ix < N; ++ix) {
                long long x = ix - N / 2, y = iy - N / 2;
                size_t i = ((size_t)b * N + iy) * N + ix;
                int inside = (x * x + y * y <= r2max_px);
                out[2 * i] = inside ? in[2 * i] : 0.0;
                out[2 * i + 1] = inside ? in[2 * i + 1] : 0.0;
            }
    return 0;
}

int orc_phase_grad(int N, int B, const double *g, const double *u, double *grad)
{
    size_t n = (size_t)B * N * N;
    for (size_t i = 0; i < n; ++i)
        grad[i] = g[2 * i + 1] * u[2 * i] - g[2 * i] * u[2 * i + 1];
    return 0;
}
