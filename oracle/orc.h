/*
 * orc.h -- CPU ORACLE for the split-step phase-screen propagation path.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product: only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.  It shares no code, header, table or
 * constant generator with the CUDA path in paper_2604_07248_b200/csrc.
 *
 * Plain C, double precision, single thread, no blocking / fusion / reordering
 * beyond what the cited definition states.  Citations are "PAPER.md:<line>"
 * (the TurPy paper text) plus the equation; readings of silent or garbled
 * passages are the numbered "Q" rows of SURVEY.md section 8(c), restated in
 * DESIGN.md section 3.
 *
 * Conventions (SURVEY.md section 8 preamble):
 *   arrays row-major, x fastest:  idx = ((b*S + s)*N + iy)*N + ix
 *   complex = interleaved (re, im) doubles;  noise inputs are float32 pairs
 *   x_i = (i - N/2)*dx ;  f_k = k/(N dx) for k < N/2, (k-N)/(N dx) otherwise
 *   forward DFT  X[k] = sum_n x[n] exp(-i 2 pi k n / N)   (unnormalised)
 *   inverse carries 1/N per axis where the definition needs a true inverse.
 *
 * Pins (tests/test_oracle_*.py): P0 FFT vs naive DFT / numpy; P1 Gaussian beam
 * width; P1b power conservation; P2 structure function; P3 filter amplitude;
 * P4 analytic mean; P5 Rytov scintillation; P6 AR recursion (incl. the
 * subharmonic coefficients under wind: the closed-form moved sinusoid); P7
 * adjoint identity; P8 finite-difference gradients; the non-paraxial term of
 * Eq. 6 on a tilted plane wave against 50-digit arithmetic; Philox-4x32-10
 * against its authors' known-answer vectors.
 * PARITY UNPINNED BY THE PAPER (defined by the survey / the open literature,
 * not by PAPER.md): the Nikishov oceanic constants (Q20; re-typed with their
 * source in tests/golden/nikishov_constants.txt and checked against that
 * file, which catches a typo but is not a pin by the paper), the
 * super-Gaussian window form (Q12), the config-4 beam (Q21).
 */
#ifndef ORC_H
#define ORC_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_PSD_KOLMOGOROV = 0, ORC_PSD_VON_KARMAN = 1, ORC_PSD_OCEAN_NIKISHOV = 2, ORC_PSD_POWER_LAW = 3 };
enum { ORC_H_FRESNEL = 0, ORC_H_ANGULAR_SPECTRUM = 1 };

typedef struct {
    int kind;            /* ORC_PSD_* */
    double L0, l0;       /* outer / inner scale [m]; von Karman only */
    double km_coeff;     /* kappa_m = km_coeff / l0 ; <=0 -> 2 pi */
    double chi_T, eps, w, eta; /* ocean: eta<=0 -> (nu^3/eps)^(1/4), nu = 1e-6 */
    double alpha, A;     /* power law (PAPER.md:331 S12, Table S1): Phi_n = A kappa^-alpha */
} orc_psd_t;

typedef struct {
    double power, cx, cy, sxx, syy, sxy, w2, I_axis, roi_sumI, roi_sumI2;
    long long roi_n;
} orc_stats_t;

/* P0: unnormalised DFT of a length-n complex line, sign=-1 forward, +1 inverse
 * (no 1/n).  n<=32 -> naive O(n^2) definition; else iterative radix-2. */
int orc_fft1d(double *a, int n, int sign);
int orc_dft1d_naive(double *a, int n, int sign);
int orc_fft2d(double *a, int N, int sign);

/* O2: phase PSD in cycles/m, Phi^f(f; dz) (PAPER.md:370 S17, :375 S18, :346 S14). */
double orc_r0(double lambda, double cn2, double dz);
double orc_psd_f(const orc_psd_t *psd, double lambda, double cn2, double dz, double f);

/* O3-O4 (PAPER.md:359 S16, :57 Eq.2, :63 Eq.3, :362). */
int orc_make_screens(int N, double dx, const orc_psd_t *psd, double lambda, int B, int S,
                     const double *cn2, const double *dz, int n_sh,
                     const float *noise, const float *noise_sh,
                     double *spectrum, double *sh_coef, double *screens);
/* synthesis only: spectrum [B][S][N][N] c128 + sh_coef [B][S][n_sh][3][3] c128 -> screens */
int orc_synthesize(int N, double dx, int B, int S, int n_sh,
                   const double *spectrum, const double *sh_coef, double *screens);
/* The imaginary part of the same synthesis: a second, statistically independent screen from the same spectrum. */
int orc_synthesize_im(int N, double dx, int B, int S, int n_sh,
                      const double *spectrum, const double *sh_coef, double *screens);
/* O5 (PAPER.md:74 Eq.4, :80 Eq.5). spectrum / sh_coef are in-out. */
int orc_evolve_screens(int N, double dx, const orc_psd_t *psd, double lambda, int B, int S,
                       const double *cn2, const double *dz, int n_sh,
                       double a, double vx, double vy, double T,
                       const float *fresh, const float *fresh_sh,
                       double *spectrum, double *sh_coef, double *screens);

/* O6 (PAPER.md:37 Eq.1, :96 Eq.6). planes/stats may be NULL. */
int orc_propagate(int N, double dx, double lambda, double n0, int B, int n_steps,
                  const double *dz, const double *screens, long long screen_batch_stride,
                  int S, int win_order, double win_sigma_frac, int h_kind,
                  const double *field_in, double *field_out, double *planes);
/* O7. planes / phase_grad may be NULL (both or neither). */
int orc_propagate_adjoint(int N, double dx, double lambda, double n0, int B, int n_steps,
                          const double *dz, const double *screens, long long screen_batch_stride,
                          int S, int win_order, double win_sigma_frac, int h_kind,
                          const double *g_out, double *g_in,
                          const double *planes, double *phase_grad);
/* O8 (PAPER.md:423 S25, :143). */
int orc_beam_stats(int N, double dx, int B, const double *field, double roi_frac,
                   orc_stats_t *stats);
/* Welford per-pixel ensemble update over B fields. */
int orc_welford(int N, int B, const double *field, double *mean, double *M2, long long *count);

/* O9 helpers (config 4). */
int orc_phase_mul(int N, int B, const double *theta, double sign, const double *in, double *out);
int orc_dft2_centered(int N, int B, int inverse, const double *in, double *out);
int orc_phase_grad(int N, int B, const double *g, const double *u, double *grad);
/* Circular receiver aperture: out = in where (ix-N/2)^2 + (iy-N/2)^2 <= r2max_px, else 0.
 * r2max_px = floor((radius/dx)^2) is decided by the caller in double (an integer decision). */
int orc_aperture(int N, int B, long long r2max_px, const double *in, double *out);

#ifdef __cplusplus
}
#endif
#endif
