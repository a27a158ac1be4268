/*
 * ssp.h -- C ABI of the B200-native split-step phase-screen propagation library.
 *
 * The product boundary.  Every entry point is `extern "C"`, takes plain pointers and
 * sizes (no torch types) and runs entirely in hand-written sm_100a CUDA kernels; there
 * is no CPU fallback.  Citations are "PAPER.md:<line>" of the TurPy paper
 * (arxiv 2604.07248) plus the equation; "Qn" are the readings listed in DESIGN.md
 * section 3.
 *
 * Conventions
 *   - Grids are square, N a power of two, 8 <= N <= 4096.  Arrays are row-major with x
 *     fastest: idx = ((b*S + s)*N + iy)*N + ix.  complex64 = interleaved (re, im) fp32.
 *   - Coordinates x_i = (i - N/2) dx.  Frequencies are in cycles/m in FFT order with the
 *     negative Nyquist: f_k = k/(N dx) for k < N/2, (k - N)/(N dx) otherwise.
 *   - Forward DFT X[k] = sum_n x[n] exp(-i 2 pi k n / N), unnormalised.
 *   - "dev" pointers are device memory of the context's device, 16-byte aligned, owned by
 *     the caller (allocate them with torch / cudaMalloc); "host" pointers are read during
 *     the call and not retained.  The library allocates only tables inside the context
 *     (twiddles, transfer-function tables, at N = 1024 up to 8 cached window maps of 4 MB)
 *     and frees them in ssp_destroy.
 *   - Calls enqueue work on the context's stream and return without synchronising,
 *     except the *_host entry points, which synchronise the stream before returning.
 *   - CUDA graphs: ssp_propagate, ssp_propagate_adjoint and ssp_beam_stats_static may be captured
 *     (cudaStreamBeginCapture on the context's stream) after ONE call with the same arguments
 *     outside capture: by then tables, TMA descriptors and the on-chip step list are cached and the
 *     call issues kernels (and one memset) only.  A first-time call under capture returns
 *     SSP_EUNSUPPORTED / SSP_ECUDA.  The screen generators upload small tables every call and are
 *     not capturable.
 *   - Return value: 0 on success, a negative ssp_status otherwise; ssp_last_error gives
 *     the text.  After an error no output buffer is guaranteed.  No exception crosses
 *     the ABI.  A context is not thread-safe.
 */
#ifndef SSP_H
#define SSP_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SSP_OK = 0,
    SSP_EINVAL = -1,        /* bad argument: N not a power of two or out of range, null
                               required pointer, S < 0, S > n_steps, a not in [0,1],
                               lambda <= 0, dz <= 0, misaligned pointer */
    SSP_EUNSUPPORTED = -2,  /* valid request this build does not implement */
    SSP_EWORKSPACE = -3,    /* workspace smaller than ssp_workspace_bytes */
    SSP_ECUDA = -4          /* CUDA runtime / driver error (text in ssp_last_error) */
} ssp_status;

typedef struct ssp_ctx ssp_ctx; /* opaque; one per (device, stream) */

typedef struct { int N; double dx; } ssp_grid;

typedef enum {
    SSP_PSD_KOLMOGOROV = 0,     /* Table S1: S17 with L0 -> inf, l0 -> 0 (Q23) */
    SSP_PSD_VON_KARMAN = 1,     /* modified von Karman, PAPER.md:370 (S17) */
    SSP_PSD_OCEAN_NIKISHOV = 2, /* Nikishov oceanic spectrum, open literature (Q20) */
    SSP_PSD_POWER_LAW = 3       /* general power-law medium, PAPER.md:331 (S12), Table S1 */
} ssp_psd_kind;

/* Phase PSD parameters.  Atmospheric kinds evaluate S17 with f in cycles/m:
 *   Phi^f(f) = 0.023 r0^(-5/3) exp(-f^2/fm^2) / (f^2 + f0^2)^(11/6),
 *   f0 = 1/L0, fm = km_coeff/(2 pi l0) (km_coeff <= 0 -> 2 pi; Q4, Q5),
 *   r0 = (0.423 k^2 Cn2 dz)^(-3/5), k = 2 pi/lambda (PAPER.md:375 S18; Q16).
 * Ocean: Phi^f(f) = (2 pi)^3 k^2 dz Phi_n(2 pi f) with Nikishov's Phi_n; cn2 is ignored;
 *   eta <= 0 -> (nu^3/eps)^(1/4), nu = 1e-6 m^2/s.
 * Power law: Phi_n(kappa) = A (kappa^2 + kappa0^2)^(-alpha/2) exp(-kappa^2/kappam^2), 3 <= alpha < 5,
 *   kappa0 = 2 pi/L0 (L0 <= 0: none), kappam = km_coeff/l0 (l0 <= 0: none), projected like the ocean
 *   spectrum; cn2 is ignored.  alpha = 11/3, A = 0.033 Cn2 is the atmospheric case. */
typedef struct {
    int kind;                  /* ssp_psd_kind */
    double L0, l0, km_coeff;   /* von Karman, power law */
    double chi_T, eps, w, eta; /* ocean */
    double alpha, A;           /* power law */
} ssp_psd;

/* Super-Gaussian absorbing window applied after every split step (north_star; Q12):
 *   W = exp(-((x^2 + y^2)/sigma^2)^(order/2)), sigma = sigma_frac N dx; order <= 0 -> off. */
typedef struct { int order; double sigma_frac; } ssp_window;

/* Per-realisation intensity statistics (PAPER.md:423 S25, :402 S22; O8 in DESIGN.md):
 *   power = sum I dx^2; (cx, cy) centroid; sxx, syy, sxy central second moments [m^2];
 *   w2 = sqrt(2 (sxx + syy)) (= w for I ~ exp(-2 r^2/w^2)); I_axis = I[N/2][N/2];
 *   ROI = [N/2 - h, N/2 + h)^2, h = floor(roi_frac N / 2) (h = 0 -> the pixel N/2):
 *   roi_sumI, roi_sumI2, roi_n  ->  spatial SI = roi_n roi_sumI2 / roi_sumI^2 - 1. */
typedef struct {
    double power, cx, cy, sxx, syy, sxy, w2, I_axis, roi_sumI, roi_sumI2;
    long long roi_n;
} ssp_stats;

/* Transfer function of the diffraction step (Q1). */
typedef enum {
    SSP_H_FRESNEL = 0,          /* H = exp(-i pi (lambda/n0) dz (fx^2 + fy^2))  (north_star) */
    SSP_H_ANGULAR_SPECTRUM = 1  /* PAPER.md:96 Eq.6, carrier removed (Q2): H = exp(i dz (sqrt(km^2 - kappa^2) - km)),
                                   km = 2 pi n0 / lambda, kappa = 2 pi |f|; evanescent bins -> 0.  Not separable: the
                                   context caches one complex64 map [N][N] per distinct (dz, conj) */
} ssp_h_kind;

/* ---- context ------------------------------------------------------------------- */

/* Create a context bound to `device` and to `cuda_stream` (a cudaStream_t passed as
 * void*; NULL = the legacy default stream).  Fails with SSP_ECUDA when no CUDA device
 * is usable.  The stream must outlive the context. */
int ssp_create(ssp_ctx **out, int device, void *cuda_stream);
int ssp_destroy(ssp_ctx *ctx);
/* Text of the last error on this context ("" if none); valid until the next call. */
const char *ssp_last_error(const ssp_ctx *ctx);
/* Library version string, e.g. "ssp 0.1 sm_100a". */
const char *ssp_version(void);
/* Number of kernels this context has launched since creation (bench bookkeeping). */
long long ssp_launch_count(const ssp_ctx *ctx);

/* Per-launch timing for measurement: while enabled, every kernel launch is bracketed by CUDA
 * events on the context's stream.  ssp_profile_report synchronises the stream, writes one line
 * per kernel class "name launches total_ms algorithmic_bytes\n" into buf (host) and clears the
 * records.  Enabling or disabling also clears them. */
int ssp_profile_enable(ssp_ctx *ctx, int on);
int ssp_profile_report(ssp_ctx *ctx, char *buf, size_t buf_bytes);

/* Bytes of device scratch any call on this (grid, B, S) may need; the caller allocates
 * it once and passes it to every call.  Independent of the context. */
size_t ssp_workspace_bytes(ssp_grid grid, int B, int S);

/* ---- screens ------------------------------------------------------------------- */

/* Screen generator (PAPER.md:359 S16; :57 Eq.2; :63 Eq.3; :362):
 *   C[ky][kx] = (a + i b) sqrt(Phi^f(|f|; dz_s)) df,  C[0][0] = 0,  df = 1/(N dx);
 *   phi_hi    = Re sum_k C[ky][kx] exp(+i 2 pi (kx ix + ky iy)/N)   (unnormalised; Q3, Q6);
 *   c_pab     = (a + i b) sqrt(Phi^f(|(b-1, a-1)| df_p)) df_p, df_p = df/3^p, p = 1..n_sh (Q7);
 *   phi_lo    = sum_p sum_{a,b != centre} Re{ c_pab exp(i 2 pi ((b-1) df_p x + (a-1) df_p y)) };
 *   phi       = phi_hi + phi_lo - mean(phi_lo).
 * cn2, dz: host [S] (one slab per screen).  d_noise: dev complex64 [B][S][N][N] of
 * N(0,1)+iN(0,1) draws; d_noise_sh: dev complex64 [B][S][n_sh][3][3] ([a][b], centre
 * unused), may be NULL when n_sh == 0.  Outputs: d_spectrum dev complex64 [B][S][N][N]
 * (the stored Fourier spectrum; may be NULL), d_sh_coef dev complex64
 * [B][S][n_sh][3][3] (may be NULL), d_screens dev fp32 [B][S][N][N] (required).
 * d_noise must not overlap d_spectrum.  0 <= n_sh <= 8. */
int ssp_make_screens(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                     int B, int S, const double *cn2, const double *dz, int n_sh,
                     const float *d_noise, const float *d_noise_sh,
                     float *d_spectrum, float *d_sh_coef, float *d_screens,
                     void *d_ws, size_t ws_bytes);

/* Autoregressive evolution on the stored spectrum (PAPER.md:80 Eq.5, :74 Eq.4; Q8-Q10):
 *   C <- a tau C + sqrt(1 - a^2) C_fresh,  tau = exp(-i 2 pi T (fx vx + fy vy)),
 * C_fresh built from the fresh noise exactly as in ssp_make_screens; the subharmonic
 * coefficients follow the same recursion with tau at their fractional frequency; the
 * screens are then resynthesised.  d_spectrum, d_sh_coef: in-out.  0 <= a <= 1. */
int ssp_evolve_screens(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                       int B, int S, const double *cn2, const double *dz, int n_sh,
                       double a, double vx, double vy, double T,
                       const float *d_fresh_noise, const float *d_fresh_noise_sh,
                       float *d_spectrum, float *d_sh_coef, float *d_screens,
                       void *d_ws, size_t ws_bytes);

/* ssp_evolve_screens with the fresh grid noise drawn inside the generator instead of read from an array: element e of
 * the [B][S][N][N] batch takes draw `first + e` of stream `stream` of ssp_fill_noise's generator under `seed` (Philox-4x32-10
 * and Box-Muller, same arithmetic), so the call equals ssp_fill_noise(seed, stream, first, B S N^2, noise) followed by
 * ssp_evolve_screens(.., noise, ..) bit for bit, without the 8 B/px write and the 8 B/px read of that array (and without
 * the array).  The subharmonic noise (tiny) stays an input.  `first` even.  Built for N >= 512 (SSP_EUNSUPPORTED below:
 * draw the noise with ssp_fill_noise and call ssp_evolve_screens). */
/* The first synthesis of the same kind: ssp_make_screens with the grid noise drawn in the generator (draw `first + e` for
 * element e), equal to ssp_fill_noise + ssp_make_screens bit for bit.  With the two seeded calls a temporal simulation
 * never holds a noise array.  N >= 512. */
int ssp_make_screens_seeded(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                            int B, int S, const double *cn2, const double *dz, int n_sh,
                            unsigned long long seed, unsigned long long stream, unsigned long long first,
                            const float *d_noise_sh, float *d_spectrum, float *d_sh_coef, float *d_screens,
                            void *d_ws, size_t ws_bytes);
int ssp_evolve_screens_seeded(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                              int B, int S, const double *cn2, const double *dz, int n_sh,
                              double a, double vx, double vy, double T,
                              unsigned long long seed, unsigned long long stream, unsigned long long first,
                              const float *d_fresh_noise_sh, float *d_spectrum, float *d_sh_coef, float *d_screens,
                              void *d_ws, size_t ws_bytes);

/* The same two calls with a second output: d_screens_im (dev fp32 [B][S][N][N]) receives the IMAGINARY part of
 * each synthesis, phi_im = Im(sum C exp(..)) + Im-part subharmonics - its mean: a second screen of the same
 * statistics, uncorrelated with the first, from the same noise and the same transforms (the part that the
 * paper's real-part screen discards, Q3).  One spectrum then yields two screens; under evolution both follow the
 * stored spectrum. */
int ssp_make_screens_pair(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                          int B, int S, const double *cn2, const double *dz, int n_sh,
                          const float *d_noise, const float *d_noise_sh,
                          float *d_spectrum, float *d_sh_coef, float *d_screens, float *d_screens_im,
                          void *d_ws, size_t ws_bytes);
int ssp_evolve_screens_pair(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda,
                            int B, int S, const double *cn2, const double *dz, int n_sh,
                            double a, double vx, double vy, double T,
                            const float *d_fresh_noise, const float *d_fresh_noise_sh,
                            float *d_spectrum, float *d_sh_coef, float *d_screens, float *d_screens_im,
                            void *d_ws, size_t ws_bytes);

/* ---- path description (host only) ------------------------------------------------ */

/* Hufnagel-Valley 5/7 profile (PAPER.md:393 S21):
 *   Cn2(h) = 0.00594 (V/27)^2 (1e-5 h)^10 exp(-h/1000) + 2.7e-16 exp(-h/1500) + A exp(-h/ground_scale),
 * h in metres above ground, V the wind speed, A the ground-level constant.  ground_scale <= 0 takes the 1000 m
 * the paper prints; the textbook profile has 100 m. */
typedef struct { double A, V, ground_scale; } ssp_hv57;
double ssp_hv57_cn2(const ssp_hv57 *p, double h);
/* Vertical path h0 .. h0 + L cut into n equal slabs: cn2[j] = slab mean of Cn2 (cn2[j] dz[j] is the S18 integral
 * of slab j), dz[j] = L/n; host double [n] each, ready for ssp_make_screens.  Optional outputs: the
 * path's Rytov variance 3.27 k^(7/6) L^(5/6) int Cn2(z) (1 - z/L)^(5/3) dz (PAPER.md:380 S19, z from the source at
 * h0) and its Fried parameter (S18). */
int ssp_hv57_path(const ssp_hv57 *p, double h0, double L, int n, double lambda, double *cn2, double *dz,
                  double *rytov, double *r0);

/* Device-side noise draws (PAPER.md:359 S16 "unit-variance complex Gaussian"; Q3, Q29).  Fills d_out (dev
 * complex64 [n], 16-byte aligned) with draws first .. first+n-1 of the stream (seed, stream); Re and Im each N(0, 1).
 * Philox-4x32-10 block i = counter (i, stream), key seed; words (x0,x1) -> draw 2i, (x2,x3) -> draw 2i+1 by Box-Muller
 * on 23-bit uniforms.  first must be even.  The result is a plain noise array for ssp_make_screens / ssp_evolve_screens
 * (their noise arguments stay inputs: any generator may fill them).  Enqueued on the context's stream. */
int ssp_fill_noise(ssp_ctx *ctx, unsigned long long seed, unsigned long long stream, unsigned long long first,
                   unsigned long long n, float *d_out);
/* The raw words of the same generator, for checking it against the published known-answer vectors of Philox-4x32-10
 * (Salmon et al., SC'11): d_out[4 j .. 4 j + 3] = the four 32-bit output words of block first_block + j (index mod 2^64)
 * of (seed, stream), i.e. counter (i mod 2^32, i >> 32, stream mod 2^32, stream >> 32), key (seed mod 2^32, seed >> 32).
 * d_out: dev uint32 [n_blocks][4], 16-byte aligned.  Enqueued on the context's stream. */
int ssp_philox_words(ssp_ctx *ctx, unsigned long long seed, unsigned long long stream, unsigned long long first_block,
                     unsigned long long n_blocks, unsigned int *d_out);

/* Screen placement (Sec. 2.4).  Host-only, double precision.
 * ssp_dz_max: the largest step the angular-spectrum transfer function (Eq. 6) supports before its phase
 * aliases on the grid: |d psi / d kappa| dkappa <= pi at kappa0 = pi/dx, dkappa = 2 pi/(N dx), i.e.
 * dz_max = (N dx / 2) sqrt(n0^2 k0^2 - kappa0^2) / kappa0 (Eq. 7 with the ratio and kappa0 corrected, Q17;
 * paraxial limit N dx^2 n0 / lambda).  0 when the arguments are invalid or n0 k0 <= kappa0.
 * ssp_place_screens: the routine of PAPER.md:109 on a piecewise-linear Cn2 profile (z_prof ascending, cn2_prof >= 0,
 * host [n_prof]; constant beyond its ends) and the caller's desired interval edges (host [n_edges], ascending):
 *   1. an interval whose Rytov variance (S19, z from the interval's start) exceeds rytov_limit is halved
 *      until every piece is within it;  2. neighbours whose union stays within the limit are merged, left to right;
 *   3. marching from the start, each end is moved to where the straight line through (last old edge within the
 *      limit, its variance) and (next old edge, its variance) meets the limit, the move halved while the result
 *      exceeds the limit (Q28);  4. an interval longer than dz_max is halved until it is not (dz_max <= 0: skip).
 * Outputs, host [max_out] each: dz[j], the slab mean cn2[j] (ready for ssp_make_screens), optionally rytov[j]; *n_out =
 * the number of intervals.  SSP_EWORKSPACE when more than max_out intervals are needed (*n_out = a lower bound on
 * the count), SSP_EUNSUPPORTED when the limit cannot be met within 2^40 halvings, SSP_EINVAL on bad arguments. */
double ssp_dz_max(ssp_grid grid, double lambda, double n0);
int ssp_place_screens(const double *z_prof, const double *cn2_prof, int n_prof, const double *edges, int n_edges,
                      double lambda, double rytov_limit, double dz_max, int max_out, double *dz, double *cn2,
                      double *rytov, int *n_out);

/* Workspace.  d_ws / ws_bytes: a caller-allocated device buffer of at least ssp_workspace_bytes(grid, B, S)
 * bytes, 16-byte aligned.  The screen calls need it (tables, subharmonic coefficients, the column-transformed
 * intermediate of a chunk of screens); the propagation calls, ssp_dft2_centered and ssp_propagate_host accept it
 * for symmetry and do not use it today (NULL / 0 is fine there). */

/* ---- propagation --------------------------------------------------------------- */

/* Split-step propagation (Eq.1; step order Q11):
 *   for j = 1..n_steps:  U <- F^-1{ F{U} H(dz_j) };  if j <= S: U <- U exp(i phi_j);  U <- U W.
 * dz: host [n_steps].  d_screens: dev fp32, screen j of field b at
 * d_screens + b*screen_batch_stride + (j-1)*N*N (stride in elements; 0 = one stack shared
 * by all fields); may be NULL when S == 0.  0 <= S <= n_steps.
 * d_field_in / d_field_out: dev complex64 [B][N][N]; may alias.
 * d_planes: optional dev complex64 [B][n_steps][N][N], the field after each complete step
 * (needed by the adjoint's phase gradient).  d_stats: optional dev ssp_stats[B] of the
 * output field with ROI fraction roi_frac. */
int ssp_propagate(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                  int B, int n_steps, const double *dz,
                  const float *d_screens, long long screen_batch_stride, int S,
                  ssp_window win, const float *d_field_in, float *d_field_out,
                  float *d_planes, ssp_stats *d_stats, double roi_frac,
                  void *d_ws, size_t ws_bytes);

/* Adjoint (conjugate transpose) of ssp_propagate (north_star; replaces autograd):
 *   for j = n_steps..1:  [grad_j = Im(G_j conj(U_j)) if j <= S];  g <- W g;
 *                        if j <= S: g <- exp(-i phi_j) g;  g <- F^-1{ conj(H(dz_j)) F{g} }.
 * G_j is the adjoint field arriving at plane j, U_j = d_planes[b][j-1].  Gradient
 * convention G = dl/dRe U + i dl/dIm U.  d_g_out / d_g_in: dev complex64 [B][N][N]; may
 * alias.  d_planes and d_phase_grad (dev fp32 [B][S][N][N]) are both given or both NULL. */
int ssp_propagate_adjoint(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                          int B, int n_steps, const double *dz,
                          const float *d_screens, long long screen_batch_stride, int S,
                          ssp_window win, const float *d_g_out, float *d_g_in,
                          const float *d_planes, float *d_phase_grad,
                          void *d_ws, size_t ws_bytes);

/* Intensity statistics of B fields (O8).  Optional per-pixel ensemble accumulation by
 * Welford's algorithm: d_mean, d_M2 dev fp32 [N][N] in-out and *count
 * (host, in-out) advanced by B; pass all three or none. */
int ssp_beam_stats(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_field, double roi_frac,
                   ssp_stats *d_stats, float *d_mean, float *d_M2, long long *count);

/* ssp_beam_stats without any allocation, for callers that may not call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same statistics (O8; PAPER.md:423 S25) of B fields
 * d_field (dev c64 [B][N][N], 16-byte aligned) into d_stats (dev ssp_stats[B], required); no ensemble accumulation.
 * The block partials live in a file-scope device array of SSP_STATS_STATIC_BYTES that every GPU loading the library
 * holds until the process exits, instead of the context's growable scratch: the call performs no cudaMalloc,
 * cudaFree or allocating library call.  Limit: B <= SSP_STATS_STATIC_MAX_FIELDS per call (SSP_EINVAL with a message
 * beyond it: split the batch, or use ssp_beam_stats); any N the library supports.  One kernel, enqueued on the
 * context's stream after a memset of the array's ticket counters; sums and their order are those of ssp_beam_stats.
 * The array is shared by ALL contexts and streams of the process on that GPU: calls that overlap on the GPU race on it
 * (serialise them on one stream or with events). */
#define SSP_STATS_STATIC_MAX_FIELDS 1024
#define SSP_STATS_STATIC_BYTES (2 * SSP_STATS_STATIC_MAX_FIELDS * 9 * 8 + SSP_STATS_STATIC_MAX_FIELDS * 4)   /* 148 KiB */
int ssp_beam_stats_static(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_field, double roi_frac,
                          ssp_stats *d_stats);

/* End-to-end form of ssp_propagate with HOST buffers: copies field and screens to the
 * device buffers given (d_field [B][N][N] c64, d_screens as above), propagates, copies
 * the output field and statistics back, and synchronises the stream.  h_* pointers are
 * host memory (pinned for full copy speed and overlap).  h_screens == NULL with S > 0: the
 * screens are already in d_screens (made there by ssp_make_screens / ssp_evolve_screens, e.g.
 * from ssp_fill_noise draws) and only the fields travel.  The batch is processed in chunks of
 * max(1, B/8) fields on two internal copy streams, so that the copies of neighbouring chunks
 * overlap the propagation; results equal ssp_propagate's. */
int ssp_propagate_host(ssp_ctx *ctx, ssp_grid grid, double lambda, double n0, int h_kind,
                       int B, int n_steps, const double *dz,
                       const float *h_screens, long long screen_batch_stride, int S,
                       ssp_window win, const float *h_field_in, float *h_field_out,
                       ssp_stats *h_stats, double roi_frac,
                       float *d_field, float *d_screens, ssp_stats *d_stats,
                       void *d_ws, size_t ws_bytes);

/* Forward-only temporal frame on the device with the screen synthesis fused into the propagation (
 * the workload of PAPER.md:76-84 when the screens are used once).  Equivalent to ssp_evolve_screens followed by
 * ssp_propagate with n_steps = S and step j = slab dz[j] -- the AR state d_spectrum / d_sh_coef advances the same way,
 * d_field_out and d_stats are the same up to fp32 rounding -- but the evolved screens are never written: the generator
 * stops after its column pass, keeps every screen's column-transformed spectrum in d_ycol (dev c64 [B][S][N][N],
 * scratch), and the split step's row kernel synthesises row iy of screen j itself (IFFT_x, real part, subharmonics,
 * analytic mean; PAPER.md:57 Eq.2, :63 Eq.3, :362) right before it applies it: 8 B/px read there instead of the
 * 12 B/px row pass plus a 4 B/px read.  Built for N = 1024 (SSP_EUNSUPPORTED otherwise), Fresnel H, window on.
 * d_ws >= ssp_workspace_bytes(grid, B, S).  Enqueued on the context's stream. */
int ssp_evolve_propagate(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, double n0,
                         int B, int S, const double *cn2, const double *dz, int n_sh,
                         double a, double vx, double vy, double T,
                         const float *d_fresh_noise, const float *d_fresh_noise_sh,
                         float *d_spectrum, float *d_sh_coef,
                         ssp_window win, const float *d_field_in, float *d_field_out,
                         ssp_stats *d_stats, double roi_frac, float *d_ycol, void *d_ws, size_t ws_bytes);

/* One temporal frame end to end from HOST fields (the workload of PAPER.md:76-84: every frame the screens evolve
 * by the autoregression of Eq. 5 and a batch of fields propagates through them).  Per chunk of ssp_frame_chunk(B)
 * fields: fresh noise is drawn on the device (ssp_fill_noise: stream 2*frame for the grid noise of the whole batch,
 * draw index = element index in [B][S][N][N]; stream 2*frame+1 for the subharmonic noise [B][S][n_sh][3][3]), the
 * chunk's screen stacks evolve (ssp_evolve_screens), its fields propagate through them (ssp_propagate with
 * n_steps = S, step dz[j] = slab dz[j], per-field stacks; launched per group of n/2, n/4, .., 1, 1 chunks), and output
 * fields and statistics return to the host; the uploads run under the first chunks' draws and evolution, the
 * downloads under the next chunks' work.  The result
 * equals those three calls on the whole batch.  Device buffers: d_field c64 [B][N][N]; d_spectrum c64
 * [B][S][N][N] and d_sh_coef c64 [B][S][n_sh][3][3], in-out (the AR state, from ssp_make_screens); d_screens fp32
 * [B][S][N][N] (out: this frame's screens); d_noise c64 [ssp_frame_chunk(B)][S][N][N] scratch; d_noise_sh c64
 * [B][S][n_sh][3][3] scratch; d_stats [B]; d_ws >= ssp_workspace_bytes(grid, ssp_frame_chunk(B), S).
 * h_adjoint_out (host c64 [B][N][N], optional; with it d_adjoint, dev c64 [B][N][N] scratch): the frame also runs the
 * adjoint split step on each group's received fields, h_adjoint_out = A^H U_out (ssp_propagate_adjoint with
 * d_g_out = the received field: the gradient of the received power (1/2) sum |U_out|^2 w.r.t. the input field, i.e.
 * the time-reversed return), and copies it back under the next group's work.  NULL: forward only.
 * Every argument is validated before the first copy is queued; if an inner call still fails, both copy streams and
 * the context's stream are drained before the error is returned.  Synchronises the stream. */
typedef struct {
    double a, vx, vy, T;            /* blending factor, wind [m/s], frame interval [s] (Eq. 4, 5) */
    unsigned long long seed, frame; /* noise streams 2*frame and 2*frame+1 of this seed */
} ssp_ar;
int ssp_frame_chunk(int B);
int ssp_frame_host(ssp_ctx *ctx, ssp_grid grid, const ssp_psd *psd, double lambda, double n0, int h_kind,
                   int B, int S, const double *cn2, const double *dz, int n_sh, const ssp_ar *ar,
                   ssp_window win, const float *h_field_in, float *h_field_out, ssp_stats *h_stats, double roi_frac,
                   float *d_field, float *d_spectrum, float *d_sh_coef, float *d_screens,
                   float *d_noise, float *d_noise_sh, ssp_stats *d_stats, void *d_ws, size_t ws_bytes,
                   float *h_adjoint_out, float *d_adjoint);

/* ---- helpers for mask systems (config 4; O9) ----------------- */

/* out = in exp(i sign theta); theta dev fp32 [N][N] shared by the B fields; in may alias out. */
int ssp_phase_mul(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_theta, double sign,
                  const float *d_in, float *d_out);
/* Lens as a DFT: centred unitary transform F_c = fftshift o fft2 o ifftshift / N
 * (inverse != 0: its inverse).  in may alias out. */
int ssp_dft2_centered(ssp_ctx *ctx, ssp_grid grid, int B, int inverse,
                      const float *d_in, float *d_out, void *d_ws, size_t ws_bytes);
/* One Adam step on a phase mask shared by B fields (D2NN training):
 *   g = (1/B) sum_b d_grad[b];  m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2;
 *   theta <- theta - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps),   t >= 1 the step count.
 * d_grad: dev fp32 [B][N][N]; d_m, d_v, d_theta: dev fp32 [N][N], updated in place. */
int ssp_adam_update(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_grad, double lr, double beta1,
                    double beta2, double eps, int t, float *d_m, float *d_v, float *d_theta);
/* Circular aperture of `radius` metres about the grid centre: out = in where
 * (ix-N/2)^2 + (iy-N/2)^2 <= floor((radius/dx)^2) (the threshold is an integer taken on the host in
 * double), else 0.  d_in / d_out: dev complex64 [B][N][N]; may alias. */
int ssp_aperture(ssp_ctx *ctx, ssp_grid grid, int B, double radius, const float *d_in, float *d_out);
/* grad[b] = Im(g[b] conj(u[b])), dev fp32 [B][N][N]; d_g, d_u dev complex64 [B][N][N]. */
int ssp_phase_grad(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_g, const float *d_u,
                   float *d_grad);
/* Per field b: d_out[b] = { Re <a,b>, Im <a,b>, sum |a|^2, sum |b|^2 } (doubles),
 * <a,b> = sum conj(a) b.  d_out: dev double [B][4]. */
int ssp_inner_products(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_a, const float *d_b,
                       double *d_out);
/* The D2NN training loss of PAPER.md:113 (mean absolute error between the processed field v and the free-space
 * result t, read as the mean modulus of the complex difference) and its gradient with respect to v:
 *   d_loss[b] = (1/N^2) sum |v - t|,   d_grad[b] = (v - t) / (N^2 |v - t|)   (0 where v == t; real-pair convention
 * G = dl/dRe v + i dl/dIm v as everywhere in this library).  d_v, d_t, d_grad: dev complex64 [B][N][N] (d_grad may
 * alias d_v); d_loss: dev double [B]. */
int ssp_mae_loss(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_v, const float *d_t, double *d_loss, float *d_grad);
/* out[b] = alpha[b] a[b] + beta[b] b[b] with per-field complex scalars; h_alpha, h_beta:
 * host double [B][2]; out may alias a or b. */
int ssp_lincomb(ssp_ctx *ctx, ssp_grid grid, int B, const double *h_alpha, const float *d_a,
                const double *h_beta, const float *d_b, float *d_out);

#ifdef __cplusplus
}
#endif
#endif /* SSP_H */
