// ssp_misc.cu -- statistics reducer (K8) and the small element-wise helpers.
//
// K8 (PAPER.md:423 S25, :143; O8): per field, raw intensity moments about the grid
// centre in pixel units: fp32 partial sums within a row, promoted to fp64 once per row, combined by
// warp shuffles into one partial per block and moment (no atomics: bit-reproducible); a one-warp-per-field
// finaliser adds the block partials in block order and turns them into ssp_stats.
#include "ssp_stats.cuh"

namespace ssp {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// grid: (blocks_per_field, B).  A block walks rows grid-stride; lanes = min(64, N/2) threads share a row
// (lane_shift = log2(lanes)), each owning float4 pairs (2 pixels) at fixed columns.  Within one row a thread sums
// I, x I, x^2 I and the ROI terms over its <= 64 pixels in fp32 (x is an exact small integer; the partial sums carry a
// relative rounding of a few 1e-7 that averages out over the >= 10^4 partials of a field), then promotes the partials
// to double once per row, where y enters.  Per-pixel fp64 accumulation ran at half the bandwidth: the fp64 pipe is narrow.
__global__ void __launch_bounds__(256) k_stats_accum(const float2 *__restrict__ field, int N, int lane_shift, int lo,
                                                      int hi, double *__restrict__ acc)
{
    const int b = blockIdx.y;
    const size_t px = (size_t)N * N;
    const float4 *f4 = reinterpret_cast<const float4 *>(field + (size_t)b * px);
    double a[ACC_N];
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) a[i] = 0.0;
    const int half = N / 2, lanes = 1 << lane_shift, rows_per_pass = 256 >> lane_shift;
    const int col0 = threadIdx.x & (lanes - 1);
    for (int iy = blockIdx.x * rows_per_pass + (threadIdx.x >> lane_shift); iy < N; iy += gridDim.x * rows_per_pass) {
        const float4 *row = f4 + (size_t)iy * half;
        const bool roi_row = iy >= lo && iy < hi;
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, r1 = 0.f, r2 = 0.f, ax = 0.f;
        for (int c = col0; c < half; c += 4 * lanes) {
            float4 u[4];                                                 // four independent loads in flight;
#pragma unroll
            for (int j = 0; j < 4; ++j) {                                // a column past the end reads as zeros: adds nothing
                const int cc = c + j * lanes;
                u[j] = cc < half ? __ldg(row + cc) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float I2[2] = {fmaf(u[j].x, u[j].x, u[j].y * u[j].y), fmaf(u[j].z, u[j].z, u[j].w * u[j].w)};
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int ix = 2 * (c + j * lanes) + e;
                    const float I = I2[e], x = (float)(ix - half), xI = x * I;
                    s0 += I;
                    s1 += xI;
                    s2 = fmaf(x, xI, s2);
                    const float Ir = (roi_row && ix >= lo && ix < hi) ? I : 0.f;
                    r1 += Ir;
                    r2 = fmaf(Ir, Ir, r2);
                    ax += (iy == half && ix == half) ? I : 0.f;
                }
            }
        }
        const double y = (double)(iy - half), d0 = (double)s0, d1 = (double)s1;
        a[ACC_I] += d0;
        a[ACC_X] += d1;
        a[ACC_XX] += (double)s2;
        a[ACC_Y] = fma(y, d0, a[ACC_Y]);
        a[ACC_YY] = fma(y * y, d0, a[ACC_YY]);
        a[ACC_XY] = fma(y, d1, a[ACC_XY]);
        a[ACC_RI] += (double)r1;
        a[ACC_RI2] += (double)r2;
        a[ACC_AXIS] += (double)ax;
    }
    // warp shuffles, then one partial per warp through shared memory, then one partial per block and moment in
    // acc[b][block][moment]; k_stats_final adds them in block order (no atomics: the result is reproducible bit by bit)
    __shared__ double part[8][ACC_N];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) {
        const double s = warp_sum(a[i]);
        if (lane == 0) part[warp][i] = s;
    }
    __syncthreads();
    if (threadIdx.x < ACC_N) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += part[w][threadIdx.x];
        acc[((size_t)b * gridDim.x + blockIdx.x) * ACC_N + threadIdx.x] = s;
    }
}

// one CTA per field: the partial records acc[b][k][moment], k < bpf, are added in a fixed order (thread j takes the
// records k = j mod 256 in ascending order, then a shuffle tree per warp, then the eight warp sums in order): no
// atomics, bit-reproducible; thread 0 finishes
__global__ void __launch_bounds__(256) k_stats_final(const double *__restrict__ acc, int bpf, double dx, long long roi_n,
                                                      ssp_stats *__restrict__ out)
{
    const int b = blockIdx.x, tid = threadIdx.x;
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    double a[ACC_N];
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) a[i] = 0.0;
    for (int k = tid; k < bpf; k += 256) {
        const double *p = acc + ((size_t)b * bpf + k) * ACC_N;
#pragma unroll
        for (int i = 0; i < ACC_N; ++i) a[i] += p[i];
    }
    __shared__ double part[8][ACC_N];
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) {
        const double s = warp_sum(a[i]);
        if ((tid & 31) == 0) part[tid >> 5][i] = s;
    }
    __syncthreads();
    if (tid == 0) {
        double t[ACC_N];
        for (int i = 0; i < ACC_N; ++i) {
            t[i] = 0.0;
            for (int w = 0; w < 8; ++w) t[i] += part[w][i];
        }
        out[b] = finalize_stats(t, dx, roi_n);
    }
}

void stats_roi(int N, double roi_frac, int *lo_out, int *hi_out, long long *roi_n)
{
    int h = (int)floor(roi_frac * N / 2.0);
    int lo = N / 2 - h, hi = N / 2 + h;
    if (h <= 0) { lo = N / 2; hi = N / 2 + 1; }
    if (lo < 0) lo = 0;
    if (hi > N) hi = N;
    *lo_out = lo; *hi_out = hi;
    *roi_n = (long long)(hi - lo) * (hi - lo);
}

int launch_stats_final(ssp_ctx *ctx, int B, int bpf, double dx, long long roi_n, const double *acc, ssp_stats *d_stats)
{
    SSP_CUDA(ctx, launch_pdl(k_stats_final, dim3(B), dim3(256), 0, ctx->stream, pdl_enabled(), acc, bpf, dx, roi_n, d_stats));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

int launch_stats(ssp_ctx *ctx, int N, double dx, int B, const float2 *field, double roi_frac,
                 ssp_stats *d_stats)
{
    int lo, hi;
    long long roi_n;
    stats_roi(N, roi_frac, &lo, &hi, &roi_n);
    int lane_shift = 0;
    while ((2 << lane_shift) <= N / 2 && lane_shift < 6) ++lane_shift;       // lanes = min(64, N/2)
    const int rows_per_pass = 256 >> lane_shift;
    // blocks per field: all B * bpf blocks resident at once (8 per SM) when the batch allows, every block the same
    // number of row passes (to within one)
    const int passes = (N + rows_per_pass - 1) / rows_per_pass;               // >= 1 (N = 8, 16: one partial pass; the kernel guards iy < N)
    int target = (ctx->num_sms * 8) / B;
    if (target < 1) target = 1;
    const int per = (passes + target - 1) / target;
    const int bpf = (passes + per - 1) / per;
    if (int rc = ensure_scratch(ctx, sizeof(double) * ACC_N * (size_t)B * bpf)) return rc;
    double *acc = reinterpret_cast<double *>(ctx->scratch);
    ctx->prof_begin("stats", 8.0 * (double)B * N * N);
    k_stats_accum<<<dim3(bpf, B), 256, 0, ctx->stream>>>(field, N, lane_shift, lo, hi, acc);
    k_stats_final<<<B, 256, 0, ctx->stream>>>(acc, bpf, dx, roi_n, d_stats);
    ctx->prof_end();
    ctx->launches += 2;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

// Welford per pixel, sequential over the B fields of this call.
__global__ void __launch_bounds__(256) k_welford(const float2 *__restrict__ field, size_t px, int B,
                                                  float *__restrict__ mean, float *__restrict__ M2, long long count0)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= px) return;
    float m = mean[i], s = M2[i];
    for (int b = 0; b < B; ++b) {
        const float2 u = __ldg(field + (size_t)b * px + i);
        const float I = fmaf(u.x, u.x, u.y * u.y);
        const float d = I - m;
        m += d / (float)(count0 + b + 1);
        s = fmaf(d, I - m, s);
    }
    mean[i] = m;
    M2[i] = s;
}

int launch_welford(ssp_ctx *ctx, int N, int B, const float2 *field, float *mean, float *M2, long long count0)
{
    const size_t px = (size_t)N * N;
    k_welford<<<(unsigned)((px + 255) / 256), 256, 0, ctx->stream>>>(field, px, B, mean, M2, count0);
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

__global__ void __launch_bounds__(256) k_phase_mul(const float *__restrict__ theta, float sign, size_t px, int B,
                                                    const float2 *in, float2 *out)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= px) return;
    float s, c;
    sincosf(__ldg(theta + i), &s, &c); // masks are in [0, 2 pi): the accurate path is cheap enough here
    s *= sign;
    for (int b = 0; b < B; ++b) {
        const float2 u = in[(size_t)b * px + i];
        out[(size_t)b * px + i] = make_float2(fmaf(u.x, c, -u.y * s), fmaf(u.x, s, u.y * c));
    }
}

// Angular-spectrum transfer function (Eq.6 without the carrier, Q2), scaled by 1/N^2:
//   H = exp(i dz (sqrt(km^2 - kappa^2) - km)) = exp(-i dz kappa^2 / (km + sqrt(km^2 - kappa^2))),
//   km = 2 pi / lam_eff, kappa^2 = 4 pi^2 (fx^2 + fy^2); kappa > km (evanescent) -> 0.
// Evaluated in double: the phase reaches hundreds of radians.
// Layout: tile-major [N/C][N (ky)][C] with C the column-tile width of the kernel that reads it, so that a
// column tile's multipliers are one contiguous 8 N C-byte block (coalesced, L2-resident).
__global__ void __launch_bounds__(256) k_h2d_table(int N, int C, double dx, double lam_eff, double dz, int conj,
                                                    float2 *__restrict__ out)
{
    const int kx = blockIdx.x * blockDim.x + threadIdx.x, ky = blockIdx.y;
    if (kx >= N) return;
    const double kPi = 3.14159265358979323846;
    const double fx = (double)((kx < N / 2) ? kx : kx - N) / ((double)N * dx);
    const double fy = (double)((ky < N / 2) ? ky : ky - N) / ((double)N * dx);
    const double km = 2.0 * kPi / lam_eff, kap2 = 4.0 * kPi * kPi * (fx * fx + fy * fy);
    float2 h = make_float2(0.f, 0.f);
    if (kap2 <= km * km) {
        double ang = -dz * kap2 / (km + sqrt(km * km - kap2));
        if (conj) ang = -ang;
        double s, c;
        sincos(ang, &s, &c);
        const double scale = 1.0 / ((double)N * (double)N);
        h = make_float2((float)(scale * c), (float)(scale * s));
    }
    out[((size_t)(kx / C) * N + ky) * C + kx % C] = h;
}

int launch_h2d_table(ssp_ctx *ctx, int N, int C, double dx, double lam_eff, double dz, int conj, float2 *out)
{
    k_h2d_table<<<dim3((N + 255) / 256, N), 256, 0, ctx->stream>>>(N, C, dx, lam_eff, dz, conj, out);
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

// Adam step on a mask shared by B fields; c1 = 1/(1-b1^t), c2 = 1/(1-b2^t), o1 = 1-b1, o2 = 1-b2
// from the host in double (1 - 0.999f in fp32 is 6e-5 off)
__global__ void __launch_bounds__(256) k_adam(size_t n, int B, const float *__restrict__ grad, float lr, float b1, float b2,
                                               float eps, float c1, float c2, float o1, float o2, float *__restrict__ m,
                                               float *__restrict__ v, float *__restrict__ theta)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float g = 0.f;
    for (int b = 0; b < B; ++b) g += grad[(size_t)b * n + i];
    g /= (float)B;
    const float mi = fmaf(b1, m[i], o1 * g);
    const float vi = fmaf(b2, v[i], o2 * g * g);
    m[i] = mi;
    v[i] = vi;
    theta[i] -= lr * (mi * c1) / (sqrtf(vi * c2) + eps);
}

int launch_adam(ssp_ctx *ctx, long long n, int B, const float *grad, float lr, float b1, float b2, float eps,
                float c1, float c2, float o1, float o2, float *m, float *v, float *theta)
{
    SSP_CUDA(ctx, launch_pdl(k_adam, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, ctx->stream, pdl_enabled(), (size_t)n, B, grad, lr, b1, b2, eps, c1, c2, o1, o2, m, v, theta));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

// circular aperture: integer test against a host-decided threshold
__global__ void __launch_bounds__(256) k_aperture(int N, long long r2max, const float2 *__restrict__ in, float2 *__restrict__ out)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const int ix = blockIdx.x * blockDim.x + threadIdx.x, iy = blockIdx.y, b = blockIdx.z;
    if (ix >= N) return;
    const long long x = ix - N / 2, y = iy - N / 2;
    const size_t i = ((size_t)b * N + iy) * N + ix;
    out[i] = (x * x + y * y <= r2max) ? in[i] : make_float2(0.f, 0.f);
}

int launch_aperture(ssp_ctx *ctx, int N, int B, long long r2max_px, const float2 *in, float2 *out)
{
    SSP_CUDA(ctx, launch_pdl(k_aperture, dim3((N + 255) / 256, N, B), dim3(256), 0, ctx->stream, pdl_enabled(), N, r2max_px, in, out));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

int launch_phase_mul(ssp_ctx *ctx, int N, int B, const float *theta, float sign, const float2 *in, float2 *out)
{
    const size_t px = (size_t)N * N;
    SSP_CUDA(ctx, launch_pdl(k_phase_mul, dim3((unsigned)((px + 255) / 256)), dim3(256), 0, ctx->stream, pdl_enabled(), theta, sign, px, B, in, out));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

__global__ void __launch_bounds__(256) k_phase_grad(const float2 *__restrict__ g, const float2 *__restrict__ u,
                                                     size_t n, float *__restrict__ grad)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float2 a = g[i], b = u[i];
    grad[i] = a.y * b.x - a.x * b.y;
}

int launch_phase_grad(ssp_ctx *ctx, long long n, const float2 *g, const float2 *u, float *grad)
{
    SSP_CUDA(ctx, launch_pdl(k_phase_grad, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, ctx->stream, pdl_enabled(), g, u, (size_t)n, grad));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

// out[b] = { Re<a,b>, Im<a,b>, |a|^2, |b|^2 },  <a,b> = sum conj(a) b
__global__ void __launch_bounds__(256) k_inner(const float2 *__restrict__ A, const float2 *__restrict__ Bf,
                                                size_t px, double *__restrict__ out)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const int b = blockIdx.y;
    double r = 0, im = 0, na = 0, nb = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < px; i += (size_t)gridDim.x * blockDim.x) {
        const float2 x = __ldg(A + (size_t)b * px + i), y = __ldg(Bf + (size_t)b * px + i);
        r += (double)x.x * y.x + (double)x.y * y.y;
        im += (double)x.x * y.y - (double)x.y * y.x;
        na += (double)x.x * x.x + (double)x.y * x.y;
        nb += (double)y.x * y.x + (double)y.y * y.y;
    }
    r = warp_sum(r); im = warp_sum(im); na = warp_sum(na); nb = warp_sum(nb);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(out + 4 * b + 0, r);
        atomicAdd(out + 4 * b + 1, im);
        atomicAdd(out + 4 * b + 2, na);
        atomicAdd(out + 4 * b + 3, nb);
    }
}

// Mean-absolute-error loss of the D2NN and its field gradient: loss[b] = (1/N^2) sum |v - t|,
// g = (v - t) / (N^2 |v - t|) (0 where v == t).  Per-block partial sums in double, then one atomic per block.
__global__ void __launch_bounds__(256) k_mae(const float2 *__restrict__ V, const float2 *__restrict__ Tg, size_t px,
                                              float inv_px, double *__restrict__ loss, float2 *__restrict__ G)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const int b = blockIdx.y;
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < px; i += (size_t)gridDim.x * blockDim.x) {
        const float2 v = __ldg(V + (size_t)b * px + i), t = __ldg(Tg + (size_t)b * px + i);
        const float dx = v.x - t.x, dy = v.y - t.y;
        const float m = sqrtf(fmaf(dx, dx, dy * dy));
        acc += (double)m;
        const float s = m > 0.f ? inv_px / m : 0.f;
        G[(size_t)b * px + i] = make_float2(dx * s, dy * s);
    }
    acc = warp_sum(acc);
    __shared__ double part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += part[w];
        atomicAdd(loss + b, s * (double)inv_px);
    }
}

int launch_mae(ssp_ctx *ctx, int N, int B, const float2 *v, const float2 *t, double *loss, float2 *g)
{
    const size_t px = (size_t)N * N;
    SSP_CUDA(ctx, cudaMemsetAsync(loss, 0, sizeof(double) * (size_t)B, ctx->stream));
    int bpf = (int)((px + 256 * 8 - 1) / (256 * 8));
    SSP_CUDA(ctx, launch_pdl(k_mae, dim3(bpf, B), dim3(256), 0, ctx->stream, pdl_enabled(), v, t, px, (float)(1.0 / (double)px), loss, g));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

int launch_inner(ssp_ctx *ctx, int N, int B, const float2 *a, const float2 *b, double *out)
{
    const size_t px = (size_t)N * N;
    SSP_CUDA(ctx, cudaMemsetAsync(out, 0, sizeof(double) * 4 * (size_t)B, ctx->stream));
    int bpf = (int)((px + 256 * 16 - 1) / (256 * 16));
    SSP_CUDA(ctx, launch_pdl(k_inner, dim3(bpf, B), dim3(256), 0, ctx->stream, pdl_enabled(), a, b, px, out));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

__global__ void __launch_bounds__(256) k_lincomb(const float2 *__restrict__ coef, const float2 *a, const float2 *b,
                                                  size_t px, float2 *out)
{
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)
    const int f = blockIdx.y;
    const float2 al = coef[2 * f], be = coef[2 * f + 1];
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < px; i += (size_t)gridDim.x * blockDim.x) {
        const float2 x = a[(size_t)f * px + i], y = b[(size_t)f * px + i];
        out[(size_t)f * px + i] = make_float2(al.x * x.x - al.y * x.y + be.x * y.x - be.y * y.y,
                                              al.x * x.y + al.y * x.x + be.x * y.y + be.y * y.x);
    }
}

int launch_lincomb(ssp_ctx *ctx, int N, int B, const float2 *coef, const float2 *a, const float2 *b, float2 *out)
{
    const size_t px = (size_t)N * N;
    int bpf = (int)((px + 256 * 4 - 1) / (256 * 4));
    SSP_CUDA(ctx, launch_pdl(k_lincomb, dim3(bpf, B), dim3(256), 0, ctx->stream, pdl_enabled(), coef, a, b, px, out));
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

} // namespace ssp
