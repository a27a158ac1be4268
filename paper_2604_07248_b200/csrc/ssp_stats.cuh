// ssp_stats.cuh -- accumulator layout and finaliser of the beam statistics (K8; PAPER.md:423 S25, :143; O8),
// shared by the stand-alone reducer (ssp_misc.cu), the epilogue of the last row kernel (ssp_kernels.cuh) and the
// on-chip small-grid kernel (ssp_small.cu).
#pragma once

#include "ssp_internal.h"

namespace ssp {

// raw intensity moments about the grid centre in pixel units, ROI sums, on-axis intensity
enum { ACC_I = 0, ACC_X, ACC_Y, ACC_XX, ACC_YY, ACC_XY, ACC_RI, ACC_RI2, ACC_AXIS, ACC_N };

// one row's sums -> the nine accumulators: y enters here, once per row, in double
enum { ROW_I = 0, ROW_X, ROW_XX, ROW_RI, ROW_RI2, ROW_AXIS, ROW_N };
__device__ __forceinline__ double row_to_acc(int moment, const double *r, double y)
{
    switch (moment) {
    case ACC_I: return r[ROW_I];
    case ACC_X: return r[ROW_X];
    case ACC_Y: return y * r[ROW_I];
    case ACC_XX: return r[ROW_XX];
    case ACC_YY: return y * y * r[ROW_I];
    case ACC_XY: return y * r[ROW_X];
    case ACC_RI: return r[ROW_RI];
    case ACC_RI2: return r[ROW_RI2];
    default: return r[ROW_AXIS];
    }
}

__device__ __forceinline__ ssp_stats finalize_stats(const double *a, double dx, long long roi_n)
{
    ssp_stats s;
    const double sI = a[ACC_I];
    s.power = sI * dx * dx;
    double cx = 0, cy = 0, sxx = 0, syy = 0, sxy = 0;
    if (sI > 0) {
        cx = a[ACC_X] / sI;
        cy = a[ACC_Y] / sI;
        sxx = a[ACC_XX] / sI - cx * cx;
        syy = a[ACC_YY] / sI - cy * cy;
        sxy = a[ACC_XY] / sI - cx * cy;
    }
    s.cx = cx * dx;
    s.cy = cy * dx;
    s.sxx = sxx * dx * dx;
    s.syy = syy * dx * dx;
    s.sxy = sxy * dx * dx;
    const double tr = s.sxx + s.syy;
    s.w2 = sqrt(2.0 * (tr > 0 ? tr : 0.0));
    s.I_axis = a[ACC_AXIS];
    s.roi_sumI = a[ACC_RI];
    s.roi_sumI2 = a[ACC_RI2];
    s.roi_n = roi_n;
    return s;
}

// Per-thread sums over the E points of one row that a thread holds in registers (layout strided by R: element (i, q) is
// pixel ix = q N/R + t + T i): fp32 within the row (x is an exact small integer), promoted to double by the caller.
template <int N, int R, int E, int T>
__device__ __forceinline__ void row_point_sums(const float2 *v, int t, int iy, int lo, int hi, double *r)
{
    constexpr int half = N / 2;
    const bool roi_row = iy >= lo && iy < hi;
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, r1 = 0.f, r2 = 0.f, ax = 0.f;
#pragma unroll
    for (int i = 0; i < E / R; ++i)
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int ix = q * (N / R) + t + T * i;
            const float2 u = v[i * R + q];
            const float I = fmaf(u.x, u.x, u.y * u.y), x = (float)(ix - half), xI = x * I;
            s0 += I;
            s1 += xI;
            s2 = fmaf(x, xI, s2);
            const float Ir = (roi_row && ix >= lo && ix < hi) ? I : 0.f;
            r1 += Ir;
            r2 = fmaf(Ir, Ir, r2);
            ax += (iy == half && ix == half) ? I : 0.f;
        }
    r[ROW_I] = (double)s0; r[ROW_X] = (double)s1; r[ROW_XX] = (double)s2;
    r[ROW_RI] = (double)r1; r[ROW_RI2] = (double)r2; r[ROW_AXIS] = (double)ax;
}

// Sum r[0..ROW_N) over groups of W consecutive lanes (W a power of two <= 32); every lane of a group ends with the sum.
template <int W>
__device__ __forceinline__ void group_sum(double *r)
{
#pragma unroll
    for (int o = W / 2; o > 0; o >>= 1)
#pragma unroll
        for (int i = 0; i < ROW_N; ++i) r[i] += __shfl_xor_sync(0xffffffffu, r[i], o);
}

} // namespace ssp
