// ssp_noalloc.cu -- beam statistics (K8; PAPER.md:423 S25, :143; O8) for callers that may not allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// ssp_beam_stats keeps its block partials in the context's scratch, which grows by cudaMalloc on demand
// (ensure_scratch).  ssp_beam_stats_static is the same reduction with the partials in g_stats_scratch below, a
// file-scope device array of fixed size that every GPU loading libssp.so holds until the process exits
// (SSP_STATS_STATIC_BYTES = 148 KiB).  The entry point calls no cudaMalloc / cudaFree and no allocating library
// routine; requests that do not fit the array are rejected.
//
// One launch instead of two: every block writes its partial record as k_stats_accum (ssp_misc.cu) does, then takes a
// ticket on its field's counter; the block that draws the last ticket adds the field's records in the fixed order of
// k_stats_final and writes ssp_stats.  No floating-point atomics: same sums in the same order as the two-kernel path.
//
// The array is shared by every call, context and stream of the process on that GPU, and keeps the last call's
// contents: the ticket counters must start at zero and are cleared on the stream before the launch; the partial
// records are fully rewritten before they are read.  Calls that overlap on the GPU (two streams, two contexts, two
// host threads) race on it.
#include <mutex>

#include "ssp_stats.cuh"

namespace ssp {

static constexpr int kMaxFields = SSP_STATS_STATIC_MAX_FIELDS;          // ticket counters
static constexpr int kMaxRecords = 2 * SSP_STATS_STATIC_MAX_FIELDS;     // block partials of one call, all fields
static constexpr size_t kRecordBytes = sizeof(double) * ACC_N * (size_t)kMaxRecords;
static constexpr size_t kScratchBytes = kRecordBytes + sizeof(unsigned) * (size_t)kMaxFields;
static_assert(kScratchBytes == SSP_STATS_STATIC_BYTES, "include/ssp.h states the size of the static scratch");

// [kMaxRecords][ACC_N] doubles, then [kMaxFields] ticket counters.  In HOST code this name is only a handle for
// cudaGetSymbolAddress -- not a device address; the kernel is given the address looked up in static_scratch().
static __device__ __align__(256) unsigned char g_stats_scratch[kScratchBytes];

static __device__ __forceinline__ double warp_sum_d(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// grid (bpf, B), 256 threads; rows and lanes as k_stats_accum: lanes = 2^lane_shift threads share a row, each owning
// float4 pairs at fixed columns; fp32 within a row, double once per row, shuffles + shared memory per block.
__global__ void __launch_bounds__(256) k_stats_static(const float2 *__restrict__ field, int N, int lane_shift, int lo,
                                                       int hi, double dx, long long roi_n, double *acc,
                                                       unsigned *tickets, ssp_stats *__restrict__ out)
{
    const int b = blockIdx.y, bpf = gridDim.x, tid = threadIdx.x;
    const size_t px = (size_t)N * N;
    const float4 *f4 = reinterpret_cast<const float4 *>(field + (size_t)b * px);
    double a[ACC_N];
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) a[i] = 0.0;
    const int half = N / 2, lanes = 1 << lane_shift, rows_per_pass = 256 >> lane_shift;
    const int col0 = tid & (lanes - 1);
    for (int iy = blockIdx.x * rows_per_pass + (tid >> lane_shift); iy < N; iy += bpf * rows_per_pass) {
        const float4 *row = f4 + (size_t)iy * half;
        const bool roi_row = iy >= lo && iy < hi;
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, r1 = 0.f, r2 = 0.f, ax = 0.f;
        for (int c = col0; c < half; c += 4 * lanes) {
            float4 u[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
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
    __shared__ double part[8][ACC_N];
    __shared__ bool last;
    const int warp = tid >> 5, lane = tid & 31;
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) {
        const double s = warp_sum_d(a[i]);
        if (lane == 0) part[warp][i] = s;
    }
    __syncthreads();
    if (tid < ACC_N) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += part[w][tid];
        acc[((size_t)b * bpf + blockIdx.x) * ACC_N + tid] = s;
        __threadfence();                                   // the record is visible device-wide before the ticket is
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();                                   // cumulative: the nine writers' records (seen through the barrier) before the ticket
        last = atomicAdd(tickets + b, 1u) == (unsigned)(bpf - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();                                       // ... and the last block sees every other block's record

    // the finaliser of k_stats_final, run by the block that drew the last ticket: thread j adds the records
    // k = j, j + 256, ... in ascending order, a shuffle tree per warp, the eight warp sums in order, thread 0 finishes
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) a[i] = 0.0;
    for (int k = tid; k < bpf; k += 256) {
        const double *p = acc + ((size_t)b * bpf + k) * ACC_N;
#pragma unroll
        for (int i = 0; i < ACC_N; ++i) a[i] += __ldcg(p + i);          // written by other SMs in this launch: not through L1
    }
#pragma unroll
    for (int i = 0; i < ACC_N; ++i) {
        const double s = warp_sum_d(a[i]);
        if (lane == 0) part[warp][i] = s;
    }
    __syncthreads();
    if (tid == 0) {
        double t[ACC_N];
        for (int i = 0; i < ACC_N; ++i) {
            t[i] = 0.0;
            for (int w = 0; w < 8; ++w) t[i] += part[w][i];
        }
        out[b] = finalize_stats(t, dx, roi_n);
        tickets[b] = 0;                                    // left clean; the entry point clears them all the same
    }
}

// Device address of g_stats_scratch on the current device: looked up once per device (the symbol has one instance
// per GPU that loaded the module), with that device current.
static cudaError_t static_scratch(int device, unsigned char **out)
{
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static unsigned char *ptr[kMaxDevices] = {};
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_stats_scratch);
        if (e != cudaSuccess) return e;
        ptr[device] = static_cast<unsigned char *>(p);
    }
    *out = ptr[device];
    return cudaSuccess;
}

} // namespace ssp

using namespace ssp;

extern "C" int ssp_beam_stats_static(ssp_ctx *ctx, ssp_grid grid, int B, const float *d_field, double roi_frac,
                                     ssp_stats *d_stats)
{
    if (!ctx) return SSP_EINVAL;
    if (!valid_N(grid.N) || !(grid.dx > 0) || B < 1 || !d_field || (reinterpret_cast<uintptr_t>(d_field) & 15) || !d_stats)
        return ctx->fail(SSP_EINVAL, "bad grid, batch, field or statistics pointer");
    if (B > kMaxFields)
        return ctx->fail(SSP_EINVAL, "ssp_beam_stats_static: B=%d exceeds the static scratch (at most %d fields per call; "
                                     "split the batch or use ssp_beam_stats)", B, kMaxFields);
    SSP_CUDA(ctx, cudaSetDevice(ctx->device));
    unsigned char *scratch = nullptr;
    SSP_CUDA(ctx, static_scratch(ctx->device, &scratch));
    double *acc = reinterpret_cast<double *>(scratch);
    unsigned *tickets = reinterpret_cast<unsigned *>(scratch + kRecordBytes);

    const int N = grid.N;
    int lo, hi;
    long long roi_n;
    stats_roi(N, roi_frac, &lo, &hi, &roi_n);
    int lane_shift = 0;
    while ((2 << lane_shift) <= N / 2 && lane_shift < 6) ++lane_shift;        // lanes = min(64, N/2)
    const int rows_per_pass = 256 >> lane_shift;
    // blocks per field as launch_stats (all blocks resident, equal row passes), capped by the records that fit
    const int passes = (N + rows_per_pass - 1) / rows_per_pass;
    int target = (ctx->num_sms * 8) / B;
    if (target > kMaxRecords / B) target = kMaxRecords / B;                  // >= 2: B <= kMaxFields
    if (target < 1) target = 1;
    const int per = (passes + target - 1) / target;
    const int bpf = (passes + per - 1) / per;

    SSP_CUDA(ctx, cudaMemsetAsync(tickets, 0, sizeof(unsigned) * (size_t)B, ctx->stream));
    k_stats_static<<<dim3(bpf, B), 256, 0, ctx->stream>>>(reinterpret_cast<const float2 *>(d_field), N, lane_shift, lo, hi,
                                                          grid.dx, roi_n, acc, tickets, d_stats);
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}
