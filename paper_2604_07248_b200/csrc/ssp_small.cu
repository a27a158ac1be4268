// ssp_small.cu -- on-chip split-step propagation for small grids (N = 64, 128).
//
// At 128^2 a split step moves 0.59 MB: two kernel launches per step cost more than the step
// (SURVEY.md section 7, H9).  Here ONE CTA keeps a whole field in shared memory (N = 128:
// 152 x 152 complex64 = 185 KB) and runs every step of the stack on it; per step only the
// screen (4 B/px) is read from HBM.  The transforms are the in-register ones of ssp_fft.cuh:
// a thread loads its points of a row or column from the shared field, and the exchange of
// the transform goes through that line's own (now free) storage, padded to N + 24 slots.
//
// Sequence (the same as ssp_propagate / ssp_propagate_adjoint issue as separate kernels):
//   row(op 0);  for k = 1..n:  col(hy_k);  row(op k)
//   row = [IFFT_x] -> * exp(+-i phi) W -> [FFT_x] -> * hx,   col = FFT_y -> * hy/N^2 -> IFFT_y.   (Eq.1)
#include "ssp_kernels.cuh"
#include "ssp_stats.cuh"

namespace ssp {

template <int N>
struct SmallCfg {
    using PR = PlanInfo<N, 0>;
    using PC = PlanInfo<N, 1>;
    static_assert(PR::E == PC::E, "row and column plans share the thread count");
    static constexpr int E = PR::E;
    static constexpr int THREADS = N * (N / E);                   // every line of the field at once
    // >= the padded line length of either plan, and = 8 mod 16 so that adjacent rows start 16 banks apart
    static constexpr int PITCH = N + 24;
    static_assert(PITCH >= PR::LINE_ELEMS && PITCH >= PC::LINE_ELEMS, "exchange fits the line's own storage");
    static constexpr size_t SMEM = sizeof(float2) * (size_t)PITCH * PITCH;
};

// exchange accessors on the shared field: a row's slots are contiguous, a column's are PITCH apart
template <int PITCH>
struct SmallRowSmem {
    static constexpr int PAD = 1;
    float2 *base;
    __device__ __forceinline__ void st(int p, float2 x) { base[p] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p]; }
    __device__ __forceinline__ void sync() { __syncthreads(); }
};
template <int PITCH>
struct SmallColSmem {
    static constexpr int PAD = 1;
    float2 *base;
    __device__ __forceinline__ void st(int p, float2 x) { base[p * PITCH] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p * PITCH]; }
    __device__ __forceinline__ void sync() { __syncthreads(); }
};

template <int N>
__global__ void __launch_bounds__(SmallCfg<N>::THREADS, 1) k_small(const SmallArgs a)
{
    using CFG = SmallCfg<N>;
    using PR = typename CFG::PR;
    using PC = typename CFG::PC;
    constexpr int E = CFG::E, PITCH = CFG::PITCH;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *F = reinterpret_cast<float2 *>(smem_raw);
    const int tid = threadIdx.x, b = blockIdx.x;
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)

    // field -> shared memory, coalesced
    const float2 *src = a.in + (size_t)b * N * N;
    for (int i = tid; i < N * N; i += CFG::THREADS) F[(i / N) * PITCH + i % N] = src[i];
    __syncthreads();

    for (int op = 0; op <= a.n_steps; ++op) {
        const SmallStep s = a.steps[op];
        float2 v[E];
        if (op > 0) { // ---- column pass: lanes walk adjacent columns
            constexpr int T = PC::T, R1 = PC::R1, RL = PC::RL;
            const int c = tid % N, t = tid / N;
            SmallColSmem<PITCH> sm{F + c};
#pragma unroll
            for (int i = 0; i < E / R1; ++i)
#pragma unroll
                for (int q = 0; q < R1; ++q) v[i * R1 + q] = F[line_index<N, 1, R1>(t, i, q) * PITCH + c];
            __syncthreads();                                      // the column is in registers: its slots are free
            fft_line<N, 1, false, false, true>(v, t, sm, a.tw_col);
#pragma unroll
            for (int i = 0; i < E / RL; ++i)
#pragma unroll
                for (int q = 0; q < RL; ++q)
                    v[i * RL + q] = cmul(v[i * RL + q], __ldg(s.hy + line_index<N, 1, RL>(t, i, q)));
            fft_line<N, 1, true, true, true>(v, t, sm, a.tw_col);
#pragma unroll
            for (int i = 0; i < E / R1; ++i)
#pragma unroll
                for (int q = 0; q < R1; ++q) F[line_index<N, 1, R1>(t, i, q) * PITCH + c] = v[i * R1 + q];
            __syncthreads();
            (void)T;
        }
        { // ---- row pass
            constexpr int T = PR::T, R1 = PR::R1, RL = PR::RL;
            const int row = tid / T, t = tid % T;
            float2 *line = F + row * PITCH;
            SmallRowSmem<PITCH> sm{line};
            RowArgs r{};
            r.phi = s.phi;
            r.phase_sign = s.phase_sign;
            r.win_on = a.win_on && s.win; r.win_qs = a.win_qs; r.win_half_order = a.win_half_order;
            const float *phi_row = s.phi ? s.phi + b * s.phi_batch_stride + (long long)row * N : nullptr;
            const bool pointwise = s.phi || r.win_on;
            if (s.first) {
#pragma unroll
                for (int i = 0; i < E / R1; ++i)
#pragma unroll
                    for (int q = 0; q < R1; ++q) v[i * R1 + q] = line[line_index<N, 0, R1>(t, i, q)];
            } else {
#pragma unroll
                for (int i = 0; i < E / RL; ++i)
#pragma unroll
                    for (int q = 0; q < RL; ++q) v[i * RL + q] = line[line_index<N, 0, RL>(t, i, q)];
            }
            __syncthreads();
            if (s.first) fft_line<N, 0, false, true, true>(v, t, sm, a.tw_row);   // inverse; strided by RL
            if (pointwise) row_pointwise<N, RL, E, T, true, false>(v, r, phi_row, t, b, row);
            if (s.second) {
                fft_line<N, 0, true, false, true>(v, t, sm, a.tw_row);           // forward, reversed plan; strided by R1
#pragma unroll
                for (int i = 0; i < E / R1; ++i)
#pragma unroll
                    for (int q = 0; q < R1; ++q) {
                        const int k = line_index<N, 0, R1>(t, i, q);
                        line[k] = s.hx ? cmul(v[i * R1 + q], __ldg(s.hx + k)) : v[i * R1 + q];
                    }
            } else {
#pragma unroll
                for (int i = 0; i < E / RL; ++i)
#pragma unroll
                    for (int q = 0; q < RL; ++q) line[line_index<N, 0, RL>(t, i, q)] = v[i * RL + q];
                if (a.stats && op == a.n_steps) {
                    // K8 on the output pixels in registers (ssp_stats.cuh): row sums -> one record per row in shared
                    // memory -> moment i summed over the rows in row order by thread i -> finished here, no extra launch
                    static_assert(T <= 32, "a row's threads sit in one warp");
                    __shared__ double part[N][ROW_N];
                    __shared__ double accs[ACC_N];
                    double rs[ROW_N];
                    row_point_sums<N, RL, E, T>(v, t, row, a.roi_lo, a.roi_hi, rs);
                    group_sum<T>(rs);
                    if (t == 0) {
#pragma unroll
                        for (int i = 0; i < ROW_N; ++i) part[row][i] = rs[i];
                    }
                    __syncthreads();
                    if (tid < ACC_N) {
                        double sum = 0.0;
#pragma unroll 1
                        for (int r2 = 0; r2 < N; ++r2) sum += row_to_acc(tid, part[r2], (double)(r2 - N / 2));
                        accs[tid] = sum;
                    }
                    __syncthreads();
                    if (tid == 0) a.stats[b] = finalize_stats(accs, a.dx, a.roi_n);
                }
            }
            __syncthreads();
        }
    }
    float2 *dst = a.out + (size_t)b * N * N;
    for (int i = tid; i < N * N; i += CFG::THREADS) dst[i] = F[(i / N) * PITCH + i % N];
}

bool small_path_available(int N) { return N == 64 || N == 128; }

template <int N>
static int launch_small_n(ssp_ctx *ctx, int B, const SmallArgs &a)
{
    using CFG = SmallCfg<N>;
    auto kern = k_small<N>;
    SSP_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CFG::SMEM));
    // algorithmic bytes of the on-chip schedule: field in + out once, one screen per step
    ctx->prof_begin("small_on_chip", (16.0 + 4.0 * a.n_screens) * (double)B * N * N);
    SSP_CUDA(ctx, launch_pdl(kern, dim3(B), dim3(CFG::THREADS), CFG::SMEM, ctx->stream, pdl_enabled(), a));
    ctx->prof_end();
    ctx->launches++;
    SSP_CUDA(ctx, cudaGetLastError());
    return SSP_OK;
}

int launch_small(ssp_ctx *ctx, int N, int B, const SmallArgs &a)
{
    if (N == 64) return launch_small_n<64>(ctx, B, a);
    if (N == 128) return launch_small_n<128>(ctx, B, a);
    return ctx->fail(SSP_EINVAL, "no on-chip path for N=%d", N);
}

} // namespace ssp
