// ssp_cluster.cu -- on-chip split-step propagation with ONE FIELD SPLIT OVER A THREAD-BLOCK CLUSTER
// (second half; H9).
//
// The single-CTA kernel of ssp_small.cu keeps a whole field in one SM's shared memory: a batch of B fields keeps B
// of the 148 SMs busy and one 128^2 step costs ~19 us of one SM's arithmetic.  Here a cluster of CS = 8 CTAs shares
// the field: CTA r holds the row slab A (rows r L .. r L + L - 1, L = N / CS) for the row passes and the column slab
// Bs (columns r L ..) for the column passes.  A pass transforms its lines locally (the in-register transforms of
// ssp_fft.cuh, exchange inside the line's own storage) and writes every result straight into the slab of the CTA that
// owns it in the other orientation -- a transpose through distributed shared memory (st.shared::cluster via
// cluster.map_shared_rank), one cluster barrier per pass.  Per step only the screen (4 B/px) comes from HBM.
//   row(op 0);  for k = 1..n:  col(hy_k);  row(op k)          (the sequence of ssp_small.cu; Eq.1)
#include <cooperative_groups.h>

#include <cstdlib>

#include "ssp_kernels.cuh"
#include "ssp_stats.cuh"

namespace cg = cooperative_groups;

namespace ssp {

template <int N>
struct ClusterCfg {
    using PR = PlanInfo<N, 0>;
    using PC = PlanInfo<N, 1>;
    static_assert(PR::E == PC::E, "row and column plans share the thread count");
    static constexpr int CS = 8;                                   // CTAs per field (portable cluster size)
    static constexpr int E = PR::E, T = N / E;
    static constexpr int L = N / CS;                               // lines per CTA and pass
    static constexpr int THREADS = L * T;
    static constexpr int PITCH = N + 24;                           // as ssp_small.cu: room for the exchange padding
    static_assert(PITCH >= PR::LINE_ELEMS && PITCH >= PC::LINE_ELEMS, "exchange fits the line's own storage");
    static constexpr int SLAB = L * PITCH;
    static constexpr size_t SMEM = sizeof(float2) * 2 * (size_t)SLAB;
};

template <int PITCH>
struct ClusterLineSmem {
    static constexpr int PAD = 1;
    float2 *base;
    __device__ __forceinline__ void st(int p, float2 x) { base[p] = x; }
    __device__ __forceinline__ float2 ld(int p) const { return base[p]; }
    __device__ __forceinline__ void sync() { __syncthreads(); }
};

template <int N>
__global__ void __launch_bounds__(ClusterCfg<N>::THREADS, 1) k_cluster(const SmallArgs a)
{
    using CFG = ClusterCfg<N>;
    using PR = typename CFG::PR;
    using PC = typename CFG::PC;
    constexpr int E = CFG::E, T = CFG::T, L = CFG::L, PITCH = CFG::PITCH, CS = CFG::CS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *A = reinterpret_cast<float2 *>(smem_raw);              // my rows:    A[row_local][ix]
    float2 *Bs = A + CFG::SLAB;                                    // my columns: Bs[col_local][iy]
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int tid = threadIdx.x, b = blockIdx.x / CS;
    const int ll = tid / T, t = tid % T;                           // local line, thread within the line
    const int gl = rank * L + ll;                                  // global row (row pass) / column (column pass)
    pdl_wait();                                                    // (ssp_internal.h: programmatic dependent launch)

    const float2 *src = a.in + ((size_t)b * N + (size_t)rank * L) * N;
    for (int i = tid; i < L * N; i += CFG::THREADS) A[(i / N) * PITCH + i % N] = src[i];
    cluster.sync();                                                // every CTA of the cluster runs: its shared memory may be written

    for (int op = 0; op <= a.n_steps; ++op) {
        const SmallStep s = a.steps[op];
        float2 v[E];
        if (op > 0) { // ---- column pass on Bs; result -> the row slabs A of the owners of the rows
            constexpr int R1 = PC::R1, RL = PC::RL;
            float2 *line = Bs + ll * PITCH;
            ClusterLineSmem<PITCH> sm{line};
#pragma unroll
            for (int i = 0; i < E / R1; ++i)
#pragma unroll
                for (int q = 0; q < R1; ++q) v[i * R1 + q] = line[line_index<N, 1, R1>(t, i, q)];
            __syncthreads();
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
                for (int q = 0; q < R1; ++q) {
                    const int iy = line_index<N, 1, R1>(t, i, q);
                    float2 *dstA = cluster.map_shared_rank(A, iy / L);
                    dstA[(iy % L) * PITCH + gl] = v[i * R1 + q];
                }
            cluster.sync();
        }
        { // ---- row pass on A; result -> the column slabs Bs of the owners of the columns (or, last op, global memory)
            constexpr int R1 = PR::R1, RL = PR::RL;
            float2 *line = A + ll * PITCH;
            ClusterLineSmem<PITCH> sm{line};
            RowArgs r{};
            r.phi = s.phi;
            r.phase_sign = s.phase_sign;
            r.win_on = a.win_on && s.win; r.win_qs = a.win_qs; r.win_half_order = a.win_half_order;
            const float *phi_row = s.phi ? s.phi + b * s.phi_batch_stride + (long long)gl * N : nullptr;
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
            if (pointwise) row_pointwise<N, RL, E, T, true, false>(v, r, phi_row, t, b, gl);
            if (s.second) {
                fft_line<N, 0, true, false, true>(v, t, sm, a.tw_row);           // forward, reversed plan; strided by R1
#pragma unroll
                for (int i = 0; i < E / R1; ++i)
#pragma unroll
                    for (int q = 0; q < R1; ++q) {
                        const int k = line_index<N, 0, R1>(t, i, q);
                        const float2 x = s.hx ? cmul(v[i * R1 + q], __ldg(s.hx + k)) : v[i * R1 + q];
                        float2 *dstB = cluster.map_shared_rank(Bs, k / L);
                        dstB[(k % L) * PITCH + gl] = x;
                    }
                cluster.sync();
            } else {
                float2 *dst = a.out + ((size_t)b * N + gl) * N;
#pragma unroll
                for (int i = 0; i < E / RL; ++i)
#pragma unroll
                    for (int q = 0; q < RL; ++q) dst[line_index<N, 0, RL>(t, i, q)] = v[i * RL + q];
                if (a.stats_acc) {
                    // K8 on the output pixels in registers: one record of the nine accumulators per row (ssp_stats.cuh),
                    // added per field in a fixed order by k_stats_final
                    static_assert(T <= 32, "a row's threads sit in one warp");
                    double rs[ROW_N];
                    row_point_sums<N, RL, E, T>(v, t, gl, a.roi_lo, a.roi_hi, rs);
                    group_sum<T>(rs);
                    const double y = (double)(gl - N / 2);
                    for (int m = t; m < ACC_N; m += T) a.stats_acc[((size_t)b * N + gl) * ACC_N + m] = row_to_acc(m, rs, y);
                }
            }
        }
    }
}

bool cluster_path_available(int N, int B)
{
    static const bool off = getenv("SSP_NO_CLUSTER") != nullptr;  // measurement switch: take the other paths
    if (off) return false;
    // one field per 8 SMs: pays while the single-CTA kernel (one SM per field) or the two-kernel path would leave
    // most of the 148 SMs idle
    // measured (forward + adjoint of 5 steps + statistics, us): 128^2: 78 / 78 / 98 / 219 at B = 1 / 4 / 16 / 64 against 283
    // for the single-CTA kernel at every B <= 64; 256^2: 205 (B <= 8) against 138-159 for the two-kernel path -- its
    // scattered 8-byte remote stores cost more than the launches they save -- so 256^2 stays on the row / column kernels
    return N == 128 && B <= 64;
}

template <int N>
static int launch_cluster_n(ssp_ctx *ctx, int B, const SmallArgs &a)
{
    using CFG = ClusterCfg<N>;
    auto kern = k_cluster<N>;
    SSP_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CFG::SMEM));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(B * CFG::CS));
    cfg.blockDim = dim3(CFG::THREADS);
    cfg.dynamicSmemBytes = CFG::SMEM;
    cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CFG::CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl_enabled() ? 2 : 1;
    ctx->prof_begin("cluster_on_chip", (16.0 + 4.0 * a.n_screens) * (double)B * N * N);
    SSP_CUDA(ctx, cudaLaunchKernelEx(&cfg, kern, a));
    ctx->prof_end();
    ctx->launches++;
    return SSP_OK;
}

int launch_cluster(ssp_ctx *ctx, int N, int B, const SmallArgs &a)
{
    if (N == 128) return launch_cluster_n<128>(ctx, B, a);
    return ctx->fail(SSP_EINVAL, "no cluster path for N=%d", N);
}

} // namespace ssp
