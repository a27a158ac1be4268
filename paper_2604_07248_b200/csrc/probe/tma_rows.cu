// tma_rows.cu -- stand-alone probe: what a plain TMA copy of column tiles reaches on this GPU, by tile width.
//
// The column kernels (ssp_col_tma.cuh) move tiles of C adjacent columns x N rows of a complex64 [rows][N] matrix with
// TMA boxes of 256 rows: every tile row is one 8 C-byte segment.  This program measures the same traffic without any
// arithmetic -- persistent CTAs, one thread each, load a tile into shared memory and store it back to a second matrix,
// NBUF tiles in flight per CTA -- and prints GB/s (read + write) and tile rows per clock and SM.  The TMA engine moves
// about 0.5-0.7 rows per clock and SM whatever their width, so 16-byte rows stop near 3 TB/s and 32-byte rows near
// 5 TB/s; from 64-byte rows on HBM is the limit (profiles/r02_tma_rows.md).  Tuning aid, not part of libssp.so:
//     python -m paper_2604_07248_b200.build --probe   ->  paper_2604_07248_b200/csrc/build/tma_rows
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <vector>
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile("{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *tm, int x, int y, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(dst)), "l"(tm), "r"(x), "r"(y), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap *tm, int x, int y, const void *src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tm), "r"(x), "r"(y), "r"(smem_u32(src)) : "memory");
}
// one thread per CTA drives everything; NBUF buffers in a ring: load tile i+NBUF-1 ahead
template <int C, int NBUF>
__global__ void k_copy(const __grid_constant__ CUtensorMap tin, const __grid_constant__ CUtensorMap tout, int N, int ROWS, int ntiles)
{
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned long long *full = reinterpret_cast<unsigned long long *>(smem);
    unsigned char *buf = smem + 128;
    const size_t tile_bytes = (size_t)ROWS * C * 8;
    const int groups = N / C, boxes = ROWS / 256;
    if (threadIdx.x != 0) return;
    for (int i = 0; i < NBUF; ++i) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    auto issue = [&](int n) {
        const int tile = blockIdx.x + n * gridDim.x, b = n % NBUF;
        const int blk = tile / groups, col0 = (tile % groups) * C;
        mbar_expect_tx(&full[b], (unsigned)tile_bytes);
        for (int j = 0; j < boxes; ++j) tma_load_2d(buf + b * tile_bytes + (size_t)j * 256 * C * 8, &tin, 2 * col0, blk * ROWS + j * 256, &full[b]);
    };
    const int mine = (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    for (int n = 0; n < NBUF && n < mine; ++n) issue(n);
    for (int n = 0; n < mine; ++n) {
        const int tile = blockIdx.x + n * gridDim.x, b = n % NBUF;
        const int blk = tile / groups, col0 = (tile % groups) * C;
        mbar_wait(&full[b], (n / NBUF) & 1);
        for (int j = 0; j < boxes; ++j) tma_store_2d(&tout, 2 * col0, blk * ROWS + j * 256, buf + b * tile_bytes + (size_t)j * 256 * C * 8);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        if (n + NBUF < mine) {
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            issue(n + NBUF);
        }
    }
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static CUtensorMap make_map(EncodeFn enc, void *base, int N, size_t rows, int C)
{
    CUtensorMap m;
    cuuint64_t dims[2] = {(cuuint64_t)2 * N, (cuuint64_t)rows}, strides[1] = {(cuuint64_t)N * 8};
    cuuint32_t box[2] = {(cuuint32_t)2 * C, 256}, es[2] = {1, 1};
    CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { printf("encode failed %d\n", (int)r); exit(1); }
    return m;
}
template <int C, int NBUF>
static void run(EncodeFn enc, float *in, float *out, int N, int ROWS, int B, int ctas_per_sm)
{
    const size_t rows = (size_t)B * ROWS;
    CUtensorMap tin = make_map(enc, in, N, rows, C), tout = make_map(enc, out, N, rows, C);
    const size_t smem = 128 + (size_t)NBUF * ROWS * C * 8;
    cudaFuncSetAttribute(k_copy<C, NBUF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int ntiles = B * (N / C), grid = 148 * ctas_per_sm;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int w = 0; w < 2; ++w) k_copy<C, NBUF><<<grid, 32, smem>>>(tin, tout, N, ROWS, ntiles);
    cudaEventRecord(e0);
    const int reps = 10;
    for (int r = 0; r < reps; ++r) k_copy<C, NBUF><<<grid, 32, smem>>>(tin, tout, N, ROWS, ntiles);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    cudaError_t e = cudaGetLastError();
    const double bytes = 16.0 * (double)rows * N;
    printf("N=%d ROWS=%d C=%d (%d-byte rows) NBUF=%d CTAs/SM=%d smem=%zu KB: %.1f GB/s  (%.3f rows/clk/SM at 1.9 GHz) %s\n", N, ROWS, C, C * 8, NBUF, ctas_per_sm,
           smem / 1024, bytes * reps / ms / 1e6, 2.0 * rows * (N / C) * reps / (ms * 1e-3) / 1.9e9 / 148, cudaGetErrorString(e));
}
int main()
{
    void *fn = nullptr; cudaDriverEntryPointQueryResult q;
    cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    EncodeFn enc = (EncodeFn)fn;
    const size_t bytes = (size_t)1 << 30;           // 1 GB in + 1 GB out: B fields of N^2 complex64 each way
    float *in, *out;
    cudaMalloc(&in, bytes); cudaMalloc(&out, bytes);
    cudaMemset(in, 1, bytes);
    // the column kernels' own shapes (tile = C columns x N rows of an N^2 field), then wider / narrower tiles
    printf("-- 1024^2 fields (k_col_tma<1024>: C = 4, two buffers, 3 CTAs/SM)\n");
    run<4, 2>(enc, in, out, 1024, 1024, 128, 3);
    run<2, 2>(enc, in, out, 1024, 1024, 128, 6);
    run<8, 2>(enc, in, out, 1024, 1024, 128, 1);
    run<8, 3>(enc, in, out, 1024, 1024, 128, 1);
    run<16, 1>(enc, in, out, 1024, 1024, 128, 1);
    printf("-- 2048^2 fields (k_col_tma<2048>: C = 4, three buffers, 1 CTA/SM; before: one buffer, 2 CTAs/SM)\n");
    run<4, 3>(enc, in, out, 2048, 2048, 32, 1);
    run<4, 1>(enc, in, out, 2048, 2048, 32, 2);
    run<2, 1>(enc, in, out, 2048, 2048, 32, 6);
    run<8, 1>(enc, in, out, 2048, 2048, 32, 1);
    printf("-- 4096^2 fields (k_col_tma<4096>: C = 2, one buffer, 2 CTAs/SM; k_col_tma_wide<4096>: C = 4, one landing buffer)\n");
    run<2, 1>(enc, in, out, 4096, 4096, 8, 2);
    run<2, 1>(enc, in, out, 4096, 4096, 8, 3);
    run<2, 3>(enc, in, out, 4096, 4096, 8, 1);
    run<4, 1>(enc, in, out, 4096, 4096, 8, 1);
    return 0;
}
