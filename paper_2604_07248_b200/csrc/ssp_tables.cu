// ssp_tables.cu -- small device tables owned by the context: FFT inter-stage twiddles,
// 1-D transfer-function tables, sign tables.  All built in double on the host (SURVEY.md
// section 7, H4: pi*lambda*dz*f^2 reaches hundreds of radians; fp32 device sincos of it
// would lose the phase), rounded once to fp32 and cached.
#include <cmath>

#include "ssp_fft.cuh"
#include <cstdlib>

#include "ssp_internal.h"

namespace ssp {

bool pdl_enabled()
{
    static const bool off = getenv("SSP_NO_PDL") != nullptr;
    return !off;
}

bool valid_N(int N) { return N >= 8 && N <= 4096 && (N & (N - 1)) == 0; }

static int upload(ssp_ctx *ctx, const std::vector<float2> &h, float2 **out)
{
    float2 *d = nullptr;
    SSP_CUDA(ctx, cudaMalloc(&d, h.size() * sizeof(float2)));
    // pageable source: cudaMemcpyAsync stages it before returning, so `h` may die afterwards
    cudaError_t e = cudaMemcpyAsync(d, h.data(), h.size() * sizeof(float2), cudaMemcpyHostToDevice, ctx->stream);
    if (e != cudaSuccess) {
        cudaFree(d);
        return ctx->fail(SSP_ECUDA, "table upload failed: %s", cudaGetErrorString(e));
    }
    *out = d;
    return SSP_OK;
}

static float2 wn(long long e, int N) // exp(-i 2 pi e / N), e reduced mod N first
{
    const double kPi = 3.14159265358979323846;
    e %= N;
    double ang = -2.0 * kPi * (double)e / (double)N;
    return make_float2((float)cos(ang), (float)sin(ang));
}

template <int N, int V>
static void fill_twiddles(std::vector<float2> &h)
{
    using PI = PlanInfo<N, V>;
    h.assign(PI::TW_TOTAL, make_float2(1.f, 0.f));
    // forward plan (R1, R2, R3)
    // first-stage tables: [k / 2][m][k % 2], so that one 16-byte load brings the twiddles of k and k + 1
    for (int k = 0; k < PI::R1; ++k)
        for (int m = 0; m < N / PI::R1; ++m)
            h[PI::TW1 + ((k / 2) * (N / PI::R1) + m) * 2 + (k & 1)] = wn((long long)m * k, N);
    for (int k = 0; k < PI::R2; ++k)
        for (int n3 = 0; n3 < PI::R3; ++n3) h[PI::TW2 + k * PI::R3 + n3] = wn((long long)PI::R1 * n3 * k, N);
    // reversed plan (RL, .., R1): first radix RL, third radix R1
    for (int k = 0; k < PI::RL; ++k)
        for (int m = 0; m < N / PI::RL; ++m)
            h[PI::TW1R + ((k / 2) * (N / PI::RL) + m) * 2 + (k & 1)] = wn((long long)m * k, N);
    for (int k = 0; k < PI::R2; ++k)
        for (int n3 = 0; n3 < PI::R1; ++n3) h[PI::TW2R + k * PI::R1 + n3] = wn((long long)PI::RL * n3 * k, N);
}

int get_twiddles(ssp_ctx *ctx, int N, int V, const float2 **out)
{
    const int key = 4 * N + V;
    auto it = ctx->twiddles.find(key);
    if (it != ctx->twiddles.end()) { *out = it->second; return SSP_OK; }
    std::vector<float2> h;
    switch (N) {
    case 8: V == 2 ? fill_twiddles<8, 2>(h) : (V ? fill_twiddles<8, 1>(h) : fill_twiddles<8, 0>(h)); break;
    case 16: V == 2 ? fill_twiddles<16, 2>(h) : (V ? fill_twiddles<16, 1>(h) : fill_twiddles<16, 0>(h)); break;
    case 32: V == 2 ? fill_twiddles<32, 2>(h) : (V ? fill_twiddles<32, 1>(h) : fill_twiddles<32, 0>(h)); break;
    case 64: V == 2 ? fill_twiddles<64, 2>(h) : (V ? fill_twiddles<64, 1>(h) : fill_twiddles<64, 0>(h)); break;
    case 128: V == 2 ? fill_twiddles<128, 2>(h) : (V ? fill_twiddles<128, 1>(h) : fill_twiddles<128, 0>(h)); break;
    case 256: V == 2 ? fill_twiddles<256, 2>(h) : (V ? fill_twiddles<256, 1>(h) : fill_twiddles<256, 0>(h)); break;
    case 512: V == 2 ? fill_twiddles<512, 2>(h) : (V ? fill_twiddles<512, 1>(h) : fill_twiddles<512, 0>(h)); break;
    case 1024: V == 2 ? fill_twiddles<1024, 2>(h) : (V ? fill_twiddles<1024, 1>(h) : fill_twiddles<1024, 0>(h)); break;
    case 2048: V == 2 ? fill_twiddles<2048, 2>(h) : (V ? fill_twiddles<2048, 1>(h) : fill_twiddles<2048, 0>(h)); break;
    case 4096: V == 2 ? fill_twiddles<4096, 2>(h) : (V ? fill_twiddles<4096, 1>(h) : fill_twiddles<4096, 0>(h)); break;
    default: return ctx->fail(SSP_EINVAL, "unsupported N=%d", N);
    }
    float2 *d = nullptr;
    if (int rc = upload(ctx, h, &d)) return rc;
    ctx->twiddles[key] = d;
    *out = d;
    return SSP_OK;
}

// h[k] = exp(-+ i pi lam_eff dz f_k^2) [/ N^2], f_k in FFT order (negative Nyquist).
// The Fresnel kernel is separable: H(kx,ky) = h[kx] h[ky]  (north_star).
int get_htable(ssp_ctx *ctx, const HKey &key, const float2 **out)
{
    auto it = ctx->htables.find(key);
    if (it != ctx->htables.end()) { *out = it->second; return SSP_OK; }
    const double kPi = 3.14159265358979323846;
    const int N = key.N;
    std::vector<float2> h(N);
    const double scale = key.scaled ? 1.0 / ((double)N * (double)N) : 1.0;
    for (int k = 0; k < N; ++k) {
        const int ks = (k < N / 2) ? k : k - N;
        const double f = (double)ks / ((double)N * key.dx);
        double ang = -kPi * key.lam_eff * key.dz * f * f;
        ang = fmod(ang, 2.0 * kPi);
        if (key.conj) ang = -ang;
        h[k] = make_float2((float)(scale * cos(ang)), (float)(scale * sin(ang)));
    }
    float2 *d = nullptr;
    if (int rc = upload(ctx, h, &d)) return rc;
    ctx->htables[key] = d;
    *out = d;
    return SSP_OK;
}

// Callers may collect several table pointers before launching (the on-chip path gathers the tables of a whole
// stack), so get_htable never frees: the cap is enforced here, once, at the entry of a propagation call.
int trim_htables(ssp_ctx *ctx)
{
    if (ctx->htables.size() <= 4096) return SSP_OK;   // unbounded dz lists: drop the cache rather than grow
    SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (auto &kv : ctx->htables) cudaFree(kv.second);
    ctx->htables.clear();
    return SSP_OK;
}

int get_h2d_table(ssp_ctx *ctx, const HKey &key, const float2 **out)
{
    auto it = ctx->h2d_tables.find(key);
    if (it != ctx->h2d_tables.end()) { *out = it->second; return SSP_OK; }
    const size_t bytes = sizeof(float2) * (size_t)key.N * key.N;
    if (ctx->h2d_bytes + bytes > ((size_t)1 << 30)) { // long dz lists on big grids: drop the cache rather than grow
        SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        for (auto &kv : ctx->h2d_tables) cudaFree(kv.second);
        ctx->h2d_tables.clear();
        ctx->h2d_bytes = 0;
    }
    float2 *d = nullptr;
    SSP_CUDA(ctx, cudaMalloc(&d, bytes));
    if (int rc = launch_h2d_table(ctx, key.N, col_tile_width(key.N), key.dx, key.lam_eff, key.dz, key.conj, d)) {
        cudaFree(d);
        return rc;
    }
    ctx->h2d_tables[key] = d;
    ctx->h2d_bytes += bytes;
    *out = d;
    return SSP_OK;
}

// s[k] = (-1)^k: the centred DFT is (-1)^k FFT((-1)^n x) / sqrt(N) per axis (N % 4 == 0).
int get_sign_table(ssp_ctx *ctx, int N, const float2 **out)
{
    auto it = ctx->sign_tables.find(N);
    if (it != ctx->sign_tables.end()) { *out = it->second; return SSP_OK; }
    std::vector<float2> h(2 * N);
    const double s = 1.0 / sqrt((double)N);
    for (int k = 0; k < N; ++k) {
        h[k] = make_float2((k & 1) ? -1.f : 1.f, 0.f);             // plain signs
        h[N + k] = make_float2((float)((k & 1) ? -s : s), 0.f);    // signs / sqrt(N)
    }
    float2 *d = nullptr;
    if (int rc = upload(ctx, h, &d)) return rc;
    ctx->sign_tables[N] = d;
    *out = d;
    return SSP_OK;
}

typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tmap_c64(ssp_ctx *ctx, const void *base, size_t cols, size_t rows, int box_cols, int box_rows,
                  CUtensorMap *out)
{
    if (!ctx->encode_tiled) {
        cudaDriverEntryPointQueryResult q;
        void *p = nullptr;
        SSP_CUDA(ctx, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q));
        if (!p || q != cudaDriverEntryPointSuccess)
            return ctx->fail(SSP_EUNSUPPORTED, "the driver does not export cuTensorMapEncodeTiled");
        ctx->encode_tiled = p;
    }
    const auto key = std::make_tuple(base, cols, rows, box_cols, box_rows);
    auto it = ctx->tmaps.find(key);
    if (it != ctx->tmaps.end()) { *out = it->second; return SSP_OK; }
    if (ctx->tmaps.size() >= 256) ctx->tmaps.clear();             // descriptors are values: nothing to free
    // complex64 as pairs of fp32: the inner dimension counts floats
    const cuuint64_t dims[2] = {(cuuint64_t)cols * 2, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)cols * sizeof(float2)};
    const cuuint32_t box[2] = {(cuuint32_t)box_cols * 2, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = reinterpret_cast<encode_tiled_fn>(ctx->encode_tiled)(
        out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(base), dims, strides, box, estr,
        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ctx->fail(SSP_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    ctx->tmaps[key] = *out;
    return SSP_OK;
}

int ensure_scratch(ssp_ctx *ctx, size_t bytes)
{
    if (bytes <= ctx->scratch_bytes) return SSP_OK;
    if (ctx->scratch) {
        SSP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->scratch);
        ctx->scratch = nullptr;
        ctx->scratch_bytes = 0;
    }
    size_t want = bytes < (1u << 16) ? (1u << 16) : bytes;
    SSP_CUDA(ctx, cudaMalloc(&ctx->scratch, want));
    ctx->scratch_bytes = want;
    return SSP_OK;
}

} // namespace ssp
