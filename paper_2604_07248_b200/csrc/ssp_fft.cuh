// ssp_fft.cuh -- in-register complex64 FFT building blocks for sm_100a.
//
// A length-N line (row or column of the field) is transformed by T = N/E threads that
// each hold E points in registers.  N = R1*R2*R3 (mixed radix, each radix <= E): every
// stage is a set of radix-R butterflies computed entirely in registers with compile-time
// twiddles; between stages the line is exchanged once through shared memory, multiplied
// by the inter-stage twiddles W_N^(rho*k) read from a table built in double precision on
// the host.  With (R1,R2) = (32,32) a 1024-point transform costs ONE shared-memory
// round trip.
//
// Index maps (decimation in frequency, in place; derivation in DESIGN.md section 6):
//   input  n = n1*(N/R1) + n2*R3 + n3,   output k = k1 + R1*k2 + R1*R2*k3
//   stage 1: butterfly m=(n2,n3):   A[k1;m]   = sum_n1 x[n1*(N/R1)+m] W_R1^(n1 k1),  *= W_N^(m k1)
//   stage 2: butterfly (k1,n3):     B[k1,k2;n3] = sum_n2 A[k1;n2,n3] W_R2^(n2 k2),   *= W_N^(R1 n3 k2)
//   stage 3: butterfly (k1,k2):     X[k]      = sum_n3 B[k1,k2;n3] W_R3^(n3 k3)
// Register layout "strided by R": thread t holds, for i in [0,E/R), j = t + T*i, the
// elements  v[i*R + q] <-> line index q*(N/R) + j.  A plan's input layout is strided by
// R1 and its output layout strided by its last radix, so the plan (R1,R2,R3) followed by
// the reversed plan (R3,R2,R1) chains register to register with no exchange in between.
#pragma once

#include <cuda_runtime.h>
#include <type_traits>
#include <utility>

namespace ssp {

__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cmul_conj(float2 a, float2 b) // a * conj(b)
{
    return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y));
}

// Packed fp32 pairs (sm_100 FFMA2 / FMUL2 / FADD2): one issue slot does both components of a complex value, and
// the SASS operand modifiers (broadcast .F32, swap .LO_HI, per-lane negate .NP) absorb the shuffles of a complex
// multiply.  Measured on B200: FFMA2 runs at the SAME 128 FMA/clk/SM as scalar FFMA (half the
// issue rate), so packing frees issue slots but no FMA-pipe time, and aligned register pairs raise register
// pressure.  It is therefore opt-in per kernel (template parameter PK), on where it measured faster.
__device__ __forceinline__ float2 f2fma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 f2mul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 f2add(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 f2sub(float2 a, float2 b) { return f2fma(make_float2(-1.f, -1.f), b, a); }
// A complex multiply by a run-time factor stays scalar under PK as well: its per-lane sign falls on a register pair
// that also carries the broadcast operand's partner, ptxas then materialises the negated pair (MOV + FADD), and the
// packed form ends at 4 issue slots / 5 pipe cycles against 4 / 4 for the scalar one.
template <bool CONJ, bool PK = false>
__device__ __forceinline__ float2 cmul_c(float2 a, float2 b)
{
    return CONJ ? cmul_conj(a, b) : cmul(a, b);
}

// cos(2 pi k / 64), k = 0..63 (double-precision values rounded once to fp32)
__host__ __device__ constexpr float cos64(int k)
{
    constexpr float t[64] = {
        1.0f, 0.9951847266721969f, 0.9807852804032304f, 0.9569403357322088f,
        0.9238795325112867f, 0.881921264348355f, 0.8314696123025452f, 0.773010453362737f,
        0.7071067811865476f, 0.6343932841636455f, 0.5555702330196023f, 0.4713967368259978f,
        0.38268343236508984f, 0.29028467725446233f, 0.19509032201612833f, 0.09801714032956077f,
        6.123233995736766e-17f, -0.09801714032956065f, -0.1950903220161282f, -0.29028467725446216f,
        -0.3826834323650897f, -0.4713967368259977f, -0.555570233019602f, -0.6343932841636454f,
        -0.7071067811865475f, -0.773010453362737f, -0.8314696123025453f, -0.8819212643483549f,
        -0.9238795325112867f, -0.9569403357322088f, -0.9807852804032304f, -0.9951847266721968f,
        -1.0f, -0.9951847266721969f, -0.9807852804032304f, -0.9569403357322089f,
        -0.9238795325112868f, -0.881921264348355f, -0.8314696123025455f, -0.7730104533627371f,
        -0.7071067811865477f, -0.6343932841636459f, -0.5555702330196022f, -0.47139673682599786f,
        -0.38268343236509034f, -0.29028467725446244f, -0.19509032201612866f, -0.09801714032956045f,
        -1.8369701987210297e-16f, 0.09801714032956009f, 0.1950903220161283f, 0.29028467725446205f,
        0.38268343236509f, 0.4713967368259976f, 0.5555702330196018f, 0.6343932841636456f,
        0.7071067811865474f, 0.7730104533627367f, 0.8314696123025452f, 0.8819212643483548f,
        0.9238795325112865f, 0.9569403357322088f, 0.9807852804032303f, 0.9951847266721969f};
    return t[k & 63];
}
__host__ __device__ constexpr float sin64(int k) { return cos64(k - 16); }

// ---- radix-R butterflies in registers: decimation in time, FMA form ----------------------------------
// One DIT butterfly (a, b) -> (a + w b, a - w b) with w = W_L^J = exp(-/+ i 2 pi J / L) (forward / inverse),
// L, J compile-time.  Trivial w (1, -/+i) cost 4 additions.  Any other w costs 6 FMAs instead of the 8
// operations of "multiply, then add and subtract":  X = a + w b as two chained FMAs per component with w's
// components as immediates, and Y = a - w b = 2 a - X as one more FMA per component.
// PK: the same butterflies on packed pairs: 2 issue slots for a trivial twiddle (the -/+i swap and sign are operand
// modifiers), 3 for any other.
template <int L, int J, bool INV, bool PK>
__device__ __forceinline__ void bfly_dit(float2 &a, float2 &b)
{
    static_assert(L <= 64, "butterfly constants are tabulated for radices up to 64");
    constexpr int k64 = (J * (64 / L)) & 63;                      // w = W_64^k64, k64 < 32 since J < L/2
    if constexpr (PK) {
    if constexpr (k64 == 0) {
        const float2 x = f2add(a, b), y = f2sub(a, b);
        a = x; b = y;
    } else if constexpr (k64 == 16) {                              // w = -i (forward), +i (inverse): w b = -/+ (-b.y, b.x)
        constexpr float s = INV ? 1.f : -1.f;
        const float2 ib = make_float2(-b.y, b.x);
        const float2 x = f2fma(make_float2(s, s), ib, a), y = f2fma(make_float2(-s, -s), ib, a);
        a = x; b = y;
    } else {
        constexpr float wr = cos64(k64);
        constexpr float wi = INV ? sin64(k64) : -sin64(k64);
        const float2 x = f2fma(make_float2(wi, wi), make_float2(-b.y, b.x), f2fma(make_float2(wr, wr), b, a));
        const float2 y = f2fma(make_float2(2.f, 2.f), a, make_float2(-x.x, -x.y));
        a = x; b = y;
    }
    } else {
    if constexpr (k64 == 0) {
        const float2 x = make_float2(a.x + b.x, a.y + b.y), y = make_float2(a.x - b.x, a.y - b.y);
        a = x; b = y;
    } else if constexpr (k64 == 16) {                              // w = -i (forward), +i (inverse)
        const float2 wb = INV ? make_float2(-b.y, b.x) : make_float2(b.y, -b.x);
        const float2 x = make_float2(a.x + wb.x, a.y + wb.y), y = make_float2(a.x - wb.x, a.y - wb.y);
        a = x; b = y;
    } else {
        constexpr float wr = cos64(k64);
        constexpr float wi = INV ? sin64(k64) : -sin64(k64);
        const float2 x = make_float2(fmaf(wr, b.x, fmaf(-wi, b.y, a.x)), fmaf(wr, b.y, fmaf(wi, b.x, a.y)));
        const float2 y = make_float2(fmaf(2.f, a.x, -x.x), fmaf(2.f, a.y, -x.y));
        a = x; b = y;
    }
    }
}

__host__ __device__ constexpr int bitrev(int i, int R)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) {
        r = (r << 1) | (i & 1);
        i >>= 1;
    }
    return r;
}

template <int R, int... I>
__device__ __forceinline__ void scramble(float2 *v, std::integer_sequence<int, I...>)
{
    float2 t[R];
    ((t[I] = v[bitrev(I, R)]), ...);
    ((v[I] = t[I]), ...);
}

// all butterflies of the level that merges transforms of length L/2 into length L
template <int R, int L, bool INV, bool PK, int... B>
__device__ __forceinline__ void dit_level(float2 *v, std::integer_sequence<int, B...>)
{
    // butterfly index B in [0, R/2): group B / (L/2), position J = B % (L/2)
    (bfly_dit<L, B % (L / 2), INV, PK>(v[(B / (L / 2)) * L + B % (L / 2)], v[(B / (L / 2)) * L + B % (L / 2) + L / 2]), ...);
}

template <int R, int L, bool INV, bool PK>
__device__ __forceinline__ void dit_levels(float2 *v)
{
    if constexpr (L <= R) {
        dit_level<R, L, INV, PK>(v, std::make_integer_sequence<int, R / 2>{});
        dit_levels<R, 2 * L, INV, PK>(v);
    }
}

// Radix-R DFT of v[0..R) in registers, natural order in and out.  R in {1,2,4,8,16,32,64}.
template <int R, bool INV, bool PK = false>
__device__ __forceinline__ void radix(float2 *v)
{
    if constexpr (R > 1) {
        scramble<R>(v, std::make_integer_sequence<int, R>{});    // bit reversal: register renaming
        dit_levels<R, 2, INV, PK>(v);
    }
}

// ---- plans -----------------------------------------------------------------------
// V = 0 ("row" variant): plans whose first and last radix agree wherever one exists, so that the
//   row kernel can run one forward-transform body twice (ssp_kernels.cuh).  N = 1024 is 32 x 32 with
//   one warp per row (a single exchange, __syncwarp only); N >= 2048 are three-stage plans with 16
//   points per thread and a named barrier per row.
// V = 1 ("column" variant): 32 points per thread and as few exchanges as possible, because a
//   column tile synchronises the whole CTA at every exchange (E = 16 measured 2664 vs 3388 GB/s).
template <int N, int V> struct Plan;
#define SSP_PLAN(N_, V_, A, B, C, E_) \
    template <> struct Plan<N_, V_> { static constexpr int R1 = A, R2 = B, R3 = C, E = E_; }
SSP_PLAN(8, 0, 8, 1, 1, 8);        SSP_PLAN(8, 1, 8, 1, 1, 8);
SSP_PLAN(16, 0, 16, 1, 1, 16);     SSP_PLAN(16, 1, 16, 1, 1, 16);
SSP_PLAN(32, 0, 32, 1, 1, 32);     SSP_PLAN(32, 1, 32, 1, 1, 32);
SSP_PLAN(64, 0, 8, 8, 1, 8);       SSP_PLAN(64, 1, 8, 8, 1, 8);
SSP_PLAN(128, 0, 16, 8, 1, 16);    SSP_PLAN(128, 1, 16, 8, 1, 16);
SSP_PLAN(256, 0, 16, 16, 1, 16);   SSP_PLAN(256, 1, 16, 16, 1, 16);
SSP_PLAN(512, 0, 16, 2, 16, 16);   SSP_PLAN(512, 1, 32, 16, 1, 32);
SSP_PLAN(1024, 0, 32, 32, 1, 32);   SSP_PLAN(1024, 1, 32, 32, 1, 32);
SSP_PLAN(2048, 0, 32, 2, 32, 32);   SSP_PLAN(2048, 1, 32, 2, 32, 32);
#ifndef SSP_P4096_COL64
#define SSP_P4096_COL64 1
#endif
#ifndef SSP_P4096_ROW64
#define SSP_P4096_ROW64 0
#endif
#if SSP_P4096_ROW64
SSP_PLAN(4096, 0, 64, 64, 1, 64);
#else
SSP_PLAN(4096, 0, 32, 4, 32, 32);
#endif
#if SSP_P4096_COL64
SSP_PLAN(4096, 1, 64, 64, 1, 64);
#else
SSP_PLAN(4096, 1, 32, 4, 32, 32);
#endif
// V = 2 ("screen column" variant): what the register-load screen generator k_screen_col runs.  Equal to V = 1
//   except at N = 4096, where the single inverse transform measured faster with short last radices than with
//   (32,4,32); at 2048 it is the shuffle plan (32,2,32) like V = 1 (4216 vs 3430 GB/s with (32,8,8)).  The TMA
//   generator (N = 512, 1024) uses V = 1.
SSP_PLAN(8, 2, 8, 1, 1, 8);        SSP_PLAN(16, 2, 16, 1, 1, 16);     SSP_PLAN(32, 2, 32, 1, 1, 32);
SSP_PLAN(64, 2, 8, 8, 1, 8);       SSP_PLAN(128, 2, 16, 8, 1, 16);    SSP_PLAN(256, 2, 16, 16, 1, 16);
SSP_PLAN(512, 2, 32, 16, 1, 32);   SSP_PLAN(1024, 2, 32, 32, 1, 32);
SSP_PLAN(2048, 2, 32, 2, 32, 32);
SSP_PLAN(4096, 2, 32, 16, 8, 32);   // ((64,64) measured here: 3387 -> 1894 GB/s: this kernel lives on resident warps)
#undef SSP_PLAN

template <int N, int V>
struct PlanInfo {
    using P = Plan<N, V>;
    static constexpr int R1 = P::R1, R2 = P::R2, R3 = P::R3, E = P::E;
    static constexpr int T = N / E;                        // threads per line
    static constexpr int NSTAGE = (R2 == 1) ? 1 : (R3 == 1 ? 2 : 3);
    static constexpr int RL = (NSTAGE == 1) ? R1 : (NSTAGE == 2 ? R2 : R3); // last radix
    static constexpr int PADQ = N / R1;                    // one pad element per PADQ positions
    static constexpr int PADQ_REV = N / RL;
    static constexpr int LINE_ELEMS = N + (R1 > RL ? R1 : RL); // padded line length (either direction), pad 1
    static constexpr int LINE_ELEMS2 = N + 2 * (R1 > RL ? R1 : RL); // the same with pad 2 (16-byte aligned rows)
    // twiddle tables (forward sign), built on the host in double:
    //   tw1 [R1/2][N/R1][2]: W_N^(m k1), the twiddles of k1 = 2p, 2p+1 adjacent (one 16-byte load)
    //   tw2 [R2][R3]: W_N^(R1 n3 k2)
    //   tw1r[RL/2][N/RL][2] and tw2r[R2][R1] for the reversed plan (R3|R2, R2, R1)
    // A plan that reads the same forwards and backwards (R1 == RL) has identical tables in both directions: they are
    // stored once, which halves the table's L1 footprint (at N = 4096: 33 KB instead of 66 KB beside the 32 KB h table).
    static constexpr bool SYM = (R1 == RL);
    static constexpr int TW1 = 0;
    static constexpr int TW2 = TW1 + N;
    static constexpr int TW1R = SYM ? TW1 : TW2 + R2 * R3;
    static constexpr int TW2R = SYM ? TW2 : TW1R + N;
    // (two-stage plans never read tw2 / tw2r; the builder still writes R2 * R1 entries there)
    static constexpr int TW_TOTAL = SYM ? TW2 + R2 * (R3 > R1 ? R3 : R1) : TW2R + R2 * R1;
};

// ---- three-stage plans (R, 2, R) with the middle stage done by warp shuffles -----------------------------
// The radix-2 middle stage of N = 2048 pairs the elements m and m + N/(2R) of the first-stage output
// (m = n2 (N/2R) + n3).  The thread that owns m is chosen so that the two partners sit 16 lanes apart in one warp:
// with LS lanes per thread step (1 for rows, C for column tiles) and G = 16/LS,
//     n2 = (t_phys / G) & 1,   n3 = (t_phys / 2G) G + t_phys % G.
// The stage is then one __shfl_xor(.., 16) per value instead of a trip through shared memory -- one exchange and
// one barrier per transform disappear -- and each half-warp still owns consecutive m, so global, tile and
// exchange accesses stay contiguous.  All index arithmetic of the kernels runs on the LOGICAL thread index m
// (fft_logical_t); input and output layouts stay "strided by R" in m.
template <int N, int V>
struct MidShuffle {
    using P = Plan<N, V>;
    static constexpr bool value = (P::R3 > 1) && (P::R2 == 2) && (P::R1 == P::R3) && (P::E == P::R1);
};
template <int N, int V, int LS>
__device__ __forceinline__ int fft_logical_t(int t_phys)
{
    if constexpr (MidShuffle<N, V>::value) {
        constexpr int G = 16 / LS;
        static_assert(LS >= 1 && LS <= 16 && (N / Plan<N, V>::E) % (2 * G) == 0, "both partners inside one warp");
        return ((t_phys / G) & 1) * Plan<N, V>::R3 + (t_phys / (2 * G)) * G + t_phys % G;
    } else return t_phys;
}

// ---- where the first-stage twiddles come from ------------------------------------------------------------------
// TwGlobal: the table in global memory (read-only path, L1-resident).  TwTmem: a per-thread copy in tensor memory
// (tcgen05.ld from the thread's own TMEM lane): for persistent kernels whose twiddles depend on the thread only, it
// takes 16 B per point and transform off the LSU data pipe, the unit these kernels saturate first.
struct TwGlobal {
    const float2 *tw;
    __device__ __forceinline__ const float2 *table() const { return tw; }
};
__device__ __forceinline__ float4 tmem_ld4(unsigned taddr)
{
    unsigned a, b, c, d;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];\n\ttcgen05.wait::ld.sync.aligned;"
                 : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(taddr) : "memory");
    return make_float4(__uint_as_float(a), __uint_as_float(b), __uint_as_float(c), __uint_as_float(d));
}
__device__ __forceinline__ void tmem_ld8(unsigned taddr, float4 &x, float4 &y)
{
    unsigned r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n\ttcgen05.wait::ld.sync.aligned;"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
    x = make_float4(__uint_as_float(r[0]), __uint_as_float(r[1]), __uint_as_float(r[2]), __uint_as_float(r[3]));
    y = make_float4(__uint_as_float(r[4]), __uint_as_float(r[5]), __uint_as_float(r[6]), __uint_as_float(r[7]));
}
__device__ __forceinline__ void tmem_st4(unsigned taddr, float4 v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};"
                 :: "r"(taddr), "r"(__float_as_uint(v.x)), "r"(__float_as_uint(v.y)), "r"(__float_as_uint(v.z)),
                    "r"(__float_as_uint(v.w)) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
struct TwTmem {
    const float2 *tw;      // the global table (for the parts a plan does not keep in TMEM)
    unsigned taddr;        // this warp's TMEM address of column 0 of the twiddle block: columns 4 p .. 4 p + 3 = twiddles of k = 2p, 2p+1
    __device__ __forceinline__ const float2 *table() const { return tw; }
};

// One complete transform of a line held in registers.
//   DIR_REV = false: plan (R1,R2,R3): input strided by R1, output strided by RL.
//   DIR_REV = true : plan (RL,..,R1): input strided by RL, output strided by R1.
// SM: exchange accessor with  st(pos, val), ld(pos), sync()  on padded positions of this line, and
// SM::PAD = pad elements per PADQ positions (1, or 2 with ld2(pos, a, b) reading two adjacent elements
// as one 16-byte access: two-stage plans only).
// TAIL_SYNC: synchronise right after the last exchange has been read, so that the caller may reuse
// the buffer at once.  A barrier placed there is cheap (the threads have just left the previous one);
// the same barrier after the last butterflies would re-align threads that have drifted apart.
template <int N, int V, bool DIR_REV, bool INV, bool TAIL_SYNC = false, bool PK = false, class SM>
__device__ __forceinline__ void fft_line(float2 *v, int t, SM &sm, const float2 *__restrict__ tw)
{
    fft_line<N, V, DIR_REV, INV, TAIL_SYNC, PK>(v, t, sm, TwGlobal{tw});
}

// HOOK: called once, right after the last exchange of the transform has been read (where TAIL_SYNC synchronises):
// the place from which a persistent kernel starts the asynchronous copy of its next line into the exchange buffer.
struct NoHook { __device__ __forceinline__ void operator()() const {} };

// PRE: called once, after the first butterflies and before the first write to the exchange buffer: where a kernel whose
// thread groups take turns on one exchange buffer waits for its turn (HOOK then hands the buffer on).
template <int N, int V, bool DIR_REV, bool INV, bool TAIL_SYNC = false, bool PK = false, class SM, class TWP, class HOOK = NoHook,
          class PRE = NoHook>
__device__ __forceinline__ void fft_line(float2 *v, int t, SM &sm, const TWP twp, HOOK hook = HOOK{}, PRE pre = PRE{})
{
    const float2 *__restrict__ tw = twp.table();
    constexpr bool TW_TMEM = std::is_same<TWP, TwTmem>::value;
    using PI = PlanInfo<N, V>;
    constexpr int E = PI::E, T = PI::T, NS = PI::NSTAGE;
    constexpr int Ra = DIR_REV ? PI::RL : PI::R1;                        // first radix
    constexpr int Rb = (NS >= 2) ? (NS == 2 ? (DIR_REV ? PI::R1 : PI::R2) : PI::R2) : 1;
    constexpr int Rc = (NS == 3) ? (DIR_REV ? PI::R1 : PI::R3) : 1;
    constexpr int PADQ = N / Ra;
    const float2 *tw1 = tw + (DIR_REV ? PI::TW1R : PI::TW1);
    const float2 *tw2 = tw + (DIR_REV ? PI::TW2R : PI::TW2);
    // padded position of line index k1 * PADQ + r, r < PADQ: one pad element per PADQ positions.  Written
    // with k1 explicit so that no division of a run-time index is left in the address arithmetic.
    constexpr int PITCH = PADQ + SM::PAD;
    static_assert(SM::PAD == 1 || NS <= 2, "16-byte exchange reads are laid out for two-stage plans");

    if constexpr (MidShuffle<N, V>::value) {
        // t is the logical index m = n2 Rc + n3; its partner (other n2) sits 16 lanes away
        static_assert(E == Ra && Ra == Rc && Rb == 2, "(R, 2, R) plans with one first-stage butterfly per thread");
        const int n2 = t / Rc, n3 = t % Rc;
        radix<Ra, INV, PK>(v);
        pre();
        const float4 *tw4 = reinterpret_cast<const float4 *>(tw1) + t;
        const float2 w2 = __ldg(tw2 + Rc + n3);                    // W_N^(Ra n3) for the k2 = 1 output
        // exchange pitches of k1 and k2: a half-warp owns one k2 and consecutive n3 (writes) / consecutive k1 (reads),
        // and 2 Rc + 1 = 1 mod 16 spreads the reads over 16 bank pairs for rows and for C-column tiles alike
        constexpr int P2 = Rc, P1 = 2 * Rc + 1;
#pragma unroll
        for (int k = 0; k < Ra; k += 2) {
            float4 w;
            if constexpr (TW_TMEM) w = tmem_ld4(twp.taddr + 2 * k);
            else w = __ldg(tw4 + (k / 2) * (N / Ra));
            float2 x[2] = {v[k], v[k + 1]};
            if (k > 0) x[0] = cmul_c<INV, PK>(x[0], make_float2(w.x, w.y));
            x[1] = cmul_c<INV, PK>(x[1], make_float2(w.z, w.w));
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const float px = __shfl_xor_sync(0xffffffffu, x[e].x, 16);
                const float py = __shfl_xor_sync(0xffffffffu, x[e].y, 16);
                // k2 = n2: own + partner for k2 = 0, (partner - own) W_N^(Ra n3) for k2 = 1
                float2 y = n2 ? make_float2(px - x[e].x, py - x[e].y) : make_float2(x[e].x + px, x[e].y + py);
                if (n2) y = cmul_c<INV, PK>(y, w2);
                sm.st((k + e) * P1 + n2 * P2 + n3, y);
            }
        }
        sm.sync();
        const int k1 = t % Ra, k2 = t / Ra;                        // output X[k1 + Ra k2 + 2 Ra k3] = X[t + 2 Ra k3]
#pragma unroll
        for (int n = 0; n < Rc; ++n) v[n] = sm.ld(k1 * P1 + k2 * P2 + n);
        if constexpr (TAIL_SYNC) sm.sync();
        hook();
        radix<Rc, INV, PK>(v);
        return;
    }

    // ---- stage 1
    constexpr int M1 = N / Ra;
#pragma unroll
    for (int i = 0; i < E / Ra; ++i) {
        radix<Ra, INV, PK>(v + i * Ra);
        if (i == 0) pre();
        if constexpr (NS >= 2) {
            const int m = t + T * i;
            const float4 *tw4 = reinterpret_cast<const float4 *>(tw1) + m;
#pragma unroll
            for (int k = 0; k < Ra; k += 2) {
                float4 w;                                         // twiddles of k and k + 1
                if constexpr (TW_TMEM) {
                    static_assert(!TW_TMEM || (E == Ra && !DIR_REV), "TMEM twiddles: one first-stage butterfly per thread");
                    w = tmem_ld4(twp.taddr + 2 * k);
                } else w = __ldg(tw4 + (k / 2) * M1);
                float2 x0 = v[i * Ra + k], x1 = v[i * Ra + k + 1];
                if (k > 0) x0 = cmul_c<INV, PK>(x0, make_float2(w.x, w.y));
                x1 = cmul_c<INV, PK>(x1, make_float2(w.z, w.w));
                sm.st(k * PITCH + m, x0);
                sm.st((k + 1) * PITCH + m, x1);
            }
        }
    }
    if constexpr (NS == 1) return;
    sm.sync();

    if constexpr (NS == 2) {
        // ---- stage 2 (last): butterfly j = k1, reads k1*Rb + n2, produces X[k1 + Ra*k2]
#pragma unroll
        for (int i = 0; i < E / Rb; ++i) {
            const int j = t + T * i;
            if constexpr (SM::PAD == 2) {
#pragma unroll
                for (int n = 0; n < Rb; n += 2) sm.ld2(j * PITCH + n, v[i * Rb + n], v[i * Rb + n + 1]);
            } else {
#pragma unroll
                for (int n = 0; n < Rb; ++n) v[i * Rb + n] = sm.ld(j * PITCH + n);
            }
        }
        if constexpr (TAIL_SYNC) sm.sync();
        hook();
#pragma unroll
        for (int i = 0; i < E / Rb; ++i) radix<Rb, INV, PK>(v + i * Rb);
    } else {
        // ---- stage 2 (middle): butterfly j = k1 + Ra*n3 (k1 fastest: with the pitch N/Ra + 1 the
        // 16 lanes of a half warp hit 16 different bank pairs), in place
#pragma unroll
        for (int i = 0; i < E / Rb; ++i) {
            const int j = t + T * i;
            const int k1 = j % Ra, n3 = j / Ra;
            const int base = k1 * PITCH + n3;
            float2 *w = v + i * Rb;
#pragma unroll
            for (int n = 0; n < Rb; ++n) w[n] = sm.ld(base + n * Rc);
            radix<Rb, INV, PK>(w);
#pragma unroll
            for (int k = 0; k < Rb; ++k) {
                float2 x = w[k];
                if (k > 0) x = cmul_c<INV, PK>(x, __ldg(tw2 + k * Rc + n3));
                sm.st(base + k * Rc, x);
            }
        }
        sm.sync();
        // ---- stage 3 (last): butterfly j = k1 + Ra*k2, reads k1*Rb*Rc + k2*Rc + n3
#pragma unroll
        for (int i = 0; i < E / Rc; ++i) {
            const int j = t + T * i;
            const int k1 = j % Ra, k2 = j / Ra;
            const int base = k1 * PITCH + k2 * Rc;
            float2 *w = v + i * Rc;
#pragma unroll
            for (int n = 0; n < Rc; ++n) w[n] = sm.ld(base + n);
        }
        if constexpr (TAIL_SYNC) sm.sync();
        hook();
#pragma unroll
        for (int i = 0; i < E / Rc; ++i) radix<Rc, INV, PK>(v + i * Rc);
    }
}

// Line index of register element q of butterfly slot i for a layout strided by R.
template <int N, int V, int R>
__device__ __forceinline__ int line_index(int t, int i, int q)
{
    return q * (N / R) + t + (N / PlanInfo<N, V>::E) * i;
}

} // namespace ssp
