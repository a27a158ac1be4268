// ssp_kernels.cuh -- row and column kernels of the fused split step (K4-K7).
//
//   k_row<N,FIRST,SECOND,GENERIC>:  [IFFT_x] -> * exp(+-i phi) W [-> save plane / phase gradient]
//                                 -> [FFT_x] -> * hx(next step)                  (Eq.1)
//   k_col<N,MODE>:                FFT_y -> * hy/N^2 -> IFFT_y on a tile of C columns (register loads)
//   k_col_tma<N>:                 the same pass with the tile moved by TMA (ssp_col_tma.cuh)
//
// One split step = one column + one row launch = two HBM round trips of the field plus one
// fp32 read of the screen: 36 B/px.  H is separable for the Fresnel
// kernel, H = hx[kx] hy[ky], both 1-D tables built in double on the host.
//
// Inverse transforms run the FORWARD code on re/im-swapped data: with s(a+ib) = b+ia,
// IFFT(x) = s(FFT(s(x))), and the swap is register renaming.  For plans whose first and last
// radix agree the output layout of a transform equals its input layout, so IFFT -> pointwise
// -> FFT is one forward-transform body executed twice in a rolled loop: half the code, which
// matters because the unrolled butterflies otherwise overflow the 32 KB instruction cache.
#pragma once

#include "ssp_internal.h"
#include "ssp_lines.cuh"
#include "ssp_stats.cuh"

namespace ssp {

template <bool SWAP>
__device__ __forceinline__ float2 swap_if(float2 x) { return SWAP ? make_float2(x.y, x.x) : x; }

template <int N>
struct SYM_PLAN { static constexpr bool value = PlanInfo<N, 0>::SYM && PlanInfo<N, 0>::NSTAGE == 2 && PlanInfo<N, 0>::E == PlanInfo<N, 0>::R1; };

// Tensor-memory layout of the persistent row kernel: a thread's lane holds 2E words of twiddle pairs, then 2E words of hx;
// warps w and w + 4 of a CTA share a lane quadrant and take consecutive column blocks of 4E.
template <int N>
struct RowTmem {
    using PI = PlanInfo<N, 0>;
    static constexpr int E = PI::E;
    static constexpr int HXOFF = 2 * E, CW = 4 * E;
    static constexpr int GROUPS = (RowCfg<N>::THREADS + 127) / 128;
    static constexpr int NEED = GROUPS * CW;
    static constexpr int COLS = NEED <= 32 ? 32 : (NEED <= 64 ? 64 : (NEED <= 128 ? 128 : (NEED <= 256 ? 256 : 512)));
    static constexpr bool OK = PI::SYM && PI::E == PI::R1 && PI::NSTAGE >= 2 && (RowCfg<N>::THREADS % 32 == 0);
};

// Pointwise stage in real space on a line held in the layout strided by RL.  SWAPPED: the registers
// hold the field re/im-swapped (it came out of an inverse transform run by the forward code); the
// result is in plain form either way.  GENERIC = false is the common split step (screen and window
// both present, nothing saved): no per-element flag tests in the unrolled body.  GENERIC = true reads
// the run-time flags: optional screen / window, saved planes, phase gradient.
template <int N, int RL, int E, int T, bool GENERIC, bool SWAPPED, bool PK = false>
__device__ __forceinline__ void row_pointwise(float2 *v, const RowArgs &a, const float *phis, int t, int b, int iy)
{
    const long long pix0 = (long long)iy * N;
    const float yc = (float)(iy - N / 2);
    const float y2 = yc * yc * a.win_qs;
    const float xf = (float)(t - N / 2);
    if constexpr (PK) {
    // Two pixels at a time: the phase reduction, the window argument and the amplitude products are packed
    // fp32 pairs ACROSS the two pixels (FMUL2 / FFMA2), only the SFU calls stay scalar; the complex multiply then
    // takes cos and sin of each pixel as broadcast scalars and the field value as the packed operand.
#pragma unroll
    for (int j = 0; j < E; j += 2) {
        const int off0 = (j % RL) * (N / RL) + T * (j / RL);      // ix = t + off, off compile-time
        const int off1 = ((j + 1) % RL) * (N / RL) + T * ((j + 1) / RL);
        float2 mr = make_float2(1.f, 1.f), mi = make_float2(0.f, 0.f);
        if (!GENERIC || a.phi) {
            sincos_reduced2(make_float2(phis[t + off0], phis[t + off1]), &mi, &mr);
            mi = f2mul(mi, make_float2(a.phase_sign, a.phase_sign));
        }
        if (!GENERIC || a.win_on) {
            float2 amp;
            if (GENERIC ? (a.win_map != nullptr) : WinMap<N>::value) {
                // cached map: the lanes of a warp read 32 consecutive floats per element (one 128-byte line)
                amp = make_float2(__ldg(a.win_map + pix0 + t + off0), __ldg(a.win_map + pix0 + t + off1));
            } else {
                const float2 xc = f2add(make_float2(xf, xf), make_float2((float)off0, (float)off1));
                amp = window_amp2(f2fma(f2mul(xc, xc), make_float2(a.win_qs, a.win_qs), make_float2(y2, y2)),
                                  a.win_half_order);
            }
            mr = f2mul(mr, amp);
            mi = f2mul(mi, amp);
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int off = e ? off1 : off0;
            const float2 u = swap_if<SWAPPED>(v[j + e]);
            if constexpr (GENERIC) {
                if (a.grad) {
                    const float2 U = a.plane_in[b * a.plane_stride + pix0 + t + off];
                    a.grad[b * a.grad_stride + pix0 + t + off] = u.y * U.x - u.x * U.y; // Im(G conj(U))
                }
            }
            const float2 r = cmul(e ? make_float2(mr.y, mi.y) : make_float2(mr.x, mi.x), u);
            if constexpr (GENERIC) {
                if (a.plane_out) a.plane_out[b * a.plane_stride + pix0 + t + off] = r;
            }
            v[j + e] = r;
        }
    }
    } else {
#pragma unroll
    for (int i = 0; i < E / RL; ++i)
#pragma unroll
        for (int q = 0; q < RL; ++q) {
            const int off = q * (N / RL) + T * i;                 // ix = t + off, off compile-time
            const float2 u = swap_if<SWAPPED>(v[i * RL + q]);
            if constexpr (GENERIC) {
                if (a.grad) {
                    const float2 U = a.plane_in[b * a.plane_stride + pix0 + t + off];
                    a.grad[b * a.grad_stride + pix0 + t + off] = u.y * U.x - u.x * U.y; // Im(G conj(U))
                }
            }
            float mr = 1.f, mi = 0.f;
            if (!GENERIC || a.phi) {
                sincos_reduced(phis[t + off], &mi, &mr);
                mi *= a.phase_sign;
            }
            if (!GENERIC || a.win_on) {
                const float xc = xf + (float)off;
                const float amp = (GENERIC && a.win_map) ? __ldg(a.win_map + pix0 + t + off)
                                                         : window_amp(fmaf(xc * xc, a.win_qs, y2), a.win_half_order);
                mr *= amp;
                mi *= amp;
            }
            const float2 r = cmul(u, make_float2(mr, mi));
            if constexpr (GENERIC) {
                if (a.plane_out) a.plane_out[b * a.plane_stride + pix0 + t + off] = r;
            }
            v[i * RL + q] = r;
        }
    }
}

// FUSE (SURVEY 8(f)-1, K3 fused into K6; forward-only temporal frames): the screen row is not read from HBM but
// synthesised here from the column-transformed spectrum row a.ycol (8 B/px instead of the 12 B/px row pass of the
// generator plus 4 B/px here) -- a third in-register transform through the same rolled forward body (IFFT_x as forward
// code on swapped data; its real part lands in .y), the subharmonic sum of k_screen_row, the result into the shared
// screen-row buffer the pointwise stage reads anyway.
template <int N, bool FIRST, bool SECOND, bool GENERIC, bool FUSE = false>
__global__ void __launch_bounds__(RowCfg<N>::THREADS, RowCfg<N>::MIN_BLOCKS) k_row(const RowArgs a)
{
    static_assert(!FUSE || (FIRST && !GENERIC && SYM_PLAN<N>::value && PlanInfo<N, 0>::T == 32), "fused screens: one warp per row");
    using PI = PlanInfo<N, 0>;
    using CFG = RowCfg<N>;
    constexpr int E = PI::E, T = PI::T, R1 = PI::R1, RL = PI::RL;
    constexpr bool SYM = (R1 == RL);                              // output layout == input layout
    constexpr bool PK = RowCfg<N>::PACKED;                        // packed fp32 pairs (ssp_fft.cuh), where measured faster
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);

    const int tid = threadIdx.x;
    const int lib = tid / T, t = fft_logical_t<N, 0, 1>(tid % T);
    RowSmem<T, CFG::WIDE> sm{smem + (size_t)lib * CFG::LINE_ELEMS, 1 + lib};
    // Persistent form (RowCfg<N>::TMEM): the CTA walks row blocks blk = blockIdx.x, + gridDim.x, ..; this thread's 16
    // twiddle pairs W_N^(t k) and the 32 hx values of its output points do not change from row to row and are read
    // from the thread's own tensor-memory lane (tcgen05.ld) instead of through the LSU data pipe.
    constexpr bool TM = RowCfg<N>::TMEM && FIRST && SECOND && !GENERIC;
    static_assert(!FUSE || MidSwapped<N>::value, "fused screens: the column kernel hands the field over swapped");
    unsigned taddr = 0;
    if constexpr (TM) {
        static_assert(!TM || RowTmem<N>::OK, "symmetric plan with one first-stage butterfly per thread");
        unsigned *slot = reinterpret_cast<unsigned *>(smem_raw + CFG::SMEM);
        if (tid < 32) tmem_alloc(slot, RowTmem<N>::COLS);
        tmem_fence_before_sync();
        __syncthreads();
        tmem_fence_after_sync();
        taddr = *slot + ((unsigned)(tid & 96) << 16) + (unsigned)(tid / 128) * RowTmem<N>::CW;
        const float4 *tw4 = reinterpret_cast<const float4 *>(a.tw + PI::TW1) + t;
#pragma unroll
        for (int p = 0; p < PI::R1 / 2; ++p) tmem_st4(taddr + 4 * p, __ldg(tw4 + p * (N / PI::R1)));
#pragma unroll
        for (int q = 0; q < PI::R1; q += 2) {
            // (no hx -- angular spectrum: the column kernel applies the whole H -- caches the factor 1)
            const float2 one = make_float2(1.f, 0.f);
            const float2 h0 = a.hx ? __ldg(a.hx + line_index<N, 0, PI::R1>(t, 0, q)) : one;
            const float2 h1 = a.hx ? __ldg(a.hx + line_index<N, 0, PI::R1>(t, 0, q + 1)) : one;
            tmem_st4(taddr + RowTmem<N>::HXOFF + 2 * q, make_float4(h0.x, h0.y, h1.x, h1.y));
        }
        tmem_wait_st();
    }
    pdl_wait();                                                   // (ssp_internal.h) everything above read constant tables only
    const long long nblk = TM ? (long long)(a.n_lines / CFG::LPB) : (long long)blockIdx.x + 1;
    for (long long blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
    const long long line = blk * CFG::LPB + lib;
    const int b = (int)(line / N), iy = (int)(line % N);
    if constexpr (TM) sm.sync();                                  // the previous row's last reads of the exchange / screen buffers

    // the screen row is streamed from HBM: fetch it asynchronously now, use it after the first transform
    float *phis = reinterpret_cast<float *>(smem_raw + CFG::SMEM_X) + (size_t)lib * N;
    if (!FUSE && (!GENERIC || a.phi)) {
        const float *g = a.phi + b * a.phi_batch_stride + (long long)iy * N;
#pragma unroll
        for (int i = 0; i < E / 4; ++i) cp_async16(phis + 4 * (t + T * i), g + 4 * (t + T * i));
        cp_async_commit();
    }
    const bool pointwise = !GENERIC || a.phi || a.win_on || a.grad || a.plane_out;

    float2 v[E];
    // FIRST (an inverse transform comes first) loads re/im-swapped when the forward code runs it
    constexpr bool SWAP_IN = FIRST && SYM;
    constexpr bool MID = MidSwapped<N>::value;                    // the column kernel left the field swapped already
    constexpr int RIN = (FIRST || SYM) ? R1 : RL;
    auto load_line = [&](auto swap_tag) {
        constexpr bool SW = decltype(swap_tag)::value;
        const float2 *src = a.in + line * N;
#pragma unroll
        for (int i = 0; i < E / RIN; ++i)
#pragma unroll
            for (int q = 0; q < RIN; ++q) {
                float2 x = src[line_index<N, 0, RIN>(t, i, q)];
                if constexpr (GENERIC) {
                    if (a.pre) {
                        const float2 pl = a.pre_line ? __ldg(a.pre_line + iy) : make_float2(1.f, 0.f);
                        x = cmul(x, cmul(pl, __ldg(a.pre + line_index<N, 0, RIN>(t, i, q))));
                    }
                }
                v[i * RIN + q] = swap_if<SW>(x);
            }
    };
    if constexpr (FUSE) {
        // ---- K3 here: Y row -> IFFT_x -> Re + subharmonics - mean -> screen-row buffer (ssp_screens.cu: k_screen_row)
        const int scr = a.scr0 + b * a.scr_stride;
        if (TM && blk != (long long)blockIdx.x) {
            cp_async_wait_all();                                  // this row of Y was copied into the exchange buffer meanwhile
            sm.sync();
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = swap_if<true>(sm.base[line_index<N, 0, R1>(t, 0, q)]);
            sm.sync();
        } else {
            const float2 *ysrc = a.ycol + ((size_t)scr * N + iy) * N;
#pragma unroll
            for (int q = 0; q < E; ++q) v[q] = swap_if<true>(ysrc[line_index<N, 0, R1>(t, 0, q)]);
        }
    } else
    if (TM && blk != (long long)blockIdx.x) {
        // persistent form: this row was copied into the warp's exchange buffer (cp.async, raw order) while the previous
        // row finished its second transform and its stores; the group committed after it is this row's screen
        if constexpr (TM) {
            cp_async_wait_group<1>();
            sm.sync();
            constexpr bool SW = SWAP_IN && !MID;
#pragma unroll
            for (int q = 0; q < RIN; ++q) v[q] = swap_if<SW>(sm.base[line_index<N, 0, RIN>(t, 0, q)]);
            sm.sync();
        }
    } else if constexpr (SWAP_IN && MID) {
        // the column kernel has left the field swapped (always so on the common path; a run-time flag otherwise)
        if (!GENERIC || a.in_swapped) load_line(std::false_type{});
        else load_line(std::true_type{});
    } else load_line(std::integral_constant<bool, SWAP_IN>{});
    auto wait_phi = [&]() {
        if (!GENERIC || a.phi) {
            cp_async_wait_all();
            sm.sync();
        }
    };

    constexpr int ROUT = SYM ? R1 : (SECOND ? R1 : RL);
    if constexpr (FUSE) {
        // pass -1: the screen row (v holds swap(Y)); pass 0: IFFT_x of the field; pass 1 (SECOND): FFT_x
        auto prefetch_next_y = [&](int pass) {
            if constexpr (TM) {
                if (pass == 1) {
                    const long long nl = line + (long long)gridDim.x * CFG::LPB;
                    if (blk + gridDim.x < nblk) {
                        sm.sync();
                        const float2 *nxt = a.ycol + ((size_t)(a.scr0 + (int)(nl / N) * a.scr_stride) * N + (int)(nl % N)) * N;
#pragma unroll
                        for (int i = 0; i < E / 2; ++i) cp_async16(sm.base + 2 * (t + T * i), nxt + 2 * (t + T * i));
                    }
                    cp_async_commit();
                }
            }
        };
#pragma unroll 1
        for (int pass = -1; pass < (SECOND ? 2 : 1); ++pass) {
            auto hook = [&]() { prefetch_next_y(pass); };
            if constexpr (TM) fft_line<N, 0, false, false, false, PK>(v, t, sm, TwTmem{a.tw, taddr}, hook);
            else fft_line<N, 0, false, false, false, PK>(v, t, sm, a.tw);
            if (pass == -1) {
                const int scr = a.scr0 + b * a.scr_stride;
                float cst = 0.f;
                if (a.n_sh > 0) {
                    cst = -__ldg(a.sh_mean + 2 * scr);
                    for (int p = 0; p < a.n_sh; ++p) {
                        const float2 *cf = a.sh_coef + ((size_t)scr * a.n_sh + p) * 9;
                        const float2 ey = __ldg(a.ex + (size_t)p * N + iy);
                        float2 d[3];
#pragma unroll
                        for (int bb = 0; bb < 3; ++bb) {
                            const float2 c0 = __ldg(cf + bb), c1 = __ldg(cf + 3 + bb), c2 = __ldg(cf + 6 + bb);
                            const float2 lo = cmul_conj(c0, ey), hi = cmul(c2, ey);
                            d[bb] = make_float2(lo.x + c1.x + hi.x, lo.y + c1.y + hi.y);
                        }
                        const float ca = d[0].x + d[2].x, sa = d[0].y - d[2].y;
                        cst += d[1].x;
                        const float2 *exp_ = a.ex + (size_t)p * N + t;
#pragma unroll
                        for (int q = 0; q < E; ++q) {
                            const float2 ex = __ldg(exp_ + (line_index<N, 0, RL>(t, 0, q) - t));
                            v[q].y = fmaf(ca, ex.x, fmaf(sa, ex.y, v[q].y));
                        }
                    }
                }
                sm.sync();
#pragma unroll
                for (int q = 0; q < E; ++q) phis[line_index<N, 0, RL>(t, 0, q)] = v[q].y + cst;
                sm.sync();
                load_line(std::false_type{});                     // the field row, as the column kernel left it (swapped)
            } else if (pass == 0) {
                row_pointwise<N, RL, E, T, false, true, PK>(v, a, phis, t, b, iy);
                sm.sync();
            }
        }
    } else
    if constexpr (SYM) {
        if constexpr (FIRST && SECOND) {
#pragma unroll 1
            for (int pass = 0; pass < 2; ++pass) {
                // the exchange buffer is reused by the next pass: a row spanning several warps synchronises
                // right after its last exchange read (TAIL), a warp-local row after the pointwise stage
                constexpr bool TAIL = (T > 32);
                if constexpr (TM) {
                    // after the second transform's exchange has been read the buffer is idle until the next row's first
                    // transform: the next row of this warp is copied into it now, under the last butterflies and the stores
                    auto prefetch_next = [&]() {
                        if (pass == 1) {
                            if (blk + gridDim.x < nblk) {
                                sm.sync();
                                const float2 *nxt = a.in + (line + (long long)gridDim.x * CFG::LPB) * N;
#pragma unroll
                                for (int i = 0; i < E / 2; ++i) cp_async16(sm.base + 2 * (t + T * i), nxt + 2 * (t + T * i));
                            }
                            cp_async_commit();
                        }
                    };
                    fft_line<N, 0, false, false, TAIL, PK>(v, t, sm, TwTmem{a.tw, taddr}, prefetch_next);
                } else fft_line<N, 0, false, false, TAIL, PK>(v, t, sm, a.tw);
                if (pass == 0) {
                    wait_phi();
                    row_pointwise<N, RL, E, T, GENERIC, true, PK>(v, a, phis, t, b, iy);
                    if constexpr (!TAIL) sm.sync();
                }
            }
        } else if constexpr (FIRST) {
            fft_line<N, 0, false, false, false, PK>(v, t, sm, a.tw);
            wait_phi();
            row_pointwise<N, RL, E, T, GENERIC, true, PK>(v, a, phis, t, b, iy);
        } else {
            if (pointwise) {
                wait_phi();
                row_pointwise<N, RL, E, T, GENERIC, false, PK>(v, a, phis, t, b, iy);
            }
            fft_line<N, 0, false, false, false, PK>(v, t, sm, a.tw);
        }
    } else {
        if constexpr (FIRST) fft_line<N, 0, false, true, SECOND, PK>(v, t, sm, a.tw); // inverse; now strided by RL
        if (pointwise) {
            wait_phi();
            row_pointwise<N, RL, E, T, GENERIC, false, PK>(v, a, phis, t, b, iy);
        }
        if constexpr (SECOND) fft_line<N, 0, true, false, false, PK>(v, t, sm, a.tw); // forward, reversed plan; strided by R1
    }

    if constexpr (FIRST && !SECOND) {
        // K8 fused into the last row kernel of a propagation (0 B/px): the output pixels are in registers.
        // Row sums in fp32, promoted to double per row, reduced over the row's lanes by shuffles; every lane group (a row,
        // or the part of a row inside one warp) writes ONE record of the nine accumulators, lanes 0..8 one moment each
        // (a 72-byte store; no shared memory, no barrier).  k_stats_final adds a field's records in a fixed order.
        if (a.stats_acc) {
            constexpr int W = StatsGroup<N>::W;
            double r[ROW_N];
            row_point_sums<N, ROUT, E, T>(v, t, iy, a.roi_lo, a.roi_hi, r);
            group_sum<W>(r);
            const size_t rec = ((size_t)blk * CFG::THREADS + tid) / W;
            const double y = (double)(iy - N / 2);
            for (int m = tid % W; m < ACC_N; m += W) a.stats_acc[rec * ACC_N + m] = row_to_acc(m, r, y);
        }
    }
    float2 *dst = a.out + line * N;
    if constexpr (TM) {
#pragma unroll
        for (int q = 0; q < ROUT; q += 4) {
            float4 ha, hb;
            tmem_ld8(taddr + RowTmem<N>::HXOFF + 2 * q, ha, hb);
            const float2 h[4] = {make_float2(ha.x, ha.y), make_float2(ha.z, ha.w), make_float2(hb.x, hb.y), make_float2(hb.z, hb.w)};
#pragma unroll
            for (int e = 0; e < 4; ++e) dst[line_index<N, 0, ROUT>(t, 0, q + e)] = cmul_c<false, PK>(v[q + e], h[e]);
        }
    } else if (a.hx) {
#pragma unroll
        for (int i = 0; i < E / ROUT; ++i)
#pragma unroll
            for (int q = 0; q < ROUT; ++q) {
                const int k = line_index<N, 0, ROUT>(t, i, q);
                dst[k] = cmul_c<false, PK>(v[i * ROUT + q], __ldg(a.hx + k));
            }
    } else {
#pragma unroll
        for (int i = 0; i < E / ROUT; ++i)
#pragma unroll
            for (int q = 0; q < ROUT; ++q) dst[line_index<N, 0, ROUT>(t, i, q)] = v[i * ROUT + q];
    }
    }   // row blocks
    if constexpr (TM) {
        tmem_fence_before_sync();
        __syncthreads();
        if (tid < 32) tmem_dealloc(*reinterpret_cast<unsigned *>(smem_raw + CFG::SMEM), RowTmem<N>::COLS);
    }
}

// MODE 0: FFT_y -> * hy -> IFFT_y.  MODE 1: FFT_y -> * hy.  MODE 2: unnormalised IFFT_y -> * hy.
template <int N, int MODE>
__global__ void __launch_bounds__(ColCfg<N>::THREADS, ColCfg<N>::MIN_BLOCKS) k_col(const ColArgs a)
{
    using PI = PlanInfo<N, 1>;
    using CFG = ColCfg<N>;
    constexpr int E = PI::E, T = PI::T, C = CFG::C;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);

    const int tid = threadIdx.x;
    const int c = tid % C, t = fft_logical_t<N, 1, C>(tid / C);
    constexpr int GROUPS = N / C;
    const int b = blockIdx.x / GROUPS, col = (blockIdx.x % GROUPS) * C + c;
    ColSmem<C> sm{smem + c};
    pdl_wait();                                                   // (ssp_internal.h: programmatic dependent launch)

    float2 v[E];
    constexpr int R1 = PI::R1, RL = PI::RL;
    const float2 *src = a.in + (size_t)b * N * N + col;
#pragma unroll
    for (int i = 0; i < E / R1; ++i)
#pragma unroll
        for (int q = 0; q < R1; ++q) v[i * R1 + q] = src[(size_t)line_index<N, 1, R1>(t, i, q) * N];

    fft_line<N, 1, false, MODE == 2, MODE == 0>(v, t, sm, a.tw); // strided by RL
    if (a.h2d) { // non-separable H(ky,kx)
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q)
                v[i * RL + q] = cmul(v[i * RL + q], __ldg(a.h2d + ((size_t)(col / C) * N + line_index<N, 1, RL>(t, i, q)) * C + c));
    } else if (a.hy) {
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q)
                v[i * RL + q] = cmul(v[i * RL + q], __ldg(a.hy + line_index<N, 1, RL>(t, i, q)));
    }
    float2 *dst = a.out + (size_t)b * N * N + col;
    if constexpr (MODE == 0) {
        fft_line<N, 1, true, true>(v, t, sm, a.tw);   // inverse, reversed plan; strided by R1
#pragma unroll
        for (int i = 0; i < E / R1; ++i)
#pragma unroll
            for (int q = 0; q < R1; ++q) dst[(size_t)line_index<N, 1, R1>(t, i, q) * N] = v[i * R1 + q];
    } else {
#pragma unroll
        for (int i = 0; i < E / RL; ++i)
#pragma unroll
            for (int q = 0; q < RL; ++q) dst[(size_t)line_index<N, 1, RL>(t, i, q) * N] = v[i * RL + q];
    }
}

} // namespace ssp
