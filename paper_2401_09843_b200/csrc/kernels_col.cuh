// kernels_col.cuh -- strided-axis ("column") passes of the padded 3-D transform (steps a1, a2, a5, a6
// of SURVEY.md section 8(a); Algorithm 3 steps 1-2 of the paper, and its reverse).
//
// The 3/2 zero-padding (Algorithm 2 step 1) and the truncation (step 5)
// are fused into the transform as a PRUNED radix-3 stage, so padded zeros are never read or written:
// with M = 3L, L = N/2, the padded line has non-zeros only at k = n (stored row n) and k = n - L
// (stored row n + L), n in [0, L); row L (the Nyquist entry) is zero by convention (A3).
//
//   inverse:  x[3r+q] = sum_n s_q[n] w_L^{+rn},   s_q[n] = (a_n + c_n w3^{-q}) W^{+qn}
//   forward:  F_q[n]  = sum_r x[3r+q] w_L^{-rn},  A_n = sum_q W^{-qn} F_q[n],  C_n = sum_q W^{-qn} w3^{+q} F_q[n]
//   with a_n / A_n = row n, c_n / C_n = row n + L, W = e^{2 pi i/(3L)}, w3 = e^{2 pi i/3}.
//
// The physical axis is kept in the decimated order p = q*L + r (physical index j = 3r + q): everything
// done in physical space is pointwise, and the forward pass consumes the same order.
//
// Tile = TC adjacent columns (TC * sizeof(complex) = 128 B, one full cache line per row) x the whole
// line.  Each length-L transform is two register stages R1 x R2 with one shared-memory exchange;
// the three sub-transforms q = 0,1,2 are done one after the other by the same threads so the input
// rows a_n, c_n are read from HBM exactly once and stay in registers.
#pragma once
#include "cx.cuh"
#include "ns_internal.h"
#include "tmem.cuh"

namespace ns {

struct ColArgs {
    long istride, ostride;    // row strides of input / output, in complex elements
    long in_slab, out_slab;   // slab strides, in complex elements
    int tiles_per_slab;       // column tiles per slab (columns / TC)
    long total_tiles;         // slabs * tiles_per_slab
    int pf_dist;              // tiles ahead to prefetch into L2 (kernels instantiated with PF): about the CTAs resident on the GPU
    // Output split over several destinations (multi-device solver, ns_mg.h: the slab exchange fused into the pass -- the rows of
    // the transformed axis are stored straight into the memory of the device that owns them, over NVLink peer access).
    // split_rows = 0: plain output.  Otherwise output row n goes to destination n / split_rows, row n % split_rows of the array
    // at peer[destination] (same slab / column offsets and row stride as the plain output); peer is a table in DEVICE memory
    // (a dynamically indexed kernel-parameter array would be copied to local memory in every thread).
    int split_rows;
    const unsigned long long* peer;
};

// address of output row `row` of the tile whose plain output base is `op` (= out + slab offset + column)
// (SPLIT is a template flag of the kernels: the plain path compiles to exactly the single-device code)
template <bool SPLIT, typename T>
__device__ __forceinline__ cx<T>* col_row(cx<T>* out, cx<T>* op, const ColArgs& g, int row) {
    if constexpr (!SPLIT) return op + (long)row * g.ostride;
    const int dst = row / g.split_rows;
    return reinterpret_cast<cx<T>*>(__ldg(g.peer + dst)) + (op - out) + (long)(row - dst * g.split_rows) * g.ostride;
}

template <int R1, int R2> struct ColP { static constexpr int value = R1 > R2 ? R1 : R2; };

// L2 prefetch of the input rows of a LATER tile (the one this SM will work on a few CTAs from now), issued while the
// current tile is in its butterflies: one tile per CTA and blocking loads leave HBM idle during the compute phases
// (ncu: DRAM 59-70 % busy, stalls = global-load latency); the prefetch keeps requests in flight.  `rows` input rows of
// 128 bytes; thread `tid` of `nthreads` takes every nthreads-th row.  Measured: it pays for the
// short lines (L = 64: a5 1.68 -> 1.52 ms, a6 1.15 -> 1.01 ms at 32 x 128^3) and loses for L = 256, so PF is a template flag.
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
template <typename T>
__device__ __forceinline__ void col_prefetch_tile(const cx<T>* __restrict__ in, const ColArgs& g, long tile, int rows, int TC, int tid,
                                                  int nthreads) {
    if (tile >= g.total_tiles) return;
    const long slab = tile / g.tiles_per_slab;
    const cx<T>* base = in + slab * g.in_slab + (long)(tile % g.tiles_per_slab) * TC;
    for (int r = tid; r < rows; r += nthreads) prefetch_l2(base + (long)r * g.istride);
}

// ------------------------------------------------------------------------------------------------
// inverse (spectral rows [0,2L) -> physical rows [0,3L)), exp(+i...)
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R1, int R2, int TC, int TPB, bool PF, bool SPLIT>
__global__ void __launch_bounds__(TC* ColP<R1, R2>::value* TPB)
col_inv_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, ColArgs g,
               Twiddles<T> tw) {
    static_assert(R1 * R2 == L && R2 >= 2, "two register stages");
    constexpr int P = ColP<R1, R2>::value;
    constexpr int TT = TC * P;  // threads per tile
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* E = reinterpret_cast<cx<T>*>(smem_raw);  // [2][TPB][L][TC]

    const int tl = threadIdx.x / TT;
    const int lt = threadIdx.x % TT;
    const int c = lt % TC, i = lt / TC;
    long tile = (long)blockIdx.x * TPB + tl;
    if (tile >= g.total_tiles) tile = g.total_tiles - 1;  // duplicate work, identical writes
    const long slab = tile / g.tiles_per_slab;
    const int col0 = (int)(tile % g.tiles_per_slab) * TC;
    const cx<T>* ip = in + slab * g.in_slab + col0 + c;
    cx<T>* op = out + slab * g.out_slab + col0 + c;
    cx<T>* Et = E + (size_t)tl * L * TC;
    constexpr size_t EBUF = (size_t)TPB * L * TC;

    cx<T> a[R1], cc[R1];
    if (i < R2) {
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int n = R2 * n1 + i;
            a[n1] = ldg(ip + (long)n * g.istride);
        }
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int n = R2 * n1 + i;
            cc[n1] = (n == 0) ? mk<T>(0, 0) : ldg(ip + (long)(L + n) * g.istride);
        }
    }
    if constexpr (PF) col_prefetch_tile<T>(in, g, (long)blockIdx.x * TPB + g.pf_dist + tl, 2 * L, TC, lt, TT);
    int buf = 0;
#pragma unroll 1
    for (int q = 0; q < 3; ++q) {
        if (i < R2) {
            cx<T> s[R1];
            if (q == 0) {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    s[n1] = a[n1] + cc[n1];
                    // prepare t1 = a - c/2, t2 = (sqrt3/2) c for q = 1, 2
                    a[n1] = mk<T>(a[n1].x - (T)0.5 * cc[n1].x, a[n1].y - (T)0.5 * cc[n1].y);
                    cc[n1] = (T)0.86602540378443864676L * cc[n1];
                }
            } else {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    const int n = R2 * n1 + i;
                    // a + c w3^{-q}:  q=1: t1 - i t2,  q=2: t1 + i t2
                    const cx<T> z = (q == 1) ? mk<T>(a[n1].x + cc[n1].y, a[n1].y - cc[n1].x)
                                             : mk<T>(a[n1].x - cc[n1].y, a[n1].y + cc[n1].x);
                    s[n1] = cmul(z, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
                }
            }
            fft_reg<R1, +1, T>(s);
#pragma unroll
            for (int r1 = 0; r1 < R1; ++r1) {
                cx<T> v = s[outpos<R1>(r1)];
                if (r1 > 0) v = cmul(v, ldg(tw.twA + r1 * R2 + i));
                Et[buf * EBUF + (size_t)(r1 * R2 + i) * TC + c] = v;
            }
        }
        __syncthreads();
        if (i < R1) {
            cx<T> y[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) y[n2] = Et[buf * EBUF + (size_t)(i * R2 + n2) * TC + c];
            fft_reg<R2, +1, T>(y);
#pragma unroll
            for (int r2 = 0; r2 < R2; ++r2) *col_row<SPLIT>(out, op, g, q * L + i + R1 * r2) = y[outpos<R2>(r2)];
        }
        buf ^= 1;
    }
}

// ------------------------------------------------------------------------------------------------
// forward (physical rows [0,3L) -> spectral rows [0,2L), truncated), exp(-i...), output * scale
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R1, int R2, int TC, int TPB, bool PF, bool SPLIT>
__global__ void __launch_bounds__(TC* ColP<R1, R2>::value* TPB)
col_fwd_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, ColArgs g, T scale,
               Twiddles<T> tw) {
    static_assert(R1 * R2 == L && R2 >= 2, "two register stages");
    constexpr int P = ColP<R1, R2>::value;
    constexpr int TT = TC * P;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* E = reinterpret_cast<cx<T>*>(smem_raw);  // [2][TPB][L][TC] exchange + [TPB][L][TC] spill of G1

    const int tl = threadIdx.x / TT;
    const int lt = threadIdx.x % TT;
    const int c = lt % TC, i = lt / TC;
    long tile = (long)blockIdx.x * TPB + tl;
    if (tile >= g.total_tiles) tile = g.total_tiles - 1;
    const long slab = tile / g.tiles_per_slab;
    const int col0 = (int)(tile % g.tiles_per_slab) * TC;
    const cx<T>* ip = in + slab * g.in_slab + col0 + c;
    cx<T>* op = out + slab * g.out_slab + col0 + c;
    cx<T>* Et = E + (size_t)tl * L * TC;
    constexpr size_t EBUF = (size_t)TPB * L * TC;
    cx<T>* G1 = E + 2 * EBUF + (size_t)tl * L * TC;

    cx<T> F0[R1];
    cx<T> x[R2];
    int buf = 0;
    if (i < R1) {
#pragma unroll
        for (int r2 = 0; r2 < R2; ++r2) x[r2] = ldg(ip + (long)(i + R1 * r2) * g.istride);
    }
    if constexpr (PF) col_prefetch_tile<T>(in, g, (long)blockIdx.x * TPB + g.pf_dist + tl, 3 * L, TC, lt, TT);
    // NEXTQ: rows of the next sub-transform are fetched while this one goes through its second stage
    // (more bytes in flight per SM; only where the registers allow it)
    constexpr bool NEXTQ = R1 * R2 <= 64;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        if (i < R1) {
            if (!NEXTQ && q > 0) {
#pragma unroll
                for (int r2 = 0; r2 < R2; ++r2) x[r2] = ldg(ip + (long)(q * L + i + R1 * r2) * g.istride);
            }
            fft_reg<R2, -1, T>(x);
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) {
                cx<T> v = x[outpos<R2>(n2)];
                if (n2 > 0) v = cmulc(v, ldg(tw.twB + n2 * R1 + i));
                Et[buf * EBUF + (size_t)(i * R2 + n2) * TC + c] = v;
            }
            if (NEXTQ && q < 2) {
#pragma unroll
                for (int r2 = 0; r2 < R2; ++r2) x[r2] = ldg(ip + (long)((q + 1) * L + i + R1 * r2) * g.istride);
            }
        }
        __syncthreads();
        if (i < R2) {
            cx<T> y[R1];
#pragma unroll
            for (int r1 = 0; r1 < R1; ++r1) y[r1] = Et[buf * EBUF + (size_t)(r1 * R2 + i) * TC + c];
            fft_reg<R1, -1, T>(y);
            if (q == 0) {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) F0[n1] = y[outpos<R1>(n1)];
            } else if (q == 1) {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    const int n = R2 * n1 + i;
                    G1[(size_t)n * TC + c] = cmulc(y[outpos<R1>(n1)], ldg(tw.w3a + n));
                }
            } else {
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    const int n = R2 * n1 + i;
                    const cx<T> g2 = cmulc(y[outpos<R1>(n1)], ldg(tw.w3b + n));
                    const cx<T> g1 = G1[(size_t)n * TC + c];
                    const cx<T> S = g1 + g2, D = g1 - g2;
                    constexpr T h3 = (T)0.86602540378443864676L;
                    const cx<T> A = F0[n1] + S;
                    // C = F0 - S/2 + i (sqrt3/2) D
                    const cx<T> C = mk<T>(F0[n1].x - (T)0.5 * S.x - h3 * D.y, F0[n1].y - (T)0.5 * S.y + h3 * D.x);
                    *col_row<SPLIT>(out, op, g, n) = scale * A;
                    *col_row<SPLIT>(out, op, g, L + n) = (n == 0) ? mk<T>(0, 0) : scale * C;
                }
            }
        }
        buf ^= 1;
    }
}

// ------------------------------------------------------------------------------------------------
// forward, long lines (R1 = 16): same transform as col_fwd_kernel, but the partial results that have to
// survive from one sub-transform q to the next (F_0 and G_1 = W^{-n} F_1, 16 complex per thread each) are
// parked in tensor memory (tmem.cuh) instead of registers / shared memory.  That removes 64 registers per
// thread and a third of the shared memory, which is what bounded the kernel at two CTAs (8 warps) per SM.
// One tile per CTA; CTAs of 4 (fp64) or 8 (fp32) warps; warp w uses TMEM lanes 32 (w % 4), columns of set w / 4.
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R2, int TC, int MINB, bool PF, bool SPLIT>
__global__ void __launch_bounds__(TC * 16, MINB)
col_fwd_tmem_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, ColArgs g, T scale, Twiddles<T> tw) {
    constexpr int R1 = 16;
    static_assert(R1 * R2 == L && R2 >= 2 && R2 <= 16, "two register stages, first of 16");
    constexpr uint32_t C16 = tmem_cols16<T>();
    constexpr uint32_t NCOLS = 128;   // (F0.x F0.y G1.x G1.y) x C16 columns per warp set, TC*16/128 warp sets
    static_assert(4 * C16 * ((TC * 16 + 127) / 128) <= NCOLS, "TMEM columns");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* E = reinterpret_cast<cx<T>*>(smem_raw);  // [2][L][TC] exchange
    __shared__ uint32_t tslot;

    const int c = threadIdx.x % TC, i = threadIdx.x / TC;
    const int warp = threadIdx.x / 32;
    const long tile = blockIdx.x;
    const long slab = tile / g.tiles_per_slab;
    const int col0 = (int)(tile % g.tiles_per_slab) * TC;
    const cx<T>* ip = in + slab * g.in_slab + col0 + c;
    cx<T>* op = out + slab * g.out_slab + col0 + c;
    constexpr size_t EBUF = (size_t)L * TC;

    if (warp == 0) tmem_alloc(&tslot, NCOLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tb = tslot + ((uint32_t)(32 * (warp % 4)) << 16) + (uint32_t)(warp / 4) * 4 * C16;
    const uint32_t tF0 = tb, tG1 = tb + 2 * C16;   // 16 complex each

    int buf = 0;
    cx<T> x[R2];
#pragma unroll
    for (int r2 = 0; r2 < R2; ++r2) x[r2] = ldg(ip + (long)(i + R1 * r2) * g.istride);
    if constexpr (PF) col_prefetch_tile<T>(in, g, tile + g.pf_dist, 3 * L, TC, threadIdx.x, TC * 16);
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        {
            fft_reg<R2, -1, T>(x);
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) {
                cx<T> v = x[outpos<R2>(n2)];
                if (n2 > 0) v = cmulc(v, ldg(tw.twB + n2 * R1 + i));
                E[buf * EBUF + (size_t)(i * R2 + n2) * TC + c] = v;
            }
        }
        // rows of the next sub-transform are fetched while this one goes through its second stage
        if (q < 2) {
#pragma unroll
            for (int r2 = 0; r2 < R2; ++r2) x[r2] = ldg(ip + (long)((q + 1) * L + i + R1 * r2) * g.istride);
        }
        __syncthreads();
        cx<T> y[R1];
        const int ii = i < R2 ? i : 0;   // threads beyond R2 (L = 128) redo column 0 and discard it
#pragma unroll
        for (int r1 = 0; r1 < R1; ++r1) y[r1] = E[buf * EBUF + (size_t)(r1 * R2 + ii) * TC + c];
        fft_reg<R1, -1, T>(y);
        constexpr int CH = tmem_cx_chunk<T>();   // complex values per TMEM access
        if (q < 2) {
            const uint32_t dst = q == 0 ? tF0 : tG1;
#pragma unroll
            for (int ch = 0; ch < 16 / CH; ++ch) {
                T px[CH], py[CH];
#pragma unroll
                for (int k = 0; k < CH; ++k) {
                    const int n1 = ch * CH + k;
                    cx<T> v = y[outpos<R1>(n1)];
                    if (q == 1) v = cmulc(v, ldg(tw.w3a + R2 * n1 + ii));
                    px[k] = v.x;
                    py[k] = v.y;
                }
                tmem_store_cx(dst + 16 * ch, px, py);
            }
        } else {
            tmem_wait_st();
#pragma unroll
            for (int ch = 0; ch < 16 / CH; ++ch) {
                T fx[CH], fy[CH], gx[CH], gy[CH];
                tmem_load_cx(tF0 + 16 * ch, fx, fy);
                tmem_load_cx(tG1 + 16 * ch, gx, gy);
                if (i < R2) {
#pragma unroll
                    for (int k = 0; k < CH; ++k) {
                        const int n1 = ch * CH + k;
                        const int n = R2 * n1 + i;
                        const cx<T> g2 = cmulc(y[outpos<R1>(n1)], ldg(tw.w3b + n));
                        const cx<T> f0 = mk<T>(fx[k], fy[k]), g1 = mk<T>(gx[k], gy[k]);
                        const cx<T> S = g1 + g2, D = g1 - g2;
                        constexpr T h3 = (T)0.86602540378443864676L;
                        const cx<T> A = f0 + S;
                        // C = F0 - S/2 + i (sqrt3/2) D
                        const cx<T> C = mk<T>(f0.x - (T)0.5 * S.x - h3 * D.y, f0.y - (T)0.5 * S.y + h3 * D.x);
                        *col_row<SPLIT>(out, op, g, n) = scale * A;
                        *col_row<SPLIT>(out, op, g, L + n) = (n == 0) ? mk<T>(0, 0) : scale * C;
                    }
                }
            }
        }
        buf ^= 1;
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tslot, NCOLS);
}

// ------------------------------------------------------------------------------------------------
// inverse, long lines (R1 = 16): same transform as col_inv_kernel with the per-thread inputs
// t1 = a - c/2, t2 = (sqrt3/2) c (needed again for q = 1, 2) parked in tensor memory, so that a third CTA
// fits on the SM (the register-resident version needs 254 registers; ncu: 1.9 warps per scheduler, stalls
// dominated by the global loads).  Thread layout and TMEM window as in col_fwd_tmem_kernel.
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R2, int TC, int MINB, bool PF, bool SPLIT>
__global__ void __launch_bounds__(TC * 16, MINB)
col_inv_tmem_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, ColArgs g, Twiddles<T> tw) {
    constexpr int R1 = 16;
    static_assert(R1 * R2 == L && R2 >= 2 && R2 <= 16, "two register stages, first of 16");
    constexpr uint32_t C16 = tmem_cols16<T>();
    constexpr uint32_t NCOLS = 128;
    static_assert(4 * C16 * ((TC * 16 + 127) / 128) <= NCOLS, "TMEM columns");
    constexpr int CH = tmem_cx_chunk<T>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* E = reinterpret_cast<cx<T>*>(smem_raw);  // [2][L][TC] exchange
    __shared__ uint32_t tslot;

    const int c = threadIdx.x % TC, i = threadIdx.x / TC;
    const int warp = threadIdx.x / 32;
    const long tile = blockIdx.x;
    const long slab = tile / g.tiles_per_slab;
    const int col0 = (int)(tile % g.tiles_per_slab) * TC;
    const cx<T>* ip = in + slab * g.in_slab + col0 + c;
    cx<T>* op = out + slab * g.out_slab + col0 + c;
    constexpr size_t EBUF = (size_t)L * TC;
    const int ii = i < R2 ? i : 0;   // threads beyond R2 (L = 128) redo column 0 of the first stage and discard it

    // the loads are issued before the TMEM allocation so that their latency overlaps it
    cx<T> s[R1], cc[R1];
#pragma unroll
    for (int n1 = 0; n1 < R1; ++n1) s[n1] = ldg(ip + (long)(R2 * n1 + ii) * g.istride);
#pragma unroll
    for (int n1 = 0; n1 < R1; ++n1) {
        const int n = R2 * n1 + ii;
        cc[n1] = (n == 0) ? mk<T>(0, 0) : ldg(ip + (long)(L + n) * g.istride);
    }
    if constexpr (PF) col_prefetch_tile<T>(in, g, tile + g.pf_dist, 2 * L, TC, threadIdx.x, TC * 16);
    if (warp == 0) tmem_alloc(&tslot, NCOLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tb = tslot + ((uint32_t)(32 * (warp % 4)) << 16) + (uint32_t)(warp / 4) * 4 * C16;
    const uint32_t tT1 = tb, tT2 = tb + 2 * C16;   // 16 complex each

    // q = 0: s = a + c; park t1 = a - c/2, t2 = (sqrt3/2) c
#pragma unroll
    for (int ch = 0; ch < 16 / CH; ++ch) {
        T ax[CH], ay[CH], bx[CH], by[CH];
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int n1 = ch * CH + k;
            ax[k] = s[n1].x - (T)0.5 * cc[n1].x;
            ay[k] = s[n1].y - (T)0.5 * cc[n1].y;
            bx[k] = (T)0.86602540378443864676L * cc[n1].x;
            by[k] = (T)0.86602540378443864676L * cc[n1].y;
            s[n1] = s[n1] + cc[n1];
        }
        tmem_store_cx(tT1 + 16 * ch, ax, ay);
        tmem_store_cx(tT2 + 16 * ch, bx, by);
    }
    int buf = 0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        if (q > 0) {
            if (q == 1) tmem_wait_st();
#pragma unroll
            for (int ch = 0; ch < 16 / CH; ++ch) {
                T ax[CH], ay[CH], bx[CH], by[CH];
                tmem_load_cx(tT1 + 16 * ch, ax, ay);
                tmem_load_cx(tT2 + 16 * ch, bx, by);
#pragma unroll
                for (int k = 0; k < CH; ++k) {
                    const int n1 = ch * CH + k;
                    const int n = R2 * n1 + ii;
                    // a + c w3^{-q}:  q=1: t1 - i t2,  q=2: t1 + i t2
                    const cx<T> z = (q == 1) ? mk<T>(ax[k] + by[k], ay[k] - bx[k]) : mk<T>(ax[k] - by[k], ay[k] + bx[k]);
                    s[n1] = cmul(z, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
                }
            }
        }
        if (i < R2) {
            fft_reg<R1, +1, T>(s);
#pragma unroll
            for (int r1 = 0; r1 < R1; ++r1) {
                cx<T> v = s[outpos<R1>(r1)];
                if (r1 > 0) v = cmul(v, ldg(tw.twA + r1 * R2 + i));
                E[buf * EBUF + (size_t)(r1 * R2 + i) * TC + c] = v;
            }
        }
        __syncthreads();
        {
            cx<T> y[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) y[n2] = E[buf * EBUF + (size_t)(i * R2 + n2) * TC + c];
            fft_reg<R2, +1, T>(y);
#pragma unroll
            for (int r2 = 0; r2 < R2; ++r2) *col_row<SPLIT>(out, op, g, q * L + i + R1 * r2) = y[outpos<R2>(r2)];
        }
        buf ^= 1;
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tslot, NCOLS);
}

}  // namespace ns
