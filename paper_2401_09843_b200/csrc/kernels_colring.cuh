// kernels_colring.cuh -- the forward strided-axis passes a5, a6 of SURVEY.md section 8(a) for long lines (L = 256) as a PERSISTENT
// kernel fed by the TMA engine: same pruned radix-3 forward transform + truncation as col_fwd_kernel in kernels_col.cuh
// (Algorithm 3 in reverse; truncation fused), different data movement.
//
// kernels_col.cuh: one tile per CTA, every thread fetches its own rows with LDG and its twiddles from L1 -- ncu shows
// `long_scoreboard` as the first stall at 2.9 warps per scheduler with DRAM 64-70 % busy (profiles/r02_full.md).  Here:
//
//  * a PRODUCER WARP issues cp.async.bulk.tensor (tensor map: box = 128 bytes x L rows of one column tile; SASS UTMALDG)
//    into a ring of STAGES whole input tiles in shared memory, completion on an mbarrier per stage; the rows of the next
//    tile are in flight while the current tile is in its butterflies, independent of how many warps are resident;
//  * THREE TEAMS of TT = TC x max(R1, R2) threads work on one tile, team q on the input rows [qL, (q+1)L) of sub-transform q:
//    3x the warps of kernels_col.cuh per tile and nothing parked between sub-transforms;
//  * the part of the stage buffer a team has consumed doubles as its exchange buffer and then holds
//    G_q[n] = W^{-qn} F_q[n] for the 3 -> 2 combine, which all threads of the CTA share;
//  * the twiddle factors a thread needs (they depend on its position in the team only, not on the tile) are parked once per
//    CTA in TENSOR MEMORY (tmem.cuh) and fetched four (fp64) at a time instead of 31 L1 loads per thread and tile.
//
// Measured (profiles/r02_experiments.md) at 512^3: fp64 a5 3.65 -> 3.20 ms, a6 2.67 -> 2.52 ms; fp32 1.96 -> 1.84, 1.40 -> 1.24 ms.  The inverse counterpart and
// the shorter lines (L = 64, 128) were built and measured too and lost against kernels_col.cuh; they are not in the library.
// Tile, register stages R1 x R2, twiddle tables and the decimated physical order are those of kernels_col.cuh.
#pragma once
#include <cuda.h>

#include <cstdint>

#include "cx.cuh"
#include "kernels_col.cuh"
#include "kernels_zfused.cuh"   // mbarrier helpers, named_bar_sync
#include "tmem.cuh"

namespace ns {

// box of the 3-D tensor (2 * columns scalars, rows, slabs) at (c0, c1, c2) -> shared memory, completion on `bar`
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

template <typename T, int L, int R1, int R2, int TC, int STAGES> struct ColRingGeo {
    static constexpr int P = R1 > R2 ? R1 : R2;
    static constexpr int TT = TC * P;                       // threads per team
    static constexpr int NT = 3 * TT + 32;                  // three teams + the producer warp
    static constexpr size_t CHUNK = (size_t)L * TC;         // complex elements of L rows of a tile
    static constexpr size_t FWD_BYTES = (STAGES * 3) * CHUNK * sizeof(cx<T>) + 2 * STAGES * sizeof(uint64_t);
    static constexpr uint32_t CHUNK_BYTES = (uint32_t)(CHUNK * sizeof(cx<T>));
    // tensor memory: per warp two twiddle sets (stage twiddles, radix-3 twiddles), each padded to a multiple of one x16 access
    static constexpr int CH = tmem_cx_chunk<T>();
    static constexpr uint32_t SETA = 16 * ((P + CH - 1) / CH);            // columns of one set (P complex values at most)
    static constexpr uint32_t WCOLS = 2 * SETA;
    static constexpr uint32_t NEED = ((3 * TT / 32 + 3) / 4) * WCOLS;
    static constexpr uint32_t NCOLS = NEED <= 32 ? 32 : NEED <= 64 ? 64 : NEED <= 128 ? 128 : NEED <= 256 ? 256 : 512;
    static_assert(NEED <= 512, "tensor memory: 512 columns per SM");
};

// Park CNT complex values per thread (value k from gen(k)) at TMEM address `base`, in chunks of one x16 access.
template <typename T, int CNT, typename Gen>
__device__ __forceinline__ void ring_park(uint32_t base, Gen gen) {
    constexpr int CH = tmem_cx_chunk<T>();
#pragma unroll
    for (int ch = 0; ch < (CNT + CH - 1) / CH; ++ch) {
        T wr[CH], wi[CH];
#pragma unroll
        for (int e = 0; e < CH; ++e) {
            const int k = ch * CH + e;
            const cx<T> w = k < CNT ? gen(k) : mk<T>(0, 0);
            wr[e] = w.x;
            wi[e] = w.y;
        }
        tmem_store_cx(base + 16 * ch, wr, wi);
    }
}

// ------------------------------------------------------------------------------------------------
// forward: physical rows [0,3L) -> spectral rows [0,2L), truncated, output * scale
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R1, int R2, int TC, int STAGES, int MINB, bool SPLIT>
__global__ void __launch_bounds__(3 * TC * ColP<R1, R2>::value + 32, MINB)
col_fwd_ring_kernel(const __grid_constant__ CUtensorMap tmap, cx<T>* __restrict__ out, ColArgs g, T scale, Twiddles<T> tw) {
    using Geo = ColRingGeo<T, L, R1, R2, TC, STAGES>;
    constexpr int TT = Geo::TT;
    constexpr size_t CHUNK = Geo::CHUNK;
    extern __shared__ __align__(128) unsigned char smem_ring[];
    cx<T>* In = reinterpret_cast<cx<T>*>(smem_ring);                               // [STAGES][3][L][TC]
    uint64_t* full = reinterpret_cast<uint64_t*>(In + (size_t)STAGES * 3 * CHUNK);  // [STAGES]
    uint64_t* empty = full + STAGES;                                              // [STAGES]

    __shared__ uint32_t tslot;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        mbar_fence_init();
    }
    if (threadIdx.x < 32) tmem_alloc(&tslot, Geo::NCOLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const long first = blockIdx.x, stride = gridDim.x;

    if (threadIdx.x >= 3 * TT) {                 // ---------------- producer warp
        if (threadIdx.x == 3 * TT) {
            tma_prefetch_desc(&tmap);
            long it = 0;
            for (long tile = first; tile < g.total_tiles; tile += stride, ++it) {
                const int s = (int)(it % STAGES);
                if (it >= STAGES) mbar_wait(empty + s, (uint32_t)(((it / STAGES) - 1) & 1));
                const int slab = (int)(tile / g.tiles_per_slab);
                const int c0 = (int)(tile % g.tiles_per_slab) * TC * 2;
                mbar_expect_tx(full + s, 3 * Geo::CHUNK_BYTES);
#pragma unroll
                for (int qq = 0; qq < 3; ++qq) tma_load_3d(In + ((size_t)s * 3 + qq) * CHUNK, &tmap, c0, qq * L, slab, full + s);
            }
        }
        return;
    }

    const int q = threadIdx.x / TT;
    const int lt = threadIdx.x % TT;
    const int c = lt % TC, i = lt / TC;
    const int bar_id = 1 + q;
    constexpr int BAR_ALL = 4;
    constexpr int CH = Geo::CH;
    // this warp's tensor-memory window: stage twiddles w_L^{n2 i} (n2 < R2), radix-3 twiddles W^{q (R2 n1 + i)} (n1 < R1)
    const int warp = threadIdx.x / 32;
    const uint32_t ttw = tslot + ((uint32_t)(32 * (warp % 4)) << 16) + (uint32_t)(warp / 4) * Geo::WCOLS;
    const uint32_t tw3 = ttw + Geo::SETA;
    {
        const int i1 = i < R1 ? i : 0, i2 = i < R2 ? i : 0;
        ring_park<T, R2>(ttw, [&](int n2) { return ldg(tw.twB + n2 * R1 + i1); });
        ring_park<T, R1>(tw3, [&](int n1) { return ldg((q == 2 ? tw.w3b : tw.w3a) + R2 * n1 + i2); });
        tmem_wait_st();
    }
    long it = 0;
    for (long tile = first; tile < g.total_tiles; tile += stride, ++it) {
        const int s = (int)(it % STAGES);
        const long slab = tile / g.tiles_per_slab;
        const int col0 = (int)(tile % g.tiles_per_slab) * TC;
        cx<T>* ob = out + slab * g.out_slab + col0;
        cx<T>* B = In + (size_t)s * 3 * CHUNK;       // the stage: [3][L][TC]
        cx<T>* Bq = B + (size_t)q * CHUNK;           // this team's rows; then its exchange buffer; then G_q
        mbar_wait(full + s, (uint32_t)((it / STAGES) & 1));
        cx<T> x[R2];
        if (i < R1) {
#pragma unroll
            for (int r2 = 0; r2 < R2; ++r2) x[r2] = Bq[(size_t)(i + R1 * r2) * TC + c];
        }
        named_bar_sync(bar_id, TT);               // every input row of the team is in registers
        if (i < R1) {
            fft_reg<R2, -1, T>(x);
#pragma unroll
            for (int ch = 0; ch < R2 / CH; ++ch) {
                T wr[CH], wi[CH];
                tmem_load_cx(ttw + 16 * ch, wr, wi);
#pragma unroll
                for (int e = 0; e < CH; ++e) {
                    const int n2 = ch * CH + e;
                    cx<T> v = x[outpos<R2>(n2)];
                    if (n2 > 0) v = cmulc(v, mk<T>(wr[e], wi[e]));
                    Bq[(size_t)(i * R2 + n2) * TC + c] = v;
                }
            }
        }
        named_bar_sync(bar_id, TT);
        cx<T> y[R1];
        if (i < R2) {
#pragma unroll
            for (int r1 = 0; r1 < R1; ++r1) y[r1] = Bq[(size_t)(r1 * R2 + i) * TC + c];
        }
        named_bar_sync(bar_id, TT);               // exchange read: the buffer may take G_q
        if (i < R2) {
            fft_reg<R1, -1, T>(y);
#pragma unroll
            for (int ch = 0; ch < R1 / CH; ++ch) {
                T wr[CH], wi[CH];
                if (q != 0) tmem_load_cx(tw3 + 16 * ch, wr, wi);          // team-uniform
#pragma unroll
                for (int e = 0; e < CH; ++e) {
                    const int n1 = ch * CH + e;
                    cx<T> v = y[outpos<R1>(n1)];
                    if (q > 0) v = cmulc(v, mk<T>(wr[e], wi[e]));
                    Bq[(size_t)(R2 * n1 + i) * TC + c] = v;
                }
            }
        }
        named_bar_sync(BAR_ALL, 3 * TT);          // F_0, G_1, G_2 of the tile are in the stage
        // 3 -> 2 combine + truncation, shared by all threads: element e = n TC + c
        for (int e = threadIdx.x; e < L * TC; e += 3 * TT) {
            const int n = e / TC;
            const cx<T> f0 = B[e], g1 = B[CHUNK + e], g2 = B[2 * CHUNK + e];
            const cx<T> S = g1 + g2, D = g1 - g2;
            constexpr T h3 = (T)0.86602540378443864676L;
            const cx<T> A = f0 + S;
            // C = F0 - S/2 + i (sqrt3/2) D
            const cx<T> Cc = mk<T>(f0.x - (T)0.5 * S.x - h3 * D.y, f0.y - (T)0.5 * S.y + h3 * D.x);
            cx<T>* op = ob + (e % TC);
            stg_stream(col_row<SPLIT>(out, op, g, n), scale * A);
            stg_stream(col_row<SPLIT>(out, op, g, L + n), (n == 0) ? mk<T>(0, 0) : scale * Cc);
        }
        named_bar_sync(BAR_ALL, 3 * TT);          // combine read: the stage goes back to the producer
        if (threadIdx.x == 0) mbar_arrive(empty + s);
    }
    tmem_fence_before_sync();
    named_bar_sync(BAR_ALL, 3 * TT);
    if (threadIdx.x < 32) tmem_dealloc(tslot, Geo::NCOLS);
}

}  // namespace ns
