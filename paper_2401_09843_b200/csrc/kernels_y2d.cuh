// kernels_y2d.cuh -- the fused contiguous-axis kernel of the TWO-DIMENSIONAL solver (the paper's solver
// exists in a 2-D and a 3-D version): per px line, pad + inverse c2r along y of (u1, u2), the trace-free
// flux, max|u|^2, forward r2c + truncate (Algorithm 2 steps 1-5) -- the M^2 physical arrays never reach HBM.
//
// In two dimensions the trace-free flux T_ij = u_i u_j - delta_ij u_2^2 has only two components, T11 = u1^2 - u2^2 and
// T12 = u1 u2 (T22 = 0; the removed part is a gradient, annihilated by the Leray projection of eq. 2.5), so a line is exactly
// ONE inverse complex transform (u1 + i u2) and ONE forward complex transform (T11 + i T12): two-for-one with nothing left
// over.  The products are formed in registers between the two transforms; tensor memory holds only the twiddles.
// Same building blocks, thread layout and input ring as kernels_zpair.cuh (one LINE per lane group instead of a line pair).
#pragma once
#include <cstdint>

#include "kernels_zpair.cuh"

namespace ns {

// in [batch][2][MM][L] complex -> out [batch][2][MM][L] complex (unnormalised transforms of T11, T12); MM = M lines per sample,
// MM % (32 / G) == 0 (a warp never straddles two samples).
template <typename T, int L, int UNITS>
__global__ void __launch_bounds__(96 * UNITS, 1)
y2d_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, unsigned MM, unsigned total_lines,
           unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    using Geo = ZPGeo<T, L>;
    constexpr int G = Geo::G, PL = Geo::PL, REGION = Geo::REGION, SLOT = Geo::SLOT;
    constexpr uint32_t NCOLS = Geo::TWCOLS <= 32 ? 32 : Geo::TWCOLS <= 64 ? 64 : 128;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tslot;

    const int unit = threadIdx.x / 96;
    const int q = (threadIdx.x % 96) / 32;
    const int warp = threadIdx.x / 32;
    const int lane = threadIdx.x & 31;
    const int lg = lane / G, t = lane % G;
    const int lgcol = lg * G;

    unsigned char* ubase = smem_raw + (size_t)unit * Geo::UNIT_BYTES;
    cx<T>* In = reinterpret_cast<cx<T>*>(ubase);
    cx<T>* Ex = In + Geo::IN_UNIT;
    uint64_t* bars = reinterpret_cast<uint64_t*>(Ex + 3 * REGION);      // [PL][2] input ring, then [1] combine-done
    uint64_t* cdone = bars + 2 * PL;
    cx<T>* Sw = Ex + q * REGION;
    const cx<T>* Ulg = In + (size_t)lg * Geo::LGPITCH;
    uint64_t* bar_lg = bars + lg * 2;
    const int bar_id = 1 + unit;
    const long cs = (long)MM * L;
    constexpr uint32_t LINE_BYTES = (uint32_t)(L * sizeof(cx<T>));

    // line number `it` of this lane group goes to slot it & 1: u1 | u2
    auto issue = [&](unsigned line, int it) {
        const unsigned b = line / MM;
        const cx<T>* src = in + ((long)line + (long)b * MM) * L;         // (b 2 MM + pp) L
        cx<T>* dst = const_cast<cx<T>*>(Ulg) + (it & 1) * SLOT;
        uint64_t* bar = bar_lg + (it & 1);
        mbar_expect_tx(bar, 2 * LINE_BYTES);
        bulk_g2s(dst, src, LINE_BYTES, bar);
        bulk_g2s(dst + L, src + cs, LINE_BYTES, bar);
    };

    if (threadIdx.x % 96 == 0) {
        for (int k = 0; k < 2 * PL; ++k) mbar_init(bars + k, 1);
        mbar_init(cdone, 3);            // one arrival per q warp (kernels_zpair.cuh: split arrive / wait)
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(&tslot, NCOLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t ttw = tslot + ((uint32_t)(32 * (warp % 4)) << 16);
    const uint32_t tw3 = ttw + 2 * Geo::C16;
    if (warp < 4) zp_park_twiddles<T, L>(ttw, tw3, t, tw);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();

    const unsigned stride = gridDim.x * UNITS * PL;
    unsigned line = (blockIdx.x * UNITS + unit) * PL + lg;        // MM % PL == 0: validity is uniform over the unit
    const bool issuer = (q == 0 && t == 0);
    if (issuer && line < total_lines) {
        issue(line, 0);
        if (line + stride < total_lines) issue(line + stride, 1);
    }

#pragma unroll 1
    for (int it = 0; line < total_lines; line += stride, ++it) {
        const unsigned b = line / MM;
        cx<T>* Oa = out + ((long)line + (long)b * MM) * L;
        mbar_wait(bar_lg + (it & 1), (uint32_t)((it >> 1) & 1));
        const cx<T>* Ua = Ulg + (it & 1) * SLOT;
        cx<T> v[16];
        zp_form_inverse<T, L, false>(v, Ua, Ua + L, q, t, tw3);
        // the regions may be overwritten only when all three warps have finished the combine of the previous line
        zp_transform<T, L>(v, Sw, lane, t, lgcol, ttw, it > 0 ? cdone : nullptr, (uint32_t)((it - 1) & 1));
        // physical values u1 + i u2 at the points p = t + G j (register zp_perm(j)); flux, conjugated, in natural order
        cx<T> w[16];
        if (umax2 != nullptr) {
            auto lmax = sq_bits((T)0);
#pragma unroll
            for (int i = 0; i < 16; ++i) lmax = umax_bits(lmax, sq_bits(v[i].x * v[i].x + v[i].y * v[i].y));
            lmax = warp_max_bits(lmax);
            if (lane == 0) atomic_max_sq(umax2 + b, lmax);
        }
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const cx<T> u = v[zp_perm<G>(j)];
            w[j] = mk<T>(u.x * u.x - u.y * u.y, -(u.x * u.y));
        }
        zp_transform<T, L>(w, Sw, lane, t, lgcol, ttw);
        zp_post_forward<T, L, false>(w, Sw, lane, q, tw3);
        named_bar_sync(bar_id, 96);
        // all three warps have consumed this line's slot: refill it with the line after next
        if (issuer && line + 2 * (unsigned long long)stride < total_lines) issue(line + 2 * stride, it + 2);
        zp_combine_store<T, L>(Ex, lgcol, Oa, Oa + cs, q, t);
        __syncwarp();                     // combine reads done: arrive; the wait is in the next inverse transform
        if (lane == 0) mbar_arrive(cdone);
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tslot, NCOLS);
}

}  // namespace ns
