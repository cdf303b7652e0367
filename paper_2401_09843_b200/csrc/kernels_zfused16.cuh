// kernels_zfused16.cuh -- 16-values-per-lane building blocks of the fused z kernel for the longest lines
// (L = N/2 in {128, 256}; the kernel itself is in kernels_zfused16t.cuh).
//
// Same mathematics as kernels_z.cuh; compared with kernels_zfused8.cuh every lane holds 16 complex values,
// so a length-L sub-transform q is 16 x G (G = L/16 lanes of one warp) with ONE warp-local shared-memory
// exchange instead of two, and half as many inter-stage twiddle loads -- the 8-per-lane kernel is bound by
// the L1 / shared-memory pipe at these lengths (profiles/r01_baseline.md).
// One warp works on the same q of 32/G neighbouring lines, so the q-dependent code does not diverge.
#pragma once
#include <cstdint>

#include "cx.cuh"
#include "kernels_zfused.cuh"   // mbarrier / bulk-copy helpers, prune3, atomic_max_nonneg
#include "kernels_zfused8.cuh"  // named_bar_sync

namespace ns {

template <int L> struct Z16Geo {
    static constexpr int G = L / 16;      // lanes per sub-transform
    static constexpr int P = G + 1;       // exchange pitch (odd: conflict-free 16-byte column reads)
    static constexpr int SZ = 16 * P;     // exchange / combine region of one sub-transform (>= L elements)
    static constexpr int UL = 32 / G;     // lines per unit (one warp = the same q of UL lines)
};

// Inverse (exp(+i)) length-L transform by G lanes.  in: v[j] = s[t + G j].
// out: v[h*G + brev<G>(r2)] = x[(t + G h) + 16 r2],  h < 16/G.
template <typename T, int L>
__device__ __forceinline__ void z16_inverse(cx<T> (&v)[16], cx<T>* __restrict__ S, int t, const Twiddles<T>& tw) {
    constexpr int G = Z16Geo<L>::G, P = Z16Geo<L>::P, Hc = 16 / G;
    fft_reg<16, +1, T>(v);
#pragma unroll
    for (int r1 = 0; r1 < 16; ++r1) {
        cx<T> w = v[brev<16>(r1)];
        if (r1 > 0) w = cmul(w, ldg(tw.z16 + r1 * G + t));
        S[r1 * P + t] = w;
    }
    __syncwarp();
#pragma unroll
    for (int h = 0; h < Hc; ++h)
#pragma unroll
        for (int tt = 0; tt < G; ++tt) v[h * G + tt] = S[(t + G * h) * P + tt];
    __syncwarp();
#pragma unroll
    for (int h = 0; h < Hc; ++h) fft_reg<G, +1, T>(v + h * G);
}

// Forward (exp(-i)) transform, exact mirror: in = layout of z16_inverse's output; out: v[brev16(j)] = F[t + G j].
template <typename T, int L>
__device__ __forceinline__ void z16_forward(cx<T> (&v)[16], cx<T>* __restrict__ S, int t, const Twiddles<T>& tw) {
    constexpr int G = Z16Geo<L>::G, P = Z16Geo<L>::P, Hc = 16 / G;
    {
        cx<T> y[16];
#pragma unroll
        for (int h = 0; h < Hc; ++h)
#pragma unroll
            for (int r2 = 0; r2 < G; ++r2) y[h * G + r2] = v[h * G + brev<G>(r2)];  // natural order in
#pragma unroll
        for (int h = 0; h < Hc; ++h) fft_reg<G, -1, T>(y + h * G);
#pragma unroll
        for (int h = 0; h < Hc; ++h)
#pragma unroll
            for (int tt = 0; tt < G; ++tt) S[(t + G * h) * P + tt] = y[h * G + brev<G>(tt)];
    }
    __syncwarp();
#pragma unroll
    for (int r1 = 0; r1 < 16; ++r1) {
        cx<T> w = S[r1 * P + t];
        if (r1 > 0) w = cmulc(w, ldg(tw.z16 + r1 * G + t));
        v[r1] = w;
    }
    __syncwarp();
    fft_reg<16, -1, T>(v);
}

}  // namespace ns
