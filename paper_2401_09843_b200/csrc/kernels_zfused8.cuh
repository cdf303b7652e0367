// kernels_zfused8.cuh -- steps a3 + a4 of SURVEY.md section 8(a) in one kernel, warp-synchronous version
// for the long lines (L = N/2 in {64, 128, 256}): per (px,py) line, pad + inverse c2r along z, the flux
// products u_i u_j, max|u|^2, forward r2c + truncate (Algorithm 2 steps 1-5).
// The M^3 physical arrays never touch HBM.
//
// Same mathematics as kernels_z.cuh / kernels_zfused.cuh (pruned radix-3 + two-for-one real transforms),
// different mapping: every lane holds 8 complex values, so each length-L sub-transform q is done by
// G = L/8 lanes of ONE warp as 8 x 8 x R3 (R3 = G/8) with warp-local shared-memory exchanges
// (__syncwarp only).  Registers per thread drop from ~255 to ~100, which lets 18+ warps share an SM.
// Block-level synchronisation (a named barrier per line, 3G threads) is needed only where the three
// sub-transforms meet (the 3 -> 2 combine + Hermitian split of each forward pair).
// Input lines of the next tile are prefetched by the TMA bulk-copy engine (cp.async.bulk + mbarrier).
#pragma once
#include <cstdint>

#include "cx.cuh"
#include "kernels_zfused.cuh"  // mbarrier / bulk-copy helpers, atomic_max_nonneg

namespace ns {

// exchange geometry (pitches chosen so that every 16-byte access pattern below is bank-conflict free)
template <int R3> struct Z8Geo;
template <> struct Z8Geo<1> { static constexpr int P1 = 9, Q = 0, SZ = 72; };
template <> struct Z8Geo<2> { static constexpr int P1 = 18, Q = 17, SZ = 144; };
template <> struct Z8Geo<4> { static constexpr int P1 = 36, Q = 33, SZ = 288; };

// Inverse (exp(+i)) length-L transform of one group of G = L/8 lanes.  in: v[j] = s[t + G j].
// out (R3 = 1): v[brev8(rA)]            = x[r1 + 8 rA],                 r1 = t
//     (R3 > 1): v[s*R3 + brevR3(rB)]    = x[r1 + 8 (rA + 8 rB)],        r1 = t / R3, rA = t % R3 + R3 s
template <typename T, int L>
__device__ __forceinline__ void z8_inverse(cx<T> (&v)[8], cx<T>* __restrict__ S, int t, const Twiddles<T>& tw) {
    constexpr int G = L / 8, R3 = G / 8;
    using Geo = Z8Geo<R3>;
    fft_reg<8, +1, T>(v);
#pragma unroll
    for (int r1 = 0; r1 < 8; ++r1) {
        cx<T> w = v[brev<8>(r1)];
        if (r1 > 0) w = cmul(w, ldg(tw.z8A + r1 * G + t));
        S[r1 * Geo::P1 + t] = w;
    }
    __syncwarp();
    const int r1 = t / R3, tb = t % R3;
#pragma unroll
    for (int ta = 0; ta < 8; ++ta) v[ta] = S[r1 * Geo::P1 + R3 * ta + tb];
    __syncwarp();
    fft_reg<8, +1, T>(v);
    if constexpr (R3 > 1) {
        cx<T> y[8];
#pragma unroll
        for (int rA = 0; rA < 8; ++rA) {
            cx<T> w = v[brev<8>(rA)];
            if (rA > 0) w = cmul(w, ldg(tw.z8C + rA * R3 + tb));
            S[rA * Geo::Q + R3 * r1 + tb] = w;
        }
        __syncwarp();
#pragma unroll
        for (int s = 0; s < 8 / R3; ++s)
#pragma unroll
            for (int b = 0; b < R3; ++b) y[s * R3 + b] = S[(tb + R3 * s) * Geo::Q + R3 * r1 + b];
        __syncwarp();
#pragma unroll
        for (int s = 0; s < 8 / R3; ++s) fft_reg<R3, +1, T>(y + s * R3);
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = y[k];
    }
}

// Forward (exp(-i)) transform, exact mirror: in = layout of z8_inverse's output; out: v[brev8(j)] = F[t + G j].
template <typename T, int L>
__device__ __forceinline__ void z8_forward(cx<T> (&v)[8], cx<T>* __restrict__ S, int t, const Twiddles<T>& tw) {
    constexpr int G = L / 8, R3 = G / 8;
    using Geo = Z8Geo<R3>;
    const int r1 = t / R3, tb = t % R3;
    if constexpr (R3 > 1) {
        cx<T> y[8];
#pragma unroll
        for (int s = 0; s < 8 / R3; ++s)
#pragma unroll
            for (int rB = 0; rB < R3; ++rB) y[s * R3 + rB] = v[s * R3 + brev<R3>(rB)];  // natural order in
#pragma unroll
        for (int s = 0; s < 8 / R3; ++s) fft_reg<R3, -1, T>(y + s * R3);
#pragma unroll
        for (int s = 0; s < 8 / R3; ++s)
#pragma unroll
            for (int b = 0; b < R3; ++b) {
                // element (rA = tb + R3 s, output index b of the radix-R3 butterfly)
                cx<T> w = y[s * R3 + brev<R3>(b)];
                if (b > 0) w = cmulc(w, ldg(tw.z8C + (tb + R3 * s) * R3 + b));
                S[(tb + R3 * s) * Geo::Q + R3 * r1 + b] = w;
            }
        __syncwarp();
#pragma unroll
        for (int rA = 0; rA < 8; ++rA) v[rA] = S[rA * Geo::Q + R3 * r1 + tb];
        __syncwarp();
    } else {
        // R3 == 1: v[brev8(rA)] holds rA; bring to natural order for the butterfly input
        cx<T> y[8];
#pragma unroll
        for (int rA = 0; rA < 8; ++rA) y[rA] = v[brev<8>(rA)];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = y[k];
    }
    fft_reg<8, -1, T>(v);
#pragma unroll
    for (int ta = 0; ta < 8; ++ta) {
        cx<T> w = v[brev<8>(ta)];
        w = cmulc(w, ldg(tw.z8B + ta * G + t));  // conj(w_L^{r1 (R3 ta + tb)})
        S[r1 * Geo::P1 + R3 * ta + tb] = w;
    }
    __syncwarp();
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = S[k * Geo::P1 + t];
    __syncwarp();
    fft_reg<8, -1, T>(v);
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// in [batch][3][MM][L] complex -> out [batch][5][MM][L] complex (unnormalised transforms of the flux components)
template <typename T, int L, int LPB, int MINB>
__global__ void __launch_bounds__(3 * (L / 8) * LPB, MINB)
z_fused8_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, long MM, long total_lines,
                unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    constexpr int G = L / 8, R3 = G / 8;
    using Geo = Z8Geo<R3>;
    constexpr int SZ = Geo::SZ;          // per sub-transform exchange / combine region (>= L elements)
    static_assert(SZ >= L, "combine region must hold a sub-transform");
    constexpr int TPL = 3 * G;           // threads per line
    constexpr int UL = TPL >= 96 ? 1 : 96 / TPL;  // lines per synchronisation unit (whole warps: 96 threads)
    constexpr int UT = UL * TPL;         // threads per unit
    static_assert(UT % 32 == 0 && LPB % UL == 0, "units are whole warps");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* In = reinterpret_cast<cx<T>*>(smem_raw);   // [LPB][3][L]
    cx<T>* Ex = In + (size_t)LPB * 3 * L;              // [LPB][3][SZ]
    uint64_t* bars = reinterpret_cast<uint64_t*>(Ex + (size_t)LPB * 3 * SZ);  // [LPB]

    const int ll = threadIdx.x / TPL;
    const int tl = threadIdx.x % TPL;   // thread within the line
    const int q = tl / G, t = tl % G;
    const cx<T>* U1 = In + (size_t)ll * 3 * L;
    const cx<T>* U2 = U1 + L;
    const cx<T>* U3 = U2 + L;
    cx<T>* Sl = Ex + (size_t)ll * 3 * SZ;   // the line's three regions
    cx<T>* S = Sl + (size_t)q * SZ;         // this sub-transform's region
    uint64_t* full = bars + ll;
    const long cs = MM * L;                 // component stride (complex) of in and out
    const long groups = (long)gridDim.x * LPB;
    constexpr uint32_t LINE_BYTES = (uint32_t)(L * sizeof(cx<T>));

    auto issue = [&](long line) {
        const long b = line / MM, pp = line % MM;
        const cx<T>* src = in + (b * 3 * MM + pp) * L;
        mbar_expect_tx(full, 3 * LINE_BYTES);
#pragma unroll
        for (int c = 0; c < 3; ++c) bulk_g2s(const_cast<cx<T>*>(U1) + c * L, src + c * cs, LINE_BYTES, full);
    };

    if (threadIdx.x == 0) {
        for (int k = 0; k < LPB; ++k) mbar_init(bars + k, 1);
        mbar_fence_init();
    }
    __syncthreads();
    long line = (long)blockIdx.x * LPB + ll;
    if (tl == 0 && line < total_lines) issue(line);
    uint32_t parity = 0;
    const int bar_id = 1 + ll / UL;

    for (; line < total_lines; line += groups, parity ^= 1) {
        const long b = line / MM, pp = line % MM;
        mbar_wait(full, parity);

        cx<T> v[8];
        T u3r[8];
        cx<T> u12[8];
        // ---------------- u3 alone
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int n = t + G * j;
            const cx<T> p3 = U3[n];
            cx<T> a, c;
            if (n == 0) { a = mk<T>(p3.x, 0); c = mk<T>(0, 0); }
            else { a = p3; c = conj(U3[L - n]); }
            v[j] = prune3(a, c, q, n, tw);
        }
        z8_inverse<T, L>(v, S, t, tw);
#pragma unroll
        for (int k = 0; k < 8; ++k) u3r[k] = v[k].x;
        // ---------------- pair (u1, u2)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int n = t + G * j;
            const cx<T> p1 = U1[n], p2 = U2[n];
            cx<T> a, c;
            if (n == 0) { a = mk<T>(p1.x, p2.x); c = mk<T>(0, 0); }
            else {
                const cx<T> m1 = U1[L - n], m2 = U2[L - n];
                a = mk<T>(p1.x - p2.y, p1.y + p2.x);
                c = mk<T>(m1.x + m2.y, m2.x - m1.y);
            }
            u12[j] = prune3(a, c, q, n, tw);
        }
        z8_inverse<T, L>(u12, S, t, tw);
        if (umax2 != nullptr) {
            auto lmax = sq_bits((T)0);
#pragma unroll
            for (int k = 0; k < 8; ++k) lmax = umax_bits(lmax, sq_bits(u12[k].x * u12[k].x + u12[k].y * u12[k].y + u3r[k] * u3r[k]));
            // lanes of a warp may belong to different lines, but (LPB | MM) to the same sample
            lmax = warp_max_bits(lmax);
            if ((threadIdx.x & 31) == 0) atomic_max_sq(umax2 + b, lmax);
        }
        // ---------------- forward pairs (T11,T22) (T12,T13) (T23,-), see kernels_z.cuh
        cx<T>* Op = out + (b * 5 * MM + pp) * L;
#pragma unroll 1
        for (int pair = 0; pair < 3; ++pair) {
            const int ca = pair == 0 ? 0 : (pair == 1 ? 1 : 4);
            const int cb = pair == 0 ? 3 : 2;  // unused for pair 2
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const cx<T> w = u12[k];
                const T w3 = u3r[k];
                v[k] = pair == 0 ? mk<T>(w.x * w.x - w3 * w3, w.y * w.y - w3 * w3) : (pair == 1 ? mk<T>(w.x * w.y, w.x * w3) : mk<T>(w.y * w3, 0));
            }
            z8_forward<T, L>(v, S, t, tw);
            // F_q[n] W^{-qn} into this sub-transform's region, natural order
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int n = t + G * j;
                cx<T> w = v[brev<8>(j)];
                if (q > 0) w = cmulc(w, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
                S[n] = w;
            }
            named_bar_sync(bar_id, UT);
            // the line's inputs were consumed long ago by all three warps: prefetch the next line
            if (pair == 0 && tl == 0 && line + groups < total_lines) issue(line + groups);
            z_combine_store<T, L, SZ, TPL>(Sl, Op + ca * cs, Op + cb * cs, pair < 2, tl);
            named_bar_sync(bar_id, UT);  // combine reads done before the regions are reused
        }
    }
}

}  // namespace ns
