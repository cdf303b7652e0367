// kernels_zfused16.cuh -- steps a3 + a4 of SURVEY.md section 8(a) in one kernel, 16-values-per-lane version
// for the longest lines (L = N/2 in {128, 256}): per (px,py) line, pad + inverse c2r along z, the flux
// products, max|u|^2, forward r2c + truncate (Algorithm 2 steps 1-5).
//
// Same mathematics as kernels_z.cuh; compared with kernels_zfused8.cuh every lane holds 16 complex values,
// so a length-L sub-transform q is 16 x G (G = L/16 lanes of one warp) with ONE warp-local shared-memory
// exchange instead of two, and half as many inter-stage twiddle loads.  The kernel is limited by the
// L1/shared-memory pipe (profiles/), so bytes through that pipe are what the layout minimises:
//   * u12 = u1 + i u2 stays in registers; the real field u3 is parked in shared memory (8 B per point) and
//     re-read while the products of each forward pair are formed, which keeps the kernel under 170 registers;
//   * one warp works on the same q of 32/G neighbouring lines, so the q-dependent code does not diverge.
// Block-level synchronisation (a named barrier per unit of 96 threads = 3 warps = 32/G lines) is needed only
// where the three sub-transforms of a line meet (3 -> 2 combine + Hermitian split of each forward pair).
// Input lines of the next iteration are prefetched by the TMA bulk-copy engine (cp.async.bulk + mbarrier).
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

// in [batch][3][MM][L] complex -> out [batch][5][MM][L] complex (unnormalised transforms of the flux components)
// UPB units (of 96 threads) per block; STASH3: park u3 in shared memory instead of registers.
template <typename T, int L, int UPB, int MINB, bool STASH3>
__global__ void __launch_bounds__(96 * UPB, MINB)
z_fused16_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, long MM, long total_lines,
                 unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    using Geo = Z16Geo<L>;
    constexpr int G = Geo::G, SZ = Geo::SZ, UL = Geo::UL;
    constexpr int LPB = UL * UPB;        // lines per block
    constexpr int TPL = 3 * G;           // threads per line
    static_assert(SZ >= L, "combine region must hold a sub-transform");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* In = reinterpret_cast<cx<T>*>(smem_raw);   // [LPB][3][L]
    cx<T>* Ex = In + (size_t)LPB * 3 * L;              // [LPB][3][SZ]
    T* St = reinterpret_cast<T*>(Ex + (size_t)LPB * 3 * SZ);  // [LPB][3][16][G] (STASH3 only)
    uint64_t* bars = reinterpret_cast<uint64_t*>(St + (STASH3 ? (size_t)LPB * 3 * L : 0));  // [LPB]

    const int unit = threadIdx.x / 96;
    const int q = (threadIdx.x % 96) / 32;          // warp within the unit
    const int lane = threadIdx.x & 31;
    const int ll = unit * UL + lane / G;             // line within the block
    const int t = lane % G;
    const int tl = q * G + t;                        // thread within the line
    const cx<T>* U1 = In + (size_t)ll * 3 * L;
    const cx<T>* U2 = U1 + L;
    const cx<T>* U3 = U2 + L;
    cx<T>* Sl = Ex + (size_t)ll * 3 * SZ;   // the line's three regions
    cx<T>* S = Sl + (size_t)q * SZ;         // this sub-transform's region
    T* S3 = St + ((size_t)ll * 3 + q) * L + t;  // this lane's column of the u3 stash, stride G
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
    const int bar_id = 1 + unit;

    for (; line < total_lines; line += groups, parity ^= 1) {
        const long b = line / MM, pp = line % MM;
        mbar_wait(full, parity);

        cx<T> v[16];
        cx<T> u12[16];
        T u3r[STASH3 ? 1 : 16];
        // ---------------- u3 alone
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int n = t + G * j;
            const cx<T> p3 = U3[n];
            cx<T> a, c;
            if (n == 0) { a = mk<T>(p3.x, 0); c = mk<T>(0, 0); }
            else { a = p3; c = conj(U3[L - n]); }
            v[j] = prune3(a, c, q, n, tw);
        }
        z16_inverse<T, L>(v, S, t, tw);
        if constexpr (STASH3) {
#pragma unroll
            for (int k = 0; k < 16; ++k) S3[k * G] = v[k].x;
        } else {
#pragma unroll
            for (int k = 0; k < 16; ++k) u3r[k] = v[k].x;
        }
        // ---------------- pair (u1, u2)
#pragma unroll
        for (int j = 0; j < 16; ++j) {
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
        z16_inverse<T, L>(u12, S, t, tw);
        if (umax2 != nullptr) {
            T lmax = 0;
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                T w3;
                if constexpr (STASH3) w3 = S3[k * G]; else w3 = u3r[k];
                lmax = fmax(lmax, u12[k].x * u12[k].x + u12[k].y * u12[k].y + w3 * w3);
            }
            // lanes of a warp belong to neighbouring lines of the same sample (LPB | MM)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) lmax = fmax(lmax, __shfl_xor_sync(0xffffffffu, lmax, o));
            if (lane == 0) atomic_max_nonneg(umax2 + b, (double)lmax);
        }
        // ---------------- forward pairs (T11,T22) (T12,T13) (T23,-), see kernels_z.cuh
        cx<T>* Op = out + (b * 5 * MM + pp) * L;
#pragma unroll 1
        for (int pair = 0; pair < 3; ++pair) {
            const int ca = pair == 0 ? 0 : (pair == 1 ? 1 : 4);
            const int cb = pair == 0 ? 3 : 2;  // unused for pair 2
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const cx<T> w = u12[k];
                T w3;
                if constexpr (STASH3) w3 = S3[k * G]; else w3 = u3r[k];
                v[k] = pair == 0 ? mk<T>(w.x * w.x - w3 * w3, w.y * w.y - w3 * w3) : (pair == 1 ? mk<T>(w.x * w.y, w.x * w3) : mk<T>(w.y * w3, 0));
            }
            z16_forward<T, L>(v, S, t, tw);
            // F_q[n] W^{-qn} into this sub-transform's region, natural order
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int n = t + G * j;
                cx<T> w = v[brev<16>(j)];
                if (q > 0) w = cmulc(w, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
                S[n] = w;
            }
            named_bar_sync(bar_id, 96);
            // the line's inputs were consumed long ago by all three warps: prefetch the next line
            if (pair == 0 && tl == 0 && line + groups < total_lines) issue(line + groups);
            {
                constexpr T h3 = (T)0.86602540378443864676L;
                for (int n = tl; n <= L / 2; n += TPL) {
                    const cx<T> f0 = Sl[n], g1 = Sl[SZ + n], g2 = Sl[2 * SZ + n];
                    const cx<T> Sm_ = g1 + g2, D = g1 - g2;
                    const cx<T> An = f0 + Sm_;
                    if (n == 0) {
                        Op[ca * cs] = mk<T>(An.x, 0);
                        if (pair < 2) Op[cb * cs] = mk<T>(An.y, 0);
                    } else {
                        const cx<T> Cn = mk<T>(f0.x - (T)0.5 * Sm_.x - h3 * D.y, f0.y - (T)0.5 * Sm_.y + h3 * D.x);
                        const int m = L - n;
                        const cx<T> f0m = Sl[m], g1m = Sl[SZ + m], g2m = Sl[2 * SZ + m];
                        const cx<T> Sm = g1m + g2m, Dm = g1m - g2m;
                        const cx<T> Am = f0m + Sm;
                        const cx<T> Cm = mk<T>(f0m.x - (T)0.5 * Sm.x - h3 * Dm.y, f0m.y - (T)0.5 * Sm.y + h3 * Dm.x);
                        Op[ca * cs + n] = mk<T>((T)0.5 * (An.x + Cm.x), (T)0.5 * (An.y - Cm.y));
                        if (pair < 2) Op[cb * cs + n] = mk<T>((T)0.5 * (An.y + Cm.y), (T)0.5 * (Cm.x - An.x));
                        if (m != n) {
                            Op[ca * cs + m] = mk<T>((T)0.5 * (Am.x + Cn.x), (T)0.5 * (Am.y - Cn.y));
                            if (pair < 2) Op[cb * cs + m] = mk<T>((T)0.5 * (Am.y + Cn.y), (T)0.5 * (Cn.x - Am.x));
                        }
                    }
                }
            }
            named_bar_sync(bar_id, 96);  // combine reads done before the regions are reused
        }
    }
}

}  // namespace ns
