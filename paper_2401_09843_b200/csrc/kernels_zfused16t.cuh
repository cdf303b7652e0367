// kernels_zfused16t.cuh -- steps a3 + a4 of SURVEY.md section 8(a) in one kernel for the longest lines
// (L = N/2 in {128, 256}): per (px,py) line, pad + inverse c2r along z, the trace-free flux products, max|u|^2,
// forward r2c + truncate (Algorithm 2 steps 1-5).  16 values per lane (kernels_zfused16.cuh)
// with the physical-space fields parked in TENSOR MEMORY instead of registers / shared memory.
//
// The kernel is latency bound and scales with the number of resident warps (profiles/r01b_tmem.md); registers and
// shared memory both cap it.  u1, u2 and u3 on the padded line (48 words per thread in fp64) live in TMEM
// (tmem.cuh), which costs neither: 128 (fp64) / 64 (fp32) columns per CTA, four CTAs per SM.  Registers then hold only
// the transform being worked on, and shared memory only the TMA input lines and the exchange / combine regions.
#pragma once
#include <cstdint>

#include "cx.cuh"
#include "kernels_zfused16.cuh"
#include "tmem.cuh"

namespace ns {

// in [batch][3][MM][L] complex -> out [batch][5][MM][L] complex (unnormalised transforms of the flux components)
// One unit (96 threads = 3 warps = the three sub-transforms q of 32/G neighbouring lines) per block.
template <typename T, int L, int MINB>
__global__ void __launch_bounds__(96, MINB)
z_fused16t_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, long MM, long total_lines,
                  unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    using Geo = Z16Geo<L>;
    constexpr int G = Geo::G, SZ = Geo::SZ, UL = Geo::UL;
    constexpr int LPB = UL;              // lines per block
    constexpr int TPL = 3 * G;           // threads per line
    constexpr uint32_t C16 = tmem_cols16<T>();                 // TMEM columns of 16 scalars
    constexpr uint32_t NCOLS = 3 * C16 <= 64 ? 64 : 128;       // u1 | u2 | u3 blocks, rounded up to a power of two
    static_assert(SZ >= L, "combine region must hold a sub-transform");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* In = reinterpret_cast<cx<T>*>(smem_raw);   // [LPB][3][L]
    cx<T>* Ex = In + (size_t)LPB * 3 * L;              // [LPB][3][SZ]
    uint64_t* bars = reinterpret_cast<uint64_t*>(Ex + (size_t)LPB * 3 * SZ);  // [LPB]
    uint32_t* tslot = reinterpret_cast<uint32_t*>(bars + LPB);

    const int q = threadIdx.x / 32;                 // warp = sub-transform q
    const int lane = threadIdx.x & 31;
    const int ll = lane / G;                         // line within the block
    const int t = lane % G;
    const int tl = q * G + t;                        // thread within the line
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
    if (q == 0) tmem_alloc(tslot, NCOLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    // this warp's TMEM window: lanes 32 q .. 32 q + 31, columns [0, 3 C16)
    const uint32_t tbase = *tslot + ((uint32_t)(32 * q) << 16);
    const uint32_t tX = tbase, tY = tbase + C16, tZ = tbase + 2 * C16;

    long line = (long)blockIdx.x * LPB + ll;
    if (tl == 0 && line < total_lines) issue(line);
    uint32_t parity = 0;

    for (; line < total_lines; line += groups, parity ^= 1) {
        const long b = line / MM, pp = line % MM;
        mbar_wait(full, parity);

        cx<T> v[16];
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
        {
            T w3[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) w3[k] = v[k].x;
            tmem_store16(tZ, w3);
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
            v[j] = prune3(a, c, q, n, tw);
        }
        z16_inverse<T, L>(v, S, t, tw);
        {
            T wx[16], wy[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) { wx[k] = v[k].x; wy[k] = v[k].y; }
            tmem_store16(tX, wx);
            tmem_store16(tY, wy);
        }
        tmem_wait_st();
        // ---------------- forward pairs (T11,T22) (T12,T13) (T23,-), see kernels_z.cuh
        cx<T>* Op = out + (b * 5 * MM + pp) * L;
#pragma unroll 1
        for (int pair = 0; pair < 3; ++pair) {
            const int ca = pair == 0 ? 0 : (pair == 1 ? 1 : 4);
            const int cb = pair == 0 ? 3 : 2;  // unused for pair 2
            {
                T w3[16];
                tmem_load16(tZ, w3);
                if (pair == 0) {
                    // v still holds u1 + i u2
                    auto lmax = sq_bits((T)0);
#pragma unroll
                    for (int k = 0; k < 16; ++k) {
                        const T x2 = v[k].x * v[k].x, y2 = v[k].y * v[k].y, z2 = w3[k] * w3[k];
                        lmax = umax_bits(lmax, sq_bits(x2 + y2 + z2));
                        v[k] = mk<T>(x2 - z2, y2 - z2);
                    }
                    if (umax2 != nullptr) {
                        // lanes of a warp belong to neighbouring lines of the same sample (LPB | MM)
                        lmax = warp_max_bits(lmax);
                        if (lane == 0) atomic_max_sq(umax2 + b, lmax);
                    }
                } else if (pair == 1) {
                    T wx[16], wy[16];
                    tmem_load16(tX, wx);
                    tmem_load16(tY, wy);
#pragma unroll
                    for (int k = 0; k < 16; ++k) v[k] = mk<T>(wx[k] * wy[k], wx[k] * w3[k]);
                } else {
                    T wy[16];
                    tmem_load16(tY, wy);
#pragma unroll
                    for (int k = 0; k < 16; ++k) v[k] = mk<T>(wy[k] * w3[k], 0);
                }
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
            named_bar_sync(1, 96);
            // the line's inputs were consumed long ago by all three warps: prefetch the next line
            if (pair == 0 && tl == 0 && line + groups < total_lines) issue(line + groups);
            z_combine_store<T, L, SZ, TPL>(Sl, Op + ca * cs, Op + cb * cs, pair < 2, tl);
            named_bar_sync(1, 96);  // combine reads done before the regions are reused
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (q == 0) tmem_dealloc(*tslot, NCOLS);
}

}  // namespace ns
