// kernels_zfused.cuh -- steps a3 + a4 of SURVEY.md section 8(a) in ONE kernel (the "beyond the model"
// fusion of SURVEY.md section 7 item 5(i)): per (px,py) line, pad + inverse c2r along z, the flux
// products u_i u_j (Algorithm 2 steps 2-3), max|u|^2, forward r2c + truncate
// (steps 4-5).  The M^3 physical arrays never touch HBM: the kernel reads 3 half
// spectra lines and writes 5.
//
// Persistent CTAs; the input lines of the NEXT tile are fetched by the TMA bulk-copy engine
// (cp.async.bulk, completion on an mbarrier) into shared memory while the current tile is being
// transformed, so HBM latency is hidden without occupancy.  Same pruned radix-3 / two-for-one math as
// kernels_z.cuh; thread layout per line: 3 (q) x P threads.
#pragma once
#include <cstdint>

#include "cx.cuh"
#include "kernels_z.cuh"

namespace ns {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}

// named barrier among `nthreads` threads of the CTA (a unit / a team), id 1..15
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// s_q[n] = (a + c w3^{-q}) W^{qn}
template <typename T>
__device__ __forceinline__ cx<T> prune3(cx<T> a, cx<T> c, int q, int n, const Twiddles<T>& tw) {
    if (q == 0) return a + c;
    constexpr T h3 = (T)0.86602540378443864676L;
    const cx<T> t1 = mk<T>(a.x - (T)0.5 * c.x, a.y - (T)0.5 * c.y);
    const cx<T> t2 = h3 * c;
    const cx<T> z = (q == 1) ? mk<T>(t1.x + t2.y, t1.y - t2.x) : mk<T>(t1.x - t2.y, t1.y + t2.x);
    return cmul(z, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
}

// in [batch][3][MM][L] complex -> out [batch][5][MM][L] complex (unnormalised transforms of the flux components)
template <typename T, int L, int R1, int R2, int LPB, int MINB>
__global__ void __launch_bounds__(3 * ZP<R1, R2>::value* LPB, MINB)
z_fused_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, long MM, long total_tiles,
               unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    static_assert(R1 * R2 == L && R2 >= 2, "two register stages");
    constexpr int P = ZP<R1, R2>::value;
    constexpr int PITCH = R2 + 1;
    constexpr int ELINE = 3 * R1 * PITCH;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* In = reinterpret_cast<cx<T>*>(smem_raw);   // [3][LPB][L]
    cx<T>* E = In + (size_t)3 * LPB * L;               // [LPB][3][R1][PITCH] exchange buffer
    cx<T>* Cb = E;   // the combine reads the exchange buffer itself
    uint64_t* full = reinterpret_cast<uint64_t*>(E + (size_t)LPB * ELINE);

    const int i = threadIdx.x % P;
    const int q = (threadIdx.x / P) % 3;
    const int ll = threadIdx.x / (3 * P);
    cx<T>* Eq = E + (size_t)ll * ELINE + (size_t)q * R1 * PITCH;
    const cx<T>* El = Cb + (size_t)ll * ELINE;
    cx<T>* Cq = Cb + (size_t)ll * ELINE + (size_t)q * R1 * PITCH;
    // element n of sub-transform qq in the combine layout (= the exchange layout, row n / R2, column n % R2)
    auto cidx = [](int qq, int n) { return qq * R1 * PITCH + (n / R2) * PITCH + (n % R2); };
    const cx<T>* U1 = In + (size_t)ll * L;
    const cx<T>* U2 = U1 + (size_t)LPB * L;
    const cx<T>* U3 = U2 + (size_t)LPB * L;
    const long cs = MM * L;  // component stride (complex) of in and out
    constexpr uint32_t COMP_BYTES = (uint32_t)(LPB * L * sizeof(cx<T>));

    auto issue = [&](long tile) {
        const long line0 = tile * LPB;
        const long b = line0 / MM, pp = line0 % MM;
        const cx<T>* src = in + (b * 3 * MM + pp) * L;
        mbar_expect_tx(full, 3 * COMP_BYTES);
#pragma unroll
        for (int c = 0; c < 3; ++c) bulk_g2s(In + (size_t)c * LPB * L, src + c * cs, COMP_BYTES, full);
    };

    if (threadIdx.x == 0) {
        mbar_init(full, 1);
        mbar_fence_init();
    }
    __syncthreads();
    long tile = blockIdx.x;
    if (threadIdx.x == 0 && tile < total_tiles) issue(tile);
    uint32_t parity = 0;

    for (; tile < total_tiles; tile += gridDim.x, parity ^= 1) {
        const long line = tile * LPB + ll;
        const long b = line / MM, pp = line % MM;
        mbar_wait(full, parity);

        T u3r[R2];
        cx<T> u12[R2];
        // ---------------- u3 alone
        if (i < R2) {
            cx<T> s[R1];
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) {
                const int n = R2 * n1 + i;
                const cx<T> p3 = U3[n];
                cx<T> a, c;
                if (n == 0) { a = mk<T>(p3.x, 0); c = mk<T>(0, 0); }
                else { a = p3; c = conj(U3[L - n]); }
                s[n1] = prune3(a, c, q, n, tw);
            }
            fft_reg<R1, +1, T>(s);
#pragma unroll
            for (int r1 = 0; r1 < R1; ++r1) {
                cx<T> v = s[outpos<R1>(r1)];
                if (r1 > 0) v = cmul(v, ldg(tw.twA + r1 * R2 + i));
                Eq[r1 * PITCH + i] = v;
            }
        }
        __syncthreads();
        if (i < R1) {
            cx<T> y[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) y[n2] = Eq[i * PITCH + n2];
            fft_reg<R2, +1, T>(y);
#pragma unroll
            for (int j = 0; j < R2; ++j) u3r[j] = y[j].x;  // u3r[j] holds r2 = brev(j)
        }
        __syncthreads();
        // ---------------- pair (u1, u2)
        if (i < R2) {
            cx<T> s[R1];
#pragma unroll
            for (int n1 = 0; n1 < R1; ++n1) {
                const int n = R2 * n1 + i;
                const cx<T> p1 = U1[n], p2 = U2[n];
                cx<T> a, c;
                if (n == 0) { a = mk<T>(p1.x, p2.x); c = mk<T>(0, 0); }
                else {
                    const cx<T> m1 = U1[L - n], m2 = U2[L - n];
                    a = mk<T>(p1.x - p2.y, p1.y + p2.x);
                    c = mk<T>(m1.x + m2.y, m2.x - m1.y);
                }
                s[n1] = prune3(a, c, q, n, tw);
            }
            fft_reg<R1, +1, T>(s);
#pragma unroll
            for (int r1 = 0; r1 < R1; ++r1) {
                cx<T> v = s[outpos<R1>(r1)];
                if (r1 > 0) v = cmul(v, ldg(tw.twA + r1 * R2 + i));
                Eq[r1 * PITCH + i] = v;
            }
        }
        __syncthreads();
        // the input lines are consumed: start fetching the next tile into the same buffer
        if (threadIdx.x == 0 && tile + gridDim.x < total_tiles) issue(tile + gridDim.x);
        if (i < R1) {
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) u12[n2] = Eq[i * PITCH + n2];
            fft_reg<R2, +1, T>(u12);  // u12[j] holds r2 = brev(j)
        }
        if (umax2 != nullptr) {
            auto lmax = sq_bits((T)0);
            if (i < R1) {
#pragma unroll
                for (int j = 0; j < R2; ++j) lmax = umax_bits(lmax, sq_bits(u12[j].x * u12[j].x + u12[j].y * u12[j].y + u3r[j] * u3r[j]));
            }
            lmax = warp_max_bits(lmax);
            if ((threadIdx.x & 31) == 0) atomic_max_sq(umax2 + b, lmax);
        }
        // ---------------- forward pairs (T11,T22) (T12,T13) (T23,-), see kernels_z.cuh
        cx<T>* Op = out + (b * 5 * MM + pp) * L;
#pragma unroll 1
        for (int pair = 0; pair < 3; ++pair) {
            const int ca = pair == 0 ? 0 : (pair == 1 ? 1 : 4);
            const int cb = pair == 0 ? 3 : 2;  // unused for pair 2
            if (i < R1) {
                cx<T> x[R2];
#pragma unroll
                for (int r2 = 0; r2 < R2; ++r2) {
                    const cx<T> w = u12[outpos<R2>(r2)];
                    const T w3 = u3r[outpos<R2>(r2)];
                    x[r2] = pair == 0 ? mk<T>(w.x * w.x - w3 * w3, w.y * w.y - w3 * w3) : (pair == 1 ? mk<T>(w.x * w.y, w.x * w3) : mk<T>(w.y * w3, 0));
                }
                fft_reg<R2, -1, T>(x);
                // pair 0: this thread overwrites the row only it has read in stage B above; later pairs: barrier above
#pragma unroll
                for (int n2 = 0; n2 < R2; ++n2) {
                    cx<T> v = x[outpos<R2>(n2)];
                    if (n2 > 0) v = cmulc(v, ldg(tw.twB + n2 * R1 + i));
                    Eq[i * PITCH + n2] = v;
                }
            }
            __syncthreads();
            if (i < R2) {
                cx<T> y[R1];
#pragma unroll
                for (int r1 = 0; r1 < R1; ++r1) y[r1] = Eq[r1 * PITCH + i];
                fft_reg<R1, -1, T>(y);
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    const int n = R2 * n1 + i;
                    cx<T> v = y[outpos<R1>(n1)];
                    if (q > 0) v = cmulc(v, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
                    Cq[n1 * PITCH + i] = v;  // when aliased: overwrites exactly the column this thread has just read
                }
            }
            __syncthreads();
            {
                constexpr T h3 = (T)0.86602540378443864676L;
                const int t = q * P + i;
                for (int n = t; n <= L / 2; n += 3 * P) {
                    const cx<T> f0 = El[cidx(0, n)], g1 = El[cidx(1, n)], g2 = El[cidx(2, n)];
                    const cx<T> S = g1 + g2, D = g1 - g2;
                    const cx<T> An = f0 + S;
                    if (n == 0) {
                        Op[ca * cs] = mk<T>(An.x, 0);
                        if (pair < 2) Op[cb * cs] = mk<T>(An.y, 0);
                    } else {
                        const cx<T> Cn = mk<T>(f0.x - (T)0.5 * S.x - h3 * D.y, f0.y - (T)0.5 * S.y + h3 * D.x);
                        const int m = L - n;
                        const cx<T> f0m = El[cidx(0, m)], g1m = El[cidx(1, m)], g2m = El[cidx(2, m)];
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
            __syncthreads();  // combine reads done before E is rewritten (next pair / next tile)
        }
    }
}

}  // namespace ns
