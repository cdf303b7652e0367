// kernels_z.cuh -- contiguous-axis (z) passes: step a3 (pad + inverse c2r + six products + max|u|)
// and step a4 (forward r2c + truncate) of SURVEY.md section 8(a); Algorithm 2 steps 2-5 and
// Algorithm 3 steps 4-5 of the paper (six products per PAPER.md:L245).
//
// Real transforms use the two-for-one trick on the same pruned radix-3 core as kernels_col.cuh:
//   inverse  z = u_a + i u_b  has spectrum Z[k] = U_a[k] + i U_b[k]; for k < 0, U[k] = conj(U[-k]), so
//            a_n = U_a[n] + i U_b[n],  c_n = conj(U_a[L-n]) + i conj(U_b[L-n])  (n >= 1), c_0 = 0,
//            and a_0 uses only the real parts of U[0] (the c2r definition: u is the real part).
//   forward  z = B_a + i B_b;  B_a^[n] = (A_n + conj(C_{L-n}))/2,  B_b^[n] = (A_n - conj(C_{L-n}))/(2i).
// The physical z axis is stored in the decimated order pz = q*L + r (physical index 3r + q).
//
// Thread layout per line: 3 (q) x P threads, q-parallel; lanes run along the line so every global
// access is contiguous.  The exchange buffer rows are padded to R2+1 elements (conflict-free
// transposes for 16-byte and 8-byte elements).
#pragma once
#include "cx.cuh"
#include "ns_internal.h"

namespace ns {

template <int R1, int R2> struct ZP { static constexpr int value = R1 > R2 ? R1 : R2; };

// Products are stored in this order (same as the spectral kernel expects): 11 12 13 22 23 33.
// Forward pairs: (11,22) (33,12) (13,23).

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* addr, double v) {
    atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

// ------------------------------------------------------------------------------------------------
// a3: in  [batch][3][MM][L] complex (kz < L),  out [batch][6][MM][3L] real,  MM = M*M lines per sample
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R1, int R2, int LPB>
__global__ void __launch_bounds__(3 * ZP<R1, R2>::value* LPB)
z_inv_prod_kernel(const cx<T>* __restrict__ in, T* __restrict__ out, long MM, long total_lines,
                  unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    static_assert(R1 * R2 == L && R2 >= 2, "two register stages");
    constexpr int P = ZP<R1, R2>::value;
    constexpr int PITCH = R2 + 1;
    constexpr int ELINE = 3 * R1 * PITCH;  // exchange elements per line per buffer
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* E = reinterpret_cast<cx<T>*>(smem_raw);  // [2][LPB][3][R1][PITCH]

    const int i = threadIdx.x % P;
    const int q = (threadIdx.x / P) % 3;
    const int ll = threadIdx.x / (3 * P);
    long line = (long)blockIdx.x * LPB + ll;
    if (line >= total_lines) line = total_lines - 1;
    const long b = line / MM, pp = line % MM;
    const cx<T>* U = in + (b * 3 * MM + pp) * L;
    const long cs = MM * L;  // component stride (complex)
    cx<T>* Eq = E + (size_t)ll * ELINE + (size_t)q * R1 * PITCH;
    constexpr size_t EBUF = (size_t)LPB * ELINE;

    cx<T> u12[R2];
    // ---------------- pair (u1, u2)
    if (i < R2) {
        cx<T> s[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int n = R2 * n1 + i;
            const cx<T> p1 = ldg(U + n), p2 = ldg(U + cs + n);
            cx<T> a, c;
            if (n == 0) {
                a = mk<T>(p1.x, p2.x);
                c = mk<T>(0, 0);
            } else {
                const cx<T> m1 = ldg(U + (L - n)), m2 = ldg(U + cs + (L - n));
                a = mk<T>(p1.x - p2.y, p1.y + p2.x);
                c = mk<T>(m1.x + m2.y, m2.x - m1.y);
            }
            // s_q[n] = (a + c w3^{-q}) W^{qn}
            if (q == 0) {
                s[n1] = a + c;
            } else {
                constexpr T h3 = (T)0.86602540378443864676L;
                const cx<T> t1 = mk<T>(a.x - (T)0.5 * c.x, a.y - (T)0.5 * c.y);
                const cx<T> t2 = h3 * c;
                const cx<T> z = (q == 1) ? mk<T>(t1.x + t2.y, t1.y - t2.x) : mk<T>(t1.x - t2.y, t1.y + t2.x);
                s[n1] = cmul(z, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
            }
        }
        fft_reg<R1, +1, T>(s);
#pragma unroll
        for (int r1 = 0; r1 < R1; ++r1) {
            cx<T> v = s[brev<R1>(r1)];
            if (r1 > 0) v = cmul(v, ldg(tw.twA + r1 * R2 + i));
            Eq[r1 * PITCH + i] = v;
        }
    }
    __syncthreads();
    if (i < R1) {
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) u12[n2] = Eq[i * PITCH + n2];
        fft_reg<R2, +1, T>(u12);
    }
    // ---------------- u3 alone (second exchange buffer: no barrier needed before writing)
    if (i < R2) {
        cx<T> s[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int n = R2 * n1 + i;
            const cx<T> p3 = ldg(U + 2 * cs + n);
            cx<T> a, c;
            if (n == 0) {
                a = mk<T>(p3.x, 0);
                c = mk<T>(0, 0);
            } else {
                a = p3;
                c = conj(ldg(U + 2 * cs + (L - n)));
            }
            if (q == 0) {
                s[n1] = a + c;
            } else {
                constexpr T h3 = (T)0.86602540378443864676L;
                const cx<T> t1 = mk<T>(a.x - (T)0.5 * c.x, a.y - (T)0.5 * c.y);
                const cx<T> t2 = h3 * c;
                const cx<T> z = (q == 1) ? mk<T>(t1.x + t2.y, t1.y - t2.x) : mk<T>(t1.x - t2.y, t1.y + t2.x);
                s[n1] = cmul(z, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
            }
        }
        fft_reg<R1, +1, T>(s);
#pragma unroll
        for (int r1 = 0; r1 < R1; ++r1) {
            cx<T> v = s[brev<R1>(r1)];
            if (r1 > 0) v = cmul(v, ldg(tw.twA + r1 * R2 + i));
            Eq[EBUF + r1 * PITCH + i] = v;
        }
    }
    __syncthreads();
    T lmax = 0;
    if (i < R1) {
        cx<T> u3[R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) u3[n2] = Eq[EBUF + i * PITCH + n2];
        fft_reg<R2, +1, T>(u3);
        constexpr int M = 3 * L;
        T* o = out + (b * 6 * MM + pp) * M + q * L + i;
        const long ps = MM * M;  // product-component stride (reals)
#pragma unroll
        for (int r2 = 0; r2 < R2; ++r2) {
            const T w1 = u12[brev<R2>(r2)].x, w2 = u12[brev<R2>(r2)].y, w3 = u3[brev<R2>(r2)].x;
            const int off = R1 * r2;
            o[off] = w1 * w1;
            o[ps + off] = w1 * w2;
            o[2 * ps + off] = w1 * w3;
            o[3 * ps + off] = w2 * w2;
            o[4 * ps + off] = w2 * w3;
            o[5 * ps + off] = w3 * w3;
            lmax = fmax(lmax, w1 * w1 + w2 * w2 + w3 * w3);
        }
    }
    if (umax2 != nullptr) {
        // all lines of a block belong to one sample only if LPB divides MM; reduce per thread -> warp -> atomic
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            // lanes of one warp may belong to different lines but, when LPB | MM, to the same sample
            lmax = fmax(lmax, __shfl_xor_sync(0xffffffffu, lmax, o));
        }
        if ((threadIdx.x & 31) == 0) atomic_max_nonneg(umax2 + b, (double)lmax);
    }
}

// ------------------------------------------------------------------------------------------------
// a4: in [batch][6][MM][3L] real,  out [batch][6][MM][L] complex (kz < L)
// ------------------------------------------------------------------------------------------------
template <typename T, int L, int R1, int R2, int LPB>
__global__ void __launch_bounds__(3 * ZP<R1, R2>::value* LPB)
z_fwd_kernel(const T* __restrict__ in, cx<T>* __restrict__ out, long MM, long total_lines,
             Twiddles<T> tw) {
    static_assert(R1 * R2 == L && R2 >= 2, "two register stages");
    constexpr int P = ZP<R1, R2>::value;
    constexpr int PITCH = R2 + 1;
    constexpr int ELINE = 3 * R1 * PITCH;
    constexpr int M = 3 * L;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* E = reinterpret_cast<cx<T>*>(smem_raw);        // [LPB][3][R1][PITCH]
    cx<T>* Cmb = E + (size_t)LPB * ELINE;                 // [LPB][3][L]

    const int i = threadIdx.x % P;
    const int q = (threadIdx.x / P) % 3;
    const int ll = threadIdx.x / (3 * P);
    long line = (long)blockIdx.x * LPB + ll;
    if (line >= total_lines) line = total_lines - 1;
    const long b = line / MM, pp = line % MM;
    const long ps = MM * M;   // input component stride (reals)
    const long cs = MM * L;   // output component stride (complex)
    const T* Bp = in + (b * 6 * MM + pp) * M;
    cx<T>* Op = out + (b * 6 * MM + pp) * L;
    cx<T>* Eq = E + (size_t)ll * ELINE + (size_t)q * R1 * PITCH;
    cx<T>* Cl = Cmb + (size_t)ll * 3 * L;

#pragma unroll 1
    for (int pair = 0; pair < 3; ++pair) {
        // (11,22) (33,12) (13,23)  with component order 11 12 13 22 23 33 = 0..5
        const int ca = pair == 0 ? 0 : (pair == 1 ? 5 : 2);
        const int cb = pair == 0 ? 3 : (pair == 1 ? 1 : 4);
        if (i < R1) {
            cx<T> x[R2];
            const T* pa = Bp + ca * ps + q * L + i;
            const T* pb = Bp + cb * ps + q * L + i;
#pragma unroll
            for (int r2 = 0; r2 < R2; ++r2) x[r2] = mk<T>(__ldg(pa + R1 * r2), __ldg(pb + R1 * r2));
            fft_reg<R2, -1, T>(x);
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) {
                cx<T> v = x[brev<R2>(n2)];
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
                cx<T> v = y[brev<R1>(n1)];
                if (q > 0) v = cmulc(v, ldg((q == 1 ? tw.w3a : tw.w3b) + n));
                Cl[q * L + n] = v;
            }
        }
        __syncthreads();
        // combine the three q and split the pair; thread t of the line handles n = t, t + 3P, ...
        {
            constexpr T h3 = (T)0.86602540378443864676L;
            const int t = q * P + i;
            for (int n = t; n <= L / 2; n += 3 * P) {
                const cx<T> f0 = Cl[n], g1 = Cl[L + n], g2 = Cl[2 * L + n];
                const cx<T> S = g1 + g2, D = g1 - g2;
                const cx<T> An = f0 + S;
                if (n == 0) {
                    Op[ca * cs] = mk<T>(An.x, 0);
                    Op[cb * cs] = mk<T>(An.y, 0);
                } else {
                    const cx<T> Cn = mk<T>(f0.x - (T)0.5 * S.x - h3 * D.y, f0.y - (T)0.5 * S.y + h3 * D.x);
                    const int m = L - n;
                    const cx<T> f0m = Cl[m], g1m = Cl[L + m], g2m = Cl[2 * L + m];
                    const cx<T> Sm = g1m + g2m, Dm = g1m - g2m;
                    const cx<T> Am = f0m + Sm;
                    const cx<T> Cm = mk<T>(f0m.x - (T)0.5 * Sm.x - h3 * Dm.y, f0m.y - (T)0.5 * Sm.y + h3 * Dm.x);
                    // B_a^[n] = (A_n + conj(C_m))/2 ; B_b^[n] = (A_n - conj(C_m))/(2i)
                    Op[ca * cs + n] = mk<T>((T)0.5 * (An.x + Cm.x), (T)0.5 * (An.y - Cm.y));
                    Op[cb * cs + n] = mk<T>((T)0.5 * (An.y + Cm.y), (T)0.5 * (Cm.x - An.x));
                    if (m != n) {
                        Op[ca * cs + m] = mk<T>((T)0.5 * (Am.x + Cn.x), (T)0.5 * (Am.y - Cn.y));
                        Op[cb * cs + m] = mk<T>((T)0.5 * (Am.y + Cn.y), (T)0.5 * (Cn.x - Am.x));
                    }
                }
            }
        }
        // next pair's first write to E happens after this thread's combine; other threads finished
        // reading E before the second barrier above, and Cmb is rewritten only after the next barrier.
    }
}

}  // namespace ns
