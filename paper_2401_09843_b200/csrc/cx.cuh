// cx.cuh -- complex arithmetic and in-register power-of-two FFT butterflies (radix up to 16).
// Part of the CUDA product path (sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace ns {

template <typename T>
struct alignas(2 * sizeof(T)) cx {
    T x, y;
};

template <typename T> __device__ __forceinline__ cx<T> mk(T x, T y) { cx<T> r; r.x = x; r.y = y; return r; }
template <typename T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <typename T> __device__ __forceinline__ cx<T> operator*(T s, cx<T> a) { return mk<T>(s * a.x, s * a.y); }
template <typename T> __device__ __forceinline__ cx<T> conj(cx<T> a) { return mk<T>(a.x, -a.y); }
// a * w
template <typename T> __device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> w) {
    return mk<T>(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
}
// a * conj(w)
template <typename T> __device__ __forceinline__ cx<T> cmulc(cx<T> a, cx<T> w) {
    return mk<T>(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}
// a * w (DIR = +1) or a * conj(w) (DIR = -1): tables hold e^{+i theta}
template <int DIR, typename T> __device__ __forceinline__ cx<T> cmul_dir(cx<T> a, cx<T> w) {
    if constexpr (DIR > 0) return cmul(a, w); else return cmulc(a, w);
}
// i * a, -i * a
template <typename T> __device__ __forceinline__ cx<T> mul_i(cx<T> a) { return mk<T>(-a.y, a.x); }
template <typename T> __device__ __forceinline__ cx<T> mul_mi(cx<T> a) { return mk<T>(a.y, -a.x); }

// Read-only cached load of a complex value (LDG.128 for double, LDG.64 for float).
template <typename T> __device__ __forceinline__ cx<T> ldg(const cx<T>* p);
template <> __device__ __forceinline__ cx<double> ldg<double>(const cx<double>* p) {
    double2 v = __ldg(reinterpret_cast<const double2*>(p));
    return mk<double>(v.x, v.y);
}
template <> __device__ __forceinline__ cx<float> ldg<float>(const cx<float>* p) {
    float2 v = __ldg(reinterpret_cast<const float2*>(p));
    return mk<float>(v.x, v.y);
}

// Cache-policy variants: small tables that every warp re-reads (keep them in L1) and streamed outputs (written once, not
// read again by this kernel: do not let them evict the tables).
template <typename T> __device__ __forceinline__ cx<T> ldg_keep(const cx<T>* p);
template <> __device__ __forceinline__ cx<double> ldg_keep<double>(const cx<double>* p) {
    double x, y;
    asm("ld.global.nc.L1::evict_last.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "l"(p));
    return mk<double>(x, y);
}
template <> __device__ __forceinline__ cx<float> ldg_keep<float>(const cx<float>* p) {
    float x, y;
    asm("ld.global.nc.L1::evict_last.v2.f32 {%0, %1}, [%2];" : "=f"(x), "=f"(y) : "l"(p));
    return mk<float>(x, y);
}
__device__ __forceinline__ void stg_stream(cx<double>* p, cx<double> v) {
    asm volatile("st.global.L1::no_allocate.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void stg_stream(cx<float>* p, cx<float> v) {
    asm volatile("st.global.L1::no_allocate.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y) : "memory");
}

// ------------------------------------------------------------------------------------------------
// d * exp(DIR * 2 pi i * M16 / 16), M16 in [0, 8), with the trivial roots special-cased.
// ------------------------------------------------------------------------------------------------
template <int DIR, int M16, typename T>
__device__ __forceinline__ cx<T> mul_root16(cx<T> d) {
    constexpr T C1 = (T)0.92387953251128675613L;  // cos(pi/8)
    constexpr T S1 = (T)0.38268343236508977173L;  // sin(pi/8)
    constexpr T S2 = (T)0.70710678118654752440L;  // sqrt(1/2)
    if constexpr (M16 == 0) {
        return d;
    } else if constexpr (M16 == 4) {
        if constexpr (DIR > 0) return mul_i(d); else return mul_mi(d);
    } else if constexpr (M16 == 2) {  // (1 + DIR i)/sqrt2
        if constexpr (DIR > 0) return mk<T>(S2 * (d.x - d.y), S2 * (d.x + d.y));
        else return mk<T>(S2 * (d.x + d.y), S2 * (d.y - d.x));
    } else if constexpr (M16 == 6) {  // (-1 + DIR i)/sqrt2
        if constexpr (DIR > 0) return mk<T>(-S2 * (d.x + d.y), S2 * (d.x - d.y));
        else return mk<T>(S2 * (d.y - d.x), -S2 * (d.x + d.y));
    } else {
        constexpr T c = (M16 == 1) ? C1 : (M16 == 3) ? S1 : (M16 == 5) ? -S1 : -C1;
        constexpr T s = (M16 == 1) ? S1 : (M16 == 3) ? C1 : (M16 == 5) ? C1 : S1;
        if constexpr (DIR > 0) return mk<T>(d.x * c - d.y * s, d.x * s + d.y * c);
        else return mk<T>(d.x * c + d.y * s, d.y * c - d.x * s);
    }
}

template <int R, int DIR, int J, typename T>
struct DifButterflies {
    static __device__ __forceinline__ void run(cx<T>* v) {
        constexpr int Hh = R / 2;
        const cx<T> a = v[J], b = v[J + Hh];
        v[J] = a + b;
        v[J + Hh] = mul_root16<DIR, J * (16 / R), T>(a - b);
        if constexpr (J + 1 < Hh) DifButterflies<R, DIR, J + 1, T>::run(v);
    }
};

template <int R>
__host__ __device__ __forceinline__ constexpr int brev(int k) {
    int r = 0;
    for (int b = 1; b < R; b <<= 1) {
        r = (r << 1) | (k & 1);
        k >>= 1;
    }
    return r;
}

// ------------------------------------------------------------------------------------------------
// Radix 16 as 4 x 4 with every twiddle multiplication folded into the additions of the second stage (FMA form):
// 144 fp operations instead of the 168 of four radix-2 levels.  A twiddle w = exp(DIR 2 pi i m/16) is written as
// w = c (p + i q) with p = 1 (|cos| >= |sin|: q = tan) or q = +-1 (p = cot), so that e = (p + i q) d costs two FMAs and
// the scale c rides on the FMAs of the radix-4 butterfly that consumes it.  Same interface as fft_reg<16>.
// ------------------------------------------------------------------------------------------------
template <typename T> struct Tw16 { T p, q, c; };
template <int DIR, int M, typename T>
__host__ __device__ constexpr Tw16<T> tw16_split() {
    // cos, sin of m pi/8
    constexpr double C[16] = {1.0, 0.92387953251128675613, 0.70710678118654752440, 0.38268343236508977173, 0.0,
                                   -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128675613, -1.0,
                                   -0.92387953251128675613, -0.70710678118654752440, -0.38268343236508977173, 0.0,
                                   0.38268343236508977173, 0.70710678118654752440, 0.92387953251128675613};
    constexpr int m = ((M % 16) + 16) % 16;
    const double co = C[m], si = (DIR > 0 ? 1.0 : -1.0) * C[(m + 12) % 16];   // sin(x) = cos(x - pi/2)
    const double aco = co < 0 ? -co : co, asi = si < 0 ? -si : si;
    if (aco >= asi) return Tw16<T>{(T)1, (T)(si / co), (T)co};
    // |sin| > |cos|: w = si (co/si + i)
    return Tw16<T>{(T)(co / si), (T)1, (T)si};
}

// e = (p + i q) d
template <int DIR, int M, typename T>
__device__ __forceinline__ cx<T> tw16_pre(cx<T> d) {
    constexpr Tw16<T> w = tw16_split<DIR, M, T>();
    if constexpr (((M % 16) + 16) % 16 == 0) return d;
    else if constexpr (w.p == (T)0) return mk<T>(-d.y, d.x);                                   // +-i: c carries the sign
    else if constexpr (w.p == (T)1) return mk<T>(d.x - w.q * d.y, d.y + w.q * d.x);
    else return mk<T>(w.p * d.x - d.y, w.p * d.y + d.x);
}

// radix-4 butterfly X_k = sum_n x_n (DIR i)^{nk} of x0, c1 e1, c2 e2, c3 e3; results to o0..o3 (X0..X3)
template <int DIR, typename T>
__device__ __forceinline__ void bf4_scaled(cx<T> x0, cx<T> e1, cx<T> e2, cx<T> e3, T c1, T c2, T r31, cx<T>& o0, cx<T>& o1, cx<T>& o2,
                                           cx<T>& o3) {
    const cx<T> t0 = mk<T>(x0.x + c2 * e2.x, x0.y + c2 * e2.y), t1 = mk<T>(x0.x - c2 * e2.x, x0.y - c2 * e2.y);
    const cx<T> u2 = mk<T>(e1.x + r31 * e3.x, e1.y + r31 * e3.y), u3 = mk<T>(e1.x - r31 * e3.x, e1.y - r31 * e3.y);
    constexpr T s = (T)DIR;
    o0 = mk<T>(t0.x + c1 * u2.x, t0.y + c1 * u2.y);
    o2 = mk<T>(t0.x - c1 * u2.x, t0.y - c1 * u2.y);
    o1 = mk<T>(t1.x - (s * c1) * u3.y, t1.y + (s * c1) * u3.x);
    o3 = mk<T>(t1.x + (s * c1) * u3.y, t1.y - (s * c1) * u3.x);
}
template <int DIR, typename T>
__device__ __forceinline__ void bf4_plain(cx<T> x0, cx<T> x1, cx<T> x2, cx<T> x3, cx<T>& o0, cx<T>& o1, cx<T>& o2, cx<T>& o3) {
    const cx<T> t0 = x0 + x2, t1 = x0 - x2, t2 = x1 + x3, d = x1 - x3;
    const cx<T> t3 = DIR > 0 ? mul_i(d) : mul_mi(d);
    o0 = t0 + t2; o2 = t0 - t2; o1 = t1 + t3; o3 = t1 - t3;
}

template <int DIR, int K1, typename T>
__device__ __forceinline__ void fft16_stage_b(cx<T>* v) {
    // group k1: registers 4 brev2(k1) + n1 hold Y(n1, k1); X[k1 + 4 k2] goes to 4 brev2(k1) + brev2(k2)
    constexpr int B = 4 * brev<4>(K1);
    const cx<T> y0 = v[B], y1 = v[B + 1], y2 = v[B + 2], y3 = v[B + 3];
    if constexpr (K1 == 0) {
        bf4_plain<DIR, T>(y0, y1, y2, y3, v[B], v[B + 2], v[B + 1], v[B + 3]);
    } else {
        constexpr Tw16<T> w1 = tw16_split<DIR, K1, T>(), w2 = tw16_split<DIR, 2 * K1, T>(), w3 = tw16_split<DIR, 3 * K1, T>();
        bf4_scaled<DIR, T>(y0, tw16_pre<DIR, K1, T>(y1), tw16_pre<DIR, 2 * K1, T>(y2), tw16_pre<DIR, 3 * K1, T>(y3), w1.c, w2.c,
                           w3.c / w1.c, v[B], v[B + 2], v[B + 1], v[B + 3]);
    }
}

template <int DIR, typename T>
__device__ __forceinline__ void fft16_fma(cx<T>* v) {
    // stage A: group n1 = registers n1 + 4 n2; Y(n1, k1) goes to register n1 + 4 brev2(k1)
#pragma unroll
    for (int n1 = 0; n1 < 4; ++n1) {
        const cx<T> x0 = v[n1], x1 = v[n1 + 4], x2 = v[n1 + 8], x3 = v[n1 + 12];
        bf4_plain<DIR, T>(x0, x1, x2, x3, v[n1], v[n1 + 8], v[n1 + 4], v[n1 + 12]);
    }
    fft16_stage_b<DIR, 0, T>(v);
    fft16_stage_b<DIR, 1, T>(v);
    fft16_stage_b<DIR, 2, T>(v);
    fft16_stage_b<DIR, 3, T>(v);
}

// radix-3 butterfly X_k = sum_n x_n w3^{DIR nk} in place (12 fp operations)
template <int DIR, typename T>
__device__ __forceinline__ void bf3(cx<T>& x0, cx<T>& x1, cx<T>& x2) {
    constexpr T h = (T)DIR * (T)0.86602540378443864676L;
    const cx<T> s = x1 + x2, d = x1 - x2;
    const cx<T> m = mk<T>(x0.x - (T)0.5 * s.x, x0.y - (T)0.5 * s.y);
    x0 = x0 + s;
    x1 = mk<T>(m.x - h * d.y, m.y + h * d.x);
    x2 = mk<T>(m.x + h * d.y, m.y - h * d.x);
}

// Lengths 6 and 12 by the prime-factor algorithm (3 x 2, 3 x 4: no twiddle factors).  Input index n = (N2 n1 + 3 n2) mod N
// (n1 < 3, n2 < N2), output index k = (N2' k1 + 3' k2) mod N by the Chinese remainder theorem; everything in place, so that
// X[k] ends at register (N2 (k mod 3) + 3 (k mod N2)) mod N.
template <int R, int DIR, typename T>
__device__ __forceinline__ void fft_pfa3(cx<T>* v) {
    constexpr int N2 = R / 3;
    static_assert(R == 6 || R == 12, "3 x 2 or 3 x 4");
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2) bf3<DIR, T>(v[(3 * n2) % R], v[(N2 + 3 * n2) % R], v[(2 * N2 + 3 * n2) % R]);
#pragma unroll
    for (int k1 = 0; k1 < 3; ++k1) {
        if constexpr (N2 == 2) {
            const cx<T> a = v[(N2 * k1) % R], b = v[(N2 * k1 + 3) % R];
            v[(N2 * k1) % R] = a + b;
            v[(N2 * k1 + 3) % R] = a - b;
        } else {
            cx<T>&r0 = v[(N2 * k1) % R], &r1 = v[(N2 * k1 + 3) % R], &r2 = v[(N2 * k1 + 6) % R], &r3 = v[(N2 * k1 + 9) % R];
            const cx<T> x0 = r0, x1 = r1, x2 = r2, x3 = r3;
            bf4_plain<DIR, T>(x0, x1, x2, x3, r0, r1, r2, r3);
        }
    }
}

// In-place FFT of v[0..R), R in {1,2,3,4,6,8,12,16}, kernel exp(DIR 2 pi i jk/R): decimation in frequency for the powers
// of two, prime-factor for 6 and 12.  Output X[k] is left at v[outpos<R>(k)].
template <int R, int DIR, typename T>
__device__ __forceinline__ void fft_reg(cx<T>* v) {
    if constexpr (R == 16) {
        fft16_fma<DIR, T>(v);
    } else if constexpr (R == 3) {
        bf3<DIR, T>(v[0], v[1], v[2]);
    } else if constexpr (R == 6 || R == 12) {
        fft_pfa3<R, DIR, T>(v);
    } else if constexpr (R >= 2) {
        DifButterflies<R, DIR, 0, T>::run(v);
        fft_reg<R / 2, DIR, T>(v);
        fft_reg<R / 2, DIR, T>(v + R / 2);
    }
}
template <int R>
__host__ __device__ __forceinline__ constexpr int outpos(int k) {
    if constexpr (R == 3) return k;
    else if constexpr (R == 6 || R == 12) return ((R / 3) * (k % 3) + 3 * (k % (R / 3))) % R;
    else return brev<R>(k);
}

}  // namespace ns
