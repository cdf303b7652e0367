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

// In-place decimation-in-frequency FFT of v[0..R), R in {1,2,4,8,16}, kernel exp(DIR 2 pi i jk/R).
// Output X[k] is left at v[brev<R>(k)].
template <int R, int DIR, typename T>
__device__ __forceinline__ void fft_reg(cx<T>* v) {
    if constexpr (R >= 2) {
        static_assert(R <= 16, "radix up to 16");
        DifButterflies<R, DIR, 0, T>::run(v);
        fft_reg<R / 2, DIR, T>(v);
        fft_reg<R / 2, DIR, T>(v + R / 2);
    }
}

template <int R>
__host__ __device__ __forceinline__ constexpr int brev(int k) {
    int r = 0;
    for (int b = 1; b < R; b <<= 1) {
        r = (r << 1) | (k & 1);
        k >>= 1;
    }
    return r;
}

}  // namespace ns
