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

// ------------------------------------------------------------------------------------------------
// Odd prime radices 3, 5, 7 (sizes 2^a 3^b 5^c 7^d) and the composite register
// lengths built from them by the prime-factor algorithm (no twiddle factors between coprime factors).
// ------------------------------------------------------------------------------------------------
// cos / sin of 2 pi m / P, P in {3, 5, 7}
template <int P> __host__ __device__ constexpr double root_cos(int m) {
    constexpr double c3[3] = {1.0, -0.5, -0.5};
    constexpr double c5[5] = {1.0, 0.30901699437494742410, -0.80901699437494742410, -0.80901699437494742410, 0.30901699437494742410};
    constexpr double c7[7] = {1.0, 0.62348980185873353053, -0.22252093395631440429, -0.90096886790241912624,
                              -0.90096886790241912624, -0.22252093395631440429, 0.62348980185873353053};
    static_assert(P == 3 || P == 5 || P == 7, "prime radix");
    return P == 3 ? c3[m % 3] : (P == 5 ? c5[m % 5] : c7[m % 7]);
}
template <int P> __host__ __device__ constexpr double root_sin(int m) {
    constexpr double s3[3] = {0.0, 0.86602540378443864676, -0.86602540378443864676};
    constexpr double s5[5] = {0.0, 0.95105651629515357212, 0.58778525229247312917, -0.58778525229247312917, -0.95105651629515357212};
    constexpr double s7[7] = {0.0, 0.78183148246802980871, 0.97492791218182360702, 0.43388373911755812048,
                              -0.43388373911755812048, -0.97492791218182360702, -0.78183148246802980871};
    return P == 3 ? s3[m % 3] : (P == 5 ? s5[m % 5] : s7[m % 7]);
}

// P-point DFT X_k = sum_n x_n exp(DIR 2 pi i nk/P), P an odd prime, on the registers v[(OFF + STR n) % MOD], in place and in
// natural order: pairs (x_j, x_{P-j}) give X_k and X_{P-k} from the same cosine sum m and sine sum s, X = m +- i DIR s.
template <int P, int DIR, int OFF, int STR, int MOD, typename T>
__device__ __forceinline__ void bf_prime(cx<T>* v) {
    constexpr int Hh = (P - 1) / 2;
    auto at = [](int n) { return (OFF + STR * n) % MOD; };
    const cx<T> x0 = v[at(0)];
    cx<T> t[Hh], d[Hh];
#pragma unroll
    for (int j = 1; j <= Hh; ++j) {
        t[j - 1] = v[at(j)] + v[at(P - j)];
        d[j - 1] = v[at(j)] - v[at(P - j)];
    }
    cx<T> sum = x0;
#pragma unroll
    for (int j = 0; j < Hh; ++j) sum = sum + t[j];
    v[at(0)] = sum;
#pragma unroll
    for (int k = 1; k <= Hh; ++k) {
        cx<T> m = x0, s = mk<T>(0, 0);
#pragma unroll
        for (int j = 1; j <= Hh; ++j) {
            const T co = (T)root_cos<P>(j * k), si = (T)root_sin<P>(j * k);
            m = mk<T>(m.x + co * t[j - 1].x, m.y + co * t[j - 1].y);
            s = mk<T>(s.x + si * d[j - 1].x, s.y + si * d[j - 1].y);
        }
        v[at(k)] = mk<T>(m.x - (T)DIR * s.y, m.y + (T)DIR * s.x);
        v[at(P - k)] = mk<T>(m.x + (T)DIR * s.y, m.y - (T)DIR * s.x);
    }
}

// Length R = P x Q by the prime-factor algorithm, P in {3, 5, 7}, Q in {2, 4} or another of those primes (gcd(P, Q) = 1).
// Input index n = (Q n1 + P n2) mod R (n1 < P, n2 < Q), output index k with k = k1 mod P, k = k2 mod Q (Chinese remainder
// theorem); everything in place, so that X[k] ends at register (Q (k mod P) + P (k mod Q)) mod R.
template <int P, int Q, int DIR, typename T, int N2 = 0>
__device__ __forceinline__ void fft_pfa_stage1(cx<T>* v) {
    if constexpr (N2 < Q) {
        bf_prime<P, DIR, (P * N2) % (P * Q), Q, P * Q, T>(v);
        fft_pfa_stage1<P, Q, DIR, T, N2 + 1>(v);
    }
}
template <int P, int Q, int DIR, typename T, int K1 = 0>
__device__ __forceinline__ void fft_pfa_stage2(cx<T>* v) {
    constexpr int R = P * Q;
    if constexpr (K1 < P) {
        if constexpr (Q == 2) {
            const cx<T> a = v[(Q * K1) % R], b = v[(Q * K1 + P) % R];
            v[(Q * K1) % R] = a + b;
            v[(Q * K1 + P) % R] = a - b;
        } else if constexpr (Q == 4) {
            cx<T>&r0 = v[(Q * K1) % R], &r1 = v[(Q * K1 + P) % R], &r2 = v[(Q * K1 + 2 * P) % R], &r3 = v[(Q * K1 + 3 * P) % R];
            const cx<T> x0 = r0, x1 = r1, x2 = r2, x3 = r3;
            bf4_plain<DIR, T>(x0, x1, x2, x3, r0, r1, r2, r3);
        } else {
            bf_prime<Q, DIR, (Q * K1) % R, P, R, T>(v);
        }
        fft_pfa_stage2<P, Q, DIR, T, K1 + 1>(v);
    }
}

// register lengths with a prime-factor decomposition P x Q (P odd prime first); 0 = none
template <int R> struct Pfa { static constexpr int P = 0, Q = 0; };
template <> struct Pfa<6>  { static constexpr int P = 3, Q = 2; };
template <> struct Pfa<12> { static constexpr int P = 3, Q = 4; };
template <> struct Pfa<10> { static constexpr int P = 5, Q = 2; };
template <> struct Pfa<20> { static constexpr int P = 5, Q = 4; };
template <> struct Pfa<14> { static constexpr int P = 7, Q = 2; };
template <> struct Pfa<28> { static constexpr int P = 7, Q = 4; };
template <> struct Pfa<15> { static constexpr int P = 3, Q = 5; };
template <> struct Pfa<21> { static constexpr int P = 3, Q = 7; };

// In-place FFT of v[0..R), kernel exp(DIR 2 pi i jk/R): decimation in frequency for R = 2^a <= 16, one butterfly for the primes
// 3, 5, 7, prime-factor for 6, 10, 12, 14, 15, 20, 21, 28.  Output X[k] is left at v[outpos<R>(k)].
template <int R, int DIR, typename T>
__device__ __forceinline__ void fft_reg(cx<T>* v) {
    if constexpr (R == 16) {
        fft16_fma<DIR, T>(v);
    } else if constexpr (R == 3) {
        bf3<DIR, T>(v[0], v[1], v[2]);
    } else if constexpr (R == 5 || R == 7) {
        bf_prime<R, DIR, 0, 1, R, T>(v);
    } else if constexpr (Pfa<R>::P != 0) {
        fft_pfa_stage1<Pfa<R>::P, Pfa<R>::Q, DIR, T>(v);
        fft_pfa_stage2<Pfa<R>::P, Pfa<R>::Q, DIR, T>(v);
    } else if constexpr (R >= 2) {
        static_assert((R & (R - 1)) == 0, "unsupported register length");
        DifButterflies<R, DIR, 0, T>::run(v);
        fft_reg<R / 2, DIR, T>(v);
        fft_reg<R / 2, DIR, T>(v + R / 2);
    }
}
template <int R>
__host__ __device__ __forceinline__ constexpr int outpos(int k) {
    if constexpr (R == 3 || R == 5 || R == 7) return k;
    else if constexpr (Pfa<R>::P != 0) return (Pfa<R>::Q * (k % Pfa<R>::P) + Pfa<R>::P * (k % Pfa<R>::Q)) % R;
    else return brev<R>(k);
}

}  // namespace ns
