// kernels_z.cuh -- mathematics shared by the contiguous-axis (z) kernels: step a3 (pad + inverse c2r +
// products + max|u|) and step a4 (forward r2c + truncate) of SURVEY.md section 8(a); Algorithm 2 steps 2-5
// and Algorithm 3 steps 4-5 of the paper (symmetric flux per PAPER.md:L245).
// The kernels themselves are in kernels_zfused.cuh / kernels_zpair.cuh (a3 and a4 fused).
//
// Real transforms use the two-for-one trick on the same pruned radix-3 core as kernels_col.cuh:
//   inverse  z = u_a + i u_b  has spectrum Z[k] = U_a[k] + i U_b[k]; for k < 0, U[k] = conj(U[-k]), so
//            a_n = U_a[n] + i U_b[n],  c_n = conj(U_a[L-n]) + i conj(U_b[L-n])  (n >= 1), c_0 = 0,
//            and a_0 uses only the real parts of U[0] (the c2r definition: u is the real part).
//   forward  z = B_a + i B_b;  B_a^[n] = (A_n + conj(C_{L-n}))/2,  B_b^[n] = (A_n - conj(C_{L-n}))/(2i).
// The physical z axis is stored in the decimated order pz = q*L + r (physical index 3r + q).
//
//
// Flux components.  The path transforms the FIVE trace-free combinations
//   T11 = u1^2 - u3^2,  T12 = u1 u2,  T13 = u1 u3,  T22 = u2^2 - u3^2,  T23 = u2 u3     (T33 = 0)
// instead of the six products of PAPER.md:L245: B_ij - T_ij = delta_ij u3^2 contributes the pure gradient
// -i k (u3^2)^ to the divergence, which the Leray projection of eq. (2.5) annihilates, so the right-hand
// side is the same to round-off (reading A13).  Stored order: 11 12 13 22 23;
// forward pairs (two-for-one): (T11,T22) (T12,T13) (T23,-).
#pragma once
#include "cx.cuh"
#include "ns_internal.h"

namespace ns {

template <int R1, int R2> struct ZP { static constexpr int value = R1 > R2 ? R1 : R2; };

// Running maximum of |u|^2 that PROPAGATES non-finite values (fmax would drop a NaN): for x >= +0 the IEEE bit patterns
// order like the values, +inf sorts above every finite value and every NaN above +inf, so an unsigned integer maximum of
// the bits keeps them.  umax2[b] holds the bits of a double; cfl_finalize / umax_read turn a non-finite maximum into a
// failed sample (NS_ERR_NONFINITE) instead of a silent dt.
__device__ __forceinline__ unsigned long long sq_bits(double v) { return (unsigned long long)__double_as_longlong(v); }
__device__ __forceinline__ unsigned int sq_bits(float v) { return __float_as_uint(v); }
template <typename U> __device__ __forceinline__ U umax_bits(U a, U b) { return a > b ? a : b; }
__device__ __forceinline__ unsigned long long warp_max_bits(unsigned long long m) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = umax_bits(m, __shfl_xor_sync(0xffffffffu, m, o));
    return m;
}
__device__ __forceinline__ unsigned int warp_max_bits(unsigned int m) { return __reduce_max_sync(0xffffffffu, m); }
__device__ __forceinline__ void atomic_max_sq(unsigned long long* addr, unsigned long long m) { atomicMax(addr, m); }
__device__ __forceinline__ void atomic_max_sq(unsigned long long* addr, unsigned int m) {
    atomicMax(addr, (unsigned long long)__double_as_longlong((double)__uint_as_float(m)));   // float -> double keeps inf / NaN
}

// 3 -> 2 radix-3 combine + Hermitian split of one forward pair (see kernels_z.cuh):
// reads F_q[n] W^{-qn} of the three sub-transforms from Sl (regions SZ apart), writes B_a^[n], B_b^[n] for
// n and L - n.  One call covers n = tl, tl + TPL, ... <= L/2 with all loads issued first.
template <typename T, int L, int SZ, int TPL>
__device__ __forceinline__ void z_combine_store(const cx<T>* __restrict__ Sl, cx<T>* __restrict__ Oa, cx<T>* __restrict__ Ob,
                                                bool two, int tl) {
    constexpr int NIT = (L / 2 + TPL) / TPL;  // iterations covering n in [0, L/2]
    constexpr T h3 = (T)0.86602540378443864676L;
    cx<T> f0[NIT], g1[NIT], g2[NIT], f0m[NIT], g1m[NIT], g2m[NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        int n = tl + it * TPL;
        if (n > L / 2) n = L / 2;             // clamped duplicate, not stored
        const int m = n == 0 ? 0 : L - n;
        f0[it] = Sl[n]; g1[it] = Sl[SZ + n]; g2[it] = Sl[2 * SZ + n];
        f0m[it] = Sl[m]; g1m[it] = Sl[SZ + m]; g2m[it] = Sl[2 * SZ + m];
    }
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int n = tl + it * TPL;
        const cx<T> Sn = g1[it] + g2[it], Dn = g1[it] - g2[it];
        const cx<T> An = f0[it] + Sn;
        const cx<T> Cn = mk<T>(f0[it].x - (T)0.5 * Sn.x - h3 * Dn.y, f0[it].y - (T)0.5 * Sn.y + h3 * Dn.x);
        const cx<T> Sm = g1m[it] + g2m[it], Dm = g1m[it] - g2m[it];
        const cx<T> Am = f0m[it] + Sm;
        const cx<T> Cm = mk<T>(f0m[it].x - (T)0.5 * Sm.x - h3 * Dm.y, f0m[it].y - (T)0.5 * Sm.y + h3 * Dm.x);
        if (n <= L / 2) {
            if (n == 0) {
                Oa[0] = mk<T>(An.x, 0);
                if (two) Ob[0] = mk<T>(An.y, 0);
            } else {
                const int m = L - n;
                Oa[n] = mk<T>((T)0.5 * (An.x + Cm.x), (T)0.5 * (An.y - Cm.y));
                if (two) Ob[n] = mk<T>((T)0.5 * (An.y + Cm.y), (T)0.5 * (Cm.x - An.x));
                if (m != n) {
                    Oa[m] = mk<T>((T)0.5 * (Am.x + Cn.x), (T)0.5 * (Am.y - Cn.y));
                    if (two) Ob[m] = mk<T>((T)0.5 * (Am.y + Cn.y), (T)0.5 * (Cn.x - Am.x));
                }
            }
        }
    }
}

}  // namespace ns
