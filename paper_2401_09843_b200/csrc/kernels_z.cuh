// kernels_z.cuh -- mathematics shared by the contiguous-axis (z) kernels: step a3 (pad + inverse c2r +
// products + max|u|) and step a4 (forward r2c + truncate) of SURVEY.md section 8(a); Algorithm 2 steps 2-5
// and Algorithm 3 steps 4-5 of the paper (symmetric flux per PAPER.md:L245).
// The kernels themselves are in kernels_zfused.cuh / kernels_zfused8.cuh (a3 and a4 fused).
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

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* addr, double v) {
    atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

}  // namespace ns
