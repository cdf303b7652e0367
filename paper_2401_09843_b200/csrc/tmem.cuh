// tmem.cuh -- Blackwell tensor memory (TMEM, 256 KB per SM: 128 lanes x 512 columns x 32 bit) used as a
// per-thread scratch pad through tcgen05.st / tcgen05.ld (SASS: STTM / LDTM).  No tensor-core math is
// involved: the fused z kernel parks its physical-space fields there so that neither registers nor shared
// memory (both of which bound its occupancy) have to hold them.  Product path only (sm_100a).
//
// Access shape .32x32b: thread i of a warp touches TMEM lane 32*(warp%4) + i, one 32-bit word per column.
// All calls are warp-collective (.sync.aligned): every lane of the warp must execute them converged.
#pragma once
#include <cstdint>

namespace ns {

// One warp allocates `ncols` columns (power of two >= 32) for the CTA and publishes the base address in *slot.
__device__ __forceinline__ void tmem_alloc(uint32_t* slot_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                     (uint32_t)__cvta_generic_to_shared(slot_smem)),
                 "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
        "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
// load + wait in ONE asm statement: the destination registers are defined when the statement ends, so the
// compiler cannot schedule a use of them ahead of tcgen05.wait::ld
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n\t"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}

// words of TMEM (columns) taken by 16 values of type T
template <typename T> __host__ __device__ constexpr uint32_t tmem_cols16() { return 16 * sizeof(T) / 4; }

// Park / fetch 16 per-thread scalars.  The caller issues tmem_wait_st() before fetching what it parked.
__device__ __forceinline__ void tmem_store16(uint32_t taddr, const double (&d)[16]) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        uint32_t r[16];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            r[2 * k] = (uint32_t)__double2loint(d[8 * h + k]);
            r[2 * k + 1] = (uint32_t)__double2hiint(d[8 * h + k]);
        }
        tmem_st16(taddr + 16 * h, r);
    }
}
__device__ __forceinline__ void tmem_store16(uint32_t taddr, const float (&d)[16]) {
    uint32_t r[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) r[k] = __float_as_uint(d[k]);
    tmem_st16(taddr, r);
}
__device__ __forceinline__ void tmem_load16(uint32_t taddr, double (&d)[16]) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        uint32_t r[16];
        tmem_ld16(taddr + 16 * h, r);
#pragma unroll
        for (int k = 0; k < 8; ++k) d[8 * h + k] = __hiloint2double((int)r[2 * k + 1], (int)r[2 * k]);
    }
}
__device__ __forceinline__ void tmem_load16(uint32_t taddr, float (&d)[16]) {
    uint32_t r[16];
    tmem_ld16(taddr, r);
#pragma unroll
    for (int k = 0; k < 16; ++k) d[k] = __uint_as_float(r[k]);
}

// One x16 access worth of scalars: 8 doubles or 16 floats (callers that must keep register pressure low work chunk by chunk).
template <typename T> __host__ __device__ constexpr int tmem_vals_per_access() { return 64 / (int)sizeof(T); }
__device__ __forceinline__ void tmem_store_vals(uint32_t taddr, const double (&d)[8]) {
    uint32_t r[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        r[2 * k] = (uint32_t)__double2loint(d[k]);
        r[2 * k + 1] = (uint32_t)__double2hiint(d[k]);
    }
    tmem_st16(taddr, r);
}
__device__ __forceinline__ void tmem_store_vals(uint32_t taddr, const float (&d)[16]) { tmem_store16(taddr, d); }
__device__ __forceinline__ void tmem_load_vals(uint32_t taddr, double (&d)[8]) {
    uint32_t r[16];
    tmem_ld16(taddr, r);
#pragma unroll
    for (int k = 0; k < 8; ++k) d[k] = __hiloint2double((int)r[2 * k + 1], (int)r[2 * k]);
}
__device__ __forceinline__ void tmem_load_vals(uint32_t taddr, float (&d)[16]) { tmem_load16(taddr, d); }

// Complex values in chunks of one x16 access: 4 complex doubles or 8 complex floats (re, im interleaved).
template <typename T> __host__ __device__ constexpr int tmem_cx_chunk() { return 16 / (2 * (int)sizeof(T) / 4); }
__device__ __forceinline__ void tmem_store_cx(uint32_t taddr, const double (&re)[4], const double (&im)[4]) {
    uint32_t r[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        r[4 * k] = (uint32_t)__double2loint(re[k]);
        r[4 * k + 1] = (uint32_t)__double2hiint(re[k]);
        r[4 * k + 2] = (uint32_t)__double2loint(im[k]);
        r[4 * k + 3] = (uint32_t)__double2hiint(im[k]);
    }
    tmem_st16(taddr, r);
}
__device__ __forceinline__ void tmem_store_cx(uint32_t taddr, const float (&re)[8], const float (&im)[8]) {
    uint32_t r[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) { r[2 * k] = __float_as_uint(re[k]); r[2 * k + 1] = __float_as_uint(im[k]); }
    tmem_st16(taddr, r);
}
__device__ __forceinline__ void tmem_load_cx(uint32_t taddr, double (&re)[4], double (&im)[4]) {
    uint32_t r[16];
    tmem_ld16(taddr, r);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        re[k] = __hiloint2double((int)r[4 * k + 1], (int)r[4 * k]);
        im[k] = __hiloint2double((int)r[4 * k + 3], (int)r[4 * k + 2]);
    }
}
__device__ __forceinline__ void tmem_load_cx(uint32_t taddr, float (&re)[8], float (&im)[8]) {
    uint32_t r[16];
    tmem_ld16(taddr, r);
#pragma unroll
    for (int k = 0; k < 8; ++k) { re[k] = __uint_as_float(r[2 * k]); im[k] = __uint_as_float(r[2 * k + 1]); }
}

}  // namespace ns
