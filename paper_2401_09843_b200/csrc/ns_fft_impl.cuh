// ns_fft_impl.cuh -- launch configuration of the FFT kernels, instantiated once per dtype.
#pragma once
#include "kernels_col.cuh"
#include "kernels_colring.cuh"
#include "kernels_z.cuh"
#include "kernels_zfused.cuh"
#include "kernels_zpair.cuh"
#include "kernels_y2d.cuh"
#include "ns_internal.h"
#include <map>
#include <mutex>
#include <utility>

namespace ns {

// Register-stage split L = R1 x R2 per supported half-length.
template <int L> struct Split;
template <> struct Split<8>   { static constexpr int R1 = 4,  R2 = 2;  };
template <> struct Split<16>  { static constexpr int R1 = 4,  R2 = 4;  };
template <> struct Split<32>  { static constexpr int R1 = 8,  R2 = 4;  };
template <> struct Split<64>  { static constexpr int R1 = 8,  R2 = 8;  };
template <> struct Split<128> { static constexpr int R1 = 16, R2 = 8;  };
template <> struct Split<256> { static constexpr int R1 = 16, R2 = 16; };
// N = 3 * 2^a (sizes with small prime factors): L = 3 * 2^(a-1), first stage 6 or 12
template <> struct Split<24>  { static constexpr int R1 = 6,  R2 = 4;  };
template <> struct Split<48>  { static constexpr int R1 = 12, R2 = 4;  };
template <> struct Split<96>  { static constexpr int R1 = 12, R2 = 8;  };
template <> struct Split<192> { static constexpr int R1 = 12, R2 = 16; };
// N = 5 * 2^a, 7 * 2^a, 15 * 2^a (radix-5 / radix-7 butterflies, prime-factor first stages 10, 14, 15, 20)
template <> struct Split<40>  { static constexpr int R1 = 10, R2 = 4;  };
template <> struct Split<80>  { static constexpr int R1 = 10, R2 = 8;  };
template <> struct Split<160> { static constexpr int R1 = 10, R2 = 16; };
template <> struct Split<320> { static constexpr int R1 = 20, R2 = 16; };
template <> struct Split<56>  { static constexpr int R1 = 14, R2 = 4;  };
template <> struct Split<112> { static constexpr int R1 = 14, R2 = 8;  };
template <> struct Split<224> { static constexpr int R1 = 14, R2 = 16; };
template <> struct Split<120> { static constexpr int R1 = 15, R2 = 8;  };
template <> struct Split<240> { static constexpr int R1 = 15, R2 = 16; };

template <int L> struct Cfg {
    static constexpr int R1 = Split<L>::R1, R2 = Split<L>::R2;
    static constexpr int P = R1 > R2 ? R1 : R2;
    // tiles per block for the column kernels: aim at 128 threads
    template <typename T> static constexpr int tpb() {
        constexpr int tt = tile_cols<T>() * P;
        return tt >= 128 ? 1 : 128 / tt;
    }
    // lines per block of the block-synchronous fused z kernel (must divide M^2): about 96-192 threads
    static constexpr int lpbf() {
        if (L % 5 == 0 || L % 7 == 0) return P <= 8 ? 8 : (P <= 14 ? 4 : 2);
        return L == 24 ? 8 : (L % 3 == 0 ? (L >= 192 ? 2 : 4) : 192 / (3 * P));
    }
    // target CTAs per SM of the fused z kernel (bounds its registers)
    static constexpr int minbf() { return (L >= 160 && (L & (L - 1)) != 0) ? 4 : 2; }
};

// Function attributes and occupancy are properties of (kernel, device): they are set / queried once per pair and remembered, not
// on every launch (one RK3 step is 19 launches; at 32^3 the step is launch bound).  Thread safe.
struct KernelSetup {
    size_t smem = 0;      // MaxDynamicSharedMemorySize already granted
    int occ = 0;          // CTAs per SM from the occupancy query (0 = not asked yet)
    bool carveout = false;
};
static std::mutex& kernel_setup_mutex() {
    static std::mutex m;
    return m;
}
static KernelSetup& kernel_setup(const void* fn) {      // call with kernel_setup_mutex() held
    static std::map<std::pair<const void*, int>, KernelSetup> table;
    int dev = 0;
    cudaGetDevice(&dev);
    return table[std::make_pair(fn, dev)];
}
template <typename K>
static cudaError_t set_smem(K kernel, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    std::lock_guard<std::mutex> lock(kernel_setup_mutex());
    KernelSetup& ks = kernel_setup((const void*)kernel);
    if (ks.smem >= bytes) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) ks.smem = bytes;
    return e;
}
template <typename K>
static cudaError_t occupancy(K kernel, int threads, size_t smem, int* occ) {
    std::lock_guard<std::mutex> lock(kernel_setup_mutex());
    KernelSetup& ks = kernel_setup((const void*)kernel);
    if (ks.occ == 0) {
        int o = 0;
        const cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kernel, threads, smem);
        if (e != cudaSuccess) return e;
        ks.occ = o < 1 ? 1 : o;
    }
    *occ = ks.occ;
    return cudaSuccess;
}

template <typename T, int L, bool PF, bool SPLIT = false>
static cudaError_t col_inv_L(cudaStream_t st, const cx<T>* in, cx<T>* out, ColArgs g, Twiddles<T> tw) {
    using C = Cfg<L>;
    constexpr int TC = tile_cols<T>(), TPB = C::template tpb<T>();
    auto k = col_inv_kernel<T, L, C::R1, C::R2, TC, TPB, PF, SPLIT>;
    const size_t smem = (size_t)2 * TPB * L * TC * sizeof(cx<T>);
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    const long blocks = (g.total_tiles + TPB - 1) / TPB;
    k<<<(unsigned)blocks, TC * C::P * TPB, smem, st>>>(in, out, g, tw);
    return cudaGetLastError();
}

template <typename T, int L, bool PF, bool SPLIT = false>
static cudaError_t col_fwd_L(cudaStream_t st, const cx<T>* in, cx<T>* out, ColArgs g, T scale, Twiddles<T> tw) {
    using C = Cfg<L>;
    constexpr int TC = tile_cols<T>(), TPB = C::template tpb<T>();
    auto k = col_fwd_kernel<T, L, C::R1, C::R2, TC, TPB, PF, SPLIT>;
    const size_t smem = (size_t)3 * TPB * L * TC * sizeof(cx<T>);
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    const long blocks = (g.total_tiles + TPB - 1) / TPB;
    k<<<(unsigned)blocks, TC * C::P * TPB, smem, st>>>(in, out, g, scale, tw);
    return cudaGetLastError();
}

// long lines (L = 128, 256): inverse pass with its inputs parked in tensor memory
template <typename T, int L, bool PF, bool SPLIT = false>
static cudaError_t col_inv_tmem_L(cudaStream_t st, const cx<T>* in, cx<T>* out, ColArgs g, Twiddles<T> tw) {
    constexpr int TC = tile_cols<T>(), R2 = L / 16;
    constexpr int MINB = sizeof(T) == 8 ? 3 : 2;
    auto k = col_inv_tmem_kernel<T, L, R2, TC, MINB, PF, SPLIT>;
    const size_t smem = (size_t)2 * L * TC * sizeof(cx<T>);
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    k<<<(unsigned)g.total_tiles, TC * 16, smem, st>>>(in, out, g, tw);
    return cudaGetLastError();
}

// long lines (L = 128, 256): forward pass with F_0 / G_1 parked in tensor memory
template <typename T, int L, bool PF, bool SPLIT = false>
static cudaError_t col_fwd_tmem_L(cudaStream_t st, const cx<T>* in, cx<T>* out, ColArgs g, T scale, Twiddles<T> tw) {
    constexpr int TC = tile_cols<T>(), R2 = L / 16;
    constexpr int MINB = sizeof(T) == 8 ? 3 : 2;
    auto k = col_fwd_tmem_kernel<T, L, R2, TC, MINB, PF, SPLIT>;
    const size_t smem = (size_t)2 * L * TC * sizeof(cx<T>);
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    k<<<(unsigned)g.total_tiles, TC * 16, smem, st>>>(in, out, g, scale, tw);
    return cudaGetLastError();
}

// ---- persistent TMA-fed forward column kernel (kernels_colring.cuh), L = 256
// cuTensorMapEncodeTiled through the runtime's driver entry point (no link dependency on libcuda)
typedef CUresult (*ns_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static ns_encode_tiled_fn ns_encode_tiled() {
    static ns_encode_tiled_fn fn = nullptr;     // device independent; benign if two threads resolve it at once
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (ns_encode_tiled_fn)p;
    }
    return fn;
}
// 3-D tensor (2 * ncols scalars, rows, slabs) over the input of a column pass; box = one column tile x L rows
template <typename T>
static cudaError_t col_tensor_map(CUtensorMap* m, const cx<T>* in, long ncols, long rows, const ColArgs& g, int L) {
    ns_encode_tiled_fn enc = ns_encode_tiled();
    if (!enc) return cudaErrorNotSupported;
    const long nslabs = g.total_tiles / g.tiles_per_slab;
    const cuuint64_t dims[3] = {(cuuint64_t)(2 * ncols), (cuuint64_t)rows, (cuuint64_t)nslabs};
    const cuuint64_t strides[2] = {(cuuint64_t)g.istride * sizeof(cx<T>), (cuuint64_t)g.in_slab * sizeof(cx<T>)};
    const cuuint32_t box[3] = {(cuuint32_t)(2 * tile_cols<T>()), (cuuint32_t)L, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(m, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)in, dims, strides,
                           box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}
// stages of the input ring / CTAs per SM: L = 256: 2 x 96 KB, one CTA of 13 (fp64) / 25 (fp32) warps per SM
template <int L> struct RingCfg { static constexpr int STAGES = 2, MINB = 1; };

template <typename T, int L, bool SPLIT = false>
static cudaError_t col_fwd_ring_L(cudaStream_t st, int num_sms, const cx<T>* in, cx<T>* out, long ncols, ColArgs g, T scale, Twiddles<T> tw) {
    using C = Cfg<L>;
    constexpr int TC = tile_cols<T>(), STAGES = RingCfg<L>::STAGES;
    using Geo = ColRingGeo<T, L, C::R1, C::R2, TC, STAGES>;
    auto k = col_fwd_ring_kernel<T, L, C::R1, C::R2, TC, STAGES, RingCfg<L>::MINB, SPLIT>;
    CUtensorMap m;
    cudaError_t e = col_tensor_map<T>(&m, in, ncols, 3 * L, g, L);
    if (e != cudaSuccess) return e;
    if ((e = set_smem(k, Geo::FWD_BYTES)) != cudaSuccess) return e;
    int occ = 0;
    if ((e = occupancy(k, Geo::NT, Geo::FWD_BYTES, &occ)) != cudaSuccess) return e;
    long grid = (long)num_sms * (occ < 1 ? 1 : occ);
    if (grid > g.total_tiles) grid = g.total_tiles;
    k<<<(unsigned)grid, Geo::NT, Geo::FWD_BYTES, st>>>(m, out, g, scale, tw);
    return cudaGetLastError();
}
template <typename T, int L>
static cudaError_t z_fused_L(cudaStream_t st, int num_sms, const cx<T>* in, cx<T>* out, long MM, long batch, unsigned long long* umax2,
                             Twiddles<T> tw) {
    using C = Cfg<L>;
    constexpr int LPB = C::lpbf();
    auto k = z_fused_kernel<T, L, C::R1, C::R2, LPB, C::minbf()>;
    const size_t smem = (size_t)LPB * (3 * L + 3 * C::R1 * (C::R2 + 1)) * sizeof(cx<T>) + 16;
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    {
        std::lock_guard<std::mutex> lock(kernel_setup_mutex());
        KernelSetup& ks = kernel_setup((const void*)k);
        if (!ks.carveout) {
            e = cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
            if (e != cudaSuccess) return e;
            ks.carveout = true;
        }
    }
    if ((MM % LPB) != 0) return cudaErrorInvalidValue;
    const long tiles = MM * batch / LPB;
    int occ = 0;
    e = occupancy(k, 3 * C::P * LPB, smem, &occ);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    long grid = (long)num_sms * occ;
    if (grid > tiles) grid = tiles;
    k<<<(unsigned)grid, 3 * C::P * LPB, smem, st>>>(in, out, MM, tiles, umax2, tw);
    return cudaGetLastError();
}

// line-pair fused z kernel (kernels_zpair.cuh), L in {64, 128, 256}: one persistent block of UNITS units per SM slot
template <typename T, int L>
static cudaError_t z_pair_L(cudaStream_t st, int num_sms, const cx<T>* in, cx<T>* out, long MM, long batch, unsigned long long* umax2,
                            Twiddles<T> tw) {
    using Geo = ZPGeo<T, L>;
    constexpr int UNITS = 4;
    auto k = z_pair_kernel<T, L, UNITS>;
    const size_t smem = (size_t)UNITS * Geo::UNIT_BYTES;
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    if ((MM % 2) != 0 || ((MM / 2) % Geo::PL) != 0) return cudaErrorInvalidValue;
    const long pairs = MM * batch / 2;
    if (MM * batch >= (1L << 31)) return cudaErrorInvalidValue;   // line indices are 32 bit in the kernel
    const long per_block = (long)UNITS * Geo::PL;
    long grid = num_sms;   // one block per SM: registers (384 threads x 168), shared memory and 512 TMEM columns all say so
    const long need = (pairs + per_block - 1) / per_block;
    if (grid > need) grid = need;
    k<<<(unsigned)grid, 96 * UNITS, smem, st>>>(in, out, (unsigned)MM, (unsigned)pairs, umax2, tw);
    return cudaGetLastError();
}

// Two kernel families, compiled in separate translation units (ns_fft_*.cu define NS_FAMILY_SMOOTH or not):
//   pow2    L = 2^a, 8..256: column kernels (+ tensor-memory variants), line-pair z kernel for L >= 64, y2d kernel
//   smooth  L = 3, 5, 7 or 15 times 2^a: column kernels + block-synchronous z kernel
#ifdef NS_FAMILY_SMOOTH
#define NS_FAM(x) x##_smooth
#define NS_DISPATCH_L(L, CALL)                                   \
    switch (L) {                                                 \
        case 24: return CALL(24);                                \
        case 48: return CALL(48);                                \
        case 96: return CALL(96);                                \
        case 192: return CALL(192);                              \
        case 40: return CALL(40);                                \
        case 80: return CALL(80);                                \
        case 160: return CALL(160);                              \
        case 320: return CALL(320);                              \
        case 56: return CALL(56);                                \
        case 112: return CALL(112);                              \
        case 224: return CALL(224);                              \
        case 120: return CALL(120);                              \
        case 240: return CALL(240);                              \
        default: return cudaErrorInvalidValue;                   \
    }
#else
#define NS_FAM(x) x##_pow2
#define NS_DISPATCH_L(L, CALL)                                   \
    switch (L) {                                                 \
        case 8: return CALL(8);                                  \
        case 16: return CALL(16);                                \
        case 32: return CALL(32);                                \
        case 64: return CALL(64);                                \
        case 128: return CALL(128);                              \
        case 256: return CALL(256);                              \
        default: return cudaErrorInvalidValue;                   \
    }
#endif

// L2 prefetch distance of the column passes in tiles (kernels_col.cuh): the CTAs resident on the GPU (2-3 per SM)
static int col_pf_dist(int num_sms, int L) {
    return (L <= 64 ? 2 : 1) * num_sms;
}
// which passes prefetch: measured per length: it pays up to L = 128; at L = 256 only for the inverse
// pass along y (a2 2.13 -> 1.93 ms at 512^3) -- along x every row of a tile lies in another 2 MB page and the extra requests lose
static bool col_pf_on(bool fwd, int L, long row_stride_bytes) {
    if (L <= 128) return true;
    return !fwd && L == 256 && row_stride_bytes < (1L << 16);
}

template <typename T>
static ColArgs make_col_args(long ncols, long nslabs, long istride, long ostride, long in_slab, long out_slab, int pf_dist,
                             const ColSplit* split) {
    ColArgs g;
    g.split_rows = split ? split->rows : 0;
    g.peer = split ? split->peer : nullptr;
    g.istride = istride;
    g.ostride = ostride;
    g.in_slab = in_slab;
    g.out_slab = out_slab;
    g.tiles_per_slab = (int)(ncols / tile_cols<T>());
    g.total_tiles = (long)g.tiles_per_slab * nslabs;
    g.pf_dist = pf_dist;
    return g;
}

template <typename T>
cudaError_t NS_FAM(launch_col_inv)(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, Twiddles<T> tw, const ColSplit* split) {
    if (ncols % tile_cols<T>() != 0) return cudaErrorInvalidValue;
    const ColArgs g = make_col_args<T>(ncols, nslabs, istride, ostride, in_slab, out_slab, col_pf_dist(num_sms, L), split);
    // measured (profiles/): parking pays at L = 128 (0.264 -> 0.216 ms at 256^3); at L = 256 the register kernel is faster
    const bool pf = col_pf_on(false, L, istride * (long)sizeof(cx<T>));
    if (split) {      // multi-device solver: output rows stored to their owners (no L2 prefetch variant)
#ifndef NS_FAMILY_SMOOTH
        if (L == 128) return col_inv_tmem_L<T, 128, false, true>(st, in, out, g, tw);
#endif
#define CALL(LL) col_inv_L<T, LL, false, true>(st, in, out, g, tw)
        NS_DISPATCH_L(L, CALL)
#undef CALL
    }
#ifndef NS_FAMILY_SMOOTH
    if (L == 128) return pf ? col_inv_tmem_L<T, 128, true>(st, in, out, g, tw) : col_inv_tmem_L<T, 128, false>(st, in, out, g, tw);
#endif
#define CALL(LL) (pf ? col_inv_L<T, LL, true>(st, in, out, g, tw) : col_inv_L<T, LL, false>(st, in, out, g, tw))
    NS_DISPATCH_L(L, CALL)
#undef CALL
}

template <typename T>
cudaError_t NS_FAM(launch_col_fwd)(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, T scale, Twiddles<T> tw, const ColSplit* split) {
    if (ncols % tile_cols<T>() != 0) return cudaErrorInvalidValue;
    const ColArgs g = make_col_args<T>(ncols, nslabs, istride, ostride, in_slab, out_slab, col_pf_dist(num_sms, L), split);
    const bool pf = col_pf_on(true, L, istride * (long)sizeof(cx<T>));
    if (split) {      // multi-device solver: output rows stored to their owners
#ifndef NS_FAMILY_SMOOTH
        if (L == 256) return col_fwd_ring_L<T, 256, true>(st, num_sms, in, out, ncols, g, scale, tw);
        if (L == 128) return col_fwd_tmem_L<T, 128, false, true>(st, in, out, g, scale, tw);
#endif
#define CALL(LL) col_fwd_L<T, LL, false, true>(st, in, out, g, scale, tw)
        NS_DISPATCH_L(L, CALL)
#undef CALL
    }
#ifndef NS_FAMILY_SMOOTH
    // long lines: the persistent TMA-fed kernel (measured at 512^3: fp64 a5 3.65 -> 3.20 ms, a6 2.67 -> 2.52 ms; fp32 1.96 -> 1.84, 1.40 -> 1.24)
    if (L == 256) return col_fwd_ring_L<T, 256>(st, num_sms, in, out, ncols, g, scale, tw);
    if (L == 128) return pf ? col_fwd_tmem_L<T, 128, true>(st, in, out, g, scale, tw) : col_fwd_tmem_L<T, 128, false>(st, in, out, g, scale, tw);
#endif
#define CALL(LL) (pf ? col_fwd_L<T, LL, true>(st, in, out, g, scale, tw) : col_fwd_L<T, LL, false>(st, in, out, g, scale, tw))
    NS_DISPATCH_L(L, CALL)
#undef CALL
}

template <typename T>
cudaError_t NS_FAM(launch_z_fused)(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long MM, long batch,
                                   unsigned long long* umax2, Twiddles<T> tw) {
#ifdef NS_FAMILY_SMOOTH
    // N = 3, 5, 7, 15 times 2^a: the block-synchronous kernel with a prime-factor first stage
#define CALL(LL) z_fused_L<T, LL>(st, num_sms, in, out, MM, batch, umax2, tw)
    NS_DISPATCH_L(L, CALL)
#undef CALL
#else
    switch (L) {
        case 256: return z_pair_L<T, 256>(st, num_sms, in, out, MM, batch, umax2, tw);
        case 128: return z_pair_L<T, 128>(st, num_sms, in, out, MM, batch, umax2, tw);
        case 64: return z_pair_L<T, 64>(st, num_sms, in, out, MM, batch, umax2, tw);
        // short lines: block-synchronous kernel
        case 8: return z_fused_L<T, 8>(st, num_sms, in, out, MM, batch, umax2, tw);
        case 16: return z_fused_L<T, 16>(st, num_sms, in, out, MM, batch, umax2, tw);
        case 32: return z_fused_L<T, 32>(st, num_sms, in, out, MM, batch, umax2, tw);
        default: return cudaErrorInvalidValue;
    }
#endif
}

#ifndef NS_FAMILY_SMOOTH
template <typename T, int L>
static cudaError_t y2d_L(cudaStream_t st, int num_sms, const cx<T>* in, cx<T>* out, long M, long batch, unsigned long long* umax2,
                         Twiddles<T> tw) {
    using Geo = ZPGeo<T, L>;
    constexpr int UNITS = 4;
    auto k = y2d_kernel<T, L, UNITS>;
    const size_t smem = (size_t)UNITS * Geo::UNIT_BYTES;
    cudaError_t e = set_smem(k, smem);
    if (e != cudaSuccess) return e;
    if ((M % Geo::PL) != 0 || M * batch >= (1L << 31)) return cudaErrorInvalidValue;
    const long lines = M * batch, per_block = (long)UNITS * Geo::PL;
    long grid = num_sms;
    const long need = (lines + per_block - 1) / per_block;
    if (grid > need) grid = need;
    k<<<(unsigned)grid, 96 * UNITS, smem, st>>>(in, out, (unsigned)M, (unsigned)lines, umax2, tw);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_y2d(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long M, long batch,
                       unsigned long long* umax2, Twiddles<T> tw) {
    switch (L) {
        case 64: return y2d_L<T, 64>(st, num_sms, in, out, M, batch, umax2, tw);
        case 128: return y2d_L<T, 128>(st, num_sms, in, out, M, batch, umax2, tw);
        case 256: return y2d_L<T, 256>(st, num_sms, in, out, M, batch, umax2, tw);
        default: return cudaErrorInvalidValue;
    }
}

// the public launchers route by family (defined once, in the pow2 translation unit)
template <typename T>
cudaError_t launch_col_inv(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, Twiddles<T> tw, const ColSplit* split) {
    if ((L & (L - 1)) == 0) return launch_col_inv_pow2<T>(st, num_sms, L, in, out, ncols, nslabs, istride, ostride, in_slab, out_slab, tw, split);
    return launch_col_inv_smooth<T>(st, num_sms, L, in, out, ncols, nslabs, istride, ostride, in_slab, out_slab, tw, split);
}
template <typename T>
cudaError_t launch_col_fwd(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, T scale, Twiddles<T> tw, const ColSplit* split) {
    if ((L & (L - 1)) == 0) return launch_col_fwd_pow2<T>(st, num_sms, L, in, out, ncols, nslabs, istride, ostride, in_slab, out_slab, scale, tw, split);
    return launch_col_fwd_smooth<T>(st, num_sms, L, in, out, ncols, nslabs, istride, ostride, in_slab, out_slab, scale, tw, split);
}
template <typename T>
cudaError_t launch_z_fused(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long MM, long batch,
                           unsigned long long* umax2, Twiddles<T> tw) {
    if ((L & (L - 1)) == 0) return launch_z_fused_pow2<T>(st, num_sms, L, in, out, MM, batch, umax2, tw);
    return launch_z_fused_smooth<T>(st, num_sms, L, in, out, MM, batch, umax2, tw);
}
#endif  // !NS_FAMILY_SMOOTH

#define NS_FFT_ARGS_COL(T) cudaStream_t, int, int, const cx<T>*, cx<T>*, long, long, long, long, long, long
#define NS_FFT_ARGS_Z(T) cudaStream_t, int, int, const cx<T>*, cx<T>*, long, long, unsigned long long*, Twiddles<T>
#ifdef NS_FAMILY_SMOOTH
#define NS_INSTANTIATE_FFT(T)                                                                   \
    template cudaError_t launch_col_inv_smooth<T>(NS_FFT_ARGS_COL(T), Twiddles<T>, const ColSplit*);             \
    template cudaError_t launch_col_fwd_smooth<T>(NS_FFT_ARGS_COL(T), T, Twiddles<T>, const ColSplit*);          \
    template cudaError_t launch_z_fused_smooth<T>(NS_FFT_ARGS_Z(T));
#else
#define NS_INSTANTIATE_FFT(T)                                                                   \
    template cudaError_t launch_col_inv_pow2<T>(NS_FFT_ARGS_COL(T), Twiddles<T>, const ColSplit*);               \
    template cudaError_t launch_col_fwd_pow2<T>(NS_FFT_ARGS_COL(T), T, Twiddles<T>, const ColSplit*);            \
    template cudaError_t launch_z_fused_pow2<T>(NS_FFT_ARGS_Z(T));                              \
    template cudaError_t launch_col_inv<T>(NS_FFT_ARGS_COL(T), Twiddles<T>, const ColSplit*);                    \
    template cudaError_t launch_col_fwd<T>(NS_FFT_ARGS_COL(T), T, Twiddles<T>, const ColSplit*);                 \
    template cudaError_t launch_z_fused<T>(NS_FFT_ARGS_Z(T));                                   \
    template cudaError_t launch_y2d<T>(NS_FFT_ARGS_Z(T));
#endif

}  // namespace ns
