// kernels_zpair.cuh -- steps a3 + a4 of SURVEY.md section 8(a) in ONE kernel for L = N/2 in {64, 128, 256}: per (px,py) line,
// pad + inverse c2r along z, the trace-free flux products, max|u|^2, forward r2c + truncate (Algorithm 2 steps 1-5,
// PAPER.md:L132-135; symmetric flux PAPER.md:L245).  The M^3 physical arrays never touch HBM.
//
// Mathematics as in kernels_z.cuh (pruned radix-3 + two-for-one real transforms).  What this kernel adds:
//
//  * LINE PAIRS.  A line needs 3 real inverse transforms (u1, u2, u3) and 5 real forward ones (T11, T12, T13, T22, T23);
//    done line by line, two-for-one leaves u3 and T23 alone in a complex transform whose imaginary half is zero.  Here a
//    lane group owns TWO neighbouring lines A, B and runs 8 complex transforms for them,
//        job 0  inverse (u3A, u3B)        job 4  inverse (u1B, u2B)
//        job 1  inverse (u1A, u2A)        job 5  forward (T11B, T22B)
//        job 2  forward (T11A, T22A)      job 6  forward (T12B, T13B)
//        job 3  forward (T12A, T13A)      job 7  forward (T23A, T23B)
//    i.e. 4 per line instead of 5: no arithmetic, shared-memory exchange or barrier is spent on zeros.
//  * ONE TRANSFORM ROUTINE.  All 8 jobs run through one copy of the code: the job loop is rolled, the forward transforms
//    use the inverse butterflies (F(x) = conj(F^-1(conj x)); the conjugations fold into the product formation and the
//    radix-3 twiddle), and forward and inverse use the same flow "radix 16 in registers -> twiddle -> warp-local exchange
//    -> radix G": a thread holds the points p = t + G j of a sub-transform before AND after it (only the register order
//    differs, a compile-time permutation), so no mirrored forward routine is needed.  The loop body is about 1/3 of the
//    unrolled per-line version and fits the 32 KB instruction cache.
//  * The physical-space fields that have to wait (4 fields of 16 values per thread: u3A, u3B and either (u1, u2) of the line
//    being worked on or T23A / T23B) are parked in TENSOR MEMORY (tmem.cuh); registers hold only the transform in flight.
//  * Inputs are fetched by the TMA bulk-copy engine into a 2-slot ring per lane group (one slot = the two half-spectrum
//    lines of one inverse job), issued two to three jobs ahead at the named barriers of the forward jobs.
//
// Thread layout: block = UNITS units of 96 threads; unit = 3 warps = the three radix-3 sub-transforms q of 32/G line pairs;
// lane group = G = L/16 lanes = one line pair; every lane holds 16 complex values.
#pragma once
#include <cstdint>

#include "cx.cuh"
#include "kernels_zfused.cuh"   // mbarrier / bulk-copy helpers, named_bar_sync, prune3
#include "tmem.cuh"

namespace ns {

template <typename T, int L> struct ZPGeo {
    static constexpr int G = L / 16;          // lanes per sub-transform = lanes per line pair
    static constexpr int Hc = 16 / G;         // radix-G transforms per lane in the second stage
    static constexpr int PL = 32 / G;         // line pairs per unit
    static constexpr int REGION = 16 * 32;    // exchange / combine region of one warp, complex elements (16 rows x 32 lanes)
    static constexpr int SLOT = 2 * L;        // one input slot: two lines of L complex
    // odd lane groups are shifted by 4 elements (64 B) when G = 4 so that the two groups of a quarter warp hit disjoint banks
    static constexpr int LGPITCH = 2 * SLOT + (G == 4 ? 4 : 0);
    static constexpr int IN_UNIT = PL * LGPITCH;                         // input ring of one unit, complex elements
    static constexpr size_t UNIT_BYTES = (size_t)(IN_UNIT + 3 * REGION) * sizeof(cx<T>) + (size_t)(PL * 2 + 2) * sizeof(uint64_t);
    static constexpr uint32_t C16 = 16 * sizeof(T) / 4;                  // TMEM columns of 16 scalars
    static constexpr uint32_t WCOLS = 4 * C16;                           // TMEM columns per warp: 4 fields
    static constexpr uint32_t TWCOLS = 4 * C16;                          // the thread's 16 inter-stage + 16 radix-3 twiddles (complex)
};

// register holding point j (p = t + G j) after a transform: output (h, r2) <-> j = h + Hc r2 sits at h G + brev_G(r2)
template <int G> __host__ __device__ constexpr int zp_perm(int j) {
    constexpr int Hc = 16 / G;
    return (j % Hc) * G + brev<G>(j / Hc);
}

// inverse of zp_perm: the point j held by register i
template <int G> __host__ __device__ constexpr int zp_unperm(int i) {
    for (int j = 0; j < 16; ++j)
        if (zp_perm<G>(j) == i) return j;
    return -1;
}

// The transform of all jobs: in v[j] = s[t + G j], out v[zp_perm(j')] = sum_n s[n] w_L^{+n k}, k = t + G j'.
// Sw: the warp's exchange region (16 rows x 32 columns, XOR-swizzled: element (row, col) at row*32 + (col ^ (row & 7))).
// ttw: tensor-memory address of the thread's inter-stage twiddles w_L^{r1 t}, r1 = 0..15 (they depend on the lane only, so
// the warps that share a TMEM lane quarter share them; fetched a few at a time they cost neither registers nor L1).
// cdone / cparity (optional): mbarrier phase to wait for before the exchange region is overwritten -- the phase the three q
// warps of the unit complete when they have finished READING the regions in the combine of the previous forward job.  The
// wait sits after the register-only first stage, so a warp that left the combine early has its input formation and a radix-16
// stage to do before it can block (the combine is split unevenly over the warps on purpose, zp_combine_store).
template <typename T, int L>
__device__ __forceinline__ void zp_transform(cx<T> (&v)[16], cx<T>* __restrict__ Sw, int lane, int t, int lgcol, uint32_t ttw,
                                             uint64_t* cdone = nullptr, uint32_t cparity = 0) {
    constexpr int G = ZPGeo<T, L>::G, Hc = ZPGeo<T, L>::Hc;
    constexpr int CH = tmem_cx_chunk<T>();
    fft_reg<16, +1, T>(v);
    if (cdone != nullptr) mbar_wait(cdone, cparity);
#pragma unroll
    for (int ch = 0; ch < 16 / CH; ++ch) {
        T wr[CH], wi[CH];
        tmem_load_cx(ttw + 16 * ch, wr, wi);
#pragma unroll
        for (int e = 0; e < CH; ++e) {
            const int r1 = ch * CH + e;
            cx<T> w = v[brev<16>(r1)];
            if (r1 > 0) w = cmul(w, mk<T>(wr[e], wi[e]));
            Sw[r1 * 32 + (lane ^ (r1 & 7))] = w;
        }
    }
    __syncwarp();
#pragma unroll
    for (int h = 0; h < Hc; ++h) {
        const int row = t + G * h;
        const cx<T>* Sr = Sw + row * 32;
        const int rm = row & 7;
#pragma unroll
        for (int tt = 0; tt < G; ++tt) {
            // column (lgcol + tt) ^ rm; for G >= 8 the XOR touches only the low three bits of tt (lgcol is a multiple of 8)
            if constexpr (G >= 8) v[h * G + tt] = Sr[lgcol + ((tt & ~7) | ((tt & 7) ^ rm))];
            else v[h * G + tt] = Sr[(lgcol + tt) ^ rm];
        }
    }
    __syncwarp();
#pragma unroll
    for (int h = 0; h < Hc; ++h) fft_reg<G, +1, T>(v + h * G);
}

// 3 -> 2 radix-3 combine + Hermitian split of one forward job: reads G_q[n] = F_q[n] W^{-qn} of the three sub-transforms
// (regions REGION apart, swizzled as above, element n at row n / G, column lgcol + n % G) and writes TWICE the two real
// transforms, 2 B_a^[n] and 2 B_b^[n], for n and L - n (kernels_z.cuh; the factor 1/2 of the Hermitian split is folded into the
// normalisation of the spectral kernel, see zp_output_scale).  The 8G + 1 values n <= L/2 are shared out unevenly on
// purpose: the q = 0 warp has no radix-3 twiddles to apply in the transforms, so it takes half of the combine
// (n < 4G), the other two a quarter each -- the three warps then reach the named barriers at about the same time.
template <typename T, int L>
__device__ __forceinline__ void zp_combine_store(const cx<T>* __restrict__ Su, int lgcol, cx<T>* __restrict__ Oa, cx<T>* __restrict__ Ob, int q,
                                                 int t) {
    constexpr int G = ZPGeo<T, L>::G, REGION = ZPGeo<T, L>::REGION;
    constexpr T h3 = (T)0.86602540378443864676L;
    auto at = [&](int qq, int n) {
        const int row = n / G, col = lgcol + n % G;
        return Su[qq * REGION + row * 32 + (col ^ (row & 7))];
    };
    // q = 0: n = t + G i, i < 4;  q = 1: n = 4G + t + G i, i < 2;  q = 2: n = 6G + t + G i, i < 2;  n = 8G = L/2: lane t = 0 of q = 2
    const int n0 = q == 0 ? t : (q == 1 ? 4 * G + t : 6 * G + t);
    // The regions hold the CONJUGATES of F_0, G_1, G_2 (zp_post_forward stores the raw output of the inverse butterflies: the
    // conjugation of F(x) = conj(F^-1(conj x)) costs nothing here, it is only signs in the additions below).  With f0, g1, g2 the
    // stored values: A' = f0 + S = conj(A),  C' = f0 - S/2 - i (sqrt3/2) D = conj(C).
    auto one = [&](cx<T> f0, cx<T> g1, cx<T> g2, cx<T>& A, cx<T>& C) {
        const cx<T> S = g1 + g2, D = g1 - g2;
        A = f0 + S;
        C = mk<T>(f0.x - (T)0.5 * S.x + h3 * D.y, f0.y - (T)0.5 * S.y - h3 * D.x);
    };
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        if (half == 1 && q != 0) break;          // warp-uniform: only the q = 0 warp has a second pair of values
        cx<T> f0[2], g1[2], g2[2], f0m[2], g1m[2], g2m[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int n = n0 + G * (2 * half + k);
            const int m = n == 0 ? 0 : L - n;
            f0[k] = at(0, n); g1[k] = at(1, n); g2[k] = at(2, n);
            f0m[k] = at(0, m); g1m[k] = at(1, m); g2m[k] = at(2, m);
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int n = n0 + G * (2 * half + k);
            cx<T> An, Cn, Am, Cm;
            one(f0[k], g1[k], g2[k], An, Cn);
            one(f0m[k], g1m[k], g2m[k], Am, Cm);
            // (An, Cn, Am, Cm are the conjugates A', C' of the quantities in the formulas of kernels_z.cuh)
            if (n == 0) {
                stg_stream(Oa, mk<T>(An.x + An.x, 0));
                stg_stream(Ob, mk<T>(-An.y - An.y, 0));
            } else {
                const int m = L - n;
                stg_stream(Oa + n, mk<T>(An.x + Cm.x, Cm.y - An.y));
                stg_stream(Ob + n, mk<T>(-An.y - Cm.y, Cm.x - An.x));
                stg_stream(Oa + m, mk<T>(Am.x + Cn.x, Cn.y - Am.y));
                stg_stream(Ob + m, mk<T>(-Am.y - Cn.y, Cn.x - Am.x));
            }
        }
    }
    if (q == 2 && t == 0) {                      // n = L/2 is its own partner
        constexpr int n = L / 2;
        cx<T> An, Cn;
        one(at(0, n), at(1, n), at(2, n), An, Cn);
        stg_stream(Oa + n, mk<T>(An.x + Cn.x, Cn.y - An.y));
        stg_stream(Ob + n, mk<T>(-An.y - Cn.y, Cn.x - An.x));
    }
}

// factor carried by the outputs of zp_combine_store relative to the plain unnormalised transform
constexpr int zp_output_scale() { return 2; }

// One warp per tensor-memory lane quarter parks the twiddles of its lanes: ttw <- w_L^{r1 t} (r1 = 0..15), tw3 <- W^{t + G j}
// (j = 0..15); both depend on the lane only, so the warps that share the quarter share them.
template <typename T, int L>
__device__ __forceinline__ void zp_park_twiddles(uint32_t ttw, uint32_t tw3, int t, const Twiddles<T>& tw) {
    constexpr int G = ZPGeo<T, L>::G, CH = tmem_cx_chunk<T>();
#pragma unroll
    for (int ch = 0; ch < 16 / CH; ++ch) {
        T wr[CH], wi[CH], vr[CH], vi[CH];
#pragma unroll
        for (int e = 0; e < CH; ++e) {
            const cx<T> w = ldg(tw.z16 + (ch * CH + e) * G + t);
            wr[e] = w.x;
            wi[e] = w.y;
            const cx<T> u = ldg(tw.w3a + t + G * (ch * CH + e));
            vr[e] = u.x;
            vi[e] = u.y;
        }
        tmem_store_cx(ttw + 16 * ch, wr, wi);
        tmem_store_cx(tw3 + 16 * ch, vr, vi);
    }
    tmem_wait_st();
}

// x with its sign flipped where `flip` is set: an integer XOR on the sign bit (ALU pipe) instead of a multiplication by +-1 (the
// fp64 pipe is the busy one in these kernels)
__device__ __forceinline__ double flip_sign(double x, bool flip) {
    return __hiloint2double(__double2hiint(x) ^ (flip ? (int)0x80000000u : 0), __double2loint(x));
}
__device__ __forceinline__ float flip_sign(float x, bool flip) { return __int_as_float(__float_as_int(x) ^ (flip ? (int)0x80000000u : 0)); }

// Input of an inverse job: v[j] = s_q[t + G j] for the two-for-one field ua + i ub with half spectra Ua, Ub (shared memory).
// Radix-3 pruning of warp q: s_q[n] = (a_n + c_n (alpha + i beta)) W^{qn},  alpha + i beta = w3^{-q}, with the third
// sub-transform taken as q = -1 (physical points 3r - 1 instead of 3r + 2: the physical order along the contiguous axis never
// leaves the kernel), so that both q != 0 warps use the same twiddles W^{n}, one of them conjugated.
// a_n = Ua[n] + i Ub[n], c_n = conj(Ua[L-n]) + i conj(Ub[L-n]) (kernels_z.cuh); n = 0: real parts only, c = 0.
// XORSIGN: the sign of the twiddle's imaginary part by flip_sign (measured faster in z_pair_kernel) or by a multiplication with
// +-1 (measured faster in y2d_kernel, whose two transforms per line leave the fp64 pipe less loaded)
template <typename T, int L, bool XORSIGN = true>
__device__ __forceinline__ void zp_form_inverse(cx<T> (&v)[16], const cx<T>* __restrict__ Ua, const cx<T>* __restrict__ Ub, int q, int t,
                                                uint32_t tw3) {
    constexpr int G = ZPGeo<T, L>::G, CH = tmem_cx_chunk<T>();
    const T alpha = q == 0 ? (T)1 : (T)-0.5;
    const T beta = q == 0 ? (T)0 : (q == 1 ? (T)-0.86602540378443864676L : (T)0.86602540378443864676L);
    const bool neg = q == 2;                // sign of the imaginary part of the twiddle: W^{+n} (q = 1), W^{-n} (q = -1)
#pragma unroll
    for (int ch = 0; ch < 16 / CH; ++ch) {
        T wr[CH], wi[CH];
        tmem_load_cx(tw3 + 16 * ch, wr, wi);
#pragma unroll
        for (int e = 0; e < CH; ++e) {
            const int j = ch * CH + e;
            const int n = t + G * j;
            const cx<T> pa = Ua[n], pb = Ub[n];
            const cx<T> ma = Ua[(L - n) & (L - 1)], mb = Ub[(L - n) & (L - 1)];
            cx<T> a = mk<T>(pa.x - pb.y, pa.y + pb.x);
            cx<T> c = mk<T>(ma.x + mb.y, mb.x - ma.y);
            if (j == 0 && n == 0) { a = mk<T>(pa.x, pb.x); c = mk<T>(0, 0); }
            // z = a + c (alpha + i beta)
            cx<T> z = mk<T>(a.x + alpha * c.x - beta * c.y, a.y + alpha * c.y + beta * c.x);
            if (q > 0) z = cmul(z, mk<T>(wr[e], XORSIGN ? flip_sign(wi[e], neg) : (neg ? (T)-1 : (T)1) * wi[e]));
            v[j] = z;
        }
    }
}

// Output of a forward job (run through the inverse butterflies on conjugated input): G_q[k] = conj(v) W^{-qk}; its CONJUGATE
// v W^{qk} goes into the warp's region in natural order, k = t + G j at row j, column lane (zp_combine_store undoes it in its signs).
template <typename T, int L, bool XORSIGN = true>
__device__ __forceinline__ void zp_post_forward(const cx<T> (&v)[16], cx<T>* __restrict__ Sw, int lane, int q, uint32_t tw3) {
    constexpr int G = ZPGeo<T, L>::G, CH = tmem_cx_chunk<T>();
    const bool neg = q == 2;
#pragma unroll
    for (int ch = 0; ch < 16 / CH; ++ch) {
        T wr[CH], wi[CH];
        tmem_load_cx(tw3 + 16 * ch, wr, wi);
#pragma unroll
        for (int e = 0; e < CH; ++e) {
            const int j = ch * CH + e;
            const cx<T> y = v[zp_perm<G>(j)];
            cx<T> w = y;
            if (q > 0) {   // G_q = conj(y) conj(r) = conj(y r), r = W^{qk}: y r is stored, the conjugation is done by the combine
                const T rx = wr[e], ry = XORSIGN ? flip_sign(wi[e], neg) : (neg ? (T)-1 : (T)1) * wi[e];
                w = mk<T>(y.x * rx - y.y * ry, y.x * ry + y.y * rx);
            }
            Sw[j * 32 + (lane ^ (j & 7))] = w;
        }
    }
}

// in [batch][3][MM][L] complex -> out [batch][5][MM][L] complex (unnormalised transforms of the flux components, order
// 11 12 13 22 23).  total_pairs = batch * MM / 2 line pairs; (MM / 2) % (32 / G) == 0 (a warp never straddles two samples).
template <typename T, int L, int UNITS>
__global__ void __launch_bounds__(96 * UNITS, 1)
z_pair_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, unsigned MM, unsigned total_pairs,
              unsigned long long* __restrict__ umax2, Twiddles<T> tw) {
    using Geo = ZPGeo<T, L>;
    constexpr int G = Geo::G, PL = Geo::PL, REGION = Geo::REGION, SLOT = Geo::SLOT;
    constexpr uint32_t C16 = Geo::C16;
    constexpr int VPA = tmem_vals_per_access<T>();   // scalars per tensor-memory access
    constexpr uint32_t NWARPS = 3 * UNITS;
    constexpr uint32_t FIELD_COLS = ((NWARPS + 3) / 4) * Geo::WCOLS;
    constexpr uint32_t COLS_NEEDED = FIELD_COLS + Geo::TWCOLS;
    constexpr uint32_t NCOLS = COLS_NEEDED <= 32 ? 32 : COLS_NEEDED <= 64 ? 64 : COLS_NEEDED <= 128 ? 128 : COLS_NEEDED <= 256 ? 256 : 512;
    static_assert(COLS_NEEDED <= 512, "tensor memory: 512 columns per SM");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tslot;

    const int unit = threadIdx.x / 96;
    const int q = (threadIdx.x % 96) / 32;          // warp of the unit = sub-transform q
    const int warp = threadIdx.x / 32;
    const int lane = threadIdx.x & 31;
    const int lg = lane / G, t = lane % G;
    const int lgcol = lg * G;


    unsigned char* ubase = smem_raw + (size_t)unit * Geo::UNIT_BYTES;
    cx<T>* In = reinterpret_cast<cx<T>*>(ubase);                       // [PL] x (2 slots x 2 lines x L), pitch LGPITCH
    cx<T>* Ex = In + Geo::IN_UNIT;                                      // [3][REGION]
    uint64_t* bars = reinterpret_cast<uint64_t*>(Ex + 3 * REGION);      // [PL][2] input ring, then [1] combine-done
    uint64_t* cdone = bars + 2 * PL;
    cx<T>* Sw = Ex + q * REGION;
    const cx<T>* Ulg = In + (size_t)lg * Geo::LGPITCH;
    uint64_t* bar_lg = bars + lg * 2;
    const int bar_id = 1 + unit;
    const long cs = (long)MM * L;                    // component stride (complex) of in and out
    constexpr uint32_t LINE_BYTES = (uint32_t)(L * sizeof(cx<T>));

    // input job jn = 3 * it + k of this lane group: k = 0 (u3A, u3B), 1 (u1A, u2A), 2 (u1B, u2B); slot jn & 1
    auto issue = [&](unsigned pr, int k, int jn) {
        const unsigned lineA = 2 * pr;
        const unsigned b = lineA / MM;                                  // in offset: (b 3 MM + pp) L = (lineA + 2 b MM) L
        const cx<T>* src = in + ((long)lineA + 2 * (long)b * MM) * L;
        cx<T>* dst = const_cast<cx<T>*>(Ulg) + (jn & 1) * SLOT;
        uint64_t* bar = bar_lg + (jn & 1);
        mbar_expect_tx(bar, 2 * LINE_BYTES);
        // k = 0: u3 of lines A and B (contiguous); k = 1, 2: u1 and u2 of line A / B (a component stride apart)
        const cx<T>* s1 = src + (k == 0 ? 2 * cs : (k == 2 ? L : 0));
        const long second = k == 0 ? L : cs;
        bulk_g2s(dst, s1, LINE_BYTES, bar);
        bulk_g2s(dst + L, s1 + second, LINE_BYTES, bar);
    };

    if (threadIdx.x % 96 == 0) {
        for (int k = 0; k < 2 * PL; ++k) mbar_init(bars + k, 1);
        mbar_init(cdone, 3);            // one arrival per q warp
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(&tslot, NCOLS);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    // this warp's TMEM window: lanes 32 (warp % 4) .. +31, columns (warp / 4) * WCOLS .. + WCOLS: four fields of C16 columns
    const uint32_t tbase = tslot + ((uint32_t)(32 * (warp % 4)) << 16) + (uint32_t)(warp / 4) * Geo::WCOLS;
    const uint32_t ttw = tslot + ((uint32_t)(32 * (warp % 4)) << 16) + FIELD_COLS;
    const uint32_t tw3 = ttw + 2 * C16;
    if (warp < 4) zp_park_twiddles<T, L>(ttw, tw3, t, tw);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();

    const unsigned stride = gridDim.x * UNITS * PL;
    unsigned pair = (blockIdx.x * UNITS + unit) * PL + lg;        // (MM/2) % PL == 0: validity is uniform over the unit
    const bool issuer = (q == 0 && t == 0);
    if (issuer && pair < total_pairs) {
#pragma unroll 1
        for (int k = 0; k < 2; ++k) issue(pair, k, k);
    }

    unsigned nfwd = 0;      // forward jobs this warp has completed = phases of cdone it has arrived on
    for (int it = 0; pair < total_pairs; pair += stride, ++it) {
        const unsigned lineA = 2 * pair;
        const unsigned b = lineA / MM;
        cx<T>* OpA = out + ((long)lineA + 4 * (long)b * MM) * L;        // out offset: (b 5 MM + pp) L
        const bool more = pair + stride < total_pairs;

#pragma unroll 1
        for (int job = 0; job < 8; ++job) {
            const bool inv = (0x13 >> job) & 1;          // jobs 0, 1, 4
            // fields (TMEM column offsets in units of C16): see the job table at the top
            //   job:   0     1     2      3      4     5      6      7
            //   fa     0     2     2      2      3     3      3      2      (inverse: re ->; forward: x)
            //   fb     1     3     3      3      0     0      0      3      (inverse: im ->; forward: y)
            //   fc     -     -     0      0      -     1      1      -      (forward: z)
            const uint32_t fa = tbase + C16 * ((0x23332220u >> (4 * job)) & 15u);
            const uint32_t fb = tbase + C16 * ((0x30003331u >> (4 * job)) & 15u);
            const uint32_t fc = tbase + C16 * (job >= 4 ? 1u : 0u);
            cx<T> v[16];
            if (inv) {
                const int k = job == 0 ? 0 : (job == 1 ? 1 : 2);
                const int jn = 3 * it + k;
                mbar_wait(bar_lg + (jn & 1), (uint32_t)((jn >> 1) & 1));
                const cx<T>* Ua = Ulg + (jn & 1) * SLOT;
                const cx<T>* Ub = Ua + L;
                zp_form_inverse<T, L>(v, Ua, Ub, q, t, tw3);
            } else {
                // products of the physical fields, conjugated (forward through the inverse butterflies), in natural order;
                // the fields are fetched from tensor memory one x16 access (VPA values) at a time to bound the live registers
                const int kind = job == 7 ? 2 : ((job == 2 || job == 5) ? 0 : 1);
                auto lmax = sq_bits((T)0);
#pragma unroll
                for (int ch = 0; ch < 16 / VPA; ++ch) {
                    T X[VPA], Y[VPA];
                    tmem_load_vals(fa + 16 * ch, X);
                    tmem_load_vals(fb + 16 * ch, Y);
                    if (kind == 2) {
#pragma unroll
                        for (int e = 0; e < VPA; ++e) v[zp_unperm<G>(ch * VPA + e)] = mk<T>(X[e], -Y[e]);
                    } else {
                        T Z[VPA];
                        tmem_load_vals(fc + 16 * ch, Z);
                        if (kind == 0) {
                            if (umax2 != nullptr) {      // stage 1 only: max |u|^2 (sticky for NaN / inf, kernels_z.cuh)
#pragma unroll
                                for (int e = 0; e < VPA; ++e) lmax = umax_bits(lmax, sq_bits(X[e] * X[e] + Y[e] * Y[e] + Z[e] * Z[e]));
                            }
#pragma unroll
                            for (int e = 0; e < VPA; ++e) {
                                const T z2 = Z[e] * Z[e];
                                v[zp_unperm<G>(ch * VPA + e)] = mk<T>(X[e] * X[e] - z2, z2 - Y[e] * Y[e]);
                            }
                        } else {
                            T W[VPA];
#pragma unroll
                            for (int e = 0; e < VPA; ++e) {
                                v[zp_unperm<G>(ch * VPA + e)] = mk<T>(X[e] * Y[e], -(X[e] * Z[e]));
                                W[e] = Y[e] * Z[e];
                            }
                            tmem_store_vals(fa + 16 * ch, W);   // T23 of this line replaces u1 (no longer needed)
                        }
                    }
                }
                if (kind == 0 && umax2 != nullptr) {   // the lines of a warp belong to one sample
                    lmax = warp_max_bits(lmax);
                    if (lane == 0) atomic_max_sq(umax2 + b, lmax);
                }
            }
            // the regions may be overwritten only when all three warps have finished the combine of the last forward job
            zp_transform<T, L>(v, Sw, lane, t, lgcol, ttw, nfwd > 0 ? cdone : nullptr, (nfwd - 1) & 1u);
            if (inv) {
#pragma unroll
                for (int ch = 0; ch < 16 / VPA; ++ch) {
                    T X[VPA], Y[VPA];
#pragma unroll
                    for (int e = 0; e < VPA; ++e) { X[e] = v[ch * VPA + e].x; Y[e] = v[ch * VPA + e].y; }
                    tmem_store_vals(fa + 16 * ch, X);
                    tmem_store_vals(fb + 16 * ch, Y);
                }
                tmem_wait_st();
            } else {
                tmem_wait_st();
                zp_post_forward<T, L>(v, Sw, lane, q, tw3);
                named_bar_sync(bar_id, 96);
                // all three warps are past the inverse jobs that read the input slots: refill them
                if (issuer && (job == 2 || job == 5)) {
                    // job 2: (u1B, u2B) of this pair and (u3A, u3B) of the next one; job 5: (u1A, u2A) of the next one
                    const int first = job == 2 ? 2 : 4, last = !more ? 2 : (job == 2 ? 3 : 4);
#pragma unroll 1
                    for (int kk = first; kk <= last; ++kk) issue(kk >= 3 ? pair + stride : pair, kk >= 3 ? kk - 3 : kk, 3 * it + kk);
                }
                cx<T>* Oa;
                cx<T>* Ob;
                if (job == 7) { Oa = OpA + 4 * cs; Ob = Oa + L; }
                else {
                    cx<T>* Ol = OpA + (job >= 4 ? L : 0);
                    const bool p0 = (job == 2 || job == 5);
                    Oa = Ol + (p0 ? 0 : 1) * cs;
                    Ob = Ol + (p0 ? 3 : 2) * cs;
                }
                zp_combine_store<T, L>(Ex, lgcol, Oa, Ob, q, t);
                // combine reads done: arrive (no wait here -- the wait is in the next zp_transform, before the regions are reused)
                __syncwarp();
                if (lane == 0) mbar_arrive(cdone);
                ++nfwd;
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tslot, NCOLS);
}

}  // namespace ns
