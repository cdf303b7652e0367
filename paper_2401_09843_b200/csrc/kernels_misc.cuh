// kernels_misc.cuh -- pointwise and reduction kernels of the product path:
//   spectral_kernel   step a7: divergence, Leray projection (eq. 2.5), dissipation
//                     (eq. 2.1-2.4) and one line of SSP-RK3 (eq. 2.6)
//   cfl_finalize      step a8: dt_b from max|u| (reading A10)
//   layout converters, energy spectrum, structure-function marginals
//   generic power-of-two FFT on the unpadded N grid, used only by ns_set_initial / ns_get_fields.
// Internal spectral layout: [batch][comp][N][N][H], H = N/2 (the identically-zero kz = N/2 column of the
// public layout is not stored, so rows are 128-byte aligned).
#pragma once
#include <cuda_pipeline.h>
#include <math_constants.h>

#include "cx.cuh"
#include "ns_internal.h"

namespace ns {

__device__ __forceinline__ int wavenum(int i, int N) { return i < N / 2 ? i : i - N; }

// ------------------------------------------------------------------------------------------------
// a7.  Th: [b][5][N][N][H] unnormalised transforms of the trace-free flux T_ij = u_i u_j - delta_ij u_3^2
//   (order 11 12 13 22 23, T33 = 0; kernels_z.cuh: the omitted part is a gradient, removed by the projection).
//   b_i = -i k_j Th_ij * scale;  Nl = b - k (k.b)/|k|^2;  R = Nl - d(|k|^2) * Us
//   mode 0: out = R
//   mode 1: out = alpha*Un + beta*Us + gamma*dt_b*R   (Un may be NULL when alpha == 0)
//           dt_b == 0 marks an inactive sample: out = Un (or Us when Un is NULL), bit exact.
//   IN-PLACE CONTRACT: out may alias Us or Un (RK stages 2 and 3 update V and U in place), so these three pointers are
//   not __restrict__; every thread reads its own entries of Us / Un before it writes the same entries of out.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256, 4)
spectral_kernel(const cx<T>* __restrict__ Bh, const cx<T>* Us, const cx<T>* Un, cx<T>* out, int N, int kmax, long total, const T* __restrict__ dtab, T scale, T alpha, T beta,
                T gamma, const double* __restrict__ dt, int mode, int Nyl, int iy0) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    // arrays [b][comp][N (kx)][Nyl (ky)][H]: the ky rows iy0 .. iy0 + Nyl - 1 of the grid (Nyl = N, iy0 = 0 except in the
    // ky-slabs of the multi-device solver, ns_mg.h)
    const int H = N / 2;
    const int iz = (int)(idx % H);
    const int iyl = (int)((idx / H) % Nyl);
    const int ix = (int)((idx / ((long)H * Nyl)) % N);
    const long b = idx / ((long)H * Nyl * N);
    const long plane = (long)N * Nyl * H;
    const long o = ((long)ix * Nyl + iyl) * H + iz;
    const cx<T>* us = Us + b * 3 * plane + o;
    cx<T>* op = out + b * 3 * plane + o;
    const int kxi = wavenum(ix, N), kyi = wavenum(iy0 + iyl, N);
    const int k2i = kxi * kxi + kyi * kyi + iz * iz;
    // truncation P_N of eq. 2.1: modes with a wavenumber component >= kmax = (user N)/2 carry nothing (kmax = N/2 unless the
    // transform grid is larger than the user's grid, ns_create); k = 0: reading A8
    const bool dead = (kxi >= kmax) || (kxi <= -kmax) || (kyi >= kmax) || (kyi <= -kmax) || (iz >= kmax) || (k2i == 0);

    cx<T> R[3] = {mk<T>(0, 0), mk<T>(0, 0), mk<T>(0, 0)};
    cx<T> u[3], un3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) u[c] = us[c * plane];
    // the second state of stages 2, 3 is fetched together with everything else (one round trip to HBM instead of two)
    const cx<T>* un = (mode != 0 && Un) ? Un + b * 3 * plane + o : nullptr;
    if (un) {
#pragma unroll
        for (int c = 0; c < 3; ++c) un3[c] = un[c * plane];
    }
    if (!dead) {
        const cx<T>* bp = Bh + b * NS_NFLUX * plane + o;
        const cx<T> B11 = ldg(bp), B12 = ldg(bp + plane), B13 = ldg(bp + 2 * plane), B22 = ldg(bp + 3 * plane),
                    B23 = ldg(bp + 4 * plane);
        const T kx = (T)kxi, ky = (T)kyi, kz = (T)iz;
        // -i z = (z.y, -z.x)
        cx<T> bb[3];
        {
            const cx<T> z0 = mk<T>(kx * B11.x + ky * B12.x + kz * B13.x, kx * B11.y + ky * B12.y + kz * B13.y);
            const cx<T> z1 = mk<T>(kx * B12.x + ky * B22.x + kz * B23.x, kx * B12.y + ky * B22.y + kz * B23.y);
            const cx<T> z2 = mk<T>(kx * B13.x + ky * B23.x, kx * B13.y + ky * B23.y);
            bb[0] = mk<T>(scale * z0.y, -scale * z0.x);
            bb[1] = mk<T>(scale * z1.y, -scale * z1.x);
            bb[2] = mk<T>(scale * z2.y, -scale * z2.x);
        }
        const T ik2 = (T)1 / (T)k2i;
        const cx<T> kb = mk<T>((kx * bb[0].x + ky * bb[1].x + kz * bb[2].x) * ik2,
                               (kx * bb[0].y + ky * bb[1].y + kz * bb[2].y) * ik2);
        const T d = dtab[k2i];
        R[0] = mk<T>(bb[0].x - kx * kb.x - d * u[0].x, bb[0].y - kx * kb.y - d * u[0].y);
        R[1] = mk<T>(bb[1].x - ky * kb.x - d * u[1].x, bb[1].y - ky * kb.y - d * u[1].y);
        R[2] = mk<T>(bb[2].x - kz * kb.x - d * u[2].x, bb[2].y - kz * kb.y - d * u[2].y);
    }
    if (mode == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) op[c * plane] = R[c];
        return;
    }
    const T dtb = (T)dt[b];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        cx<T> r;
        if (un) {
            const cx<T> n = un3[c];
            if (dtb == (T)0) r = n;
            else r = mk<T>(alpha * n.x + beta * u[c].x + gamma * dtb * R[c].x, alpha * n.y + beta * u[c].y + gamma * dtb * R[c].y);
        } else {
            if (dtb == (T)0) r = u[c];
            else r = mk<T>(beta * u[c].x + gamma * dtb * R[c].x, beta * u[c].y + gamma * dtb * R[c].y);
        }
        op[c * plane] = r;
    }
}

// ------------------------------------------------------------------------------------------------
// time-step bookkeeping (device resident: no host sync inside a step)
// ------------------------------------------------------------------------------------------------
// umax2[b] holds the bits of max |u|^2 over the padded grid at the start of the step (by-product of a3 in stage 1; a
// non-finite field gives +inf or NaN there, kernels_z.cuh).  A sample whose maximum is not finite is marked in bad[b]
// and frozen (dt_b = 0): the host reports NS_ERR_NONFINITE at its next synchronising call.
__device__ __forceinline__ bool nonfinite_sq(unsigned long long bits) {
    const double um2 = __longlong_as_double((long long)bits);
    return !(um2 < CUDART_INF);
}
static __global__ void set_dt_uniform_kernel(double* dt, double* t, double value, const unsigned long long* umax2, int* bad, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    if (nonfinite_sq(umax2[b])) { bad[b] = 1; value = 0.0; }
    dt[b] = value;
    t[b] += value;
}
static __global__ void set_dt_array_kernel(double* dt, double* t, const double* src, const unsigned long long* umax2, int* bad, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    double value = src[b];
    if (nonfinite_sq(umax2[b])) { bad[b] = 1; value = 0.0; }
    dt[b] = value;
    t[b] += value;
}
// dt_b = min(cfl * dx / umax_b, t_end - t_b); 0 for finished samples.
static __global__ void cfl_finalize_kernel(double* dt, double* t, const unsigned long long* umax2, int* bad, double cfl, double dx,
                                    double t_end, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const double remaining = t_end - t[b];
    double v = 0.0;
    if (nonfinite_sq(umax2[b])) {
        bad[b] = 1;
    } else if (remaining > 0.0) {
        const double um = sqrt(__longlong_as_double((long long)umax2[b]));
        v = um > 0.0 ? cfl * dx / um : remaining;
        if (!(v < remaining)) v = remaining;
    }
    dt[b] = v;
    t[b] += v;
}
static __global__ void umax_read_kernel(double* out, const unsigned long long* umax2, int* bad, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    if (nonfinite_sq(umax2[b])) bad[b] = 1;
    out[b] = sqrt(__longlong_as_double((long long)umax2[b]));   // +inf / NaN for a non-finite field
}

// ------------------------------------------------------------------------------------------------
// layout converters: public [.][N][N][N/2+1]  <->  internal [.][N][N][N/2]
// ------------------------------------------------------------------------------------------------
// Nu = the user's grid size (public arrays), N >= Nu the transform grid of the handle (internal arrays): a mode k of the
// user's grid sits at stored index k mod Nu there and k mod N here; modes with |k_i| >= Nu/2 are zero here.
__device__ __forceinline__ int embed_index(int i, int N, int Nu) {   // internal index -> public index, -1 if outside K_Nu
    const int k = wavenum(i, N);
    if (k >= Nu / 2 || k <= -(Nu / 2)) return -1;
    return k >= 0 ? k : k + Nu;
}
template <typename T>
__global__ void to_internal_kernel(const cx<T>* __restrict__ pub, cx<T>* __restrict__ in, int N, int Nu, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2, Hu = Nu / 2;
    const int iz = (int)(idx % H);
    const long row = idx / H;  // (cube, ix, iy)
    const int iy = (int)(row % N), ix = (int)((row / N) % N);
    const long cube = row / ((long)N * N);
    const int jx = embed_index(ix, N, Nu), jy = embed_index(iy, N, Nu);
    cx<T> v = mk<T>(0, 0);
    if (jx >= 0 && jy >= 0 && iz < Hu) v = pub[((cube * Nu + jx) * Nu + jy) * (Hu + 1) + iz];
    in[idx] = v;
}
template <typename T>
__global__ void to_public_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ pub, int N, int Nu, long total_pub) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total_pub) return;
    const int H = N / 2, Hu = Nu / 2;
    const int iz = (int)(idx % (Hu + 1));
    const long row = idx / (Hu + 1);
    const int jy = (int)(row % Nu), jx = (int)((row / Nu) % Nu);
    const long cube = row / ((long)Nu * Nu);
    cx<T> v = mk<T>(0, 0);
    if (iz != Hu && jx != Hu && jy != Hu) {
        const int ix = jx < Hu ? jx : jx - Nu + N, iy = jy < Hu ? jy : jy - Nu + N;
        v = in[((cube * N + ix) * N + iy) * H + iz];
    }
    pub[idx] = v;
}

// ------------------------------------------------------------------------------------------------
// energy spectrum: E[b][K] += w/2 |u_hat|^2, K = floor(|k| + 1/2)
// ENS: enstrophy spectrum, |u_hat|^2 replaced by |k x u_hat|^2 (vorticity omega_hat = i k x u_hat)
// grid = (chunks, batch); dynamic smem nbins doubles
// ------------------------------------------------------------------------------------------------
template <typename T, bool ENS>
__global__ void energy_spectrum_kernel(const cx<T>* __restrict__ U, double* __restrict__ E, int N, int nbins) {
    extern __shared__ double bins[];
    for (int i = threadIdx.x; i < nbins; i += blockDim.x) bins[i] = 0.0;
    __syncthreads();
    const int H = N / 2;
    const long plane = (long)N * N * H;
    const long b = blockIdx.y;
    const cx<T>* u = U + b * 3 * plane;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < plane; idx += (long)gridDim.x * blockDim.x) {
        const int iz = (int)(idx % H), iy = (int)((idx / H) % N), ix = (int)(idx / ((long)H * N));
        if (ix == N / 2 || iy == N / 2) continue;
        const double kx = wavenum(ix, N), ky = wavenum(iy, N), kz = iz;
        const int bin = (int)floor(sqrt(kx * kx + ky * ky + kz * kz) + 0.5);
        if (bin >= nbins) continue;
        double e = 0.0;
        if constexpr (ENS) {
            const cx<T> a = u[idx], b2 = u[plane + idx], c3 = u[2 * plane + idx];
            const double ax = a.x, ay = a.y, bx = b2.x, by = b2.y, cxr = c3.x, cyi = c3.y;
            // k x u, real and imaginary parts separately (the factor i does not change the modulus)
            const double w1r = ky * cxr - kz * bx, w1i = ky * cyi - kz * by;
            const double w2r = kz * ax - kx * cxr, w2i = kz * ay - kx * cyi;
            const double w3r = kx * bx - ky * ax, w3i = kx * by - ky * ay;
            e = w1r * w1r + w1i * w1i + w2r * w2r + w2i * w2i + w3r * w3r + w3i * w3i;
        } else {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const cx<T> v = u[c * plane + idx];
                e += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
            }
        }
        atomicAdd(&bins[bin], (iz == 0 ? 0.5 : 1.0) * e);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += blockDim.x)
        if (bins[i] != 0.0) atomicAdd(&E[b * nbins + i], bins[i]);
}

// ------------------------------------------------------------------------------------------------
// structure function through its exact spectral form:
//   S2(l) = (1/3) sum_d sum_k 2 (1 - cos(k_d l dx)) w_k |u_hat_k|^2
// marginals: e[b][d][i] = sum over the other two indices of w |u_hat|^2, i = stored index along d
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void sf_marginals_kernel(const cx<T>* __restrict__ U, double* __restrict__ marg, int N) {
    extern __shared__ double bins[];  // [3][N]
    for (int i = threadIdx.x; i < 3 * N; i += blockDim.x) bins[i] = 0.0;
    __syncthreads();
    const int H = N / 2;
    const long plane = (long)N * N * H;
    const long b = blockIdx.y;
    const cx<T>* u = U + b * 3 * plane;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < plane; idx += (long)gridDim.x * blockDim.x) {
        const int iz = (int)(idx % H), iy = (int)((idx / H) % N), ix = (int)(idx / ((long)H * N));
        if (ix == N / 2 || iy == N / 2) continue;
        double e = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const cx<T> v = u[c * plane + idx];
            e += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
        }
        e *= (iz == 0 ? 1.0 : 2.0);
        atomicAdd(&bins[ix], e);
        atomicAdd(&bins[N + iy], e);
        atomicAdd(&bins[2 * N + iz], e);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 3 * N; i += blockDim.x)
        if (bins[i] != 0.0) atomicAdd(&marg[b * 3 * N + i], bins[i]);
}
// one block per sample, thread per l
static __global__ void sf_finalize_kernel(const double* __restrict__ marg, double* __restrict__ S, int N, int Nu, int nl) {
    const int b = blockIdx.x;
    for (int l = 1 + threadIdx.x; l <= nl; l += blockDim.x) {
        double acc = 0.0;
        for (int d = 0; d < 3; ++d)
            for (int i = 0; i < N; ++i) {
                const double e = marg[(b * 3 + d) * N + i];
                if (e == 0.0) continue;
                const int k = (d == 2) ? i : wavenum(i, N);
                // cos(k l dx) = cos(2 pi k l / Nu), dx = 2 pi / Nu the user's grid spacing, with exact argument reduction
                const long kl = ((long)k * l) % Nu;
                acc += 2.0 * (1.0 - cospi(2.0 * (double)kl / (double)Nu)) * e;
            }
        S[b * nl + (l - 1)] = acc / 3.0;
    }
}

// G consecutive radix-2 DIT levels s .. s+G-1 of the tile in shared memory S[n][9] (8 lines), done in registers: the 2^G
// elements base + t 2^(s-1) of a block of 2^(s-1+G) (a sub-sequence of length m is a whole number of such blocks).
template <typename T, int G>
__device__ __forceinline__ void generic_dit_pass(cx<T>* __restrict__ S, int s, int n, int sign, const cx<T>* __restrict__ gtw) {
    constexpr int TL = 8, PITCH = TL + 1, R = 1 << G;
    const int half0 = 1 << (s - 1);
    const int items = (n >> G) * TL;
    for (int e = threadIdx.x; e < items; e += blockDim.x) {
        const int c = e % TL, gi = e / TL;
        const int o = gi & (half0 - 1);
        const int base = ((gi >> (s - 1)) << (s - 1 + G)) + o;
        cx<T> v[R];
#pragma unroll
        for (int t = 0; t < R; ++t) v[t] = S[(base + t * half0) * PITCH + c];
#pragma unroll
        for (int l = 0; l < G; ++l) {
            const int dt = 1 << l;
#pragma unroll
            for (int t = 0; t < R; ++t) {
                if (t & dt) continue;
                const int j = o + (t & (dt - 1)) * half0;                  // position within the half of level s + l
                cx<T> w = ldg(gtw + (long)j * (n >> (s + l)));              // w_{2^(s+l)}^j from the order-n table
                if (sign < 0) w = conj(w);
                const cx<T> a = v[t], bq = cmul(v[t + dt], w);
                v[t] = a + bq;
                v[t + dt] = a - bq;
            }
        }
#pragma unroll
        for (int t = 0; t < R; ++t) S[(base + t * half0) * PITCH + c] = v[t];
    }
}

// ------------------------------------------------------------------------------------------------
// unpadded N-grid transforms for ns_set_initial / ns_get_fields / the physical-space statistics (NOT on the hot path):
// a shared-memory FFT on tiles of 8 lines of a full complex [cubes][n][n][n] array, in place, n = p 2^a with p in {1, 3, 5, 7, 15}.
//   axis 0: element stride n*n, axis 1: n, axis 2: 1.  dim = 2: the same on [planes][n][n] (axes 1 and 2).
// n = p m, p in {3, 5, 7, 15}: the p decimated sequences x[p r + q] are transformed by radix-2 stages (m = 2^a) and combined by
// one radix-p stage, X[k + m t] = sum_q w_n^{q (k + m t)} F_q[k].  Twiddles come from the table gtw[j] = exp(+2 pi i j / n).
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
generic_fft_kernel(cx<T>* __restrict__ A, int n, int log2m, int nsub, int axis, int sign, long total_tiles,
                   const cx<T>* __restrict__ gtw, int dim) {
    constexpr int TL = 8;  // lines per tile
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* S = reinterpret_cast<cx<T>*>(smem_raw);  // [n][TL+1]
    constexpr int PITCH = TL + 1;
    const long tile = blockIdx.x;
    if (tile >= total_tiles) return;
    const int m = 1 << log2m;          // n = nsub m, nsub in {1, 3, 5, 7, 15}
    // dim = 3: cubes [n][n][n], n^2 lines per cube and axis; dim = 2: planes [n][n] (axes 1 and 2 only), n lines per plane
    const long n2 = (long)n * n;
    const long lines = dim == 3 ? n2 : n;
    const long tiles_per_cube = lines / TL;
    const long cube = tile / tiles_per_cube;
    const long l0 = (tile % tiles_per_cube) * TL;  // first line id within the cube
    cx<T>* base = A + cube * (dim == 3 ? n2 * n : n2);
    const long es = axis == 0 ? n2 : (axis == 1 ? n : 1);
    // line id l -> offset of element 0
    auto line_base = [&](long l) -> long {
        if (axis == 0) return l;
        if (axis == 1) return dim == 3 ? (l / n) * n2 + (l % n) : l;
        return l * n;
    };
    auto root = [&](int j) -> cx<T> {   // exp(sign 2 pi i j / n), 0 <= j < n
        const cx<T> w = ldg(gtw + j);
        return sign > 0 ? w : conj(w);
    };
    // load: element j = nsub r + q goes to q m + bitrev_m(r); asynchronous copies (LDGSTS), so that all of a thread's loads
    // are in flight at once without holding registers
    for (int e = threadIdx.x; e < n * TL; e += blockDim.x) {
        int j, c;
        if (axis == 2) { j = e % n; c = e / n; } else { c = e % TL; j = e / TL; }
        const int q = j % nsub, r = j / nsub;
        const int rr = log2m == 0 ? 0 : (int)(__brev((unsigned)r) >> (32 - log2m));
        __pipeline_memcpy_async(&S[(q * m + rr) * PITCH + c], &base[line_base(l0 + c) + (long)j * es], sizeof(cx<T>));
    }
    __pipeline_commit();
    __pipeline_wait_prior(0);
    __syncthreads();
    // radix-2 decimation-in-time levels 1..log2m, up to three levels per pass in registers (one barrier and one trip through
    // shared memory per pass instead of per level)
    for (int s = 1; s <= log2m;) {
        const int G = log2m - s + 1 >= 3 ? 3 : log2m - s + 1;
        if (G == 3) generic_dit_pass<T, 3>(S, s, n, sign, gtw);
        else if (G == 2) generic_dit_pass<T, 2>(S, s, n, sign, gtw);
        else generic_dit_pass<T, 1>(S, s, n, sign, gtw);
        s += G;
        __syncthreads();
    }
    if (nsub == 3) {
        const T h = (T)sign * (T)0.86602540378443864676L;
        for (int e = threadIdx.x; e < m * TL; e += blockDim.x) {
            const int c = e % TL, k = e / TL;
            const cx<T> f0 = S[k * PITCH + c];
            const cx<T> f1 = cmul(S[(m + k) * PITCH + c], root(k));
            const cx<T> f2 = cmul(S[(2 * m + k) * PITCH + c], root(2 * k));
            const cx<T> sm = f1 + f2, d = f1 - f2;
            const cx<T> mm = mk<T>(f0.x - (T)0.5 * sm.x, f0.y - (T)0.5 * sm.y);
            S[k * PITCH + c] = f0 + sm;
            S[(m + k) * PITCH + c] = mk<T>(mm.x - h * d.y, mm.y + h * d.x);
            S[(2 * m + k) * PITCH + c] = mk<T>(mm.x + h * d.y, mm.y - h * d.x);
        }
        __syncthreads();
    } else if (nsub > 1) {
        // odd factor 5, 7 or 15: the plain nsub-point combine, X[k + m t] = sum_q w_n^{qk} F_q[k] w_nsub^{qt}
        for (int e = threadIdx.x; e < m * TL; e += blockDim.x) {
            const int c = e % TL, k = e / TL;
            cx<T> f[15];
            for (int q = 0; q < nsub; ++q) f[q] = q == 0 ? S[k * PITCH + c] : cmul(S[(q * m + k) * PITCH + c], root((q * k) % n));
            for (int t = 0; t < nsub; ++t) {
                cx<T> acc = f[0];
                for (int q = 1; q < nsub; ++q) acc = acc + cmul(f[q], root(((q * t) % nsub) * m));
                S[(t * m + k) * PITCH + c] = acc;
            }
        }
        __syncthreads();
    }
    for (int e = threadIdx.x; e < n * TL; e += blockDim.x) {
        int j, c;
        if (axis == 2) { j = e % n; c = e / n; } else { c = e % TL; j = e / TL; }
        base[line_base(l0 + c) + (long)j * es] = S[j * PITCH + c];
    }
}

// Fallback of generic_fft_kernel for a grid size n that is not p 2^a (p in {1, 3, 5, 7, 15}): the plain O(n^2) DFT of tiles of
// 8 lines, X[k] = sum_j x[j] exp(sign 2 pi i jk/n), roots from the table gtw[j] = exp(+2 pi i j/n).  Only the physical-space
// entry points (ns_set_initial, ns_get_fields, S_p, moments) of handles with such a size use it; never on the hot path.
template <typename T>
__global__ void __launch_bounds__(256)
dft_lines_kernel(cx<T>* __restrict__ A, int n, int axis, int sign, long total_tiles, const cx<T>* __restrict__ gtw, int dim) {
    constexpr int TL = 8, PITCH = TL + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* S = reinterpret_cast<cx<T>*>(smem_raw);   // [n][PITCH] input
    cx<T>* O = S + (size_t)n * PITCH;                // [n][PITCH] output
    const long tile = blockIdx.x;
    if (tile >= total_tiles) return;
    // dim = 3: cubes [n][n][n], n^2 lines per cube and axis; dim = 2: planes [n][n] (axes 1 and 2 only), n lines per plane
    const long nn = (long)n * n;
    const long n2 = dim == 3 ? nn : n;                // lines per cube / plane
    const long tiles_per_cube = (n2 + TL - 1) / TL;   // the last tile may be ragged (line count not a multiple of 8)
    const long cube = tile / tiles_per_cube;
    const long l0 = (tile % tiles_per_cube) * TL;
    cx<T>* base = A + cube * (dim == 3 ? nn * n : nn);
    const long es = axis == 0 ? nn : (axis == 1 ? n : 1);
    auto line_base = [&](long l) -> long {
        if (axis == 0) return l;
        if (axis == 1) return dim == 3 ? (l / n) * nn + (l % n) : l;
        return l * n;
    };
    for (int e = threadIdx.x; e < n * TL; e += blockDim.x) {
        int j, c;
        if (axis == 2) { j = e % n; c = e / n; } else { c = e % TL; j = e / TL; }
        S[j * PITCH + c] = l0 + c < n2 ? base[line_base(l0 + c) + (long)j * es] : mk<T>(0, 0);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < n * TL; e += blockDim.x) {
        const int c = e % TL, k = e / TL;
        T ar = 0, ai = 0;
        int r = 0;                                   // (j k) mod n
        for (int j = 0; j < n; ++j) {
            const cx<T> w = ldg(gtw + r);
            const cx<T> x = S[j * PITCH + c];
            const T wy = sign > 0 ? w.y : -w.y;
            ar += x.x * w.x - x.y * wy;
            ai += x.x * wy + x.y * w.x;
            r += k;
            if (r >= n) r -= n;
        }
        O[k * PITCH + c] = mk<T>(ar, ai);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < n * TL; e += blockDim.x) {
        int j, c;
        if (axis == 2) { j = e % n; c = e / n; } else { c = e % TL; j = e / TL; }
        if (l0 + c < n2) base[line_base(l0 + c) + (long)j * es] = O[j * PITCH + c];
    }
}

template <typename T>
__global__ void real_to_complex_kernel(const T* __restrict__ in, cx<T>* __restrict__ out, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < total) out[idx] = mk<T>(in[idx], 0);
}
template <typename T>
__global__ void complex_to_real_kernel(const cx<T>* __restrict__ in, T* __restrict__ out, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < total) out[idx] = in[idx].x;
}

// W: [batch][3][N][N][N] full complex unnormalised spectra -> U internal, scaled 1/N^3, Nyquist zeroed,
// Leray-projected for k != 0 (eq. 2.5 projector; reading A11).
template <typename T>
__global__ void init_project_kernel(const cx<T>* __restrict__ W, cx<T>* __restrict__ U, int N, int Nu, long total, T scale) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2;
    const int iz = (int)(idx % H);
    const int iy = (int)((idx / H) % N);
    const int ix = (int)((idx / ((long)H * N)) % N);
    const long b = idx / ((long)H * N * N);
    const long plane = (long)N * N * H, cube = (long)Nu * Nu * Nu;
    const long o = ((long)ix * N + iy) * H + iz;
    cx<T> u[3];
    const int jx = embed_index(ix, N, Nu), jy = embed_index(iy, N, Nu);
    const bool nyq = jx < 0 || jy < 0 || iz >= Nu / 2;      // outside K_Nu (incl. the Nyquist planes of the user's grid)
#pragma unroll
    for (int c = 0; c < 3; ++c) u[c] = nyq ? mk<T>(0, 0) : scale * W[(b * 3 + c) * cube + ((long)jx * Nu + jy) * Nu + iz];
    const int kxi = wavenum(ix, N), kyi = wavenum(iy, N);
    const int k2i = kxi * kxi + kyi * kyi + iz * iz;
    if (!nyq && k2i > 0) {
        const T kx = (T)kxi, ky = (T)kyi, kz = (T)iz, ik2 = (T)1 / (T)k2i;
        const cx<T> ku = mk<T>((kx * u[0].x + ky * u[1].x + kz * u[2].x) * ik2, (kx * u[0].y + ky * u[1].y + kz * u[2].y) * ik2);
        u[0] = mk<T>(u[0].x - kx * ku.x, u[0].y - kx * ku.y);
        u[1] = mk<T>(u[1].x - ky * ku.x, u[1].y - ky * ku.y);
        u[2] = mk<T>(u[2].x - kz * ku.x, u[2].y - kz * ku.y);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) U[(b * 3 + c) * plane + o] = u[c];
}

// U internal (transform grid N) -> W full complex Hermitian spectrum on the user's Nu grid (kz < 0 from conj of (-k)).
template <typename T>
__global__ void expand_hermitian_kernel(const cx<T>* __restrict__ U, cx<T>* __restrict__ W, int N, int Nu, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2, Hu = Nu / 2;
    const int jz = (int)(idx % Nu);
    const int jy = (int)((idx / Nu) % Nu);
    const int jx = (int)((idx / ((long)Nu * Nu)) % Nu);
    const long cubei = idx / ((long)Nu * Nu * Nu);
    const long plane = (long)N * N * H;
    cx<T> v = mk<T>(0, 0);
    if (jx != Hu && jy != Hu && jz != Hu) {
        const int kx = jx < Hu ? jx : jx - Nu, ky = jy < Hu ? jy : jy - Nu, kz = jz < Hu ? jz : jz - Nu;
        if (kz >= 0) {
            v = U[cubei * plane + ((long)(kx >= 0 ? kx : kx + N) * N + (ky >= 0 ? ky : ky + N)) * H + kz];
        } else {
            v = conj(U[cubei * plane + ((long)(kx > 0 ? N - kx : -kx) * N + (ky > 0 ? N - ky : -ky)) * H - kz]);
        }
    }
    W[idx] = v;
}

// ------------------------------------------------------------------------------------------------
// structure function of order p in physical space: S[b][l-1] += sum_x sum_d |u(x + l e_d) - u(x)|^p
// u: [batch][3][N][N][N] reals; grid = (chunks, nl, batch); one shift l per blockIdx.y
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void sf_p_kernel(const T* __restrict__ u, double* __restrict__ S, int N, int nl, double p) {
    const long np = (long)N * N * N;
    const int l = blockIdx.y + 1;
    const long b = blockIdx.z;
    const T* ub = u + b * 3 * np;
    const double hp = 0.5 * p;
    double acc = 0.0;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < np; idx += (long)gridDim.x * blockDim.x) {
        const int iz = (int)(idx % N), iy = (int)((idx / N) % N), ix = (int)(idx / ((long)N * N));
        const long ox = ((long)((ix + l) % N) * N + iy) * N + iz;
        const long oy = ((long)ix * N + (iy + l) % N) * N + iz;
        const long oz = ((long)ix * N + iy) * N + (iz + l) % N;
        double rx = 0.0, ry = 0.0, rz = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double a = (double)ub[c * np + idx];
            const double dx = (double)ub[c * np + ox] - a, dy = (double)ub[c * np + oy] - a, dz = (double)ub[c * np + oz] - a;
            rx += dx * dx; ry += dy * dy; rz += dz * dz;
        }
        acc += (p == 2.0) ? rx + ry + rz : pow(rx, hp) + pow(ry, hp) + pow(rz, hp);
    }
    __shared__ double red[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) atomicAdd(&S[b * nl + (l - 1)], v);
    }
}

static __global__ void scale_kernel(double* __restrict__ a, double s, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] *= s;
}

// pointwise mean and (population) variance over the batch: u [batch][n] -> mean [n], var [n]
template <typename T>
__global__ void ensemble_moments_kernel(const T* __restrict__ u, T* __restrict__ mean, T* __restrict__ var, long n, int batch) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double m = 0.0;
    for (int b = 0; b < batch; ++b) m += (double)u[(long)b * n + i];
    m /= (double)batch;
    double v = 0.0;
    for (int b = 0; b < batch; ++b) {
        const double d = (double)u[(long)b * n + i] - m;
        v += d * d;
    }
    mean[i] = (T)m;
    var[i] = (T)(v / (double)batch);
}

}  // namespace ns
