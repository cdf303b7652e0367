// kernels_misc2d.cuh -- pointwise and reduction kernels of the TWO-DIMENSIONAL solver:
//   spectral2d_kernel  divergence, Leray projection (eq. 2.5), dissipation (eq. 2.1-2.4) and one line of
//                      SSP-RK3 (eq. 2.6) on the torus [0,2pi)^2
//   layout converters, initial projection, Hermitian expansion, ring spectra.
// Internal spectral layout: [batch][2][N][H], H = N/2 (index [b][comp][ikx][iky], iky >= 0 fastest; the identically-zero
// ky = N/2 column of the public layout [N][N/2+1] is not stored).
#pragma once
#include "cx.cuh"
#include "kernels_misc.cuh"

namespace ns {

// Th: [b][2][N][H] unnormalised transforms of the trace-free flux T11 = u1^2 - u2^2, T12 = u1 u2 (T22 = 0).
//   b_1 = -i (kx T11 + ky T12) scale,  b_2 = -i kx T12 scale;  Nl = b - k (k.b)/|k|^2;  R = Nl - d(|k|^2) Us
//   mode 0: out = R;  mode 1: out = alpha Un + beta Us + gamma dt_b R  (dt_b == 0: sample untouched, bit exact).
//   In-place contract as spectral_kernel: out may alias Us or Un.
template <typename T>
__global__ void __launch_bounds__(256)
spectral2d_kernel(const cx<T>* __restrict__ Th, const cx<T>* Us, const cx<T>* Un, cx<T>* out, int N, int kmax, long total,
                  const T* __restrict__ dtab, T scale, T alpha, T beta, T gamma, const double* __restrict__ dt, int mode) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2;
    const int iy = (int)(idx % H);
    const int ix = (int)((idx / H) % N);
    const long b = idx / ((long)H * N);
    const long plane = (long)N * H;
    const long o = (long)ix * H + iy;
    const cx<T>* us = Us + b * 2 * plane + o;
    cx<T>* op = out + b * 2 * plane + o;
    const int kxi = wavenum(ix, N);
    const int k2i = kxi * kxi + iy * iy;
    // P_N of the user's grid: modes with a component >= kmax = (user N)/2 carry nothing (kmax = N/2 unless the transform grid is larger)
    const bool dead = (kxi >= kmax) || (kxi <= -kmax) || (iy >= kmax) || (k2i == 0);
    cx<T> R[2] = {mk<T>(0, 0), mk<T>(0, 0)};
    const cx<T> u0 = us[0], u1 = us[plane];
    if (!dead) {
        const cx<T>* tp = Th + b * 2 * plane + o;
        const cx<T> T11 = ldg(tp), T12 = ldg(tp + plane);
        const T kx = (T)kxi, ky = (T)iy;
        const cx<T> z0 = mk<T>(kx * T11.x + ky * T12.x, kx * T11.y + ky * T12.y);
        const cx<T> z1 = mk<T>(kx * T12.x, kx * T12.y);
        const cx<T> b0 = mk<T>(scale * z0.y, -scale * z0.x), b1 = mk<T>(scale * z1.y, -scale * z1.x);   // -i z
        const T ik2 = (T)1 / (T)k2i;
        const cx<T> kb = mk<T>((kx * b0.x + ky * b1.x) * ik2, (kx * b0.y + ky * b1.y) * ik2);
        const T d = dtab[k2i];
        R[0] = mk<T>(b0.x - kx * kb.x - d * u0.x, b0.y - kx * kb.y - d * u0.y);
        R[1] = mk<T>(b1.x - ky * kb.x - d * u1.x, b1.y - ky * kb.y - d * u1.y);
    }
    if (mode == 0) {
        op[0] = R[0];
        op[plane] = R[1];
        return;
    }
    const T dtb = (T)dt[b];
    const cx<T> u[2] = {u0, u1};
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        cx<T> r;
        if (Un) {
            const cx<T> n = Un[b * 2 * plane + o + c * plane];
            r = dtb == (T)0 ? n : mk<T>(alpha * n.x + beta * u[c].x + gamma * dtb * R[c].x, alpha * n.y + beta * u[c].y + gamma * dtb * R[c].y);
        } else {
            r = dtb == (T)0 ? u[c] : mk<T>(beta * u[c].x + gamma * dtb * R[c].x, beta * u[c].y + gamma * dtb * R[c].y);
        }
        op[c * plane] = r;
    }
}

// public [.][Nu][Nu/2+1] (the user's grid) <-> internal [.][N][N/2] (the transform grid N >= Nu; modes outside K_Nu are zero)
__device__ __forceinline__ int embed_index2d(int i, int N, int Nu) {   // internal index -> public index, -1 if outside K_Nu
    const int k = wavenum(i, N);
    if (k >= Nu / 2 || k <= -(Nu / 2)) return -1;
    return k >= 0 ? k : k + Nu;
}
template <typename T>
__global__ void to_internal2d_kernel(const cx<T>* __restrict__ pub, cx<T>* __restrict__ in, int N, int Nu, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2, Hu = Nu / 2;
    const int iy = (int)(idx % H);
    const long row = idx / H;  // (plane, ix)
    const int ix = (int)(row % N);
    const long pl = row / N;
    const int jx = embed_index2d(ix, N, Nu);
    cx<T> v = mk<T>(0, 0);
    if (jx >= 0 && iy < Hu) v = pub[(pl * Nu + jx) * (Hu + 1) + iy];
    in[idx] = v;
}
template <typename T>
__global__ void to_public2d_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ pub, int N, int Nu, long total_pub) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total_pub) return;
    const int H = N / 2, Hu = Nu / 2;
    const int iy = (int)(idx % (Hu + 1));
    const long row = idx / (Hu + 1);
    const int jx = (int)(row % Nu);
    const long pl = row / Nu;
    cx<T> v = mk<T>(0, 0);
    if (iy != Hu && jx != Hu) v = in[(pl * N + (jx < Hu ? jx : jx - Nu + N)) * H + iy];
    pub[idx] = v;
}

// W: [batch][2][Nu][Nu] full complex unnormalised spectra on the user's grid -> U internal, scaled, Nyquist lines zeroed,
// Leray-projected (k != 0)
template <typename T>
__global__ void init_project2d_kernel(const cx<T>* __restrict__ W, cx<T>* __restrict__ U, int N, int Nu, long total, T scale) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2;
    const int iy = (int)(idx % H);
    const int ix = (int)((idx / H) % N);
    const long b = idx / ((long)H * N);
    const long plane = (long)N * H, sq = (long)Nu * Nu;
    const int jx = embed_index2d(ix, N, Nu);
    const bool nyq = jx < 0 || iy >= Nu / 2;
    cx<T> u[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) u[c] = nyq ? mk<T>(0, 0) : scale * W[(b * 2 + c) * sq + (long)jx * Nu + iy];
    const int kxi = wavenum(ix, N);
    const int k2i = kxi * kxi + iy * iy;
    if (!nyq && k2i > 0) {
        const T kx = (T)kxi, ky = (T)iy, ik2 = (T)1 / (T)k2i;
        const cx<T> ku = mk<T>((kx * u[0].x + ky * u[1].x) * ik2, (kx * u[0].y + ky * u[1].y) * ik2);
        u[0] = mk<T>(u[0].x - kx * ku.x, u[0].y - kx * ku.y);
        u[1] = mk<T>(u[1].x - ky * ku.x, u[1].y - ky * ku.y);
    }
    U[(b * 2) * plane + (long)ix * H + iy] = u[0];
    U[(b * 2 + 1) * plane + (long)ix * H + iy] = u[1];
}

// U internal -> W full complex Hermitian spectrum on the user's Nu grid (ky < 0 from conj of (-k))
template <typename T>
__global__ void expand_hermitian2d_kernel(const cx<T>* __restrict__ U, cx<T>* __restrict__ W, int N, int Nu, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2, Hu = Nu / 2;
    const int jy = (int)(idx % Nu);
    const int jx = (int)((idx / Nu) % Nu);
    const long pl = idx / ((long)Nu * Nu);
    const long plane = (long)N * H;
    cx<T> v = mk<T>(0, 0);
    if (jx != Hu && jy != Hu) {
        const int kx = jx < Hu ? jx : jx - Nu, ky = jy < Hu ? jy : jy - Nu;
        if (ky >= 0) v = U[pl * plane + (long)(kx >= 0 ? kx : kx + N) * H + ky];
        else v = conj(U[pl * plane + (long)(kx > 0 ? N - kx : -kx) * H - ky]);
    }
    W[idx] = v;
}

// ring spectra: E[b][K] += w/2 |u_hat|^2 (ENS: |kx u2 - ky u1|^2), K = floor(|k| + 1/2); grid = (chunks, batch)
template <typename T, bool ENS>
__global__ void spectrum2d_kernel(const cx<T>* __restrict__ U, double* __restrict__ E, int N, int nbins) {
    extern __shared__ double bins[];
    for (int i = threadIdx.x; i < nbins; i += blockDim.x) bins[i] = 0.0;
    __syncthreads();
    const int H = N / 2;
    const long plane = (long)N * H;
    const long b = blockIdx.y;
    const cx<T>* u = U + b * 2 * plane;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < plane; idx += (long)gridDim.x * blockDim.x) {
        const int iy = (int)(idx % H), ix = (int)(idx / H);
        if (ix == N / 2) continue;
        const double kx = wavenum(ix, N), ky = iy;
        const int bin = (int)floor(sqrt(kx * kx + ky * ky) + 0.5);
        if (bin >= nbins) continue;
        const cx<T> a = u[idx], c = u[plane + idx];
        double e;
        if constexpr (ENS) {
            const double wr = kx * (double)c.x - ky * (double)a.x, wi = kx * (double)c.y - ky * (double)a.y;
            e = wr * wr + wi * wi;
        } else {
            e = (double)a.x * a.x + (double)a.y * a.y + (double)c.x * c.x + (double)c.y * c.y;
        }
        atomicAdd(&bins[bin], (iy == 0 ? 0.5 : 1.0) * e);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += blockDim.x)
        if (bins[i] != 0.0) atomicAdd(&E[b * nbins + i], bins[i]);
}

}  // namespace ns
