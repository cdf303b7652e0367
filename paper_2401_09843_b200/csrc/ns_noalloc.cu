// ns_noalloc.cu -- the allocation-free entry point of include/ns_noalloc.h: the energy spectrum (reading A14) of a
// caller-held spectral state, its bins accumulated in a file-scope static __device__ scratch array.  No cudaMalloc / cudaFree and
// no allocating library call anywhere in this file.  Self-contained: it shares no state with the solver handles of ns_solver.cu.
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/ns_noalloc.h"
#include "cx.cuh"

using namespace ns;

// The scratch: batch * nbins partial sums.  Resident on every GPU that loads the library, from load until exit.
// In HOST code this name is a host-side stand-in, not a device address: only the pointer cudaGetSymbolAddress returns (per device)
// may be handed to a kernel.
static __device__ __align__(256) double g_noalloc_bins[NS_NOALLOC_MAX_VALUES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
double* g_scratch_addr[MAX_DEVICES] = {};   // device address of g_noalloc_bins, per device ordinal (resolved once)

// set-up, once per device, with that device current
cudaError_t scratch_address(int dev, double** out) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (g_scratch_addr[dev] == nullptr) {
        double* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_bins);
        if (e != cudaSuccess) return e;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

__global__ void noalloc_clear_kernel(double* __restrict__ bins, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) bins[i] = 0.0;
}

// E[b][K] += w/2 |u_hat|^2, K = floor(|k| + 1/2), over the public layout [batch][3][N][N][N/2+1]; grid = (chunks, batch);
// dynamic shared memory: nbins doubles (block-local bins, then one atomic per non-empty bin and block into the scratch)
template <typename T>
__global__ void __launch_bounds__(256)
noalloc_spectrum_kernel(const cx<T>* __restrict__ U, double* __restrict__ bins_g, int N, int nbins) {
    extern __shared__ double bins[];
    for (int i = threadIdx.x; i < nbins; i += blockDim.x) bins[i] = 0.0;
    __syncthreads();
    const int Hp = N / 2 + 1;
    const long plane = (long)N * N * Hp;
    const long b = blockIdx.y;
    const cx<T>* u = U + b * 3 * plane;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < plane; idx += (long)gridDim.x * blockDim.x) {
        const int iz = (int)(idx % Hp), iy = (int)((idx / Hp) % N), ix = (int)(idx / ((long)Hp * N));
        if (ix == N / 2 || iy == N / 2 || iz == N / 2) continue;      // Nyquist planes carry nothing (reading A3)
        const double kx = ix < N / 2 ? ix : ix - N, ky = iy < N / 2 ? iy : iy - N, kz = iz;
        const int bin = (int)floor(sqrt(kx * kx + ky * ky + kz * kz) + 0.5);
        if (bin >= nbins) continue;
        double e = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const cx<T> v = u[c * plane + idx];
            e += (double)v.x * (double)v.x + (double)v.y * (double)v.y;
        }
        atomicAdd(&bins[bin], (iz == 0 ? 0.5 : 1.0) * e);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += blockDim.x)
        if (bins[i] != 0.0) atomicAdd(&bins_g[b * nbins + i], bins[i]);
}

__global__ void noalloc_copy_kernel(const double* __restrict__ bins, double* __restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = bins[i];
}

int fail(char* errbuf, int errbuf_len, int code, const char* msg) {
    if (errbuf && errbuf_len > 0) snprintf(errbuf, (size_t)errbuf_len, "%s", msg);
    return code;
}

}  // namespace

extern "C" int ns_noalloc_energy_spectrum(const void* u_hat_dev, int N, int batch, ns_dtype dtype, int nbins, double* E_out,
                                          ns_memspace out_ms, void* cuda_stream, char* errbuf, int errbuf_len) {
    char msg[256];
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (!u_hat_dev || !E_out) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "u_hat_dev or E_out is NULL");
    if (dtype != NS_F64 && dtype != NS_F32) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "unknown dtype");
    if (out_ms != NS_HOST && out_ms != NS_DEVICE) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "unknown memspace for E_out");
    if (N < 2 || N > 4096 || (N % 2) != 0) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "N must be even with 2 <= N <= 4096");
    if (batch < 1 || batch > 65535) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "batch must be in [1, 65535]");
    if (nbins < 1 || nbins > 4096) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "nbins must be in [1, 4096]");
    if ((long)batch * nbins > NS_NOALLOC_MAX_VALUES) {
        snprintf(msg, sizeof msg, "batch * nbins = %ld exceeds the static scratch of %d doubles (NS_NOALLOC_MAX_VALUES): split the batch",
                 (long)batch * nbins, NS_NOALLOC_MAX_VALUES);
        return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, msg);
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        snprintf(msg, sizeof msg, "no usable CUDA device (no CPU fallback): %s", cudaGetErrorString(e));
        return fail(errbuf, errbuf_len, NS_ERR_CUDA, msg);
    }
    if (dev < 0 || dev >= MAX_DEVICES) return fail(errbuf, errbuf_len, NS_ERR_INVALID_ARG, "device ordinal beyond 63");
    double* scratch = nullptr;
    if ((e = scratch_address(dev, &scratch)) != cudaSuccess) {
        cudaGetLastError();
        snprintf(msg, sizeof msg, "cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
        return fail(errbuf, errbuf_len, NS_ERR_CUDA, msg);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n = batch * nbins;
    const long plane = (long)N * N * (N / 2 + 1);
    long chunks = (plane + 256L * 16 - 1) / (256L * 16);
    if (chunks > 1024) chunks = 1024;
    // the array keeps the last call's contents: clear what this call accumulates into
    noalloc_clear_kernel<<<(n + 255) / 256, 256, 0, st>>>(scratch, n);
    const size_t smem = (size_t)nbins * sizeof(double);      // <= 32 KB: no attribute needed
    if (dtype == NS_F64)
        noalloc_spectrum_kernel<double><<<dim3((unsigned)chunks, (unsigned)batch), 256, smem, st>>>((const cx<double>*)u_hat_dev, scratch, N, nbins);
    else
        noalloc_spectrum_kernel<float><<<dim3((unsigned)chunks, (unsigned)batch), 256, smem, st>>>((const cx<float>*)u_hat_dev, scratch, N, nbins);
    if (out_ms == NS_DEVICE) {
        noalloc_copy_kernel<<<(n + 255) / 256, 256, 0, st>>>(scratch, E_out, n);
    } else {
        e = cudaMemcpyAsync(E_out, scratch, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) {
            snprintf(msg, sizeof msg, "copy to host: %s", cudaGetErrorString(e));
            return fail(errbuf, errbuf_len, NS_ERR_CUDA, msg);
        }
    }
    if ((e = cudaGetLastError()) != cudaSuccess) {
        snprintf(msg, sizeof msg, "kernel launch: %s", cudaGetErrorString(e));
        return fail(errbuf, errbuf_len, NS_ERR_CUDA, msg);
    }
    return NS_OK;
}
