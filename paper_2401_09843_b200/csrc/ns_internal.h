// ns_internal.h -- launcher interface between the host-side solver (ns_solver.cu) and the FFT kernel
// translation units (ns_fft_f64.cu / ns_fft_f32.cu).  Product path only.
#pragma once
#include <cuda_runtime.h>

#include "cx.cuh"

namespace ns {

template <typename T>
struct Twiddles {
    const cx<T>* tw3;  // [2L]  exp(+2 pi i n / (3L))
    const cx<T>* twL;  // [L]   exp(+2 pi i n / L)
};

// true if the pruned transform of half-length L = N/2 is supported
bool fft_supported(int L);

// columns per tile of the strided passes (128 bytes per row)
template <typename T> constexpr int tile_cols() { return 128 / (2 * (int)sizeof(T)); }

// Strided-axis passes.  `ncols` contiguous columns per slab (multiple of tile_cols<T>()), `nslabs` slabs.
// Input rows [0,2L) -> output rows [0,3L) (inverse) or the reverse (forward, output multiplied by scale).
template <typename T>
cudaError_t launch_col_inv(cudaStream_t st, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, Twiddles<T> tw);
template <typename T>
cudaError_t launch_col_fwd(cudaStream_t st, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, T scale, Twiddles<T> tw);
// z passes.  in/out layouts documented in kernels_z.cuh.  umax2 may be NULL.
template <typename T>
cudaError_t launch_z_inv_prod(cudaStream_t st, int L, const cx<T>* in, T* phys, long MM, long batch,
                              unsigned long long* umax2, Twiddles<T> tw);
template <typename T>
cudaError_t launch_z_fwd(cudaStream_t st, int L, const T* phys, cx<T>* out, long MM, long batch, Twiddles<T> tw);

}  // namespace ns
