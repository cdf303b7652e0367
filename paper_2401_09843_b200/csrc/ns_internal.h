// ns_internal.h -- launcher interface between the host-side solver (ns_solver.cu) and the FFT kernel
// translation units (ns_fft_f64.cu / ns_fft_f32.cu).  Product path only.
#pragma once
#include <cuda_runtime.h>

#include "cx.cuh"

namespace ns {

// number of flux components carried through a4-a7: the five trace-free combinations of kernels_z.cuh
constexpr int NS_NFLUX = 5;

// Twiddle tables, laid out so that the lanes of a warp read consecutive entries:
//   twA[r1 * R2 + n2] = twB[n2 * R1 + r1] = exp(+2 pi i r1 n2 / L)      (inter-stage twiddles, L = R1 R2)
//   w3a[n] = exp(+2 pi i n / (3L)),  w3b[n] = exp(+2 pi i 2n / (3L)),  n < L   (pruned radix-3 twiddles)
template <typename T>
struct Twiddles {
    const cx<T>* twA;
    const cx<T>* twB;
    const cx<T>* w3a;
    const cx<T>* w3b;
    // table of the 16-values-per-lane z kernel (kernels_zpair.cuh), G = L/16 (L >= 64 only):
    //   z16[r1*G + t] = w_L^{r1 t},  r1 < 16, t < G
    const cx<T>* z16;
    // gN[j] = exp(+2 pi i j / N), j < N = 2L: the unpadded N-grid transforms (generic_fft_kernel)
    const cx<T>* gN;
};
// number of complex entries of the table block and its host-side construction (long double arguments);
// make_twiddles() returns the views into a device copy of that block
inline size_t twiddle_table_len(int L) { return (size_t)10 * L; }
// register-stage split L = R1 x R2 used by the kernels (needed by the host to build twA / twB)
void fft_split(int L, int* R1, int* R2);

// true if the pruned transform of half-length L = N/2 is supported
bool fft_supported(int L);

// columns per tile of the strided passes (128 bytes per row)
template <typename T> constexpr int tile_cols() { return 128 / (2 * (int)sizeof(T)); }

// Output of a strided-axis pass split over several destinations (multi-device solver): output row n is stored to row
// n % rows of the array at peer[n / rows]; `peer` is a table IN DEVICE MEMORY of the launching device holding the destination
// base addresses (device pointers, possibly of other devices with peer access enabled); `base` = peer[0], the address the
// plain-output offsets are taken against.
struct ColSplit {
    int rows;
    const unsigned long long* peer;
};

// Strided-axis passes.  `ncols` contiguous columns per slab (multiple of tile_cols<T>()), `nslabs` slabs.
// Input rows [0,2L) -> output rows [0,3L) (inverse) or the reverse (forward, output multiplied by scale).
template <typename T>
cudaError_t launch_col_inv(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, Twiddles<T> tw, const ColSplit* split = nullptr);
template <typename T>
cudaError_t launch_col_fwd(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,
                           long istride, long ostride, long in_slab, long out_slab, T scale, Twiddles<T> tw, const ColSplit* split = nullptr);
// fused a3+a4 (kernels_zpair.cuh; kernels_zfused.cuh for L <= 32): in [batch][3][MM][L] -> out [batch][NS_NFLUX][MM][L];
// persistent grid sized from num_sms (the SM count of the solver's device) and the CTAs per SM.  umax2 may be NULL.
template <typename T>
cudaError_t launch_z_fused(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long MM, long batch,
                           unsigned long long* umax2, Twiddles<T> tw);

// the same three launchers per kernel family (ns_fft_impl.cuh): L = 2^a / L = 3, 5, 7, 15 times 2^a
#define NS_DECL_FAMILY(FAM)                                                                                                        \
    template <typename T>                                                                                                          \
    cudaError_t launch_col_inv_##FAM(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,    \
                                     long istride, long ostride, long in_slab, long out_slab, Twiddles<T> tw,                     \
                                     const ColSplit* split);                                                                       \
    template <typename T>                                                                                                          \
    cudaError_t launch_col_fwd_##FAM(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long ncols, long nslabs,    \
                                     long istride, long ostride, long in_slab, long out_slab, T scale, Twiddles<T> tw,            \
                                     const ColSplit* split);                                                                       \
    template <typename T>                                                                                                          \
    cudaError_t launch_z_fused_##FAM(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long MM, long batch,        \
                                     unsigned long long* umax2, Twiddles<T> tw);
NS_DECL_FAMILY(pow2)
NS_DECL_FAMILY(smooth)
#undef NS_DECL_FAMILY

// factor carried by the output of launch_z_fused / launch_y2d relative to the plain unnormalised transform (the kernels of
// kernels_zpair.cuh fold the 1/2 of their Hermitian split into the normalisation of the spectral kernel)
int z_fused_output_scale(int L);

// fused contiguous-axis kernel of the 2-D solver (kernels_y2d.cuh), L in {64, 128, 256}: in [batch][2][M][L] -> out [batch][2][M][L]
template <typename T>
cudaError_t launch_y2d(cudaStream_t st, int num_sms, int L, const cx<T>* in, cx<T>* out, long M, long batch,
                       unsigned long long* umax2, Twiddles<T> tw);

}  // namespace ns
