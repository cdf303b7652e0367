// fp64 instantiation of the FFT pass kernels for the sizes N = 3, 5, 7, 15 times 2^a.
#define NS_FAMILY_SMOOTH
#include "ns_fft_impl.cuh"
namespace ns {
NS_INSTANTIATE_FFT(double)
}  // namespace ns
