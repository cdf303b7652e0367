// fp32 instantiation of the FFT pass kernels.
#include "ns_fft_impl.cuh"
namespace ns {
NS_INSTANTIATE_FFT(float)
}  // namespace ns
