// fp64 instantiation of the FFT pass kernels.
#include "ns_fft_impl.cuh"
namespace ns {
NS_INSTANTIATE_FFT(double)
bool fft_supported(int L) { return L == 8 || L == 16 || L == 32 || L == 64 || L == 128 || L == 256; }
}  // namespace ns
