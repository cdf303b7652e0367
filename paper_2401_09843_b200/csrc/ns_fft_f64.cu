// fp64 instantiation of the FFT pass kernels.
#include "ns_fft_impl.cuh"
namespace ns {
NS_INSTANTIATE_FFT(double)
bool fft_supported(int L) {
    int R1 = 0, R2 = 0;
    fft_split(L, &R1, &R2);
    return R1 != 0;
}
int z_fused_output_scale(int L) { return (L == 64 || L == 128 || L == 256) ? zp_output_scale() : 1; }
#define NS_SPLIT_CASE(LL) case LL: *R1 = Split<LL>::R1; *R2 = Split<LL>::R2; break;
void fft_split(int L, int* R1, int* R2) {
    switch (L) {
        NS_SPLIT_CASE(8) NS_SPLIT_CASE(16) NS_SPLIT_CASE(32) NS_SPLIT_CASE(64) NS_SPLIT_CASE(128) NS_SPLIT_CASE(256)
        NS_SPLIT_CASE(24) NS_SPLIT_CASE(48) NS_SPLIT_CASE(96) NS_SPLIT_CASE(192)
        NS_SPLIT_CASE(40) NS_SPLIT_CASE(80) NS_SPLIT_CASE(160) NS_SPLIT_CASE(320)
        NS_SPLIT_CASE(56) NS_SPLIT_CASE(112) NS_SPLIT_CASE(224)
        NS_SPLIT_CASE(120) NS_SPLIT_CASE(240)
        default: *R1 = 0; *R2 = 0;
    }
}
}  // namespace ns
