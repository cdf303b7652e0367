// fp64 instantiation of the FFT pass kernels.
#include "ns_fft_impl.cuh"
namespace ns {
NS_INSTANTIATE_FFT(double)
bool fft_supported(int L) {
    return L == 8 || L == 16 || L == 32 || L == 64 || L == 128 || L == 256 || L == 24 || L == 48 || L == 96 || L == 192;
}
int z_fused_output_scale(int L) { return (L == 64 || L == 128 || L == 256) ? zp_output_scale() : 1; }
void fft_split(int L, int* R1, int* R2) {
    switch (L) {
        case 8: *R1 = Split<8>::R1; *R2 = Split<8>::R2; break;
        case 16: *R1 = Split<16>::R1; *R2 = Split<16>::R2; break;
        case 32: *R1 = Split<32>::R1; *R2 = Split<32>::R2; break;
        case 64: *R1 = Split<64>::R1; *R2 = Split<64>::R2; break;
        case 128: *R1 = Split<128>::R1; *R2 = Split<128>::R2; break;
        case 256: *R1 = Split<256>::R1; *R2 = Split<256>::R2; break;
        case 24: *R1 = Split<24>::R1; *R2 = Split<24>::R2; break;
        case 48: *R1 = Split<48>::R1; *R2 = Split<48>::R2; break;
        case 96: *R1 = Split<96>::R1; *R2 = Split<96>::R2; break;
        case 192: *R1 = Split<192>::R1; *R2 = Split<192>::R2; break;
        default: *R1 = 0; *R2 = 0;
    }
}
}  // namespace ns
