// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_12() { return Launch<3, 4>::ops(); }
FftOps ops_16() { return Launch<4, 4>::ops(); }
FftOps ops_20() { return Launch<5, 4>::ops(); }
FftOps ops_24() { return Launch<4, 6>::ops(); }
FftOps ops_30() { return Launch<5, 6>::ops(); }
FftOps ops_32() { return Launch<4, 8>::ops(); }
}  // namespace bsefft
