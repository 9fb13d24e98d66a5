// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_64() { return Launch<8, 8>::ops(); }
FftOps ops_72() { return Launch<6, 12>::ops(); }
FftOps ops_80() { return Launch<8, 10>::ops(); }
}  // namespace bsefft
