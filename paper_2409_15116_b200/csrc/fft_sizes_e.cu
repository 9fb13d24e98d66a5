// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_120() { return Launch<10, 12>::ops(); }
FftOps ops_128() { return Launch<8, 16>::ops(); }
}  // namespace bsefft
