// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_160() { return Launch<10, 16>::ops(); }
}  // namespace bsefft
