// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_108() { return Launch<9, 12>::ops(); }
}  // namespace bsefft
