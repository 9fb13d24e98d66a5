// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_96() { return Launch<8, 12>::ops(); }
FftOps ops_100() { return Launch<10, 10>::ops(); }
}  // namespace bsefft
