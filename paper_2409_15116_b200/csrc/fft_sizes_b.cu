// Instantiations of the two-pass FFT kernels (fft_kernels.cuh) for a group of grid edges n = R1 * R2.
#include "fft_kernels.cuh"
namespace bsefft {
FftOps ops_36() { return Launch<6, 6>::ops(); }
FftOps ops_40() { return Launch<5, 8>::ops(); }
FftOps ops_48() { return Launch<6, 8>::ops(); }
FftOps ops_60() { return Launch<6, 10>::ops(); }
}  // namespace bsefft
