// FP64 peak probe: the roofline denominators for the dense contractions (a1, a5, a7, a11) are measured, not
// assumed.  DMMA chain: 8 independent mma.sync.m8n8k4.f64 accumulators per warp; DFMA chain: 8 independent
// fma.rn.f64 chains per thread.  Both saturate every SM (148 x 4 CTAs x 256 threads).
#include "bse_internal.h"

namespace {

__global__ void __launch_bounds__(256) dmma_chain_kernel(double *out, int iters, double a0, double b0) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = a0 + threadIdx.x * 1e-9, b = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) dfma_chain_kernel(double *out, int iters, double a0, double b0) {
    double c[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i] = i;
    const double a = a0 + threadIdx.x * 1e-9, b = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) c[i] = fma(c[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i];
    if (s == 123.456) out[0] = s;
}

}  // namespace

extern "C" int bse_probe_fp64_peak(double *dmma_tflops, double *dfma_tflops, void *stream) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        bse_set_error("no CUDA device");
        return BSE_ECUDA;
    }
    cudaStream_t s = (cudaStream_t)stream;
    cudaDeviceProp prop;
    BSE_CUDA(cudaGetDeviceProperties(&prop, 0));
    const int blocks = prop.multiProcessorCount * 4, threads = 256, iters = 4096;
    double *d = nullptr;
    BSE_CUDA(cudaMalloc(&d, 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best_mma = 1e30f, best_fma = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        float ms;
        cudaEventRecord(e0, s);
        dmma_chain_kernel<<<blocks, threads, 0, s>>>(d, iters, 1.0000001, 0.5);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_mma) best_mma = ms;
        cudaEventRecord(e0, s);
        dfma_chain_kernel<<<blocks, threads, 0, s>>>(d, iters, 0.9999999, 1e-3);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_fma) best_fma = ms;
    }
    BSE_CUDA(cudaGetLastError());
    const double warps = (double)blocks * threads / 32.0;
    if (dmma_tflops) *dmma_tflops = warps * iters * 8.0 * (2.0 * 8 * 8 * 4) / (best_mma * 1e-3) / 1e12;
    if (dfma_tflops) *dfma_tflops = (double)blocks * threads * iters * 8.0 * 2.0 / (best_fma * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    return BSE_OK;
}
