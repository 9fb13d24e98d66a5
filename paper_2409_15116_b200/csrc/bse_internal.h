// Internal declarations shared by the CUDA translation units of libbse_b200.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/bse.h"

#define BSE_MAX_RADIX_PASSES 12

// ---------------------------------------------------------------------------------------------------------
// FFT plan: one length n for all three axes (cubic grid).  In-place decimation-in-frequency passes over
// shared memory; after all passes position p of a line holds frequency rev[p]  (pos[rev[p]] = p).
struct FftPlan {
    int n = 0;           // points per axis
    int ld = 0;          // padded line length in shared memory (complex elements), n + 1
    int npass = 0;
    int radix[BSE_MAX_RADIX_PASSES];
    int R = 0;           // floor(sqrt(msq_max))
    int W = 0;           // kept m3 columns in the plane pass: m3 = 0..R  -> W = R + 1
    int NS = 0;          // number of half sticks (m2, m3): m3 > 0 or (m3 == 0 and m2 >= 0), inside the disk
    long long npw_h = 0;
    // device tables
    double2 *tw = nullptr;        // [n]   exp(-2 pi i t / n)
    int *pos = nullptr;           // [n]   position of frequency k after the DIF passes
    int *rev = nullptr;           // [n]   frequency held at position p
    int *kk_fwd = nullptr;        // [2][W] column slot of (row parity, m3) in the forward plane pass
    int *kk_inv = nullptr;        // [2][W] same for the inverse plane pass
    int *stick_off_fwd = nullptr; // [NS]  smem offset of stick (m2,m3) after the forward plane pass
    int *stick_off_inv = nullptr; // [NS]  smem offset where stick (m2,m3) is loaded in the inverse plane pass
    int *stick_off_mir = nullptr; // [NS]  smem offset of the mirrored (-m2, 0) entry, -1 if none
    int *fmap = nullptr;          // [NS][n] forward stick pass: (stick, position t) -> index in H or -1
    int *imap = nullptr;          // [NS][n] inverse stick pass: (stick, t = m1 mod n) -> h, -1 (zero), or -2-h (conj)
    double *vc12 = nullptr;       // [npw_h] sqrt(4 pi)/|G|, 0 at G = 0
    double *vc12n = nullptr;      // [npw_h] vc12 / N   (forward FFT normalisation folded in)
};

// ---------------------------------------------------------------------------------------------------------
struct bse_handle {
    int n = 0;
    long long N = 0;
    double L = 0, Omega = 0, dV = 0, ecut = 0, eta = 0;
    int msq_max = 0;
    int Nv = 0, Npdep = 0;
    unsigned flags = 0;
    cudaStream_t stream = nullptr;
    const double *u = nullptr;       // device [Nv][N]
    const double *phi = nullptr;     // device [Npdep][2 Npw_h]
    double *u_owned = nullptr, *phi_owned = nullptr;
    std::vector<int> mill;           // host [npw_h][3]
    FftPlan fft;
    double *f2 = nullptr;            // device [Npdep]  2 lambda/(1-lambda)
    // screen / pair list
    double *Mmat = nullptr;          // device [Nv][Nv]  sum_r u_v^2 u_w^2
    int *rowcnt = nullptr, *rowptr = nullptr;   // device [Nv], [Nv+1]
    int *pid = nullptr;              // device [Nv][Nv] pair index or -1 (v <= w)
    int2 *pairs = nullptr;           // device [P]
    int *adj_ptr = nullptr;          // device [Nv+1] directed adjacency (both directions)
    int2 *adj = nullptr;             // device [nadj] (w, pair index), sorted by w within a row
    long long P = -1, nadj = 0;
    bool built = false;
    // tau store
    double *tau_r = nullptr;         // [P][N]
    double2 *tau_g = nullptr;        // [P][npw_h]
    size_t tau_bytes = 0;            // capacity of the store (grow-only)
    // workspaces (sized for a pair batch)
    long long Pb = 0;                // pair-batch capacity
    double2 *Z = nullptr;            // [Pb][n][NS]
    double2 *X = nullptr;            // [Pb][npw_h]
    double2 *T = nullptr;            // [Pb][npw_h]
    double *Dm = nullptr;            // [Pb][Npdep]
    double *part = nullptr;          // split-K partials
    size_t part_bytes = 0;
    double *Sov = nullptr;           // [B*Nv][Nv] P_c overlaps
    size_t Sov_elems = 0;
    double *tau_batch = nullptr;     // [Pb][N] scratch for PW / STREAM modes
    double *a_dev = nullptr, *out_dev = nullptr;   // staging for the host-pointer entry point
    size_t a_dev_bytes = 0;
    // profiling
    bool prof = false;
    double st_ms[BSE_ST_COUNT] = {0};
    long long st_launch[BSE_ST_COUNT] = {0};
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
};

void bse_set_error(const std::string &msg);
int bse_cuda_fail(cudaError_t e, const char *what);

#define BSE_CUDA(call)                                                        \
    do {                                                                      \
        cudaError_t e__ = (call);                                             \
        if (e__ != cudaSuccess) return bse_cuda_fail(e__, #call);             \
    } while (0)

// ---- kernels' host launchers (each returns a BSE_* status) -------------------------------------------------
// fft_kernels.cu
int bse_fft_smem_bytes_plane(const FftPlan &pl);
int bse_launch_fwd_plane(const FftPlan &pl, const double *fields, const int2 *pairs, long long p0, int count,
                         long long N, double2 *Z, cudaStream_t s);
int bse_launch_fwd_stick(const FftPlan &pl, const double2 *Z, int count, double2 *X, const double *scale,
                         cudaStream_t s);
int bse_launch_inv_stick(const FftPlan &pl, const double2 *T, int count, double2 *Z, cudaStream_t s);
int bse_launch_inv_plane(const FftPlan &pl, const double2 *Z, int count, long long N, double *out, cudaStream_t s);

// gemm_dmma.cu
enum { EPI_PARTIAL = 0, EPI_TAU = 1, EPI_SUB = 2 };
// C[M][N] (+)= A[M][K] * B[N][K]^T, split-K partials into `part` then reduced: C = alpha * colscale[n] * sum
int bse_gemm_dot(const double *A, long long lda, const double *B, long long ldb, int M, int N, long long K,
                 bool squareA, bool squareB, double *part, size_t part_bytes, double *C, long long ldc,
                 double alpha, const double *colscale, cudaStream_t s);
// NN form: acc = A[M][K] * B[K][N];  EPI_TAU: C = colscale2[n>>1] * (Xin + acc);  EPI_SUB: C = C - acc
int bse_gemm_nn(const double *A, long long lda, const double *B, long long ldb, int M, long long N, int K,
                int epi, const double *Xin, const double *colscale2, double *C, long long ldc, cudaStream_t s);

// k1x_kernels.cu
int bse_launch_pairlist(bse_handle *h);                 // M -> rowcnt,rowptr,pid,pairs (count only if pairs==nullptr)
int bse_launch_accumulate(bse_handle *h, const double *tau, long long p_first, long long p_count,
                          const double *a, double *acc, int B, bool zero_init);
