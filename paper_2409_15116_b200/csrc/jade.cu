// JADE localisation of the occupied orbitals (eq. 12-15): produces the U that bse_rotate and
// the screen of eq. 16 presuppose.
//   A^(k)_vw = <psi_v| M^(k) |psi_w>, M^(1..6) = cos / sin (2 pi x / L), ... (eq. 13, 15)   weighted copy + split-K DMMA GEMM
//   U_0 = eigenvectors of A^(1), by the same Jacobi machinery run on A^(1) alone, columns by ascending eigenvalue
//   sweeps of concurrent Givens rotations over round-robin rounds of disjoint pairs (readings J1-J4 of DESIGN.md): all
//   angles of a round from the matrices as they stand, then A^(k) <- R^T A^(k) R, V <- V R
// The paper accumulates the rotations of a concurrent loop into one N_occ^3 matrix product (its A100 / cuBLAS design); on B200
// the seven N_v x N_v matrices (56 MB at N_v = 1024) live in the 126 MB L2, so a round is applied directly as row and column
// pair updates (O(N_v^2) per round instead of O(N_v^3)), and one whole sweep is replayed as a CUDA graph.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>
#include <vector>

#include "bse_internal.h"

namespace {

// round-robin tournament (reading J2): pair k of round r with m = Nv rounded up to even
__device__ __forceinline__ void rr_pair(int r, int k, int m, int &p, int &q) {
    int a, b;
    if (k == 0) { a = m - 1; b = r; }
    else { a = (r + k) % (m - 1); b = (r - k + (m - 1)) % (m - 1); }
    p = a < b ? a : b;
    q = a < b ? b : a;
}

// wbuf[v][j] = psi[v][k0 + j] * M(k0 + j), M = cos or sin of 2 pi i_axis / n
__global__ void __launch_bounds__(256)
jade_weight_kernel(const double *__restrict__ psi, long long N, int n, long long k0, long long kc, int axis, int use_sin,
                   const double *__restrict__ cs_tab /* [2][n]: cos, sin of 2 pi i / n */, double *__restrict__ wbuf) {
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= kc) return;
    const long long k = k0 + j;
    const int i3 = (int)(k % n), i2 = (int)((k / n) % n), i1 = (int)(k / ((long long)n * n));
    const int idx = axis == 0 ? i1 : (axis == 1 ? i2 : i3);
    const double w = cs_tab[(use_sin ? n : 0) + idx];
    const long long v = blockIdx.y;
    wbuf[v * kc + j] = psi[v * N + k] * w;
}

// angles of one round: cs[k] = (c, s) for pair k; smax <- max |s| (bits of a non-negative double compare as integers)
__global__ void __launch_bounds__(256)
jade_angles_kernel(const double *__restrict__ A, int K, int Nv, int m, int r, double2 *__restrict__ cs,
                   unsigned long long *__restrict__ smax) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m / 2) return;
    int p, q;
    rr_pair(r, k, m, p, q);
    if (q >= Nv) { cs[k] = make_double2(1.0, 0.0); return; }      // pair with the padding index: no rotation
    double g11 = 0.0, g22 = 0.0, g12 = 0.0;
    for (int n = 0; n < K; ++n) {
        const double *a = A + (long long)n * Nv * Nv;
        const double h1 = a[(long long)p * Nv + p] - a[(long long)q * Nv + q];
        const double h2 = 2.0 * a[(long long)p * Nv + q];
        g11 = fma(h1, h1, g11);
        g22 = fma(h2, h2, g22);
        g12 = fma(h1, h2, g12);
    }
    const double ton = g11 - g22, toff = 2.0 * g12;
    const double theta = 0.5 * atan2(toff, ton + sqrt(ton * ton + toff * toff));
    double s, c;
    sincos(theta, &s, &c);
    cs[k] = make_double2(c, s);
    atomicMax(smax, (unsigned long long)__double_as_longlong(fabs(s)));
}

// columns: X[i][p], X[i][q] <- c X[i][p] + s X[i][q], -s X[i][p] + c X[i][q] for every row i of the K + 1 matrices (A's and V)
__global__ void __launch_bounds__(256)
jade_cols_kernel(double *__restrict__ A, int Kp1, int Nv, int m, int r, const double2 *__restrict__ cs) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m / 2) return;
    int p, q;
    rr_pair(r, k, m, p, q);
    if (q >= Nv) return;
    const double2 t = cs[k];
    double *row = A + ((long long)blockIdx.z * Nv + blockIdx.y) * Nv;
    const double xp = row[p], xq = row[q];
    row[p] = t.x * xp + t.y * xq;
    row[q] = -t.y * xp + t.x * xq;
}

// rows: X[p][j], X[q][j] <- c X[p][j] + s X[q][j], -s X[p][j] + c X[q][j] for every column j of the K matrices A
__global__ void __launch_bounds__(256)
jade_rows_kernel(double *__restrict__ A, int Nv, int m, int r, const double2 *__restrict__ cs) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Nv) return;
    int p, q;
    rr_pair(r, blockIdx.y, m, p, q);
    if (q >= Nv) return;
    const double2 t = cs[blockIdx.y];
    double *a = A + (long long)blockIdx.z * Nv * Nv;
    const double xp = a[(long long)p * Nv + j], xq = a[(long long)q * Nv + j];
    a[(long long)p * Nv + j] = t.x * xp + t.y * xq;
    a[(long long)q * Nv + j] = -t.y * xp + t.x * xq;
}

__global__ void jade_identity_kernel(double *__restrict__ V, int Nv) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < (long long)Nv * Nv) V[i] = (i / Nv == i % Nv) ? 1.0 : 0.0;
}
// dst[i][j] = src[i][perm[j]]
__global__ void jade_permute_cols_kernel(const double *__restrict__ src, const int *__restrict__ perm, double *__restrict__ dst,
                                         int Nv, long long ldd) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (j < Nv) dst[(long long)i * ldd + j] = src[(long long)i * Nv + perm[j]];
}
__global__ void jade_diag_kernel(const double *__restrict__ A, int K, int Nv, double *__restrict__ d) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < K * Nv) d[i] = A[((long long)(i / Nv) * Nv + i % Nv) * Nv + i % Nv];
}
// dst [rows][ldd] <- src [rows][lds] (first cols columns)
__global__ void jade_copy2d_kernel(const double *__restrict__ src, long long lds, double *__restrict__ dst, long long ldd, int cols) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (j < cols) dst[(long long)i * ldd + j] = src[(long long)i * lds + j];
}

struct Jade {
    int Nv, m, K;
    double *A = nullptr;        // [K + 1][Nv][Nv]: the K matrices, then V
    double2 *cs = nullptr;
    unsigned long long *smax = nullptr;
    cudaStream_t s = nullptr;
    cudaGraphExec_t exec[2] = {nullptr, nullptr};   // sweep graphs for K = 1 (eigen-initialisation) and K = 6
};

// one sweep (m - 1 rounds, 3 launches each) on the first K matrices (+ V, always at index Kall)
void enqueue_sweep(const Jade &J, int K, int Kall) {
    const int Nv = J.Nv, m = J.m, half = m / 2;
    double *V = J.A + (long long)Kall * Nv * Nv;
    for (int r = 0; r < m - 1; ++r) {
        jade_angles_kernel<<<(half + 255) / 256, 256, 0, J.s>>>(J.A, K, Nv, m, r, J.cs, J.smax);
        jade_cols_kernel<<<dim3((half + 255) / 256, Nv, K), 256, 0, J.s>>>(J.A, K, Nv, m, r, J.cs);
        jade_cols_kernel<<<dim3((half + 255) / 256, Nv, 1), 256, 0, J.s>>>(V, 1, Nv, m, r, J.cs);
        jade_rows_kernel<<<dim3((Nv + 255) / 256, half, K), 256, 0, J.s>>>(J.A, Nv, m, r, J.cs);
    }
}

// sweeps until max |sin theta| of a sweep < tol; returns the number of sweeps done, or < 0 for a BSE_* error
int run_sweeps(Jade &J, int K, int Kall, double tol, int max_sweeps, int slot) {
    if (!J.exec[slot]) {
        cudaGraph_t g;
        if (cudaStreamBeginCapture(J.s, cudaStreamCaptureModeThreadLocal) != cudaSuccess) return BSE_ECUDA;
        enqueue_sweep(J, K, Kall);
        if (cudaStreamEndCapture(J.s, &g) != cudaSuccess) return BSE_ECUDA;
        if (cudaGraphInstantiate(&J.exec[slot], g, 0) != cudaSuccess) { cudaGraphDestroy(g); return BSE_ECUDA; }
        cudaGraphDestroy(g);
    }
    int done = 0;
    for (; done < max_sweeps;) {
        if (cudaMemsetAsync(J.smax, 0, 8, J.s) != cudaSuccess) return BSE_ECUDA;
        if (cudaGraphLaunch(J.exec[slot], J.s) != cudaSuccess) return BSE_ECUDA;
        unsigned long long bits = 0;
        if (cudaMemcpyAsync(&bits, J.smax, 8, cudaMemcpyDeviceToHost, J.s) != cudaSuccess) return BSE_ECUDA;
        if (cudaStreamSynchronize(J.s) != cudaSuccess) return BSE_ECUDA;
        ++done;
        double smax;
        static_assert(sizeof(double) == sizeof(unsigned long long), "");
        memcpy(&smax, &bits, 8);
        if (smax < tol) break;
    }
    return done;
}

}  // namespace

extern "C" int bse_jade(const int grid[3], const double cell[9], int Nv, const double *psi, double *U, double *psi_loc,
                        double tol, int max_sweeps, int init_eig, int *sweeps, double *spread, void *stream) {
    if (!grid || !cell || !psi || !U || Nv <= 0 || max_sweeps < 0 || !(tol >= 0)) {
        bse_set_error("bse_jade: null pointer or bad size");
        return BSE_EINVAL;
    }
    const int n = grid[0];
    const double L = cell[0];
    if (grid[1] != n || grid[2] != n || n <= 0 || (n & 1) || !(L > 0)) {
        bse_set_error("bse_jade: cubic cells and cubic grids with even n only");
        return BSE_EUNSUPPORTED;
    }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            if (std::fabs(cell[3 * i + j] - (i == j ? L : 0.0)) > 1e-12 * L) {
                bse_set_error("bse_jade: cubic cells only");
                return BSE_EUNSUPPORTED;
            }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        bse_set_error("no CUDA device: this library has no CPU fallback");
        return BSE_ECUDA;
    }
    const long long N = (long long)n * n * n;
    const double dV = L * L * L / (double)N;
    const int K = 6;
    const long long nv2 = (long long)Nv * Nv;
    const long long lds = (Nv + 1) & ~1;
    cudaStream_t user = (cudaStream_t)stream;
    Jade J;
    J.Nv = Nv; J.m = Nv + (Nv & 1); J.K = K;
    cudaEvent_t ev = nullptr;
    double *wbuf = nullptr, *part = nullptr, *tabs = nullptr, *T = nullptr, *Vt = nullptr, *diag = nullptr, *Vp = nullptr;
    int *perm_d = nullptr;
    int rc = BSE_OK, done = 0;
    // chunk of grid points whose weighted copy is formed at a time (<= 1 GB), split-K workspace
    long long kc = std::max<long long>(4096, std::min<long long>(N, ((long long)1 << 27) / Nv)) & ~1LL;
    const size_t part_bytes = std::max<size_t>((size_t)64 << 20, (size_t)nv2 * 8 * 4);
    std::vector<double> tab_h(2 * (size_t)n), diag_h((size_t)K * Nv);
    for (int i = 0; i < n; ++i) {
        const long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)i / (long double)n;
        tab_h[i] = (double)cosl(ang);
        tab_h[n + i] = (double)sinl(ang);
    }
#define JCUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = bse_cuda_fail(e__, #call); goto cleanup; } } while (0)
#define JRC(call) do { rc = (call); if (rc) goto cleanup; } while (0)
    {
        JCUDA(cudaStreamCreateWithFlags(&J.s, cudaStreamNonBlocking));
        JCUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        JCUDA(cudaEventRecord(ev, user));                        // after whatever produced psi on the caller's stream
        JCUDA(cudaStreamWaitEvent(J.s, ev, 0));
        JCUDA(cudaMalloc(&J.A, (size_t)(K + 1) * nv2 * 8));
        JCUDA(cudaMalloc(&J.cs, (size_t)(J.m / 2) * 16));
        JCUDA(cudaMalloc(&J.smax, 8));
        JCUDA(cudaMalloc(&wbuf, (size_t)Nv * kc * 8));
        JCUDA(cudaMalloc(&part, part_bytes));
        JCUDA(cudaMalloc(&tabs, tab_h.size() * 8));
        JCUDA(cudaMalloc(&T, (size_t)Nv * lds * 8));
        JCUDA(cudaMalloc(&Vt, (size_t)Nv * lds * 8));
        JCUDA(cudaMalloc(&Vp, (size_t)Nv * lds * 8));
        JCUDA(cudaMalloc(&diag, (size_t)K * Nv * 8));
        JCUDA(cudaMalloc(&perm_d, (size_t)Nv * 4));
        JCUDA(cudaMemcpyAsync(tabs, tab_h.data(), tab_h.size() * 8, cudaMemcpyHostToDevice, J.s));
        JCUDA(cudaMemsetAsync(T, 0, (size_t)Nv * lds * 8, J.s));         // the padding column of the GEMM operands stays zero
        JCUDA(cudaMemsetAsync(Vt, 0, (size_t)Nv * lds * 8, J.s));
        JCUDA(cudaMemsetAsync(Vp, 0, (size_t)Nv * lds * 8, J.s));
        double *V = J.A + (long long)K * nv2;
        // ---- A^(k) (eq. 15): weighted copy of a chunk of grid points, then the split-K dot GEMM accumulating over the chunks
        for (long long k0 = 0; k0 < N; k0 += kc) {
            const long long c = std::min(kc, N - k0);
            for (int k = 0; k < K; ++k) {
                jade_weight_kernel<<<dim3((unsigned)((c + 255) / 256), Nv), 256, 0, J.s>>>(psi, N, n, k0, c, k / 2, k & 1, tabs, wbuf);
                JCUDA(cudaGetLastError());
                JRC(bse_gemm_dot(wbuf, c, psi + k0, N, Nv, Nv, c, false, false, part, part_bytes, J.A + k * nv2, Nv, dV, nullptr,
                                 J.s, k0 > 0));
            }
        }
        double sumsq = 0.0;
        if (spread) {                                            // sum_k Tr B^(k) = 3 sum_v ||psi_v||^2 because cos^2 + sin^2 = 1
            double *ss = wbuf;                                   // scratch: [Nv][2]
            JRC(bse_launch_row_sumsq(psi, psi, N, Nv, ss, J.s));
            std::vector<double> h2((size_t)2 * Nv);
            JCUDA(cudaMemcpyAsync(h2.data(), ss, h2.size() * 8, cudaMemcpyDeviceToHost, J.s));
            jade_diag_kernel<<<(K * Nv + 255) / 256, 256, 0, J.s>>>(J.A, K, Nv, diag);
            JCUDA(cudaMemcpyAsync(diag_h.data(), diag, diag_h.size() * 8, cudaMemcpyDeviceToHost, J.s));
            JCUDA(cudaStreamSynchronize(J.s));
            for (int v = 0; v < Nv; ++v) sumsq += dV * h2[2 * v];
            double d2 = 0.0;
            for (double x : diag_h) d2 += x * x;
            spread[0] = 3.0 * sumsq - d2;
        }
        jade_identity_kernel<<<(unsigned)((nv2 + 255) / 256), 256, 0, J.s>>>(V, Nv);
        JCUDA(cudaGetLastError());
        if (init_eig) {
            // ---- V_0 = eigenvectors of A^(1): Jacobi sweeps on a copy of A^(1) alone, columns sorted by
            // ascending eigenvalue, then A^(k) <- V_0^T A^(k) V_0 as DMMA GEMMs
            double *A1 = wbuf;                                   // scratch copy (wbuf holds >= Nv * 4096 doubles >= nv2 for Nv <= 4096)
            if ((size_t)nv2 > (size_t)Nv * kc) { bse_set_error("bse_jade: Nv too large for the scratch buffer"); rc = BSE_EUNSUPPORTED; goto cleanup; }
            JCUDA(cudaMemcpyAsync(A1, J.A, (size_t)nv2 * 8, cudaMemcpyDeviceToDevice, J.s));
            Jade J1 = J;
            J1.A = nullptr;
            // the K = 1 problem lives in its own [2][Nv][Nv] buffer: matrix, then V
            JCUDA(cudaMalloc(&J1.A, (size_t)2 * nv2 * 8));
            JCUDA(cudaMemcpyAsync(J1.A, A1, (size_t)nv2 * 8, cudaMemcpyDeviceToDevice, J.s));
            jade_identity_kernel<<<(unsigned)((nv2 + 255) / 256), 256, 0, J.s>>>(J1.A + nv2, Nv);
            J1.exec[0] = J1.exec[1] = nullptr;
            const int d1 = run_sweeps(J1, 1, 1, 1e-15, 100, 0);
            if (J1.exec[0]) cudaGraphExecDestroy(J1.exec[0]);
            if (d1 < 0) { cudaFree(J1.A); rc = d1; bse_set_error("bse_jade: eigen-initialisation failed"); goto cleanup; }
            std::vector<double> ev_h((size_t)Nv);
            jade_diag_kernel<<<(Nv + 255) / 256, 256, 0, J.s>>>(J1.A, 1, Nv, diag);
            cudaMemcpyAsync(ev_h.data(), diag, (size_t)Nv * 8, cudaMemcpyDeviceToHost, J.s);
            cudaStreamSynchronize(J.s);
            std::vector<int> perm((size_t)Nv);
            std::iota(perm.begin(), perm.end(), 0);
            std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return ev_h[a] < ev_h[b]; });
            cudaMemcpyAsync(perm_d, perm.data(), (size_t)Nv * 4, cudaMemcpyHostToDevice, J.s);
            jade_permute_cols_kernel<<<dim3((Nv + 255) / 256, Nv), 256, 0, J.s>>>(J1.A + nv2, perm_d, V, Nv, Nv);
            cudaStreamSynchronize(J.s);
            cudaFree(J1.A);
            JCUDA(cudaGetLastError());
            // padded copies for the GEMM tile loader (16-byte rows), V_0^T
            jade_copy2d_kernel<<<dim3((Nv + 255) / 256, Nv), 256, 0, J.s>>>(V, Nv, Vp, lds, Nv);
            JRC(bse_launch_transpose(V, Nv, Vt, lds, Nv, J.s));
            for (int k = 0; k < K; ++k) {
                jade_copy2d_kernel<<<dim3((Nv + 255) / 256, Nv), 256, 0, J.s>>>(J.A + k * nv2, Nv, T, lds, Nv);
                // W = A V_0  (into wbuf, padded), then A <- V_0^T W
                JRC(bse_gemm_nn(T, lds, Vp, lds, Nv, lds, Nv, EPI_STORE, nullptr, nullptr, wbuf, lds, J.s));
                JRC(bse_gemm_nn(Vt, lds, wbuf, lds, Nv, lds, Nv, EPI_STORE, nullptr, nullptr, T, lds, J.s));
                jade_copy2d_kernel<<<dim3((Nv + 255) / 256, Nv), 256, 0, J.s>>>(T, lds, J.A + k * nv2, Nv, Nv);
            }
            JCUDA(cudaGetLastError());
        }
        // ---- the JADE sweeps
        done = run_sweeps(J, K, K, tol, max_sweeps, 1);
        if (done < 0) { rc = done; bse_set_error("bse_jade: sweep launch failed"); goto cleanup; }
        if (sweeps) *sweeps = done;
        if (spread) {
            jade_diag_kernel<<<(K * Nv + 255) / 256, 256, 0, J.s>>>(J.A, K, Nv, diag);
            JCUDA(cudaMemcpyAsync(diag_h.data(), diag, diag_h.size() * 8, cudaMemcpyDeviceToHost, J.s));
            JCUDA(cudaStreamSynchronize(J.s));
            double d2 = 0.0;
            for (double x : diag_h) d2 += x * x;
            spread[1] = 3.0 * sumsq - d2;
        }
        // ---- U = V^T (reading J4), psi~ = U psi (eq. 12)
        JRC(bse_launch_transpose(V, Nv, U, Nv, Nv, J.s));
        if (psi_loc) {
            JRC(bse_launch_transpose(V, Nv, Vt, lds, Nv, J.s));
            JRC(bse_gemm_nn(Vt, lds, psi, N, Nv, N, Nv, EPI_STORE, nullptr, nullptr, psi_loc, N, J.s));
        }
        JCUDA(cudaEventRecord(ev, J.s));
        JCUDA(cudaStreamWaitEvent(user, ev, 0));                 // the caller's stream sees U / psi_loc
        JCUDA(cudaStreamSynchronize(J.s));
    }
cleanup:
#undef JCUDA
#undef JRC
    if (J.s) cudaStreamSynchronize(J.s);
    for (cudaGraphExec_t e : J.exec) if (e) cudaGraphExecDestroy(e);
    cudaFree(J.A); cudaFree(J.cs); cudaFree(J.smax); cudaFree(wbuf); cudaFree(part); cudaFree(tabs); cudaFree(T); cudaFree(Vt);
    cudaFree(Vp); cudaFree(diag); cudaFree(perm_d);
    if (ev) cudaEventDestroy(ev);
    if (J.s) cudaStreamDestroy(J.s);
    return rc;
}
