// FP64 tensor-core (DMMA, mma.sync.m8n8k4.f64) GEMMs for the dense contractions of the path:
//   a1  screen          M_vw   = sum_r u_v^2 u_w^2                       (eq. 16)   dot form, split-K
//   a5  PDEP projection c_{a,p}= 2 sum_{H\0} Re(conj phi_a x_p)          (eq. 11)   dot form, split-K
//   a7  back-projection y_p(G) = sum_a phi_a(G) f_a c_{a,p}, fused a8    (eq. 9, 11)              NN form
//   a11 P_c             S = dV acc u^T (dot form), out = acc - S u (NN)
// tcgen05.mma has no f64 kind on sm_100a, so the FP64 tensor path is the warp-level DMMA; operands are staged
// with cp.async (LDGSTS) through a 3-stage shared-memory ring.  CTA tile 64 x 64 x 16, 4 warps of 32 x 32.
#include "bse_internal.h"

namespace {

constexpr int BN = 64, BK = 16, STAGES = 3;
// CTA tile BMT x 64 x 16 with BMT = 64 (4 warps) or 128 (8 warps); every warp owns 32 x 32
constexpr int LDK = BK + 4;    // K-major tile row stride (doubles): conflict-free fragment reads
constexpr int LDN = BN + 4;    // N-major tile row stride
constexpr int B_TILE_K = BN * LDK;
constexpr int B_TILE_N = BK * LDN;

// 16-byte cp.async that reads only `sz` (0, 8 or 16) bytes from global and zero-fills the rest
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int sz) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// load a K-major tile: rows [r0, r0+64) of a [rows][K] matrix, k in [k0, k0+16) -> smem [64][LDK]
template <int ROWS, int NT>
__device__ __forceinline__ void load_tile_k(double *sm, const double *g, long long ld, int rows, int r0,
                                            long long k0, long long kend) {
    // ROWS rows x BK/2 chunks of 16 B, NT threads
#pragma unroll
    for (int i = 0; i < ROWS * (BK / 2) / NT; ++i) {
        const int c = threadIdx.x + i * NT;
        const int r = c / (BK / 2), kc = (c % (BK / 2)) * 2;
        const long long left = kend - (k0 + kc);
        const bool ok = (r0 + r < rows) && (left > 0);
        const double *src = ok ? g + (long long)(r0 + r) * ld + k0 + kc : g;
        cp_async16(sm + r * LDK + kc, src, ok ? (left >= 2 ? 16 : 8) : 0);
    }
}
// load an N-major tile: k rows [k0,k0+16) of a [K][N] matrix, columns [c0, c0+64) -> smem [16][LDN]
template <int NT>
__device__ __forceinline__ void load_tile_n(double *sm, const double *g, long long ld, long long cols, long long c0,
                                            int k0, int kend) {
    // BK rows x 32 chunks
#pragma unroll
    for (int i = 0; i < BK * 32 / NT; ++i) {
        const int c = threadIdx.x + i * NT;
        const int r = c >> 5, cc = (c & 31) * 2;
        const long long left = cols - (c0 + cc);
        const bool ok = (k0 + r < kend) && (left > 0);
        const double *src = ok ? g + (long long)(k0 + r) * ld + c0 + cc : g;
        cp_async16(sm + r * LDN + cc, src, ok ? (left >= 2 ? 16 : 8) : 0);
    }
}

// BN_MAJOR = false: B is [N][K] (dot form).  true: B is [K][N] (NN form).
// EPI_PARTIAL: store raw accumulators to part[z][M][Ntot]  (split-K, K range per blockIdx.z)
// EPI_TAU    : C[m][n] = cs2[n>>1] * (Xin[m][n] + acc)
// EPI_SUB    : C[m][n] = C[m][n] - acc
// EPI_STORE  : C[m][n] = acc
template <int BM, bool BN_MAJOR, int EPI, bool SQA, bool SQB>
__global__ void __launch_bounds__(2 * BM)
dgemm_kernel(const double *__restrict__ A, long long lda, const double *__restrict__ B, long long ldb, int M,
             long long Ntot, long long K, long long kchunk, double *__restrict__ C, long long ldc,
             const double *__restrict__ Xin, const double *__restrict__ cs2) {
    extern __shared__ __align__(16) double sm[];
    constexpr int THREADS = 2 * BM, A_TILE = BM * LDK;
    double *As = sm;
    double *Bs = sm + STAGES * A_TILE;
    constexpr int B_TILE = BN_MAJOR ? B_TILE_N : B_TILE_K;

    // NN form: 1-D grid with the m tile fastest, so the CTAs that share one [K][64] panel of B (the big operand: u or Phi)
    // run back to back and the panel is read from HBM once.  Dot form: (n tile, m tile, k split).
    const int tm_ = (M + BM - 1) / BM;
    const int m0 = (BN_MAJOR ? (int)(blockIdx.x % tm_) : (int)blockIdx.y) * BM;
    const long long n0 = (long long)(BN_MAJOR ? blockIdx.x / tm_ : blockIdx.x) * BN;
    const long long kbeg = (long long)blockIdx.z * kchunk;
    const long long kend = (kbeg + kchunk < K) ? kbeg + kchunk : K;
    const int nk = (int)((kend - kbeg + BK - 1) / BK);
    if (SQA && SQB && n0 + BN <= m0) return;      // screen SYRK: M is symmetric, only tiles touching v <= w are formed
    (void)THREADS;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;
    const int lr = lane >> 2, lc = lane & 3;

    // EPI_TAU / EPI_SUB: the accumulators start from the epilogue operand (Xin, resp. C), whose global loads then overlap
    // the cp.async prologue instead of sitting exposed after the k loop; EPI_SUB multiplies with -A (C - A B).
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            acc[i][j][0] = acc[i][j][1] = 0.0;
            if (EPI == EPI_TAU || EPI == EPI_SUB) {
                const int m = m0 + wm + i * 8 + lr;
                const long long nn = n0 + wn + j * 8 + 2 * lc;
                if (m < M && nn + 1 < Ntot) {
                    const double *src = (EPI == EPI_TAU ? Xin : C) + (long long)m * ldc + nn;
                    const double2 x = __ldcs(reinterpret_cast<const double2 *>(src));
                    acc[i][j][0] = x.x; acc[i][j][1] = x.y;
                } else if (m < M && nn < Ntot) {
                    acc[i][j][0] = ((EPI == EPI_TAU ? Xin : C) + (long long)m * ldc + nn)[0];
                }
            }
        }

    auto issue = [&](int kt) {
        if (kt < nk) {
            const int st = kt % STAGES;
            const long long k0 = kbeg + (long long)kt * BK;
            load_tile_k<BM, THREADS>(As + st * A_TILE, A, lda, M, m0, k0, kend);
            if (BN_MAJOR) load_tile_n<THREADS>(Bs + st * B_TILE, B, ldb, Ntot, n0, (int)k0, (int)kend);
            else load_tile_k<BN, THREADS>(Bs + st * B_TILE, B, ldb, (int)Ntot, (int)n0, k0, kend);
        }
        cp_commit();
    };
#pragma unroll
    for (int i = 0; i < STAGES - 1; ++i) issue(i);
    for (int kt = 0; kt < nk; ++kt) {
        cp_wait<STAGES - 2>();
        __syncthreads();
        issue(kt + STAGES - 1);
        const double *as = As + (kt % STAGES) * A_TILE;
        const double *bs = Bs + (kt % STAGES) * B_TILE;
        if (SQA && SQB && m0 + wm >= (int)n0 + wn + 32) continue;   // SYRK: a warp tile entirely below the diagonal idles
#pragma unroll
        for (int kk = 0; kk < BK; kk += 4) {
            double af[4], bf[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                af[i] = as[(wm + i * 8 + lr) * LDK + kk + lc];
                if (SQA) af[i] *= af[i];
                if (EPI == EPI_SUB) af[i] = -af[i];
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                bf[j] = BN_MAJOR ? bs[(kk + lc) * LDN + wn + j * 8 + lr] : bs[(wn + j * 8 + lr) * LDK + kk + lc];
                if (SQB) bf[j] *= bf[j];
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cp_wait<0>();

    // epilogue: thread holds C[row = lr][col = 2*lc, 2*lc+1] of each 8x8 tile
    double *Cout = C;
    if (EPI == EPI_PARTIAL) Cout = C + (long long)blockIdx.z * M * ldc;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int m = m0 + wm + i * 8 + lr;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const long long nn = n0 + wn + j * 8 + 2 * lc;
            if (nn >= Ntot) continue;     // Ntot even for every caller that reaches the vector store below
            double v0 = acc[i][j][0], v1 = acc[i][j][1];
            double *dst = Cout + (long long)m * ldc + nn;
            if (EPI == EPI_TAU) {
                const double sc = cs2[nn >> 1];
                v0 *= sc;
                v1 *= sc;
            }
            if (EPI == EPI_PARTIAL) {          // ldc may be odd here: scalar stores
                dst[0] = v0;
                if (nn + 1 < Ntot) dst[1] = v1;
            } else if (nn + 1 < Ntot) {
                *reinterpret_cast<double2 *>(dst) = make_double2(v0, v1);
            } else {
                dst[0] = v0;
            }
        }
    }
}

// C[m][n] = alpha * colscale[n] * sum_z part[z][m][n], fixed order (deterministic)
__global__ void splitk_reduce_kernel(const double *__restrict__ part, int splits, long long MN, int N,
                                     double *__restrict__ C, long long ldc, double alpha,
                                     const double *__restrict__ colscale, int accumulate) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= MN) return;
    double s = 0.0;
    for (int z = 0; z < splits; ++z) s += part[(long long)z * MN + i];
    s *= alpha;
    const long long m = i / N;
    const int n = (int)(i - m * N);
    if (colscale) s *= colscale[n];
    C[m * ldc + n] = accumulate ? C[m * ldc + n] + s : s;
}

constexpr int smem_dot(int bm) { return STAGES * (bm * LDK + B_TILE_K) * 8; }
constexpr int smem_nn(int bm) { return STAGES * (bm * LDK + B_TILE_N) * 8; }

// CTA tile height: 64 rows (4 warps).  The 128-row form (8 warps, the 64-column operand tile shared by twice as many warps) is
// kept behind bse_debug_set("gemm_bm", 128) for A/B timing: it measured slower wherever it differed (cfg 5 pdep_project 468 vs
// 354 ms, pdep_backproject 410 vs 337 ms, P_c equal): half as many CTAs to balance over 148 SMs and two CTAs per SM instead of 3-4.
int g_bm_override = 0;
inline int pick_bm(int) { return g_bm_override == 128 ? 128 : 64; }

// Dynamic shared-memory opt-in of one kernel instantiation.  cudaFuncSetAttribute is thread-safe and idempotent, so it is
// simply issued before every launch (a few hundred ns on the host) instead of remembering pointers in a shared table.
template <typename KernelT>
int prep(KernelT k, int smem) {
    BSE_CUDA(cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    return BSE_OK;
}

template <int BM, bool BN_MAJOR, int EPI, bool SQA, bool SQB>
int launch(dim3 grid, int smem, cudaStream_t s, const double *A, long long lda, const double *B, long long ldb, int M,
           long long N, long long K, long long kchunk, double *C, long long ldc, const double *Xin, const double *cs2) {
    auto k = dgemm_kernel<BM, BN_MAJOR, EPI, SQA, SQB>;
    int rc = prep(k, smem);
    if (rc) return rc;
    k<<<grid, 2 * BM, smem, s>>>(A, lda, B, ldb, M, N, K, kchunk, C, ldc, Xin, cs2);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

}  // namespace

void bse_gemm_set_bm(int bm) { g_bm_override = bm; }

int bse_gemm_dot(const double *A, long long lda, const double *B, long long ldb, int M, int N, long long K,
                 bool squareA, bool squareB, double *part, size_t part_bytes, double *C, long long ldc,
                 double alpha, const double *colscale, cudaStream_t s, bool accumulate) {
    if (M <= 0 || N <= 0) return BSE_OK;
    const int BM = pick_bm(M);
    const int tm = (M + BM - 1) / BM, tn = (N + BN - 1) / BN;
    const long long ksteps = (K + BK - 1) / BK;
    long long tiles = (long long)tm * tn;
    if (squareA && squareB) {                                   // SYRK: tiles that touch v <= w
        tiles = 0;
        for (int i = 0; i < tm; ++i)
            for (int j = 0; j < tn; ++j) tiles += ((long long)(j + 1) * BN > (long long)i * BM) ? 1 : 0;
    }
    // split K so that the CTAs fill the machine in whole waves.  A CTA of 64 rows (4 warps, 60 KB of shared memory) is
    // resident 3 to an SM, so a wave is 444 CTAs and costs 3 units (one unit = one CTA on an SM whose DMMA pipe is saturated,
    // which takes ~8 warps); the last, partial wave puts c = ceil(r / 148) CTAs on an SM and costs c units, or ~1.7 when
    // c = 1 (4 warps do not saturate the pipe).  Measured: 304 CTAs ran 1.5x longer than 288; cfg 4's projection at 576 CTAs
    // (one wave + 132) reached 0.69 of the DMMA peak, at 288 (two per SM) 0.86.  The SYRK squares its operands on the way to
    // the fragments and needs all three resident CTAs to hide that: two per SM ran at 0.44 against 0.66 with three, so there a
    // partial wave costs as much as a full one.  More, shorter CTAs only add prologue and partial-sum traffic, so a larger
    // split must win by 2 %.
    const long long sms = 148;
    long long smax = ksteps / 8;
    const long long cap = (long long)(part_bytes / ((size_t)M * N * 8));
    if (cap < 1) { bse_set_error("bse_gemm_dot: split-K workspace too small"); return BSE_ENOMEM; }
    if (smax > cap) smax = cap;
    if (smax < 1) smax = 1;
    long long splits = 1;
    double best = -1.0;
    const long long res = BM == 128 ? 2 : 3;                    // resident CTAs per SM
    for (long long sp = 1; sp <= smax; ++sp) {
        const long long ctas = tiles * sp;
        const long long full = ctas / (res * sms), r = ctas % (res * sms);
        double t = (double)(full * res);
        if (r) {
            const long long c = (r + sms - 1) / sms;
            t += (squareA && squareB) ? (double)res : (c == 1 && BM == 64) ? 1.7 : (double)c;
        }
        const double eff = ((double)ctas / (double)sms) / t;
        if (eff > best + 0.02) { best = eff; splits = sp; }
        if (ctas >= 5 * res * sms) break;
    }
    long long kchunk = ((ksteps + splits - 1) / splits) * BK;
    splits = (K + kchunk - 1) / kchunk;
    dim3 grid(tn, tm, (unsigned)splits);
    int rc;
    if (squareA && squareB)
        rc = BM == 128 ? launch<128, false, EPI_PARTIAL, true, true>(grid, smem_dot(128), s, A, lda, B, ldb, M, N, K, kchunk, part, N, nullptr, nullptr)
                       : launch<64, false, EPI_PARTIAL, true, true>(grid, smem_dot(64), s, A, lda, B, ldb, M, N, K, kchunk, part, N, nullptr, nullptr);
    else
        rc = BM == 128 ? launch<128, false, EPI_PARTIAL, false, false>(grid, smem_dot(128), s, A, lda, B, ldb, M, N, K, kchunk, part, N, nullptr, nullptr)
                       : launch<64, false, EPI_PARTIAL, false, false>(grid, smem_dot(64), s, A, lda, B, ldb, M, N, K, kchunk, part, N, nullptr, nullptr);
    if (rc) return rc;
    const long long MN = (long long)M * N;
    splitk_reduce_kernel<<<(unsigned)((MN + 255) / 256), 256, 0, s>>>(part, (int)splits, MN, N, C, ldc, alpha, colscale,
                                                                       accumulate ? 1 : 0);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_gemm_nn(const double *A, long long lda, const double *B, long long ldb, int M, long long N, int K, int epi,
                const double *Xin, const double *colscale2, double *C, long long ldc, cudaStream_t s) {
    if (M <= 0 || N <= 0) return BSE_OK;
    const int BM = pick_bm(M);
    const int tm = (M + BM - 1) / BM;
    const long long tn = (N + BN - 1) / BN;
    if (tn * tm > 2147483647LL) { bse_set_error("bse_gemm_nn: too many tiles"); return BSE_EUNSUPPORTED; }
    dim3 grid((unsigned)(tn * tm), 1, 1);
#define BSE_NN(EPI, XIN, CS2)                                                                                                  \
    (BM == 128 ? launch<128, true, EPI, false, false>(grid, smem_nn(128), s, A, lda, B, ldb, M, N, K, K, C, ldc, XIN, CS2)      \
               : launch<64, true, EPI, false, false>(grid, smem_nn(64), s, A, lda, B, ldb, M, N, K, K, C, ldc, XIN, CS2))
    if (epi == EPI_TAU) return BSE_NN(EPI_TAU, Xin, colscale2);
    if (epi == EPI_SUB) return BSE_NN(EPI_SUB, nullptr, nullptr);
    if (epi == EPI_STORE) return BSE_NN(EPI_STORE, nullptr, nullptr);
#undef BSE_NN
    bse_set_error("bse_gemm_nn: bad epilogue");
    return BSE_EINVAL;
}

// ---------------------------------------------------------------------------------------------------------
// Allocation-free screen (include/bse.h: bse_screen_overlap_static).  The split-K partial sums of the SYRK above normally
// live in the handle's cudaMalloc'ed workspace; callers that may not allocate (CUDA graph capture, serving loops) get the
// same kernels with the partial sums in a fixed array that is part of the library image: every GPU that loads the library
// holds these 8 MiB until the process exits.  In HOST code the name g_screen_scratch is only a stand-in of the symbol, not a
// device address: the address comes from cudaGetSymbolAddress, once per device, with that device current.
#include <mutex>

constexpr size_t SCREEN_SCRATCH_BYTES = (size_t)BSE_SCREEN_STATIC_BYTES;
static __device__ __align__(256) double g_screen_scratch[SCREEN_SCRATCH_BYTES / 8];

namespace {
constexpr int MAX_DEVICES = 64;
double *g_screen_scratch_addr[MAX_DEVICES] = {nullptr};         // device address of g_screen_scratch on device d
std::mutex g_screen_scratch_mutex;

int screen_scratch_address(double **out) {
    int dev = -1;
    BSE_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) { bse_set_error("bse_screen_overlap_static: device ordinal out of range"); return BSE_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_screen_scratch_mutex);
    if (!g_screen_scratch_addr[dev]) {
        double *p = nullptr;
        BSE_CUDA(cudaGetSymbolAddress((void **)&p, g_screen_scratch));
        if (!p) { bse_set_error("bse_screen_overlap_static: cudaGetSymbolAddress returned a null address"); return BSE_ECUDA; }
        g_screen_scratch_addr[dev] = p;
    }
    *out = g_screen_scratch_addr[dev];
    return BSE_OK;
}
}  // namespace

extern "C" int bse_screen_overlap_static(const double *u, int Nv, long long N, double *M, void *stream) {
    if (!u || !M || Nv <= 0 || N <= 0) { bse_set_error("bse_screen_overlap_static: null pointer or empty size"); return BSE_EINVAL; }
    if ((N & 1) || ((uintptr_t)u & 15)) {
        bse_set_error("bse_screen_overlap_static: N must be even and u 16-byte aligned (16-byte operand loads)");
        return BSE_EINVAL;
    }
    const size_t need = (size_t)Nv * (size_t)Nv * 8;              // one set of partial sums (split-K factor 1)
    if (need > SCREEN_SCRATCH_BYTES) {
        bse_set_error("bse_screen_overlap_static: Nv = " + std::to_string(Nv) + " needs " + std::to_string(need) +
                      " bytes of split-K scratch, the static array holds " + std::to_string(SCREEN_SCRATCH_BYTES) +
                      " (Nv <= " + std::to_string(BSE_SCREEN_STATIC_MAX_NV) + ")");
        return BSE_EINVAL;
    }
    double *part = nullptr;
    int rc;
    if ((rc = screen_scratch_address(&part))) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    // the array keeps the previous call's partial sums, and the SYRK writes only the tiles that touch v <= w: clear it, so that
    // the tiles below the diagonal reduce to zero instead of to whatever an earlier call left there
    BSE_CUDA(cudaMemsetAsync(part, 0, SCREEN_SCRATCH_BYTES, s));
    return bse_gemm_dot(u, N, u, N, Nv, Nv, N, true, true, part, SCREEN_SCRATCH_BYTES, M, Nv, 1.0, nullptr, s, false);
}
