// Internal declarations shared by the CUDA translation units of libbse_b200.  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/bse.h"

// ---------------------------------------------------------------------------------------------------------
// FFT plan: one length n = R1 * R2 for all three axes (cubic grid); two register-butterfly passes per axis
// (fft_kernels.cuh).  Sticks = (m2, m3) columns of the sphere's disk with m3 > 0 or (m3 == 0 and m2 >= 0), ordered
// by (m2 mod n, m3).
struct FftPlan {
    int n = 0, R1 = 0, R2 = 0;
    long long N = 0;     // n^3
    int R = 0;           // floor(sqrt(msq_max))
    int W = 0;           // kept m3 columns in the plane pass: m3 = 0..R  -> W = R + 1
    int NS = 0;          // number of half sticks
    long long npw_h = 0;
    const void *ops = nullptr;    // bsefft::FftOps of this n
    int compact_inv = -1;         // inverse plane kernel: -1 automatic, 0 never compact, k > 1 compact sized for k CTAs / SM
    int pipe = -1;                // plane passes: -1 automatic, 0 one-plane-per-CTA kernels, 1 pipelined kernels (fft_pipe.cuh)
    int pipe_lc = 0;              // > 0: cap on the lines per slab of the pipelined kernels (test knob)
    // device tables
    double2 *tw = nullptr;        // [n]   exp(-2 pi i t / n)
    int *soff = nullptr;          // [n]   stick index of (t2 = m2 mod n, m3) is soff[t2] + m3
    int *wmax = nullptr;          // [n]   largest m3 with a stick at t2, -1 if none
    int *wmin = nullptr;          // [n]   smallest stored m3 at t2 (1 for m2 < 0)
    int *hmapT = nullptr;         // [n][NS] (t1 = m1 mod n, stick) -> h in H, -1 outside, -2-h conj of entry h
    double *vc12 = nullptr;       // [npw_h] sqrt(4 pi)/|G|, 0 at G = 0
    double *vc12n = nullptr;      // [npw_h] vc12 / (2N)  (forward normalisation and the untangling 1/2 folded in)
    double *inv2n = nullptr;      // [npw_h] 1 / (2N)     (forward transform without the Coulomb factor, PW wrapper)
    double *vcn = nullptr;        // [npw_h] v_c / (2N) = vc12^2 / (2N)  (Hartree potential of K1e)
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
    FftPlan fft;                     // the problem grid n
    FftPlan ffta;                    // coarser apply grid of the PW layout (n_a >= 3R+1), if one exists
    const FftPlan *ap = nullptr;     // grid the apply runs on: &ffta or &fft
    double *f2 = nullptr;            // device [Npdep]  2 lambda/(1-lambda)
    // screen / pair list
    double *Mmat = nullptr;          // device [Nv][Nv]  sum_r u_v^2 u_w^2
    int *rowcnt = nullptr, *rowptr = nullptr;   // device [Nv], [Nv+1]
    int *pid = nullptr;              // device [Nv][Nv] pair index or -1 (v <= w)
    int2 *pairs = nullptr;           // device [P]
    int *adj_ptr = nullptr;          // device [Nv+1] directed adjacency (both directions)
    int2 *adj = nullptr;             // device [nadj] (w, pair index), sorted by w within a row
    long long P = -1, nadj = 0;
    std::vector<int> adj_h;          // host copy of adj, flattened (w, pair)
    struct RowBatch { int v0, v1, u0, nu; };   // rows rowlist[v0 .. v1); its unique pairs are batch_pairs[u0, u0 + nu)
    std::vector<RowBatch> batches;
    int *batch_pairs = nullptr;      // device: pair indices of every batch, concatenated
    int *eslot = nullptr;            // device [nadj]: slot of directed entry e inside its batch
    int *rowlist = nullptr;          // device [Nv]: rows in batch order (clusters of the pair graph)
    double uniq_share = 1.0;         // P / (sum of nu): share of the inverted fields that is algorithmic work
    std::vector<int> adj_ptr_h;      // host copy of adj_ptr (row batches of the batched tau modes)
    bool built = false;
    // row-sharded operation (bse_set_rows): this handle owns the output rows [row0, row1); the tau store then
    // holds only the Pa pairs that touch one of them (pairs_act, ascending pair index; eslot_act[e] = slot of directed entry e)
    int row0 = 0, row1 = 0;                // row1 = Nv when unrestricted
    bool rows_set = false;
    long long Pa = 0;                      // pairs in the tau store (= P when unrestricted)
    int2 *pairs_act = nullptr;             // device [Pa] (restricted only; else the store follows `pairs`)
    int *eslot_act = nullptr;              // device [nadj] (restricted only)
    // tau store
    double *tau_r = nullptr;         // [P][N]
    double2 *tau_g = nullptr;        // [P][npw_h]
    float2 *tau_g32 = nullptr;       // [P][npw_h] single-precision store (BSE_TAU_F32) instead of tau_g
    size_t tau_bytes = 0;            // capacity of the store (grow-only)
    // workspaces (sized for a pair batch)
    long long Pb = 0;                // pairs per batch (Pb_alloc rounded down to whole 64-row GEMM tiles)
    long long Pb_alloc = 0;          // fields the batch workspaces hold
    double2 *Z = nullptr;            // [Pb_alloc][n][NS]
    double2 *X = nullptr;            // [Pb][npw_h]
    double2 *T = nullptr;            // [Pb][npw_h]
    double *Dm = nullptr;            // [Pb][Npdep]
    double *part = nullptr;          // split-K partials
    size_t part_bytes = 0;
    double *Sov = nullptr;           // [B*Nv][Nv] P_c overlaps
    size_t Sov_elems = 0;
    double *tau_batch = nullptr;     // [Pacc][N] tau(r) of one row batch (PW / STREAM modes)
    // PW layout (a12): u on H, its weighted copy for <u_w|.>, real-space staging of one group of Bg trial blocks
    double2 *uG = nullptr, *uGw = nullptr;         // [Nv][npw_h]
    double *a_r = nullptr, *acc_r = nullptr;       // [Bg][Nv][N]
    int Bg = 0, rows_cap = 0;                      // acc_r holds rows_cap rows per block (row batches)
    bool Bg_final = false, plan_ok = false;
    std::vector<int> plan_adj_h, plan_adj_ptr_h;   // the adjacency the row batches were planned for (exact comparison)
    // debug / test knobs (bse_debug_set; never read from the environment): caps that only ever lower a limit
    long long dbg_max_group = 0, dbg_max_batch = 0;   // 0 = no cap; either one set keeps the apply on the group / row-batch path
    long long dbg_in_chunks = 0;                      // column slabs bse_set_inputs_host copies u in (0 = automatic)
    long long dbg_pc_rows = 0;                        // cap of the rows per chunk of P_c (0 = no cap)
    long long dbg_slab_planes = 0;                    // cap of the planes per slab (0 = no cap)
    long long dbg_slab_rows = 0;                      // cap of the rows per chunk of the plane-slab apply; -1 = never use it
    // plane-slab streaming of the PW-layout apply: a_r = [B][Nv][SN], tau_batch = [P][SN],
    // acc_r = [B][slab_rc][SN], SN = R2 n_a^2 points of the slab { i1 = s + R1 k2 }
    bool slab_mode = false, plan_allow_slab = true, plan_mix = false;
    int slab_rc = 0;                                  // rows per chunk
    int slab_S = 0, slab_M = 0;                       // the slab split n_a = S * M chosen by the plan (fewest slabs that fit)
    size_t a_r_elems = 0;                             // capacity of a_r in doubles
    long long slab_pz = 0;                            // slab fields that fit the stick-plane buffer Z
    int *rowid = nullptr;                             // device [Nv]: rows in the order the chunks take them
    int dbg_compact_inv = -1;                         // -1 = automatic choice of the inverse plane kernel
    long long Pacc = 0;                            // capacity of tau_batch in directed entries                         // Bg is already the most that fits
    // K1e workspaces (grow-only): dens / vH [B][N] (REAL) or one block's a(r) [Nv][Na] + [1][Na] + product rows [Pb][Na] (PW)
    double *k1e_ws = nullptr;
    size_t k1e_bytes = 0;
    // combined K1e / K1x call (bse_apply_k1): while mix_on, accumulate_all folds ce * 2 u_v vH[b] into the accumulated rows
    bool mix_on = false;
    double mix_ce = 0.0, mix_cd = 1.0;
    int mix_B = 0;
    const double *mix_u = nullptr;                 // orbitals on the grid the apply runs on; nullptr: made on the fly from uG
    const double *mix_vH = nullptr;                // [nb][N] Hartree potentials of the blocks being accumulated
    bool uG_valid = false, u_a_valid = false;      // uG / uGw / u_a hold the current orbitals (stale after bse_set_inputs_host)
    int u_bl = -1;                                 // 1: every orbital is band-limited to S (checked once), 0: not, -1: unknown
    double2 *accG = nullptr;                       // [rows][npw_h] rows on H for the P_c overlaps of the REAL layout
    long long accG_rows = 0;
    double *Ut = nullptr;                          // [Nv][ldS] transposed copy of the rotation matrix (bse_rotate)
    double *u_a = nullptr;                         // [Nv][Na] orbitals on the apply grid (PW layout with a coarser grid)
    double *a_dev = nullptr, *out_dev = nullptr;   // staging for the host-pointer entry point
    size_t a_dev_bytes = 0;
    cudaStream_t s_in = nullptr, s_out = nullptr;  // copy streams of the pipelined host-pointer apply
    std::vector<cudaEvent_t> ev_pipe;
    // host-pointer apply, non-pipelined form: the copy of a overlaps the tau rebuild (STREAM), finished row chunks of P_c
    // leave for the host while the next chunk is projected
    bool tau_prefilled = false;                    // bse_apply_k1x_host has rebuilt tau for the apply that follows
    double *d2h_host = nullptr;                    // host image of out_dev (non-null only inside bse_apply_k1x_host)
    long long d2h_rows_done = 0;                   // leading rows of out_dev already on their way to d2h_host
    cudaEvent_t ev_d2h = nullptr;
    // bse_set_inputs_host copies on s_in, u in column slabs: bse_build_tau screens slab c as soon as it has arrived
    bool inputs_pending = false;                   // a copy is in flight that the library's stream has not yet waited for
    int in_chunks = 0;                             // column slabs of the last copy of u (0: u was not copied)
    long long in_kc = 0;                           // grid points per slab
    std::vector<cudaEvent_t> ev_in;                // [c] slab c of u is on the device
    cudaEvent_t ev_in_done = nullptr;              // everything bse_set_inputs_host enqueued is on the device
    // profiling
    bool prof = false;
    double st_ms[BSE_ST_COUNT] = {0};
    long long st_launch[BSE_ST_COUNT] = {0};
    double st_flops[BSE_ST_COUNT] = {0}, st_bytes[BSE_ST_COUNT] = {0};   // algorithmic work of the launches so far
    double st_handoff[BSE_ST_COUNT] = {0};                               // + bytes of the Z hand-off between plane and stick pass
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    cudaEvent_t ev_fill0 = nullptr, ev_fill1 = nullptr;   // around the last fill of the tau store
    bool fill_timed = false;
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
int bse_fft_select(FftPlan &pl);     // sets R1, R2, ops for pl.n; BSE_EUNSUPPORTED if there is no kernel for n
// fields: [.][N]; pairs == nullptr: plain transform of field p0+p.  scale: [npw_h] table applied in the stick pass.
// fwd_stick: scatter != nullptr (device array): field p is written to X + scatter[p] * npw_h instead of X + p * npw_h.
// np > 0: the fields hold np planes each (one slab, N = np n^2 is then the field stride) instead of n
int bse_launch_fwd_plane(const FftPlan &pl, const double *fields, const int2 *pairs, long long p0, int count,
                         long long N, double2 *Z, cudaStream_t s, int np = 0);
int bse_launch_fwd_stick(const FftPlan &pl, const double2 *Z, int count, double2 *X, const double *scale,
                         cudaStream_t s, const int *scatter = nullptr);
// gather != nullptr: field p is read from T + gather[g0 + p] * npw_h (pair indices of a row batch)
// T32 != nullptr: read the coefficients from this single-precision copy instead of T (BSE_TAU_F32)
int bse_launch_inv_stick(const FftPlan &pl, const double2 *T, int count, double2 *Z, cudaStream_t s,
                         const int *gather = nullptr, int g0 = 0, const float2 *T32 = nullptr);
// subtract: out <- out - transform instead of out <- transform (P_c update of the REAL layout)
int bse_launch_inv_plane(const FftPlan &pl, const double2 *Z, int count, long long N, double *out, cudaStream_t s,
                         bool subtract = false, int np = 0);
// slab forms of the stick passes (fft_kernels.cuh): the planes i1 = slab + S k, k < M, only (n = S M, M <= 32).  Zs[count][M][NS].
// forward: field p goes to row (p / rc) * row_ld + row0 + p % rc of X; accumulate: X += (slabs 1 .. R1-1) instead of X =
int bse_launch_inv_stick_slab(const FftPlan &pl, int S, int M, const double2 *T, int count, double2 *Zs, cudaStream_t s, int slab,
                              const int *gather = nullptr, int g0 = 0, const float2 *T32 = nullptr);
int bse_launch_fwd_stick_slab(const FftPlan &pl, int S, int M, const double2 *Zs, int count, double2 *X, const double *scale,
                              cudaStream_t s, int slab, bool accumulate, int rc, long long row_ld, long long row0);

// gemm_dmma.cu
enum { EPI_PARTIAL = 0, EPI_TAU = 1, EPI_SUB = 2, EPI_STORE = 3 };
// C[M][N] (+)= A[M][K] * B[N][K]^T, split-K partials into `part` then reduced: C = alpha * colscale[n] * sum
int bse_gemm_dot(const double *A, long long lda, const double *B, long long ldb, int M, int N, long long K,
                 bool squareA, bool squareB, double *part, size_t part_bytes, double *C, long long ldc,
                 double alpha, const double *colscale, cudaStream_t s, bool accumulate = false);   // accumulate: C += instead of C =
void bse_gemm_set_bm(int bm);      // test / tuning knob: force the CTA tile height (64 or 128; 0 = automatic)
// NN form: acc = A[M][K] * B[K][N];  EPI_TAU: C = colscale2[n>>1] * (Xin + acc);  EPI_SUB: C = C - acc;  EPI_STORE: C = acc
int bse_gemm_nn(const double *A, long long lda, const double *B, long long ldb, int M, long long N, int K,
                int epi, const double *Xin, const double *colscale2, double *C, long long ldc, cudaStream_t s);

// k1x_kernels.cu
int bse_launch_pairlist(bse_handle *h);                 // M -> rowcnt,rowptr,pid,pairs (count only if pairs==nullptr)
// row-complete accumulation of the rows rows[0 .. nrows) (device array): tau_b[eslot[e]] for every directed entry e of
// those rows; local: acc row index = position in the batch instead of the row id
int bse_launch_accumulate_rows(bse_handle *h, long long N, const double *tau_b, const int *eslot, const int *rows,
                               int nrows, const double *a, double *acc, long long acc_ld, bool local, int B);
// K1e (eq. 4): dens[b][r] = sum_v u[v][r] a[b][v][r];  out[b * out_ld + i][r] = 2 u[v0 + i][r] vH[b][r], i < nrows
// u: the orbitals v0 .. v0 + nv (nv < 0: all Nv, v0 = 0); add: dens += instead of dens =
int bse_launch_k1e_density(const double *u, const double *a, double *dens, int Nv, long long N, int B, cudaStream_t s,
                           int v0 = 0, int nv = -1, bool add = false);
int bse_launch_k1e_product(const double *u, const double *vH, double *out, int v0, int nrows, long long out_ld,
                           long long N, int B, cudaStream_t s);
// acc row <- cd * acc row + 2 ce * u[v] * vH[b] on nrows rows (rows: device row ids or nullptr = identity)
int bse_launch_k1_mix(const double *u, const double *vH, double *acc, const int *rows, int nrows, long long acc_ld,
                      bool local, long long N, int nb, double ce, double cd, cudaStream_t s);
// out[2 row] = sum_k x[row][k]^2, out[2 row + 1] = sum_k (x[row][k] - y[row][k])^2 (rows of len doubles)
int bse_launch_row_sumsq(const double *x, const double *y, long long len, int rows, double *out, cudaStream_t s);
// dst[j][i] = src[i][j], n x n, leading dimensions lds / ldd
int bse_launch_transpose(const double *src, long long lds, double *dst, long long ldd, int n, cudaStream_t s);
// dst[i] = (float) src[i], count doubles (tau(G) of a pair batch into the single-precision store)
int bse_launch_to_f32(const double *src, float *dst, long long count, cudaStream_t s);
// dst[w][k] = Omega * wt * src[w][k], wt = 2 for G != 0 and (1, 0) on (re, im) of G = 0 (entry 0 of H)
int bse_launch_weight_pw(const double2 *src, double2 *dst, long long npw_h, long long rows, double Omega,
                         cudaStream_t s);
int bse_launch_accumulate(bse_handle *h, const double *tau, long long p_first, long long p_count,
                          const double *a, double *acc, int B, bool zero_init);
