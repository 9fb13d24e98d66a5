// C-ABI entry points of libbse_b200 (include/bse.h): host-side tables, orchestration of the kernel sequence.
// Path:  a1 screen -> pair list -> per pair batch [a2+a3 plane pass, a3+a4 stick pass,
// a5+a6 projection DGEMM, a7+a8 back-projection DGEMM, a9 inverse stick + plane pass] ; apply: a10 accumulate,
// a11 P_c (two DGEMMs).  No CPU fallback: every numeric step is a kernel in this library.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "bse_internal.h"

static thread_local std::string g_err;
void bse_set_error(const std::string &msg) { g_err = msg; }
int bse_cuda_fail(cudaError_t e, const char *what) {
    g_err = std::string("CUDA error: ") + cudaGetErrorString(e) + " at " + what;
    return e == cudaErrorMemoryAllocation ? BSE_ENOMEM : BSE_ECUDA;
}
extern "C" const char *bse_last_error(void) { return g_err.c_str(); }
extern "C" const char *bse_version(void) { return "bse_b200 0.1 (sm_100a, fp64)"; }

static const char *k_stage_names[BSE_ST_COUNT] = {
    "screen_syrk", "pair_list", "fwd_plane", "fwd_stick", "pdep_project", "pdep_backproject",
    "inv_stick", "inv_plane", "k1x_accumulate", "pc_overlap", "pc_update", "k1e_density", "k1e_product"};
extern "C" const char *bse_stage_name(int s) { return (s >= 0 && s < BSE_ST_COUNT) ? k_stage_names[s] : "?"; }

namespace {

template <typename T>
int upload(T *&dst, const std::vector<T> &src) {
    BSE_CUDA(cudaMalloc(&dst, std::max<size_t>(src.size(), 1) * sizeof(T)));
    if (!src.empty()) BSE_CUDA(cudaMemcpy(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return BSE_OK;
}

// the accumulate launchers handle the trial blocks 8, 4, 2 or 1 at a time
static int acc_launches(int nb) { return nb / 8 + ((nb & 4) ? 1 : 0) + ((nb & 2) ? 1 : 0) + (nb & 1); }
// accumulate_rows: all whole groups of 8 blocks in ONE launch
static int acc_rows_launches(int nb) { return (nb >= 8 ? 1 : 0) + ((nb & 4) ? 1 : 0) + ((nb & 2) ? 1 : 0) + (nb & 1); }

struct StageTimer {
    bse_handle *h; int st;
    int launches = 1;                              // kernels the stage call launches (set by the caller when not one)
    // bytes: algorithmic HBM bytes by SURVEY 8(d) (fields, coefficients on H, GEMM operands); handoff: bytes of the stick-plane
    // intermediate Z, which exists only because the 3-D transform is split into two kernels (implementation traffic)
    StageTimer(bse_handle *h_, int st_, double flops, double bytes, double handoff = 0.0) : h(h_), st(st_) {
        h->st_flops[st] += flops;
        h->st_bytes[st] += bytes;
        h->st_handoff[st] += handoff;
        if (h->prof) cudaEventRecord(h->ev0, h->stream);
    }
    ~StageTimer() {
        h->st_launch[st] += launches;
        if (h->prof) {
            cudaEventRecord(h->ev1, h->stream);
            cudaEventSynchronize(h->ev1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, h->ev0, h->ev1);
            h->st_ms[st] += ms;
        }
    }
};

// Tables of one FFT grid of edge n (the problem's grid, or the coarser apply grid of the PW layout).  The order of H is
// the normative one of the PROBLEM grid h->n whatever n is, so PW arrays mean the same thing on both grids.
int build_fft_plan(bse_handle *h, FftPlan &pl, int n) {
    pl.n = n;
    pl.N = (long long)n * n * n;
    const int nkey = h->n;
    int rc;
    if ((rc = bse_fft_select(pl))) return rc;
    const int msq = h->msq_max;
    const int R = (int)std::floor(std::sqrt((double)msq) + 1e-9);
    pl.R = R;
    pl.W = R + 1;
    // half sphere H in the normative order
    struct M3 { int m1, m2, m3; long long key; };
    std::vector<M3> H;
    for (int m1 = -R; m1 <= R; ++m1)
        for (int m2 = -R; m2 <= R; ++m2)
            for (int m3 = -R; m3 <= R; ++m3) {
                if (m1 * m1 + m2 * m2 + m3 * m3 > msq) continue;
                const bool half = (m3 > 0) || (m3 == 0 && m2 > 0) || (m3 == 0 && m2 == 0 && m1 >= 0);
                if (!half) continue;
                const long long key = ((long long)((m1 + nkey) % nkey) * nkey + (m2 + nkey) % nkey) * nkey + (m3 + nkey) % nkey;
                H.push_back({m1, m2, m3, key});
            }
    std::sort(H.begin(), H.end(), [](const M3 &a, const M3 &b) { return a.key < b.key; });
    pl.npw_h = (long long)H.size();
    const int D = 2 * R + 1;
    std::vector<int> hidx((size_t)D * D * D, -1);
    auto hid = [&](int m1, int m2, int m3) -> int & { return hidx[((size_t)(m1 + R) * D + (m2 + R)) * D + (m3 + R)]; };
    h->mill.resize(H.size() * 3);
    std::vector<double> vc12(H.size()), vc12n(H.size()), inv2n(H.size()), vcn(H.size());
    const double twopi_L = 2.0 * M_PI / h->L;
    for (size_t i = 0; i < H.size(); ++i) {
        hid(H[i].m1, H[i].m2, H[i].m3) = (int)i;
        h->mill[3 * i] = H[i].m1; h->mill[3 * i + 1] = H[i].m2; h->mill[3 * i + 2] = H[i].m3;
        const int q = H[i].m1 * H[i].m1 + H[i].m2 * H[i].m2 + H[i].m3 * H[i].m3;
        vc12[i] = q == 0 ? 0.0 : std::sqrt(4.0 * M_PI) / (twopi_L * std::sqrt((double)q));
        vc12n[i] = vc12[i] / (2.0 * (double)pl.N);
        inv2n[i] = 1.0 / (2.0 * (double)pl.N);
        vcn[i] = vc12[i] * vc12[i] / (2.0 * (double)pl.N);
    }
    // half sticks ordered by (t2 = m2 mod n, m3): stick index = soff[t2] + m3 for wmin[t2] <= m3 <= wmax[t2]
    std::vector<int> soff(n, 0), wmax(n, -1), wmin(n, 0);
    struct St { int m2, m3; };
    std::vector<St> sticks;
    for (int t2 = 0; t2 < n; ++t2) {
        const int m2 = t2 < n / 2 ? t2 : t2 - n;
        if (std::abs(m2) > R || 2 * t2 == n) continue;
        const int lo = m2 < 0 ? 1 : 0;
        int hi = -1;
        for (int m3 = 0; m3 <= R; ++m3)
            if (m2 * m2 + m3 * m3 <= msq) hi = m3;
        wmin[t2] = lo;
        wmax[t2] = hi;
        soff[t2] = (int)sticks.size() - lo;
        for (int m3 = lo; m3 <= hi; ++m3) sticks.push_back({m2, m3});
    }
    pl.NS = (int)sticks.size();
    std::vector<int> hmapT((size_t)n * pl.NS, -1);
    for (int s = 0; s < pl.NS; ++s) {
        const int m2 = sticks[s].m2, m3 = sticks[s].m3;
        for (int t1 = 0; t1 < n; ++t1) {
            const int m1 = t1 < n / 2 ? t1 : t1 - n;
            int v = -1;
            if (2 * t1 != n && std::abs(m1) <= R && m1 * m1 + m2 * m2 + m3 * m3 <= msq) {
                v = hid(m1, m2, m3);
                if (v < 0) v = -2 - hid(-m1, -m2, -m3);      // only the (0,0) stick, m1 < 0
            }
            hmapT[(size_t)t1 * pl.NS + s] = v;
        }
    }
    std::vector<double2> tw(n);
    for (int t = 0; t < n; ++t) {
        const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)t / (long double)n;
        tw[t] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
    if ((rc = upload(pl.tw, tw))) return rc;
    if ((rc = upload(pl.soff, soff))) return rc;
    if ((rc = upload(pl.wmax, wmax))) return rc;
    if ((rc = upload(pl.wmin, wmin))) return rc;
    if ((rc = upload(pl.hmapT, hmapT))) return rc;
    if ((rc = upload(pl.vc12, vc12))) return rc;
    if ((rc = upload(pl.vc12n, vc12n))) return rc;
    if ((rc = upload(pl.inv2n, inv2n))) return rc;
    if ((rc = upload(pl.vcn, vcn))) return rc;
    return BSE_OK;
}

void free_plan(FftPlan &pl) {
    cudaFree(pl.tw); cudaFree(pl.soff); cudaFree(pl.wmax); cudaFree(pl.wmin); cudaFree(pl.hmapT);
    cudaFree(pl.vc12); cudaFree(pl.vc12n); cudaFree(pl.inv2n); cudaFree(pl.vcn);
}

inline long long ldD(const bse_handle *h) { return (h->Npdep + 1) & ~1; }
inline long long ldS(const bse_handle *h) { return (h->Nv + 1) & ~1; }

// ---------------------------------------------------------------------------------------------------------
// Stage wrappers: one kernel sequence + its event timer + its ALGORITHMIC flops and compulsory HBM bytes (the roofline
// model of DESIGN.md section 6; bse_profile_model returns the sums).  lg = log2(n); z = bytes of one field's stick
// planes Z; g = bytes of one field on H.
struct Model {
    double lg, N8, z, g, plane_flops, stick_flops;
    explicit Model(const FftPlan &pl) {
        const double n = pl.n;
        lg = std::log2(n);
        N8 = 8.0 * (double)pl.N;
        z = 16.0 * n * pl.NS;
        g = 16.0 * (double)pl.npw_h;
        plane_flops = 2.5 * n * n * n * lg + 5.0 * n * n * pl.W * lg;         // n^2 real rows + n W kept columns
        stick_flops = 5.0 * n * lg * pl.NS;
    }
};

int st_fwd_plane(bse_handle *h, const FftPlan &pl, const double *fields, const int2 *pairs, long long p0, int cnt) {
    const Model m(pl);
    StageTimer t(h, BSE_ST_FWD_PLANE, cnt * m.plane_flops, cnt * m.N8, cnt * m.z);
    return bse_launch_fwd_plane(pl, fields, pairs, p0, cnt, pl.N, h->Z, h->stream);
}
int st_fwd_stick(bse_handle *h, const FftPlan &pl, int cnt, double2 *X, const double *scale, const int *scatter = nullptr) {
    const Model m(pl);
    StageTimer t(h, BSE_ST_FWD_STICK, cnt * m.stick_flops, cnt * m.g, cnt * m.z);
    return bse_launch_fwd_stick(pl, h->Z, cnt, X, scale, h->stream, scatter);
}
int st_inv_stick(bse_handle *h, const FftPlan &pl, const double2 *T, int cnt) {
    const Model m(pl);
    StageTimer t(h, BSE_ST_INV_STICK, cnt * m.stick_flops, cnt * m.g, cnt * m.z);
    return bse_launch_inv_stick(pl, T, cnt, h->Z, h->stream);
}
int st_inv_plane(bse_handle *h, const FftPlan &pl, int cnt, double *out) {
    const Model m(pl);
    StageTimer t(h, BSE_ST_INV_PLANE, cnt * m.plane_flops, cnt * m.N8, cnt * m.z);
    return bse_launch_inv_plane(pl, h->Z, cnt, pl.N, out, h->stream);
}
// C[M][Nn] = alpha colscale[n] sum_k A[m][k] B[n][k]   (split-K DMMA)
int st_gemm_dot(bse_handle *h, int stage, const double *A, long long lda, const double *B, long long ldb, int M, int Nn,
                long long K, bool sq, double *C, long long ldc, double alpha, const double *colscale, bool accumulate = false) {
    const double flops = sq ? (double)M * (Nn + 1) * (double)K : 2.0 * M * Nn * (double)K;
    const double bytes = sq ? 8.0 * M * (double)K : 8.0 * ((double)M * K + (double)Nn * K);
    StageTimer t(h, stage, flops, bytes);
    return bse_gemm_dot(A, lda, B, ldb, M, Nn, K, sq, sq, h->part, h->part_bytes, C, ldc, alpha, colscale, h->stream, accumulate);
}
// NN form with the EPI_TAU / EPI_SUB epilogue: reads A [M][K], B [K][Nn], one [M][Nn] operand, writes [M][Nn]
int st_gemm_nn(bse_handle *h, int stage, const double *A, long long lda, const double *B, long long ldb, int M,
               long long Nn, int K, int epi, const double *Xin, const double *cs2, double *C, long long ldc) {
    StageTimer t(h, stage, 2.0 * M * (double)Nn * K, 8.0 * (2.0 * M * (double)Nn + (double)K * Nn));
    return bse_gemm_nn(A, lda, B, ldb, M, Nn, K, epi, Xin, cs2, C, ldc, h->stream);
}
// a10 for the pairs [p0, p0+cnt): compulsory traffic = tau of the batch; a and acc once per call (charged to the
// first batch); flops 2 nb N per directed pair
int st_accumulate(bse_handle *h, const double *tau, long long p0, long long cnt, const double *a, double *acc, int nb,
                  bool first) {
    const Model m(h->fft);
    const double directed = (double)h->nadj * (double)cnt / (double)std::max<long long>(h->P, 1);
    StageTimer t(h, BSE_ST_ACCUM, 2.0 * nb * (double)h->N * directed,
                 m.N8 * ((double)cnt + (first ? 2.0 * nb * h->Nv : 0.0)));
    t.launches = acc_launches(nb);
    return bse_launch_accumulate(h, tau, p0, cnt, a, acc, nb, first);
}

// tau for pairs [p0, p0+cnt): a2..a8 into dstG ([cnt][npw_h] complex), then a9 into dstR ([cnt][N]) if given
int run_pair_batch(bse_handle *h, const int2 *plist, long long p0, int cnt, double2 *dstG, double *dstR) {
    const FftPlan &pl = h->fft;
    const long long K2 = 2 * pl.npw_h;
    int rc;
    if ((rc = st_fwd_plane(h, pl, h->u, plist, p0, cnt))) return rc;
    if ((rc = st_fwd_stick(h, pl, cnt, h->X, pl.vc12n))) return rc;
    if ((rc = st_gemm_dot(h, BSE_ST_PROJECT, (const double *)h->X, K2, h->phi, K2, cnt, h->Npdep, K2, false, h->Dm,
                          ldD(h), 1.0, h->f2))) return rc;
    if ((rc = st_gemm_nn(h, BSE_ST_BACKPROJECT, h->Dm, ldD(h), h->phi, K2, cnt, K2, h->Npdep, EPI_TAU,
                         (const double *)h->X, pl.vc12, (double *)dstG, K2))) return rc;
    if (dstR) {
        if ((rc = st_inv_stick(h, pl, dstG, cnt))) return rc;
        if ((rc = st_inv_plane(h, pl, cnt, dstR))) return rc;
    }
    return BSE_OK;
}

int ensure_sov(bse_handle *h, long long rows) {
    const long long lds = ldS(h);
    if (h->Sov_elems < (size_t)(rows * lds)) {
        cudaFree(h->Sov);
        h->Sov = nullptr;
        h->Sov_elems = 0;
        BSE_CUDA(cudaMalloc(&h->Sov, (size_t)(rows * lds) * 8));
        h->Sov_elems = (size_t)(rows * lds);
    }
    return BSE_OK;
}

// P_c on `rows` vectors of length K held in x: S = x ub^T (split-K dot GEMM; ub carries the inner
// product's weights), x -= S uk (NN GEMM).  REAL: ub = uk = u, alpha = dV.  PW: ub = uGw, uk = uG, alpha = 1.
int p_c_rows(bse_handle *h, double *x, long long rows, long long K, const double *ub, const double *uk, double alpha) {
    const long long lds = ldS(h);
    int rc;
    if ((rc = ensure_sov(h, rows))) return rc;
    long long mc = rows;
    const long long per_row = (long long)h->Nv * 8 * 2;
    const long long chunk_bytes = (long long)std::min<size_t>(h->part_bytes, (size_t)64 << 20);
    if (rows * per_row > chunk_bytes) mc = std::max<long long>(64, (chunk_bytes / per_row) / 64 * 64);
    // host-pointer apply: finished chunks leave for the host while the next is projected, and what stays exposed at the end is
    // the LAST chunk's copy: ~16 chunks instead of 4 (cfg 5: 8.1 GB -> 2 GB behind the last projection)
    if (h->d2h_host && x == h->out_dev) mc = std::min(mc, std::max<long long>(256, ((rows + 15) / 16 + 63) / 64 * 64));
    if (h->dbg_pc_rows >= 1) mc = std::min(mc, h->dbg_pc_rows);
    for (long long r0 = 0; r0 < rows; r0 += mc) {
        const int m = (int)std::min(mc, rows - r0);
        if ((rc = st_gemm_dot(h, BSE_ST_PC_OVERLAP, x + r0 * K, K, ub, K, m, h->Nv, K, false, h->Sov + r0 * lds, lds,
                              alpha, nullptr))) return rc;
        if ((rc = st_gemm_nn(h, BSE_ST_PC_UPDATE, h->Sov + r0 * lds, lds, uk, K, m, K, h->Nv, EPI_SUB, nullptr, nullptr,
                             x + r0 * K, K))) return rc;
        if (h->d2h_host && x == h->out_dev && r0 == h->d2h_rows_done) {      // rows [r0, r0 + m) are final: send them off
            BSE_CUDA(cudaEventRecord(h->ev_d2h, h->stream));
            BSE_CUDA(cudaStreamWaitEvent(h->s_out, h->ev_d2h, 0));
            BSE_CUDA(cudaMemcpyAsync(h->d2h_host + r0 * K, x + r0 * K, (size_t)m * K * 8, cudaMemcpyDeviceToHost, h->s_out));
            h->d2h_rows_done = r0 + m;
        }
    }
    return BSE_OK;
}

// u_w(G) on H for the PW layout (a12): forward transform of every orbital, no pair product, scale 1/(2N) -> uG;
// uGw = Omega * wt(G) * uG with wt = 2 (G != 0), (1, 0) on (re, im) of G = 0, so that the half-sphere real dot product
// sum_k uGw[w][k] x[k] equals <u_w|x> = Omega sum_{G in S} conj(u_w(G)) x(G)   (S14).
int ensure_u_pw(bse_handle *h) {
    if (h->uG && h->uG_valid) return BSE_OK;
    const FftPlan &pl = h->fft;
    const size_t bytes = (size_t)h->Nv * pl.npw_h * 16;
    if (!h->uG) {                             // kept across bse_set_inputs_host: new orbitals are transformed into the same buffers
        BSE_CUDA(cudaMalloc(&h->uG, bytes));
        BSE_CUDA(cudaMalloc(&h->uGw, bytes));
    }
    int rc;
    for (long long v0 = 0; v0 < h->Nv; v0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, h->Nv - v0);
        if ((rc = st_fwd_plane(h, pl, h->u, nullptr, v0, cnt))) return rc;
        if ((rc = st_fwd_stick(h, pl, cnt, h->uG + v0 * pl.npw_h, pl.inv2n))) return rc;
    }
    if ((rc = bse_launch_weight_pw(h->uG, h->uGw, pl.npw_h, h->Nv, h->Omega, h->stream))) return rc;
    h->uG_valid = true;                       // only once every fill has been enqueued without error
    return BSE_OK;
}

// Is every orbital band-limited to S?  Forms T_S u_v (forward transform, truncation to S, inverse transform) and requires
// ||u_v - T_S u_v|| <= 1e-12 ||u_v||: a norm comparison (Parseval) would only see leakage above ~1e-6 in amplitude.
// Decided once per set of inputs.  Plane-wave orbitals are, by construction.
int ensure_k1e_ws(bse_handle *h, size_t bytes);     // grow-only scratch, defined with the K1e helpers below

int check_band_limited(bse_handle *h) {
    if (h->u_bl >= 0) return BSE_OK;
    int rc;
    if ((rc = ensure_u_pw(h))) return rc;
    const FftPlan &pl = h->fft;
    const long long Nv = h->Nv;
    const int chunk = (int)std::min<long long>(std::min<long long>(h->Pb, 32), Nv);
    if ((rc = ensure_k1e_ws(h, (size_t)chunk * h->N * 8))) return rc;      // T_S u of a few orbitals at a time
    if ((rc = ensure_sov(h, 2))) return rc;                              // >= 2 Nv doubles of scratch
    for (long long v0 = 0; v0 < Nv; v0 += chunk) {
        const int cnt = (int)std::min<long long>(chunk, Nv - v0);
        if ((rc = st_inv_stick(h, pl, h->uG + v0 * pl.npw_h, cnt))) return rc;
        if ((rc = st_inv_plane(h, pl, cnt, h->k1e_ws))) return rc;
        if ((rc = bse_launch_row_sumsq(h->u + v0 * h->N, h->k1e_ws, h->N, cnt, h->Sov + 2 * v0, h->stream))) return rc;
    }
    std::vector<double> host((size_t)2 * Nv);
    BSE_CUDA(cudaMemcpyAsync(host.data(), h->Sov, host.size() * 8, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    bool ok = true;
    for (long long v = 0; v < Nv; ++v)                                   // || u_v - T_S u_v || <= 1e-12 || u_v ||
        if (!(host[2 * v + 1] <= 1e-24 * host[2 * v])) ok = false;
    h->u_bl = ok ? 1 : 0;
    return BSE_OK;
}

// P_c on REAL-layout rows when u is band-limited to S: <u_w|x> = Omega sum_S conj(u_w(G)) x(G) needs x only on S, so the
// overlaps come from one pruned forward transform per row and a GEMM over 2 N_pw_h instead of N (16x fewer flops);
// and so does the correction: x -= inverse transform of (S u)(G), fused into the inverse plane pass (x itself is not
// truncated: S15).
int p_c_rows_real(bse_handle *h, double *x, long long rows) {
    int rc;
    if ((rc = check_band_limited(h))) return rc;
    if (h->u_bl != 1) return p_c_rows(h, x, rows, h->N, h->u, h->u, h->dV);
    const FftPlan &pl = h->fft;
    const long long npw_h = pl.npw_h, K2 = 2 * npw_h, lds = ldS(h);
    if (h->accG_rows < rows) {
        cudaFree(h->accG);
        h->accG = nullptr; h->accG_rows = 0;
        BSE_CUDA(cudaMalloc(&h->accG, (size_t)rows * npw_h * 16));
        h->accG_rows = rows;
    }
    for (long long r0 = 0; r0 < rows; r0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, rows - r0);
        if ((rc = st_fwd_plane(h, pl, x, nullptr, r0, cnt))) return rc;
        if ((rc = st_fwd_stick(h, pl, cnt, h->accG + r0 * npw_h, pl.inv2n))) return rc;
    }
    if ((rc = ensure_sov(h, rows))) return rc;
    long long mc = rows;
    const long long per_row = (long long)h->Nv * 8 * 2;
    if (rows * per_row > (long long)h->part_bytes) mc = std::max<long long>(64, (long long)(h->part_bytes / per_row) / 64 * 64);
    const Model m(pl);
    for (long long r0 = 0; r0 < rows; r0 += mc) {
        const int mm = (int)std::min(mc, rows - r0);
        double *ag = (double *)(h->accG + r0 * npw_h);
        if ((rc = st_gemm_dot(h, BSE_ST_PC_OVERLAP, ag, K2, (const double *)h->uGw, K2, mm, h->Nv, K2, false,
                              h->Sov + r0 * lds, lds, 1.0, nullptr))) return rc;
        if (h->Nv < 48) {        // few orbitals: the real-space DGEMM update (2 Nv N flops per row) beats a transform per row
            if ((rc = st_gemm_nn(h, BSE_ST_PC_UPDATE, h->Sov + r0 * lds, lds, h->u, h->N, mm, h->N, h->Nv, EPI_SUB, nullptr,
                                 nullptr, x + r0 * h->N, h->N))) return rc;
            continue;
        }
        // the correction sum_w S_w u_w is band-limited too: form it on H (small NN GEMM over the rows' coefficients, which
        // are no longer needed) and subtract its inverse transform in the plane pass's store
        if ((rc = st_gemm_nn(h, BSE_ST_PC_UPDATE, h->Sov + r0 * lds, lds, (const double *)h->uG, K2, mm, K2, h->Nv, EPI_STORE,
                             nullptr, nullptr, ag, K2))) return rc;
        for (long long c0 = 0; c0 < mm; c0 += h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, mm - c0);
            if ((rc = st_inv_stick(h, pl, h->accG + (r0 + c0) * npw_h, cnt))) return rc;
            StageTimer t(h, BSE_ST_PC_UPDATE, cnt * m.plane_flops, cnt * 2.0 * m.N8, cnt * m.z);
            if ((rc = bse_launch_inv_plane(pl, h->Z, cnt, pl.N, x + (r0 + c0) * h->N, h->stream, true))) return rc;
        }
    }
    return BSE_OK;
}


// pair-batch workspaces Z, X, T, Dm for `pb` fields (tau_batch follows lazily); called at create and again after the
// pair list is known if one row of the adjacency has more entries than the batch holds
int alloc_batch_ws(bse_handle *h, long long pb) {
    cudaFree(h->Z); cudaFree(h->X); cudaFree(h->T); cudaFree(h->Dm); cudaFree(h->tau_batch);
    h->Z = h->X = h->T = nullptr; h->Dm = nullptr; h->tau_batch = nullptr;
    h->Pb = 0;
    if (cudaMalloc(&h->Z, (size_t)pb * h->n * h->fft.NS * 16) || cudaMalloc(&h->X, (size_t)pb * h->fft.npw_h * 16) ||
        cudaMalloc(&h->T, (size_t)pb * h->fft.npw_h * 16) || cudaMalloc(&h->Dm, (size_t)pb * ldD(h) * 8)) {
        (void)cudaGetLastError();
        bse_set_error("out of device memory (pair-batch workspaces)");
        return BSE_ENOMEM;
    }
    h->Pb_alloc = pb;
    h->Pb = pb >= 64 ? pb / 64 * 64 : pb;          // whole 64-row CTA tiles in the PDEP GEMMs (297 pairs cost as much as 320)
    return BSE_OK;
}

// tau store of the REAL / PW modes (grow-only); BSE_TAU_STREAM uses the PW store as a transient that is refilled inside
// every apply call (tau(G) is 16 N / N_pw_h ~ 16x smaller than tau(r), which stays streamed in batches)
int ensure_tau_store(bse_handle *h, bool real) {
    const bool f32 = !real && (h->flags & BSE_TAU_F32);         // tau(G) kept as complex64 (single precision)
    const size_t need = real ? (size_t)h->Pa * h->N * 8 : (size_t)h->Pa * h->fft.npw_h * (f32 ? 8 : 16);
    const bool have = real ? h->tau_r != nullptr : (f32 ? h->tau_g32 != nullptr : h->tau_g != nullptr);
    if (need <= h->tau_bytes && have) return BSE_OK;
    cudaFree(h->tau_r); h->tau_r = nullptr;
    cudaFree(h->tau_g); h->tau_g = nullptr;
    cudaFree(h->tau_g32); h->tau_g32 = nullptr;
    h->tau_bytes = 0;
    size_t free_b = 0, total_b = 0;
    cudaMemGetInfo(&free_b, &total_b);
    if (need + ((size_t)256 << 20) > free_b) {
        char msg[160];
        snprintf(msg, sizeof msg, "tau store needs %.2f GB, %.2f GB free%s", need / 1e9, free_b / 1e9,
                 real ? ": use BSE_TAU_PW or BSE_TAU_STREAM" : "");
        bse_set_error(msg);
        return BSE_ENOMEM;
    }
    if (real) BSE_CUDA(cudaMalloc(&h->tau_r, need));
    else if (f32) BSE_CUDA(cudaMalloc(&h->tau_g32, need));
    else BSE_CUDA(cudaMalloc(&h->tau_g, need));
    h->tau_bytes = need;
    return BSE_OK;
}

int fill_tau_store(bse_handle *h, bool real) {
    int rc;
    cudaEventRecord(h->ev_fill0, h->stream);        // device time of the pair integrals alone (bse_last_tau_fill_ms)
    const int2 *plist = h->rows_set ? h->pairs_act : h->pairs;       // row-sharded: only the pairs that touch an owned row
    for (long long p0 = 0; p0 < h->Pa; p0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, h->Pa - p0);
        if (real) rc = run_pair_batch(h, plist, p0, cnt, h->T, h->tau_r + p0 * h->N);
        else if (h->tau_g32) {                                   // the batch in double (workspace T), rounded once into the store
            rc = run_pair_batch(h, plist, p0, cnt, h->T, nullptr);
            if (!rc) rc = bse_launch_to_f32((const double *)h->T, (float *)(h->tau_g32 + p0 * h->fft.npw_h),
                                            2 * (long long)cnt * h->fft.npw_h, h->stream);
        } else rc = run_pair_batch(h, plist, p0, cnt, h->tau_g + p0 * h->fft.npw_h, nullptr);
        if (rc) return rc;
    }
    cudaEventRecord(h->ev_fill1, h->stream);
    h->fill_timed = true;
    return BSE_OK;
}

// Row batches of the batched tau modes.  A batch is a CLUSTER of rows grown greedily over the pair graph: starting from
// the lowest row not yet placed, the row with the most neighbours already inside the batch is added while the pairs the
// batch touches (each counted once: a pair with both ends inside serves both rows) fit the tau(r) batch buffer and the
// rows fit acc_r.  Compact clusters share pairs (fewer tau(r) inversions than rows in list order) and touch few
// distinct neighbours (fewer re-reads of a).  rowlist holds the rows of all batches, batch after batch.
int plan_row_batches(bse_handle *h, int rows_cap) {
    const std::vector<int> &ap = h->adj_ptr_h;
    const int Nv = h->Nv;
    h->batches.clear();
    std::vector<int> pairs_all, eslot((size_t)h->nadj), mark((size_t)std::max<long long>(h->P, 1), -1), rowlist;
    std::vector<int> cur, score((size_t)Nv, 0), touched;
    std::vector<char> placed((size_t)Nv, 0);
    rowlist.reserve(Nv);
    int next_seed = 0, tag = 0;
    while ((int)rowlist.size() < Nv) {
        while (placed[next_seed]) ++next_seed;
        cur.clear();
        touched.clear();
        const int r0 = (int)rowlist.size();
        int v = next_seed;
        for (;;) {
            int fresh = 0;
            for (int e = ap[v]; e < ap[v + 1]; ++e) fresh += mark[h->adj_h[2 * e + 1]] != tag ? 1 : 0;
            if ((int)rowlist.size() > r0 && (long long)cur.size() + fresh > h->Pacc) break;
            placed[v] = 1;
            rowlist.push_back(v);
            for (int e = ap[v]; e < ap[v + 1]; ++e) {
                const int pidx = h->adj_h[2 * e + 1], u = h->adj_h[2 * e];
                if (mark[pidx] != tag) { mark[pidx] = tag; cur.push_back(pidx); }
                if (!placed[u]) { if (score[u]++ == 0) touched.push_back(u); }
            }
            if ((int)rowlist.size() - r0 >= rows_cap || (int)rowlist.size() >= Nv) break;
            int best = -1, bs = 0;                              // most neighbours already in the batch; ties: lowest row
            for (int u : touched)
                if (!placed[u] && (score[u] > bs || (score[u] == bs && u < best))) { bs = score[u]; best = u; }
            if (best < 0) {                                     // the component is exhausted: continue with the next unplaced row
                int s2 = next_seed;
                while (s2 < Nv && placed[s2]) ++s2;
                if (s2 >= Nv) break;
                best = s2;
            }
            v = best;
        }
        for (int u : touched) score[u] = 0;
        std::sort(cur.begin(), cur.end());                     // ascending pair index: sequential reads of the tau(G) store
        for (int i = r0; i < (int)rowlist.size(); ++i) {
            const int row = rowlist[i];
            for (int e = ap[row]; e < ap[row + 1]; ++e)
                eslot[e] = (int)(std::lower_bound(cur.begin(), cur.end(), h->adj_h[2 * e + 1]) - cur.begin());
        }
        h->batches.push_back({r0, (int)rowlist.size(), (int)pairs_all.size(), (int)cur.size()});
        pairs_all.insert(pairs_all.end(), cur.begin(), cur.end());
        ++tag;
    }
    h->uniq_share = (double)h->P / (double)std::max<size_t>(pairs_all.size(), 1);
    cudaFree(h->batch_pairs); cudaFree(h->eslot); cudaFree(h->rowlist);
    h->batch_pairs = h->eslot = h->rowlist = nullptr;
    BSE_CUDA(cudaMalloc(&h->batch_pairs, std::max<size_t>(pairs_all.size(), 1) * 4));
    BSE_CUDA(cudaMalloc(&h->eslot, std::max<size_t>(eslot.size(), 1) * 4));
    BSE_CUDA(cudaMalloc(&h->rowlist, (size_t)Nv * 4));
    BSE_CUDA(cudaMemcpyAsync(h->batch_pairs, pairs_all.data(), pairs_all.size() * 4, cudaMemcpyHostToDevice, h->stream));
    BSE_CUDA(cudaMemcpyAsync(h->eslot, eslot.data(), eslot.size() * 4, cudaMemcpyHostToDevice, h->stream));
    BSE_CUDA(cudaMemcpyAsync(h->rowlist, rowlist.data(), (size_t)Nv * 4, cudaMemcpyHostToDevice, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));                // the host vectors go out of scope
    return BSE_OK;
}

// Memory plan of the apply, made from what is free at the first call (and again if B grows or the list changes):
//   tau_batch [Pacc][N]   tau(r) of the directed entries of one row batch (batched tau modes)
//   a_r  [Bg][Nv][N]      PW layout: real-space trial blocks of one group (every neighbour of a row may be needed)
//   acc_r[Bg][rows_cap][N] PW layout: accumulated rows of the current row batch (all Nv rows with BSE_TAU_REAL)
// A larger row batch re-reads a fewer times and lets rows that share neighbours hit L2, a larger group inverts tau fewer
// times: 60 % of the free memory goes to the group, the rest to the batch.
int plan_apply_memory(bse_handle *h, int B, bool allow_slab = true, bool mix = false) {
    const bool pw = (h->flags & BSE_VEC_PW) != 0;
    const bool batched = (h->flags & BSE_TAU_MASK) != BSE_TAU_REAL;
    if (h->plan_ok && (h->plan_allow_slab != allow_slab || (mix && !h->plan_mix))) h->plan_ok = false;
    // the plan is kept only for the very adjacency it was made for (a rebuilt list with the same pair count but other
    // pairs must not reuse the old batches / eslot) and while the group still holds B blocks
    const bool same_list = !batched || (h->plan_adj_ptr_h == h->adj_ptr_h && h->plan_adj_h == h->adj_h);
    if (h->plan_ok && same_list && (!pw || h->Bg >= B || h->Bg_final)) return BSE_OK;
    cudaFree(h->tau_batch); cudaFree(h->a_r); cudaFree(h->acc_r);
    h->tau_batch = h->a_r = h->acc_r = nullptr;
    h->Bg = 0; h->Pacc = 0; h->rows_cap = 0; h->plan_ok = false;
    h->slab_mode = false; h->slab_rc = 0; h->plan_allow_slab = allow_slab; h->plan_mix = mix;
    size_t free_b = 0, total_b = 0;
    cudaMemGetInfo(&free_b, &total_b);
    // Plane-slab streaming (PW layout, tau on H): the whole apply runs on one slab of R2 planes at a time, with a(r) of ALL B
    // blocks and tau(r) of ALL pairs resident for that slab, so every field is inverse-transformed exactly once per call (no
    // trial-block groups, no pair shared between two row batches).  Every slab sweeps the coefficient arrays once, which costs
    // more than it saves while the group path below holds ALL B blocks in one group (cfg 3-4: measured 43 vs 37 ms, 814 vs
    // 735 ms), so the slab path is taken when that path would need several groups (cfg 5: 2.5 vs 3.3 s), on row-sharded
    // handles, and when a slab knob asks for it.
    bool one_group = false;
    if (pw && batched) {
        const double N8g = 8.0 * (double)h->ap->N, availg = 0.92 * (double)free_b - 512.0 * 1048576.0;
        const double avgd = std::max(1.0, (double)h->nadj / h->Nv);
        int maxd = 1;
        for (int v = 0; v < h->Nv; ++v) maxd = std::max(maxd, h->adj_ptr_h[v + 1] - h->adj_ptr_h[v]);
        const double want = (double)std::max<long long>(maxd, std::min<long long>(h->nadj, 256));
        const double rest = availg - (double)B * h->Nv * N8g;
        one_group = rest > 0 && rest / (N8g * (1.0 + 2.0 * B / avgd)) >= want;
    }
    const bool slab_forced = h->rows_set || h->dbg_slab_rows >= 1 || h->dbg_slab_planes >= 1;
    if (pw && batched && allow_slab && h->dbg_max_group < 1 && h->dbg_max_batch < 1 && h->dbg_slab_rows >= 0 &&
        (slab_forced || !one_group)) {
        const FftPlan &pl = *h->ap;
        const double avail_s = 0.92 * (double)free_b - 512.0 * 1048576.0;
        // the slab split n_a = S * M (any factorisation with M <= 16 and S <= 16, fft_slab.cuh): the fewest slabs whose working set fits,
        // because every slab sweeps all coefficient arrays once.  dbg_slab_planes caps M (tests: several slabs on small grids).
        long long rc = 0, pz = 0;
        int Ssel = 0, Msel = 0;
        double SN8 = 0.0;
        // M <= 16: 32 M <= 512 threads per CTA keeps the slab stick kernels at two CTAs per SM with 128 registers; measured at
        // cfg 5 (complex64 store, where memory would allow more): M = 20 costs 114 ms per sweep against 73 ms at M = 15
        for (int M = std::min(pl.n, 16); M >= 1; --M) {
            if (pl.n % M || pl.n / M > 16) continue;           // the slab stick kernels keep <= 16 folded terms per thread
            if (h->dbg_slab_planes >= 1 && M > h->dbg_slab_planes) continue;
            SN8 = 8.0 * (double)M * pl.n * pl.n;
            // a(r) of all blocks + tau(r) of all (owned) pairs; the combined call also keeps u and v_H of the slab (k1e_ws)
            const double fixed = ((double)B * h->Nv + (double)h->Pa + (mix ? (double)h->Nv + 2.0 * B : 0.0)) * SN8;
            pz = (long long)(((double)h->Pb_alloc * h->n * h->fft.NS) / ((double)M * pl.NS));
            rc = (long long)((avail_s - fixed) / ((double)B * SN8));
            rc = std::min<long long>(rc, std::min<long long>(pz / B, 65535 / B));
            rc = std::min<long long>(rc, std::min<long long>(h->Nv, 256));
            if (h->dbg_slab_rows >= 1) rc = std::min<long long>(rc, h->dbg_slab_rows);
            if (rc >= std::min<long long>(h->Nv, 32) || (h->dbg_slab_rows >= 1 && rc >= 1) || (M == 1 && rc >= 1)) {
                Ssel = pl.n / M; Msel = M;
                break;
            }
            rc = 0;
        }
        if (Msel >= 1 && rc >= 1) {
            BSE_CUDA(cudaMalloc(&h->a_r, (size_t)((double)B * h->Nv * SN8)));
            h->a_r_elems = (size_t)((double)B * h->Nv * SN8 / 8.0);
            BSE_CUDA(cudaMalloc(&h->tau_batch, (size_t)std::max<double>((double)h->Pa * SN8, 8.0)));
            BSE_CUDA(cudaMalloc(&h->acc_r, (size_t)((double)B * rc * SN8)));
            if (!h->rowid) {
                std::vector<int> ids((size_t)h->Nv);
                for (int v = 0; v < h->Nv; ++v) ids[v] = v;
                BSE_CUDA(cudaMalloc(&h->rowid, (size_t)h->Nv * 4));
                BSE_CUDA(cudaMemcpy(h->rowid, ids.data(), (size_t)h->Nv * 4, cudaMemcpyHostToDevice));
            }
            h->slab_mode = true; h->slab_rc = (int)rc; h->slab_pz = pz; h->slab_S = Ssel; h->slab_M = Msel;
            h->Bg = B; h->Bg_final = false;
            h->plan_ok = true;
            h->plan_adj_ptr_h = h->adj_ptr_h;
            h->plan_adj_h = h->adj_h;
            return BSE_OK;
        }
    }
    const double N8 = 8.0 * (double)h->ap->N;      // staging lives on the apply grid
    const double avail = 0.92 * (double)free_b - 512.0 * 1048576.0;   // leave the caller some room
    const double avgdeg = std::max(1.0, (double)h->nadj / h->Nv);
    int maxdeg = 1;
    for (int v = 0; v < h->Nv; ++v) maxdeg = std::max(maxdeg, h->adj_ptr_h[v + 1] - h->adj_ptr_h[v]);
    auto nomem = [&](const char *what, double need) {
        char msg[200];
        snprintf(msg, sizeof msg, "%s needs %.2f GB, %.2f GB free", what, need / 1e9, free_b / 1e9);
        bse_set_error(msg);
        return BSE_ENOMEM;
    };
    long long bg = 0, pacc = 0, rows_cap = 0;
    if (!pw) {
        if (batched) {
            pacc = (long long)std::min<double>((double)h->nadj, 0.9 * avail / N8);
            if (pacc < maxdeg) return nomem("tau(r) of one row of pairs", maxdeg * N8);
        }
    } else if (!batched) {
        bg = (long long)std::min<double>(B, avail / (2.0 * h->Nv * N8));
        if (bg < 1) return nomem("real-space staging of one trial block (PW layout)", 2.0 * h->Nv * N8);
        rows_cap = h->Nv;
    } else {
        // tau(r) of every directed entry is re-made once per group, so take the fewest groups whose row batch still
        // holds max(longest row, min(nadj, 256)) entries; then the smallest group size with that many groups
        const long long want = std::max<long long>(maxdeg, std::min<long long>(h->nadj, 256));
        auto pacc_of = [&](long long g) {
            const double rest = avail - (double)g * h->Nv * N8;
            return rest <= 0 ? 0LL : (long long)std::min<double>((double)h->nadj, rest / (N8 * (1.0 + 2.0 * g / avgdeg)));
        };
        bg = B;
        while (bg >= 1 && pacc_of(bg) < want) --bg;
        if (bg < 1) return nomem("real-space staging of one trial block plus one row batch (PW layout)",
                                 (h->Nv + 2.0 * want) * N8);
        const long long groups = (B + bg - 1) / bg;
        while (bg > 1 && (B + bg - 2) / (bg - 1) == groups) --bg;
        pacc = pacc_of(bg);
        rows_cap = std::min<long long>(h->Nv, std::max<long long>(1, (long long)(2.0 * pacc / avgdeg)));
    }
    // test knobs (bse_debug_set): cap B_g / the row batch so that small cases exercise several groups and several row
    // batches (tests/test_gpu_parity.py); they never raise a limit
    if (h->dbg_max_group >= 1 && bg > h->dbg_max_group) bg = h->dbg_max_group;
    if (h->dbg_max_batch >= 1) {
        const long long cap_p = std::max<long long>(h->dbg_max_batch, maxdeg);
        if (pacc > cap_p) {
            pacc = cap_p;
            if (pw && batched) rows_cap = std::min<long long>(h->Nv, std::max<long long>(1, (long long)(2.0 * pacc / avgdeg)));
        }
    }
    if (pacc) BSE_CUDA(cudaMalloc(&h->tau_batch, (size_t)pacc * h->ap->N * 8));
    if (bg) {
        BSE_CUDA(cudaMalloc(&h->a_r, (size_t)bg * h->Nv * h->ap->N * 8));
        h->a_r_elems = (size_t)bg * h->Nv * h->ap->N;
        BSE_CUDA(cudaMalloc(&h->acc_r, (size_t)bg * rows_cap * h->ap->N * 8));
    }
    h->Bg = (int)bg; h->Bg_final = bg < B; h->Pacc = pacc; h->rows_cap = (int)rows_cap;
    if (batched) {
        int rc = plan_row_batches(h, pw ? (int)rows_cap : h->Nv);
        if (rc) return rc;
    }
    h->plan_ok = true;
    h->plan_adj_ptr_h = h->adj_ptr_h;
    h->plan_adj_h = h->adj_h;
    return BSE_OK;
}

// ---- K1e helpers (eq. 4): workspace, Hartree potential in place, orbitals on the apply grid
int ensure_k1e_ws(bse_handle *h, size_t bytes) {
    if (h->k1e_bytes >= bytes) return BSE_OK;
    cudaFree(h->k1e_ws);
    h->k1e_ws = nullptr; h->k1e_bytes = 0;
    if (cudaMalloc(&h->k1e_ws, bytes) != cudaSuccess) {
        // the K1x apply plan holds the free memory: drop it (the next apply plans again around this workspace)
        (void)cudaGetLastError();
        h->k1e_ws = nullptr;
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        cudaFree(h->tau_batch); cudaFree(h->a_r); cudaFree(h->acc_r);
        h->tau_batch = h->a_r = h->acc_r = nullptr;
        h->Bg = 0; h->Pacc = 0; h->rows_cap = 0; h->plan_ok = false;
        BSE_CUDA(cudaMalloc(&h->k1e_ws, bytes));
    }
    h->k1e_bytes = bytes;
    return BSE_OK;
}

// n -> v_H in place for cnt fields held at buf ([cnt][pl.N]): forward transform with the v_c / N scaling (a3 + a4 with
// v_c instead of v_c^{1/2}), inverse transform (a9)
int hartree_in_place(bse_handle *h, const FftPlan &pl, double *buf, int nfields) {
    int rc;
    for (int c0 = 0; c0 < nfields; c0 += (int)h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, nfields - c0);
        if ((rc = st_fwd_plane(h, pl, buf, nullptr, c0, cnt))) return rc;
        if ((rc = st_fwd_stick(h, pl, cnt, h->X, pl.vcn))) return rc;
        if ((rc = st_inv_stick(h, pl, h->X, cnt))) return rc;
        if ((rc = st_inv_plane(h, pl, cnt, buf + (long long)c0 * pl.N))) return rc;
    }
    return BSE_OK;
}

// orbitals on the apply grid of the PW layout: u_a = inverse transform of u(G) on n_a (u is band-limited to S)
int ensure_u_apply(bse_handle *h) {
    if (h->ap == &h->fft || (h->u_a && h->u_a_valid)) return BSE_OK;
    const FftPlan &pl = *h->ap;
    int rc;
    if ((rc = ensure_u_pw(h))) return rc;
    if (!h->u_a && cudaMalloc(&h->u_a, (size_t)h->Nv * pl.N * 8) != cudaSuccess) {
        // the K1x apply plan holds the free memory: drop it (the next K1x apply plans again, with u_a in place)
        (void)cudaGetLastError();
        h->u_a = nullptr;
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        cudaFree(h->tau_batch); cudaFree(h->a_r); cudaFree(h->acc_r);
        h->tau_batch = h->a_r = h->acc_r = nullptr;
        h->Bg = 0; h->Pacc = 0; h->rows_cap = 0; h->plan_ok = false;
        BSE_CUDA(cudaMalloc(&h->u_a, (size_t)h->Nv * pl.N * 8));
    }
    for (long long v0 = 0; v0 < h->Nv; v0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, h->Nv - v0);
        if ((rc = st_inv_stick(h, pl, h->uG + v0 * pl.npw_h, cnt))) return rc;
        if ((rc = st_inv_plane(h, pl, cnt, h->u_a + v0 * pl.N))) return rc;
    }
    h->u_a_valid = true;
    return BSE_OK;
}

// forward transform of `rows` accumulated fields of each of nb blocks into the PW output (a12): acc(G) on H
int rows_to_pw(bse_handle *h, const double *acc, long long acc_ld, int rows, int nb, double2 *out_pw, const int *dest) {
    const FftPlan &pl = *h->ap;
    const long long npw_h = pl.npw_h;
    int rc;
    for (int b = 0; b < nb; ++b)
        for (int r0 = 0; r0 < rows; r0 += (int)h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, rows - r0);
            if ((rc = st_fwd_plane(h, pl, acc + (long long)b * acc_ld * pl.N, nullptr, r0, cnt))) return rc;
            // field p of the launch is row dest[r0 + p] (device array; nullptr: row r0 + p) of block b
            if ((rc = st_fwd_stick(h, pl, cnt, out_pw + (long long)b * h->Nv * npw_h + (dest ? 0 : r0 * npw_h), pl.inv2n,
                                   dest ? dest + r0 : nullptr))) return rc;
        }
    return BSE_OK;
}

// a9 + a10 for nb trial blocks a = [nb][Nv][N] (real space).
//   REAL vec layout: acc_real = out ([nb][Nv][N]), out_pw = nullptr.
//   PW vec layout:   acc_real = nullptr, rows are accumulated in h->acc_r and transformed to out_pw ([nb][Nv][npw_h]).
// BSE_TAU_REAL: one launch over the symmetric pair list.  BSE_TAU_PW / STREAM: row batches; the batch holds tau(r) of every
// directed entry of its rows (inverse FFT gathered from the tau(G) store), so each output row is written once.
int accumulate_all(bse_handle *h, const double *a, int nb, double *acc_real, double2 *out_pw) {
    const unsigned mode = h->flags & BSE_TAU_MASK;
    int rc;
    if (mode == BSE_TAU_REAL) {
        double *acc = acc_real ? acc_real : h->acc_r;
        if ((rc = st_accumulate(h, h->tau_r, 0, h->P, a, acc, nb, true))) return rc;
        if (h->mix_on) {
            StageTimer t(h, BSE_ST_K1E_PRODUCT, 3.0 * nb * h->Nv * (double)h->ap->N, 8.0 * h->ap->N * (2.0 * nb * h->Nv + h->Nv + nb));
            if ((rc = bse_launch_k1_mix(h->mix_u, h->mix_vH, acc, nullptr, h->Nv, h->Nv, false, h->ap->N, nb, h->mix_ce,
                                        h->mix_cd, h->stream))) return rc;
        }
        return out_pw ? rows_to_pw(h, acc, h->Nv, h->Nv, nb, out_pw, nullptr) : BSE_OK;
    }
    const FftPlan &pl = *h->ap;
    const Model m(pl);
    const std::vector<int> &ap = h->adj_ptr_h;
    const double uniq = h->uniq_share;        // share of the inverted fields that is algorithmic work (each pair once)
    for (const bse_handle::RowBatch &bt : h->batches) {
        const int r0 = bt.v0, rows = bt.v1 - bt.v0;               // rows rowlist[r0 .. r0 + rows)
        for (int c0 = 0; c0 < bt.nu; c0 += (int)h->Pb) {              // tau(G) -> tau(r) of the batch's pairs
            const int c = (int)std::min<long long>(h->Pb, bt.nu - c0);
            { StageTimer t(h, BSE_ST_INV_STICK, uniq * c * m.stick_flops, uniq * c * m.g, uniq * c * m.z);
              if ((rc = bse_launch_inv_stick(pl, h->tau_g, c, h->Z, h->stream, h->batch_pairs, bt.u0 + c0, h->tau_g32))) return rc; }
            { StageTimer t(h, BSE_ST_INV_PLANE, uniq * c * m.plane_flops, uniq * c * m.N8, uniq * c * m.z);
              if ((rc = bse_launch_inv_plane(pl, h->Z, c, pl.N, h->tau_batch + (long long)c0 * pl.N, h->stream))) return rc; }
        }
        { StageTimer t(h, BSE_ST_ACCUM, 2.0 * nb * (double)pl.N * (double)h->nadj * rows / h->Nv,
                       m.N8 * (uniq * bt.nu + nb * rows + (r0 == 0 ? (double)nb * h->Nv : 0.0)));
          t.launches = acc_rows_launches(nb);
          if (acc_real) rc = bse_launch_accumulate_rows(h, pl.N, h->tau_batch, h->eslot, h->rowlist + r0, rows, a, acc_real, h->Nv, false, nb);
          else rc = bse_launch_accumulate_rows(h, pl.N, h->tau_batch, h->eslot, h->rowlist + r0, rows, a, h->acc_r, h->rows_cap, true, nb);
          if (rc) return rc; }
        if (h->mix_on) {
            StageTimer t(h, BSE_ST_K1E_PRODUCT, 3.0 * nb * rows * (double)pl.N, m.N8 * (2.0 * nb * rows + rows + nb));
            if (acc_real) rc = bse_launch_k1_mix(h->mix_u, h->mix_vH, acc_real, h->rowlist + r0, rows, h->Nv, false, pl.N, nb,
                                                 h->mix_ce, h->mix_cd, h->stream);
            else if (h->mix_u) rc = bse_launch_k1_mix(h->mix_u, h->mix_vH, h->acc_r, h->rowlist + r0, rows, h->rows_cap, true, pl.N,
                                                      nb, h->mix_ce, h->mix_cd, h->stream);
            else {                                                    // the rows' orbitals on the apply grid, on the fly
                double *ub = h->k1e_ws + (long long)h->mix_B * pl.N;
                for (int c0 = 0; c0 < rows && !rc; c0 += (int)h->Pb) {
                    const int c = (int)std::min<long long>(h->Pb, rows - c0);
                    if ((rc = bse_launch_inv_stick(pl, h->uG, c, h->Z, h->stream, h->rowlist, r0 + c0))) break;
                    if ((rc = bse_launch_inv_plane(pl, h->Z, c, pl.N, ub, h->stream))) break;
                    rc = bse_launch_k1_mix(ub, h->mix_vH, h->acc_r + (long long)c0 * pl.N, nullptr, c, h->rows_cap, true, pl.N, nb,
                                           h->mix_ce, h->mix_cd, h->stream);
                }
            }
            if (rc) return rc;
        }
        if (out_pw && (rc = rows_to_pw(h, h->acc_r, h->rows_cap, rows, nb, out_pw, h->rowlist + r0))) return rc;
    }
    return BSE_OK;
}

// PW layout, plane-slab streaming (a9 + a10 + a12 on one slab of planes at a time; see plan_apply_memory and the slab stick
// kernels of fft_kernels.cuh).  For slab s = { i1 = s + R1 k2 }:  a(G) -> a(r) on the slab for all B blocks, tau(G) -> tau(r)
// on the slab for all pairs, then chunks of rows: accumulate (eq. 5), forward plane pass, forward slab stick pass that
// accumulates the slab's share of acc(G) into out.  P_c follows on the finished coefficients.
int apply_pw_slab(bse_handle *h, const double2 *a, double2 *out, int B) {
    const FftPlan &pl = *h->ap;
    const Model m(pl);
    const int S = h->slab_S, M = h->slab_M;
    const long long SN = (long long)M * pl.n * pl.n, npw_h = pl.npw_h, Nv = h->Nv;
    const double share = (double)M / pl.n;               // one slab's share of a whole-field pass
    const long long nloc = h->row1 - h->row0;            // out holds the owned rows only: [B][nloc][npw_h]
    int rc;
    auto to_slab = [&](const double2 *src, long long fields, double *dst, int s, const float2 *src32 = nullptr) -> int {
        for (long long f0 = 0; f0 < fields; f0 += h->slab_pz) {
            const int cnt = (int)std::min<long long>(h->slab_pz, fields - f0);
            { StageTimer t(h, BSE_ST_INV_STICK, cnt * m.stick_flops * share, cnt * m.g * share, cnt * m.z * share);
              if (int r = bse_launch_inv_stick_slab(pl, S, M, src32 ? nullptr : src + f0 * npw_h, cnt, h->Z, h->stream, s, nullptr, 0,
                                                    src32 ? src32 + f0 * npw_h : nullptr)) return r; }
            { StageTimer t(h, BSE_ST_INV_PLANE, cnt * m.plane_flops * share, cnt * m.N8 * share, cnt * m.z * share);
              if (int r = bse_launch_inv_plane(pl, h->Z, cnt, SN, dst + f0 * SN, h->stream, false, M)) return r; }
        }
        return BSE_OK;
    };
    // combined call (eq. 1, bse_apply_k1): k1e_ws = u_slab [Nv][SN] | vH_slab [B][SN] | vG [B][npw_h].  A first sweep over the
    // slabs forms the transition density n_b = sum_v u_v a_bv slab by slab and accumulates v_c n_b(G) into vG (eq. 4); the main
    // sweep then adds 2 ce u_v v_H[b] to the accumulated rows before their forward transform, so P_c is applied once.
    double *u_slab = h->k1e_ws, *vH_slab = h->k1e_ws ? h->k1e_ws + Nv * SN : nullptr;
    double2 *vG = h->k1e_ws ? (double2 *)(vH_slab + (long long)B * SN) : nullptr;
    if (h->mix_on) {
        for (int s = 0; s < S; ++s) {
            if ((rc = to_slab(a, (long long)B * Nv, h->a_r, s))) return rc;
            if ((rc = to_slab(h->uG, Nv, u_slab, s))) return rc;
            { StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * B * Nv * (double)SN, 8.0 * SN * (double)(B * Nv + Nv + B));
              if ((rc = bse_launch_k1e_density(u_slab, h->a_r, vH_slab, h->Nv, SN, B, h->stream))) return rc; }
            { StageTimer t(h, BSE_ST_FWD_PLANE, B * m.plane_flops * share, B * m.N8 * share, B * m.z * share);
              if ((rc = bse_launch_fwd_plane(pl, vH_slab, nullptr, 0, B, SN, h->Z, h->stream, M))) return rc; }
            { StageTimer t(h, BSE_ST_FWD_STICK, B * m.stick_flops * share, B * m.g * share, B * m.z * share);
              if ((rc = bse_launch_fwd_stick_slab(pl, S, M, h->Z, B, vG, pl.vcn, h->stream, s, s > 0, B, 0, 0))) return rc; }
        }
    }
    for (int s = 0; s < S; ++s) {
        if ((rc = to_slab(a, (long long)B * Nv, h->a_r, s))) return rc;
        if ((rc = to_slab(h->tau_g, h->Pa, h->tau_batch, s, h->tau_g32))) return rc;
        if (h->mix_on) {
            if ((rc = to_slab(h->uG, Nv, u_slab, s))) return rc;
            if ((rc = to_slab(vG, B, vH_slab, s))) return rc;
        }
        for (long long v0 = h->row0; v0 < h->row1; v0 += h->slab_rc) {       // the owned rows (all of them unless bse_set_rows)
            const int rows = (int)std::min<long long>(h->slab_rc, h->row1 - v0);
            const double directed = (double)(h->adj_ptr_h[v0 + rows] - h->adj_ptr_h[v0]);
            { StageTimer t(h, BSE_ST_ACCUM, 2.0 * B * (double)SN * directed,
                           8.0 * SN * ((double)h->Pa * rows / nloc + (double)B * rows + (v0 == h->row0 ? (double)B * Nv : 0.0)));
              t.launches = acc_rows_launches(B);
              if ((rc = bse_launch_accumulate_rows(h, SN, h->tau_batch, h->eslot_act, h->rowid + v0, rows, h->a_r, h->acc_r, rows,
                                                   true, B))) return rc; }
            if (h->mix_on) {
                StageTimer t(h, BSE_ST_K1E_PRODUCT, 3.0 * B * rows * (double)SN, 8.0 * SN * (2.0 * B * rows + rows + B));
                if ((rc = bse_launch_k1_mix(u_slab, vH_slab, h->acc_r, h->rowid + v0, rows, rows, true, SN, B, h->mix_ce, h->mix_cd,
                                            h->stream))) return rc;
            }
            const int cnt = B * rows;
            { StageTimer t(h, BSE_ST_FWD_PLANE, cnt * m.plane_flops * share, cnt * m.N8 * share, cnt * m.z * share);
              if ((rc = bse_launch_fwd_plane(pl, h->acc_r, nullptr, 0, cnt, SN, h->Z, h->stream, M))) return rc; }
            { StageTimer t(h, BSE_ST_FWD_STICK, cnt * m.stick_flops * share, cnt * m.g * share, cnt * m.z * share);
              if ((rc = bse_launch_fwd_stick_slab(pl, S, M, h->Z, cnt, out, pl.inv2n, h->stream, s, s > 0, rows, nloc, v0 - h->row0))) return rc; }
        }
    }
    return p_c_rows(h, (double *)out, (long long)B * nloc, 2 * npw_h, (const double *)h->uGw, (const double *)h->uG, 1.0);
}

// PW layout (a12): a, out = [B][Nv][npw_h] complex on H
int apply_pw(bse_handle *h, const double2 *a, double2 *out, int B) {
    const FftPlan &pl = *h->ap;
    int rc;
    if ((rc = ensure_u_pw(h))) return rc;
    if (h->slab_mode) return apply_pw_slab(h, a, out, B);
    if (h->rows_set) { bse_set_error("row-sharded apply needs the plane-slab path (PW layout, tau on H, enough memory)"); return BSE_EUNSUPPORTED; }
    const long long Nv = h->Nv, npw_h = pl.npw_h;
    for (int b0 = 0; b0 < B; b0 += h->Bg) {
        const int nb = std::min(h->Bg, B - b0);
        const long long fields = (long long)nb * Nv;
        const double2 *ag = a + (long long)b0 * Nv * npw_h;
        for (long long f0 = 0; f0 < fields; f0 += h->Pb) {           // a(G) -> a(r)
            const int cnt = (int)std::min<long long>(h->Pb, fields - f0);
            if ((rc = st_inv_stick(h, pl, ag + f0 * npw_h, cnt))) return rc;
            if ((rc = st_inv_plane(h, pl, cnt, h->a_r + f0 * pl.N))) return rc;
        }
        if (h->mix_on) {                                              // v_H of this group's blocks (K1e part of bse_apply_k1)
            double *vH = h->k1e_ws;
            if (h->mix_u) {
                StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * nb * Nv * (double)pl.N, 8.0 * pl.N * (double)(nb * Nv + Nv + nb));
                if ((rc = bse_launch_k1e_density(h->mix_u, h->a_r, vH, h->Nv, pl.N, nb, h->stream))) return rc;
            } else {                                                  // u on the apply grid made on the fly, Pb orbitals at a time
                double *ub = h->k1e_ws + (long long)B * pl.N;
                for (long long v0 = 0; v0 < Nv; v0 += h->Pb) {
                    const int cnt = (int)std::min<long long>(h->Pb, Nv - v0);
                    if ((rc = st_inv_stick(h, pl, h->uG + v0 * npw_h, cnt))) return rc;
                    if ((rc = st_inv_plane(h, pl, cnt, ub))) return rc;
                    StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * nb * cnt * (double)pl.N, 8.0 * pl.N * (double)(nb * cnt + cnt + nb));
                    if ((rc = bse_launch_k1e_density(ub, h->a_r, vH, h->Nv, pl.N, nb, h->stream, (int)v0, cnt, v0 > 0))) return rc;
                }
            }
            if ((rc = hartree_in_place(h, pl, vH, nb))) return rc;
            h->mix_vH = vH;
        }
        if ((rc = accumulate_all(h, h->a_r, nb, nullptr, out + (long long)b0 * Nv * npw_h))) return rc;
    }
    // P_c in PW: S = <u_w|acc> (real dot GEMM against the weighted copy), out -= S u(G)
    return p_c_rows(h, (double *)out, (long long)B * Nv, 2 * npw_h, (const double *)h->uGw, (const double *)h->uG, 1.0);
}

}  // namespace

extern "C" int bse_create(bse_handle **hout, const int grid[3], const double cell[9], double ecut, int Nv,
                          const double *u, int Npdep, const double *phi, const double *lambda, double eta,
                          unsigned flags, void *stream) {
    if (!hout || !grid || !cell || !u || !phi || !lambda) { bse_set_error("null pointer"); return BSE_EINVAL; }
    *hout = nullptr;
    if (grid[0] <= 0 || grid[1] <= 0 || grid[2] <= 0 || Nv <= 0 || Npdep <= 0 || !(ecut > 0) || !(eta >= 0)) {
        bse_set_error("non-positive size, ecut <= 0 or eta < 0");
        return BSE_EINVAL;
    }
    if (grid[0] != grid[1] || grid[1] != grid[2] || (grid[0] & 1)) {
        bse_set_error("this version supports cubic grids with even n only");
        return BSE_EUNSUPPORTED;
    }
    const double L = cell[0];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            const double want = (i == j) ? L : 0.0;
            if (!(L > 0) || std::fabs(cell[3 * i + j] - want) > 1e-12 * std::fabs(L)) {
                bse_set_error("this version supports cubic cells only");
                return (L > 0) ? BSE_EUNSUPPORTED : BSE_EINVAL;
            }
        }
    for (int a = 0; a < Npdep; ++a)
        if (!(lambda[a] < 1.0)) { bse_set_error("lambda >= 1"); return BSE_EINVAL; }
    if ((flags & BSE_TAU_MASK) == 3u) { bse_set_error("bad tau storage flag"); return BSE_EINVAL; }
    if ((flags & BSE_TAU_F32) && (flags & BSE_TAU_MASK) == BSE_TAU_REAL) {
        bse_set_error("BSE_TAU_F32 needs BSE_TAU_PW or BSE_TAU_STREAM");
        return BSE_EINVAL;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        bse_set_error("no CUDA device: this library has no CPU fallback");
        return BSE_ECUDA;
    }
    bse_handle *h = new (std::nothrow) bse_handle();
    if (!h) return BSE_ENOMEM;
    h->n = grid[0];
    h->N = (long long)h->n * h->n * h->n;
    h->L = L; h->Omega = L * L * L; h->dV = h->Omega / (double)h->N;
    h->ecut = ecut; h->eta = eta; h->Nv = Nv; h->Npdep = Npdep; h->flags = flags;
    h->row0 = 0; h->row1 = Nv;
    h->stream = (cudaStream_t)stream;
    h->msq_max = (int)std::floor(2.0 * ecut * (L / (2.0 * M_PI)) * (L / (2.0 * M_PI)) * (1.0 + 1e-12));
    const int R = (int)std::floor(std::sqrt((double)h->msq_max) + 1e-9);
    int rc = BSE_OK;
    auto fail = [&](int code) { bse_destroy(h); return code; };
    if (2 * R >= h->n) { bse_set_error("sphere does not fit the grid (R >= n/2)"); return fail(BSE_EINVAL); }
    if ((rc = build_fft_plan(h, h->fft, h->n))) return fail(rc);
    // Apply grid of the PW layout: tau(r) a(r) is a product of two functions band-limited to |m| <= R per axis, so its
    // components inside S are alias-free on any grid with n_a >= 3R + 1; the apply then moves (n_a / n)^3 of the bytes.
    // (The REAL layout is defined on the problem grid, and a BSE_TAU_REAL store holds tau on it, so both keep n.)
    h->ap = &h->fft;
    if ((flags & BSE_VEC_PW) && (flags & BSE_TAU_MASK) != BSE_TAU_REAL) {
        static const int sizes[] = {12, 16, 20, 24, 30, 32, 36, 40, 48, 60, 64, 72, 80, 96, 100, 108, 120, 128, 144, 160};
        for (int na : sizes)
            if (na >= 3 * R + 1 && na < h->n) {
                if ((rc = build_fft_plan(h, h->ffta, na))) return fail(rc);
                h->ap = &h->ffta;
                break;
            }
    }
    if ((long long)Npdep > 2 * (h->fft.npw_h - 1)) { bse_set_error("Npdep > 2 (Npw_h - 1)"); return fail(BSE_EINVAL); }
    const long long K2 = 2 * h->fft.npw_h;
    if (flags & BSE_PTR_HOST) {
        if (cudaMalloc(&h->u_owned, (size_t)Nv * h->N * 8) != cudaSuccess ||
            cudaMalloc(&h->phi_owned, (size_t)Npdep * K2 * 8) != cudaSuccess) {
            bse_set_error("out of device memory for u / phi");
            return fail(BSE_ENOMEM);
        }
        if (cudaMemcpyAsync(h->u_owned, u, (size_t)Nv * h->N * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
            cudaMemcpyAsync(h->phi_owned, phi, (size_t)Npdep * K2 * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess) {
            bse_set_error("host-to-device copy of u / phi failed");
            return fail(BSE_ECUDA);
        }
        h->u = h->u_owned; h->phi = h->phi_owned;
    } else {
        h->u = u; h->phi = phi;
    }
    std::vector<double> f2(Npdep);
    for (int a = 0; a < Npdep; ++a) f2[a] = 2.0 * lambda[a] / (1.0 - lambda[a]);   // factor 2: half-sphere sum
    if ((rc = upload(h->f2, f2))) return fail(rc);

    // fixed-size buffers
    const size_t nv2 = (size_t)Nv * Nv;
    if (cudaMalloc(&h->Mmat, nv2 * 8) || cudaMalloc(&h->rowcnt, (size_t)Nv * 4) || cudaMalloc(&h->rowptr, (size_t)(Nv + 1) * 4) ||
        cudaMalloc(&h->pid, nv2 * 4) || cudaMalloc(&h->pairs, ((size_t)Nv * (Nv + 1) / 2) * 8) ||
        cudaMalloc(&h->adj_ptr, (size_t)(Nv + 1) * 4) || cudaMalloc(&h->adj, nv2 * 8)) {
        bse_set_error("out of device memory (pair tables)");
        return fail(BSE_ENOMEM);
    }
    // pair-batch workspaces
    size_t free_b = 0, total_b = 0;
    cudaMemGetInfo(&free_b, &total_b);
    const size_t per_pair = (size_t)h->n * h->fft.NS * 16 + 2 * (size_t)h->fft.npw_h * 16 + (size_t)ldD(h) * 8;
    const size_t per_pair_r = (size_t)h->N * 8;   // tau_batch, allocated lazily (PW / STREAM / get_tau)
    size_t budget = std::min<size_t>((size_t)12 << 30, free_b / 4);
    long long Pb = (long long)(budget / (per_pair + per_pair_r));
    Pb = std::max<long long>(1, std::min<long long>(Pb, 512));
    h->part_bytes = std::max<size_t>((size_t)128 << 20, nv2 * 8 * 2);    // split-K partial sums: room for 13 splits of the screen at N_v = 1024
    if ((rc = alloc_batch_ws(h, Pb))) return fail(rc);
    if (cudaMalloc(&h->part, h->part_bytes)) {
        bse_set_error("out of device memory (workspaces)");
        return fail(BSE_ENOMEM);
    }
    cudaEventCreate(&h->ev0);
    cudaEventCreate(&h->ev1);
    cudaEventCreate(&h->ev_fill0);
    cudaEventCreate(&h->ev_fill1);
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) { bse_set_error("stream sync failed"); return fail(BSE_ECUDA); }
    *hout = h;
    return BSE_OK;
}

extern "C" int bse_destroy(bse_handle *h) {
    if (!h) return BSE_OK;
    cudaStreamSynchronize(h->stream);
    if (h->s_in) cudaStreamSynchronize(h->s_in);
    if (h->s_out) cudaStreamSynchronize(h->s_out);
    free_plan(h->fft);
    free_plan(h->ffta);
    cudaFree(h->u_owned); cudaFree(h->phi_owned); cudaFree(h->f2); cudaFree(h->Mmat); cudaFree(h->rowcnt);
    cudaFree(h->rowptr); cudaFree(h->pid); cudaFree(h->pairs); cudaFree(h->adj_ptr); cudaFree(h->adj);
    cudaFree(h->tau_r); cudaFree(h->tau_g); cudaFree(h->tau_g32); cudaFree(h->Z); cudaFree(h->X); cudaFree(h->T); cudaFree(h->Dm);
    cudaFree(h->part); cudaFree(h->Sov); cudaFree(h->tau_batch); cudaFree(h->a_dev); cudaFree(h->out_dev);
    cudaFree(h->uG); cudaFree(h->uGw); cudaFree(h->a_r); cudaFree(h->acc_r);
    cudaFree(h->batch_pairs); cudaFree(h->eslot); cudaFree(h->rowlist); cudaFree(h->rowid); cudaFree(h->pairs_act); cudaFree(h->eslot_act); cudaFree(h->k1e_ws); cudaFree(h->u_a); cudaFree(h->Ut); cudaFree(h->accG);
    for (cudaEvent_t e : h->ev_pipe) cudaEventDestroy(e);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
    if (h->ev_d2h) cudaEventDestroy(h->ev_d2h);
    if (h->ev_in_done) cudaEventDestroy(h->ev_in_done);
    for (cudaEvent_t e : h->ev_in) cudaEventDestroy(e);
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    if (h->ev_fill0) cudaEventDestroy(h->ev_fill0);
    if (h->ev_fill1) cudaEventDestroy(h->ev_fill1);
    delete h;
    return BSE_OK;
}

// Row-sharded operation (Fig. 2: the N_occ orbitals of A_s block-distributed over band groups):
// this handle owns the output rows [v0, v1).  bse_build_tau then keeps tau only for the pairs that touch an owned row, and
// bse_apply_k1x takes the FULL (all-gathered) trial blocks a [B][Nv][.] and writes the owned rows out [B][v1 - v0][.].
extern "C" int bse_set_rows(bse_handle *h, int v0, int v1) {
    if (!h) { bse_set_error("null handle"); return BSE_EINVAL; }
    if (v0 < 0 || v1 > h->Nv || v0 >= v1) { bse_set_error("bse_set_rows: need 0 <= v0 < v1 <= Nv"); return BSE_EINVAL; }
    if (!(h->flags & BSE_VEC_PW) || (h->flags & BSE_TAU_MASK) == BSE_TAU_REAL) {
        bse_set_error("bse_set_rows needs BSE_VEC_PW with BSE_TAU_PW or BSE_TAU_STREAM");
        return BSE_EUNSUPPORTED;
    }
    h->row0 = v0; h->row1 = v1;
    h->rows_set = !(v0 == 0 && v1 == h->Nv);
    h->built = false;
    h->plan_ok = false;
    return BSE_OK;
}

// the library's stream waits for whatever bse_set_inputs_host left in flight on the copy stream
static int wait_inputs(bse_handle *h) {
    if (h->inputs_pending) {
        BSE_CUDA(cudaStreamWaitEvent(h->stream, h->ev_in_done, 0));
        h->inputs_pending = false;
    }
    h->in_chunks = 0;
    return BSE_OK;
}

extern "C" int bse_build_tau(bse_handle *h) {
    if (!h) { bse_set_error("null handle"); return BSE_EINVAL; }
    int rc;
    h->built = false;
    // a1: M = (u^2)(u^2)^T, then the threshold decision and the list, all on the device
    if (h->inputs_pending && h->in_chunks > 1) {
        // u is still arriving from the host in column slabs: M accumulates slab after slab (the sum over grid points in
        // slab order), so the copy hides the screen
        for (int c = 0; c < h->in_chunks; ++c) {
            const long long k0 = c * h->in_kc, kc = std::min<long long>(h->in_kc, h->N - k0);
            BSE_CUDA(cudaStreamWaitEvent(h->stream, h->ev_in[c], 0));
            if ((rc = st_gemm_dot(h, BSE_ST_SCREEN, h->u + k0, h->N, h->u + k0, h->N, h->Nv, h->Nv, kc, true, h->Mmat, h->Nv,
                                  1.0, nullptr, c > 0))) return rc;
        }
    } else {
        if ((rc = wait_inputs(h))) return rc;
        if ((rc = st_gemm_dot(h, BSE_ST_SCREEN, h->u, h->N, h->u, h->N, h->Nv, h->Nv, h->N, true, h->Mmat, h->Nv, 1.0,
                              nullptr))) return rc;
    }
    if ((rc = wait_inputs(h))) return rc;
    { StageTimer t(h, BSE_ST_PAIRLIST, 0.0, 8.0 * h->Nv * (double)h->Nv);
      if ((rc = bse_launch_pairlist(h))) return rc; }
    const unsigned mode = h->flags & BSE_TAU_MASK;
    if (mode != BSE_TAU_STREAM) {
        if ((rc = ensure_tau_store(h, mode == BSE_TAU_REAL))) return rc;
        if ((rc = fill_tau_store(h, mode == BSE_TAU_REAL))) return rc;
    }
    h->built = true;
    return BSE_OK;
}

extern "C" int bse_apply_k1x(bse_handle *h, const double *a, double *out, int B) {
    if (!h || !a || !out || B <= 0) { bse_set_error("null pointer or B <= 0"); return BSE_EINVAL; }
    if (!h->built) { bse_set_error("bse_apply_k1x before bse_build_tau"); return BSE_ESTATE; }
    if (a == out) { bse_set_error("out must not alias a"); return BSE_EINVAL; }
    int rc;
    if ((h->flags & BSE_TAU_MASK) == BSE_TAU_STREAM) {       // tau rebuilt inside every apply: tau(G) transient, tau(r) streamed
        if (!h->tau_prefilled) {
            if ((rc = ensure_tau_store(h, false))) return rc;
            if ((rc = fill_tau_store(h, false))) return rc;
        }
        h->tau_prefilled = false;
    }
    if ((rc = plan_apply_memory(h, B))) return rc;
    if (h->flags & BSE_VEC_PW) return apply_pw(h, (const double2 *)a, (double2 *)out, B);
    if ((rc = accumulate_all(h, a, B, out, nullptr))) return rc;
    return p_c_rows_real(h, out, (long long)B * h->Nv);
}

extern "C" int bse_apply_k1x_host(bse_handle *h, const double *a_host, double *out_host, int B) {
    if (!h || !a_host || !out_host || B <= 0) { bse_set_error("null pointer or B <= 0"); return BSE_EINVAL; }
    const size_t bytes = (h->flags & BSE_VEC_PW) ? (size_t)B * h->Nv * h->fft.npw_h * 16 : (size_t)B * h->Nv * h->N * 8;
    if (h->a_dev_bytes < bytes) {
        cudaFree(h->a_dev); cudaFree(h->out_dev);
        h->a_dev = h->out_dev = nullptr; h->a_dev_bytes = 0;
        BSE_CUDA(cudaMalloc(&h->a_dev, bytes));
        BSE_CUDA(cudaMalloc(&h->out_dev, bytes));
        h->a_dev_bytes = bytes;
    }
    if ((h->flags & BSE_TAU_MASK) == BSE_TAU_REAL && B > 1) {
        // tau(r) is resident, so blocks are independent: copy block b+1 in and block b-1 out (two copy streams, PCIe is full
        // duplex) while block b is applied; the call ends ~one block after the last input byte arrives
        if (!h->s_in) {
            BSE_CUDA(cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
            BSE_CUDA(cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
        }
        while ((int)h->ev_pipe.size() < 2 * B + 1) {
            cudaEvent_t e;
            BSE_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            h->ev_pipe.push_back(e);
        }
        const size_t per = bytes / B, per_d = per / 8;
        BSE_CUDA(cudaEventRecord(h->ev_pipe[2 * B], h->stream));             // earlier work on the library's stream first
        BSE_CUDA(cudaStreamWaitEvent(h->s_in, h->ev_pipe[2 * B], 0));
        for (int b = 0; b < B; ++b) {
            BSE_CUDA(cudaMemcpyAsync(h->a_dev + b * per_d, a_host + b * per_d, per, cudaMemcpyHostToDevice, h->s_in));
            BSE_CUDA(cudaEventRecord(h->ev_pipe[b], h->s_in));
        }
        for (int b = 0; b < B; ++b) {
            BSE_CUDA(cudaStreamWaitEvent(h->stream, h->ev_pipe[b], 0));
            const int rc = bse_apply_k1x(h, h->a_dev + b * per_d, h->out_dev + b * per_d, 1);
            if (rc) return rc;
            BSE_CUDA(cudaEventRecord(h->ev_pipe[B + b], h->stream));
            BSE_CUDA(cudaStreamWaitEvent(h->s_out, h->ev_pipe[B + b], 0));
            BSE_CUDA(cudaMemcpyAsync(out_host + b * per_d, h->out_dev + b * per_d, per, cudaMemcpyDeviceToHost, h->s_out));
        }
        BSE_CUDA(cudaStreamSynchronize(h->s_out));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        return BSE_OK;
    }
    // one apply over all blocks: a arrives on the copy stream while tau is rebuilt (STREAM), and every row chunk P_c has
    // finished leaves on the other copy stream while the next one is projected (p_c_rows)
    if (!h->s_in) {
        BSE_CUDA(cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
        BSE_CUDA(cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
    }
    if (!h->ev_d2h) BSE_CUDA(cudaEventCreateWithFlags(&h->ev_d2h, cudaEventDisableTiming));
    BSE_CUDA(cudaEventRecord(h->ev_d2h, h->stream));                         // earlier work on the library's stream first
    BSE_CUDA(cudaStreamWaitEvent(h->s_in, h->ev_d2h, 0));
    BSE_CUDA(cudaMemcpyAsync(h->a_dev, a_host, bytes, cudaMemcpyHostToDevice, h->s_in));
    BSE_CUDA(cudaEventRecord(h->ev_d2h, h->s_in));
    int rc = BSE_OK;
    if (h->built && (h->flags & BSE_TAU_MASK) == BSE_TAU_STREAM) {
        if ((rc = ensure_tau_store(h, false)) == BSE_OK && (rc = fill_tau_store(h, false)) == BSE_OK) h->tau_prefilled = true;
    }
    BSE_CUDA(cudaStreamWaitEvent(h->stream, h->ev_d2h, 0));
    if (rc == BSE_OK) {
        h->d2h_host = out_host;
        h->d2h_rows_done = 0;
        rc = bse_apply_k1x(h, h->a_dev, h->out_dev, B);
        h->d2h_host = nullptr;
    }
    h->tau_prefilled = false;
    if (rc) { cudaStreamSynchronize(h->s_in); cudaStreamSynchronize(h->s_out); return rc; }
    const size_t done = (size_t)h->d2h_rows_done * (bytes / ((size_t)B * h->Nv));   // bytes per row: the vector length * 8
    if (done < bytes)
        BSE_CUDA(cudaMemcpyAsync((char *)out_host + done, (char *)h->out_dev + done, bytes - done, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->s_out));
    return BSE_OK;
}

// New orbitals / PDEP vectors of the same sizes from HOST memory into the buffers a BSE_PTR_HOST handle owns (no
// reallocation): the per-step input refresh of a caller whose orbitals change (bench.py's e2e step).  Invalidates tau.
extern "C" int bse_set_inputs_host(bse_handle *h, const double *u_host, const double *phi_host) {
    if (!h || (!u_host && !phi_host)) { bse_set_error("null pointer"); return BSE_EINVAL; }
    if (!h->u_owned || !h->phi_owned) { bse_set_error("bse_set_inputs_host needs a handle created with BSE_PTR_HOST"); return BSE_ESTATE; }
    if (!h->s_in) {
        BSE_CUDA(cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
        BSE_CUDA(cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
    }
    if (!h->ev_in_done) BSE_CUDA(cudaEventCreateWithFlags(&h->ev_in_done, cudaEventDisableTiming));
    BSE_CUDA(cudaEventRecord(h->ev_in_done, h->stream));                     // readers of the old arrays first
    BSE_CUDA(cudaStreamWaitEvent(h->s_in, h->ev_in_done, 0));
    h->in_chunks = 0;
    if (u_host) {
        // column slabs (all orbitals on a range of grid points): the screen of bse_build_tau is a sum over grid points and
        // starts on slab 0 while the others are on their way.  Small arrays go in one piece.
        const size_t ub = (size_t)h->Nv * h->N * 8;
        const int nch = h->dbg_in_chunks >= 1 ? (int)h->dbg_in_chunks : (ub >= ((size_t)256 << 20) ? 8 : 1);
        const long long kc = nch == 1 ? h->N : ((h->N + nch - 1) / nch + 1023) / 1024 * 1024;
        const int used = (int)((h->N + kc - 1) / kc);
        while ((int)h->ev_in.size() < used) {
            cudaEvent_t e;
            BSE_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            h->ev_in.push_back(e);
        }
        for (int c = 0; c < used; ++c) {
            const long long k0 = c * kc, kw = std::min<long long>(kc, h->N - k0);
            BSE_CUDA(cudaMemcpy2DAsync(h->u_owned + k0, (size_t)h->N * 8, u_host + k0, (size_t)h->N * 8, (size_t)kw * 8, h->Nv,
                                       cudaMemcpyHostToDevice, h->s_in));
            BSE_CUDA(cudaEventRecord(h->ev_in[c], h->s_in));
        }
        h->in_chunks = used;
        h->in_kc = kc;
    }
    if (phi_host) BSE_CUDA(cudaMemcpyAsync(h->phi_owned, phi_host, (size_t)h->Npdep * h->fft.npw_h * 16, cudaMemcpyHostToDevice, h->s_in));
    BSE_CUDA(cudaEventRecord(h->ev_in_done, h->s_in));
    h->inputs_pending = true;
    h->built = false;
    if (u_host) { h->uG_valid = false; h->u_a_valid = false; h->u_bl = -1; }     // derived copies are refilled in place, lazily
    return BSE_OK;
}

// ------------------------------------------------------------------------------------------------ K1e (eq. 4)
extern "C" int bse_apply_k1e(bse_handle *h, const double *a, double *out, int B) {
    if (!h || !a || !out || B <= 0) { bse_set_error("null pointer or B <= 0"); return BSE_EINVAL; }
    if (a == out) { bse_set_error("out must not alias a"); return BSE_EINVAL; }
    int rc;
    if ((rc = wait_inputs(h))) return rc;
    const long long Nv = h->Nv;
    if (!(h->flags & BSE_VEC_PW)) {
        const FftPlan &pl = h->fft;
        const double N8 = 8.0 * (double)pl.N;
        if ((rc = ensure_k1e_ws(h, (size_t)B * pl.N * 8))) return rc;
        { StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * B * Nv * (double)pl.N, N8 * (B * Nv + Nv + B));
          if ((rc = bse_launch_k1e_density(h->u, a, h->k1e_ws, h->Nv, pl.N, B, h->stream))) return rc; }
        if ((rc = hartree_in_place(h, pl, h->k1e_ws, B))) return rc;
        { StageTimer t(h, BSE_ST_K1E_PRODUCT, 2.0 * B * Nv * (double)pl.N, N8 * (B * Nv + Nv + B));
          if ((rc = bse_launch_k1e_product(h->u, h->k1e_ws, out, 0, h->Nv, Nv, pl.N, B, h->stream))) return rc; }
        return p_c_rows_real(h, out, (long long)B * Nv);
    }
    // PW layout: one block at a time on the apply grid: a(G) -> a(r), density, Hartree, products in row chunks -> out(G)
    const FftPlan &pl = *h->ap;
    const double N8 = 8.0 * (double)pl.N;
    const long long npw_h = pl.npw_h;
    if ((rc = ensure_u_pw(h))) return rc;
    if ((rc = ensure_u_apply(h))) return rc;
    const double *ua = h->u_a ? h->u_a : h->u;
    // staging: the K1x plan's buffers when they exist (they took the free memory), else own workspace
    double *a_r = (h->a_r && h->a_r_elems >= (size_t)Nv * pl.N) ? h->a_r : nullptr;
    double *dens = (h->tau_batch && h->Pacc >= h->Pb + 1) ? h->tau_batch : nullptr;
    if (!a_r || !dens) {
        if ((rc = ensure_k1e_ws(h, (size_t)((a_r ? 0 : Nv) + (dens ? 0 : 1 + h->Pb)) * pl.N * 8))) return rc;
        // ensure_k1e_ws may have dropped the K1x plan's buffers to make room: look at them again
        if (a_r && !h->a_r) a_r = nullptr;
        if (dens && !h->tau_batch) dens = nullptr;
        if ((rc = ensure_k1e_ws(h, (size_t)((a_r ? 0 : Nv) + (dens ? 0 : 1 + h->Pb)) * pl.N * 8))) return rc;
        double *ws = h->k1e_ws;
        if (!a_r) { a_r = ws; ws += Nv * pl.N; }
        if (!dens) dens = ws;
    }
    double *prod = dens + pl.N;
    const double2 *ag = (const double2 *)a;
    double2 *og = (double2 *)out;
    for (int b = 0; b < B; ++b) {
        for (long long v0 = 0; v0 < Nv; v0 += h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, Nv - v0);
            if ((rc = st_inv_stick(h, pl, ag + ((long long)b * Nv + v0) * npw_h, cnt))) return rc;
            if ((rc = st_inv_plane(h, pl, cnt, a_r + v0 * pl.N))) return rc;
        }
        { StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * Nv * (double)pl.N, N8 * (2.0 * Nv + 1));
          if ((rc = bse_launch_k1e_density(ua, a_r, dens, h->Nv, pl.N, 1, h->stream))) return rc; }
        if ((rc = hartree_in_place(h, pl, dens, 1))) return rc;
        for (long long v0 = 0; v0 < Nv; v0 += h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, Nv - v0);
            { StageTimer t(h, BSE_ST_K1E_PRODUCT, 2.0 * cnt * (double)pl.N, N8 * (2.0 * cnt + 1));
              if ((rc = bse_launch_k1e_product(ua, dens, prod, (int)v0, cnt, h->Pb, pl.N, 1, h->stream))) return rc; }
            if ((rc = st_fwd_plane(h, pl, prod, nullptr, 0, cnt))) return rc;
            if ((rc = st_fwd_stick(h, pl, cnt, og + ((long long)b * Nv + v0) * npw_h, pl.inv2n))) return rc;
        }
    }
    return p_c_rows(h, (double *)out, (long long)B * Nv, 2 * npw_h, (const double *)h->uGw, (const double *)h->uG, 1.0);
}

// ---- K1e split for the row-sharded operation.  eq. 4 sums over ALL occupied states inside the integral:
// each rank forms the Hartree potential of its own rows' share of the transition density, the shares are summed over the ranks
// (an all-reduce of B * N_pw_h coefficients - "communications between band groups are required only when a summation over
// occupied states is carried out"), and every rank finishes its own rows.  PW layout only.
//   vG[b](G) = v_c(G) * sum_{v in [v0, v1)} [u_v a_bv](G)  on H        a_rows: [B][v1 - v0][npw_h] (the owned rows of each block)
extern "C" int bse_k1e_hartree_partial(bse_handle *h, const double *a_rows, int v0, int v1, int B, double *vG) {
    if (!h || !a_rows || !vG || B <= 0 || v0 < 0 || v1 > h->Nv || v0 >= v1) { bse_set_error("bad argument"); return BSE_EINVAL; }
    if (!(h->flags & BSE_VEC_PW)) { bse_set_error("bse_k1e_hartree_partial needs BSE_VEC_PW"); return BSE_EUNSUPPORTED; }
    const FftPlan &pl = *h->ap;
    const long long npw_h = pl.npw_h, nloc = v1 - v0;
    const double N8 = 8.0 * (double)pl.N;
    int rc;
    if ((rc = wait_inputs(h))) return rc;
    if ((rc = ensure_u_pw(h))) return rc;
    if ((rc = ensure_u_apply(h))) return rc;
    const double *ua = h->u_a ? h->u_a : h->u;
    if ((rc = ensure_k1e_ws(h, (size_t)(h->Pb + 1) * pl.N * 8))) return rc;
    double *dens = h->k1e_ws, *chunk = h->k1e_ws + pl.N;
    const double2 *ag = (const double2 *)a_rows;
    for (int b = 0; b < B; ++b) {
        for (long long c0 = 0; c0 < nloc; c0 += h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, nloc - c0);
            if ((rc = st_inv_stick(h, pl, ag + ((long long)b * nloc + c0) * npw_h, cnt))) return rc;
            if ((rc = st_inv_plane(h, pl, cnt, chunk))) return rc;
            StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * cnt * (double)pl.N, N8 * (2.0 * cnt + 1));
            if ((rc = bse_launch_k1e_density(ua + (v0 + c0) * pl.N, chunk, dens, cnt, pl.N, 1, h->stream, 0, cnt, c0 > 0))) return rc;
        }
        if ((rc = st_fwd_plane(h, pl, dens, nullptr, 0, 1))) return rc;
        if ((rc = st_fwd_stick(h, pl, 1, (double2 *)vG + (long long)b * npw_h, pl.vcn))) return rc;
    }
    return BSE_OK;
}

//   out_rows[b, v - v0] = P_c [ 2 u_v v_H[b] ] truncated to S,  v_H[b](r) = sum_{G in S} vG[b](G) e^{iG.r}   (vG summed over the ranks)
extern "C" int bse_k1e_from_hartree(bse_handle *h, const double *vG, int v0, int v1, int B, double *out_rows) {
    if (!h || !vG || !out_rows || B <= 0 || v0 < 0 || v1 > h->Nv || v0 >= v1) { bse_set_error("bad argument"); return BSE_EINVAL; }
    if (!(h->flags & BSE_VEC_PW)) { bse_set_error("bse_k1e_from_hartree needs BSE_VEC_PW"); return BSE_EUNSUPPORTED; }
    const FftPlan &pl = *h->ap;
    const long long npw_h = pl.npw_h, nloc = v1 - v0;
    const double N8 = 8.0 * (double)pl.N;
    int rc;
    if ((rc = wait_inputs(h))) return rc;
    if ((rc = ensure_u_pw(h))) return rc;
    if ((rc = ensure_u_apply(h))) return rc;
    const double *ua = h->u_a ? h->u_a : h->u;
    if ((rc = ensure_k1e_ws(h, (size_t)(h->Pb + 1) * pl.N * 8))) return rc;
    double *vH = h->k1e_ws, *prod = h->k1e_ws + pl.N;
    double2 *og = (double2 *)out_rows;
    for (int b = 0; b < B; ++b) {
        if ((rc = st_inv_stick(h, pl, (const double2 *)vG + (long long)b * npw_h, 1))) return rc;
        if ((rc = st_inv_plane(h, pl, 1, vH))) return rc;
        for (long long c0 = 0; c0 < nloc; c0 += h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, nloc - c0);
            { StageTimer t(h, BSE_ST_K1E_PRODUCT, 2.0 * cnt * (double)pl.N, N8 * (2.0 * cnt + 1));
              if ((rc = bse_launch_k1e_product(ua, vH, prod, (int)(v0 + c0), cnt, h->Pb, pl.N, 1, h->stream))) return rc; }
            if ((rc = st_fwd_plane(h, pl, prod, nullptr, 0, cnt))) return rc;
            if ((rc = st_fwd_stick(h, pl, cnt, og + ((long long)b * nloc + c0) * npw_h, pl.inv2n))) return rc;
        }
    }
    return p_c_rows(h, out_rows, (long long)B * nloc, 2 * npw_h, (const double *)h->uGw, (const double *)h->uG, 1.0);
}

// Two-body kernel in one call (eq. 1: K1e and K1d enter with one P_c): out = P_c( ce * 2 u_v v_H + cd * sum_v' tau_vv' a_v' )
extern "C" int bse_apply_k1(bse_handle *h, const double *a, double *out, int B, double ce, double cd) {
    if (!h || !a || !out || B <= 0) { bse_set_error("null pointer or B <= 0"); return BSE_EINVAL; }
    if (!h->built) { bse_set_error("bse_apply_k1 before bse_build_tau"); return BSE_ESTATE; }
    if (a == out) { bse_set_error("out must not alias a"); return BSE_EINVAL; }
    int rc;
    const bool pw = (h->flags & BSE_VEC_PW) != 0;
    const bool batched = (h->flags & BSE_TAU_MASK) != BSE_TAU_REAL;
    if (h->rows_set) { bse_set_error("bse_apply_k1 is not available on a row-sharded handle"); return BSE_EUNSUPPORTED; }
    if (pw && batched) {
        // plane-slab path (the one bse_apply_k1x takes) with room kept for u and v_H of one slab
        if ((rc = ensure_u_pw(h))) return rc;
        if ((h->flags & BSE_TAU_MASK) == BSE_TAU_STREAM) {
            if ((rc = ensure_tau_store(h, false))) return rc;
            if ((rc = fill_tau_store(h, false))) return rc;
        }
        if (h->u_a) {                                           // a copy left by bse_apply_k1e: give its memory to the plan
            BSE_CUDA(cudaStreamSynchronize(h->stream));
            cudaFree(h->u_a);
            h->u_a = nullptr; h->u_a_valid = false;
            h->plan_ok = false;
        }
        if (!h->plan_ok || (h->slab_mode && !h->plan_mix)) {     // about to plan: the K1e scratch of another call would eat the slab's room
            BSE_CUDA(cudaStreamSynchronize(h->stream));
            cudaFree(h->k1e_ws);
            h->k1e_ws = nullptr; h->k1e_bytes = 0;
        }
        if ((rc = plan_apply_memory(h, B, true, true))) return rc;
        if (h->slab_mode) {
            const size_t SN = (size_t)h->slab_M * h->ap->n * h->ap->n;
            if ((rc = ensure_k1e_ws(h, ((size_t)h->Nv + B) * SN * 8 + (size_t)B * h->ap->npw_h * 16))) return rc;
            if (!h->slab_mode || !h->plan_ok) { bse_set_error("bse_apply_k1: the slab workspace did not fit"); return BSE_ENOMEM; }
            h->mix_ce = ce; h->mix_cd = cd; h->mix_B = B;
            h->mix_on = true;
            rc = apply_pw(h, (const double2 *)a, (double2 *)out, B);
            h->mix_on = false;
            return rc;
        }
    }
    const bool fly = pw && h->ap != &h->fft && batched;         // u on the apply grid is made on
    if (pw && (rc = ensure_u_pw(h))) return rc;                 // the fly from u(G), Pb orbitals at a time: no [Nv][Na] copy
    if (pw && !fly && (rc = ensure_u_apply(h))) return rc;
    if (fly && h->u_a) {                                        // a copy left by bse_apply_k1e: give its memory to the plan
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        cudaFree(h->u_a);
        h->u_a = nullptr; h->u_a_valid = false;
        h->plan_ok = false;
    }
    if ((rc = ensure_k1e_ws(h, (size_t)(B + (fly ? h->Pb : 0)) * h->ap->N * 8))) return rc;
    if ((h->flags & BSE_TAU_MASK) == BSE_TAU_STREAM && !(pw && batched)) {
        if ((rc = ensure_tau_store(h, false))) return rc;
        if ((rc = fill_tau_store(h, false))) return rc;
    }
    if ((rc = plan_apply_memory(h, B, pw && batched, pw && batched))) return rc;   // group / row-batch path (same plan as above)
    h->mix_ce = ce; h->mix_cd = cd; h->mix_B = B;
    h->mix_u = fly ? nullptr : ((pw && h->u_a) ? h->u_a : h->u);
    if (pw) {
        h->mix_on = true;
        rc = apply_pw(h, (const double2 *)a, (double2 *)out, B);
        h->mix_on = false;
        return rc;
    }
    const FftPlan &pl = h->fft;
    { StageTimer t(h, BSE_ST_K1E_DENSITY, 2.0 * B * h->Nv * (double)pl.N, 8.0 * pl.N * (double)(B * h->Nv + h->Nv + B));
      if ((rc = bse_launch_k1e_density(h->u, a, h->k1e_ws, h->Nv, pl.N, B, h->stream))) return rc; }
    if ((rc = hartree_in_place(h, pl, h->k1e_ws, B))) return rc;
    h->mix_vH = h->k1e_ws;
    h->mix_on = true;
    rc = accumulate_all(h, a, B, out, nullptr);
    h->mix_on = false;
    if (rc) return rc;
    return p_c_rows_real(h, out, (long long)B * h->Nv);
}

// KS <-> localised representation of the trial blocks (eq. 12): y[b] = U x[b] or U^T x[b]
extern "C" int bse_rotate(bse_handle *h, const double *U, int transpose, const double *x, double *y, int B) {
    if (!h || !U || !x || !y || B <= 0) { bse_set_error("null pointer or B <= 0"); return BSE_EINVAL; }
    if (x == y) { bse_set_error("y must not alias x"); return BSE_EINVAL; }
    const long long K = (h->flags & BSE_VEC_PW) ? 2 * h->fft.npw_h : h->N;
    const long long lds = ldS(h);
    const double *A = U;
    long long lda = h->Nv;
    int rc;
    if (transpose) {
        if (!h->Ut) BSE_CUDA(cudaMalloc(&h->Ut, (size_t)h->Nv * lds * 8));
        if ((rc = bse_launch_transpose(U, h->Nv, h->Ut, lds, h->Nv, h->stream))) return rc;
        A = h->Ut;
        lda = lds;
    }
    if (h->Nv & 1) {                       // the tile loader copies 16 B at a time: odd row lengths go through a padded copy
        if (!transpose) {
            if (!h->Ut) BSE_CUDA(cudaMalloc(&h->Ut, (size_t)h->Nv * lds * 8));
            BSE_CUDA(cudaMemcpy2DAsync(h->Ut, (size_t)lds * 8, U, (size_t)h->Nv * 8, (size_t)h->Nv * 8, h->Nv,
                                       cudaMemcpyDeviceToDevice, h->stream));
            A = h->Ut;
            lda = lds;
        }
    }
    for (int b = 0; b < B; ++b)
        if ((rc = bse_gemm_nn(A, lda, x + (long long)b * h->Nv * K, K, h->Nv, K, h->Nv, EPI_STORE, nullptr, nullptr,
                              y + (long long)b * h->Nv * K, K, h->stream))) return rc;
    return BSE_OK;
}

// ------------------------------------------------------------------------------------------------ accessors
extern "C" int bse_npw_half(const bse_handle *h, long long *npw_h) {
    if (!h || !npw_h) return BSE_EINVAL;
    *npw_h = h->fft.npw_h;
    return BSE_OK;
}
extern "C" int bse_gvectors(const bse_handle *h, int *mill) {
    if (!h || !mill) return BSE_EINVAL;
    std::memcpy(mill, h->mill.data(), h->mill.size() * sizeof(int));
    return BSE_OK;
}
extern "C" int bse_num_pairs(const bse_handle *h, long long *P) {
    if (!h || !P) return BSE_EINVAL;
    if (h->P < 0) { bse_set_error("no pair list yet"); return BSE_ESTATE; }
    *P = h->P;
    return BSE_OK;
}
extern "C" int bse_get_pairs(const bse_handle *h, int *pairs) {
    if (!h || !pairs) return BSE_EINVAL;
    if (h->P < 0) { bse_set_error("no pair list yet"); return BSE_ESTATE; }
    BSE_CUDA(cudaMemcpyAsync(pairs, h->pairs, (size_t)h->P * 8, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    return BSE_OK;
}
extern "C" int bse_get_overlap(const bse_handle *h, double *O) {
    if (!h || !O) return BSE_EINVAL;
    if (h->P < 0) { bse_set_error("no screen yet"); return BSE_ESTATE; }
    const int Nv = h->Nv;
    std::vector<double> M((size_t)Nv * Nv);
    BSE_CUDA(cudaMemcpyAsync(M.data(), h->Mmat, M.size() * 8, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    for (int v = 0; v < Nv; ++v)             // the device holds the upper triangle (v <= w) only
        for (int w = v; w < Nv; ++w)
            O[(size_t)v * Nv + w] = O[(size_t)w * Nv + v] =
                M[(size_t)v * Nv + w] / std::sqrt(M[(size_t)v * Nv + v] * M[(size_t)w * Nv + w]);
    return BSE_OK;
}
extern "C" int bse_get_tau(bse_handle *h, long long first, long long count, double *dst, unsigned layout) {
    if (!h || !dst || first < 0 || count < 0) return BSE_EINVAL;
    if (!h->built) { bse_set_error("bse_get_tau before bse_build_tau"); return BSE_ESTATE; }
    if (first + count > h->P) { bse_set_error("pair range out of bounds"); return BSE_EINVAL; }
    const unsigned mode = h->flags & BSE_TAU_MASK;
    const long long npw_h = h->fft.npw_h;
    if (layout == BSE_TAU_REAL && mode == BSE_TAU_REAL && !h->rows_set) {
        BSE_CUDA(cudaMemcpyAsync(dst, h->tau_r + first * h->N, (size_t)count * h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
        return BSE_OK;
    }
    if (layout == BSE_TAU_PW && mode == BSE_TAU_PW && !h->rows_set && !h->tau_g32) {
        BSE_CUDA(cudaMemcpyAsync(dst, h->tau_g + first * npw_h, (size_t)count * npw_h * 16, cudaMemcpyDeviceToDevice, h->stream));
        return BSE_OK;
    }
    if (layout != BSE_TAU_REAL && layout != BSE_TAU_PW) { bse_set_error("bad layout"); return BSE_EINVAL; }
    // recompute batch by batch straight into dst
    int rc;
    for (long long p0 = first; p0 < first + count; p0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, first + count - p0);
        if (layout == BSE_TAU_PW) rc = run_pair_batch(h, h->pairs, p0, cnt, (double2 *)dst + (p0 - first) * npw_h, nullptr);
        else rc = run_pair_batch(h, h->pairs, p0, cnt, h->T, dst + (p0 - first) * h->N);
        if (rc) return rc;
    }
    return BSE_OK;
}

// Debug / test knobs (they only ever lower a limit or pick between equivalent kernels; results do not change)
extern "C" int bse_debug_set(bse_handle *h, const char *key, long long value) {
    if (!h || !key) { bse_set_error("null pointer"); return BSE_EINVAL; }
    const std::string k(key);
    if (k == "max_group") { h->dbg_max_group = value; h->plan_ok = false; }
    else if (k == "max_batch") { h->dbg_max_batch = value; h->plan_ok = false; }
    else if (k == "compact_inv") { h->fft.compact_inv = h->ffta.compact_inv = (int)value; }
    else if (k == "pipe") { h->fft.pipe = h->ffta.pipe = (int)value; }
    else if (k == "pipe_lc") { h->fft.pipe_lc = h->ffta.pipe_lc = (int)value; }
    else if (k == "slab_rows") { h->dbg_slab_rows = value; h->plan_ok = false; }
    else if (k == "gemm_bm") { bse_gemm_set_bm((int)value); }       // process-wide: CTA tile height of the DMMA GEMMs
    else if (k == "slab_planes") { h->dbg_slab_planes = value; h->plan_ok = false; }
    else if (k == "pc_rows") { h->dbg_pc_rows = value; }
    else if (k == "in_chunks") { h->dbg_in_chunks = value; }
    else { bse_set_error("bse_debug_set: unknown key " + k); return BSE_EINVAL; }
    return BSE_OK;
}

// Device time of the most recent fill of the tau store (a2..a8(+a9) for all P pairs): inside bse_build_tau for BSE_TAU_REAL / PW,
// inside bse_apply_k1x / bse_apply_k1 for BSE_TAU_STREAM.  Synchronises on the closing event.
extern "C" int bse_last_tau_fill_ms(bse_handle *h, double *ms) {
    if (!h || !ms) { bse_set_error("null pointer"); return BSE_EINVAL; }
    if (!h->fill_timed) { bse_set_error("no tau fill yet"); return BSE_ESTATE; }
    BSE_CUDA(cudaEventSynchronize(h->ev_fill1));
    float f = 0.f;
    BSE_CUDA(cudaEventElapsedTime(&f, h->ev_fill0, h->ev_fill1));
    *ms = f;
    return BSE_OK;
}

extern "C" int bse_profile_enable(bse_handle *h, int enable) {
    if (!h) return BSE_EINVAL;
    h->prof = enable != 0;
    return BSE_OK;
}
extern "C" int bse_profile_reset(bse_handle *h) {
    if (!h) return BSE_EINVAL;
    for (int i = 0; i < BSE_ST_COUNT; ++i) { h->st_ms[i] = 0; h->st_launch[i] = 0; h->st_flops[i] = 0; h->st_bytes[i] = 0; h->st_handoff[i] = 0; }
    return BSE_OK;
}
extern "C" int bse_profile_get(const bse_handle *h, double *ms, long long *launches) {
    if (!h) return BSE_EINVAL;
    for (int i = 0; i < BSE_ST_COUNT; ++i) {
        if (ms) ms[i] = h->st_ms[i];
        if (launches) launches[i] = h->st_launch[i];
    }
    return BSE_OK;
}
extern "C" int bse_profile_model(const bse_handle *h, double *flops, double *bytes) {
    if (!h) return BSE_EINVAL;
    for (int i = 0; i < BSE_ST_COUNT; ++i) {
        if (flops) flops[i] = h->st_flops[i];
        if (bytes) bytes[i] = h->st_bytes[i];
    }
    return BSE_OK;
}
extern "C" int bse_profile_handoff(const bse_handle *h, double *bytes) {
    if (!h || !bytes) return BSE_EINVAL;
    for (int i = 0; i < BSE_ST_COUNT; ++i) bytes[i] = h->st_handoff[i];
    return BSE_OK;
}
