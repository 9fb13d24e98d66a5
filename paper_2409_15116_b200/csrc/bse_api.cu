// C-ABI entry points of libbse_b200 (include/bse.h): host-side tables, orchestration of the kernel sequence.
// Path:  a1 screen -> pair list -> per pair batch [a2+a3 plane pass, a3+a4 stick pass,
// a5+a6 projection DGEMM, a7+a8 back-projection DGEMM, a9 inverse stick + plane pass] ; apply: a10 accumulate,
// a11 P_c (two DGEMMs).  No CPU fallback: every numeric step is a kernel in this library.
#include <algorithm>
#include <cmath>
#include <cstdio>
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
    "inv_stick", "inv_plane", "k1x_accumulate", "pc_overlap", "pc_update"};
extern "C" const char *bse_stage_name(int s) { return (s >= 0 && s < BSE_ST_COUNT) ? k_stage_names[s] : "?"; }

namespace {

template <typename T>
int upload(T *&dst, const std::vector<T> &src) {
    BSE_CUDA(cudaMalloc(&dst, std::max<size_t>(src.size(), 1) * sizeof(T)));
    if (!src.empty()) BSE_CUDA(cudaMemcpy(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return BSE_OK;
}

struct StageTimer {
    bse_handle *h; int st;
    StageTimer(bse_handle *h_, int st_) : h(h_), st(st_) {
        if (h->prof) cudaEventRecord(h->ev0, h->stream);
    }
    ~StageTimer() {
        h->st_launch[st] += 1;
        if (h->prof) {
            cudaEventRecord(h->ev1, h->stream);
            cudaEventSynchronize(h->ev1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, h->ev0, h->ev1);
            h->st_ms[st] += ms;
        }
    }
};

int build_fft_plan(bse_handle *h) {
    FftPlan &pl = h->fft;
    const int n = h->n;
    pl.n = n;
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
                const long long key = ((long long)((m1 + n) % n) * n + (m2 + n) % n) * n + (m3 + n) % n;
                H.push_back({m1, m2, m3, key});
            }
    std::sort(H.begin(), H.end(), [](const M3 &a, const M3 &b) { return a.key < b.key; });
    pl.npw_h = (long long)H.size();
    const int D = 2 * R + 1;
    std::vector<int> hidx((size_t)D * D * D, -1);
    auto hid = [&](int m1, int m2, int m3) -> int & { return hidx[((size_t)(m1 + R) * D + (m2 + R)) * D + (m3 + R)]; };
    h->mill.resize(H.size() * 3);
    std::vector<double> vc12(H.size()), vc12n(H.size()), inv2n(H.size());
    const double twopi_L = 2.0 * M_PI / h->L;
    for (size_t i = 0; i < H.size(); ++i) {
        hid(H[i].m1, H[i].m2, H[i].m3) = (int)i;
        h->mill[3 * i] = H[i].m1; h->mill[3 * i + 1] = H[i].m2; h->mill[3 * i + 2] = H[i].m3;
        const int q = H[i].m1 * H[i].m1 + H[i].m2 * H[i].m2 + H[i].m3 * H[i].m3;
        vc12[i] = q == 0 ? 0.0 : std::sqrt(4.0 * M_PI) / (twopi_L * std::sqrt((double)q));
        vc12n[i] = vc12[i] / (2.0 * (double)h->N);
        inv2n[i] = 1.0 / (2.0 * (double)h->N);
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
    return BSE_OK;
}

void free_plan(FftPlan &pl) {
    cudaFree(pl.tw); cudaFree(pl.soff); cudaFree(pl.wmax); cudaFree(pl.wmin); cudaFree(pl.hmapT);
    cudaFree(pl.vc12); cudaFree(pl.vc12n); cudaFree(pl.inv2n);
}

inline long long ldD(const bse_handle *h) { return (h->Npdep + 1) & ~1; }
inline long long ldS(const bse_handle *h) { return (h->Nv + 1) & ~1; }

// tau for pairs [p0, p0+cnt): a2..a8 into dstG ([cnt][npw_h] complex), then a9 into dstR ([cnt][N]) if given
int run_pair_batch(bse_handle *h, long long p0, int cnt, double2 *dstG, double *dstR) {
    const FftPlan &pl = h->fft;
    int rc;
    { StageTimer t(h, BSE_ST_FWD_PLANE);
      if ((rc = bse_launch_fwd_plane(pl, h->u, h->pairs, p0, cnt, h->N, h->Z, h->stream))) return rc; }
    { StageTimer t(h, BSE_ST_FWD_STICK);
      if ((rc = bse_launch_fwd_stick(pl, h->Z, cnt, h->X, pl.vc12n, h->stream))) return rc; }
    const long long K2 = 2 * pl.npw_h;
    { StageTimer t(h, BSE_ST_PROJECT);
      if ((rc = bse_gemm_dot((const double *)h->X, K2, h->phi, K2, cnt, h->Npdep, K2, false, false, h->part,
                             h->part_bytes, h->Dm, ldD(h), 1.0, h->f2, h->stream))) return rc; }
    { StageTimer t(h, BSE_ST_BACKPROJECT);
      if ((rc = bse_gemm_nn(h->Dm, ldD(h), h->phi, K2, cnt, K2, h->Npdep, EPI_TAU, (const double *)h->X, pl.vc12,
                            (double *)dstG, K2, h->stream))) return rc; }
    if (dstR) {
        { StageTimer t(h, BSE_ST_INV_STICK);
          if ((rc = bse_launch_inv_stick(pl, dstG, cnt, h->Z, h->stream))) return rc; }
        { StageTimer t(h, BSE_ST_INV_PLANE);
          if ((rc = bse_launch_inv_plane(pl, h->Z, cnt, h->N, dstR, h->stream))) return rc; }
    }
    return BSE_OK;
}

int ensure_tau_batch(bse_handle *h) {
    if (!h->tau_batch) BSE_CUDA(cudaMalloc(&h->tau_batch, (size_t)h->Pb * h->N * 8));
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

int p_c_project(bse_handle *h, double *out, int B) {
    // out currently holds acc.  S = dV acc u^T (split-K dot GEMM), out -= S u (NN GEMM)
    const long long rows = (long long)B * h->Nv;
    const long long lds = ldS(h);
    int rc0;
    if ((rc0 = ensure_sov(h, rows))) return rc0;
    long long mc = rows;
    const long long per_row = (long long)h->Nv * 8 * 2;
    if (rows * per_row > (long long)h->part_bytes) mc = std::max<long long>(64, (long long)(h->part_bytes / per_row) / 64 * 64);
    int rc;
    for (long long r0 = 0; r0 < rows; r0 += mc) {
        const int m = (int)std::min(mc, rows - r0);
        { StageTimer t(h, BSE_ST_PC_OVERLAP);
          if ((rc = bse_gemm_dot(out + r0 * h->N, h->N, h->u, h->N, m, h->Nv, h->N, false, false, h->part,
                                 h->part_bytes, h->Sov + r0 * lds, lds, h->dV, nullptr, h->stream))) return rc; }
        { StageTimer t(h, BSE_ST_PC_UPDATE);
          if ((rc = bse_gemm_nn(h->Sov + r0 * lds, lds, h->u, h->N, m, h->N, h->Nv, EPI_SUB, nullptr, nullptr,
                                out + r0 * h->N, h->N, h->stream))) return rc; }
    }
    return BSE_OK;
}


// u_w(G) on H for the PW layout (a12): forward transform of every orbital, no pair product, scale 1/(2N) -> uG;
// uGw = Omega * wt(G) * uG with wt = 2 (G != 0), (1, 0) on (re, im) of G = 0, so that the half-sphere real dot product
// sum_k uGw[w][k] x[k] equals <u_w|x> = Omega sum_{G in S} conj(u_w(G)) x(G)   (S14).
int ensure_u_pw(bse_handle *h) {
    if (h->uG) return BSE_OK;
    const FftPlan &pl = h->fft;
    const size_t bytes = (size_t)h->Nv * pl.npw_h * 16;
    BSE_CUDA(cudaMalloc(&h->uG, bytes));
    BSE_CUDA(cudaMalloc(&h->uGw, bytes));
    int rc;
    for (long long v0 = 0; v0 < h->Nv; v0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, h->Nv - v0);
        { StageTimer t(h, BSE_ST_FWD_PLANE);
          if ((rc = bse_launch_fwd_plane(pl, h->u, nullptr, v0, cnt, h->N, h->Z, h->stream))) return rc; }
        { StageTimer t(h, BSE_ST_FWD_STICK);
          if ((rc = bse_launch_fwd_stick(pl, h->Z, cnt, h->uG + v0 * pl.npw_h, pl.inv2n, h->stream))) return rc; }
    }
    return bse_launch_weight_pw(h->uG, h->uGw, pl.npw_h, h->Nv, h->Omega, h->stream);
}

// real-space staging of one group of trial blocks: a_r, acc_r = [Bg][Nv][N]; Bg from the memory that is free now
int ensure_vec_stage(bse_handle *h, int B) {
    const size_t per_block = (size_t)h->Nv * h->N * 8 * 2;
    if (h->Bg >= 1 && (h->Bg >= B || h->Bg_final)) return BSE_OK;
    cudaFree(h->a_r); cudaFree(h->acc_r);
    h->a_r = h->acc_r = nullptr; h->Bg = 0;
    size_t free_b = 0, total_b = 0;
    cudaMemGetInfo(&free_b, &total_b);
    const size_t reserve = (size_t)512 << 20;
    long long bg = free_b > reserve ? (long long)((free_b - reserve) / per_block) : 0;
    if (bg < 1) {
        char msg[200];
        snprintf(msg, sizeof msg, "PW layout needs %.2f GB of real-space staging per trial block, %.2f GB free",
                 per_block / 1e9, free_b / 1e9);
        bse_set_error(msg);
        return BSE_ENOMEM;
    }
    h->Bg_final = bg < B;
    if (bg > B) bg = B;
    BSE_CUDA(cudaMalloc(&h->a_r, (size_t)bg * h->Nv * h->N * 8));
    BSE_CUDA(cudaMalloc(&h->acc_r, (size_t)bg * h->Nv * h->N * 8));
    h->Bg = (int)bg;
    return BSE_OK;
}

// acc (real space, [nb][Nv][N]) for the listed pairs: tau from the store or rebuilt per batch   (a9, a10)
int accumulate_all(bse_handle *h, const double *a, double *acc, int nb) {
    const unsigned mode = h->flags & BSE_TAU_MASK;
    int rc;
    if (mode == BSE_TAU_REAL) {
        StageTimer t(h, BSE_ST_ACCUM);
        return bse_launch_accumulate(h, h->tau_r, 0, h->P, a, acc, nb, true);
    }
    if ((rc = ensure_tau_batch(h))) return rc;
    for (long long p0 = 0; p0 < h->P; p0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, h->P - p0);
        if (mode == BSE_TAU_PW) {
            { StageTimer t(h, BSE_ST_INV_STICK);
              if ((rc = bse_launch_inv_stick(h->fft, h->tau_g + p0 * h->fft.npw_h, cnt, h->Z, h->stream))) return rc; }
            { StageTimer t(h, BSE_ST_INV_PLANE);
              if ((rc = bse_launch_inv_plane(h->fft, h->Z, cnt, h->N, h->tau_batch, h->stream))) return rc; }
        } else {
            if ((rc = run_pair_batch(h, p0, cnt, h->T, h->tau_batch))) return rc;
        }
        StageTimer t(h, BSE_ST_ACCUM);
        if ((rc = bse_launch_accumulate(h, h->tau_batch, p0, cnt, a, acc, nb, p0 == 0))) return rc;
    }
    return BSE_OK;
}

// PW layout (a12): a, out = [B][Nv][npw_h] complex on H
int apply_pw(bse_handle *h, const double2 *a, double2 *out, int B) {
    const FftPlan &pl = h->fft;
    int rc;
    if ((rc = ensure_u_pw(h))) return rc;
    if ((rc = ensure_vec_stage(h, B))) return rc;
    const long long Nv = h->Nv, npw_h = pl.npw_h;
    for (int b0 = 0; b0 < B; b0 += h->Bg) {
        const int nb = std::min(h->Bg, B - b0);
        const long long fields = (long long)nb * Nv;
        const double2 *ag = a + (long long)b0 * Nv * npw_h;
        double2 *og = out + (long long)b0 * Nv * npw_h;
        for (long long f0 = 0; f0 < fields; f0 += h->Pb) {           // a(G) -> a(r)
            const int cnt = (int)std::min<long long>(h->Pb, fields - f0);
            { StageTimer t(h, BSE_ST_INV_STICK);
              if ((rc = bse_launch_inv_stick(pl, ag + f0 * npw_h, cnt, h->Z, h->stream))) return rc; }
            { StageTimer t(h, BSE_ST_INV_PLANE);
              if ((rc = bse_launch_inv_plane(pl, h->Z, cnt, h->N, h->a_r + f0 * h->N, h->stream))) return rc; }
        }
        if ((rc = accumulate_all(h, h->a_r, h->acc_r, nb))) return rc;
        for (long long f0 = 0; f0 < fields; f0 += h->Pb) {           // acc(r) -> acc(G), truncated to S (S15)
            const int cnt = (int)std::min<long long>(h->Pb, fields - f0);
            { StageTimer t(h, BSE_ST_FWD_PLANE);
              if ((rc = bse_launch_fwd_plane(pl, h->acc_r, nullptr, f0, cnt, h->N, h->Z, h->stream))) return rc; }
            { StageTimer t(h, BSE_ST_FWD_STICK);
              if ((rc = bse_launch_fwd_stick(pl, h->Z, cnt, og + f0 * npw_h, pl.inv2n, h->stream))) return rc; }
        }
    }
    // P_c in PW: S = <u_w|acc> (real dot GEMM against the weighted copy), out -= S u(G)
    const long long rows = (long long)B * Nv, K2 = 2 * npw_h, lds = ldS(h);
    if ((rc = ensure_sov(h, rows))) return rc;
    long long mc = rows;
    const long long per_row = Nv * 8 * 2;
    if (rows * per_row > (long long)h->part_bytes) mc = std::max<long long>(64, (long long)(h->part_bytes / per_row) / 64 * 64);
    double *o = (double *)out;
    for (long long r0 = 0; r0 < rows; r0 += mc) {
        const int m = (int)std::min(mc, rows - r0);
        { StageTimer t(h, BSE_ST_PC_OVERLAP);
          if ((rc = bse_gemm_dot(o + r0 * K2, K2, (const double *)h->uGw, K2, m, h->Nv, K2, false, false, h->part,
                                 h->part_bytes, h->Sov + r0 * lds, lds, 1.0, nullptr, h->stream))) return rc; }
        { StageTimer t(h, BSE_ST_PC_UPDATE);
          if ((rc = bse_gemm_nn(h->Sov + r0 * lds, lds, (const double *)h->uG, K2, m, K2, h->Nv, EPI_SUB, nullptr, nullptr,
                                o + r0 * K2, K2, h->stream))) return rc; }
    }
    return BSE_OK;
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
    h->stream = (cudaStream_t)stream;
    h->msq_max = (int)std::floor(2.0 * ecut * (L / (2.0 * M_PI)) * (L / (2.0 * M_PI)) * (1.0 + 1e-12));
    const int R = (int)std::floor(std::sqrt((double)h->msq_max) + 1e-9);
    int rc = BSE_OK;
    auto fail = [&](int code) { bse_destroy(h); return code; };
    if (2 * R >= h->n) { bse_set_error("sphere does not fit the grid (R >= n/2)"); return fail(BSE_EINVAL); }
    if ((rc = build_fft_plan(h))) return fail(rc);
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
    size_t budget = std::min<size_t>((size_t)6 << 30, free_b / 4);
    long long Pb = (long long)(budget / (per_pair + per_pair_r));
    Pb = std::max<long long>(1, std::min<long long>(Pb, 256));
    h->Pb = Pb;
    h->part_bytes = std::max<size_t>((size_t)64 << 20, nv2 * 8 * 2);
    if (cudaMalloc(&h->Z, (size_t)Pb * h->n * h->fft.NS * 16) || cudaMalloc(&h->X, (size_t)Pb * h->fft.npw_h * 16) ||
        cudaMalloc(&h->T, (size_t)Pb * h->fft.npw_h * 16) || cudaMalloc(&h->Dm, (size_t)Pb * ldD(h) * 8) ||
        cudaMalloc(&h->part, h->part_bytes)) {
        bse_set_error("out of device memory (workspaces)");
        return fail(BSE_ENOMEM);
    }
    cudaEventCreate(&h->ev0);
    cudaEventCreate(&h->ev1);
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) { bse_set_error("stream sync failed"); return fail(BSE_ECUDA); }
    *hout = h;
    return BSE_OK;
}

extern "C" int bse_destroy(bse_handle *h) {
    if (!h) return BSE_OK;
    cudaStreamSynchronize(h->stream);
    free_plan(h->fft);
    cudaFree(h->u_owned); cudaFree(h->phi_owned); cudaFree(h->f2); cudaFree(h->Mmat); cudaFree(h->rowcnt);
    cudaFree(h->rowptr); cudaFree(h->pid); cudaFree(h->pairs); cudaFree(h->adj_ptr); cudaFree(h->adj);
    cudaFree(h->tau_r); cudaFree(h->tau_g); cudaFree(h->Z); cudaFree(h->X); cudaFree(h->T); cudaFree(h->Dm);
    cudaFree(h->part); cudaFree(h->Sov); cudaFree(h->tau_batch); cudaFree(h->a_dev); cudaFree(h->out_dev);
    cudaFree(h->uG); cudaFree(h->uGw); cudaFree(h->a_r); cudaFree(h->acc_r);
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    delete h;
    return BSE_OK;
}

extern "C" int bse_build_tau(bse_handle *h) {
    if (!h) { bse_set_error("null handle"); return BSE_EINVAL; }
    int rc;
    h->built = false;
    // a1: M = (u^2)(u^2)^T, then the threshold decision and the list, all on the device
    { StageTimer t(h, BSE_ST_SCREEN);
      if ((rc = bse_gemm_dot(h->u, h->N, h->u, h->N, h->Nv, h->Nv, h->N, true, true, h->part, h->part_bytes, h->Mmat,
                             h->Nv, 1.0, nullptr, h->stream))) return rc; }
    { StageTimer t(h, BSE_ST_PAIRLIST);
      if ((rc = bse_launch_pairlist(h))) return rc; }
    const unsigned mode = h->flags & BSE_TAU_MASK;
    if (mode != BSE_TAU_STREAM) {
        const size_t need = (mode == BSE_TAU_REAL) ? (size_t)h->P * h->N * 8 : (size_t)h->P * h->fft.npw_h * 16;
        if (need > h->tau_bytes) {            // grow-only store: a rebuild with the same list allocates nothing
            cudaFree(h->tau_r); h->tau_r = nullptr;
            cudaFree(h->tau_g); h->tau_g = nullptr;
            h->tau_bytes = 0;
            size_t free_b = 0, total_b = 0;
            cudaMemGetInfo(&free_b, &total_b);
            if (need + ((size_t)256 << 20) > free_b) {
                char msg[160];
                snprintf(msg, sizeof msg, "tau store needs %.2f GB, %.2f GB free: use BSE_TAU_PW or BSE_TAU_STREAM",
                         need / 1e9, free_b / 1e9);
                bse_set_error(msg);
                return BSE_ENOMEM;
            }
            if (mode == BSE_TAU_REAL) BSE_CUDA(cudaMalloc(&h->tau_r, need));
            else BSE_CUDA(cudaMalloc(&h->tau_g, need));
            h->tau_bytes = need;
        }
        for (long long p0 = 0; p0 < h->P; p0 += h->Pb) {
            const int cnt = (int)std::min<long long>(h->Pb, h->P - p0);
            if (mode == BSE_TAU_REAL) rc = run_pair_batch(h, p0, cnt, h->T, h->tau_r + p0 * h->N);
            else rc = run_pair_batch(h, p0, cnt, h->tau_g + p0 * h->fft.npw_h, nullptr);
            if (rc) return rc;
        }
    }
    h->built = true;
    return BSE_OK;
}

extern "C" int bse_apply_k1x(bse_handle *h, const double *a, double *out, int B) {
    if (!h || !a || !out || B <= 0) { bse_set_error("null pointer or B <= 0"); return BSE_EINVAL; }
    if (!h->built) { bse_set_error("bse_apply_k1x before bse_build_tau"); return BSE_ESTATE; }
    if (a == out) { bse_set_error("out must not alias a"); return BSE_EINVAL; }
    int rc;
    if (h->flags & BSE_VEC_PW) return apply_pw(h, (const double2 *)a, (double2 *)out, B);
    if ((rc = accumulate_all(h, a, out, B))) return rc;
    return p_c_project(h, out, B);
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
    BSE_CUDA(cudaMemcpyAsync(h->a_dev, a_host, bytes, cudaMemcpyHostToDevice, h->stream));
    const int rc = bse_apply_k1x(h, h->a_dev, h->out_dev, B);
    if (rc) return rc;
    BSE_CUDA(cudaMemcpyAsync(out_host, h->out_dev, bytes, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
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
    for (int v = 0; v < Nv; ++v)
        for (int w = 0; w < Nv; ++w)
            O[(size_t)v * Nv + w] = M[(size_t)v * Nv + w] / std::sqrt(M[(size_t)v * Nv + v] * M[(size_t)w * Nv + w]);
    return BSE_OK;
}
extern "C" int bse_get_tau(bse_handle *h, long long first, long long count, double *dst, unsigned layout) {
    if (!h || !dst || first < 0 || count < 0) return BSE_EINVAL;
    if (!h->built) { bse_set_error("bse_get_tau before bse_build_tau"); return BSE_ESTATE; }
    if (first + count > h->P) { bse_set_error("pair range out of bounds"); return BSE_EINVAL; }
    const unsigned mode = h->flags & BSE_TAU_MASK;
    const long long npw_h = h->fft.npw_h;
    if (layout == BSE_TAU_REAL && mode == BSE_TAU_REAL) {
        BSE_CUDA(cudaMemcpyAsync(dst, h->tau_r + first * h->N, (size_t)count * h->N * 8, cudaMemcpyDeviceToDevice, h->stream));
        return BSE_OK;
    }
    if (layout == BSE_TAU_PW && mode == BSE_TAU_PW) {
        BSE_CUDA(cudaMemcpyAsync(dst, h->tau_g + first * npw_h, (size_t)count * npw_h * 16, cudaMemcpyDeviceToDevice, h->stream));
        return BSE_OK;
    }
    if (layout != BSE_TAU_REAL && layout != BSE_TAU_PW) { bse_set_error("bad layout"); return BSE_EINVAL; }
    // recompute batch by batch straight into dst
    int rc;
    for (long long p0 = first; p0 < first + count; p0 += h->Pb) {
        const int cnt = (int)std::min<long long>(h->Pb, first + count - p0);
        if (layout == BSE_TAU_PW) rc = run_pair_batch(h, p0, cnt, (double2 *)dst + (p0 - first) * npw_h, nullptr);
        else rc = run_pair_batch(h, p0, cnt, h->T, dst + (p0 - first) * h->N);
        if (rc) return rc;
    }
    return BSE_OK;
}

extern "C" int bse_profile_enable(bse_handle *h, int enable) {
    if (!h) return BSE_EINVAL;
    h->prof = enable != 0;
    return BSE_OK;
}
extern "C" int bse_profile_reset(bse_handle *h) {
    if (!h) return BSE_EINVAL;
    for (int i = 0; i < BSE_ST_COUNT; ++i) { h->st_ms[i] = 0; h->st_launch[i] = 0; }
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
