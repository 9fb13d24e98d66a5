// Size dispatch of the two-pass FFT kernels (fft_kernels.cuh).  Each supported grid edge n = R1 * R2 is instantiated in
// one of the fft_sizes_*.cu translation units (compiled in parallel); this file holds the table and the launch wrappers.
#include <algorithm>

#include "fft_kernels.cuh"
#include "fft_slab.cuh"

namespace bsefft {
FftOps ops_12(); FftOps ops_16(); FftOps ops_20(); FftOps ops_24(); FftOps ops_30(); FftOps ops_32(); FftOps ops_36();
FftOps ops_40(); FftOps ops_48(); FftOps ops_60(); FftOps ops_64(); FftOps ops_72(); FftOps ops_80(); FftOps ops_96();
FftOps ops_100(); FftOps ops_108(); FftOps ops_120(); FftOps ops_128(); FftOps ops_144(); FftOps ops_160();
}  // namespace bsefft

using bsefft::FftOps;
using bsefft::PlanDev;

static const FftOps *find_ops(int n) {
    static const FftOps table[] = {
        bsefft::ops_12(), bsefft::ops_16(), bsefft::ops_20(), bsefft::ops_24(), bsefft::ops_30(), bsefft::ops_32(),
        bsefft::ops_36(), bsefft::ops_40(), bsefft::ops_48(), bsefft::ops_60(), bsefft::ops_64(), bsefft::ops_72(),
        bsefft::ops_80(), bsefft::ops_96(), bsefft::ops_100(), bsefft::ops_108(), bsefft::ops_120(), bsefft::ops_128(), bsefft::ops_144(),
        bsefft::ops_160()};
    for (const FftOps &o : table)
        if (o.n == n) return &o;
    return nullptr;
}

int bse_fft_select(FftPlan &pl) {
    const FftOps *o = find_ops(pl.n);
    if (!o) {
        bse_set_error("no FFT kernel for this grid edge (supported n: 12 16 20 24 30 32 36 40 48 60 64 72 80 96 100 108 120 128 144 160)");
        return BSE_EUNSUPPORTED;
    }
    pl.R1 = o->R1; pl.R2 = o->R2; pl.ops = o;
    return BSE_OK;
}

static PlanDev to_dev(const FftPlan &pl, int np = 0) {
    PlanDev d;
    d.R = pl.R; d.W = pl.W; d.NS = pl.NS;
    d.np = np > 0 ? np : pl.n;
    d.pipe = pl.pipe; d.pipe_lc = pl.pipe_lc;
    d.magicW = (1 << 20) / (pl.W > 0 ? pl.W : 1) + 1;
    d.tw = pl.tw; d.soff = pl.soff; d.wmax = pl.wmax; d.wmin = pl.wmin; d.hmapT = pl.hmapT;
    return d;
}

int bse_launch_fwd_plane(const FftPlan &pl, const double *fields, const int2 *pairs, long long p0, int count,
                         long long N, double2 *Z, cudaStream_t s, int np) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->fwd_plane(to_dev(pl, np), fields, pairs, p0, count, N, Z, s);
}
int bse_launch_inv_plane(const FftPlan &pl, const double2 *Z, int count, long long N, double *out, cudaStream_t s,
                         bool subtract, int np) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->inv_plane(to_dev(pl, np), Z, count, N, out, s, subtract ? 1 : 0, pl.compact_inv);
}
// slab stick passes: any factorisation n = S * M with M <= 32 (fft_slab.cuh); M = A * B with A the largest divisor <= sqrt(M)
static int slab_split(int M) {
    int A = 1;
    for (int a = 1; a * a <= M; ++a)
        if (M % a == 0) A = a;
    return A;
}
// the fields of a launch are spread over the CTAs of a stick group
static int slab_per_cta(int groups, int count) {
    // two CTAs are resident per SM (64 registers, 480 threads): ~16 waves of 296 CTAs, so that the last, partial wave costs
    // little (with 4 waves of CTAs that walk over 250 fields each, the tail was a sixth of the launch)
    const int want = std::max(1, (148 * 2 * 16 + groups - 1) / groups);   // field chunks per stick group
    return std::max(1, (count + want - 1) / want);
}
int bse_launch_inv_stick_slab(const FftPlan &pl, int S, int M, const double2 *T, int count, double2 *Zs, cudaStream_t s, int slab,
                              const int *gather, int g0, const float2 *T32) {
    if (count <= 0) return BSE_OK;
    if (S * M != pl.n || M > 32 || M < 1 || S > 16) { bse_set_error("slab stick pass: bad factorisation"); return BSE_EINVAL; }
    const PlanDev P = to_dev(pl);
    const int TS = bsefft::SLAB_TS, A = slab_split(M), groups = (pl.NS + TS - 1) / TS;
    const int NQt = S <= 4 ? 4 : (S <= 8 ? 8 : (S <= 12 ? 12 : 16)), Bt = M / A;
    const int smem = (2 * M * (TS + 1) + NQt * M + A * A + M + Bt * Bt) * 16;     // C | D | root tables (fft_slab.cuh)
    const int per = slab_per_cta(groups, count);
    const dim3 grid(groups, (count + per - 1) / per);
    const bool small = TS * M <= 512;
#define BSE_SLAB_PICK(name, ...) \
    (small ? (S <= 4 ? bsefft::name<4, 512, ##__VA_ARGS__> : (S <= 8 ? bsefft::name<8, 512, ##__VA_ARGS__> : (S <= 12 ? bsefft::name<12, 512, ##__VA_ARGS__> : bsefft::name<16, 512, ##__VA_ARGS__>))) \
           : (S <= 4 ? bsefft::name<4, 1024, ##__VA_ARGS__> : (S <= 8 ? bsefft::name<8, 1024, ##__VA_ARGS__> : (S <= 12 ? bsefft::name<12, 1024, ##__VA_ARGS__> : bsefft::name<16, 1024, ##__VA_ARGS__>))))
    // staged gathers (cp.async, one field ahead) where two CTAs per SM still fit beside the staging area
    const int stage_bytes = NQt * TS * M * 16;
    const bool staged = !T32 && small && per > 1 && 2 * (smem + stage_bytes + 1024) <= 232448;
    const int smem_all = smem + (staged ? stage_bytes : 0);
    auto kern = T32 ? BSE_SLAB_PICK(inv_stick_slab_kernel, true, false)
                    : (staged ? BSE_SLAB_PICK(inv_stick_slab_kernel, false, true) : BSE_SLAB_PICK(inv_stick_slab_kernel, false, false));
    if (smem_all > 48 * 1024) BSE_CUDA(cudaFuncSetAttribute((const void *)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_all));
    kern<<<grid, TS * M, smem_all, s>>>(P, pl.n, S, M, A, T, pl.npw_h, Zs, gather, g0, slab, count, per, T32,
                                        bsefft::slab_const(pl.n, M, A));
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}
int bse_launch_fwd_stick_slab(const FftPlan &pl, int S, int M, const double2 *Zs, int count, double2 *X, const double *scale,
                              cudaStream_t s, int slab, bool accumulate, int rc_rows, long long row_ld, long long row0) {
    if (count <= 0) return BSE_OK;
    if (S * M != pl.n || M > 32 || M < 1 || S > 16) { bse_set_error("slab stick pass: bad factorisation"); return BSE_EINVAL; }
    const PlanDev P = to_dev(pl);
    const int TS = bsefft::SLAB_TS, A = slab_split(M), groups = (pl.NS + TS - 1) / TS;
    const int NQt = S <= 4 ? 4 : (S <= 8 ? 8 : (S <= 12 ? 12 : 16)), Bt = M / A;
    const int smem = (2 * M * (TS + 1) + NQt * M + A * A + M + Bt * Bt) * 16;     // C | D | root tables (fft_slab.cuh)
    const int per = count >= 2048 ? 8 : (count >= 1024 ? 4 : 1);     // few fields per CTA: the read-modify-writes of many short CTAs overlap better than
                                               // a long walk; a few amortise the index map and the root tables (cfg 5: 1 / 4 / 8 / 16 fields: 245 / 224 / 220 / 218 ms)
    const dim3 grid(groups, (count + per - 1) / per);
    const bool small = TS * M <= 512;
    auto kern = BSE_SLAB_PICK(fwd_stick_slab_kernel);
    kern<<<grid, TS * M, smem, s>>>(P, pl.n, S, M, A, Zs, X, pl.npw_h, scale, slab, accumulate ? 1 : 0, rc_rows, row_ld, row0,
                                    count, per, bsefft::slab_const(pl.n, M, A));
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}
int bse_launch_fwd_stick(const FftPlan &pl, const double2 *Z, int count, double2 *X, const double *scale,
                         cudaStream_t s, const int *scatter) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->fwd_stick(to_dev(pl), Z, count, X, pl.npw_h, scale, s, scatter);
}
int bse_launch_inv_stick(const FftPlan &pl, const double2 *T, int count, double2 *Z, cudaStream_t s,
                         const int *gather, int g0, const float2 *T32) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->inv_stick(to_dev(pl), T, count, pl.npw_h, Z, s, gather, g0, T32);
}
