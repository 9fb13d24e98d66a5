// Size dispatch of the two-pass FFT kernels (fft_kernels.cuh).  Each supported grid edge n = R1 * R2 is instantiated in
// one of the fft_sizes_*.cu translation units (compiled in parallel); this file holds the table and the launch wrappers.
#include "fft_kernels.cuh"

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
int bse_launch_inv_stick_slab(const FftPlan &pl, const double2 *T, int count, double2 *Zs, cudaStream_t s, int slab,
                              const int *gather, int g0) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->inv_stick_slab(to_dev(pl), T, count, pl.npw_h, Zs, s, gather, g0, slab);
}
int bse_launch_fwd_stick_slab(const FftPlan &pl, const double2 *Zs, int count, double2 *X, const double *scale, cudaStream_t s,
                              int slab, bool accumulate, int rc, long long row_ld, long long row0) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->fwd_stick_slab(to_dev(pl), Zs, count, X, pl.npw_h, scale, s, slab, accumulate ? 1 : 0, rc,
                                                    row_ld, row0);
}
int bse_launch_fwd_stick(const FftPlan &pl, const double2 *Z, int count, double2 *X, const double *scale,
                         cudaStream_t s, const int *scatter) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->fwd_stick(to_dev(pl), Z, count, X, pl.npw_h, scale, s, scatter);
}
int bse_launch_inv_stick(const FftPlan &pl, const double2 *T, int count, double2 *Z, cudaStream_t s,
                         const int *gather, int g0) {
    if (count <= 0) return BSE_OK;
    return ((const FftOps *)pl.ops)->inv_stick(to_dev(pl), T, count, pl.npw_h, Z, s, gather, g0);
}
