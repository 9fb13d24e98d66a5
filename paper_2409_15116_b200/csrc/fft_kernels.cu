// Batched, pruned 3-D FFT kernels (fp64) for the pair-density -> PW_h and PW_h -> real-space transforms.
//
// Steps a2, a3, a4 and a9 of SURVEY.md 8(a) ("FFTs within a band group"; eq. 6/9/10):
//   forward:  rho_p(r) = u_v(r) u_w(r)  --plane pass-->  Z[p][i1][stick]  --stick pass-->  x_p(G) on H
//   inverse:  tau_p(G) on H  --stick pass-->  Z[p][i1][stick]  --plane pass-->  tau_p(r)
//
// Plane pass: one CTA owns one contiguous n x n plane of fixed i1 in shared memory.  Two real rows are packed
// into one complex line (row 2j -> real part, row 2j+1 -> imaginary part), transformed along i3 with in-place
// radix-{2,3,4,5} decimation-in-frequency passes, untangled in place, and only the columns m3 = 0..R (sphere
// radius) go through the transform along i2; only the (m2, m3) inside the sphere's disk ("sticks") leave the SM.
// Stick pass: a CTA owns a tile of sticks for all i1, transforms along i1, and applies the v_c^{1/2}/N scaling
// while gathering to the half sphere H (forward) or scatters from H (inverse).
// The pair product is fused into the plane pass's load, so rho_p(r) never exists in HBM.
#include "bse_internal.h"

namespace {

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// multiply by s*i  (s = +1 or -1)
__device__ __forceinline__ double2 muli(double2 a, double s) { return make_double2(-s * a.y, s * a.x); }

// One in-place DIF pass of radix r over `nlines` lines living in shared memory.
//   COL = false: element e of line l is C[l*ld + e]
//   COL = true : element e of line l is C[(e>>1)*ld + kk[(e&1)*W + l]]   (columns of the packed plane)
//   sgn = -1 forward (e^{-i...}), +1 inverse.
template <bool COL>
__device__ __forceinline__ void fft_pass(double2 *C, const double2 *tw, const int *kk, int W, int n, int ld,
                                         int nlines, int Lc, int r, double sgn) {
    const int m = Lc / r;
    const int nb = n / r;
    const int tws = n / Lc;
    const int total = nlines * nb;
    for (int w = threadIdx.x; w < total; w += blockDim.x) {
        const int line = w % nlines;
        const int b = w / nlines;
        const int blk = b / m;
        const int j = b - blk * m;
        const int base = blk * Lc + j;
        int off[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            if (q < r) {
                const int e = base + q * m;
                off[q] = COL ? ((e >> 1) * ld + kk[(e & 1) * W + line]) : (line * ld + e);
            }
        }
        double2 y0, y1, y2, y3, y4;
        if (r == 4) {
            double2 x0 = C[off[0]], x1 = C[off[1]], x2 = C[off[2]], x3 = C[off[3]];
            double2 a = cadd(x0, x2), bb = csub(x0, x2), c = cadd(x1, x3), d = muli(csub(x1, x3), sgn);
            y0 = cadd(a, c); y2 = csub(a, c); y1 = cadd(bb, d); y3 = csub(bb, d);
        } else if (r == 2) {
            double2 x0 = C[off[0]], x1 = C[off[1]];
            y0 = cadd(x0, x1); y1 = csub(x0, x1);
        } else if (r == 3) {
            double2 x0 = C[off[0]], x1 = C[off[1]], x2 = C[off[2]];
            double2 t1 = cadd(x1, x2);
            double2 t2 = make_double2(x0.x - 0.5 * t1.x, x0.y - 0.5 * t1.y);
            const double s3 = sgn * 0.86602540378443864676;
            double2 d = csub(x1, x2);
            double2 t3 = make_double2(-s3 * d.y, s3 * d.x);   // i * s3 * d
            y0 = cadd(x0, t1); y1 = cadd(t2, t3); y2 = csub(t2, t3);
        } else {  // r == 5
            double2 x0 = C[off[0]], x1 = C[off[1]], x2 = C[off[2]], x3 = C[off[3]], x4 = C[off[4]];
            const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410;
            const double s1 = sgn * 0.95105651629515357212, s2 = sgn * 0.58778525229247312917;
            double2 a1 = cadd(x1, x4), a2 = cadd(x2, x3), b1 = csub(x1, x4), b2 = csub(x2, x3);
            y0 = make_double2(x0.x + a1.x + a2.x, x0.y + a1.y + a2.y);
            double2 p1 = make_double2(x0.x + c1 * a1.x + c2 * a2.x, x0.y + c1 * a1.y + c2 * a2.y);
            double2 p2 = make_double2(x0.x + c2 * a1.x + c1 * a2.x, x0.y + c2 * a1.y + c1 * a2.y);
            double2 q1 = make_double2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
            double2 q2 = make_double2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
            double2 iq1 = make_double2(-q1.y, q1.x), iq2 = make_double2(-q2.y, q2.x);
            y1 = cadd(p1, iq1); y4 = csub(p1, iq1); y2 = cadd(p2, iq2); y3 = csub(p2, iq2);
        }
        // twiddles w_Lc^{j q}: table index j*q*tws < n
        if (m > 1 && j > 0) {
            const int t1 = j * tws;
            double2 w1 = tw[t1]; w1.y *= -sgn;     // table holds e^{-i}, forward uses it as is (sgn=-1)
            y1 = cmul(y1, w1);
            if (r > 2) { double2 w2 = tw[2 * t1]; w2.y *= -sgn; y2 = cmul(y2, w2); }
            if (r > 3) { double2 w3 = tw[3 * t1]; w3.y *= -sgn; y3 = cmul(y3, w3); }
            if (r > 4) { double2 w4 = tw[4 * t1]; w4.y *= -sgn; y4 = cmul(y4, w4); }
        }
        C[off[0]] = y0; C[off[1]] = y1;
        if (r > 2) C[off[2]] = y2;
        if (r > 3) C[off[3]] = y3;
        if (r > 4) C[off[4]] = y4;
    }
}

struct PlanDev {
    int n, ld, npass, W, NS;
    int radix[BSE_MAX_RADIX_PASSES];
    const double2 *tw;
    const int *pos, *rev, *kk_fwd, *kk_inv, *stick_off_fwd, *stick_off_inv, *stick_off_mir, *fmap, *imap;
};

PlanDev to_dev(const FftPlan &pl) {
    PlanDev d;
    d.n = pl.n; d.ld = pl.ld; d.npass = pl.npass; d.W = pl.W; d.NS = pl.NS;
    for (int i = 0; i < BSE_MAX_RADIX_PASSES; ++i) d.radix[i] = pl.radix[i];
    d.tw = pl.tw; d.pos = pl.pos; d.rev = pl.rev; d.kk_fwd = pl.kk_fwd; d.kk_inv = pl.kk_inv;
    d.stick_off_fwd = pl.stick_off_fwd; d.stick_off_inv = pl.stick_off_inv; d.stick_off_mir = pl.stick_off_mir;
    d.fmap = pl.fmap; d.imap = pl.imap;
    return d;
}

// shared memory carve-up of the plane kernels: C[(n/2)*ld] | tw[n] | pos[n] | kk[2W]
__device__ __forceinline__ void carve(unsigned char *smem, int n, int ld, double2 *&C, double2 *&tw, int *&pos,
                                      int *&kk) {
    C = reinterpret_cast<double2 *>(smem);
    tw = C + (size_t)(n / 2) * ld;
    pos = reinterpret_cast<int *>(tw + n);
    kk = pos + n;
}

// ---------------------------------------------------------------------------------------------------------
// forward plane pass.  grid = (n planes, count pairs).  fields: [.][N]; pair (v,w) = pairs[p0+p], or when
// pairs == nullptr the single field p0+p (no product: step a12's forward wrapper).
__global__ void __launch_bounds__(1024, 1)
fwd_plane_kernel(PlanDev P, const double *__restrict__ fields, const int2 *__restrict__ pairs, long long p0,
                 long long N, double2 *__restrict__ Z) {
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C, *tw; int *pos, *kk;
    const int n = P.n, ld = P.ld, W = P.W;
    carve(smem, n, ld, C, tw, pos, kk);
    for (int i = threadIdx.x; i < n; i += blockDim.x) { tw[i] = P.tw[i]; pos[i] = P.pos[i]; }
    for (int i = threadIdx.x; i < 2 * W; i += blockDim.x) kk[i] = P.kk_fwd[i];

    const int i1 = blockIdx.x;
    const long long p = blockIdx.y;
    const double *fv, *fw = nullptr;
    if (pairs) {
        const int2 vw = pairs[p0 + p];
        fv = fields + (long long)vw.x * N + (long long)i1 * n * n;
        fw = fields + (long long)vw.y * N + (long long)i1 * n * n;
    } else {
        fv = fields + (p0 + p) * N + (long long)i1 * n * n;
    }
    // a2: pair density, packed two rows per complex line
    const int half = n * n / 2;
    for (int idx = threadIdx.x; idx < half; idx += blockDim.x) {
        const int e = 2 * idx;
        const int i2 = e / n, i3 = e - i2 * n;
        double2 a = *reinterpret_cast<const double2 *>(fv + e);
        if (fw) {
            const double2 b = *reinterpret_cast<const double2 *>(fw + e);
            a.x *= b.x; a.y *= b.y;
        }
        double *dst = reinterpret_cast<double *>(&C[(i2 >> 1) * ld + i3]) + (i2 & 1);
        dst[0] = a.x;
        dst[2] = a.y;
    }
    __syncthreads();
    // a3 (i3): n/2 complex lines of length n
    int Lc = n;
    for (int ps = 0; ps < P.npass; ++ps) {
        fft_pass<false>(C, tw, kk, W, n, ld, n / 2, Lc, P.radix[ps], -1.0);
        Lc /= P.radix[ps];
        __syncthreads();
    }
    // untangle rows 2j / 2j+1 for m3 = 0..R, in place: A -> slot pos[k], B -> slot pos[n-k] (k=0: pos[n/2])
    const int nl = n / 2;
    for (int idx = threadIdx.x; idx < nl * W; idx += blockDim.x) {
        const int j = idx % nl, k = idx / nl;
        if (k == 0) {
            const double2 z = C[j * ld + pos[0]];
            C[j * ld + pos[0]] = make_double2(z.x, 0.0);
            C[j * ld + pos[n / 2]] = make_double2(z.y, 0.0);
        } else {
            const int oa = j * ld + pos[k], ob = j * ld + pos[n - k];
            const double2 a = C[oa], b = C[ob];
            C[oa] = make_double2(0.5 * (a.x + b.x), 0.5 * (a.y - b.y));
            C[ob] = make_double2(0.5 * (a.y + b.y), -0.5 * (a.x - b.x));
        }
    }
    __syncthreads();
    // a3 (i2): W columns of length n
    Lc = n;
    for (int ps = 0; ps < P.npass; ++ps) {
        fft_pass<true>(C, tw, kk, W, n, ld, W, Lc, P.radix[ps], -1.0);
        Lc /= P.radix[ps];
        __syncthreads();
    }
    double2 *z = Z + (p * n + i1) * (long long)P.NS;
    for (int s = threadIdx.x; s < P.NS; s += blockDim.x) z[s] = C[P.stick_off_fwd[s]];
}

// ---------------------------------------------------------------------------------------------------------
// inverse plane pass.  grid = (n planes, count).  Z[p][i1][NS] -> out[p][N] real.
__global__ void __launch_bounds__(1024, 1)
inv_plane_kernel(PlanDev P, const double2 *__restrict__ Z, long long N, double *__restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C, *tw; int *pos, *kk;
    const int n = P.n, ld = P.ld, W = P.W;
    carve(smem, n, ld, C, tw, pos, kk);
    for (int i = threadIdx.x; i < n; i += blockDim.x) { tw[i] = P.tw[i]; pos[i] = P.pos[i]; }
    for (int i = threadIdx.x; i < 2 * W; i += blockDim.x) kk[i] = P.kk_inv[i];
    const int i1 = blockIdx.x;
    const long long p = blockIdx.y;
    const int nl = n / 2;
    for (int i = threadIdx.x; i < nl * ld; i += blockDim.x) C[i] = make_double2(0.0, 0.0);
    __syncthreads();
    const double2 *z = Z + (p * n + i1) * (long long)P.NS;
    for (int s = threadIdx.x; s < P.NS; s += blockDim.x) {
        const double2 v = z[s];
        C[P.stick_off_inv[s]] = v;
        const int mo = P.stick_off_mir[s];
        if (mo >= 0) C[mo] = make_double2(v.x, -v.y);
    }
    __syncthreads();
    int Lc = n;
    for (int ps = 0; ps < P.npass; ++ps) {
        fft_pass<true>(C, tw, kk, W, n, ld, W, Lc, P.radix[ps], +1.0);
        Lc /= P.radix[ps];
        __syncthreads();
    }
    // tangle: Z_j[k] = Ga[k] + i Gb[k], Z_j[n-k] = conj(Ga[k]) + i conj(Gb[k]);  Ga at slot k, Gb at slot n-k
    for (int idx = threadIdx.x; idx < nl * W; idx += blockDim.x) {
        const int j = idx % nl, k = idx / nl;
        if (k == 0) {
            const double2 a = C[j * ld], b = C[j * ld + n / 2];
            C[j * ld] = make_double2(a.x, b.x);
            C[j * ld + n / 2] = make_double2(0.0, 0.0);
        } else {
            const int oa = j * ld + k, ob = j * ld + n - k;
            const double2 a = C[oa], b = C[ob];
            C[oa] = make_double2(a.x - b.y, a.y + b.x);
            C[ob] = make_double2(a.x + b.y, b.x - a.y);
        }
    }
    __syncthreads();
    Lc = n;
    for (int ps = 0; ps < P.npass; ++ps) {
        fft_pass<false>(C, tw, kk, W, n, ld, nl, Lc, P.radix[ps], +1.0);
        Lc /= P.radix[ps];
        __syncthreads();
    }
    double *o = out + p * N + (long long)i1 * n * n;
    const int half = n * n / 2;
    for (int idx = threadIdx.x; idx < half; idx += blockDim.x) {
        const int e = 2 * idx;
        const int i2 = e / n, i3 = e - i2 * n;
        const int t = pos[i2];
        const double *src = reinterpret_cast<const double *>(&C[(t >> 1) * ld]) + (t & 1);
        double2 v;
        v.x = src[2 * pos[i3]];
        v.y = src[2 * pos[i3 + 1]];
        *reinterpret_cast<double2 *>(o + e) = v;
    }
}

// ---------------------------------------------------------------------------------------------------------
// stick passes.  grid = (ceil(NS/TS), count).  smem: C[TS*ld] | tw[n]
constexpr int TS = 16;

__global__ void __launch_bounds__(256)
fwd_stick_kernel(PlanDev P, const double2 *__restrict__ Z, double2 *__restrict__ X, long long npw_h,
                 const double *__restrict__ scale) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int n = P.n, ld = P.ld, NS = P.NS;
    double2 *C = reinterpret_cast<double2 *>(smem);
    double2 *tw = C + TS * ld;
    for (int i = threadIdx.x; i < n; i += blockDim.x) tw[i] = P.tw[i];
    const int s0 = blockIdx.x * TS;
    const int ns = min(TS, NS - s0);
    const long long p = blockIdx.y;
    const double2 *z = Z + p * n * (long long)NS;
    for (int w = threadIdx.x; w < TS * n; w += blockDim.x) {
        const int s = w % TS, t = w / TS;
        C[s * ld + t] = (s < ns) ? z[(long long)t * NS + s0 + s] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    int Lc = n;
    for (int ps = 0; ps < P.npass; ++ps) {
        fft_pass<false>(C, tw, nullptr, 0, n, ld, TS, Lc, P.radix[ps], -1.0);
        Lc /= P.radix[ps];
        __syncthreads();
    }
    // a4: x(G) = v_c^{1/2}(G) rho(G) (1/N folded into scale), gathered to H
    double2 *x = X + p * npw_h;
    for (int w = threadIdx.x; w < ns * n; w += blockDim.x) {
        const int s = w % ns, t = w / ns;
        const int hh = P.fmap[(long long)(s0 + s) * n + t];
        if (hh >= 0) {
            const double sc = scale[hh];
            const double2 v = C[s * ld + t];
            x[hh] = make_double2(v.x * sc, v.y * sc);
        }
    }
}

__global__ void __launch_bounds__(256)
inv_stick_kernel(PlanDev P, const double2 *__restrict__ T, long long npw_h, double2 *__restrict__ Z) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int n = P.n, ld = P.ld, NS = P.NS;
    double2 *C = reinterpret_cast<double2 *>(smem);
    double2 *tw = C + TS * ld;
    for (int i = threadIdx.x; i < n; i += blockDim.x) tw[i] = P.tw[i];
    const int s0 = blockIdx.x * TS;
    const int ns = min(TS, NS - s0);
    const long long p = blockIdx.y;
    const double2 *tg = T + p * npw_h;
    for (int w = threadIdx.x; w < TS * n; w += blockDim.x) {
        const int s = w % TS, t = w / TS;
        double2 v = make_double2(0.0, 0.0);
        if (s < ns) {
            const int code = P.imap[(long long)(s0 + s) * n + t];
            if (code >= 0) v = tg[code];
            else if (code <= -2) { v = tg[-2 - code]; v.y = -v.y; }
        }
        C[s * ld + t] = v;
    }
    __syncthreads();
    int Lc = n;
    for (int ps = 0; ps < P.npass; ++ps) {
        fft_pass<false>(C, tw, nullptr, 0, n, ld, TS, Lc, P.radix[ps], +1.0);
        Lc /= P.radix[ps];
        __syncthreads();
    }
    double2 *z = Z + p * n * (long long)NS;
    for (int w = threadIdx.x; w < ns * n; w += blockDim.x) {
        const int s = w % ns, t = w / ns;
        z[(long long)P.rev[t] * NS + s0 + s] = C[s * ld + t];
    }
}

int plane_threads(int n) { return n <= 32 ? 128 : (n <= 64 ? 256 : (n <= 96 ? 512 : 1024)); }

}  // namespace

int bse_fft_smem_bytes_plane(const FftPlan &pl) {
    return (pl.n / 2) * pl.ld * 16 + pl.n * 16 + pl.n * 4 + 2 * pl.W * 4 + 16;
}

static int set_smem(const void *fn, int bytes) {
    if (bytes > 48 * 1024) BSE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    return BSE_OK;
}

int bse_launch_fwd_plane(const FftPlan &pl, const double *fields, const int2 *pairs, long long p0, int count,
                         long long N, double2 *Z, cudaStream_t s) {
    if (count <= 0) return BSE_OK;
    const int smem = bse_fft_smem_bytes_plane(pl);
    int rc = set_smem((const void *)fwd_plane_kernel, smem);
    if (rc) return rc;
    for (int c0 = 0; c0 < count; c0 += 65535) {
        const int c = count - c0 < 65535 ? count - c0 : 65535;
        fwd_plane_kernel<<<dim3(pl.n, c), plane_threads(pl.n), smem, s>>>(
            to_dev(pl), fields, pairs, p0 + c0, N, Z + (long long)c0 * pl.n * pl.NS);
    }
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_inv_plane(const FftPlan &pl, const double2 *Z, int count, long long N, double *out, cudaStream_t s) {
    if (count <= 0) return BSE_OK;
    const int smem = bse_fft_smem_bytes_plane(pl);
    int rc = set_smem((const void *)inv_plane_kernel, smem);
    if (rc) return rc;
    for (int c0 = 0; c0 < count; c0 += 65535) {
        const int c = count - c0 < 65535 ? count - c0 : 65535;
        inv_plane_kernel<<<dim3(pl.n, c), plane_threads(pl.n), smem, s>>>(
            to_dev(pl), Z + (long long)c0 * pl.n * pl.NS, N, out + (long long)c0 * N);
    }
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_fwd_stick(const FftPlan &pl, const double2 *Z, int count, double2 *X, const double *scale,
                         cudaStream_t s) {
    if (count <= 0) return BSE_OK;
    const int smem = TS * pl.ld * 16 + pl.n * 16;
    for (int c0 = 0; c0 < count; c0 += 65535) {
        const int c = count - c0 < 65535 ? count - c0 : 65535;
        fwd_stick_kernel<<<dim3((pl.NS + TS - 1) / TS, c), 256, smem, s>>>(
            to_dev(pl), Z + (long long)c0 * pl.n * pl.NS, X + (long long)c0 * pl.npw_h, pl.npw_h, scale);
    }
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_inv_stick(const FftPlan &pl, const double2 *T, int count, double2 *Z, cudaStream_t s) {
    if (count <= 0) return BSE_OK;
    const int smem = TS * pl.ld * 16 + pl.n * 16;
    for (int c0 = 0; c0 < count; c0 += 65535) {
        const int c = count - c0 < 65535 ? count - c0 : 65535;
        inv_stick_kernel<<<dim3((pl.NS + TS - 1) / TS, c), 256, smem, s>>>(
            to_dev(pl), T + (long long)c0 * pl.npw_h, pl.npw_h, Z + (long long)c0 * pl.n * pl.NS);
    }
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}
