// Batched, pruned 3-D FFT kernels (fp64), templated on the two-pass factorisation n = R1 * R2 (R2 even).
//
// Steps a2, a3, a4, a9 (and the a12 wrappers) of SURVEY.md 8(a)  ("FFTs within a band group"; eq. 6/9/10):
//   forward:  rho_p(r) = u_v(r) u_w(r)  --plane pass-->  Z[p][i1][stick]  --stick pass-->  x_p(G) on H
//   inverse:  tau_p(G) on H  --stick pass-->  Z[p][i1][stick]  --plane pass-->  tau_p(r)
//
// Every 1-D transform of length n is two in-place decimation-in-frequency passes whose butterflies (sizes R1, R2 <= 16)
// live in registers (fft_codelets.cuh), so a line crosses shared memory twice:
//   pass 1: thread (line, j)   takes elements e = j + q R2 (q < R1), R1-point DFT, times w_n^{jq}, back to the same places
//   pass 2: thread (line, blk) takes elements e = blk R2 + q (q < R2), R2-point DFT; place blk R2 + k2 then holds
//           frequency blk + R1 k2.
// Logical element e of a line sits at shared-memory slot natslot(e) = (e / R2) (R2+1) + e % R2 (odd group stride: the
// strided accesses of pass 2 and of the column passes are bank-conflict free).
//
// Plane pass (one CTA = one n x n plane of fixed i1, two real rows packed per complex line):
//   forward  P1 rows pass 1 straight from global memory (pair product fused: rho never exists in HBM)
//            P2 rows pass 2, only frequencies |m3| <= R are written back
//            P3 columns pass 1 with the two-row untangling fused into its load (columns m3 = 0..R only)
//            P4 columns pass 2 straight to global memory: only the (m2, m3) sticks inside the sphere's disk leave the SM
//   inverse  I1 columns pass 1 straight from the sticks in global memory, I2 columns pass 2 + tangling of row pairs,
//            I3 rows pass 1 (zero padding by predicate), I4 rows pass 2 straight to global memory.
// Stick pass (one CTA = TS sticks of one pair, all i1): S1 from global, S2 to global with the v_c^{1/2}/N scaling and the
// gather to the half sphere H (forward) / scatter from H (inverse) fused.
#pragma once
#include <cstdint>

#include "bse_internal.h"
#include "fft_codelets.cuh"

namespace bsefft {

struct PlanDev {
    int R, W, NS;
    int np;                 // planes per field handled by the plane kernels: n (whole fields) or R2 (one slab, see below)
    const double2 *tw;      // [n] exp(-2 pi i t / n)
    const int *soff;        // [n] stick index of (t2, m3) is soff[t2] + m3
    const int *wmax;        // [n] largest m3 of a stick at t2 = m2 mod n, -1 if none
    const int *wmin;        // [n] smallest m3 stored (1 for m2 < 0: the (m2<0, m3=0) sticks are mirrors)
    const int *hmapT;       // [n][NS] (t1 = m1 mod n, stick) -> h in H, -1 outside the sphere, -2-h: conj of entry h
    int pipe;               // plane passes: -1 automatic, 0 the one-plane-per-CTA kernels, 1 the pipelined kernels (fft_pipe.cuh)
    int pipe_lc;            // > 0: at most this many packed lines per slab of the pipelined kernels (test knob)
    int magicW;             // 2^20 / W + 1: task / W == (task * magicW) >> 20 for task < 4096, W <= 160 (no integer division)
};

// coefficient h of a field kept in double (t) or, when t32 != nullptr, in single precision
__device__ __forceinline__ double2 ldcoef(const double2 *t, const float2 *t32, int h) {
    if (t32) { const float2 f = t32[h]; return make_double2((double)f.x, (double)f.y); }
    return t[h];
}

template <int R1, int R2>
struct Geo {
    static constexpr int n = R1 * R2;
    static constexpr int R2p = R2 + 1;
    static constexpr int LD = R1 * R2p + ((R2 % 8) ? ((R2 - R1 * R2p) % 8 + 8) % 8 : 0);   // plane line stride (complex)
    static constexpr int LDS = (R1 * R2p) | 1;                                            // stick line stride
    static constexpr int LDC = (R1 * R2p) | 1;                                            // compact column stride
    static constexpr int TS = 32;                                                          // sticks per CTA
    static __host__ __device__ constexpr int natslot(int e) { return (e / R2) * R2p + e % R2; }
    static __host__ __device__ constexpr int fwdslot(int k) { return (k % R1) * R2p + k / R1; }
    static constexpr int plane_smem = (n / 2) * LD * 16 + n * 16 + 3 * n * 4;
    // plane kernels: as many CTAs per SM as shared memory allows (they are the only overlap of one plane's load / store
    // phases with another's butterflies), and per CTA the threads that leave each of them >= ~112 registers
    static constexpr int plane_tasks = (n / 2) * R2;
    static constexpr int smem_ctas = 232448 / (plane_smem + 1024) < 1 ? 1 : 232448 / (plane_smem + 1024);
    static constexpr int thr_cap0 = 65536 / (100 * (smem_ctas > 6 ? 6 : smem_ctas)) / 32 * 32;
    static constexpr int thr_cap = thr_cap0 > 512 ? 512 : (thr_cap0 < 64 ? 64 : thr_cap0);
    static constexpr int plane_iters = (plane_tasks + thr_cap - 1) / thr_cap;
    static constexpr int plane_thr = (((plane_tasks + plane_iters - 1) / plane_iters + 31) / 32 * 32) < 64
                                         ? 64 : ((plane_tasks + plane_iters - 1) / plane_iters + 31) / 32 * 32;
    static constexpr int reg_ctas = 65536 / (plane_thr * 100);          // keep >= 100 registers per thread
    static constexpr int plane_minb = smem_ctas < reg_ctas ? (smem_ctas < 1 ? 1 : smem_ctas) : (reg_ctas < 1 ? 1 : reg_ctas);
    static constexpr int stick_smem = TS * LDS * 16;
};

// shared memory carve-up of the plane kernels: C[(n/2)*LD] | tw[n] | soff[n] | wmax[n] | wmin[n]
template <int R1, int R2>
__device__ __forceinline__ void plane_tables(unsigned char *smem, const PlanDev &P, double2 *&C, double2 *&tw,
                                             int *&soff, int *&wmax, int *&wmin) {
    using G = Geo<R1, R2>;
    constexpr int n = G::n;
    C = reinterpret_cast<double2 *>(smem);
    tw = C + (size_t)(n / 2) * G::LD;
    soff = reinterpret_cast<int *>(tw + n);
    wmax = soff + n;
    wmin = wmax + n;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        tw[i] = P.tw[i]; soff[i] = P.soff[i]; wmax[i] = P.wmax[i]; wmin[i] = P.wmin[i];
    }
}

// ---------------------------------------------------------------------------------------------------------
// forward plane pass.  grid = (n planes, count).  fields: [.][N]; pair (v,w) = pairs[p0+p], or when pairs == nullptr
// the single field p0+p (no product: forward wrapper of the PW layout, step a12).
// Output carries a factor 2 (the 1/2 of the two-row untangling is folded into the stick pass's scale).
template <int R1, int R2>
__global__ void __launch_bounds__(Geo<R1, R2>::plane_thr, Geo<R1, R2>::plane_minb)
fwd_plane_kernel(PlanDev P, const double *__restrict__ fields, const int2 *__restrict__ pairs, long long p0,
                 long long N, double2 *__restrict__ Z) {
    using G = Geo<R1, R2>;
    constexpr int n = G::n, LD = G::LD, R2p = G::R2p;
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C, *tw; int *soff, *wmax, *wmin;
    plane_tables<R1, R2>(smem, P, C, tw, soff, wmax, wmin);
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
    __syncthreads();
    // P1 (a2 + rows pass 1)
    for (int task = threadIdx.x; task < (n / 2) * R2; task += blockDim.x) {
        const int l = task / R2, j = task - l * R2;
        const double *ra = fv + (2 * l) * n + j, *rb = ra + n;
        double2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) x[q] = make_double2(ra[q * R2], rb[q * R2]);
        if (fw) {
            const double *wa = fw + (2 * l) * n + j, *wb = wa + n;
#pragma unroll
            for (int q = 0; q < R1; ++q) { x[q].x *= wa[q * R2]; x[q].y *= wb[q * R2]; }
        }
        Dft<R1, -1>::run(x);
        twiddle_powers<R1>(x, tw[j]);
#pragma unroll
        for (int q = 0; q < R1; ++q) C[l * LD + q * R2p + j] = x[q];
    }
    __syncthreads();
    // P2 (rows pass 2): frequency k = blk + R1 k2 lands in slot blk R2p + k2 = fwdslot(k)
    const int R = P.R, W = P.W;
    for (int task = threadIdx.x; task < (n / 2) * R1; task += blockDim.x) {
        const int l = task / R1, blk = task - l * R1;
        double2 *c = C + l * LD + blk * R2p;
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = c[q];
        Dft<R2, -1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            const int k = blk + R1 * k2;
            if (k <= R || k >= n - R) c[k2] = x[k2];
        }
    }
    __syncthreads();
    // P3 (untangle rows 2l / 2l+1 + columns pass 1), columns m3 = 0..R; two DFTs per thread (rows j = 2jp, 2jp+1)
    for (int task = threadIdx.x; task < W * (R2 / 2); task += blockDim.x) {
        const int jp = task / W, m3 = task - jp * W;
        const int sa = G::fwdslot(m3), sb = G::fwdslot(m3 ? n - m3 : n / 2);
        double2 xa[R1], xb[R1];
        const int sbr = m3 ? sb : sa;          // m3 = 0: with zb := za the formulas below give (2 za.x, 0) and (2 za.y, 0): no branch
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int l = jp + q * (R2 / 2);
            const double2 za = C[l * LD + sa], zb = C[l * LD + sbr];
            xa[q] = make_double2(za.x + zb.x, za.y - zb.y);           // za + conj(zb)      = 2 A[m3]
            xb[q] = make_double2(za.y + zb.y, zb.x - za.x);           // (za - conj(zb))/i  = 2 B[m3]
        }
        Dft<R1, -1>::run(xa);
        Dft<R1, -1>::run(xb);
        twiddle_powers<R1>(xa, tw[2 * jp]);
        twiddle_powers<R1>(xb, tw[2 * jp + 1]);
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int l = jp + q * (R2 / 2);
            C[l * LD + sa] = xa[q];
            C[l * LD + sb] = xb[q];
        }
    }
    __syncthreads();
    // P4 (columns pass 2): only sticks inside the disk leave the SM
    double2 *z = Z + (p * P.np + i1) * (long long)P.NS;
    for (int task = threadIdx.x; task < W * R1; task += blockDim.x) {
        const int blk = task / W, m3 = task - blk * W;
        const int sa = G::fwdslot(m3), sb = G::fwdslot(m3 ? n - m3 : n / 2);
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = C[(blk * (R2 / 2) + (q >> 1)) * LD + ((q & 1) ? sb : sa)];
        Dft<R2, -1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            const int t2 = blk + R1 * k2;
            if (m3 <= wmax[t2] && m3 >= wmin[t2]) z[soff[t2] + m3] = x[k2];
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// inverse plane pass.  grid = (n planes, count).  Z[p][i1][NS] -> out[p][N] real.
template <int R1, int R2, bool SUB>
__global__ void __launch_bounds__(Geo<R1, R2>::plane_thr, Geo<R1, R2>::plane_minb)
inv_plane_kernel(PlanDev P, const double2 *__restrict__ Z, long long N, double *__restrict__ out) {
    using G = Geo<R1, R2>;
    constexpr int n = G::n, LD = G::LD, R2p = G::R2p;
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C, *tw; int *soff, *wmax, *wmin;
    plane_tables<R1, R2>(smem, P, C, tw, soff, wmax, wmin);
    const int i1 = blockIdx.x;
    const long long p = blockIdx.y;
    const int R = P.R, W = P.W;
    const double2 *z = Z + (p * P.np + i1) * (long long)P.NS;
    __syncthreads();
    // I1 (columns pass 1 from the sticks; (m2<0, m3=0) is the conjugate of (-m2, 0))
    for (int task = threadIdx.x; task < W * R2; task += blockDim.x) {
        const int j = task / W, m3 = task - j * W;
        const int na = G::natslot(m3), nb = G::natslot(m3 ? n - m3 : n / 2);
        double2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int t2 = j + q * R2;
            double2 v = make_double2(0.0, 0.0);
            if (m3 <= wmax[t2]) {
                if (m3 >= wmin[t2]) v = z[soff[t2] + m3];
                else { v = z[soff[n - t2]]; v.y = -v.y; }
            }
            x[q] = v;
        }
        Dft<R1, +1>::run(x);
        twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int e = j + q * R2;
            C[(e >> 1) * LD + ((e & 1) ? nb : na)] = x[q];
        }
    }
    __syncthreads();
    // I2 (columns pass 2 + tangle): Z_l[k] = A[k] + i B[k], Z_l[n-k] = conj(A[k]) + i conj(B[k])
    for (int task = threadIdx.x; task < W * R1; task += blockDim.x) {
        const int blk = task / W, m3 = task - blk * W;
        const int na = G::natslot(m3), nb = G::natslot(m3 ? n - m3 : n / 2);
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = C[(blk * (R2 / 2) + (q >> 1)) * LD + ((q & 1) ? nb : na)];
        Dft<R2, +1>::run(x);
#pragma unroll
        for (int t = 0; t < R2 / 2; ++t) {
            const double2 a = x[2 * t], b = x[2 * t + 1];
            double2 *c = C + (blk * (R2 / 2) + t) * LD;
            if (m3 == 0) {
                c[na] = make_double2(a.x, b.x);
            } else {
                c[na] = make_double2(a.x - b.y, a.y + b.x);
                c[nb] = make_double2(a.x + b.y, b.x - a.y);
            }
        }
    }
    __syncthreads();
    // I3 (rows pass 1; frequencies outside |m3| <= R are zero by predicate, never read)
    for (int task = threadIdx.x; task < (n / 2) * R2; task += blockDim.x) {
        const int l = task / R2, j = task - l * R2;
        double2 *c = C + l * LD + j;
        double2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int e = j + q * R2;
            x[q] = (e <= R || e >= n - R) ? c[q * R2p] : make_double2(0.0, 0.0);
        }
        Dft<R1, +1>::run(x);
        twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
        for (int q = 0; q < R1; ++q) c[q * R2p] = x[q];
    }
    __syncthreads();
    // I4 (rows pass 2 to global): line l packs the rows held at column places 2l, 2l+1 (place p holds row p/R2 + R1 (p%R2))
    double *o = out + p * N + (long long)i1 * n * n;
    for (int task = threadIdx.x; task < (n / 2) * R1; task += blockDim.x) {
        const int l = task / R1, blk = task - l * R1;
        const double2 *c = C + l * LD + blk * R2p;
        const int pa = 2 * l, pb = 2 * l + 1;
        double *oa = o + (pa / R2 + R1 * (pa % R2)) * n + blk;
        double *ob = o + (pb / R2 + R1 * (pb % R2)) * n + blk;
        double olda[SUB ? R2 : 1], oldb[SUB ? R2 : 1];
        if (SUB) {                             // out <- out - transform (P_c update): the old values are fetched before the
#pragma unroll                                 // butterfly so that their latency hides behind it
            for (int k2 = 0; k2 < R2; ++k2) { olda[k2] = oa[R1 * k2]; oldb[k2] = ob[R1 * k2]; }
        }
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = c[q];
        Dft<R2, +1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            if (SUB) { oa[R1 * k2] = olda[k2] - x[k2].x; ob[R1 * k2] = oldb[k2] - x[k2].y; }
            else { oa[R1 * k2] = x[k2].x; ob[R1 * k2] = x[k2].y; }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// inverse plane pass, COMPACT form for large planes.  The full-plane kernel above keeps n/2 lines of n complex in shared
// memory (n^2 * 8 B: 115 KB at n = 120, 166 KB at 144), so one CTA per SM and every global phase exposed.  Only the W = R+1
// columns m3 <= R carry data until the rows pass expands them, so this form keeps the columns compact, Cc[W][LDC], runs the
// two column passes there, and expands LC lines at a time through a small line buffer Wk[LC][LD] (rows pass 1 with the
// two-row tangle fused into its load, rows pass 2 straight to global).  82 + 25 KB at n = 120: two CTAs per SM.
// dynamic smem: Cc[W * LDC] | Wk[LC * LD] | tables (tw, soff, wmax, wmin)
template <int R1, int R2, bool SUB>
__global__ void __launch_bounds__(256)
inv_plane_compact_kernel(PlanDev P, const double2 *__restrict__ Z, long long N, double *__restrict__ out, int LC) {
    using G = Geo<R1, R2>;
    constexpr int n = G::n, LD = G::LD, R2p = G::R2p, LDC = G::LDC;
    extern __shared__ __align__(16) unsigned char smem[];
    const int R = P.R, W = P.W;
    double2 *Cc = reinterpret_cast<double2 *>(smem);
    double2 *Wk = Cc + (size_t)W * LDC;
    double2 *tw = Wk + (size_t)LC * LD;
    int *soff = reinterpret_cast<int *>(tw + n);
    int *wmax = soff + n, *wmin = wmax + n;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        tw[i] = P.tw[i]; soff[i] = P.soff[i]; wmax[i] = P.wmax[i]; wmin[i] = P.wmin[i];
    }
    const int i1 = blockIdx.x;
    const long long p = blockIdx.y;
    const double2 *z = Z + (p * P.np + i1) * (long long)P.NS;
    __syncthreads();
    // I1 (columns pass 1 from the sticks): column m3 lives at Cc[m3 * LDC + natslot(i2 index)]
    for (int task = threadIdx.x; task < W * R2; task += blockDim.x) {
        const int j = task / W, m3 = task - j * W;
        double2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int t2 = j + q * R2;
            double2 v = make_double2(0.0, 0.0);
            if (m3 <= wmax[t2]) {
                if (m3 >= wmin[t2]) v = z[soff[t2] + m3];
                else { v = z[soff[n - t2]]; v.y = -v.y; }
            }
            x[q] = v;
        }
        Dft<R1, +1>::run(x);
        twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
        for (int q = 0; q < R1; ++q) Cc[m3 * LDC + q * R2p + j] = x[q];
    }
    __syncthreads();
    // I2 (columns pass 2, in place): slot blk * R2p + k2 then holds row blk + R1 k2 of column m3
    for (int task = threadIdx.x; task < W * R1; task += blockDim.x) {
        const int blk = task / W, m3 = task - blk * W;
        double2 *c = Cc + m3 * LDC + blk * R2p;
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = c[q];
        Dft<R2, +1>::run(x);
#pragma unroll
        for (int q = 0; q < R2; ++q) c[q] = x[q];
    }
    __syncthreads();
    double *o = out + p * N + (long long)i1 * n * n;
    for (int l0 = 0; l0 < n / 2; l0 += LC) {
        const int nl = min(LC, n / 2 - l0);
        // I3 (rows pass 1): line l packs the rows at column places 2l, 2l+1:  Z_l[k] = A[k] + i B[k],
        // Z_l[n-k] = conj(A[k]) + i conj(B[k]); everything outside |m3| <= R is zero
        for (int task = threadIdx.x; task < nl * R2; task += blockDim.x) {
            const int ll = task / R2, j = task - ll * R2;
            const int l = l0 + ll;
            const int sa = G::natslot(2 * l), sb = G::natslot(2 * l + 1);
            double2 x[R1];
#pragma unroll
            for (int q = 0; q < R1; ++q) {
                const int e = j + q * R2;
                double2 v = make_double2(0.0, 0.0);
                if (e <= R) {
                    const double2 a = Cc[e * LDC + sa], b = Cc[e * LDC + sb];
                    v = e ? make_double2(a.x - b.y, a.y + b.x) : make_double2(a.x, b.x);
                } else if (e >= n - R) {
                    const double2 a = Cc[(n - e) * LDC + sa], b = Cc[(n - e) * LDC + sb];
                    v = make_double2(a.x + b.y, b.x - a.y);
                }
                x[q] = v;
            }
            Dft<R1, +1>::run(x);
            twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
            for (int q = 0; q < R1; ++q) Wk[ll * LD + q * R2p + j] = x[q];
        }
        __syncthreads();
        // I4 (rows pass 2 to global): place p holds row p / R2 + R1 (p % R2)
        for (int task = threadIdx.x; task < nl * R1; task += blockDim.x) {
            const int ll = task / R1, blk = task - ll * R1;
            const int l = l0 + ll;
            const double2 *c = Wk + ll * LD + blk * R2p;
            const int pa = 2 * l, pb = 2 * l + 1;
            double *oa = o + (pa / R2 + R1 * (pa % R2)) * n + blk;
            double *ob = o + (pb / R2 + R1 * (pb % R2)) * n + blk;
            double olda[SUB ? R2 : 1], oldb[SUB ? R2 : 1];
            if (SUB) {
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) { olda[k2] = oa[R1 * k2]; oldb[k2] = ob[R1 * k2]; }
            }
            double2 x[R2];
#pragma unroll
            for (int q = 0; q < R2; ++q) x[q] = c[q];
            Dft<R2, +1>::run(x);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                if (SUB) { oa[R1 * k2] = olda[k2] - x[k2].x; ob[R1 * k2] = oldb[k2] - x[k2].y; }
                else { oa[R1 * k2] = x[k2].x; ob[R1 * k2] = x[k2].y; }
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------------------
// stick passes.  grid = (ceil(NS/TS), count), 256 threads.  smem: C[TS*LDS]
template <int R1, int R2>
__global__ void __launch_bounds__(256)
fwd_stick_kernel(PlanDev P, const double2 *__restrict__ Z, double2 *__restrict__ X, long long npw_h,
                 const double *__restrict__ scale, const int *__restrict__ scatter, int s_off) {
    using G = Geo<R1, R2>;
    constexpr int n = G::n, LDS = G::LDS, R2p = G::R2p, TS = G::TS;
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C = reinterpret_cast<double2 *>(smem);
    const double2 *tw = P.tw;                 // read through L1: no table copy, no barrier before the first load
    const int NS = P.NS;
    const int s0 = blockIdx.x * TS;
    const long long p = blockIdx.y;
    const double2 *z = Z + p * n * (long long)NS;
    for (int task = threadIdx.x; task < TS * R2; task += blockDim.x) {
        const int j = task / TS, sl = task - j * TS;
        const int s = s0 + sl;
        if (s >= NS) continue;
        double2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) x[q] = z[(long long)(j + q * R2) * NS + s];
        Dft<R1, -1>::run(x);
        twiddle_powers<R1>(x, tw[j]);
#pragma unroll
        for (int q = 0; q < R1; ++q) C[sl * LDS + q * R2p + j] = x[q];
    }
    __syncthreads();
    // a4: x(G) = scale(G) * rho(G), gathered to H  (scale = v_c^{1/2}/(2N) for tau, 1/(2N) for the PW wrapper)
    double2 *xo = X + (scatter ? (long long)scatter[s_off + p] : p) * npw_h;
    for (int task = threadIdx.x; task < TS * R1; task += blockDim.x) {
        const int blk = task / TS, sl = task - blk * TS;
        const int s = s0 + sl;
        if (s >= NS) continue;
        int hh[R2];                           // the targets on H: fetched before the butterfly, their latency hides behind it
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) hh[k2] = P.hmapT[(blk + R1 * k2) * NS + s];
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = C[sl * LDS + blk * R2p + q];
        Dft<R2, -1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            if (hh[k2] >= 0) {
                const double sc = scale[hh[k2]];
                xo[hh[k2]] = make_double2(x[k2].x * sc, x[k2].y * sc);
            }
        }
    }
}

template <int R1, int R2, bool F32>
__global__ void __launch_bounds__(256)
inv_stick_kernel(PlanDev P, const double2 *__restrict__ T, long long npw_h, double2 *__restrict__ Z,
                 const int *__restrict__ gather, int g0, const float2 *__restrict__ T32) {
    using G = Geo<R1, R2>;
    constexpr int n = G::n, LDS = G::LDS, R2p = G::R2p, TS = G::TS;
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C = reinterpret_cast<double2 *>(smem);
    const double2 *tw = P.tw;                 // read through L1: no table copy, no barrier before the first load
    const int NS = P.NS;
    const int s0 = blockIdx.x * TS;
    const long long p = blockIdx.y;
    // T32 != nullptr: the coefficients are kept in single precision (BSE_TAU_F32) and widened on load
    const long long toff = (gather ? (long long)gather[g0 + p] : p) * npw_h;
    const double2 *tg = T + toff;
    const float2 *tg32 = F32 ? T32 + toff : nullptr;
    for (int task = threadIdx.x; task < TS * R2; task += blockDim.x) {
        const int j = task / TS, sl = task - j * TS;
        const int s = s0 + sl;
        if (s >= NS) continue;
        double2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) {
            const int code = P.hmapT[(j + q * R2) * NS + s];
            double2 v = make_double2(0.0, 0.0);
            if (code >= 0) v = F32 ? ldcoef(tg, tg32, code) : tg[code];
            else if (code <= -2) { v = F32 ? ldcoef(tg, tg32, -2 - code) : tg[-2 - code]; v.y = -v.y; }
            x[q] = v;
        }
        Dft<R1, +1>::run(x);
        twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
        for (int q = 0; q < R1; ++q) C[sl * LDS + q * R2p + j] = x[q];
    }
    __syncthreads();
    double2 *z = Z + p * n * (long long)NS;
    for (int task = threadIdx.x; task < TS * R1; task += blockDim.x) {
        const int blk = task / TS, sl = task - blk * TS;
        const int s = s0 + sl;
        if (s >= NS) continue;
        double2 x[R2];
#pragma unroll
        for (int q = 0; q < R2; ++q) x[q] = C[sl * LDS + blk * R2p + q];
        Dft<R2, +1>::run(x);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) z[(long long)(blk + R1 * k2) * NS + s] = x[k2];
    }
}


}  // namespace bsefft
#include "fft_pipe.cuh"
namespace bsefft {

// ---------------------------------------------------------------------------------------------------------
// host launchers for one factorisation; collected in a table by fft_kernels.cu
struct FftOps {
    int n, R1, R2, plane_smem;
    int (*fwd_plane)(const PlanDev &, const double *, const int2 *, long long, int, long long, double2 *, cudaStream_t);
    int (*inv_plane)(const PlanDev &, const double2 *, int, long long, double *, cudaStream_t, int, int);
    int (*fwd_stick)(const PlanDev &, const double2 *, int, double2 *, long long, const double *, cudaStream_t, const int *);
    int (*inv_stick)(const PlanDev &, const double2 *, int, long long, double2 *, cudaStream_t, const int *, int, const float2 *);
};

inline int plane_threads(int tasks) {
    const int iters = (tasks + 511) / 512;
    const int t = ((tasks + iters - 1) / iters + 31) / 32 * 32;
    return t < 64 ? 64 : t;
}

template <int R1, int R2>
struct Launch {
    using G = Geo<R1, R2>;
    static int set_smem(const void *fn, int bytes, bool plane = false) {
        if (bytes > 48 * 1024) BSE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
        if (plane && bytes >= 64 * 1024)   // large planes: take the whole carve-out so that smem_ctas CTAs fit
            BSE_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        return BSE_OK;
    }
    // ---- pipelined plane passes (fft_pipe.cuh) ----
    using PG = PipeGeo<R1, R2>;
    static constexpr int SMEM_MAX = 232448;                     // opt-in limit of one CTA on sm_100
    // automatic choice (measured): where one full plane fills the SM (n >= 120), the inverse pass
    // (cfg 5: 230 -> 210 ms) and the single-field forward pass (-11 %); the pair-density forward pass stages two fields, which
    // leaves it 9 lines per slab at n = 160 (slower), and on smaller planes the one-plane kernels run more warps per SM
    static bool use_pipe(const PlanDev &P, bool inverse, bool pair) {
        return P.pipe > 0 || (P.pipe < 0 && G::smem_ctas == 1 && (inverse || !pair));
    }
    // lines per slab: as many as fit beside the fixed buffers, at most one rows-pass task per thread, slabs of equal size
    static int pick_lc(int fixed, int per_line, int knob) {
        int lc = (SMEM_MAX - fixed) / per_line;
        const int cap = (PIPE_THREADS + R2 - 1) / R2;
        if (lc > cap) lc = cap;
        if (lc > G::n / 2) lc = G::n / 2;
        if (lc < 2) return 0;
        const int ns = (G::n / 2 + lc - 1) / lc;
        lc = (G::n / 2 + ns - 1) / ns;
        if (knob > 0 && lc > knob) lc = knob;
        return lc;
    }
    static int persistent_grid(const void *kern, int smem, long long total, int *grid) {
        int dev = 0, sms = 0, occ = 0;
        BSE_CUDA(cudaGetDevice(&dev));
        BSE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        BSE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        BSE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        BSE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, PIPE_THREADS, smem));
        if (occ < 1) return BSE_EUNSUPPORTED;
        const long long g = (long long)occ * sms;
        *grid = (int)(total < g ? total : g);
        return BSE_OK;
    }
    static int inv_plane_pipe(const PlanDev &P, const double2 *Z, int count, long long N, double *out, cudaStream_t s) {
        // bulk copies move 16-byte aligned pieces: a caller's buffer at an odd multiple of 8 bytes takes the one-plane kernels
        if ((((uintptr_t)out | (uintptr_t)Z) & 15) || (N & 1)) return BSE_EUNSUPPORTED;
        const int LC = pick_lc(PG::inv_smem(P.W, P.NS, 0), G::LD * 16 + 2 * G::n * 8, P.pipe_lc);
        if (LC < 2) return BSE_EUNSUPPORTED;
        const int smem = PG::inv_smem(P.W, P.NS, LC);
        const long long total = (long long)count * P.np;
        int grid = 0;
        const int rc = persistent_grid((const void *)inv_plane_pipe_kernel<R1, R2>, smem, total, &grid);
        if (rc) return rc;
        inv_plane_pipe_kernel<R1, R2><<<grid, PIPE_THREADS, smem, s>>>(P, Z, N, out, total, LC);
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    static int fwd_plane_pipe(const PlanDev &P, const double *fields, const int2 *pairs, long long p0, int count, long long N,
                              double2 *Z, cudaStream_t s) {
        if (((uintptr_t)fields & 15) || (N & 1)) return BSE_EUNSUPPORTED;      // see inv_plane_pipe
        const int nf = pairs ? 2 : 1, NST = 2;
        const int LC = pick_lc(PG::fwd_smem(P.W, 0, NST, nf), G::LD * 16 + NST * nf * 2 * G::n * 8, P.pipe_lc);
        if (LC < 2) return BSE_EUNSUPPORTED;
        const int smem = PG::fwd_smem(P.W, LC, NST, nf);
        const long long total = (long long)count * P.np;
        int grid = 0;
        const int rc = persistent_grid((const void *)fwd_plane_pipe_kernel<R1, R2>, smem, total, &grid);
        if (rc) return rc;
        fwd_plane_pipe_kernel<R1, R2><<<grid, PIPE_THREADS, smem, s>>>(P, fields, pairs, p0, N, Z, total, LC, NST);
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    static int fwd_plane(const PlanDev &P, const double *fields, const int2 *pairs, long long p0, int count, long long N,
                         double2 *Z, cudaStream_t s) {
        if (use_pipe(P, false, pairs != nullptr)) {
            int rc = fwd_plane_pipe(P, fields, pairs, p0, count, N, Z, s);
            if (rc != BSE_EUNSUPPORTED) return rc;
        }
        int rc = set_smem((const void *)fwd_plane_kernel<R1, R2>, G::plane_smem, true);
        if (rc) return rc;
        const int threads = G::plane_thr;
        for (int c0 = 0; c0 < count; c0 += 65535) {
            const int c = count - c0 < 65535 ? count - c0 : 65535;
            fwd_plane_kernel<R1, R2><<<dim3(P.np, c), threads, G::plane_smem, s>>>(
                P, fields, pairs, p0 + c0, N, Z + (long long)c0 * P.np * P.NS);
        }
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    static int inv_plane(const PlanDev &P, const double2 *Z, int count, long long N, double *out, cudaStream_t s, int sub,
                         int force) {
        if (!sub && force < 0 && use_pipe(P, true, false)) {
            int rc = inv_plane_pipe(P, Z, count, N, out, s);
            if (rc != BSE_EUNSUPPORTED) return rc;
        }
        // large planes (one full-plane CTA per SM): the compact form, if two of its CTAs fit an SM
        // force = k (test / tuning knob of the plan, bse_debug_set): the compact form sized for k CTAs per SM (0: never, -1: auto)
        const int tables = G::n * 16 + 3 * G::n * 4;
        const int per_sm = force > 1 ? force : 2;
        const int share = (232448 - per_sm * 1024) / per_sm;
        int LC = (share - P.W * G::LDC * 16 - tables) / (G::LD * 16);
        if (LC > G::n / 2) LC = G::n / 2;
        const bool fits = LC >= 4;
        const bool use = force >= 0 ? (force != 0 && fits) : (G::smem_ctas == 1 && fits);
        if (use) {
            const int smem_c = (P.W * G::LDC + LC * G::LD) * 16 + tables;
            auto kern = sub ? inv_plane_compact_kernel<R1, R2, true> : inv_plane_compact_kernel<R1, R2, false>;
            int rc = set_smem((const void *)kern, smem_c, true);
            if (rc) return rc;
            int threads = ((LC * R2 + 31) / 32) * 32;
            if (threads > 256) threads = 256;
            if (threads < 64) threads = 64;
            for (int c0 = 0; c0 < count; c0 += 65535) {
                const int c = count - c0 < 65535 ? count - c0 : 65535;
                kern<<<dim3(P.np, c), threads, smem_c, s>>>(P, Z + (long long)c0 * P.np * P.NS, N, out + (long long)c0 * N, LC);
            }
            BSE_CUDA(cudaGetLastError());
            return BSE_OK;
        }
        auto kern = sub ? inv_plane_kernel<R1, R2, true> : inv_plane_kernel<R1, R2, false>;
        int rc = set_smem((const void *)kern, G::plane_smem, true);
        if (rc) return rc;
        const int threads = G::plane_thr;
        for (int c0 = 0; c0 < count; c0 += 65535) {
            const int c = count - c0 < 65535 ? count - c0 : 65535;
            kern<<<dim3(P.np, c), threads, G::plane_smem, s>>>(P, Z + (long long)c0 * P.np * P.NS, N, out + (long long)c0 * N);
        }
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    static int fwd_stick(const PlanDev &P, const double2 *Z, int count, double2 *X, long long npw_h, const double *scale,
                         cudaStream_t s, const int *scatter) {
        int rc = set_smem((const void *)fwd_stick_kernel<R1, R2>, G::stick_smem);
        if (rc) return rc;
        for (int c0 = 0; c0 < count; c0 += 65535) {
            const int c = count - c0 < 65535 ? count - c0 : 65535;
            fwd_stick_kernel<R1, R2><<<dim3((P.NS + G::TS - 1) / G::TS, c), 256, G::stick_smem, s>>>(
                P, Z + (long long)c0 * G::n * P.NS, scatter ? X : X + (long long)c0 * npw_h, npw_h, scale, scatter, c0);
        }
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    static int inv_stick(const PlanDev &P, const double2 *T, int count, long long npw_h, double2 *Z, cudaStream_t s,
                         const int *gather, int g0, const float2 *T32) {
        auto kern = T32 ? inv_stick_kernel<R1, R2, true> : inv_stick_kernel<R1, R2, false>;
        int rc = set_smem((const void *)kern, G::stick_smem);
        if (rc) return rc;
        for (int c0 = 0; c0 < count; c0 += 65535) {
            const int c = count - c0 < 65535 ? count - c0 : 65535;
            kern<<<dim3((P.NS + G::TS - 1) / G::TS, c), 256, G::stick_smem, s>>>(
                P, gather ? T : T + (long long)c0 * npw_h, npw_h, Z + (long long)c0 * G::n * P.NS, gather, g0 + c0,
                (T32 && !gather) ? T32 + (long long)c0 * npw_h : T32);
        }
        BSE_CUDA(cudaGetLastError());
        return BSE_OK;
    }
    static FftOps ops() {
        return FftOps{G::n, R1, R2, G::plane_smem, fwd_plane, inv_plane, fwd_stick, inv_stick};
    }
};

}  // namespace bsefft
