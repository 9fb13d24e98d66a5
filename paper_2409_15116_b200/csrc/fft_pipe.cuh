// Pipelined plane passes: persistent CTAs, bulk-copy (TMA) staging, compact columns.
//
// Same transforms as fwd_plane_kernel / inv_plane_kernel of fft_kernels.cuh (steps a2, a3, a9 and the a12 wrappers of
// SURVEY.md 8(a)), organised so that every byte that crosses HBM moves asynchronously:
//   * a CTA is persistent and walks over (field, plane) items it, it + gridDim.x, ...
//   * inverse: the NS sticks of one plane are ONE contiguous NS*16-byte piece of Z: a single cp.async.bulk
//     (global -> shared, completion on an mbarrier) fetches the NEXT item's sticks while the current one is transformed;
//     the rows pass works on slabs of LC packed lines, its results (2 LC contiguous real rows) are collected in shared
//     memory and leave with one cp.async.bulk (shared -> global) per slab, which drains while the next slab is computed
//   * forward: the 2 LC real rows of a slab are contiguous in the field: one bulk copy per field and slab into a ring
//     of NST stages (the pair's second orbital into the same stage; the product is formed when the rows pass reads
//     them), issued NST slabs ahead - also across items, so the loads keep flowing during the column passes
//   * only the columns |m3| <= R survive the rows pass, so between the rows and the columns passes the plane is kept
//     compact (W columns of n), which is what makes room for the staging buffers at n = 120 ... 160.
// The threads only ever move data between shared memory and registers (the sticks of the forward pass are the
// exception: 16-byte stores in runs of W).  Arithmetic, its order inside a line and the butterflies are those of the
// kernels in fft_kernels.cuh; the results agree to rounding (the two-row packing pairs other rows).
#pragma once
#include <cstdint>

namespace bsefft {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// global -> shared, bytes % 16 == 0, both addresses 16-byte aligned; completion counted on the mbarrier
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// shared -> global, as one bulk group
__device__ __forceinline__ void bulk_store(void *dst, const void *src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src_smem)),
                 "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// generic-proxy writes to shared memory -> visible to the async proxy (before a bulk store reads them)
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

constexpr int PIPE_THREADS = 256;

// shared-memory sizes (bytes) of the pipelined kernels for LC lines per slab; the host launchers and the kernels use
// the same carve-up
template <int R1, int R2>
struct PipeGeo {
    using G = Geo<R1, R2>;
    static constexpr int n = G::n;
    static constexpr int LDL = (n / 2) | 1;                          // forward: column stride of the compact store (lines)
    static constexpr int tables = n * 16 + 3 * n * 4;
    static __host__ __device__ int pad16(int b) { return (b + 15) & ~15; }
    // inverse: Cc[W*LDC] | Wk[LC*LD] | Os[2 LC n] | Zs[NS] | tables | mbar
    // (one extra compact column and one extra stick that stay zero: what the predicates of the one-plane kernels skip is
    // read from there, so the field loop has no divergent branches)
    static __host__ __device__ int inv_smem(int W, int NS, int LC) {
        return (W + 1) * G::LDC * 16 + LC * G::LD * 16 + 2 * LC * n * 8 + (NS + 1) * 16 + pad16(tables) + 16;
    }
    // forward: Cc[2W*LDL] | Wk[LC*LD] | raw[NST][nf][2 LC n] | tables | mbar[NST]
    // (column 2W of the compact store takes the pruned frequencies |m3| > R: the rows pass stores without branching)
    static __host__ __device__ int fwd_smem(int W, int LC, int nst, int nf) {
        return (2 * W + 1) * LDL * 16 + LC * G::LD * 16 + nst * nf * 2 * LC * n * 8 + pad16(tables) + 16 * nst;
    }
};

// ---------------------------------------------------------------------------------------------------------
// inverse plane pass, pipelined.  Z[item][NS] -> out (real planes).  item = p * np + i1.
template <int R1, int R2>
__global__ void __launch_bounds__(PIPE_THREADS)
inv_plane_pipe_kernel(PlanDev P, const double2 *__restrict__ Z, long long N, double *__restrict__ out, long long total,
                      int LC) {
    using G = Geo<R1, R2>;
    using PG = PipeGeo<R1, R2>;
    constexpr int n = G::n, LD = G::LD, R2p = G::R2p, LDC = G::LDC;
    extern __shared__ __align__(16) unsigned char smem[];
    const int R = P.R, W = P.W, NS = P.NS;
    double2 *Cc = reinterpret_cast<double2 *>(smem);                 // [W + 1][LDC], column W stays zero
    double2 *Wk = Cc + (size_t)(W + 1) * LDC;
    double *Os = reinterpret_cast<double *>(Wk + (size_t)LC * LD);
    double2 *Zs = reinterpret_cast<double2 *>(Os + (size_t)2 * LC * n);   // [NS + 1], stick NS stays zero
    double2 *tw = Zs + NS + 1;
    int *soff = reinterpret_cast<int *>(tw + n);
    int *wmax = soff + n, *wmin = wmax + n;
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(reinterpret_cast<unsigned char *>(tw) + PG::pad16(PG::tables));
    const uint32_t bar = smem_u32(mbar);
    const int tid = threadIdx.x;
    for (int i = tid; i < n; i += blockDim.x) {
        tw[i] = P.tw[i]; soff[i] = P.soff[i]; wmax[i] = P.wmax[i]; wmin[i] = P.wmin[i];
    }
    for (int i = tid; i < LDC; i += blockDim.x) Cc[(size_t)W * LDC + i] = make_double2(0.0, 0.0);
    if (tid == 0) { Zs[NS] = make_double2(0.0, 0.0); mbar_init(bar, 1); mbar_fence_init(); }
    __syncthreads();
    long long it = blockIdx.x;
    const uint32_t zbytes = (uint32_t)NS * 16u;
    if (tid == 0 && it < total) { mbar_expect_tx(bar, zbytes); bulk_load(Zs, Z + it * NS, zbytes, bar); }
    uint32_t parity = 0;
    for (; it < total; it += gridDim.x) {
        const long long p = it / P.np;
        const int i1 = (int)(it - p * P.np);
        mbar_wait(bar, parity);
        parity ^= 1u;
        // I1 (columns pass 1 from the staged sticks; (m2<0, m3=0) is the conjugate of (-m2, 0))
        for (int task = tid; task < W * R2; task += blockDim.x) {
            const int j = (task * P.magicW) >> 20, m3 = task - j * W;                  // task / W
            double2 x[R1];
#pragma unroll
            for (int q = 0; q < R1; ++q) {
                const int t2 = j + q * R2;
                const bool in = m3 <= wmax[t2], own = m3 >= wmin[t2];        // own: stored; else the mirror (-m2, 0), conjugated
                const int idx = in ? soff[own ? t2 : n - t2] + (own ? m3 : 0) : NS;     // NS: the zero stick
                double2 v = Zs[idx];
                if (in && !own) v.y = -v.y;
                x[q] = v;
            }
            Dft<R1, +1>::run(x);
            twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
            for (int q = 0; q < R1; ++q) Cc[m3 * LDC + q * R2p + j] = x[q];
        }
        __syncthreads();
        // the stick buffer is free: fetch the next item's sticks behind the rest of this one
        if (tid == 0 && it + gridDim.x < total) {
            mbar_expect_tx(bar, zbytes);
            bulk_load(Zs, Z + (it + gridDim.x) * NS, zbytes, bar);
        }
        // I2 (columns pass 2, in place): slot blk * R2p + k2 = fwdslot(row) then holds row blk + R1 k2 of column m3
        for (int task = tid; task < W * R1; task += blockDim.x) {
            const int blk = (task * P.magicW) >> 20, m3 = task - blk * W;              // task / W
            double2 *c = Cc + m3 * LDC + blk * R2p;
            double2 x[R2];
#pragma unroll
            for (int q = 0; q < R2; ++q) x[q] = c[q];
            Dft<R2, +1>::run(x);
            // column m3 = 0 is the transform of a Hermitian column: real up to rounding; the rows pass uses its real parts
#pragma unroll
            for (int q = 0; q < R2; ++q) c[q] = m3 ? x[q] : make_double2(x[q].x, 0.0);
        }
        __syncthreads();
        double *o = out + p * N + (long long)i1 * n * n;
        for (int l0 = 0; l0 < n / 2; l0 += LC) {
            const int nl = min(LC, n / 2 - l0);
            // I3 (rows pass 1): line l packs rows 2l, 2l+1:  Z_l[k] = A[k] + i B[k], Z_l[n-k] = conj(A[k]) + i conj(B[k])
            for (int task = tid; task < nl * R2; task += blockDim.x) {
                const int ll = task / R2, j = task - ll * R2;
                const int l = l0 + ll;
                const int sa = G::fwdslot(2 * l), sb = G::fwdslot(2 * l + 1);
                double2 x[R1];
#pragma unroll
                for (int q = 0; q < R1; ++q) {
                    const int e = j + q * R2;
                    const bool lo = e <= R;
                    const int col = lo ? e : (e >= n - R ? n - e : W);       // W: the zero column
                    const double sg = lo ? 1.0 : -1.0;
                    const double2 a = Cc[col * LDC + sa], b = Cc[col * LDC + sb];
                    x[q] = make_double2(fma(-sg, b.y, a.x), fma(sg, a.y, b.x));
                }
                Dft<R1, +1>::run(x);
                twiddle_powers<R1>(x, cconj(tw[j]));
#pragma unroll
                for (int q = 0; q < R1; ++q) Wk[ll * LD + q * R2p + j] = x[q];
            }
            if (tid == 0) bulk_wait_read();          // the previous slab's store has finished reading Os
            __syncthreads();
            // I4 (rows pass 2): real rows 2l, 2l+1 collected in Os
            for (int task = tid; task < nl * R1; task += blockDim.x) {
                const int ll = task / R1, blk = task - ll * R1;
                const double2 *c = Wk + ll * LD + blk * R2p;
                double *oa = Os + (2 * ll) * n + blk, *ob = oa + n;
                double2 x[R2];
#pragma unroll
                for (int q = 0; q < R2; ++q) x[q] = c[q];
                Dft<R2, +1>::run(x);
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) { oa[R1 * k2] = x[k2].x; ob[R1 * k2] = x[k2].y; }
            }
            fence_async_smem();
            __syncthreads();
            if (tid == 0) bulk_store(o + (long long)2 * l0 * n, Os, (uint32_t)(2 * nl * n * 8));
        }
    }
    if (tid == 0) bulk_wait_all();
}

// ---------------------------------------------------------------------------------------------------------
// forward plane pass, pipelined.  fields / pairs / p0 / N as fwd_plane_kernel; item = p * np + i1 -> Z[item][NS].
// Output carries the factor 2 of the two-row untangling, as fwd_plane_kernel's.
template <int R1, int R2>
__global__ void __launch_bounds__(PIPE_THREADS)
fwd_plane_pipe_kernel(PlanDev P, const double *__restrict__ fields, const int2 *__restrict__ pairs, long long p0,
                      long long N, double2 *__restrict__ Z, long long total, int LC, int NST) {
    using G = Geo<R1, R2>;
    using PG = PipeGeo<R1, R2>;
    constexpr int n = G::n, LD = G::LD, R2p = G::R2p, LDL = PG::LDL;
    extern __shared__ __align__(16) unsigned char smem[];
    const int R = P.R, W = P.W;
    const int nf = pairs ? 2 : 1;
    double2 *Cc = reinterpret_cast<double2 *>(smem);                 // [2W + 1][LDL]: column m3 and, at W + m3, column n - m3
    double2 *Wk = Cc + (size_t)(2 * W + 1) * LDL;
    double *raw = reinterpret_cast<double *>(Wk + (size_t)LC * LD);
    const int stage_dbl = nf * 2 * LC * n;
    double2 *tw = reinterpret_cast<double2 *>(raw + (size_t)NST * stage_dbl);
    int *soff = reinterpret_cast<int *>(tw + n);
    int *wmax = soff + n, *wmin = wmax + n;
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(reinterpret_cast<unsigned char *>(tw) + PG::pad16(PG::tables));
    const int tid = threadIdx.x;
    for (int i = tid; i < n; i += blockDim.x) {
        tw[i] = P.tw[i]; soff[i] = P.soff[i]; wmax[i] = P.wmax[i]; wmin[i] = P.wmin[i];
    }
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) mbar_init(smem_u32(mbar + 2 * s), 1);
        mbar_fence_init();
    }
    __syncthreads();
    const int ns = (n / 2 + LC - 1) / LC;                            // slabs per item
    // my slabs are numbered g = k * ns + s over my items k = 0, 1, ...; slab g lives in stage g % NST
    const long long my_items = blockIdx.x < total ? (total - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const long long my_slabs = my_items * ns;
    auto issue = [&](long long g) {                                  // thread 0 only
        const long long k = g / ns;
        const int s = (int)(g - k * ns);
        const long long it = blockIdx.x + k * gridDim.x;
        const long long p = it / P.np;
        const int i1 = (int)(it - p * P.np);
        const int l0 = s * LC, nl = min(LC, n / 2 - l0);
        const uint32_t bytes = (uint32_t)(2 * nl * n * 8);
        const int st = (int)(g % NST);
        const uint32_t bar = smem_u32(mbar + 2 * st);
        double *dst = raw + (size_t)st * stage_dbl;
        const long long off = (long long)i1 * n * n + (long long)2 * l0 * n;
        mbar_expect_tx(bar, bytes * nf);
        if (pairs) {
            const int2 vw = pairs[p0 + p];
            bulk_load(dst, fields + (long long)vw.x * N + off, bytes, bar);
            bulk_load(dst + 2 * LC * n, fields + (long long)vw.y * N + off, bytes, bar);
        } else {
            bulk_load(dst, fields + (p0 + p) * N + off, bytes, bar);
        }
    };
    if (tid == 0)
        for (long long g = 0; g < NST && g < my_slabs; ++g) issue(g);
    long long g = 0;
    for (long long it = blockIdx.x; it < total; it += gridDim.x) {
        for (int l0 = 0; l0 < n / 2; l0 += LC, ++g) {
            const int nl = min(LC, n / 2 - l0);
            const int st = (int)(g % NST);
            mbar_wait(smem_u32(mbar + 2 * st), (uint32_t)((g / NST) & 1));
            const double *rv = raw + (size_t)st * stage_dbl, *rw = rv + 2 * LC * n;
            // P1 (a2 + rows pass 1) from the staged rows
            for (int task = tid; task < nl * R2; task += blockDim.x) {
                const int ll = task / R2, j = task - ll * R2;
                const double *ra = rv + (2 * ll) * n + j, *rb = ra + n;
                double2 x[R1];
#pragma unroll
                for (int q = 0; q < R1; ++q) x[q] = make_double2(ra[q * R2], rb[q * R2]);
                if (nf == 2) {
                    const double *wa = rw + (2 * ll) * n + j, *wb = wa + n;
#pragma unroll
                    for (int q = 0; q < R1; ++q) { x[q].x *= wa[q * R2]; x[q].y *= wb[q * R2]; }
                }
                Dft<R1, -1>::run(x);
                twiddle_powers<R1>(x, tw[j]);
#pragma unroll
                for (int q = 0; q < R1; ++q) Wk[ll * LD + q * R2p + j] = x[q];
            }
            __syncthreads();
            // the stage is free: fetch the slab NST ahead (possibly of a later item) into it
            if (tid == 0 && g + NST < my_slabs) issue(g + NST);
            // P2 (rows pass 2): frequencies |m3| <= R go to the compact store, line l of column m3 / W + (n - m3)
            for (int task = tid; task < nl * R1; task += blockDim.x) {
                const int ll = task / R1, blk = task - ll * R1;
                const double2 *c = Wk + ll * LD + blk * R2p;
                double2 x[R2];
#pragma unroll
                for (int q = 0; q < R2; ++q) x[q] = c[q];
                Dft<R2, -1>::run(x);
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const int k = blk + R1 * k2;
                    const int col = k <= R ? k : (k >= n - R ? W + n - k : 2 * W);      // 2W: pruned, never read
                    Cc[col * LDL + l0 + ll] = x[k2];
                }
            }
            __syncthreads();
        }
        // P3 (untangle rows 2l / 2l+1 + columns pass 1), columns m3 = 0..R; two DFTs per thread (rows j = 2jp, 2jp+1)
        for (int task = tid; task < W * (R2 / 2); task += blockDim.x) {
            const int jp = (task * P.magicW) >> 20, m3 = task - jp * W;                // task / W
            double2 *ca = Cc + m3 * LDL, *cb = Cc + (W + m3) * LDL;
            double2 xa[R1], xb[R1];
            const double2 *cbr = m3 ? cb : ca;   // m3 = 0: with zb := za the formulas give (2 za.x, 0) and (2 za.y, 0): no branch
#pragma unroll
            for (int q = 0; q < R1; ++q) {
                const int l = jp + q * (R2 / 2);
                const double2 za = ca[l], zb = cbr[l];
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
                ca[l] = xa[q];
                cb[l] = xb[q];
            }
        }
        __syncthreads();
        // P4 (columns pass 2): only sticks inside the disk leave the SM
        double2 *z = Z + it * (long long)P.NS;
        for (int task = tid; task < W * R1; task += blockDim.x) {
            const int blk = (task * P.magicW) >> 20, m3 = task - blk * W;              // task / W
            const double2 *ca = Cc + m3 * LDL + blk * (R2 / 2), *cb = Cc + (W + m3) * LDL + blk * (R2 / 2);
            double2 x[R2];
#pragma unroll
            for (int q = 0; q < R2; ++q) x[q] = (q & 1) ? cb[q >> 1] : ca[q >> 1];
            Dft<R2, -1>::run(x);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                const int t2 = blk + R1 * k2;
                if (m3 <= wmax[t2] && m3 >= wmin[t2]) z[soff[t2] + m3] = x[k2];
            }
        }
        __syncthreads();                 // the compact store is rewritten by the next item's P2
    }
}

}  // namespace bsefft
