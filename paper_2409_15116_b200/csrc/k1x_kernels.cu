// Pair screen decision + pair list (eq. 16) and the K1x accumulation (eq. 5):
//   keep (v<=w) iff v == w or M_vw / sqrt(M_vv M_ww) >= eta;   list in lexicographic order
//   acc[b,v,r] = sum_{w : (v,w) or (w,v) kept} tau_{vw}(r) a[b,w,r]
#include <algorithm>

#include "bse_internal.h"

namespace {

__device__ __forceinline__ bool keep_pair(const double *M, int Nv, int v, int w, double eta) {
    if (v == w) return true;
    const double o = M[(long long)v * Nv + w] / sqrt(M[(long long)v * Nv + v] * M[(long long)w * Nv + w]);
    return o >= eta;
}

// exclusive scan of vals[0..n) in place (global memory), total returned to every thread; one CTA of 1024 threads
__device__ int block_exclusive_scan(int *vals, int n, int *smem_warp /*[33]*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int carry = 0;
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        const int x = (i < n) ? vals[i] : 0;
        int incl = x;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += y;
        }
        if (lane == 31) smem_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int w = smem_warp[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, w, d);
                if (lane >= d) w += y;
            }
            smem_warp[lane] = w;                      // inclusive warp totals
        }
        __syncthreads();
        const int before = (warp ? smem_warp[warp - 1] : 0) + carry;
        if (i < n) vals[i] = before + incl - x;
        carry += smem_warp[31];
        __syncthreads();
    }
    return carry;
}

// a1 decision + pair list + directed adjacency in ONE launch (one CTA, warp per row, lanes over w: coalesced rows of M,
// ballot prefix keeps the lexicographic order).  pid is written symmetrically (pid[v][w] = pid[w][v] = pair index or -1).
__global__ void __launch_bounds__(1024)
pairlist_kernel(const double *__restrict__ M, int Nv, double eta, int *__restrict__ rowptr, int2 *__restrict__ pairs,
                int *__restrict__ pid, int *__restrict__ adj_ptr, int2 *__restrict__ adj) {
    __shared__ int sw[33];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    for (int v = warp; v < Nv; v += nwarp) {                                  // kept pairs per row (w >= v)
        int c = 0;
        for (int w0 = v & ~31; w0 < Nv; w0 += 32) {
            const int w = w0 + lane;
            const bool k = (w >= v && w < Nv) ? keep_pair(M, Nv, v, w, eta) : false;
            c += __popc(__ballot_sync(0xffffffffu, k));
        }
        if (lane == 0) rowptr[v] = c;
    }
    __syncthreads();
    const int P = block_exclusive_scan(rowptr, Nv, sw);
    if (threadIdx.x == 0) rowptr[Nv] = P;
    __syncthreads();
    for (int v = warp; v < Nv; v += nwarp) {                                  // fill pairs and the symmetric pid
        int base = rowptr[v];
        for (int w0 = v & ~31; w0 < Nv; w0 += 32) {
            const int w = w0 + lane;
            const bool in = (w >= v && w < Nv);
            const bool k = in ? keep_pair(M, Nv, v, w, eta) : false;
            const unsigned bal = __ballot_sync(0xffffffffu, k);
            const int idx = base + __popc(bal & ((1u << lane) - 1u));
            if (in) {
                const int val = k ? idx : -1;
                if (k) pairs[idx] = make_int2(v, w);
                pid[(long long)v * Nv + w] = val;
                pid[(long long)w * Nv + v] = val;
            }
            base += __popc(bal);
        }
    }
    __syncthreads();
    for (int t = warp; t < Nv; t += nwarp) {                                  // directed entries per row
        int c = 0;
        for (int x0 = 0; x0 < Nv; x0 += 32) {
            const int x = x0 + lane;
            c += __popc(__ballot_sync(0xffffffffu, x < Nv && pid[(long long)t * Nv + x] >= 0));
        }
        if (lane == 0) adj_ptr[t] = c;
    }
    __syncthreads();
    const int nadj = block_exclusive_scan(adj_ptr, Nv, sw);
    if (threadIdx.x == 0) adj_ptr[Nv] = nadj;
    __syncthreads();
    for (int t = warp; t < Nv; t += nwarp) {
        int base = adj_ptr[t];
        for (int x0 = 0; x0 < Nv; x0 += 32) {
            const int x = x0 + lane;
            const int p = (x < Nv) ? pid[(long long)t * Nv + x] : -1;
            const unsigned bal = __ballot_sync(0xffffffffu, p >= 0);
            if (p >= 0) adj[base + __popc(bal & ((1u << lane) - 1u))] = make_int2(x, p);
            base += __popc(bal);
        }
    }
}

// grid = (Nv, ceil(N / (2*blockDim))).  v varies fastest across resident CTAs, so the CTAs in flight share one
// r-tile and a[b][w][tile] / tau_p[tile] are served from L2 after their first touch.
template <int BB>
__global__ void __launch_bounds__(256)
accumulate_kernel(const double *__restrict__ tau, long long p_first, long long p_count,
                  const int *__restrict__ adj_ptr, const int2 *__restrict__ adj, const double *__restrict__ a,
                  double *__restrict__ acc, int Nv, long long N, int b0, int zero_init) {
    const int v = blockIdx.x;
    const long long r = 2 * ((long long)blockIdx.y * blockDim.x + threadIdx.x);
    const int e0 = adj_ptr[v], e1 = adj_ptr[v + 1];
    double2 s[BB];
#pragma unroll
    for (int b = 0; b < BB; ++b) s[b] = make_double2(0.0, 0.0);
    bool any = false;
    for (int e = e0; e < e1; ++e) {
        const int2 wp = adj[e];
        const long long p = wp.y - p_first;
        if (p < 0 || p >= p_count) continue;
        any = true;
        if (r < N) {
            const double2 t = *reinterpret_cast<const double2 *>(tau + p * N + r);   // re-used by row w: keep in L2
#pragma unroll
            for (int b = 0; b < BB; ++b) {
                const double2 x = *reinterpret_cast<const double2 *>(a + ((long long)(b0 + b) * Nv + wp.x) * N + r);
                s[b].x = fma(t.x, x.x, s[b].x);
                s[b].y = fma(t.y, x.y, s[b].y);
            }
        }
    }
    if (r >= N) return;
    if (!any && !zero_init) return;
#pragma unroll
    for (int b = 0; b < BB; ++b) {
        double2 *dst = reinterpret_cast<double2 *>(acc + ((long long)(b0 + b) * Nv + v) * N + r);
        if (zero_init) {
            *dst = s[b];
        } else {
            const double2 o = *dst;
            *dst = make_double2(o.x + s[b].x, o.y + s[b].y);
        }
    }
}

// Row-complete form used with the batched tau modes: the batch holds tau(r) of every pair that its rows
// rows[0 .. gridDim.x) touch, once (a pair with both ends in the batch serves both rows); eslot[e] is the slot of
// directed entry e in the batch.  Each output row is written once, never re-read:
//   acc[b * acc_ld + (local ? i : v)][r] = sum_{e in row v} tau_b[eslot[e]][r] * a[b][adj[e].x][r],  v = rows[i]
// grid = (rows, ceil(N / (2*blockDim))); rows vary fastest across resident CTAs, so they share the r-tile of a in L2.
template <int BB, bool GROUPS>
__global__ void __launch_bounds__(256)
accumulate_rows_kernel(const double *__restrict__ tau_dir, const int *__restrict__ eslot,
                       const int *__restrict__ rows, const int *__restrict__ adj_ptr,
                       const int2 *__restrict__ adj, const double *__restrict__ a, double *__restrict__ acc, int Nv,
                       long long N, int b0, long long acc_ld, int local, int ngroups) {
    // ngroups > 1: blockIdx.x = row * ngroups + g, the CTA takes the blocks b0 + g BB .. of its row.  The CTAs of one row and
    // tile then run side by side, so tau(r) of the row's pairs comes from HBM once and from L2 for the other groups
    const int ri = GROUPS ? blockIdx.x / ngroups : blockIdx.x;
    if (GROUPS) b0 += (blockIdx.x - ri * ngroups) * BB;
    const int v = rows[ri];                          // the batch is a cluster of rows, not a range
    const int arow = local ? ri : v;                 // acc_r of the PW layout holds the batch's rows in batch order
    const long long r = 2 * ((long long)blockIdx.y * blockDim.x + threadIdx.x);
    if (r >= N) return;
    const int ea = adj_ptr[v], eb = adj_ptr[v + 1];
    double2 s[BB];
#pragma unroll
    for (int b = 0; b < BB; ++b) s[b] = make_double2(0.0, 0.0);
    for (int e = ea; e < eb; ++e) {
        const int w = adj[e].x;
        // tau is read once per use: streaming load, so that it does not push the re-used a tiles out of L2
        const long long slot = eslot ? eslot[e] : adj[e].y;      // no slot table: the buffer holds tau of every pair, by pair index
        const double2 t = __ldcs(reinterpret_cast<const double2 *>(tau_dir + slot * N + r));
#pragma unroll
        for (int b = 0; b < BB; ++b) {
            const double2 x = *reinterpret_cast<const double2 *>(a + ((long long)(b0 + b) * Nv + w) * N + r);
            s[b].x = fma(t.x, x.x, s[b].x);
            s[b].y = fma(t.y, x.y, s[b].y);
        }
    }
#pragma unroll
    for (int b = 0; b < BB; ++b)
        __stcs(reinterpret_cast<double2 *>(acc + ((long long)(b0 + b) * acc_ld + arow) * N + r), s[b]);
}

// K1e (eq. 4): transition density n[b][r] = sum_v u[v][r] a[b][v][r] and the product 2 u[v][r] vH[b][r].
// grid = (ceil(N / (2*blockDim)), ceil(B / BB)); u[v] tiles are shared by the BB blocks of a CTA.
template <int BB>
__global__ void __launch_bounds__(256)
k1e_density_kernel(const double *__restrict__ u, const double *__restrict__ a, double *__restrict__ dens, int Nv,
                   long long N, int B, int v0, int nv, int add) {
    const long long r = 2 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);
    if (r >= N) return;
    const int b0 = blockIdx.y * BB;
    double2 s[BB];
#pragma unroll
    for (int b = 0; b < BB; ++b) s[b] = make_double2(0.0, 0.0);
    for (int v = 0; v < nv; ++v) {                     // u holds the orbitals v0 .. v0 + nv (a chunk), a all Nv of them
        const double2 x = *reinterpret_cast<const double2 *>(u + (long long)v * N + r);
#pragma unroll
        for (int b = 0; b < BB; ++b) {
            if (b0 + b < B) {
                const double2 y = __ldcs(reinterpret_cast<const double2 *>(a + ((long long)(b0 + b) * Nv + v0 + v) * N + r));
                s[b].x = fma(x.x, y.x, s[b].x);
                s[b].y = fma(x.y, y.y, s[b].y);
            }
        }
    }
#pragma unroll
    for (int b = 0; b < BB; ++b)
        if (b0 + b < B) {
            double2 *dst = reinterpret_cast<double2 *>(dens + (long long)(b0 + b) * N + r);
            if (add) { const double2 o = *dst; s[b].x += o.x; s[b].y += o.y; }
            *dst = s[b];
        }
}

// out[(b * out_ld + v - v0)][r] = 2 u[v][r] vH[b][r] for v in [v0, v0 + gridDim.y), b < B
__global__ void __launch_bounds__(256)
k1e_product_kernel(const double *__restrict__ u, const double *__restrict__ vH, double *__restrict__ out, int v0,
                   long long out_ld, long long N, int B) {
    const long long r = 2 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);
    if (r >= N) return;
    const int v = v0 + blockIdx.y;
    const double2 x = *reinterpret_cast<const double2 *>(u + (long long)v * N + r);
    for (int b = 0; b < B; ++b) {
        const double2 y = *reinterpret_cast<const double2 *>(vH + (long long)b * N + r);
        __stcs(reinterpret_cast<double2 *>(out + ((long long)b * out_ld + blockIdx.y) * N + r),
               make_double2(2.0 * x.x * y.x, 2.0 * x.y * y.y));
    }
}

// Combined two-body kernel (eq. 1: K1e - K1d share one P_c): acc row <- cd * acc row + ce2 * u[v][r] * vH[b][r] on the rows of
// a batch (rows == nullptr: row i = i); acc row index = position in the batch (local) or the row id.
__global__ void __launch_bounds__(256)
k1_mix_kernel(const double *__restrict__ u, const double *__restrict__ vH, double *__restrict__ acc,
              const int *__restrict__ rows, long long acc_ld, int local, long long N, int nb, double ce2, double cd) {
    const long long r = 2 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);
    if (r >= N) return;
    const int i = blockIdx.y;
    const int v = rows ? rows[i] : i;
    const int arow = local ? i : v;
    const double2 x = *reinterpret_cast<const double2 *>(u + (long long)v * N + r);
    for (int b = 0; b < nb; ++b) {
        const double2 y = *reinterpret_cast<const double2 *>(vH + (long long)b * N + r);
        double2 *dst = reinterpret_cast<double2 *>(acc + ((long long)b * acc_ld + arow) * N + r);
        const double2 p = *dst;
        *dst = make_double2(fma(ce2 * x.x, y.x, cd * p.x), fma(ce2 * x.y, y.y, cd * p.y));
    }
}

// out[2 row] = sum_k x[row][k]^2, out[2 row + 1] = sum_k (x[row][k] - y[row][k])^2; one CTA per row, fixed-order tree
__global__ void __launch_bounds__(256)
row_sumsq_kernel(const double *__restrict__ x, const double *__restrict__ y, long long len, double *__restrict__ out) {
    __shared__ double red[256], red2[256];
    const double *row = x + (long long)blockIdx.x * len, *row2 = y + (long long)blockIdx.x * len;
    double s = 0.0, d = 0.0;
    for (long long k = threadIdx.x; k < len; k += 256) {
        const double a = row[k], e = a - row2[k];
        s = fma(a, a, s);
        d = fma(e, e, d);
    }
    red[threadIdx.x] = s;
    red2[threadIdx.x] = d;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) { red[threadIdx.x] += red[threadIdx.x + w]; red2[threadIdx.x] += red2[threadIdx.x + w]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        out[2 * blockIdx.x] = red[0];
        out[2 * blockIdx.x + 1] = red2[0];
    }
}

__global__ void transpose_kernel(const double *__restrict__ src, long long lds, double *__restrict__ dst, long long ldd, int n) {
    const int i = blockIdx.y * blockDim.y + threadIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && j < n) dst[(long long)j * ldd + i] = src[(long long)i * lds + j];
}

__global__ void weight_pw_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst, long long npw_h,
                                 long long total, double Omega) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const double2 c = src[i];
    dst[i] = (i % npw_h == 0) ? make_double2(Omega * c.x, 0.0) : make_double2(2.0 * Omega * c.x, 2.0 * Omega * c.y);
}

__global__ void to_f32_kernel(const double *__restrict__ src, float *__restrict__ dst, long long count) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) dst[i] = (float)src[i];
}

}  // namespace

int bse_launch_to_f32(const double *src, float *dst, long long count, cudaStream_t s) {
    to_f32_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(src, dst, count);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_weight_pw(const double2 *src, double2 *dst, long long npw_h, long long rows, double Omega,
                         cudaStream_t s) {
    const long long total = npw_h * rows;
    weight_pw_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(src, dst, npw_h, total, Omega);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_pairlist(bse_handle *h) {
    const int Nv = h->Nv;
    pairlist_kernel<<<1, 1024, 0, h->stream>>>(h->Mmat, Nv, h->eta, h->rowptr, h->pairs, h->pid, h->adj_ptr, h->adj);
    BSE_CUDA(cudaGetLastError());
    int P = 0, nadj = 0;
    BSE_CUDA(cudaMemcpyAsync(&P, h->rowptr + Nv, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    h->adj_ptr_h.resize(Nv + 1);
    BSE_CUDA(cudaMemcpyAsync(h->adj_ptr_h.data(), h->adj_ptr, (size_t)(Nv + 1) * 4, cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    h->P = P;
    h->nadj = nadj = h->adj_ptr_h[Nv];
    h->adj_h.clear();
    if ((h->flags & BSE_TAU_MASK) != BSE_TAU_REAL) {   // (w, pair) of every directed entry: row batches are planned on the host
        h->adj_h.resize((size_t)nadj * 2);
        BSE_CUDA(cudaMemcpyAsync(h->adj_h.data(), h->adj, (size_t)nadj * 8, cudaMemcpyDeviceToHost, h->stream));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
    }
    h->Pa = P;
    cudaFree(h->pairs_act); cudaFree(h->eslot_act);
    h->pairs_act = nullptr; h->eslot_act = nullptr;
    if (h->rows_set) {
        // the pairs that touch a row of [row0, row1), in ascending pair index; slot of every directed entry of those rows
        std::vector<int2> pairs_h((size_t)std::max(P, 1));
        BSE_CUDA(cudaMemcpyAsync(pairs_h.data(), h->pairs, (size_t)P * 8, cudaMemcpyDeviceToHost, h->stream));
        BSE_CUDA(cudaStreamSynchronize(h->stream));
        std::vector<int> slot((size_t)std::max(P, 1), -1), eslot((size_t)std::max(nadj, 1), -1);
        std::vector<int2> act;
        for (int p = 0; p < P; ++p) {
            const int2 vw = pairs_h[p];
            if ((vw.x >= h->row0 && vw.x < h->row1) || (vw.y >= h->row0 && vw.y < h->row1)) {
                slot[p] = (int)act.size();
                act.push_back(vw);
            }
        }
        for (int v = h->row0; v < h->row1; ++v)
            for (int e = h->adj_ptr_h[v]; e < h->adj_ptr_h[v + 1]; ++e) eslot[e] = slot[h->adj_h[2 * (size_t)e + 1]];
        h->Pa = (long long)act.size();
        BSE_CUDA(cudaMalloc(&h->pairs_act, std::max<size_t>(act.size(), 1) * 8));
        BSE_CUDA(cudaMalloc(&h->eslot_act, std::max<size_t>(eslot.size(), 1) * 4));
        BSE_CUDA(cudaMemcpy(h->pairs_act, act.data(), act.size() * 8, cudaMemcpyHostToDevice));
        BSE_CUDA(cudaMemcpy(h->eslot_act, eslot.data(), eslot.size() * 4, cudaMemcpyHostToDevice));
    }
    return BSE_OK;
}

int bse_launch_accumulate(bse_handle *h, const double *tau, long long p_first, long long p_count, const double *a,
                          double *acc, int B, bool zero_init) {
    const int threads = 256;
    const long long tiles = (h->N / 2 + threads - 1) / threads;
    dim3 grid(h->Nv, (unsigned)tiles);
    int b0 = 0;
    while (b0 < B) {
        const int left = B - b0;
        if (left >= 8) {
            accumulate_kernel<8><<<grid, threads, 0, h->stream>>>(tau, p_first, p_count, h->adj_ptr, h->adj, a, acc,
                                                                    h->Nv, h->N, b0, zero_init ? 1 : 0);
            b0 += 8;
        } else if (left >= 4) {
            accumulate_kernel<4><<<grid, threads, 0, h->stream>>>(tau, p_first, p_count, h->adj_ptr, h->adj, a, acc,
                                                                    h->Nv, h->N, b0, zero_init ? 1 : 0);
            b0 += 4;
        } else if (left >= 2) {
            accumulate_kernel<2><<<grid, threads, 0, h->stream>>>(tau, p_first, p_count, h->adj_ptr, h->adj, a, acc,
                                                                    h->Nv, h->N, b0, zero_init ? 1 : 0);
            b0 += 2;
        } else {
            accumulate_kernel<1><<<grid, threads, 0, h->stream>>>(tau, p_first, p_count, h->adj_ptr, h->adj, a, acc,
                                                                    h->Nv, h->N, b0, zero_init ? 1 : 0);
            b0 += 1;
        }
    }
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_accumulate_rows(bse_handle *h, long long N, const double *tau_dir, const int *eslot, const int *rows,
                               int nrows, const double *a, double *acc, long long acc_ld, bool local, int B) {
    const int threads = 256;
    const long long tiles = (N / 2 + threads - 1) / threads;
    dim3 grid(nrows, (unsigned)tiles);
    int b0 = 0;
    const int ng = B / 8;                            // whole groups of 8 blocks: one launch, the groups of a row side by side
    if (ng > 1) {
        accumulate_rows_kernel<8, true><<<dim3(nrows * ng, (unsigned)tiles), threads, 0, h->stream>>>(
            tau_dir, eslot, rows, h->adj_ptr, h->adj, a, acc, h->Nv, N, 0, acc_ld, local ? 1 : 0, ng);
        b0 = 8 * ng;
    }
#define BSE_ROWS(BB)                                                                                              \
    accumulate_rows_kernel<BB, false><<<grid, threads, 0, h->stream>>>(tau_dir, eslot, rows, h->adj_ptr, h->adj, a, acc, h->Nv, \
                                                                N, b0, acc_ld, local ? 1 : 0, 1)
    while (b0 < B) {
        const int left = B - b0;
        if (left >= 8) { BSE_ROWS(8); b0 += 8; }
        else if (left >= 4) { BSE_ROWS(4); b0 += 4; }
        else if (left >= 2) { BSE_ROWS(2); b0 += 2; }
        else { BSE_ROWS(1); b0 += 1; }
    }
#undef BSE_ROWS
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_k1e_density(const double *u, const double *a, double *dens, int Nv, long long N, int B, cudaStream_t s,
                           int v0, int nv, bool add) {
    const int threads = 256;
    const unsigned tiles = (unsigned)((N / 2 + threads - 1) / threads);
    if (nv < 0) nv = Nv;
    k1e_density_kernel<4><<<dim3(tiles, (B + 3) / 4), threads, 0, s>>>(u, a, dens, Nv, N, B, v0, nv, add ? 1 : 0);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_k1e_product(const double *u, const double *vH, double *out, int v0, int nrows, long long out_ld,
                           long long N, int B, cudaStream_t s) {
    const int threads = 256;
    const unsigned tiles = (unsigned)((N / 2 + threads - 1) / threads);
    k1e_product_kernel<<<dim3(tiles, nrows), threads, 0, s>>>(u, vH, out, v0, out_ld, N, B);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_transpose(const double *src, long long lds, double *dst, long long ldd, int n, cudaStream_t s) {
    dim3 blk(32, 8), grd((n + 31) / 32, (n + 7) / 8);
    transpose_kernel<<<grd, blk, 0, s>>>(src, lds, dst, ldd, n);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_k1_mix(const double *u, const double *vH, double *acc, const int *rows, int nrows, long long acc_ld,
                      bool local, long long N, int nb, double ce, double cd, cudaStream_t s) {
    const int threads = 256;
    const unsigned tiles = (unsigned)((N / 2 + threads - 1) / threads);
    k1_mix_kernel<<<dim3(tiles, nrows), threads, 0, s>>>(u, vH, acc, rows, acc_ld, local ? 1 : 0, N, nb, 2.0 * ce, cd);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_row_sumsq(const double *x, const double *y, long long len, int rows, double *out, cudaStream_t s) {
    row_sumsq_kernel<<<rows, 256, 0, s>>>(x, y, len, out);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}
