// Pair screen decision + pair list (eq. 16) and the K1x accumulation (eq. 5):
//   keep (v<=w) iff v == w or M_vw / sqrt(M_vv M_ww) >= eta;   list in lexicographic order
//   acc[b,v,r] = sum_{w : (v,w) or (w,v) kept} tau_{vw}(r) a[b,w,r]
#include "bse_internal.h"

namespace {

__device__ __forceinline__ bool keep_pair(const double *M, int Nv, int v, int w, double eta) {
    if (v == w) return true;
    const double o = M[(long long)v * Nv + w] / sqrt(M[(long long)v * Nv + v] * M[(long long)w * Nv + w]);
    return o >= eta;
}

__global__ void row_count_kernel(const double *__restrict__ M, int Nv, double eta, int *__restrict__ cnt) {
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= Nv) return;
    int c = 0;
    for (int w = v; w < Nv; ++w) c += keep_pair(M, Nv, v, w, eta) ? 1 : 0;
    cnt[v] = c;
}

// exclusive scan of cnt[0..n) into ptr[0..n]; one CTA, staged through shared memory in chunks
__global__ void scan_kernel(const int *__restrict__ cnt, int n, int *__restrict__ ptr) {
    __shared__ int buf[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        buf[threadIdx.x] = (i < n) ? cnt[i] : 0;
        __syncthreads();
        if (threadIdx.x == 0) {
            int run = carry;
            for (int k = 0; k < 1024; ++k) { const int c = buf[k]; buf[k] = run; run += c; }
            carry = run;
        }
        __syncthreads();
        if (i < n) ptr[i] = buf[threadIdx.x];
        __syncthreads();
    }
    if (threadIdx.x == 0) ptr[n] = carry;
}

__global__ void fill_pairs_kernel(const double *__restrict__ M, int Nv, double eta, const int *__restrict__ rowptr,
                                  int2 *__restrict__ pairs, int *__restrict__ pid) {
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= Nv) return;
    int idx = rowptr[v];
    for (int w = 0; w < v; ++w) pid[(long long)v * Nv + w] = -1;
    for (int w = v; w < Nv; ++w) {
        if (keep_pair(M, Nv, v, w, eta)) {
            pairs[idx] = make_int2(v, w);
            pid[(long long)v * Nv + w] = idx++;
        } else {
            pid[(long long)v * Nv + w] = -1;
        }
    }
}

__global__ void adj_count_kernel(const int *__restrict__ pid, int Nv, int *__restrict__ cnt) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nv) return;
    int c = 0;
    for (int x = 0; x < Nv; ++x) {
        const int p = (x < t) ? pid[(long long)x * Nv + t] : pid[(long long)t * Nv + x];
        c += (p >= 0) ? 1 : 0;
    }
    cnt[t] = c;
}

__global__ void adj_fill_kernel(const int *__restrict__ pid, int Nv, const int *__restrict__ ptr,
                                int2 *__restrict__ adj) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nv) return;
    int idx = ptr[t];
    for (int x = 0; x < Nv; ++x) {
        const int p = (x < t) ? pid[(long long)x * Nv + t] : pid[(long long)t * Nv + x];
        if (p >= 0) adj[idx++] = make_int2(x, p);
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
            const double2 t = *reinterpret_cast<const double2 *>(tau + p * N + r);
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

__global__ void weight_pw_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst, long long npw_h,
                                 long long total, double Omega) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const double2 c = src[i];
    dst[i] = (i % npw_h == 0) ? make_double2(Omega * c.x, 0.0) : make_double2(2.0 * Omega * c.x, 2.0 * Omega * c.y);
}

}  // namespace

int bse_launch_weight_pw(const double2 *src, double2 *dst, long long npw_h, long long rows, double Omega,
                         cudaStream_t s) {
    const long long total = npw_h * rows;
    weight_pw_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(src, dst, npw_h, total, Omega);
    BSE_CUDA(cudaGetLastError());
    return BSE_OK;
}

int bse_launch_pairlist(bse_handle *h) {
    const int Nv = h->Nv;
    const int nb = (Nv + 127) / 128;
    row_count_kernel<<<nb, 128, 0, h->stream>>>(h->Mmat, Nv, h->eta, h->rowcnt);
    scan_kernel<<<1, 1024, 0, h->stream>>>(h->rowcnt, Nv, h->rowptr);
    fill_pairs_kernel<<<nb, 128, 0, h->stream>>>(h->Mmat, Nv, h->eta, h->rowptr, h->pairs, h->pid);
    adj_count_kernel<<<nb, 128, 0, h->stream>>>(h->pid, Nv, h->rowcnt);
    scan_kernel<<<1, 1024, 0, h->stream>>>(h->rowcnt, Nv, h->adj_ptr);
    adj_fill_kernel<<<nb, 128, 0, h->stream>>>(h->pid, Nv, h->adj_ptr, h->adj);
    BSE_CUDA(cudaGetLastError());
    int P = 0, nadj = 0;
    BSE_CUDA(cudaMemcpyAsync(&P, h->rowptr + Nv, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaMemcpyAsync(&nadj, h->adj_ptr + Nv, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    BSE_CUDA(cudaStreamSynchronize(h->stream));
    h->P = P;
    h->nadj = nadj;
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
