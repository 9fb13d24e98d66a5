// Slab forms of the stick passes (included by fft_kernels.cu only: the kernels are not templates).
#pragma once
#include "fft_kernels.cuh"

namespace bsefft {

// ---------------------------------------------------------------------------------------------------------
// SLAB stick passes (plane-slab streaming of the PW-layout apply).  A product tau(r) a(r) is local in
// r, so the apply may run on one subset of the i1 planes at a time; for ANY factorisation n = S M the slab
// s = { i1 = s + S k : k < M } splits the 1-D transform along i1 exactly (one decimation step):
//   inverse:  x[s + S k] = sum_{j < M} e^{+2 pi i k j / M}  y_s[j],    y_s[j] = sum_{q < S} X[j + q M] e^{+2 pi i s (j + q M) / n}
//   forward:  X[t1] = sum_s e^{-2 pi i s t1 / n}  Y_s[t1 mod M],      Y_s[j] = sum_{k < M} x[s + S k] e^{-2 pi i k j / M}
// so every slab costs one fold over the (at most 2R+1) non-zero coefficients of a stick plus one M-point transform, all
// slabs together S sweeps over the coefficients on H, and the forward pass ACCUMULATES its slab's contribution into X (slab 0
// stores).  The host picks the smallest S whose slab fits the free memory (fewest sweeps).  Zs[p][k][NS].
// CTA = TS sticks of one field, TS * M threads (the plan keeps M <= 16: 512 threads, two CTAs per SM): thread (j, stick) folds residue class j (<= S stick-coalesced
// gathers, four in flight at a time).  The M-point transform runs out of shared memory as two passes of the split
// M = A B (A + B terms per thread instead of M), input index j = j1 B + j2, output index k = k1 + A k2:
//   z[k1][j2] = w_M^{k1 j2} sum_{j1 < A} y[j1 B + j2] w_A^{k1 j1},      x[k1 + A k2] = sum_{j2 < B} z[k1][j2] w_B^{k2 j2}
// with every root taken from the table tw[t] = e^{-2 pi i t / n} (A | M | n), conjugated for the inverse.
// dynamic smem: C[M][TS + 1] | D[M][TS + 1]
constexpr int SLAB_TS = 32;

// v * w (SIGN < 0, forward) or v * conj(w) (SIGN > 0, inverse)
template <int SIGN>
__device__ __forceinline__ double2 cmul_s(double2 v, double2 w) {
    return SIGN < 0 ? make_double2(v.x * w.x - v.y * w.y, v.x * w.y + v.y * w.x)
                    : make_double2(v.x * w.x + v.y * w.y, v.y * w.x - v.x * w.y);
}

// M-point transform of the TS sticks held in C[j][stick]; thread t (< M) of lane sl returns the value of index
// k = k1 + A k2, k1 = t / B, k2 = t % B.  D is the second buffer; contains one __syncthreads (every thread must call) and
// expects C complete (a barrier) on entry.
// Host-computed constants of one split n = S M, M = A B (no integer division in the kernels): the root strides n/A, n/B, n/M
// and the multiplier that turns t / B into a multiply-shift (exact for t < 64, B <= 32).
struct SlabConst {
    int B, nA, nB, nM, magicB;
};
inline SlabConst slab_const(int n, int M, int A) {
    const int B = M / A;
    return SlabConst{B, n / A, n / B, n / M, (65536 + B - 1) / B};
}

// Root tables of one CTA in shared memory (every entry is read by all lanes of a warp at once: broadcasts), filled once by
// slab_tables:  Wf[q M + j] = tw[slab (j + q M) mod n]  (the fold),  W1[k1 A + j1] = w_A^{k1 j1},  Wm[t] = w_M^{k1 j2} (t = k1 B + j2),
// W2[k2 B + j2] = w_B^{k2 j2};  all as tw[.] = e^{-2 pi i ./n}, conjugated by cmul_s for the inverse.
struct SlabTables {
    const double2 *Wf, *W1, *Wm, *W2;
};
__device__ __forceinline__ int slab_table_size(int NQ, int M, int A, int B) { return NQ * M + A * A + M + B * B; }
__device__ __forceinline__ SlabTables slab_tables(double2 *base, const double2 *__restrict__ tw, int n, int NQ, int M, int A,
                                                  int B, int slab, const SlabConst sc) {
    double2 *Wf = base, *W1 = Wf + NQ * M, *Wm = W1 + A * A, *W2 = Wm + M;
    for (int i = threadIdx.x; i < NQ * M; i += blockDim.x) Wf[i] = tw[(int)(((long long)slab * i) % n)];   // i = q M + j = t1
    for (int i = threadIdx.x; i < A * A; i += blockDim.x) W1[i] = tw[(((i / A) * (i % A)) % A) * sc.nA];
    for (int i = threadIdx.x; i < M; i += blockDim.x) Wm[i] = tw[(i / B) * (i % B) * sc.nM];
    for (int i = threadIdx.x; i < B * B; i += blockDim.x) W2[i] = tw[(((i / B) * (i % B)) % B) * sc.nB];
    return SlabTables{Wf, W1, Wm, W2};
}

template <int SIGN>
__device__ __forceinline__ double2 slab_dft(const double2 *C, double2 *D, const SlabTables &tb, int A, int B, int t, int sl,
                                            int &k_out, const SlabConst sc) {
    constexpr int LDT = SLAB_TS + 1;
    const int k1 = (t * sc.magicB) >> 16, r2 = t - k1 * B;      // t / B, t % B.  pass 1: (k1, j2 = r2); pass 2: (k1, k2 = r2)
    double2 z = make_double2(0.0, 0.0);
    {
        const double2 *c = C + r2 * LDT + sl, *w = tb.W1 + k1 * A;
        for (int j1 = 0; j1 < A; ++j1) {
            const double2 p = cmul_s<SIGN>(c[j1 * B * LDT], w[j1]);
            z.x += p.x;
            z.y += p.y;
        }
        z = cmul_s<SIGN>(z, tb.Wm[t]);                          // w_M^{k1 j2}
    }
    D[t * LDT + sl] = z;                                        // D[k1 B + j2]
    __syncthreads();
    double2 x = make_double2(0.0, 0.0);
    {
        const double2 *d = D + k1 * B * LDT + sl, *w = tb.W2 + r2 * B;
        for (int j2 = 0; j2 < B; ++j2) {
            const double2 p = cmul_s<SIGN>(d[j2 * LDT], w[j2]);
            x.x += p.x;
            x.y += p.y;
        }
    }
    k_out = k1 + A * r2;
    return x;
}

// Both kernels: grid = (stick groups, field chunks).  A CTA keeps ITS sticks and walks over the fields of its chunk, so the
// index map of a stick (which coefficient of H each of its <= S folded terms is) is read once into registers and every field
// costs one round of independent, stick-coalesced gathers (no index load in front of them).  S <= 16.
// NQ = S rounded up to a multiple of 4 (template: the index registers are a compile-time array); MAXT = 512 or 1024 bounds the
// CTA (32 M threads), so that slabs of <= 16 planes get 128 registers per thread.
// STAGED (double coefficients, where the staging area fits beside two CTAs per SM): the NQ gathers of the NEXT field go to
// G[q][thread] by cp.async while this field's M-point transform runs; a thread reads back only what it copied itself.
template <int NQ, int MAXT, bool F32, bool STAGED>
__global__ void __launch_bounds__(MAXT, MAXT <= 512 ? 2 : 1)
inv_stick_slab_kernel(PlanDev P, int n, int S, int M, int A, const double2 *__restrict__ T, long long npw_h,
                      double2 *__restrict__ Zs, const int *__restrict__ gather, int g0, int slab, int count, int per_cta,
                      const float2 *__restrict__ T32, const SlabConst sc) {
    constexpr int TS = SLAB_TS, LDT = TS + 1;
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C = reinterpret_cast<double2 *>(smem);
    double2 *D = C + M * LDT;
    const int NS = P.NS, R = P.R;
    const int sl = threadIdx.x % TS, j = threadIdx.x / TS;      // lanes run over sticks: coalesced gathers
    const int sidx = blockIdx.x * TS + sl;
    const int Bm = sc.B;                                        // M / A
    const SlabTables tb = slab_tables(D + M * LDT, P.tw, n, NQ, M, A, Bm, slab, sc);
    double2 *G = D + M * LDT + slab_table_size(NQ, M, A, Bm);
    __syncthreads();
    int code[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int t1 = j + q * M;
        code[q] = (q < S && sidx < NS && (t1 <= R || t1 >= n - R)) ? P.hmapT[(long long)t1 * NS + sidx] : -1;   // |m1| <= R
    }
    const double2 *wf = tb.Wf + j;                              // wf[q M] = e^{-2 pi i slab t1 / n} for t1 = j + q M
    const int p_end = min(count, (int)(blockIdx.y + 1) * per_cta);
    auto stage_field = [&](int p) {
        const double2 *tg = T + (gather ? (long long)gather[g0 + p] : (long long)p) * npw_h;
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int c = code[q];
            const double2 *src = c >= 0 ? tg + c : (c <= -2 ? tg + (-2 - c) : tg);
            const unsigned dst = (unsigned)__cvta_generic_to_shared(G + q * blockDim.x + threadIdx.x);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(c == -1 ? 0 : 16));
        }
        asm volatile("cp.async.commit_group;\n" ::);
    };
    if (STAGED && (int)(blockIdx.y * per_cta) < p_end) stage_field(blockIdx.y * per_cta);
    for (int p = blockIdx.y * per_cta; p < p_end; ++p) {
        const long long toff = (gather ? (long long)gather[g0 + p] : (long long)p) * npw_h;
        const double2 *tg = T + toff;
        const float2 *tg32 = F32 ? T32 + toff : nullptr;        // coefficients kept in single precision (BSE_TAU_F32)
        double2 y = make_double2(0.0, 0.0);
        if (STAGED) {
            asm volatile("cp.async.wait_group 0;\n" ::: "memory");
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                double2 v = G[q * blockDim.x + threadIdx.x];
                if (code[q] <= -2) v.y = -v.y;
                const double2 pr = cmul_s<+1>(v, wf[q * M]);
                y.x += pr.x;
                y.y += pr.y;
            }
            if (p + 1 < p_end) stage_field(p + 1);
        } else
#pragma unroll
        for (int q0 = 0; q0 < NQ; q0 += 4) {
            double2 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int c = code[q0 + u];
                v[u] = make_double2(0.0, 0.0);
                if (F32) {
                    if (c >= 0) { const float2 f = tg32[c]; v[u] = make_double2((double)f.x, (double)f.y); }
                    else if (c <= -2) { const float2 f = tg32[-2 - c]; v[u] = make_double2((double)f.x, -(double)f.y); }
                } else {
                    if (c >= 0) v[u] = tg[c];
                    else if (c <= -2) { v[u] = tg[-2 - c]; v[u].y = -v[u].y; }
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const double2 pr = cmul_s<+1>(v[u], wf[(q0 + u) * M]);    // times e^{+2 pi i slab t1 / n}
                y.x += pr.x;
                y.y += pr.y;
            }
        }
        __syncthreads();                                        // the previous field's transform has left C and D
        C[j * LDT + sl] = y;
        __syncthreads();
        int k;
        const double2 x = slab_dft<+1>(C, D, tb, A, Bm, j, sl, k, sc);
        if (sidx < NS) Zs[((long long)p * M + k) * NS + sidx] = x;
    }
}

// field p of the launch goes to row  (p / rc) * row_ld + row0 + (p % rc)  of X (the rows of a chunk, block after block)
template <int NQ, int MAXT>
__global__ void __launch_bounds__(MAXT, MAXT <= 512 ? 2 : 1)
fwd_stick_slab_kernel(PlanDev P, int n, int S, int M, int A, const double2 *__restrict__ Zs, double2 *__restrict__ X,
                      long long npw_h, const double *__restrict__ scale, int slab, int accumulate, int rc, long long row_ld,
                      long long row0, int count, int per_cta, const SlabConst sc) {
    constexpr int TS = SLAB_TS, LDT = TS + 1;
    extern __shared__ __align__(16) unsigned char smem[];
    double2 *C = reinterpret_cast<double2 *>(smem);
    double2 *D = C + M * LDT;
    const int NS = P.NS, R = P.R;
    const int sl = threadIdx.x % TS, t = threadIdx.x / TS;
    const int sidx = blockIdx.x * TS + sl;
    const SlabTables tb = slab_tables(D + M * LDT, P.tw, n, NQ, M, A, sc.B, slab, sc);   // first used after the barriers below
    // this thread's output residue j = k1 + A k2 (what slab_dft returns for thread t) and its targets on H, with their scale
    const int Bf = sc.B, tq = (t * sc.magicB) >> 16, j = tq + A * (t - tq * Bf);     // Bf = M / A; j = t / Bf + A (t % Bf)
    int hh[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int t1 = j + q * M;
        hh[q] = (q < S && sidx < NS && (t1 <= R || t1 >= n - R)) ? P.hmapT[(long long)t1 * NS + sidx] : -1;
    }
    const double2 *wf = tb.Wf + j;
    const int p_end = min(count, (int)(blockIdx.y + 1) * per_cta);
    const double2 *zp = Zs + ((long long)blockIdx.y * per_cta * M + t) * NS + sidx;     // plane k = t of the slab
    double2 znext = (sidx < NS && (int)(blockIdx.y * per_cta) < p_end) ? *zp : make_double2(0.0, 0.0);
    for (int p = blockIdx.y * per_cta; p < p_end; ++p) {
        const double2 zin = znext;
        zp += (long long)M * NS;
        if (sidx < NS && p + 1 < p_end) znext = *zp;            // the next field's value travels behind this field's transform
        double2 *xo = X + ((p / rc) * row_ld + row0 + (p % rc)) * npw_h;
        __syncthreads();
        C[t * LDT + sl] = zin;
        __syncthreads();
        int jj;                                                 // Y[j] = sum_k x[k] e^{-2 pi i k j / M}
        const double2 y = slab_dft<-1>(C, D, tb, A, Bf, t, sl, jj, sc);
        // one read-modify-write after the other (measured: a batch of reads followed by a batch of writes is slower)
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            if (hh[q] >= 0) {
                const double2 pr = cmul_s<-1>(y, wf[q * M]);    // times e^{-2 pi i slab t1 / n}
                const double sc = scale[hh[q]];
                double2 v = make_double2(pr.x * sc, pr.y * sc);
                if (accumulate) { const double2 o = xo[hh[q]]; v.x += o.x; v.y += o.y; }
                xo[hh[q]] = v;
            }
        }
    }
}

}  // namespace bsefft
