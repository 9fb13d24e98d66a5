// In-register complex DFT codelets (fp64) for sizes 2,3,4,5 (hand-written butterflies) and 6,8,9,10,12,16
// (one Cooley-Tukey split inside the thread, roots folded to immediates after unrolling).
//   Dft<R,S>::run(x): x[k] <- sum_j x[j] exp(S * 2 pi i j k / R),  natural order in and out.  S = -1 forward, +1 inverse.
// Used by the two-pass (n = R1*R2) plane and stick kernels of fft_kernels.cu: each thread transforms R1 or R2
// elements held in registers, so a line of length n crosses shared memory twice instead of log_4(n) times.
#pragma once
#include <cuda_runtime.h>

namespace bsefft {

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cconj(double2 a) { return make_double2(a.x, -a.y); }
// a * (S*i)
template <int S>
__device__ __forceinline__ double2 muli(double2 a) { return S > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x); }

template <int R> struct Roots;
#include "fft_roots.inc"

// a * exp(S * 2 pi i m / R); m is a compile-time constant after unrolling, so the branches fold away
template <int R, int S>
__device__ __forceinline__ double2 mul_root(double2 a, int m) {
    m %= R;
    if (m == 0) return a;
    if (2 * m == R) return make_double2(-a.x, -a.y);
    if (4 * m == R) return muli<S>(a);
    if (4 * m == 3 * R) return muli<-S>(a);
    const double c = Roots<R>::c(m), s = (S > 0 ? 1.0 : -1.0) * Roots<R>::s(m);
    return make_double2(a.x * c - a.y * s, a.x * s + a.y * c);
}

template <int R, int S> struct Dft;

template <int S> struct Dft<1, S> {
    static __device__ __forceinline__ void run(double2 (&)[1]) {}
};
template <int S> struct Dft<2, S> {
    static __device__ __forceinline__ void run(double2 (&x)[2]) {
        const double2 a = x[0], b = x[1];
        x[0] = cadd(a, b); x[1] = csub(a, b);
    }
};
template <int S> struct Dft<3, S> {
    static __device__ __forceinline__ void run(double2 (&x)[3]) {
        const double s3 = (S > 0 ? 1.0 : -1.0) * 0.86602540378443864676;
        const double2 t1 = cadd(x[1], x[2]);
        const double2 t2 = make_double2(x[0].x - 0.5 * t1.x, x[0].y - 0.5 * t1.y);
        const double2 d = csub(x[1], x[2]);
        const double2 t3 = make_double2(-s3 * d.y, s3 * d.x);
        x[0] = cadd(x[0], t1); x[1] = cadd(t2, t3); x[2] = csub(t2, t3);
    }
};
template <int S> struct Dft<4, S> {
    static __device__ __forceinline__ void run(double2 (&x)[4]) {
        const double2 a = cadd(x[0], x[2]), b = csub(x[0], x[2]), c = cadd(x[1], x[3]), d = muli<S>(csub(x[1], x[3]));
        x[0] = cadd(a, c); x[2] = csub(a, c); x[1] = cadd(b, d); x[3] = csub(b, d);
    }
};
template <int S> struct Dft<5, S> {
    static __device__ __forceinline__ void run(double2 (&x)[5]) {
        const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410;
        const double sg = (S > 0 ? 1.0 : -1.0);
        const double s1 = sg * 0.95105651629515357212, s2 = sg * 0.58778525229247312917;
        const double2 a1 = cadd(x[1], x[4]), a2 = cadd(x[2], x[3]), b1 = csub(x[1], x[4]), b2 = csub(x[2], x[3]);
        const double2 x0 = x[0];
        const double2 p1 = make_double2(x0.x + c1 * a1.x + c2 * a2.x, x0.y + c1 * a1.y + c2 * a2.y);
        const double2 p2 = make_double2(x0.x + c2 * a1.x + c1 * a2.x, x0.y + c2 * a1.y + c1 * a2.y);
        const double2 q1 = make_double2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
        const double2 q2 = make_double2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
        const double2 iq1 = make_double2(-q1.y, q1.x), iq2 = make_double2(-q2.y, q2.x);
        x[0] = make_double2(x0.x + a1.x + a2.x, x0.y + a1.y + a2.y);
        x[1] = cadd(p1, iq1); x[4] = csub(p1, iq1); x[2] = cadd(p2, iq2); x[3] = csub(p2, iq2);
    }
};

// R = A * B:  X[k1 + A k2] = sum_b w_R^{b k1} w_B^{b k2} [ sum_a x[a B + b] w_A^{a k1} ]
template <int R, int A, int B, int S>
__device__ __forceinline__ void dft_split(double2 (&x)[R]) {
    double2 t[B][A];
#pragma unroll
    for (int b = 0; b < B; ++b) {
#pragma unroll
        for (int a = 0; a < A; ++a) t[b][a] = x[a * B + b];
        Dft<A, S>::run(t[b]);
#pragma unroll
        for (int k1 = 1; k1 < A; ++k1) t[b][k1] = mul_root<R, S>(t[b][k1], b * k1);
    }
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) {
        double2 u[B];
#pragma unroll
        for (int b = 0; b < B; ++b) u[b] = t[b][k1];
        Dft<B, S>::run(u);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) x[k1 + A * k2] = u[k2];
    }
}
template <int S> struct Dft<6, S> { static __device__ __forceinline__ void run(double2 (&x)[6]) { dft_split<6, 3, 2, S>(x); } };
template <int S> struct Dft<8, S> { static __device__ __forceinline__ void run(double2 (&x)[8]) { dft_split<8, 4, 2, S>(x); } };
template <int S> struct Dft<9, S> { static __device__ __forceinline__ void run(double2 (&x)[9]) { dft_split<9, 3, 3, S>(x); } };
template <int S> struct Dft<10, S> { static __device__ __forceinline__ void run(double2 (&x)[10]) { dft_split<10, 5, 2, S>(x); } };
template <int S> struct Dft<12, S> { static __device__ __forceinline__ void run(double2 (&x)[12]) { dft_split<12, 3, 4, S>(x); } };
template <int S> struct Dft<16, S> { static __device__ __forceinline__ void run(double2 (&x)[16]) { dft_split<16, 4, 4, S>(x); } };

// y[q] *= w^q for q = 1..R-1 given w = w_n^{S j}: powers by squaring (depth log2 R, keeps rounding at a few ulp)
template <int R>
__device__ __forceinline__ void twiddle_powers(double2 (&y)[R], double2 w) {
    double2 p[R];
    p[1 % R] = w;
#pragma unroll
    for (int q = 2; q < R; ++q) p[q] = (q & 1) ? cmul(p[q - 1], w) : cmul(p[q / 2], p[q / 2]);
#pragma unroll
    for (int q = 1; q < R; ++q) y[q] = cmul(y[q], p[q]);
}

}  // namespace bsefft
