// Batched 1-D complex128 FFT engine (Stockham autosort, one radix per pass, butterflies in registers,
// passes exchanged through shared memory).  Unnormalised; SIGN = +1 is the transform used by I
// (exp(+2 pi i jk/L)), SIGN = -1 the one used by I^+ (include/jdft.h).
//
// A CTA transforms T pencils of length L at once.  Shared-memory layout is [L][TP] double2 with the
// pencil index fastest (TP >= T; TP odd when the caller transposes through it), so consecutive threads
// touch consecutive 16-byte words in every pass.  The first pass takes its inputs from a loader functor
// ld(row, t) and the last pass hands its outputs to a store functor st(row, t, value), so callers fuse
// the global-memory side (zero fill, pruning, V multiply, ...) into the butterflies.
//
// Lengths in SpecPlan<> (32 48 64 72 80 96 100 120 128 144 160 192 216 256) run with compile-time radices up to 16
// (two or three passes); any other
// 2/3/5-smooth length runs the same code with the radices 4, 2, 3, 5 taken from FftPlan at run time.
#pragma once
#include <cuda_runtime.h>
#include <type_traits>
#include "jdft_internal.h"

namespace jfft {

// ---------------------------------------------------------------- compile-time trigonometry
struct CS { double c, s; };

constexpr double cx_sin_small(double x) {  // |x| <= pi/4
    const double x2 = x * x;
    double r = 1.0;
    for (int n = 27; n >= 3; n -= 2) r = 1.0 - x2 / (double)((n - 1) * n) * r;
    return x * r;
}
constexpr double cx_cos_small(double x) {  // |x| <= pi/4
    const double x2 = x * x;
    double r = 1.0;
    for (int n = 26; n >= 2; n -= 2) r = 1.0 - x2 / (double)((n - 1) * n) * r;
    return r;
}
// (cos, sin)(2 pi e / R), 0 <= e < R, reduced to the first octant with integer arithmetic
constexpr CS cx_cs(int e, int R) {
    const double pi = 3.14159265358979323846264338327950288;
    const int num = 8 * e;
    const int oct = num / R;
    const int rem = num % R;
    const double phi = (oct & 1) ? (pi * (double)(R - rem)) / (4.0 * R) : (pi * (double)rem) / (4.0 * R);
    const double c = cx_cos_small(phi), s = cx_sin_small(phi);
    switch (oct) {
        case 0: return CS{c, s};
        case 1: return CS{s, c};
        case 2: return CS{-s, c};
        case 3: return CS{-c, s};
        case 4: return CS{-c, -s};
        case 5: return CS{-s, -c};
        case 6: return CS{s, -c};
        default: return CS{c, -s};
    }
}

template <int B, int E, class F>
__device__ __forceinline__ void static_for(F &&f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// ---------------------------------------------------------------- complex helpers
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * (SIGN i)
template <int SIGN>
__device__ __forceinline__ double2 mul_i(double2 a) {
    return SIGN > 0 ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}
// x * exp(SIGN 2 pi i E / R), E and R compile-time
template <int SIGN, int E, int R>
__device__ __forceinline__ double2 mul_w(double2 x) {
    constexpr int e = ((E % R) + R) % R;
    if constexpr (e == 0) {
        return x;
    } else if constexpr ((4 * e) % R == 0) {
        constexpr int q = (4 * e) / R;
        if constexpr (q == 1) return mul_i<SIGN>(x);
        else if constexpr (q == 2) return make_double2(-x.x, -x.y);
        else return mul_i<-SIGN>(x);
    } else {
        constexpr CS w = cx_cs(e, R);
        constexpr double c = w.c;
        constexpr double s = SIGN > 0 ? w.s : -w.s;
        return make_double2(x.x * c - x.y * s, x.x * s + x.y * c);
    }
}

// ---------------------------------------------------------------- in-register DFTs
// a[n] <- sum_k a[k] exp(SIGN 2 pi i n k / R), natural order in and out.
template <int R, int SIGN>
struct Dft;

template <int SIGN>
struct Dft<1, SIGN> {
    static __device__ __forceinline__ void run(double2 (&)[1]) {}
};
template <int SIGN>
struct Dft<2, SIGN> {
    static __device__ __forceinline__ void run(double2 (&a)[2]) {
        const double2 t = a[0];
        a[0] = cadd(t, a[1]);
        a[1] = csub(t, a[1]);
    }
};
template <int SIGN>
struct Dft<3, SIGN> {
    static __device__ __forceinline__ void run(double2 (&a)[3]) {
        constexpr double h = 0.86602540378443864676372317075294;  // sin(pi/3)
        const double2 t1 = cadd(a[1], a[2]);
        const double2 t2 = make_double2(a[0].x - 0.5 * t1.x, a[0].y - 0.5 * t1.y);
        const double2 d = csub(a[1], a[2]);
        const double2 t3 = mul_i<SIGN>(make_double2(h * d.x, h * d.y));
        a[0] = cadd(a[0], t1);
        a[1] = cadd(t2, t3);
        a[2] = csub(t2, t3);
    }
};
template <int SIGN>
struct Dft<4, SIGN> {
    static __device__ __forceinline__ void run(double2 (&a)[4]) {
        const double2 t0 = cadd(a[0], a[2]), t1 = csub(a[0], a[2]);
        const double2 t2 = cadd(a[1], a[3]), t3 = mul_i<SIGN>(csub(a[1], a[3]));
        a[0] = cadd(t0, t2);
        a[2] = csub(t0, t2);
        a[1] = cadd(t1, t3);
        a[3] = csub(t1, t3);
    }
};
template <int SIGN>
struct Dft<5, SIGN> {
    static __device__ __forceinline__ void run(double2 (&a)[5]) {
        constexpr double c1 = 0.30901699437494742410229341718282;   // cos(2 pi/5)
        constexpr double c2 = -0.80901699437494742410229341718282;  // cos(4 pi/5)
        constexpr double s1 = 0.95105651629515357211643933337938;   // sin(2 pi/5)
        constexpr double s2 = 0.58778525229247312916870595463907;   // sin(4 pi/5)
        const double2 p14 = cadd(a[1], a[4]), m14 = csub(a[1], a[4]);
        const double2 p23 = cadd(a[2], a[3]), m23 = csub(a[2], a[3]);
        const double2 r1 = make_double2(a[0].x + c1 * p14.x + c2 * p23.x, a[0].y + c1 * p14.y + c2 * p23.y);
        const double2 r2 = make_double2(a[0].x + c2 * p14.x + c1 * p23.x, a[0].y + c2 * p14.y + c1 * p23.y);
        const double2 i1 = mul_i<SIGN>(make_double2(s1 * m14.x + s2 * m23.x, s1 * m14.y + s2 * m23.y));
        const double2 i2 = mul_i<SIGN>(make_double2(s2 * m14.x - s1 * m23.x, s2 * m14.y - s1 * m23.y));
        a[0] = make_double2(a[0].x + p14.x + p23.x, a[0].y + p14.y + p23.y);
        a[1] = cadd(r1, i1);
        a[4] = csub(r1, i1);
        a[2] = cadd(r2, i2);
        a[3] = csub(r2, i2);
    }
};

// R = R1 R2 by Cooley-Tukey in registers: k = R2 k1 + k2, n = n1 + R1 n2,
// w_R^{nk} = w_R1^{n1 k1} w_R^{n1 k2} w_R2^{n2 k2}
template <int R1, int R2, int SIGN>
__device__ __forceinline__ void dft_composite(double2 (&a)[R1 * R2]) {
    constexpr int R = R1 * R2;
    double2 b[R2][R1];
    static_for<0, R2>([&](auto K2) {
        constexpr int k2 = decltype(K2)::value;
        double2 t[R1];
#pragma unroll
        for (int k1 = 0; k1 < R1; k1++) t[k1] = a[R2 * k1 + k2];
        Dft<R1, SIGN>::run(t);
        static_for<0, R1>([&](auto N1) {
            constexpr int n1 = decltype(N1)::value;
            b[k2][n1] = mul_w<SIGN, n1 * k2, R>(t[n1]);
        });
    });
#pragma unroll
    for (int n1 = 0; n1 < R1; n1++) {
        double2 t[R2];
#pragma unroll
        for (int k2 = 0; k2 < R2; k2++) t[k2] = b[k2][n1];
        Dft<R2, SIGN>::run(t);
#pragma unroll
        for (int n2 = 0; n2 < R2; n2++) a[n1 + R1 * n2] = t[n2];
    }
}
#define JFFT_COMPOSITE(R, R1, R2)                                                              \
    template <int SIGN>                                                                         \
    struct Dft<R, SIGN> {                                                                       \
        static __device__ __forceinline__ void run(double2 (&a)[R]) { dft_composite<R1, R2, SIGN>(a); } \
    };
JFFT_COMPOSITE(6, 2, 3)
JFFT_COMPOSITE(8, 2, 4)
JFFT_COMPOSITE(9, 3, 3)
JFFT_COMPOSITE(10, 2, 5)
JFFT_COMPOSITE(12, 3, 4)
JFFT_COMPOSITE(15, 3, 5)
JFFT_COMPOSITE(16, 4, 4)
#undef JFFT_COMPOSITE

// ---------------------------------------------------------------- compile-time plans
template <int L>
struct SpecPlan {
    static constexpr int npass = 0;  // no specialisation
    static constexpr int r0 = 1, r1 = 1, r2 = 1;
    static constexpr int radix(int) { return 1; }
};
#define JFFT_SPEC2(L, A, B)                                                 \
    template <>                                                              \
    struct SpecPlan<L> {                                                     \
        static constexpr int npass = 2;                                      \
        static constexpr int r0 = A, r1 = B, r2 = 1;                         \
        static constexpr int radix(int i) { return i == 0 ? A : B; }         \
    };
#define JFFT_SPEC3(L, A, B, C)                                               \
    template <>                                                              \
    struct SpecPlan<L> {                                                     \
        static constexpr int npass = 3;                                      \
        static constexpr int r0 = A, r1 = B, r2 = C;                         \
        static constexpr int radix(int i) { return i == 0 ? A : (i == 1 ? B : C); } \
    };
JFFT_SPEC2(32, 4, 8)
JFFT_SPEC2(48, 6, 8)
JFFT_SPEC2(96, 8, 12)
JFFT_SPEC2(100, 10, 10)
JFFT_SPEC2(120, 8, 15)
JFFT_SPEC2(144, 12, 12)
JFFT_SPEC2(160, 10, 16)
JFFT_SPEC2(192, 12, 16)
JFFT_SPEC2(256, 16, 16)
JFFT_SPEC2(64, 8, 8)
JFFT_SPEC2(72, 8, 9)
JFFT_SPEC2(80, 8, 10)
JFFT_SPEC2(128, 8, 16)
JFFT_SPEC3(216, 6, 6, 6)
#undef JFFT_SPEC2
#undef JFFT_SPEC3

inline bool has_spec(int L) {
    switch (L) {
        case 32: case 48: case 64: case 72: case 80: case 96: case 100: case 120: case 128: case 144: case 160: case 192:
        case 216: case 256: return true;
        default: return false;
    }
}

// ---------------------------------------------------------------- one Stockham pass
// Current sub-length n = L / s (s = product of the radices already applied), m = n / R.
// Butterfly bf = p s + q (p < m, q < s) reads rows bf + k L/R and writes rows q + s (R p + j),
// output j multiplied by w_n^{p j} = w_L^{p s j}.
template <int R, int SIGN, int T, int TP, int NT, class Ld, class St>
__device__ __forceinline__ void stockham_pass(const int L, const int s, const bool first, const bool last,
                                              const double2 *__restrict__ tw, const double2 *cur, double2 *nxt,
                                              Ld &ld, St &st) {
    const int nbf = L / R;
    for (int w = threadIdx.x; w < nbf * T; w += NT) {
        const int t = w % T, bf = w / T;
        double2 a[R];
#pragma unroll
        for (int k = 0; k < R; k++) {
            const int row = bf + k * nbf;
            a[k] = first ? ld(row, t) : cur[row * TP + t];
        }
        Dft<R, SIGN>::run(a);
        const int q = bf % s, pb = bf - q;
        if (!last) {
#pragma unroll
            for (int j = 1; j < R; j++) {
                double2 wv = tw[pb * j];
                if (SIGN < 0) wv.y = -wv.y;
                a[j] = cmul(a[j], wv);
            }
        }
        const int ob = q + pb * R;
#pragma unroll
        for (int j = 0; j < R; j++) {
            const int row = ob + s * j;
            if (last) st(row, t, a[j]);
            else nxt[row * TP + t] = a[j];
        }
    }
}

// index (0/1) of the buffer that is free for the store functor of the last pass when pass 0 writes buffer 0
__host__ __device__ inline int fft_out_buf(int npass) { return (npass - 1) & 1; }

// Full transform of T pencils.  Pass 0 reads ld and writes bufA; pass i >= 1 reads the buffer pass i-1
// wrote and writes the other one; the last pass writes through st.  All threads of the CTA must call this.
// The caller synchronises before (if ld reads shared memory written by other threads) and after (if st
// writes shared memory read by other threads).
template <int LT, int SIGN, int T, int TP, int NT, class Ld, class St>
__device__ __forceinline__ void fft_run(const FftPlan &plan, const double2 *__restrict__ tw, double2 *bufA,
                                        double2 *bufB, Ld ld, St st) {
    if constexpr (LT > 0) {
        using P = SpecPlan<LT>;
        static_assert(P::npass >= 1, "no specialised plan for this length");
        static_for<0, P::npass>([&](auto IP) {
            constexpr int ip = decltype(IP)::value;
            constexpr int R = P::radix(ip);
            int s = 1;
#pragma unroll
            for (int i = 0; i < ip; i++) s *= P::radix(i);
            double2 *dst = (ip & 1) ? bufB : bufA;
            const double2 *src = (ip & 1) ? bufA : bufB;
            stockham_pass<R, SIGN, T, TP, NT>(LT, s, ip == 0, ip == P::npass - 1, tw, src, dst, ld, st);
            if (ip != P::npass - 1) __syncthreads();
        });
    } else {
        const int L = plan.L;
        int s = 1;
        for (int ip = 0; ip < plan.npass; ip++) {
            const int R = plan.radix[ip];
            double2 *dst = (ip & 1) ? bufB : bufA;
            const double2 *src = (ip & 1) ? bufA : bufB;
            const bool first = ip == 0, last = ip == plan.npass - 1;
            switch (R) {
                case 1: stockham_pass<1, SIGN, T, TP, NT>(L, s, first, last, tw, src, dst, ld, st); break;
                case 2: stockham_pass<2, SIGN, T, TP, NT>(L, s, first, last, tw, src, dst, ld, st); break;
                case 3: stockham_pass<3, SIGN, T, TP, NT>(L, s, first, last, tw, src, dst, ld, st); break;
                case 4: stockham_pass<4, SIGN, T, TP, NT>(L, s, first, last, tw, src, dst, ld, st); break;
                default: stockham_pass<5, SIGN, T, TP, NT>(L, s, first, last, tw, src, dst, ld, st); break;
            }
            s *= R;
            if (!last) __syncthreads();
        }
    }
}

template <int LT>
__host__ __device__ inline int fft_npass(const FftPlan &plan) {
    if constexpr (LT > 0) return SpecPlan<LT>::npass;
    else return plan.npass;
}

}  // namespace jfft
