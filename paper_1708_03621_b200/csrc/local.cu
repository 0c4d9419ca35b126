// FFT-based operators: I, I^+, J, the local + kinetic part of H, and the diagonal L, O.
// Pipeline of one band batch of apply_H (SURVEY.md 3.3 / DESIGN.md section 5):
//   K1 k_cols_inv   scatter sphere -> columns  (+) inverse FFT along axis 2   (occupied (i0,i1) columns only)
//   K2 k_rows<inv>  inverse FFT along axis 1, compact columns -> dense planes  (occupied i0 planes only)
//   K3 k_planes<V>  inverse FFT along axis 0 (+) * V_loc (+) forward FFT along axis 0 (real-space psi never stored)
//   K4 k_rows<fwd>  forward FFT along axis 1, dense planes -> compact columns
//   K5 k_cols_fwd   forward FFT along axis 2 (+) gather box -> sphere (+) + Omega ke C   (the -1/2 L C term)
// Intermediates: W1 [nbatch][ncol][S2] and W2 [nbatch][npl][S1][S2] (c128) in the caller's workspace.
#include <cmath>
#include "tma.cuh"
#include "fft.cuh"
#include "cols_tuned.cuh"

using namespace jfft;

namespace {

constexpr int kT = 8;      // pencils per CTA
constexpr int kNT = 128;   // threads per CTA
// threads per CTA of the column kernels: the work items of a pass, (L / radix) x kT, should be whole rounds
template <int LT> struct ColsNT { static constexpr int v = kNT; };
template <> struct ColsNT<216> { static constexpr int v = 288; };   // 6 x 6 x 6: 36 x 8 items in every pass
template <> struct ColsNT<32> { static constexpr int v = 64; };     // 4 x 8: 64 and 32 items

__device__ __forceinline__ int wrapi(int m, int S) {
    int r = m % S;
    return r < 0 ? r + S : r;
}

// ------------------------------------------------------------------------------------------------ K1
template <int LT>
__global__ void __launch_bounds__(ColsNT<LT>::v) k_cols_inv(const FftPlan plan, const double2 *__restrict__ tw, const int ncol,
                                                  const int64_t nG, const int *__restrict__ col_n0,
                                                  const int *__restrict__ col_m2lo, const double2 *__restrict__ C,
                                                  double2 *__restrict__ W1) {
    constexpr int T = kT, TP = kT + 1, NT = ColsNT<LT>::v;
    const int L = LT > 0 ? LT : plan.L;
    extern __shared__ double2 smem[];
    double2 *bufA = smem, *bufB = smem + L * TP;
    __shared__ int s_n0[T + 1], s_m2[T];
    const int tid = threadIdx.x, c0 = blockIdx.x * T, b = blockIdx.y;
    const int nc = min(T, ncol - c0);
    if (tid <= T) s_n0[tid] = col_n0[min(c0 + tid, ncol)];
    if (tid < T) s_m2[tid] = col_m2lo[min(c0 + tid, ncol - 1)];
    for (int e = tid; e < L * TP; e += NT) bufB[e] = make_double2(0.0, 0.0);
    __syncthreads();
    const int nbeg = s_n0[0], nend = s_n0[nc];
    const double2 *Cb = C + (size_t)b * nG;
    for (int e = tid; e < nend - nbeg; e += NT) {
        const int n = nbeg + e;
        int t = 0;
        while (n >= s_n0[t + 1]) t++;
        const int row = wrapi(s_m2[t] + (n - s_n0[t]), L);
        bufB[row * TP + t] = Cb[n];
    }
    __syncthreads();
    double2 *out = fft_out_buf(fft_npass<LT>(plan)) ? bufB : bufA;
    fft_run<LT, +1, T, TP, NT>(
        plan, tw, bufA, bufB, [&](int row, int t) { return bufB[row * TP + t]; },
        [&](int row, int t, double2 v) { out[row * TP + t] = v; });
    __syncthreads();
    double2 *Wb = W1 + ((size_t)b * ncol + c0) * L;
    for (int e = tid; e < nc * L; e += NT) {
        const int t = e / L, row = e - t * L;
        Wb[e] = out[row * TP + t];
    }
}

// ------------------------------------------------------------------------------------------------ K5
// out[b][n] = scale * (F_2 W1)[column of n][m2 of n]  (+ kin * ke[n] * C[b][n])
template <int LT>
__global__ void __launch_bounds__(ColsNT<LT>::v) k_cols_fwd(const FftPlan plan, const double2 *__restrict__ tw, const int ncol,
                                                  const int64_t nG, const int *__restrict__ col_n0,
                                                  const int *__restrict__ col_m2lo, const double2 *__restrict__ W1,
                                                  const double scale, const double kin, const double *__restrict__ ke,
                                                  const double2 *__restrict__ C, double2 *__restrict__ outC) {
    constexpr int T = kT, TP = kT + 1, NT = ColsNT<LT>::v;
    const int L = LT > 0 ? LT : plan.L;
    extern __shared__ double2 smem[];
    double2 *bufA = smem, *bufB = smem + L * TP;
    __shared__ int s_n0[T + 1], s_m2[T];
    const int tid = threadIdx.x, c0 = blockIdx.x * T, b = blockIdx.y;
    const int nc = min(T, ncol - c0);
    if (tid <= T) s_n0[tid] = col_n0[min(c0 + tid, ncol)];
    if (tid < T) s_m2[tid] = col_m2lo[min(c0 + tid, ncol - 1)];
    const double2 *Wb = W1 + ((size_t)b * ncol + c0) * L;
    for (int e = tid; e < T * L; e += NT) {
        const int t = e / L, row = e - t * L;
        bufB[row * TP + t] = t < nc ? Wb[e] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    double2 *out = fft_out_buf(fft_npass<LT>(plan)) ? bufB : bufA;
    fft_run<LT, -1, T, TP, NT>(
        plan, tw, bufA, bufB, [&](int row, int t) { return bufB[row * TP + t]; },
        [&](int row, int t, double2 v) { out[row * TP + t] = v; });
    __syncthreads();
    const int nbeg = s_n0[0], nend = s_n0[nc];
    const double2 *Cb = C + (size_t)b * nG;
    double2 *Ob = outC + (size_t)b * nG;
    for (int e = tid; e < nend - nbeg; e += NT) {
        const int n = nbeg + e;
        int t = 0;
        while (n >= s_n0[t + 1]) t++;
        const int row = wrapi(s_m2[t] + (n - s_n0[t]), L);
        double2 v = out[row * TP + t];
        v.x *= scale;
        v.y *= scale;
        if (kin != 0.0) {
            const double f = kin * ke[n];
            const double2 c = Cb[n];
            v.x = fma(f, c.x, v.x);
            v.y = fma(f, c.y, v.y);
        }
        Ob[n] = v;
    }
}

// ------------------------------------------------------------------------------------------------ K2 / K4
// FWD == false: W1 columns -> (inverse FFT along axis 1) -> W2 planes.   FWD == true: the reverse, forward FFT.
template <int LT, bool FWD>
__global__ void __launch_bounds__(kNT) k_rows(const FftPlan plan, const double2 *__restrict__ tw, const int S2,
                                              const int npl, const int ncol, const int *__restrict__ rowcol,
                                              double2 *__restrict__ W1, double2 *__restrict__ W2) {
    constexpr int T = kT, TP = kT, NT = kNT;
    const int L = LT > 0 ? LT : plan.L;  // = S1
    extern __shared__ double2 smem[];
    double2 *bufA = smem, *bufB = smem + L * TP;
    int *s_rowcol = reinterpret_cast<int *>(smem + 2 * L * TP);
    const int tid = threadIdx.x, t0 = blockIdx.x * T, p = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_rowcol[i] = rowcol[p * L + i];
    __syncthreads();
    double2 *W1b = W1 + (size_t)b * ncol * S2 + t0;
    double2 *W2b = W2 + ((size_t)b * npl + p) * L * S2 + t0;
    const int tmax = S2 - t0;
    if (!FWD) {
        fft_run<LT, +1, T, TP, NT>(
            plan, tw, bufA, bufB,
            [&](int row, int t) {
                const int c = s_rowcol[row];
                return (c >= 0 && t < tmax) ? W1b[(size_t)c * S2 + t] : make_double2(0.0, 0.0);
            },
            [&](int row, int t, double2 v) {
                if (t < tmax) W2b[(size_t)row * S2 + t] = v;
            });
    } else {
        fft_run<LT, -1, T, TP, NT>(
            plan, tw, bufA, bufB,
            [&](int row, int t) { return t < tmax ? W2b[(size_t)row * S2 + t] : make_double2(0.0, 0.0); },
            [&](int row, int t, double2 v) {
                const int c = s_rowcol[row];
                if (c >= 0 && t < tmax) W1b[(size_t)c * S2 + t] = v;
            });
    }
}

// ------------------------------------------------------------------------------------------------ K3
// MODE 0: W2 -> inverse axis 0 -> * V -> forward axis 0 -> W2 (in place; each CTA owns its pencils)
// MODE 1: W2 -> inverse axis 0 -> psi (full box)          [last step of I]
// MODE 2: psi (full box) -> forward axis 0 -> W2           [first step of I^+]
template <int LT, int MODE>
__global__ void __launch_bounds__(kNT) k_planes(const FftPlan plan, const double2 *__restrict__ tw, const int S1,
                                                const int S2, const int npl, const int *__restrict__ planeof,
                                                double2 *__restrict__ W2, const double *__restrict__ V,
                                                double2 *__restrict__ psi) {
    constexpr int T = kT, TP = kT, NT = kNT;
    const int L = LT > 0 ? LT : plan.L;  // = S0
    extern __shared__ double2 smem[];
    double2 *bufA = smem, *bufB = smem + L * TP;
    int *s_planeof = reinterpret_cast<int *>(smem + 2 * L * TP);
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
    const int tmax = S2 - t0;
    auto ld_w2 = [&](int row, int t) {
        const int p = s_planeof[row];
        return (p >= 0 && t < tmax) ? W2b[p * plane + t] : make_double2(0.0, 0.0);
    };
    auto st_w2 = [&](int row, int t, double2 v) {
        const int p = s_planeof[row];
        if (p >= 0 && t < tmax) W2b[p * plane + t] = v;
    };
    if (MODE == 0) {
        const int np = fft_npass<LT>(plan);
        double2 *X = fft_out_buf(np) ? bufB : bufA;
        double2 *Y = fft_out_buf(np) ? bufA : bufB;
        const double *Vb = V + (size_t)i1 * S2 + t0;
        fft_run<LT, +1, T, TP, NT>(plan, tw, bufA, bufB, ld_w2, [&](int row, int t, double2 v) {
            const double f = t < tmax ? Vb[row * plane + t] : 0.0;
            X[row * TP + t] = make_double2(v.x * f, v.y * f);
        });
        __syncthreads();
        fft_run<LT, -1, T, TP, NT>(plan, tw, Y, X, [&](int row, int t) { return X[row * TP + t]; }, st_w2);
    } else if (MODE == 1) {
        double2 *pb = psi + (size_t)b * L * plane + (size_t)i1 * S2 + t0;
        fft_run<LT, +1, T, TP, NT>(plan, tw, bufA, bufB, ld_w2, [&](int row, int t, double2 v) {
            if (t < tmax) pb[row * plane + t] = v;
        });
    } else {
        const double2 *pb = psi + (size_t)b * L * plane + (size_t)i1 * S2 + t0;
        fft_run<LT, -1, T, TP, NT>(
            plan, tw, bufA, bufB,
            [&](int row, int t) { return t < tmax ? pb[row * plane + t] : make_double2(0.0, 0.0); }, st_w2);
    }
}

// ================================================================================================ tuned kernels
// Two-pass specialised lengths (L = R1 R2: 32, 64, 72, 80, 128) run the kernels below instead of k_rows / k_planes<0>:
//  * 16 pencils per CTA (256-byte global segments), thread count = 16 x (work items of the heaviest pass / 16) so
//    that no thread idles at a barrier while others compute a butterfly;
//  * ONE shared-memory tile [L][16] (half the footprint of the ping-pong engine -> twice the resident CTAs);
//  * in k_planes_fused the inverse transform runs the radices (R1, R2) and the forward transform (R2, R1): the last
//    inverse pass leaves a thread holding rows bf + R1 j (j < R2), which are exactly the inputs of the first forward
//    pass, so IDFT_R2 -> * V_loc -> DFT_R2 happens in registers: 4 instead of 6 shared-memory tile transfers and
//    3 instead of 4 barriers per pencil pair.
template <int LT>
struct Tuned {
    static constexpr bool ok = SpecPlan<LT>::npass == 2;
    static constexpr int R1 = SpecPlan<LT>::r0, R2 = SpecPlan<LT>::r1;
    static constexpr int T = 16;
    // threads = T x (butterflies of the pass that must run in one round = the R2 pass) rounded so the R1 pass is whole rounds
    static constexpr int NB1 = ok ? LT / R1 : 1, NB2 = ok ? LT / R2 : 1;   // butterflies per pencil in the R1 / R2 pass
    static constexpr int NBT = (NB1 % NB2 == 0) ? NB2 : (NB1 > NB2 ? NB1 : NB2);
    static constexpr int NT = T * NBT;
};

template <int R, int SIGN>
__device__ __forceinline__ void twiddle_rows(double2 (&a)[R], const double2 *__restrict__ tw, const int bf) {
#pragma unroll
    for (int j = 1; j < R; j++) {
        double2 wv = __ldg(tw + bf * j);
        if (SIGN < 0) wv.y = -wv.y;
        a[j] = cmul(a[j], wv);
    }
}

// resident CTAs per SM the register allocation of k_planes_fused is bounded for (measured: DESIGN.md section 12, table of experiments)
// default: registers the fused middle radix needs (16 complex values + V factors for radix 15/16) against 64 K per SM
template <int LT> struct PlanesMinB {
    static constexpr int need = Tuned<LT>::R2 >= 12 ? 128 : 96;
    static constexpr int fit = 65536 / (Tuned<LT>::NT * need);
    static constexpr int v = fit < 1 ? 1 : (fit > 6 ? 6 : fit);
};
#ifndef PLANES_MINB_80
#define PLANES_MINB_80 6
#endif
template <> struct PlanesMinB<80> { static constexpr int v = PLANES_MINB_80; };
template <> struct PlanesMinB<72> { static constexpr int v = 6; };
// K3 tuned: W2 -> IFFT axis 0 -> * V -> FFT axis 0 -> W2 (in place)
template <int LT>
__global__ void __launch_bounds__(Tuned<LT>::NT, PlanesMinB<LT>::v) k_planes_fused(const double2 *__restrict__ tw, const int S1, const int S2,
                                                                const int npl, const int *__restrict__ planeof,
                                                                double2 *__restrict__ W2, const double *__restrict__ V) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, NT = C::NT, L = LT;
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_planeof[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
    const double *Vb = V + (size_t)i1 * S2 + t0;
    const int tmax = S2 - t0;
    // pass 0 of the inverse transform: radix R1, rows bf + k R2 -> rows bf R1 + j, twiddle w^(bf j)
    for (int w = tid; w < R2 * T; w += NT) {
        const int t = w % T, bf = w / T;
        double2 a[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            const int p = s_planeof[bf + k * R2];
            a[k] = (p >= 0 && t < tmax) ? W2b[p * plane + t] : make_double2(0.0, 0.0);
        }
        Dft<R1, +1>::run(a);
        twiddle_rows<R1, +1>(a, tw, bf);
#pragma unroll
        for (int j = 0; j < R1; j++) A[(bf * R1 + j) * T + t] = a[j];
    }
    __syncthreads();
    // last inverse pass (radix R2) -> * V -> first forward pass (radix R2), all in registers
    {
        static_assert(R1 * T <= NT, "the fused middle pass must run in one round");
        const int t = tid % T, bf = tid / T;
        const bool act = tid < R1 * T;
        double2 a[R2];
        if (act) {
#pragma unroll
            for (int k = 0; k < R2; k++) a[k] = A[(bf + k * R1) * T + t];
        }
        __syncthreads();
        if (act) {
            Dft<R2, +1>::run(a);
#pragma unroll
            for (int j = 0; j < R2; j++) {
                const double f = t < tmax ? __ldg(Vb + (size_t)(bf + R1 * j) * plane + t) : 0.0;
                a[j].x *= f;
                a[j].y *= f;
            }
            Dft<R2, -1>::run(a);
            twiddle_rows<R2, -1>(a, tw, bf);
#pragma unroll
            for (int j = 0; j < R2; j++) A[(bf * R2 + j) * T + t] = a[j];
        }
    }
    __syncthreads();
    // last forward pass: radix R1, rows bf + k R2 -> rows bf + R2 j (only the occupied planes are stored)
    for (int w = tid; w < R2 * T; w += NT) {
        const int t = w % T, bf = w / T;
        double2 a[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) a[k] = A[(bf + k * R2) * T + t];
        Dft<R1, -1>::run(a);
#pragma unroll
        for (int j = 0; j < R1; j++) {
            const int p = s_planeof[bf + R2 * j];
            if (p >= 0 && t < tmax) W2b[p * plane + t] = a[j];
        }
    }
}

// K3 with TWO adjacent pencils per thread (lengths whose fused radix is <= 10, so 2 x R2 complex values fit in
// registers): the twiddle, plane-map and V reads are shared by the pair and W2 / V move as 256-bit / 128-bit words,
// which cuts the load/store instruction count per pencil by ~30 % on the pipe that bounds k_planes_fused.
// Shared tile [L][T] with the even pencils in the first half of a row and the odd ones in the second, so both
// 16-byte accesses of a thread are lane-contiguous.  Requires S2 even (32-byte alignment of a pencil pair).
// Radix-8 butterflies pruned to the sphere's extent along axis 0 (PR = true, R1 = 8): when the planes
// [2 R2, 6 R2) hold no sphere point (|m0| < 2 R2, true for every workload of BASELINE.json at 80 and 128), inputs
// 2..5 of every first-pass butterfly are zero and outputs 2..5 of every last-pass butterfly are discarded.
// dft8_in0167: a[n] <- a0 + a1 w^n + a6 w^6n + a7 w^7n, w = exp(SIGN 2 pi i / 8)  (a[2..5] ignored on entry)
template <int SIGN>
__device__ __forceinline__ void dft8_in0167(double2 (&a)[8]) {
    const double2 j6 = mul_i<SIGN>(a[6]);
    const double2 e0 = cadd(a[0], a[6]), e2 = csub(a[0], a[6]), e1 = csub(a[0], j6), e3 = cadd(a[0], j6);
    const double2 u = mul_w<SIGN, 1, 8>(a[1]), v = mul_w<SIGN, 7, 8>(a[7]);
    const double2 o0 = cadd(a[1], a[7]), o2 = mul_i<SIGN>(csub(a[1], a[7]));
    const double2 o1 = cadd(u, v), o3 = mul_i<SIGN>(csub(u, v));
    a[0] = cadd(e0, o0); a[4] = csub(e0, o0);
    a[1] = cadd(e1, o1); a[5] = csub(e1, o1);
    a[2] = cadd(e2, o2); a[6] = csub(e2, o2);
    a[3] = cadd(e3, o3); a[7] = csub(e3, o3);
}
// dft8_out0167: outputs 0, 1, 6, 7 of the full length-8 DFT (a[2..5] undefined on exit)
template <int SIGN>
__device__ __forceinline__ void dft8_out0167(double2 (&a)[8]) {
    const double2 s0 = cadd(a[0], a[4]), s1 = cadd(a[1], a[5]), s2 = cadd(a[2], a[6]), s3 = cadd(a[3], a[7]);
    const double2 d0 = csub(a[0], a[4]), d1 = csub(a[1], a[5]), d2 = csub(a[2], a[6]), d3 = csub(a[3], a[7]);
    const double2 j2 = mul_i<SIGN>(d2), j3 = mul_i<SIGN>(d3);
    a[0] = cadd(cadd(s0, s2), cadd(s1, s3));
    a[6] = csub(csub(s0, s2), mul_i<SIGN>(csub(s1, s3)));
    a[1] = cadd(cadd(d0, j2), mul_w<SIGN, 1, 8>(cadd(d1, j3)));
    a[7] = cadd(csub(d0, j2), mul_w<SIGN, 7, 8>(csub(d1, j3)));
}

template <int LT>
struct Pair {
    static constexpr int T = LT == 72 ? 32 : 16;       // pencils per CTA
    static constexpr int H = T / 2;                    // threads per butterfly row
    static constexpr int G = 1;                        // tiles (adjacent i1 rows) per CTA (2 at length 80 measured slower)
    static constexpr int NTG = Tuned<LT>::NBT * H;     // threads per tile
    static constexpr int NT = G * NTG;
    static constexpr bool ok = Tuned<LT>::ok && Tuned<LT>::R2 <= 10 && Tuned<LT>::R1 <= 10;
};
__device__ __forceinline__ void ld256(const double2 *p, double2 &a, double2 &b) {
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a.x), "=d"(a.y), "=d"(b.x), "=d"(b.y) : "l"(p));
}
__device__ __forceinline__ void st256(double2 *p, const double2 a, const double2 b) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y) : "memory");
}
template <int LT, bool PR = false>
__global__ void __launch_bounds__(Pair<LT>::NT) k_planes_fused2(const double2 *__restrict__ tw, const int S1, const int S2,
                                                                const int npl, const int *__restrict__ planeof,
                                                                double2 *__restrict__ W2, const double *__restrict__ V) {
    using C = Tuned<LT>;
    using Q = Pair<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = Q::T, H = Q::H, NT = Q::NTG, L = LT;
    static_assert(R1 * H <= NT, "the fused middle pass must run in one round");
    extern __shared__ double2 smem[];
    __shared__ int s_planeof[L];
    const int grp = threadIdx.x / NT, tid = threadIdx.x % NT;  // tile of this thread inside the CTA, index inside the tile
    double2 *A = smem + grp * L * T;
    const int t0 = blockIdx.x * T, i1 = blockIdx.y * Q::G + grp, b = blockIdx.z;
    for (int i = threadIdx.x; i < L; i += Q::NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const bool live = i1 < S1;
    const size_t plane = (size_t)S1 * S2;
    double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
    const double *Vb = V + (size_t)i1 * S2 + t0;
    const int tmax = live ? S2 - t0 : 0;  // even; 0 switches every global access of an idle tile group off
    for (int w = tid; w < R2 * H; w += NT) {
        const int l = w % H, bf = w / H;
        double2 a0[R1], a1[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            if (PR && k >= 2 && k < 6) continue;
            const int p = s_planeof[bf + k * R2];
            a0[k] = a1[k] = make_double2(0.0, 0.0);
            if (p >= 0 && 2 * l < tmax) ld256(W2b + p * plane + 2 * l, a0[k], a1[k]);
        }
        if constexpr (PR) {
            dft8_in0167<+1>(a0);
            dft8_in0167<+1>(a1);
        } else {
            Dft<R1, +1>::run(a0);
            Dft<R1, +1>::run(a1);
        }
#pragma unroll
        for (int j = 1; j < R1; j++) {
            const double2 wv = __ldg(tw + bf * j);
            a0[j] = cmul(a0[j], wv);
            a1[j] = cmul(a1[j], wv);
        }
#pragma unroll
        for (int j = 0; j < R1; j++) {
            A[(bf * R1 + j) * T + l] = a0[j];
            A[(bf * R1 + j) * T + H + l] = a1[j];
        }
    }
    __syncthreads();
    {
        const int l = tid % H, bf = tid / H;
        const bool act = tid < R1 * H;
        double2 a0[R2], a1[R2];
        if (act) {
#pragma unroll
            for (int k = 0; k < R2; k++) {
                a0[k] = A[(bf + k * R1) * T + l];
                a1[k] = A[(bf + k * R1) * T + H + l];
            }
        }
        __syncthreads();
        if (act) {
            Dft<R2, +1>::run(a0);
            Dft<R2, +1>::run(a1);
#pragma unroll
            for (int j = 0; j < R2; j++) {
                double2 f = make_double2(0.0, 0.0);
                if (2 * l < tmax) f = __ldg(reinterpret_cast<const double2 *>(Vb + (size_t)(bf + R1 * j) * plane + 2 * l));
                a0[j].x *= f.x;
                a0[j].y *= f.x;
                a1[j].x *= f.y;
                a1[j].y *= f.y;
            }
            Dft<R2, -1>::run(a0);
            Dft<R2, -1>::run(a1);
#pragma unroll
            for (int j = 1; j < R2; j++) {
                double2 wv = __ldg(tw + bf * j);
                wv.y = -wv.y;
                a0[j] = cmul(a0[j], wv);
                a1[j] = cmul(a1[j], wv);
            }
#pragma unroll
            for (int j = 0; j < R2; j++) {
                A[(bf * R2 + j) * T + l] = a0[j];
                A[(bf * R2 + j) * T + H + l] = a1[j];
            }
        }
    }
    __syncthreads();
    for (int w = tid; w < R2 * H; w += NT) {
        const int l = w % H, bf = w / H;
        double2 a0[R1], a1[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            a0[k] = A[(bf + k * R2) * T + l];
            a1[k] = A[(bf + k * R2) * T + H + l];
        }
        if constexpr (PR) {
            dft8_out0167<-1>(a0);
            dft8_out0167<-1>(a1);
        } else {
            Dft<R1, -1>::run(a0);
            Dft<R1, -1>::run(a1);
        }
#pragma unroll
        for (int j = 0; j < R1; j++) {
            if (PR && j >= 2 && j < 6) continue;
            const int p = s_planeof[bf + R2 * j];
            if (p >= 0 && 2 * l < tmax) st256(W2b + p * plane + 2 * l, a0[j], a1[j]);
        }
    }
}

// K3 hybrid for lengths 128 and 80: the first and last pass (radix 8, global side) handle TWO adjacent pencils per thread with
// 256-bit loads/stores and shared twiddle / plane-map reads, in ONE round of all 128 threads; the fused middle pass
// (radix 16, one pencil per thread: two would not fit in registers) is unchanged.  Tile rows keep the even pencils in
// the first half and the odd ones in the second; middle-pass lane x works on pencil 2x (x < 8) or 2(x-8)+1, so every
// shared-memory access of a quarter-warp is one contiguous 128-byte row segment.  Requires S2 even.
template <int LT>
struct Hyb {  // threads = the larger of the pair passes' and the middle pass' work items
    static constexpr int PAIRS = Tuned<LT>::R2 * (Tuned<LT>::T / 2), MID = Tuned<LT>::R1 * Tuned<LT>::T;
    static constexpr int NT = PAIRS > MID ? PAIRS : MID;
    static constexpr int MINB = LT == 128 ? 4 : 5;   // measured
};
template <int LT, bool PR = false>
__global__ void __launch_bounds__(Hyb<LT>::NT, (PR && LT == 80) ? 6 : Hyb<LT>::MINB) k_planes_fused_h(const double2 *__restrict__ tw, const int S1,
                                                                                     const int S2, const int npl,
                                                                                     const int *__restrict__ planeof,
                                                                                     double2 *__restrict__ W2,
                                                                                     const double *__restrict__ V) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, H = T / 2, NT = Hyb<LT>::NT, L = LT;
    static_assert(R2 * H <= NT && R1 * T <= NT, "pair passes and the fused middle pass must each be one round");
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_planeof[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
    const double *Vb = V + (size_t)i1 * S2 + t0;
    const int tmax = S2 - t0;  // even
    if (tid < R2 * H) {
        const int l = tid % H, bf = tid / H;
        double2 a0[R1], a1[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            if (PR && k >= 2 && k < 6) continue;
            const int p = s_planeof[bf + k * R2];
            a0[k] = a1[k] = make_double2(0.0, 0.0);
            if (p >= 0 && 2 * l < tmax) ld256(W2b + p * plane + 2 * l, a0[k], a1[k]);
        }
        if constexpr (PR) {
            dft8_in0167<+1>(a0);
            dft8_in0167<+1>(a1);
        } else {
            Dft<R1, +1>::run(a0);
            Dft<R1, +1>::run(a1);
        }
#pragma unroll
        for (int j = 1; j < R1; j++) {
            const double2 wv = __ldg(tw + bf * j);
            a0[j] = cmul(a0[j], wv);
            a1[j] = cmul(a1[j], wv);
        }
#pragma unroll
        for (int j = 0; j < R1; j++) {
            A[(bf * R1 + j) * T + l] = a0[j];
            A[(bf * R1 + j) * T + H + l] = a1[j];
        }
    }
    __syncthreads();
    {
        const int x = tid % T, bf = tid / T;             // x = slot inside the tile row
        const int t = x < H ? 2 * x : 2 * (x - H) + 1;   // pencil stored in that slot
        const bool act = tid < R1 * T;
        double2 a[R2];
        if (act) {
#pragma unroll
            for (int k = 0; k < R2; k++) a[k] = A[(bf + k * R1) * T + x];
        }
        __syncthreads();
        if (act) {
            Dft<R2, +1>::run(a);
#pragma unroll
            for (int j = 0; j < R2; j++) {
                const double f = t < tmax ? __ldg(Vb + (size_t)(bf + R1 * j) * plane + t) : 0.0;
                a[j].x *= f;
                a[j].y *= f;
            }
            Dft<R2, -1>::run(a);
            twiddle_rows<R2, -1>(a, tw, bf);
#pragma unroll
            for (int j = 0; j < R2; j++) A[(bf * R2 + j) * T + x] = a[j];
        }
    }
    __syncthreads();
    if (tid < R2 * H) {
        const int l = tid % H, bf = tid / H;
        double2 a0[R1], a1[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            a0[k] = A[(bf + k * R2) * T + l];
            a1[k] = A[(bf + k * R2) * T + H + l];
        }
        if constexpr (PR) {
            dft8_out0167<-1>(a0);
            dft8_out0167<-1>(a1);
        } else {
            Dft<R1, -1>::run(a0);
            Dft<R1, -1>::run(a1);
        }
#pragma unroll
        for (int j = 0; j < R1; j++) {
            if (PR && j >= 2 && j < 6) continue;
            const int p = s_planeof[bf + R2 * j];
            if (p >= 0 && 2 * l < tmax) st256(W2b + p * plane + 2 * l, a0[j], a1[j]);
        }
    }
}

// K2 / K4 hybrid (same idea as k_planes_fused_h): the first pass works on pencil pairs with 256-bit loads and shared
// twiddle / row-map reads, the last pass on single pencils with lane x -> pencil 2x | 2(x-8)+1.  Requires S2 even.
template <int LT, bool FWD>
__global__ void __launch_bounds__(Hyb<LT>::NT) k_rows_hyb(const double2 *__restrict__ tw, const int S2, const int npl,
                                                          const int ncol, const int *__restrict__ rowcol,
                                                          double2 *__restrict__ W1, double2 *__restrict__ W2) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, H = T / 2, NT = Hyb<LT>::NT, L = LT;
    constexpr int SIGN = FWD ? -1 : +1;
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_rowcol[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, p = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_rowcol[i] = rowcol[p * L + i];
    __syncthreads();
    double2 *W1b = W1 + (size_t)b * ncol * S2 + t0;
    double2 *W2b = W2 + ((size_t)b * npl + p) * L * S2 + t0;
    const int tmax = S2 - t0;  // even
    if (tid < R2 * H) {
        const int l = tid % H, bf = tid / H;
        double2 a0[R1], a1[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            const int row = bf + k * R2;
            a0[k] = a1[k] = make_double2(0.0, 0.0);
            if (FWD) {
                if (2 * l < tmax) ld256(W2b + (size_t)row * S2 + 2 * l, a0[k], a1[k]);
            } else {
                const int c = s_rowcol[row];
                if (c >= 0 && 2 * l < tmax) ld256(W1b + (size_t)c * S2 + 2 * l, a0[k], a1[k]);
            }
        }
        Dft<R1, SIGN>::run(a0);
        Dft<R1, SIGN>::run(a1);
#pragma unroll
        for (int j = 1; j < R1; j++) {
            double2 wv = __ldg(tw + bf * j);
            if (SIGN < 0) wv.y = -wv.y;
            a0[j] = cmul(a0[j], wv);
            a1[j] = cmul(a1[j], wv);
        }
#pragma unroll
        for (int j = 0; j < R1; j++) {
            A[(bf * R1 + j) * T + l] = a0[j];
            A[(bf * R1 + j) * T + H + l] = a1[j];
        }
    }
    __syncthreads();
    if (tid < R1 * T) {
        const int x = tid % T, bf = tid / T;
        const int t = x < H ? 2 * x : 2 * (x - H) + 1;
        double2 a[R2];
#pragma unroll
        for (int k = 0; k < R2; k++) a[k] = A[(bf + k * R1) * T + x];
        Dft<R2, SIGN>::run(a);
#pragma unroll
        for (int j = 0; j < R2; j++) {
            const int row = bf + R1 * j;
            if (FWD) {
                const int c = s_rowcol[row];
                if (c >= 0 && t < tmax) W1b[(size_t)c * S2 + t] = a[j];
            } else {
                if (t < tmax) W2b[(size_t)row * S2 + t] = a[j];
            }
        }
    }
}

// Last pass of I (MODE 1: occupied planes of W2 -> full real-space block) and first pass of I^+ / J (MODE 2: the
// reverse), same hybrid as k_rows_hyb: pencil pairs with 256-bit loads in the first pass, single pencils in the last.
template <int LT, int MODE, bool PR = false>   // PR: pruned radix-8 first pass of I (MODE 1), see dft8_in0167
__global__ void __launch_bounds__(Hyb<LT>::NT) k_planes_io_hyb(const double2 *__restrict__ tw, const int S1, const int S2,
                                                               const int npl, const int *__restrict__ planeof,
                                                               double2 *__restrict__ W2, double2 *__restrict__ psi) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, H = T / 2, NT = Hyb<LT>::NT, L = LT;
    constexpr int SIGN = MODE == 1 ? +1 : -1;
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_planeof[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
    double2 *pb = psi + (size_t)b * L * plane + (size_t)i1 * S2 + t0;
    const int tmax = S2 - t0;  // even
    if (tid < R2 * H) {
        const int l = tid % H, bf = tid / H;
        double2 a0[R1], a1[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            if (PR && MODE == 1 && k >= 2 && k < 6) continue;
            const int row = bf + k * R2;
            a0[k] = a1[k] = make_double2(0.0, 0.0);
            if (MODE == 1) {
                const int p = s_planeof[row];
                if (p >= 0 && 2 * l < tmax) ld256(W2b + p * plane + 2 * l, a0[k], a1[k]);
            } else {
                if (2 * l < tmax) ld256(pb + row * plane + 2 * l, a0[k], a1[k]);
            }
        }
        if constexpr (PR && MODE == 1) {
            dft8_in0167<SIGN>(a0);
            dft8_in0167<SIGN>(a1);
        } else {
            Dft<R1, SIGN>::run(a0);
            Dft<R1, SIGN>::run(a1);
        }
#pragma unroll
        for (int j = 1; j < R1; j++) {
            double2 wv = __ldg(tw + bf * j);
            if (SIGN < 0) wv.y = -wv.y;
            a0[j] = cmul(a0[j], wv);
            a1[j] = cmul(a1[j], wv);
        }
#pragma unroll
        for (int j = 0; j < R1; j++) {
            A[(bf * R1 + j) * T + l] = a0[j];
            A[(bf * R1 + j) * T + H + l] = a1[j];
        }
    }
    __syncthreads();
    if (tid < R1 * T) {
        const int x = tid % T, bf = tid / T;
        const int t = x < H ? 2 * x : 2 * (x - H) + 1;
        double2 a[R2];
#pragma unroll
        for (int k = 0; k < R2; k++) a[k] = A[(bf + k * R1) * T + x];
        Dft<R2, SIGN>::run(a);
#pragma unroll
        for (int j = 0; j < R2; j++) {
            const int row = bf + R1 * j;
            if (MODE == 1) {
                if (t < tmax) pb[row * plane + t] = a[j];
            } else {
                const int p = s_planeof[row];
                if (p >= 0 && t < tmax) W2b[p * plane + t] = a[j];
            }
        }
    }
}

// Density with the hybrid first pass (pencil pairs, 256-bit loads) of k_planes_io_hyb and register accumulators.
template <int LT, bool PR = false>   // PR: pruned radix-8 first pass, see dft8_in0167
__global__ void __launch_bounds__(Hyb<LT>::NT) k_planes_density_hyb(const double2 *__restrict__ tw, const int S1, const int S2,
                                                                    const int npl, const int *__restrict__ planeof,
                                                                    const double2 *__restrict__ W2, const double *__restrict__ f,
                                                                    const int nbt, double *__restrict__ n, const int accumulate) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, H = T / 2, NT = Hyb<LT>::NT, L = LT;
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_planeof[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    const int tmax = S2 - t0;  // even
    const int x = tid % T, bfl = tid / T;
    const int tl = x < H ? 2 * x : 2 * (x - H) + 1;
    const bool act = tid < R1 * T;
    double acc[R2];
#pragma unroll
    for (int j = 0; j < R2; j++) acc[j] = 0.0;
    for (int b = 0; b < nbt; b++) {
        const double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
        if (tid < R2 * H) {
            const int l = tid % H, bf = tid / H;
            double2 a0[R1], a1[R1];
#pragma unroll
            for (int k = 0; k < R1; k++) {
                if (PR && k >= 2 && k < 6) continue;
                const int p = s_planeof[bf + k * R2];
                a0[k] = a1[k] = make_double2(0.0, 0.0);
                if (p >= 0 && 2 * l < tmax) ld256(W2b + p * plane + 2 * l, a0[k], a1[k]);
            }
            if constexpr (PR) {
                dft8_in0167<+1>(a0);
                dft8_in0167<+1>(a1);
            } else {
                Dft<R1, +1>::run(a0);
                Dft<R1, +1>::run(a1);
            }
#pragma unroll
            for (int j = 1; j < R1; j++) {
                const double2 wv = __ldg(tw + bf * j);
                a0[j] = cmul(a0[j], wv);
                a1[j] = cmul(a1[j], wv);
            }
#pragma unroll
            for (int j = 0; j < R1; j++) {
                A[(bf * R1 + j) * T + l] = a0[j];
                A[(bf * R1 + j) * T + H + l] = a1[j];
            }
        }
        __syncthreads();
        if (act) {
            const double fb = f[b];
            double2 a[R2];
#pragma unroll
            for (int k = 0; k < R2; k++) a[k] = A[(bfl + k * R1) * T + x];
            Dft<R2, +1>::run(a);
#pragma unroll
            for (int j = 0; j < R2; j++) acc[j] = fma(fb, a[j].x * a[j].x + a[j].y * a[j].y, acc[j]);
        }
        __syncthreads();
    }
    if (act && tl < tmax) {
        double *o = n + (size_t)i1 * S2 + t0 + tl;
#pragma unroll
        for (int j = 0; j < R2; j++) {
            double *q = o + (size_t)(bfl + R1 * j) * plane;
            *q = accumulate ? *q + acc[j] : acc[j];
        }
    }
}

// Density, tuned: last pass of I for the two-pass lengths with the |psi|^2 accumulators in REGISTERS.  A CTA owns the
// tile (i1, 16 adjacent i2) and walks the bands of the batch in order; in the last pass (radix R2, one round) a
// thread always produces the same rows bf + R1 j of the same pencil, so it keeps their R2 partial sums itself.
template <int LT>
__global__ void __launch_bounds__(Tuned<LT>::NT) k_planes_density_tuned(const double2 *__restrict__ tw, const int S1, const int S2,
                                                                        const int npl, const int *__restrict__ planeof,
                                                                        const double2 *__restrict__ W2,
                                                                        const double *__restrict__ f, const int nbt,
                                                                        double *__restrict__ n, const int accumulate) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, NT = C::NT, L = LT;
    static_assert(R1 * T <= NT, "the last pass must run in one round");
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_planeof[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    const int tmax = S2 - t0;
    const int tl = tid % T, bfl = tid / T;
    const bool act = tid < R1 * T;
    double acc[R2];
#pragma unroll
    for (int j = 0; j < R2; j++) acc[j] = 0.0;
    for (int b = 0; b < nbt; b++) {
        const double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
        for (int w = tid; w < R2 * T; w += NT) {
            const int t = w % T, bf = w / T;
            double2 a[R1];
#pragma unroll
            for (int k = 0; k < R1; k++) {
                const int p = s_planeof[bf + k * R2];
                a[k] = (p >= 0 && t < tmax) ? W2b[p * plane + t] : make_double2(0.0, 0.0);
            }
            Dft<R1, +1>::run(a);
            twiddle_rows<R1, +1>(a, tw, bf);
#pragma unroll
            for (int j = 0; j < R1; j++) A[(bf * R1 + j) * T + t] = a[j];
        }
        __syncthreads();
        if (act) {
            const double fb = f[b];
            double2 a[R2];
#pragma unroll
            for (int k = 0; k < R2; k++) a[k] = A[(bfl + k * R1) * T + tl];
            Dft<R2, +1>::run(a);
#pragma unroll
            for (int j = 0; j < R2; j++) acc[j] = fma(fb, a[j].x * a[j].x + a[j].y * a[j].y, acc[j]);
        }
        __syncthreads();
    }
    if (act && tl < tmax) {
        double *o = n + (size_t)i1 * S2 + t0 + tl;
#pragma unroll
        for (int j = 0; j < R2; j++) {
            double *q = o + (size_t)(bfl + R1 * j) * plane;
            *q = accumulate ? *q + acc[j] : acc[j];
        }
    }
}

// K2 / K4 tuned: one transform along axis 1 between compact columns (W1) and compact planes (W2)
template <int LT, bool FWD>
__global__ void __launch_bounds__(Tuned<LT>::NT) k_rows_tuned(const double2 *__restrict__ tw, const int S2, const int npl,
                                                              const int ncol, const int *__restrict__ rowcol,
                                                              double2 *__restrict__ W1, double2 *__restrict__ W2) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = C::T, NT = C::NT, L = LT;
    constexpr int SIGN = FWD ? -1 : +1;
    extern __shared__ double2 smem[];
    double2 *A = smem;
    __shared__ int s_rowcol[L];
    const int tid = threadIdx.x, t0 = blockIdx.x * T, p = blockIdx.y, b = blockIdx.z;
    for (int i = tid; i < L; i += NT) s_rowcol[i] = rowcol[p * L + i];
    __syncthreads();
    double2 *W1b = W1 + (size_t)b * ncol * S2 + t0;
    double2 *W2b = W2 + ((size_t)b * npl + p) * L * S2 + t0;
    const int tmax = S2 - t0;
    for (int w = tid; w < R2 * T; w += NT) {
        const int t = w % T, bf = w / T;
        double2 a[R1];
#pragma unroll
        for (int k = 0; k < R1; k++) {
            const int row = bf + k * R2;
            if (FWD) {
                a[k] = t < tmax ? W2b[(size_t)row * S2 + t] : make_double2(0.0, 0.0);
            } else {
                const int c = s_rowcol[row];
                a[k] = (c >= 0 && t < tmax) ? W1b[(size_t)c * S2 + t] : make_double2(0.0, 0.0);
            }
        }
        Dft<R1, SIGN>::run(a);
        twiddle_rows<R1, SIGN>(a, tw, bf);
#pragma unroll
        for (int j = 0; j < R1; j++) A[(bf * R1 + j) * T + t] = a[j];
    }
    __syncthreads();
    for (int w = tid; w < R1 * T; w += NT) {
        const int t = w % T, bf = w / T;
        double2 a[R2];
#pragma unroll
        for (int k = 0; k < R2; k++) a[k] = A[(bf + k * R1) * T + t];
        Dft<R2, SIGN>::run(a);
#pragma unroll
        for (int j = 0; j < R2; j++) {
            const int row = bf + R1 * j;
            if (FWD) {
                const int c = s_rowcol[row];
                if (c >= 0 && t < tmax) W1b[(size_t)c * S2 + t] = a[j];
            } else {
                if (t < tmax) W2b[(size_t)row * S2 + t] = a[j];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ density
// n[j] (+)= sum_b f[b] |psi_b[j]|^2 for the nbt bands of a batch: the last pass of I with an
// accumulate-|psi|^2 epilogue instead of a store.  One CTA owns a tile (i1, kT adjacent i2) of the box and walks the
// bands of the batch in order, so the sum has a fixed order and needs no atomics; psi never reaches HBM.
template <int LT>
__global__ void __launch_bounds__(kNT) k_planes_density(const FftPlan plan, const double2 *__restrict__ tw, const int S1,
                                                        const int S2, const int npl, const int *__restrict__ planeof,
                                                        const double2 *__restrict__ W2, const double *__restrict__ f,
                                                        const int nbt, double *__restrict__ n, const int accumulate) {
    constexpr int T = kT, TP = kT, NT = kNT;
    const int L = LT > 0 ? LT : plan.L;  // = S0
    extern __shared__ double2 smem[];
    double2 *bufA = smem, *bufB = smem + L * TP;
    double *acc = reinterpret_cast<double *>(smem + 2 * L * TP);
    int *s_planeof = reinterpret_cast<int *>(acc + L * TP);
    const int tid = threadIdx.x, t0 = blockIdx.x * T, i1 = blockIdx.y;
    for (int i = tid; i < L; i += NT) s_planeof[i] = planeof[i];
    for (int i = tid; i < L * TP; i += NT) acc[i] = 0.0;
    __syncthreads();
    const size_t plane = (size_t)S1 * S2;
    const int tmax = S2 - t0;
    for (int b = 0; b < nbt; b++) {
        const double2 *W2b = W2 + (size_t)b * npl * plane + (size_t)i1 * S2 + t0;
        const double fb = f[b];
        fft_run<LT, +1, T, TP, NT>(
            plan, tw, bufA, bufB,
            [&](int row, int t) {
                const int p = s_planeof[row];
                return (p >= 0 && t < tmax) ? W2b[p * plane + t] : make_double2(0.0, 0.0);
            },
            [&](int row, int t, double2 v) { acc[row * TP + t] += fb * (v.x * v.x + v.y * v.y); });
        __syncthreads();
    }
    double *nb_ = n + (size_t)i1 * S2 + t0;
    for (int e = tid; e < L * T; e += NT) {
        const int row = e / T, t = e - row * T;
        if (t < tmax) {
            double *o = nb_ + (size_t)row * plane + t;
            *o = accumulate ? *o + acc[row * TP + t] : acc[row * TP + t];
        }
    }
}

// ------------------------------------------------------------------------------------------------ gradient / divergence
// ("gradient and divergence operators apply in reciprocal space (where they are diagonal)")
// q(n) = G^T (iG[n] + k) Cartesian; Gm = the 3x3 G row-major (row i = reciprocal vector b_i).
struct Mat3 { double g[9], k[3]; };
__device__ __forceinline__ void q_of(const Mat3 &m, const int32_t *__restrict__ iG, const int64_t n, double (&q)[3]) {
    const double t0 = iG[3 * n] + m.k[0], t1 = iG[3 * n + 1] + m.k[1], t2 = iG[3 * n + 2] + m.k[2];
#pragma unroll
    for (int d = 0; d < 3; d++) q[d] = m.g[d] * t0 + m.g[3 + d] * t1 + m.g[6 + d] * t2;
}
// out[d][b][n] = i q_d C[b][n]
__global__ void k_gradient(const Mat3 m, const int32_t *__restrict__ iG, const int64_t nG, const int64_t total,
                           const double2 *__restrict__ C, double2 *__restrict__ out) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        double q[3];
        q_of(m, iG, i % nG, q);
        const double2 c = C[i];
#pragma unroll
        for (int d = 0; d < 3; d++) out[d * total + i] = make_double2(-q[d] * c.y, q[d] * c.x);
    }
}
// out[b][n] = f * sum_d i q_d X[d][b][n]
__global__ void k_divergence(const Mat3 m, const int32_t *__restrict__ iG, const int64_t nG, const int64_t total,
                             const double f, const double2 *__restrict__ X, double2 *__restrict__ out) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        double q[3];
        q_of(m, iG, i % nG, q);
        double sr = 0.0, si = 0.0;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            const double2 x = X[d * total + i];
            sr -= q[d] * x.y;
            si += q[d] * x.x;
        }
        out[i] = make_double2(f * sr, f * si);
    }
}

// Real fields, two for one (Listing 1 on half-sphere storage, jdft_pcm_hessian_real).  The 3 nb gradient components
// c = d nb + ib of real fields are Hermitian-symmetric spectra G_c; a pair (2p, 2p+1) rides through the COMPLEX pipeline
// as Z_p = G_2p + i G_2p+1 (its real-space image is g_2p + i g_2p+1, so the real epsilon acts on both at once) and is
// separated afterwards: G'_2p[n] = (Z'[n] + conj(Z'[-n])) / 2,  G'_2p+1[n] = (Z'[n] - conj(Z'[-n])) / (2 i).
// Gamma-point bases only: the canonical order is inversion symmetric, -n = nG - 1 - n, origin n0 = (nG - 1) / 2, and
// the stored half is n0 .. nG - 1:  phi~[n0 + h] = ph[h],  phi~[n0 - h] = conj(ph[h]),  Im phi~[n0] ignored.
__device__ __forceinline__ double2 half_ext(const double2 *__restrict__ ph, const int64_t n, const int64_t n0) {
    if (n > n0) return ph[n - n0];
    if (n < n0) { const double2 v = ph[n0 - n]; return make_double2(v.x, -v.y); }
    return make_double2(ph[0].x, 0.0);
}
// Z[p][n] = i q_d(n) phi~_ib[n] + i * (i q_d'(n) phi~_ib'[n]),  (d, ib) = component 2p, (d', ib') = component 2p + 1
__global__ void k_grad_pack_real(const Mat3 m, const int32_t *__restrict__ iG, const int64_t nG, const int nb, const int npair,
                                 const double2 *__restrict__ phi_h, double2 *__restrict__ Z) {
    const int64_t n0 = (nG - 1) / 2, nGh = n0 + 1, total = (int64_t)npair * nG;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int p = (int)(i / nG);
        const int64_t n = i - (int64_t)p * nG;
        double q[3];
        q_of(m, iG, n, q);
        const int c0 = 2 * p, c1 = 2 * p + 1;
        const double2 a = half_ext(phi_h + (size_t)(c0 % nb) * nGh, n, n0);
        // i q a = (-q a.y, q a.x)
        const double qa = q[c0 / nb];
        double zr = -qa * a.y, zi = qa * a.x;
        if (c1 < 3 * nb) {
            const double2 bb = half_ext(phi_h + (size_t)(c1 % nb) * nGh, n, n0);
            const double qb = q[c1 / nb];
            // + i * (i qb bb) = i * (-qb bb.y, qb bb.x) = (-qb bb.x, -qb bb.y)
            zr -= qb * bb.x;
            zi -= qb * bb.y;
        }
        Z[i] = make_double2(zr, zi);
    }
}
// out_h[ib][h] = f * sum_d i q_d(n) G'_{d nb + ib}[n],  n = n0 + h
__global__ void k_unpack_div_real(const Mat3 m, const int32_t *__restrict__ iG, const int64_t nG, const int nb, const double f,
                                  const double2 *__restrict__ Z, double2 *__restrict__ out_h) {
    const int64_t n0 = (nG - 1) / 2, nGh = n0 + 1, total = (int64_t)nb * nGh;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int ib = (int)(i / nGh);
        const int64_t h = i - (int64_t)ib * nGh, n = n0 + h, nm = n0 - h;
        double q[3];
        q_of(m, iG, n, q);
        double sr = 0.0, si = 0.0;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            const int c = d * nb + ib;
            const double2 *Zp = Z + (size_t)(c >> 1) * nG;
            const double2 zp = Zp[n], zm = Zp[nm];
            double gr, gi;
            if ((c & 1) == 0) {   // (z+ + conj(z-)) / 2
                gr = 0.5 * (zp.x + zm.x);
                gi = 0.5 * (zp.y - zm.y);
            } else {              // (z+ - conj(z-)) / (2 i) = (Im-part difference, -Re-part difference) / 2
                gr = 0.5 * (zp.y + zm.y);
                gi = -0.5 * (zp.x - zm.x);
            }
            sr -= q[d] * gi;      // i q g = (-q gi, q gr)
            si += q[d] * gr;
        }
        out_h[i] = make_double2(f * sr, f * si);
    }
}

// ------------------------------------------------------------------------------------------------ diagonal ops
// out[b][n] = (f0 + f1 * ke[n]) * C[b][n]
__global__ void k_diag(const int64_t nG, const int64_t total, const double f0, const double f1,
                       const double *__restrict__ ke, const double2 *__restrict__ C, double2 *__restrict__ out) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const double f = f0 + f1 * ke[i % nG];
        const double2 c = C[i];
        out[i] = make_double2(f * c.x, f * c.y);
    }
}

#include "planes_tma.cuh"

// ------------------------------------------------------------------------------------------------ launch helpers
// the 256-bit global accesses of the pair / hybrid kernels need 32-byte aligned arrays (the ABI only asks for 16)
inline bool aligned32(const void *a, const void *b = nullptr) { return ((((uintptr_t)a) | ((uintptr_t)b)) & 31) == 0; }

// (static __shared__ tables count against the 48 KB default too, hence the 40 KB threshold)
template <class K>
cudaError_t ensure_smem(K kernel, size_t bytes, int device) {
    return bytes <= 40 * 1024 ? cudaSuccess : jdft_ensure_smem((const void *)kernel, bytes, device);
}

#define SPEC_SWITCH(L, force_generic, ...)                    \
    do {                                                      \
        const int l__ = (force_generic) ? 0 : (L);            \
        switch (l__) {                                        \
            case 32: { constexpr int LT = 32; __VA_ARGS__; } break;  \
            case 48: { constexpr int LT = 48; __VA_ARGS__; } break;  \
            case 96: { constexpr int LT = 96; __VA_ARGS__; } break;  \
            case 100: { constexpr int LT = 100; __VA_ARGS__; } break; \
            case 120: { constexpr int LT = 120; __VA_ARGS__; } break; \
            case 144: { constexpr int LT = 144; __VA_ARGS__; } break; \
            case 160: { constexpr int LT = 160; __VA_ARGS__; } break; \
            case 192: { constexpr int LT = 192; __VA_ARGS__; } break; \
            case 256: { constexpr int LT = 256; __VA_ARGS__; } break; \
            case 64: { constexpr int LT = 64; __VA_ARGS__; } break;  \
            case 72: { constexpr int LT = 72; __VA_ARGS__; } break;  \
            case 80: { constexpr int LT = 80; __VA_ARGS__; } break;  \
            case 128: { constexpr int LT = 128; __VA_ARGS__; } break; \
            case 216: { constexpr int LT = 216; __VA_ARGS__; } break; \
            default: { constexpr int LT = 0; __VA_ARGS__; } break;   \
        }                                                     \
    } while (0)

struct Bufs {
    double2 *W1, *W2;
};

Bufs carve(const jdft_basis *b, int nbatch, size_t ws_offset = 0) {
    Bufs w;
    w.W1 = reinterpret_cast<double2 *>(static_cast<char *>(b->ws) + ws_offset);
    w.W2 = w.W1 + (size_t)nbatch * b->ncol * b->S[2];
    return w;
}

int launch_cols_inv(const jdft_basis *b, const double2 *C, int nbt, double2 *W1, cudaStream_t st) {
    const int L = b->S[2];
    const size_t smem = 2 * (size_t)L * (kT + 1) * sizeof(double2);
    dim3 grid((b->ncol + kT - 1) / kT, nbt);
    jdft_prof_begin(b, JDFT_K_COLS_INV, st);
    SPEC_SWITCH(L, b->opt_force_generic, {
        if constexpr (jcols::Cfg<LT>::ok) {
            using F = jcols::Cfg<LT>;
            dim3 g2((b->ncol + F::T - 1) / F::T, nbt);
            // pruned radix-8 first pass when no sphere point has |m2| >= 2 NB0 (rows [2 NB0, 6 NB0) empty)
            const bool pr = F::R0 == 8 && b->opt_prune && b->mmin[2] > -2 * F::NB0 && b->mmax[2] < 2 * F::NB0;
            // first pass straight from the sphere where a column has >= 16 first-pass butterflies (half-warps along one
            // column's rows); measured: 128: 0.844 -> 0.705 ms (config 5), 216: 1.903 -> 1.767 ms (config 4), 80 (10
            // butterflies): 0.0491 -> 0.0502 ms, so shorter columns keep the staged scatter
            constexpr bool kDirect = F::NB0 >= 16;
            const bool direct = kDirect && b->opt_cols_direct;
            if constexpr (kDirect) {
                if (direct && pr) {
                    JDFT_CUDA(ensure_smem(jcols::k_cols_inv_tuned<LT, F::R0 == 8, true>, F::smem, b->device));
                    jcols::k_cols_inv_tuned<LT, F::R0 == 8, true><<<g2, F::NT, F::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, C, W1);
                } else if (direct) {
                    JDFT_CUDA(ensure_smem(jcols::k_cols_inv_tuned<LT, false, true>, F::smem, b->device));
                    jcols::k_cols_inv_tuned<LT, false, true><<<g2, F::NT, F::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, C, W1);
                }
            }
            if (!direct && pr) {
                JDFT_CUDA(ensure_smem(jcols::k_cols_inv_tuned<LT, F::R0 == 8>, F::smem, b->device));
                jcols::k_cols_inv_tuned<LT, F::R0 == 8><<<g2, F::NT, F::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, C, W1);
            } else if (!direct) {
                JDFT_CUDA(ensure_smem(jcols::k_cols_inv_tuned<LT>, F::smem, b->device));
                jcols::k_cols_inv_tuned<LT><<<g2, F::NT, F::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, C, W1);
            }
        } else {
            JDFT_CUDA(ensure_smem(k_cols_inv<LT>, smem, b->device));
            k_cols_inv<LT><<<grid, ColsNT<LT>::v, smem, st>>>(b->plan[2], b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, C, W1);
        }
    });
    jdft_prof_end(b, JDFT_K_COLS_INV, st);
    JDFT_LAUNCH_CHECK("k_cols_inv");
    return JDFT_OK;
}

int launch_cols_fwd(const jdft_basis *b, const double2 *W1, int nbt, double scale, double kin, const double2 *C,
                    double2 *out, cudaStream_t st) {
    const int L = b->S[2];
    const size_t smem = 2 * (size_t)L * (kT + 1) * sizeof(double2);
    dim3 grid((b->ncol + kT - 1) / kT, nbt);
    jdft_prof_begin(b, JDFT_K_COLS_FWD, st);
    SPEC_SWITCH(L, b->opt_force_generic, {
        if constexpr (jcols::Cfg<LT>::ok) {
            using F = jcols::Cfg<LT>;
            using FR = jcols::Cfg<LT, true>;
            // reversed plan (16, 8) with the radix-8 last pass pruned, when no sphere point has |m2| >= 2 (L / 8); measured:
            // 1.116 -> 0.949 ms at 128 (0.78 -> 0.91 of the HBM roofline), no gain at 80 = 8 x 10 (kept on the forward plan)
            constexpr bool kRev = F::NP == 2 && F::R0 == 8 && F::R1 == 16;
            const bool rev = kRev && b->opt_prune && b->mmin[2] > -2 * (LT / 8) && b->mmax[2] < 2 * (LT / 8);
            // ... and its last pass writing the sphere straight from registers ("cols_direct"): 0.951 -> 0.878 ms at 128
            // (0.92 -> 0.99 of the HBM roofline); on the forward plans the same change is slower (216: 1.85 -> 2.03 ms,
            // 80: 0.0635 -> 0.0697 ms: radix-6 / radix-10 last passes with lanes along the pencil), so they keep the gather
            if constexpr (kRev) {
                if (rev) {
                    dim3 g2((b->ncol + FR::T - 1) / FR::T, nbt);
                    if (b->opt_cols_direct) {
                        JDFT_CUDA(ensure_smem(jcols::k_cols_fwd_tuned<LT, true, true>, FR::smem, b->device));
                        jcols::k_cols_fwd_tuned<LT, true, true><<<g2, FR::NT, FR::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo,
                                                                                         W1, scale, kin, b->d_ke, C, out);
                    } else {
                        JDFT_CUDA(ensure_smem(jcols::k_cols_fwd_tuned<LT, true>, FR::smem, b->device));
                        jcols::k_cols_fwd_tuned<LT, true><<<g2, FR::NT, FR::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, W1,
                                                                                   scale, kin, b->d_ke, C, out);
                    }
                }
            }
            if (!rev) {
                JDFT_CUDA(ensure_smem(jcols::k_cols_fwd_tuned<LT>, F::smem, b->device));
                dim3 g2((b->ncol + F::T - 1) / F::T, nbt);
                jcols::k_cols_fwd_tuned<LT><<<g2, F::NT, F::smem, st>>>(b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, W1,
                                                                   scale, kin, b->d_ke, C, out);
            }
        } else {
            JDFT_CUDA(ensure_smem(k_cols_fwd<LT>, smem, b->device));
            k_cols_fwd<LT><<<grid, ColsNT<LT>::v, smem, st>>>(b->plan[2], b->d_tw[2], b->ncol, b->nG, b->d_col_n0, b->d_col_m2lo, W1,
                                                    scale, kin, b->d_ke, C, out);
    }
    });
    jdft_prof_end(b, JDFT_K_COLS_FWD, st);
    JDFT_LAUNCH_CHECK("k_cols_fwd");
    return JDFT_OK;
}

template <bool FWD>
int launch_rows(const jdft_basis *b, int nbt, double2 *W1, double2 *W2, cudaStream_t st) {
    const int L = b->S[1];
    const size_t smem = 2 * (size_t)L * kT * sizeof(double2) + (size_t)L * sizeof(int);
    dim3 grid((b->S[2] + kT - 1) / kT, b->npl, nbt);
    jdft_prof_begin(b, FWD ? JDFT_K_ROWS_FWD : JDFT_K_ROWS_INV, st);
    SPEC_SWITCH(L, b->opt_force_generic, {
        if constexpr (LT == 128) {  // measured: 1.07 -> 0.94 ms at 128 (91 % of the HBM roofline), slower at 80
            if (b->S[2] % 2 == 0 && b->opt_pair && aligned32(W1, W2)) {
                using C = Tuned<LT>;
                const size_t sm2 = (size_t)L * C::T * sizeof(double2);
                JDFT_CUDA(ensure_smem(k_rows_hyb<LT, FWD>, sm2, b->device));
                dim3 g2((b->S[2] + C::T - 1) / C::T, b->npl, nbt);
                k_rows_hyb<LT, FWD><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[1], b->S[2], b->npl, b->ncol, b->d_rowcol, W1, W2);
                jdft_prof_end(b, FWD ? JDFT_K_ROWS_FWD : JDFT_K_ROWS_INV, st);
                JDFT_LAUNCH_CHECK("k_rows_hyb");
                return JDFT_OK;
            }
        }
        if constexpr (Tuned<LT>::ok) {
            using C = Tuned<LT>;
            const size_t sm2 = (size_t)L * C::T * sizeof(double2);
            JDFT_CUDA(ensure_smem(k_rows_tuned<LT, FWD>, sm2, b->device));
            dim3 g2((b->S[2] + C::T - 1) / C::T, b->npl, nbt);
            k_rows_tuned<LT, FWD><<<g2, C::NT, sm2, st>>>(b->d_tw[1], b->S[2], b->npl, b->ncol, b->d_rowcol, W1, W2);
        } else {
            JDFT_CUDA(ensure_smem(k_rows<LT, FWD>, smem, b->device));
            k_rows<LT, FWD><<<grid, kNT, smem, st>>>(b->plan[1], b->d_tw[1], b->S[2], b->npl, b->ncol, b->d_rowcol, W1, W2);
        }
    });
    jdft_prof_end(b, FWD ? JDFT_K_ROWS_FWD : JDFT_K_ROWS_INV, st);
    JDFT_LAUNCH_CHECK("k_rows");
    return JDFT_OK;
}

// occupied planes: i0 in [0, m0lo + npl) and [L + m0lo, L); the pruned radix-8 butterflies need [2 R2, 6 R2) empty
template <class C>
bool planes_prunable(const jdft_basis *b, int L) {
    return C::R1 == 8 && b->opt_prune && b->m0lo < 0 && b->m0lo + b->npl <= 2 * C::R2 && L + b->m0lo >= 6 * C::R2;
}

// K3 through TMA (planes_tma.cuh): returns 1 if launched, 0 if this shape / pointer cannot take the path, < 0 on error
template <int LT>
int try_planes_tma(const jdft_basis *b, int nbt, double2 *W2, const double *V, cudaStream_t st) {
    if constexpr (!PlanesTma<LT>::ok) {
        return 0;
    } else {
        using Q = PlanesTma<LT>;
        const int S1 = b->S[1], S2 = b->S[2], npl = b->npl;
        JdftEncodeTiledFn enc = jdft_tensor_map_encoder();
        const size_t smem = Q::smem_bytes(npl);
        if (!enc || !b->opt_tma || npl > 256 || S1 > 65536 || smem > 200 * 1024 || (((uintptr_t)W2) & 15)) return 0;
        CUtensorMap tm;
        const cuuint64_t gdim[3] = {(cuuint64_t)2 * S2, (cuuint64_t)S1, (cuuint64_t)nbt * npl};
        const cuuint64_t gstr[2] = {(cuuint64_t)S2 * 16, (cuuint64_t)S1 * S2 * 16};
        const cuuint32_t box[3] = {32, 1, (cuuint32_t)npl}, estr[3] = {1, 1, 1};
        if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, W2, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return 0;
        const int ntx = (S2 + Q::T - 1) / Q::T;
        const int64_t ntiles = (int64_t)ntx * S1 * nbt;
        if (ntiles >= ((int64_t)1 << 31)) return 0;
        const int grid = (int)(ntiles < (int64_t)b->num_sms * Q::MINB ? ntiles : (int64_t)b->num_sms * Q::MINB);
        const bool pr = planes_prunable<Tuned<LT>>(b, LT);
        jdft_prof_begin(b, JDFT_K_PLANES, st);
        if (pr) {
            JDFT_CUDA(jdft_ensure_smem((const void *)k_planes_tma<LT, true>, smem, b->device));
            k_planes_tma<LT, true><<<grid, Q::NT, smem, st>>>(tm, b->d_tw[0], S1, S2, npl, b->d_planeof, V, ntx, (int)ntiles);
        } else {
            JDFT_CUDA(jdft_ensure_smem((const void *)k_planes_tma<LT, false>, smem, b->device));
            k_planes_tma<LT, false><<<grid, Q::NT, smem, st>>>(tm, b->d_tw[0], S1, S2, npl, b->d_planeof, V, ntx, (int)ntiles);
        }
        jdft_prof_end(b, JDFT_K_PLANES, st);
        JDFT_LAUNCH_CHECK("k_planes_tma");
        return 1;
    }
}

template <int MODE>
int launch_planes(const jdft_basis *b, int nbt, double2 *W2, const double *V, double2 *psi, cudaStream_t st) {
    const int L = b->S[0];
    const size_t smem = 2 * (size_t)L * kT * sizeof(double2) + (size_t)L * sizeof(int);
    dim3 grid((b->S[2] + kT - 1) / kT, b->S[1], nbt);
    if (MODE == 0 && b->opt_tma) {
        int took = 0;
        SPEC_SWITCH(L, b->opt_force_generic, { took = try_planes_tma<LT>(b, nbt, W2, V, st); });
        if (took != 0) return took < 0 ? took : JDFT_OK;
    }
    jdft_prof_begin(b, JDFT_K_PLANES, st);
    SPEC_SWITCH(L, b->opt_force_generic, {
        if constexpr (MODE == 0 && Pair<LT>::ok && LT == 72) {  // measured: +7 % at 72 (32 pencils/CTA), -12 % at 80 (16 pencils, 80 threads)
            if (b->S[2] % 2 == 0 && b->opt_pair && aligned32(W2) && (((uintptr_t)V) & 15) == 0) {
                using Q = Pair<LT>;
                const size_t sm2 = (size_t)Q::G * L * Q::T * sizeof(double2);
                dim3 g2((b->S[2] + Q::T - 1) / Q::T, (b->S[1] + Q::G - 1) / Q::G, nbt);
                if (planes_prunable<Tuned<LT>>(b, L)) {
                    JDFT_CUDA(ensure_smem(k_planes_fused2<LT, true>, sm2, b->device));
                    k_planes_fused2<LT, true><<<g2, Q::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, V);
                } else {
                    JDFT_CUDA(ensure_smem(k_planes_fused2<LT>, sm2, b->device));
                    k_planes_fused2<LT><<<g2, Q::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, V);
                }
                jdft_prof_end(b, JDFT_K_PLANES, st);
                JDFT_LAUNCH_CHECK("k_planes_fused2");
                return JDFT_OK;
            }
        }
        if constexpr (MODE != 0 && (LT == 128 || LT == 80)) {
            if (b->S[2] % 2 == 0 && b->opt_pair && aligned32(W2, psi)) {
                using C = Tuned<LT>;
                const size_t sm2 = (size_t)L * C::T * sizeof(double2);
                dim3 g2((b->S[2] + C::T - 1) / C::T, b->S[1], nbt);
                if (MODE == 1 && planes_prunable<C>(b, L)) {
                    JDFT_CUDA(ensure_smem(k_planes_io_hyb<LT, MODE, MODE == 1>, sm2, b->device));
                    k_planes_io_hyb<LT, MODE, MODE == 1><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, psi);
                } else {
                    JDFT_CUDA(ensure_smem(k_planes_io_hyb<LT, MODE>, sm2, b->device));
                    k_planes_io_hyb<LT, MODE><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, psi);
                }
                jdft_prof_end(b, JDFT_K_PLANES, st);
                JDFT_LAUNCH_CHECK("k_planes_io_hyb");
                return JDFT_OK;
            }
        }
        if constexpr (MODE == 0 && (LT == 128 || LT == 80)) {  // 72 runs the full pair kernel above (hybrid measured slower)
            if (b->S[2] % 2 == 0 && b->opt_pair && aligned32(W2)) {
                using C = Tuned<LT>;
                const size_t sm2 = (size_t)L * C::T * sizeof(double2);
                dim3 g2((b->S[2] + C::T - 1) / C::T, b->S[1], nbt);
                if (planes_prunable<C>(b, L)) {
                    JDFT_CUDA(ensure_smem(k_planes_fused_h<LT, true>, sm2, b->device));
                    k_planes_fused_h<LT, true><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, V);
                } else {
                    JDFT_CUDA(ensure_smem(k_planes_fused_h<LT>, sm2, b->device));
                    k_planes_fused_h<LT><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, V);
                }
                jdft_prof_end(b, JDFT_K_PLANES, st);
                JDFT_LAUNCH_CHECK("k_planes_fused_h");
                return JDFT_OK;
            }
        }
        if constexpr (MODE == 0 && Tuned<LT>::ok) {
            using C = Tuned<LT>;
            const size_t sm2 = (size_t)L * C::T * sizeof(double2);
            JDFT_CUDA(ensure_smem(k_planes_fused<LT>, sm2, b->device));
            dim3 g2((b->S[2] + C::T - 1) / C::T, b->S[1], nbt);
            k_planes_fused<LT><<<g2, C::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, V);
        } else {
            JDFT_CUDA(ensure_smem(k_planes<LT, MODE>, smem, b->device));
            k_planes<LT, MODE><<<grid, kNT, smem, st>>>(b->plan[0], b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, W2, V, psi);
        }
    });
    jdft_prof_end(b, JDFT_K_PLANES, st);
    JDFT_LAUNCH_CHECK("k_planes");
    return JDFT_OK;
}

int check_common(const jdft_basis *b, const void *in, const void *out, int nb, const char *who) {
    if (!b) return jdft_fail(JDFT_EINVAL, "%s: null basis", who);
    if (nb < 0) return jdft_fail(JDFT_EINVAL, "%s: negative band count", who);
    if (nb > 0 && (!in || !out)) return jdft_fail(JDFT_EINVAL, "%s: null data pointer", who);
    if ((((uintptr_t)in) | ((uintptr_t)out)) & 15) return jdft_fail(JDFT_EINVAL, "%s: data pointer not 16-byte aligned", who);
    return JDFT_OK;
}

}  // namespace

// HC = I^+ (Vloc .* I C) + Omega ke C  for all nb bands, in band batches
int jdft_local_H(const jdft_basis *b, const double *Vloc, const double *C_, int nb, double *HC_, cudaStream_t st,
                 size_t ws_offset, double scale, double kin) {
    if (kin < 0.0) kin = b->volume;
    const int nbatch = jdft_band_batch(b, nb, ws_offset);
    if (nb > 0 && nbatch == 0) return jdft_fail(JDFT_EWORKSPACE, "apply_H: workspace missing or smaller than one band (%zu bytes)", jdft_fft_bytes_per_band(b));
    const double2 *C = reinterpret_cast<const double2 *>(C_);
    double2 *HC = reinterpret_cast<double2 *>(HC_);
    int rc;
    for (int b0 = 0; b0 < nb; b0 += nbatch) {
        const int nbt = nb - b0 < nbatch ? nb - b0 : nbatch;
        const Bufs w = carve(b, nbatch, ws_offset);
        const double2 *Cb = C + (size_t)b0 * b->nG;
        if ((rc = launch_cols_inv(b, Cb, nbt, w.W1, st))) return rc;
        if ((rc = launch_rows<false>(b, nbt, w.W1, w.W2, st))) return rc;
        if ((rc = launch_planes<0>(b, nbt, w.W2, Vloc, nullptr, st))) return rc;
        if ((rc = launch_rows<true>(b, nbt, w.W1, w.W2, st))) return rc;
        if ((rc = launch_cols_fwd(b, w.W1, nbt, scale, kin, Cb, HC + (size_t)b0 * b->nG, st))) return rc;
    }
    return JDFT_OK;
}

extern "C" int jdft_apply_I(const jdft_basis *b, const double *C_, int nb, double *psi_, jdft_stream s) {
    int rc = check_common(b, C_, psi_, nb, "apply_I");
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)s;
    const int nbatch = jdft_band_batch(b, nb);
    if (nb > 0 && nbatch == 0) return jdft_fail(JDFT_EWORKSPACE, "apply_I: workspace missing or smaller than one band");
    const double2 *C = reinterpret_cast<const double2 *>(C_);
    double2 *psi = reinterpret_cast<double2 *>(psi_);
    for (int b0 = 0; b0 < nb; b0 += nbatch) {
        const int nbt = nb - b0 < nbatch ? nb - b0 : nbatch;
        const Bufs w = carve(b, nbatch);
        if ((rc = launch_cols_inv(b, C + (size_t)b0 * b->nG, nbt, w.W1, st))) return rc;
        if ((rc = launch_rows<false>(b, nbt, w.W1, w.W2, st))) return rc;
        if ((rc = launch_planes<1>(b, nbt, w.W2, nullptr, psi + (size_t)b0 * b->N, st))) return rc;
    }
    return JDFT_OK;
}

static int idag_scaled(const jdft_basis *b, const double *psi_, int nb, double *C_, double scale, jdft_stream s,
                       const char *who) {
    int rc = check_common(b, psi_, C_, nb, who);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)s;
    const int nbatch = jdft_band_batch(b, nb);
    if (nb > 0 && nbatch == 0) return jdft_fail(JDFT_EWORKSPACE, "%s: workspace missing or smaller than one band", who);
    double2 *psi = reinterpret_cast<double2 *>(const_cast<double *>(psi_));
    double2 *C = reinterpret_cast<double2 *>(C_);
    for (int b0 = 0; b0 < nb; b0 += nbatch) {
        const int nbt = nb - b0 < nbatch ? nb - b0 : nbatch;
        const Bufs w = carve(b, nbatch);
        if ((rc = launch_planes<2>(b, nbt, w.W2, nullptr, psi + (size_t)b0 * b->N, st))) return rc;
        if ((rc = launch_rows<true>(b, nbt, w.W1, w.W2, st))) return rc;
        if ((rc = launch_cols_fwd(b, w.W1, nbt, scale, 0.0, C + (size_t)b0 * b->nG, C + (size_t)b0 * b->nG, st))) return rc;
    }
    return JDFT_OK;
}

extern "C" int jdft_apply_Idag(const jdft_basis *b, const double *psi, int nb, double *C, jdft_stream s) {
    return idag_scaled(b, psi, nb, C, 1.0, s, "apply_Idag");
}

extern "C" int jdft_apply_J(const jdft_basis *b, const double *psi, int nb, double *C, jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "apply_J: null basis");
    return idag_scaled(b, psi, nb, C, 1.0 / (double)b->N, s, "apply_J");
}

extern "C" int jdft_density(const jdft_basis *b, const double *C_, int nb, const double *f, double *n, int accumulate,
                            jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "density: null basis");
    if (nb < 0) return jdft_fail(JDFT_EINVAL, "density: negative band count");
    if (!n || (nb > 0 && (!C_ || !f))) return jdft_fail(JDFT_EINVAL, "density: null data pointer");
    if (((uintptr_t)C_) & 15) return jdft_fail(JDFT_EINVAL, "density: C not 16-byte aligned");
    cudaStream_t st = (cudaStream_t)s;
    if (nb == 0) {
        if (!accumulate) JDFT_CUDA(cudaMemsetAsync(n, 0, (size_t)b->N * 8, st));
        return JDFT_OK;
    }
    const int nbatch = jdft_band_batch(b, nb);
    if (nbatch == 0) return jdft_fail(JDFT_EWORKSPACE, "density: workspace missing or smaller than one band");
    const double2 *C = reinterpret_cast<const double2 *>(C_);
    const int L = b->S[0];
    const size_t smem = 2 * (size_t)L * kT * sizeof(double2) + (size_t)L * kT * sizeof(double) + (size_t)L * sizeof(int);
    dim3 grid((b->S[2] + kT - 1) / kT, b->S[1]);
    int rc;
    for (int b0 = 0; b0 < nb; b0 += nbatch) {
        const int nbt = nb - b0 < nbatch ? nb - b0 : nbatch;
        const Bufs w = carve(b, nbatch);
        if ((rc = launch_cols_inv(b, C + (size_t)b0 * b->nG, nbt, w.W1, st))) return rc;
        if ((rc = launch_rows<false>(b, nbt, w.W1, w.W2, st))) return rc;
        const int acc = (accumulate || b0 > 0) ? 1 : 0;
        jdft_prof_begin(b, JDFT_K_PLANES, st);
        SPEC_SWITCH(L, b->opt_force_generic, {
            bool hyb = false;
            if constexpr (LT == 128) {  // measured: 3.20 -> 2.73 ms on config 3; slower at 80
                if (b->S[2] % 2 == 0 && b->opt_pair && aligned32(w.W2)) {
                    using C = Tuned<LT>;
                    const size_t sm2 = (size_t)L * C::T * sizeof(double2);
                    dim3 g2((b->S[2] + C::T - 1) / C::T, b->S[1]);
                    if (planes_prunable<C>(b, L)) {
                        JDFT_CUDA(ensure_smem(k_planes_density_hyb<LT, true>, sm2, b->device));
                        k_planes_density_hyb<LT, true><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof,
                                                                                     w.W2, f + b0, nbt, n, acc);
                    } else {
                        JDFT_CUDA(ensure_smem(k_planes_density_hyb<LT>, sm2, b->device));
                        k_planes_density_hyb<LT><<<g2, Hyb<LT>::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, w.W2,
                                                                          f + b0, nbt, n, acc);
                    }
                    hyb = true;
                }
            }
            if (hyb) {
            } else if constexpr (Tuned<LT>::ok) {
                using C = Tuned<LT>;
                const size_t sm2 = (size_t)L * C::T * sizeof(double2);
                JDFT_CUDA(ensure_smem(k_planes_density_tuned<LT>, sm2, b->device));
                dim3 g2((b->S[2] + C::T - 1) / C::T, b->S[1]);
                k_planes_density_tuned<LT><<<g2, C::NT, sm2, st>>>(b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, w.W2,
                                                                   f + b0, nbt, n, acc);
            } else {
                JDFT_CUDA(ensure_smem(k_planes_density<LT>, smem, b->device));
                k_planes_density<LT><<<grid, kNT, smem, st>>>(b->plan[0], b->d_tw[0], b->S[1], b->S[2], b->npl, b->d_planeof, w.W2,
                                                              f + b0, nbt, n, acc);
            }
        });
        jdft_prof_end(b, JDFT_K_PLANES, st);
        JDFT_LAUNCH_CHECK("k_planes_density");
    }
    return JDFT_OK;
}

namespace {
Mat3 mat3_of(const jdft_basis *b) {
    Mat3 m;
    for (int i = 0; i < 9; i++) m.g[i] = b->G[i];
    for (int i = 0; i < 3; i++) m.k[i] = b->k[i];
    return m;
}
int elementwise_grid(const jdft_basis *b, int64_t total) {
    const int64_t blocks = (total + 255) / 256, cap = (int64_t)b->num_sms * 16;
    return (int)(blocks > cap ? cap : blocks);
}
int launch_gradient(const jdft_basis *b, const double *C, int nb, double *out, cudaStream_t st) {
    const int64_t total = (int64_t)nb * b->nG;
    jdft_prof_begin(b, JDFT_K_DIAG, st);
    k_gradient<<<elementwise_grid(b, total), 256, 0, st>>>(mat3_of(b), b->d_iG, b->nG, total, reinterpret_cast<const double2 *>(C),
                                                        reinterpret_cast<double2 *>(out));
    jdft_prof_end(b, JDFT_K_DIAG, st);
    JDFT_LAUNCH_CHECK("k_gradient");
    return JDFT_OK;
}
int launch_divergence(const jdft_basis *b, const double *X, int nb, double f, double *out, cudaStream_t st) {
    const int64_t total = (int64_t)nb * b->nG;
    jdft_prof_begin(b, JDFT_K_DIAG, st);
    k_divergence<<<elementwise_grid(b, total), 256, 0, st>>>(mat3_of(b), b->d_iG, b->nG, total, f, reinterpret_cast<const double2 *>(X),
                                                          reinterpret_cast<double2 *>(out));
    jdft_prof_end(b, JDFT_K_DIAG, st);
    JDFT_LAUNCH_CHECK("k_divergence");
    return JDFT_OK;
}
}  // namespace

extern "C" int jdft_gradient(const jdft_basis *b, const double *C, int nb, double *out, jdft_stream s) {
    int rc = check_common(b, C, out, nb, "gradient");
    if (rc) return rc;
    if (nb == 0) return JDFT_OK;
    return launch_gradient(b, C, nb, out, (cudaStream_t)s);
}

extern "C" int jdft_divergence(const jdft_basis *b, const double *X, int nb, double *out, jdft_stream s) {
    int rc = check_common(b, X, out, nb, "divergence");
    if (rc) return rc;
    if (nb == 0) return JDFT_OK;
    return launch_divergence(b, X, nb, 1.0, out, (cudaStream_t)s);
}

// Listing 1 of the paper: hessian(phi) = (-1/4 pi) divergence(J(epsilon * I(gradient(phi)))).  The three gradient
// components run through the fused pruned pipeline as 3 nb "bands" (epsilon multiply inside K3, 1/N of J in K5's
// gather); the component block lives at the front of the workspace and is transformed in place.
extern "C" int jdft_pcm_hessian(const jdft_basis *b, const double *epsilon, const double *phi, int nb, double *out,
                                jdft_stream s) {
    int rc = check_common(b, phi, out, nb, "pcm_hessian");
    if (rc) return rc;
    if (!epsilon) return jdft_fail(JDFT_EINVAL, "pcm_hessian: null epsilon");
    if (nb == 0) return JDFT_OK;
    cudaStream_t st = (cudaStream_t)s;
    const size_t gbytes = (((size_t)3 * nb * b->nG * 16) + 255) & ~(size_t)255;
    if (!b->ws || jdft_band_batch(b, 3 * nb, gbytes) == 0)
        return jdft_fail(JDFT_EWORKSPACE, "pcm_hessian: workspace must hold 3 nb nG c128 (%zu bytes) plus one band of FFT scratch", gbytes);
    double *g = static_cast<double *>(b->ws);
    if ((rc = launch_gradient(b, phi, nb, g, st))) return rc;
    if ((rc = jdft_local_H(b, epsilon, g, 3 * nb, g, st, gbytes, 1.0 / (double)b->N, 0.0))) return rc;
    return launch_divergence(b, g, nb, -1.0 / (4.0 * M_PI), out, st);
}

// Listing 1 on REAL fields in half-sphere storage (include/jdft.h): 3 nb real gradient components travel as
// ceil(3 nb / 2) complex fields through the fused pruned pipeline -- half the FFT work and bytes of jdft_pcm_hessian.
extern "C" int jdft_pcm_hessian_real(const jdft_basis *b, const double *epsilon, const double *phi_h, int nb, double *out_h,
                                     jdft_stream s) {
    int rc = check_common(b, phi_h, out_h, nb, "pcm_hessian_real");
    if (rc) return rc;
    if (!epsilon) return jdft_fail(JDFT_EINVAL, "pcm_hessian_real: null epsilon");
    if (b->k[0] != 0.0 || b->k[1] != 0.0 || b->k[2] != 0.0 || b->nG % 2 == 0)
        return jdft_fail(JDFT_EINVAL, "pcm_hessian_real: half-sphere storage needs a Gamma-point basis (k = 0)");
    if (nb == 0) return JDFT_OK;
    cudaStream_t st = (cudaStream_t)s;
    const int npair = (3 * nb + 1) / 2;
    const size_t zbytes = (((size_t)npair * b->nG * 16) + 255) & ~(size_t)255;
    if (!b->ws || jdft_band_batch(b, npair, zbytes) == 0)
        return jdft_fail(JDFT_EWORKSPACE, "pcm_hessian_real: workspace must hold ceil(3 nb / 2) nG c128 (%zu bytes) plus one band of FFT scratch", zbytes);
    double *Z = static_cast<double *>(b->ws);
    jdft_prof_begin(b, JDFT_K_DIAG, st);
    k_grad_pack_real<<<elementwise_grid(b, (int64_t)npair * b->nG), 256, 0, st>>>(mat3_of(b), b->d_iG, b->nG, nb, npair,
                                                                                 reinterpret_cast<const double2 *>(phi_h),
                                                                                 reinterpret_cast<double2 *>(Z));
    jdft_prof_end(b, JDFT_K_DIAG, st);
    JDFT_LAUNCH_CHECK("k_grad_pack_real");
    if ((rc = jdft_local_H(b, epsilon, Z, npair, Z, st, zbytes, 1.0 / (double)b->N, 0.0))) return rc;
    jdft_prof_begin(b, JDFT_K_DIAG, st);
    k_unpack_div_real<<<elementwise_grid(b, (int64_t)nb * ((b->nG + 1) / 2)), 256, 0, st>>>(
        mat3_of(b), b->d_iG, b->nG, nb, -1.0 / (4.0 * M_PI), reinterpret_cast<const double2 *>(Z), reinterpret_cast<double2 *>(out_h));
    jdft_prof_end(b, JDFT_K_DIAG, st);
    JDFT_LAUNCH_CHECK("k_unpack_div_real");
    return JDFT_OK;
}

static int diag_op(const jdft_basis *b, const double *C, int nb, double *out, double f0, double f1, jdft_stream s,
                   const char *who) {
    int rc = check_common(b, C, out, nb, who);
    if (rc) return rc;
    const int64_t total = (int64_t)nb * b->nG;
    if (total == 0) return JDFT_OK;
    jdft_prof_begin(b, JDFT_K_DIAG, (cudaStream_t)s);
    k_diag<<<elementwise_grid(b, total), 256, 0, (cudaStream_t)s>>>(b->nG, total, f0, f1, b->d_ke, reinterpret_cast<const double2 *>(C),
                                                      reinterpret_cast<double2 *>(out));
    jdft_prof_end(b, JDFT_K_DIAG, (cudaStream_t)s);
    JDFT_LAUNCH_CHECK(who);
    return JDFT_OK;
}

extern "C" int jdft_apply_L(const jdft_basis *b, const double *C, int nb, double *LC, jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "apply_L: null basis");
    return diag_op(b, C, nb, LC, 0.0, -2.0 * b->volume, s, "apply_L");
}

extern "C" int jdft_apply_O(const jdft_basis *b, const double *C, int nb, double *OC, jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "apply_O: null basis");
    return diag_op(b, C, nb, OC, b->volume, 0.0, s, "apply_O");
}
