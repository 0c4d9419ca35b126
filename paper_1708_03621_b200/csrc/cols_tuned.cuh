// Tuned column kernels (K1: scatter + inverse FFT along axis 2; K5: forward FFT along axis 2 + gather + kinetic)
// for the lengths that have compile-time plans (fft.cuh SpecPlan).  Included by local.cu only.
//
// Both kernels were bound by shared-memory bandwidth, not HBM (ncu of the staged variants: L1/shared pipe 61-85 %, DRAM 38-57 %), so the design
// goal is fewer shared-memory tile transfers than the ping-pong engine needs:
//   K1  no zero fill (the first pass tests "is this row inside the column's sphere run" instead), and the last pass
//       writes W1 straight from registers with the lanes of a warp running along the pencil (consecutive rows ->
//       128..512-byte global segments), so there is no transposition through shared memory;
//   K5  the first pass reads W1 straight from global memory the same way (lanes along the pencil) and writes its
//       butterflies into an XOR-swizzled tile, so the load staging disappears as well.
// Tiles are [L][TP] c128 with TP = T + 1 (T pencils per CTA); the swizzled tile uses stride T inside the same buffer.
// DIRECT variants (option "cols_direct", default on where measured faster): the sphere side goes without shared memory too --
// K1's first pass reads each column's run (contiguous in n) straight into its butterflies, K5's pruned last pass at
// length 128 writes the run straight from registers with the kinetic term; lanes run along one column's rows, so the
// global accesses are contiguous segments and the column search, the scatter / gather crossing and a barrier go away
// (config 5: K1 0.844 -> 0.705 ms = 0.76 -> 0.90 of the HBM roofline; K5 0.951 -> 0.878 ms = 0.92 -> 0.99).
#pragma once
#include "fft.cuh"

namespace jcols {
using namespace jfft;

// REV (two-pass plans only): the radices in reversed order (128 = 16 x 8 instead of 8 x 16), so that the LAST pass is the
// radix-8 one and can be output-pruned (K5) the way K1's first pass is input-pruned.
template <int LT, bool REV = false>
struct Cfg {
    using P = SpecPlan<LT>;
    static constexpr int NP = P::npass;
    static constexpr bool ok = NP == 2 || NP == 3;
    static constexpr int R0 = (REV && NP == 2) ? P::r1 : P::r0, R1 = (REV && NP == 2) ? P::r0 : P::r1, R2 = P::r2;
    static constexpr int RL = NP == 3 ? R2 : R1;               // radix of the last pass
    static constexpr int T = NP == 3 ? 8 : 16;                  // pencils per CTA
    static constexpr int TP = T + 1;
    // resident CTAs per SM the register allocation is bounded for (latency-bound kernels: more warps in flight win)
    static constexpr int RMAX = R0 > R1 ? (R0 > R2 ? R0 : R2) : (R1 > R2 ? R1 : R2);
    static constexpr int FIT = ok ? 65536 / (T * (LT / R0) / ((NP == 2 && LT / R0 == 2 * (LT / RL)) ? 2 : 1) * (RMAX >= 15 ? 80 : (RMAX >= 12 ? 72 : 40))) : 1;
    static constexpr int MINB_DEF = FIT < 1 ? 1 : (FIT > 6 ? 6 : FIT);
    // measured choices for the lengths of the five workloads (profiles/), the rule for the rest
    static constexpr int MINB_INV = LT == 216 ? 5 : (LT == 128 ? 6 : MINB_DEF), MINB_FWD = REV ? 4 : (LT == 216 ? 4 : (LT == 128 ? 6 : MINB_DEF));
    static constexpr int NBL = ok ? LT / RL : 1;                // butterflies per pencil in the last pass
    static constexpr int NB0 = ok ? LT / R0 : 1;                // ... in the first pass
    // ONE swizzled tile [L][T]; the shared -> shared passes run in a single round (threads = their work items) and
    // in place: every thread reads its butterfly, barrier, writes it back
    // first pass in ROUNDS0 rounds: 2 when it has twice the butterflies of the last pass (128 = 8 x 16), so that no
    // thread idles in the (heavier) last pass; both rounds are read before the barrier of the in-place update
    static constexpr int ROUNDS0 = (NP == 2 && NB0 == 2 * NBL) ? 2 : 1;
    static constexpr int NT = T * NB0 / ROUNDS0;
    static constexpr int NB1 = ok ? LT / R1 : 1;                // butterflies per pencil in the middle pass (3-pass plans)
    static_assert(NP != 3 || NB1 * T == NT, "middle pass must be exactly one round");
    static constexpr size_t smem = (size_t)LT * T * sizeof(double2);
    // swizzled position of (row, pencil t): conflict-free for lanes along t, along butterflies and along rows
    static __device__ __forceinline__ int sw(int row, int t) { return row * T + (t ^ ((row + row / R0) & (T - 1))); }
};

__device__ __forceinline__ int wrap_row(int m, int L) {
    int r = m % L;
    return r < 0 ? r + L : r;
}

// column t of sphere entry n among the CTA's T columns: largest t with s_n0[t] <= n (branch-free binary search)
template <int T>
__device__ __forceinline__ int find_col(const int *s_n0, const int n) {
    int t = 0;
#pragma unroll
    for (int h = T / 2; h >= 1; h >>= 1)
        if (n >= s_n0[t + h]) t += h;
    return t;
}

template <int R, int SIGN>
__device__ __forceinline__ void tw_mul(double2 (&a)[R], const double2 *__restrict__ tw, const int pb) {
#pragma unroll
    for (int j = 1; j < R; j++) {
        double2 wv = __ldg(tw + pb * j);
        if (SIGN < 0) wv.y = -wv.y;
        a[j] = cmul(a[j], wv);
    }
}

// middle pass of a three-pass plan, in place in the swizzled tile, one round, pencil index fastest:
// radix R1, s = R0 (Stockham: rows bf + k NB1 -> rows q + pb R1 + s j, twiddle w^(pb j), q = bf mod s, pb = bf - q)
template <int LT, int SIGN>
__device__ __forceinline__ void mid_pass_inplace(double2 *X, const double2 *__restrict__ tw) {
    using F = Cfg<LT>;
    constexpr int R = F::R1, nbf = F::NB1, s = F::R0, T = F::T;
    const int t = threadIdx.x % T, bf = threadIdx.x / T;
    double2 a[R];
#pragma unroll
    for (int k = 0; k < R; k++) a[k] = X[F::sw(bf + k * nbf, t)];
    __syncthreads();
    Dft<R, SIGN>::run(a);
    const int q = bf % s, pb = bf - q;
    tw_mul<R, SIGN>(a, tw, pb);
#pragma unroll
    for (int j = 0; j < R; j++) X[F::sw(q + pb * R + s * j, t)] = a[j];
    __syncthreads();
}

// ------------------------------------------------------------------------------------------------ K1
// PR (radix-8 first pass only): every column's sphere run lies in rows [0, 2 NB0) u [6 NB0, L) (|m2| < 2 NB0, true for
// the cubic workloads of BASELINE.json), so inputs 2..5 of every first-pass butterfly are zero: they are neither read
// nor tested, and the butterfly is the pruned dft8_in0167 (16 instead of 24 complex additions).
template <int SIGN>
__device__ __forceinline__ void dft8_in0167_c(double2 (&a)[8]) {
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

// DIRECT: the first pass takes its inputs straight from the sphere (column t's run is contiguous in n; the lanes of a
// warp run along the butterfly index, i.e. along consecutive rows of one column -> contiguous global segments), so the
// scatter into the tile, its column search and two of the barriers disappear.
template <int LT, bool PR = false, bool DIRECT = false>
__global__ void __launch_bounds__(Cfg<LT>::NT, Cfg<LT>::MINB_INV) k_cols_inv_tuned(const double2 *__restrict__ tw, const int ncol,
                                                                const int64_t nG, const int *__restrict__ col_n0,
                                                                const int *__restrict__ col_m2lo,
                                                                const double2 *__restrict__ C, double2 *__restrict__ W1) {
    using F = Cfg<LT>;
    constexpr int T = F::T, TP = F::TP, NT = F::NT, L = LT, R0 = F::R0, R1 = F::R1, RL = F::RL, NBL = F::NBL, NB0 = F::NB0;
    extern __shared__ double2 smem[];
    double2 *X = smem;
    __shared__ int s_n0[T + 1], s_m2w[T];
    const int tid = threadIdx.x, c0 = blockIdx.x * T, b = blockIdx.y;
    const int nc = min(T, ncol - c0);
    if (tid <= T) s_n0[tid] = col_n0[min(c0 + tid, ncol)];
    if (tid < T) s_m2w[tid] = wrap_row(col_m2lo[min(c0 + tid, ncol - 1)], L);
    __syncthreads();
    const double2 *Cb = C + (size_t)b * nG;
    double2 *Wb = W1 + ((size_t)b * ncol + c0) * L;
    const int nbeg = s_n0[0], nend = s_n0[nc];
    if constexpr (DIRECT) {
        constexpr int RD = F::ROUNDS0;
        double2 a[RD][R0];
#pragma unroll
        for (int r = 0; r < RD; r++) {
            const int w = tid + r * NT;
            const int bf = w % NB0, t = w / NB0;
            const int m2w = s_m2w[t], n0 = s_n0[t], len = t < nc ? s_n0[t + 1] - n0 : 0;
#pragma unroll
            for (int k = 0; k < R0; k++) {
                if (PR && k >= 2 && k < 6) continue;
                int off = bf + k * NB0 - m2w;
                if (off < 0) off += L;
                a[r][k] = make_double2(0.0, 0.0);
                if (off < len) a[r][k] = Cb[n0 + off];
            }
        }
#pragma unroll
        for (int r = 0; r < RD; r++) {
            const int w = tid + r * NT;
            const int bf = w % NB0, t = w / NB0;
            if constexpr (PR && R0 == 8) dft8_in0167_c<+1>(a[r]);
            else Dft<R0, +1>::run(a[r]);
            tw_mul<R0, +1>(a[r], tw, bf);
#pragma unroll
            for (int j = 0; j < R0; j++) X[F::sw(bf * R0 + j, t)] = a[r][j];
        }
        __syncthreads();
    } else {
        // scatter the sphere runs of the nc columns (contiguous in n) into the tile; nothing else of it is read
        // (the sphere reads are issued four deep before the first dependent shared-memory store: their HBM latency was
        //  the largest single stall of the kernel in the ncu source page)
        constexpr int U = F::NP == 3 ? 1 : 4;   // measured: pays at 128 (0.874 -> 0.847 ms at U = 4) and 80, not at 216 (40 registers)
        for (int e0 = tid; e0 < nend - nbeg; e0 += U * NT) {
            double2 v[U];
#pragma unroll
            for (int u = 0; u < U; u++) {
                const int e = e0 + u * NT;
                if (e < nend - nbeg) v[u] = Cb[nbeg + e];
            }
#pragma unroll
            for (int u = 0; u < U; u++) {
                const int e = e0 + u * NT;
                if (e < nend - nbeg) {
                    const int n = nbeg + e;
                    const int t = find_col<T>(s_n0, n);
                    int row = s_m2w[t] + (n - s_n0[t]);
                    if (row >= L) row -= L;
                    X[F::sw(row, t)] = v[u];
                }
            }
        }
        __syncthreads();
        // pass 0 (radix R0, s = 1), in place: rows bf + k NB0 (zero outside the run) -> rows bf R0 + j; every round is
        // read before the barrier, written after it
        {
            constexpr int RD = F::ROUNDS0;
            double2 a[RD][R0];
#pragma unroll
            for (int r = 0; r < RD; r++) {
                const int w = tid + r * NT;
                const int t = w % T, bf = w / T;
                const int m2w = s_m2w[t], len = t < nc ? s_n0[t + 1] - s_n0[t] : 0;
#pragma unroll
                for (int k = 0; k < R0; k++) {
                    if (PR && k >= 2 && k < 6) continue;
                    const int row = bf + k * NB0;
                    int off = row - m2w;
                    if (off < 0) off += L;
                    a[r][k] = make_double2(0.0, 0.0);
                    if (off < len) a[r][k] = X[F::sw(row, t)];
                }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < RD; r++) {
                const int w = tid + r * NT;
                const int t = w % T, bf = w / T;
                if constexpr (PR && R0 == 8) dft8_in0167_c<+1>(a[r]);
                else Dft<R0, +1>::run(a[r]);
                tw_mul<R0, +1>(a[r], tw, bf);
#pragma unroll
                for (int j = 0; j < R0; j++) X[F::sw(bf * R0 + j, t)] = a[r][j];
            }
        }
        __syncthreads();
    }
    {
        if constexpr (F::NP == 3) mid_pass_inplace<LT, +1>(X, tw);
        // last pass (radix RL): lanes run along the pencil, outputs go straight to W1[column][row]
        for (int w = tid; w < NBL * T; w += NT) {
            const int bf = w % NBL, t = w / NBL;
            double2 a[RL];
#pragma unroll
            for (int k = 0; k < RL; k++) a[k] = X[F::sw(bf + k * NBL, t)];
            Dft<RL, +1>::run(a);
            if (t < nc) {
#pragma unroll
                for (int j = 0; j < RL; j++) Wb[(size_t)t * L + bf + NBL * j] = a[j];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ K5
// out[b][n] = scale * (F_2 W1)[column of n][m2 of n]  (+ kin * ke[n] * C[b][n])
template <int SIGN>
__device__ __forceinline__ void dft8_out0167_c(double2 (&a)[8]) {   // outputs 0, 1, 6, 7 of the length-8 DFT (a[2..5] undefined on exit)
    const double2 s0 = cadd(a[0], a[4]), s1 = cadd(a[1], a[5]), s2 = cadd(a[2], a[6]), s3 = cadd(a[3], a[7]);
    const double2 d0 = csub(a[0], a[4]), d1 = csub(a[1], a[5]), d2 = csub(a[2], a[6]), d3 = csub(a[3], a[7]);
    const double2 j2 = mul_i<SIGN>(d2), j3 = mul_i<SIGN>(d3);
    a[0] = cadd(cadd(s0, s2), cadd(s1, s3));
    a[6] = csub(csub(s0, s2), mul_i<SIGN>(csub(s1, s3)));
    a[1] = cadd(cadd(d0, j2), mul_w<SIGN, 1, 8>(cadd(d1, j3)));
    a[7] = cadd(csub(d0, j2), mul_w<SIGN, 7, 8>(csub(d1, j3)));
}

// REV = true: reversed radix order with the radix-8 LAST pass pruned to outputs 0, 1, 6, 7 (rows [2 NBL, 6 NBL) hold no
// sphere point, the gather never reads them); the launcher checks |m2| < 2 NBL.
// DIRECT: the last pass runs with the lanes of a warp along the pencil and writes the sphere run of its column straight from
// registers (consecutive rows of a column are consecutive n), with the kinetic term; the in-place write-back, the
// gather with its column search and one barrier disappear.
template <int LT, bool REV = false, bool DIRECT = false>
__global__ void __launch_bounds__(Cfg<LT, REV>::NT, Cfg<LT, REV>::MINB_FWD) k_cols_fwd_tuned(const double2 *__restrict__ tw, const int ncol,
                                                                const int64_t nG, const int *__restrict__ col_n0,
                                                                const int *__restrict__ col_m2lo,
                                                                const double2 *__restrict__ W1, const double scale,
                                                                const double kin, const double *__restrict__ ke,
                                                                const double2 *__restrict__ C, double2 *__restrict__ outC) {
    using F = Cfg<LT, REV>;
    constexpr int T = F::T, TP = F::TP, NT = F::NT, L = LT, R0 = F::R0, R1 = F::R1, RL = F::RL, NBL = F::NBL, NB0 = F::NB0;
    static_assert(!REV || (F::NP == 2 && RL == 8), "the reversed plan ends with the radix-8 pass");
    extern __shared__ double2 smem[];
    double2 *X = smem;
    __shared__ int s_n0[T + 1], s_m2w[T];
    const int tid = threadIdx.x, c0 = blockIdx.x * T, b = blockIdx.y;
    const int nc = min(T, ncol - c0);
    for (int i = tid; i <= T; i += NT) s_n0[i] = col_n0[min(c0 + i, ncol)];
    for (int i = tid; i < T; i += NT) s_m2w[i] = wrap_row(col_m2lo[min(c0 + i, ncol - 1)], L);
    if (kin != 0.0 && LT == 128) {   // measured: 1.126 -> 1.116 ms at 128; slower at 80 and 216
        // the gather at the end reads C and ke of this CTA's sphere run (contiguous in n) straight from HBM, and nothing
        // hides that latency there (ncu: 45 % of the warp samples on long-scoreboard stalls): ask L2 for those lines now,
        // one prefetch per thread, so they arrive while the transform runs
        const int pb = __ldg(col_n0 + c0), pe = __ldg(col_n0 + min(c0 + T, ncol));
        const char *pc = reinterpret_cast<const char *>(C + (size_t)b * nG + pb);
        const char *pk = reinterpret_cast<const char *>(ke + pb);
        const int nc_lines = ((pe - pb) * 16 + 127) / 128, nk_lines = ((pe - pb) * 8 + 127) / 128;
        for (int e = tid; e < nc_lines + nk_lines; e += NT) {
            const char *a = e < nc_lines ? pc + e * 128 : pk + (e - nc_lines) * 128;
            asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
        }
    }
    // pass 0 (radix R0, s = 1): lanes run along the pencil, inputs straight from W1[column][row]
    const double2 *Wb = W1 + ((size_t)b * ncol + c0) * L;
    {
        for (int w = tid; w < NB0 * T; w += NT) {
            const int bf = w % NB0, t = w / NB0;
            double2 a[R0];
#pragma unroll
            for (int k = 0; k < R0; k++) a[k] = t < nc ? Wb[(size_t)t * L + bf + k * NB0] : make_double2(0.0, 0.0);
            Dft<R0, -1>::run(a);
            tw_mul<R0, -1>(a, tw, bf);
#pragma unroll
            for (int j = 0; j < R0; j++) X[F::sw(bf * R0 + j, t)] = a[j];
        }
        __syncthreads();
        if constexpr (F::NP == 3) mid_pass_inplace<LT, -1>(X, tw);
        if constexpr (DIRECT) {
            const double2 *Cb = C + (size_t)b * nG;
            double2 *Ob = outC + (size_t)b * nG;
            for (int w = tid; w < NBL * T; w += NT) {
                const int bf = w % NBL, t = w / NBL;
                double2 a[RL];
#pragma unroll
                for (int k = 0; k < RL; k++) a[k] = X[F::sw(bf + k * NBL, t)];
                const int m2w = s_m2w[t], n0 = s_n0[t], len = t < nc ? s_n0[t + 1] - n0 : 0;
                if constexpr (REV) dft8_out0167_c<-1>(a);
                else Dft<RL, -1>::run(a);
                constexpr int J4 = 4;   // outputs whose C / ke reads are in flight together
#pragma unroll
                for (int j0 = 0; j0 < (REV ? J4 : RL); j0 += J4) {   // REV: the one chunk of outputs 0, 1, 6, 7
                    double2 c[J4];
                    double f[J4];
                    int n[J4];
#pragma unroll
                    for (int u = 0; u < J4; u++) {
                        const int j = REV ? (u < 2 ? u : u + 4) : j0 + u;
                        c[u] = make_double2(0.0, 0.0);
                        f[u] = 0.0;
                        n[u] = -1;
                        if (j < RL) {
                            int off = bf + NBL * j - m2w;
                            if (off < 0) off += L;
                            if (off < len) {
                                n[u] = n0 + off;
                                if (kin != 0.0) {
                                    c[u] = Cb[n[u]];
                                    f[u] = kin * ke[n[u]];
                                }
                            }
                        }
                    }
#pragma unroll
                    for (int u = 0; u < J4; u++) {
                        const int j = REV ? (u < 2 ? u : u + 4) : j0 + u;
                        if (j < RL && n[u] >= 0) {
                            double2 v = a[j];
                            v.x = fma(f[u], c[u].x, v.x * scale);
                            v.y = fma(f[u], c[u].y, v.y * scale);
                            Ob[n[u]] = v;
                        }
                    }
                }
            }
            return;
        }
        // last pass (radix RL), in place: a thread reads and writes the same rows bf + NBL k of its pencil
        for (int w = tid; w < NBL * T; w += NT) {
            const int t = w % T, bf = w / T;
            double2 a[RL];
#pragma unroll
            for (int k = 0; k < RL; k++) a[k] = X[F::sw(bf + k * NBL, t)];
            if constexpr (REV) dft8_out0167_c<-1>(a);
            else Dft<RL, -1>::run(a);
#pragma unroll
            for (int j = 0; j < RL; j++) {
                if (REV && j >= 2 && j < 6) continue;
                X[F::sw(bf + NBL * j, t)] = a[j];
            }
        }
    }
    __syncthreads();
    // gather the sphere runs (contiguous in n) and add the kinetic term
    const int nbeg = s_n0[0], nend = s_n0[nc];
    const double2 *Cb = C + (size_t)b * nG;
    double2 *Ob = outC + (size_t)b * nG;
    constexpr int U = LT == 128 ? 4 : 1;   // global reads of C and ke U deep, then the shared-memory gathers and the stores
    for (int e0 = tid; e0 < nend - nbeg; e0 += U * NT) {
        double2 c[U];
        double f[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int e = e0 + u * NT;
            c[u] = make_double2(0.0, 0.0);
            f[u] = 0.0;
            if (kin != 0.0 && e < nend - nbeg) {
                c[u] = Cb[nbeg + e];
                f[u] = kin * ke[nbeg + e];
            }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int e = e0 + u * NT;
            if (e < nend - nbeg) {
                const int n = nbeg + e;
                const int t = find_col<T>(s_n0, n);
                int row = s_m2w[t] + (n - s_n0[t]);
                if (row >= L) row -= L;
                double2 v = X[F::sw(row, t)];
                v.x = fma(f[u], c[u].x, v.x * scale);
                v.y = fma(f[u], c[u].y, v.y * scale);
                Ob[n] = v;
            }
        }
    }
}

}  // namespace jcols
