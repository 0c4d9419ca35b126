// Complex FP64 GEMMs on the FP64 tensor pipe (DMMA, mma.sync.m8n8k4.f64) for the nonlocal projectors and the
// subspace overlap.  tcgen05 has no FP64 kind, so on sm_100a the FP64 tensor path is
// the warp-level DMMA; one complex MAC tile = four real DMMAs (Cr += ArBr -/+ AiBi, Ci += ArBi +/- AiBr) in the 4M
// kernels, THREE in the 3M (Karatsuba) kernels that serve the large contractions (see k_gemm_dotk below).
//
//   k_gemm_dotk   Out[r][c] = sum_k X[r][k] * conj?(Y[c][k])     both operands K-contiguous (K = nG), split-K with
//                 a fixed-order reduction (deterministic, no atomics): P^+ C, C1^+ C2, and D.B for dense D
//   k_gemm_expand Out[r][n] (+)= sum_j A[r][j] * Pm[j][n]        K = nproj, n contiguous: P (D P^+ C)
//
//                 (epilogue: Out = A Pm + addscale Add, which serves HC += ..., and Omega C + ... of O_us)
//   k_splitk_reduce[_block]  fixed-order split-K reduction with the scale, the real diagonal or the per-atom block D
//
// Tiles: 64 x 64 per CTA (4M), 4 warps of 32 x 32 (4 x 4 DMMA tiles of 8 x 8); 64 x 48 (3M: three accumulator sets);
// BK = 8, 4-stage cp.async pipeline (6 stages in the 3M expand kernel).
// Shared-memory layout of a K-contiguous operand: per group of 4 k, a dense [64 rows][4 k] block of c128
// (64 B per row, so the 8 lanes of a quarter-warp read 128 contiguous bytes), blocks skewed by 64 B.
#include <cstring>
#include "jdft_internal.h"
#include "tma.cuh"

namespace {

constexpr int BM = 64, BN = 64, BK = 8, STAGES = 4, NTHREADS = 128;
constexpr int KBLK_BYTES = 64 * 64 + 64;               // one [64][4] block + skew
constexpr int OPK_BYTES = (BK / 4) * KBLK_BYTES;        // K-contiguous operand, one stage
constexpr int PROW_BYTES = BN * 16 + 32;                // n-contiguous operand: row stride
constexpr int OPN_BYTES = BK * PROW_BYTES;

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, bool valid) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma(double &c0, double &c1, const double a, const double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// load one stage of a K-contiguous operand: rows [row0, row0+64) of M [nrows][ld], k in [k0, k0+BK), zero beyond kend/nrows
template <int BKT = BK, int ROWS = 64>   // ROWS: rows of the tile that are used (the rest of the 64-row block is never read)
__device__ __forceinline__ void load_opk(char *dst, const double2 *M, int64_t ld, int nrows, int row0, int64_t k0,
                                         int64_t kend, int tid) {
    static_assert((ROWS * BKT) % NTHREADS == 0, "whole rounds");
#pragma unroll
    for (int i = 0; i < (ROWS * BKT) / NTHREADS; i++) {
        const int e = tid + i * NTHREADS;
        const int r = e / BKT, kk = e % BKT;
        const int64_t k = k0 + kk;
        const bool ok = (row0 + r < nrows) && (k < kend);
        const double2 *src = ok ? M + (size_t)(row0 + r) * ld + k : M;
        cp_async16(dst + (kk / 4) * KBLK_BYTES + r * 64 + (kk % 4) * 16, src, ok);
    }
}

// ---------------------------------------------------------------------------------------------- dot-K GEMM
// BN_ = 64, or 48 when the column extent is a multiple of 48 but not of 64 (np = 288, 864: no zero-padded DMMAs)
// M3: the complex product by the 3M (Karatsuba) scheme -- three real DMMAs per complex tile product instead of four:
//   t1 = xr yr,  t2 = xi e,  t3 = (xr + xi)(yr + e)   (e = +-yi),   real = t1 - t2,  imag = t3 - t1 - t2
// (three accumulator sets; one operand sum per fragment).  Normwise as accurate as the 4M
// scheme (Higham, Accuracy and Stability, ch. 23: 3M is normwise stable), which is what the per-band relative L2
// tolerance measures; 25 % fewer tensor instructions.
// TMA: the operand stages are filled by cp.async.bulk.tensor (one elected thread, 2 D boxes {4 k, rows} that land as the
// same [rows][4] blocks the fragment loads expect, mbarrier-signalled, out-of-range rows / k zero-filled by the TMA unit)
// instead of 7 predicated cp.async with 64-bit address arithmetic per thread and k-tile.
template <bool CONJY, bool TRI, int BN_, bool M3 = false, int ST = STAGES, int BKT = BK, bool TMA = false>
__global__ void __launch_bounds__(NTHREADS, M3 ? 2 : 1) k_gemm_dotk(const __grid_constant__ CUtensorMap tmX,
                                                        const __grid_constant__ CUtensorMap tmY,
                                                        const double2 *__restrict__ X, const int Rn,
                                                        const double2 *__restrict__ Y, const int Cn, const int64_t K,
                                                        const int ktiles_per_split, double2 *__restrict__ part) {
    extern __shared__ __align__(128) char smem[];
    constexpr int KBLK = TMA ? 64 * 64 : KBLK_BYTES;   // pitch of one [64][4] block (the skew only serves cp.async writes)
    constexpr int OPKT = (BKT / 4) * KBLK;             // one stage of a K-contiguous operand
    char *sX = smem, *sY = smem + ST * OPKT;
    __shared__ __align__(8) uint64_t full[ST];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NTL = BN_ / 16;   // 8-wide DMMA tiles per warp along the columns
    const int wr = (warp >> 1) * 32, wc = (warp & 1) * (BN_ / 2);
    // tri: X == Y and the result is Hermitian; blockIdx.x enumerates, row tile by row tile, the tiles that reach the
    // diagonal or lie below it (first column of the tile <= last row of the tile); the reduction mirrors the rest
    int tr = blockIdx.y, tc = blockIdx.x;
    if constexpr (TRI) {
        const int tcol = (Cn + BN_ - 1) / BN_;
        int t = blockIdx.x;
        tr = 0;
        for (;;) {
            const int nt = min(tcol, ((tr + 1) * BM - 1) / BN_ + 1);
            if (t < nt) break;
            t -= nt;
            tr++;
        }
        tc = t;
    }
    const int row0 = tr * BM, col0 = tc * BN_;
    // rows of Y this tile owns (the loader fills the rest of its 64 rows with zeros); 64: exactly the original code path
    const int cend = BN_ == 64 ? Cn : min(Cn, col0 + BN_);
    const int64_t ktiles = (K + BKT - 1) / BKT;
    const int64_t kt0 = (int64_t)blockIdx.z * ktiles_per_split;
    int64_t kt1 = kt0 + ktiles_per_split;
    if (kt1 > ktiles) kt1 = ktiles;
    const int nkt = (int)(kt1 - kt0);

    // 4M: cr = real, ci = imag accumulators.  3M: cr = k1, ci = k2, c3 = k3 accumulators.
    double cr[4][NTL][2], ci[4][NTL][2], c3[M3 ? 4 : 1][M3 ? NTL : 1][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < NTL; j++) {
            cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0;
            if constexpr (M3) c3[i][j][0] = c3[i][j][1] = 0.0;
        }

    // one stage: (BKT / 4) boxes of {4 k, 64 rows} for X and {4 k, BN_ rows} for Y
    auto tma_stage = [&](int slot, int64_t kt) {
        constexpr uint32_t bytes = (BKT / 4) * (64 + BN_) * 64;
        jtma::mbar_expect_tx(&full[slot], bytes);
#pragma unroll
        for (int q = 0; q < BKT / 4; q++) {
            const int c0 = (int)(2 * (kt * BKT + 4 * q));   // coordinate in doubles along K
            jtma::tma_load_2d(sX + slot * OPKT + q * KBLK, &tmX, c0, row0, &full[slot]);
            jtma::tma_load_2d(sY + slot * OPKT + q * KBLK, &tmY, c0, col0, &full[slot]);
        }
    };
    if constexpr (TMA) {
        if (tid == 0) {
            for (int s = 0; s < ST; s++) jtma::mbar_init(&full[s], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        if (tid == 0)
            for (int s = 0; s < ST - 1 && s < nkt; s++) tma_stage(s, kt0 + s);
    } else {
        for (int s = 0; s < ST - 1; s++) {
            if (s < nkt) {
                load_opk<BKT>(sX + s * OPKT, X, K, Rn, row0, (kt0 + s) * BKT, K, tid);
                load_opk<BKT, BN_>(sY + s * OPKT, Y, K, cend, col0, (kt0 + s) * BKT, K, tid);
            }
            cp_async_commit();
        }
    }
    const int fo = (lane >> 2) * 64 + (lane & 3) * 16;  // fragment offset inside a [64][4] block
    for (int kt = 0; kt < nkt; kt++) {
        if constexpr (TMA) {
            jtma::mbar_wait(&full[kt % ST], (kt / ST) & 1);
            __syncthreads();   // everyone is done with the stage of k-tile kt - 1, which is refilled now
            const int nx = kt + ST - 1;
            if (tid == 0 && nx < nkt) tma_stage(nx % ST, kt0 + nx);
        } else {
            cp_async_wait<ST - 2>();
            __syncthreads();
            if constexpr (!M3) {   // 4M kernels: refill issued right away (the late issue below costs them registers)
                const int nx = kt + ST - 1;
                if (nx < nkt) {
                    const int slot = nx % ST;
                    load_opk<BKT>(sX + slot * OPKT, X, K, Rn, row0, (kt0 + nx) * BKT, K, tid);
                    load_opk<BKT, BN_>(sY + slot * OPKT, Y, K, cend, col0, (kt0 + nx) * BKT, K, tid);
                }
                cp_async_commit();
            }
        }
        const char *bx = sX + (kt % ST) * OPKT, *by = sY + (kt % ST) * OPKT;
#pragma unroll
        for (int kk = 0; kk < BKT / 4; kk++) {
            double2 a[4], bq[NTL];
#pragma unroll
            for (int i = 0; i < 4; i++)
                a[i] = *reinterpret_cast<const double2 *>(bx + kk * KBLK + (wr + 8 * i) * 64 + fo);
#pragma unroll
            for (int j = 0; j < NTL; j++)
                bq[j] = *reinterpret_cast<const double2 *>(by + kk * KBLK + (wc + 8 * j) * 64 + fo);
            if constexpr (!TMA && M3) {
                // the refill of the stage consumed in the previous k-tile is issued AFTER this k-tile's last fragment loads: a
                // shared-memory load right behind the cp.async batch waited for it (ncu: 5 % of the warp samples)
                if (kk == BKT / 4 - 1) {
                    const int nx = kt + ST - 1;
                    if (nx < nkt) {
                        const int slot = nx % ST;
                        load_opk<BKT>(sX + slot * OPKT, X, K, Rn, row0, (kt0 + nx) * BKT, K, tid);
                        load_opk<BKT, BN_>(sY + slot * OPKT, Y, K, cend, col0, (kt0 + nx) * BKT, K, tid);
                    }
                    cp_async_commit();
                }
            }
            if constexpr (M3) {
                double sa[4], sb[NTL], e[NTL];
#pragma unroll
                for (int i = 0; i < 4; i++) sa[i] = a[i].x + a[i].y;
#pragma unroll
                for (int j = 0; j < NTL; j++) {
                    e[j] = CONJY ? -bq[j].y : bq[j].y;   // X (yr + i e)
                    sb[j] = bq[j].x + e[j];
                }
#pragma unroll
                for (int i = 0; i < 4; i++)
#pragma unroll
                    for (int j = 0; j < NTL; j++) {
                        dmma(cr[i][j][0], cr[i][j][1], a[i].x, bq[j].x);   // t1 = xr yr
                        dmma(ci[i][j][0], ci[i][j][1], a[i].y, e[j]);      // t2 = xi e
                        dmma(c3[i][j][0], c3[i][j][1], sa[i], sb[j]);      // t3 = (xr + xi)(yr + e)
                    }
            } else {
#pragma unroll
                for (int i = 0; i < 4; i++)
#pragma unroll
                    for (int j = 0; j < NTL; j++) {
                        // X (Yr -/+ i Yi):  conj: Cr += XrYr + XiYi, Ci += XiYr - XrYi ; else Cr += XrYr - XiYi, Ci += XiYr + XrYi
                        const double yi = CONJY ? bq[j].y : -bq[j].y;
                        dmma(cr[i][j][0], cr[i][j][1], a[i].x, bq[j].x);
                        dmma(ci[i][j][0], ci[i][j][1], a[i].y, bq[j].x);
                        dmma(cr[i][j][0], cr[i][j][1], a[i].y, yi);
                        dmma(ci[i][j][0], ci[i][j][1], a[i].x, -yi);
                    }
            }
        }
    }
    if constexpr (M3) {
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = 0; j < NTL; j++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const double t1 = cr[i][j][h], t2 = ci[i][j][h], t3 = c3[i][j][h];
                    cr[i][j][h] = t1 - t2;
                    ci[i][j][h] = (t3 - t1) - t2;
                }
    }
    if constexpr (!TMA) cp_async_wait<0>();
    double2 *P = part + (size_t)blockIdx.z * Rn * Cn;
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const int r = row0 + wr + 8 * i + (lane >> 2);
        if (r >= Rn) continue;
#pragma unroll
        for (int j = 0; j < NTL; j++) {
            const int c = col0 + wc + 8 * j + 2 * (lane & 3);
            if (c < Cn) P[(size_t)r * Cn + c] = make_double2(cr[i][j][0], ci[i][j][0]);
            if (c + 1 < Cn) P[(size_t)r * Cn + c + 1] = make_double2(cr[i][j][1], ci[i][j][1]);
        }
    }
}

// Out[i] = scale * dscale[c] * sum_s part[s][i]   (fixed order)
// tri = column tile width (0: off): only tiles reaching or below the diagonal were computed; the rest is the conjugate
// transpose (Hermitian result)
__global__ void k_splitk_reduce(const double2 *__restrict__ part, const int nsplit, const int64_t total, const int Cn,
                                const double scale, const double *__restrict__ dscale, double2 *__restrict__ Out,
                                const int tri, const int accumulate) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        int64_t src = i;
        bool cj = false;
        if (tri) {
            const int r = (int)(i / Cn), c = (int)(i % Cn);
            if ((c / tri) * tri > (r / BM) * BM + BM - 1) { src = (int64_t)c * Cn + r; cj = true; }   // tile not computed: mirror
        }
        double sr = 0.0, si = 0.0;
        for (int s = 0; s < nsplit; s++) {
            const double2 v = part[(size_t)s * total + src];
            sr += v.x;
            si += v.y;
        }
        if (cj) si = -si;
        const double f = dscale ? scale * dscale[i % Cn] : scale;
        double2 o = make_double2(f * sr, f * si);
        if (accumulate) { const double2 w = Out[i]; o.x += w.x; o.y += w.y; }
        Out[i] = o;
    }
}

// Block-diagonal D (per-atom Hermitian blocks c128[Cn / nblk][nblk][nblk], D_mode = nblk) applied in the reduction:
// Out[r][a nblk + j] = scale * sum_l D[a][j][l] * (sum_s part[s][r][a nblk + l]).  One thread per (row, atom); the
// nblk reduced values stay in registers (nblk <= NBMAX), so the partials are read once.
template <int NBMAX>
__global__ void k_splitk_reduce_block(const double2 *__restrict__ part, const int nsplit, const int Rn, const int Cn,
                                      const int nblk, const double scale, const double2 *__restrict__ Dblk,
                                      double2 *__restrict__ Out) {
    const int natom = Cn / nblk;
    const int64_t total = (int64_t)Rn * Cn, items = (int64_t)Rn * natom;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < items; i += (int64_t)gridDim.x * blockDim.x) {
        const int r = (int)(i / natom), a = (int)(i % natom);
        const size_t base = (size_t)r * Cn + (size_t)a * nblk;
        double2 red[NBMAX];
#pragma unroll
        for (int l = 0; l < NBMAX; l++) {
            red[l] = make_double2(0.0, 0.0);
            if (l < nblk)
                for (int s = 0; s < nsplit; s++) {
                    const double2 v = part[(size_t)s * total + base + l];
                    red[l].x += v.x;
                    red[l].y += v.y;
                }
        }
        const double2 *Da = Dblk + (size_t)a * nblk * nblk;
        for (int j = 0; j < nblk; j++) {
            double sr = 0.0, si = 0.0;
#pragma unroll
            for (int l = 0; l < NBMAX; l++)
                if (l < nblk) {
                    const double2 d = Da[j * nblk + l];
                    sr += d.x * red[l].x - d.y * red[l].y;
                    si += d.x * red[l].y + d.y * red[l].x;
                }
            Out[base + j] = make_double2(scale * sr, scale * si);
        }
    }
}
// any block size: one thread per output element, the block row re-reduced per element (blocks > 16 are rare)
__global__ void k_splitk_reduce_block_any(const double2 *__restrict__ part, const int nsplit, const int Rn, const int Cn,
                                          const int nblk, const double scale, const double2 *__restrict__ Dblk,
                                          double2 *__restrict__ Out) {
    const int64_t total = (int64_t)Rn * Cn;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i % Cn), a = c / nblk, j = c % nblk;
        const size_t base = (size_t)(i - c) + (size_t)a * nblk;
        const double2 *Da = Dblk + ((size_t)a * nblk + j) * nblk;
        double sr = 0.0, si = 0.0;
        for (int l = 0; l < nblk; l++) {
            double rr = 0.0, ri = 0.0;
            for (int s = 0; s < nsplit; s++) {
                const double2 v = part[(size_t)s * total + base + l];
                rr += v.x;
                ri += v.y;
            }
            const double2 d = Da[l];
            sr += d.x * rr - d.y * ri;
            si += d.x * ri + d.y * rr;
        }
        Out[i] = make_double2(scale * sr, scale * si);
    }
}

// ---------------------------------------------------------------------------------------------- expand GEMM
// BN_ x (WM x WN warps): 64 x (2 x 2) is the default tile; 56 x (4 x 1) exists because for some n extents it fills the
// 148 x 3 CTA slots in whole waves where 64 leaves a half-empty tail wave (config 2: 1.68 -> 1.93 waves).
template <int BN_, int WM, int WN, bool M3 = false, int ST = STAGES>
__global__ void __launch_bounds__(NTHREADS, M3 ? 2 : 3) k_gemm_expand(const double2 *__restrict__ A, const int Rn,
                                                          const double2 *__restrict__ Pm, const int K, const int64_t Nn,
                                                          double2 *Out, const double2 *Add,
                                                          const double addscale) {
    extern __shared__ __align__(16) char smem[];
    constexpr int MTL = BM / (8 * WM), NTL = BN_ / (8 * WN);   // 8 x 8 DMMA tiles per warp along rows / columns
    constexpr int PROW = BN_ * 16 + 32, OPN = BK * PROW;
    static_assert(WM * WN * 32 == NTHREADS && MTL * 8 * WM == BM && NTL * 8 * WN == BN_, "warp layout");
    char *sA = smem, *sP = smem + ST * OPK_BYTES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wr = (warp / WN) * (8 * MTL), wc = (warp % WN) * (8 * NTL);
    // row tile fastest: the CTAs that share one n-tile of P (all band tiles) run at the same time, so P comes from HBM
    // once and from L2 otherwise (ncu, config 5: 14.7 GB of DRAM reads per launch with the n-tile fastest)
    const int row0 = blockIdx.x * BM;
    const int64_t n0 = (int64_t)blockIdx.y * BN_;
    const int nkt = (K + BK - 1) / BK;
    // pull the tile the epilogue adds to towards L2 shortly before it is needed (PF_AHEAD k-tiles before the end: early
    // enough to cover the HBM latency, late enough that the lines are still resident -- a CTA lives for ~140 us at K = 864)
    constexpr int PF_AHEAD = 12;
    auto prefetch_out = [&]() {
        for (int e = tid; e < BM * ((BN_ * 16 + 127) / 128); e += NTHREADS) {
            const int r = e / ((BN_ * 16 + 127) / 128), seg = e % ((BN_ * 16 + 127) / 128);
            if (row0 + r < Rn && n0 + seg * 8 < Nn)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(Add + (size_t)(row0 + r) * Nn + n0 + seg * 8));
        }
    };
    if (Add && (!M3 || nkt <= PF_AHEAD)) prefetch_out();   // short K (4M kernel): at the start

    double cr[MTL][NTL][2], ci[MTL][NTL][2], c3[M3 ? MTL : 1][M3 ? NTL : 1][2];   // 3M: k1, k2, k3 (see k_gemm_dotk)
#pragma unroll
    for (int i = 0; i < MTL; i++)
#pragma unroll
        for (int j = 0; j < NTL; j++) {
            cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0;
            if constexpr (M3) c3[i][j][0] = c3[i][j][1] = 0.0;
        }

    auto load_p = [&](char *dst, int k0) {
#pragma unroll
        for (int i = 0; i < (BK * BN_ + NTHREADS - 1) / NTHREADS; i++) {
            const int e = tid + i * NTHREADS;
            if ((BK * BN_) % NTHREADS != 0 && e >= BK * BN_) break;
            const int kk = e / BN_, nn = e % BN_;
            const bool ok = (k0 + kk < K) && (n0 + nn < Nn);
            const double2 *src = ok ? Pm + (size_t)(k0 + kk) * Nn + n0 + nn : Pm;
            cp_async16(dst + kk * PROW + nn * 16, src, ok);
        }
    };
    for (int s = 0; s < ST - 1; s++) {
        if (s < nkt) {
            load_opk(sA + s * OPK_BYTES, A, K, Rn, row0, (int64_t)s * BK, K, tid);
            load_p(sP + s * OPN, s * BK);
        }
        cp_async_commit();
    }
    const int fa = (lane >> 2) * 64 + (lane & 3) * 16;
    const int fp = (lane & 3) * PROW + (lane >> 2) * 16;
    for (int kt = 0; kt < nkt; kt++) {
        cp_async_wait<ST - 2>();
        __syncthreads();
        if (M3 && Add && kt == nkt - PF_AHEAD) prefetch_out();
        if constexpr (!M3) {   // 4M kernels (3 CTAs per SM, 168 registers): refill issued right away
            const int nx = kt + ST - 1;
            if (nx < nkt) {
                const int slot = nx % ST;
                load_opk(sA + slot * OPK_BYTES, A, K, Rn, row0, (int64_t)nx * BK, K, tid);
                load_p(sP + slot * OPN, nx * BK);
            }
            cp_async_commit();
        }
        const char *ba = sA + (kt % ST) * OPK_BYTES, *bp = sP + (kt % ST) * OPN;
#pragma unroll
        for (int kk = 0; kk < BK / 4; kk++) {
            double2 a[MTL], bq[NTL];
#pragma unroll
            for (int i = 0; i < MTL; i++)
                a[i] = *reinterpret_cast<const double2 *>(ba + kk * KBLK_BYTES + (wr + 8 * i) * 64 + fa);
#pragma unroll
            for (int j = 0; j < NTL; j++)
                bq[j] = *reinterpret_cast<const double2 *>(bp + kk * 4 * PROW + (wc + 8 * j) * 16 + fp);
            if (M3 && kk == BK / 4 - 1) {   // refill issued after the k-tile's last fragment loads (see k_gemm_dotk): 10.97 -> 10.80 ms at config 5
                const int nx = kt + ST - 1;
                if (nx < nkt) {
                    const int slot = nx % ST;
                    load_opk(sA + slot * OPK_BYTES, A, K, Rn, row0, (int64_t)nx * BK, K, tid);
                    load_p(sP + slot * OPN, nx * BK);
                }
                cp_async_commit();
            }
            if constexpr (M3) {
                double sa[MTL], sb[NTL];
#pragma unroll
                for (int i = 0; i < MTL; i++) sa[i] = a[i].x + a[i].y;
#pragma unroll
                for (int j = 0; j < NTL; j++) sb[j] = bq[j].x + bq[j].y;
#pragma unroll
                for (int i = 0; i < MTL; i++)
#pragma unroll
                    for (int j = 0; j < NTL; j++) {
                        dmma(cr[i][j][0], cr[i][j][1], a[i].x, bq[j].x);
                        dmma(ci[i][j][0], ci[i][j][1], a[i].y, bq[j].y);
                        dmma(c3[i][j][0], c3[i][j][1], sa[i], sb[j]);
                    }
            } else {
#pragma unroll
                for (int i = 0; i < MTL; i++)
#pragma unroll
                    for (int j = 0; j < NTL; j++) {
                        dmma(cr[i][j][0], cr[i][j][1], a[i].x, bq[j].x);
                        dmma(ci[i][j][0], ci[i][j][1], a[i].y, bq[j].x);
                        dmma(cr[i][j][0], cr[i][j][1], a[i].y, -bq[j].y);
                        dmma(ci[i][j][0], ci[i][j][1], a[i].x, bq[j].y);
                    }
            }
        }
    }
    cp_async_wait<0>();
    if constexpr (M3) {
#pragma unroll
        for (int i = 0; i < MTL; i++)
#pragma unroll
            for (int j = 0; j < NTL; j++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const double t1 = cr[i][j][h], t2 = ci[i][j][h], t3 = c3[i][j][h];
                    cr[i][j][h] = t1 - t2;
                    ci[i][j][h] = (t3 - t1) - t2;
                }
    }
#pragma unroll
    for (int i = 0; i < MTL; i++) {
        const int r = row0 + wr + 8 * i + (lane >> 2);
        if (r >= Rn) continue;
#pragma unroll
        for (int j = 0; j < NTL; j++) {
            const int64_t n = n0 + wc + 8 * j + 2 * (lane & 3);
            double2 *o = Out + (size_t)r * Nn + n;
            const double2 *ad = Add + (size_t)r * Nn + n;   // Add may alias Out (accumulate): each element is read, then written, by this thread only
            if (n < Nn) {
                double2 v = make_double2(cr[i][j][0], ci[i][j][0]);
                if (Add) { const double2 w = ad[0]; v.x = fma(addscale, w.x, v.x); v.y = fma(addscale, w.y, v.y); }
                o[0] = v;
            }
            if (n + 1 < Nn) {
                double2 v = make_double2(cr[i][j][1], ci[i][j][1]);
                if (Add) { const double2 w = ad[1]; v.x = fma(addscale, w.x, v.x); v.y = fma(addscale, w.y, v.y); }
                o[1] = v;
            }
        }
    }
}

template <class K>
cudaError_t ensure_smem(K kernel, size_t bytes, int device) {
    return jdft_ensure_smem((const void *)kernel, bytes, device);
}

}  // namespace

int jdft_gemm_dotk(const jdft_basis *b, const double *X, int Rn, const double *Y, int Cn, int64_t K, int conjY,
                   double scale, const double *dscale, double *Out, void *scratch, size_t scratch_bytes,
                   cudaStream_t st, const double *dblock, int nblk, int accumulate) {
    if (Rn <= 0 || Cn <= 0) return JDFT_OK;
    if (dblock && (nblk < 1 || Cn % nblk != 0 || dscale || accumulate))
        return jdft_fail(JDFT_EINVAL, "gemm: block-diagonal D needs nproj %% block == 0");
    // X^+ X is Hermitian: compute the lower-triangle tiles only and mirror them in the reduction
    const int tri = (X == Y && Rn == Cn && conjY && !dscale && !dblock && BM == BN) ? 1 : 0;
    const int trow = (Rn + BM - 1) / BM;
    // column tile: 48 instead of 64 when that removes a noticeable share of zero padding (np = 288: 320 -> 288 columns)
    const int pad64 = ((Cn + 63) / 64) * 64, pad48 = ((Cn + 47) / 48) * 48;
    int bn = (!tri && Cn > 64 && pad48 * 100 < pad64 * 93) ? 48 : 64;  // measured: pays at 10 % padding (np = 288), not at 3.6 % (np = 864)
    // 3M scheme (three DMMAs per complex tile product; 64 x 48 tiles, its three accumulator sets leave no room for
    // 64 x 64): taken when 0.8 x its padded width beats the 4M choice and K is long enough to matter
    const bool m3 = b->opt_gemm3m && K >= 512 && (tri ? Cn >= 128 : pad48 * 80 < (bn == 48 ? pad48 : pad64) * 100);
    if (m3) bn = 48;   // (64 x 32 tiles at 3 CTAs per SM measured 7 % slower)
    // pipeline of the 3M kernels: measured on config 3 (P^+ C, 1.70 ms): 6 stages of 8 -> 1.78 ms, 3 stages of 16 -> 1.89 ms
    constexpr int ST3 = STAGES, BK3 = BK;
    const int bk = m3 ? BK3 : BK;
    const int64_t ktiles = (K + bk - 1) / bk;
    const int tcol = (Cn + bn - 1) / bn;
    int tiles = trow * tcol;
    if (tri) {
        tiles = 0;
        for (int tr = 0; tr < trow; tr++) {
            const int nt = ((tr + 1) * BM - 1) / bn + 1;
            tiles += nt < tcol ? nt : tcol;
        }
    }
    const size_t one = (size_t)Rn * Cn * 16;
    // Split K so that the grid fills whole waves of the SMs x 2 resident CTAs (184 registers x 128 threads):
    // among 1..6 waves take the smallest count whose fill tiles*nsplit / (waves*slots) is within 2 % of the best (stop at 97 %).
    const int64_t slots = (int64_t)b->num_sms * 2;
    const int64_t min_kt = 128 / bk;                                         // at least 128 k per slice
    const int64_t max_by_k = ktiles / min_kt > 0 ? ktiles / min_kt : 1;
    const int64_t max_by_ws = (int64_t)(scratch_bytes / one);
    if (max_by_ws < 1) return jdft_fail(JDFT_EWORKSPACE, "gemm: workspace too small for a %d x %d result", Rn, Cn);
    int64_t nsplit = 1;
    double best = -1.0;
    for (int64_t w = 1; w <= 6; w++) {
        int64_t ns = (w * slots) / tiles;
        if (ns > max_by_k) ns = max_by_k;
        if (ns > max_by_ws) ns = max_by_ws;
        if (ns < 1) ns = 1;
        const int64_t ctas = ns * tiles;
        const int64_t waves = (ctas + slots - 1) / slots;
        const double fill = (double)ctas / (double)(waves * slots);
        if (fill > best + 0.02) { best = fill; nsplit = ns; }   // more waves (more partials) only for > 2 % better fill
        if (best >= 0.97) break;
    }
    int64_t per = (ktiles + nsplit - 1) / nsplit;
    if (per < 1) per = 1;
    nsplit = (ktiles + per - 1) / per;
    if (nsplit < 1) nsplit = 1;
    // TMA operand staging (option "gemm_tma"): both operands need 16-byte aligned rows (K even or ... always: c128) and
    // extents that fit the tensor-map fields; the 3M kernels only (they are the ones on the hot path)
    CUtensorMap tmX, tmY;
    memset(&tmX, 0, sizeof(tmX));
    memset(&tmY, 0, sizeof(tmY));
    bool tma = false;
    if (m3 && b->opt_gemm_tma && K < ((int64_t)1 << 30)) {
        JdftEncodeTiledFn enc = jdft_tensor_map_encoder();
        const cuuint64_t strX[1] = {(cuuint64_t)K * 16};
        const cuuint64_t dimX[2] = {(cuuint64_t)2 * K, (cuuint64_t)Rn}, dimY[2] = {(cuuint64_t)2 * K, (cuuint64_t)Cn};
        const cuuint32_t boxX[2] = {8, 64}, boxY[2] = {8, (cuuint32_t)bn}, es[2] = {1, 1};
        tma = enc &&
              enc(&tmX, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)X, dimX, strX, boxX, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS &&
              enc(&tmY, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)Y, dimY, strX, boxY, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
    }
    const size_t smem = m3 ? 2 * ST3 * (BK3 / 4) * (tma ? 4096 : KBLK_BYTES) + (tma ? 128 : 0) : 2 * STAGES * OPK_BYTES;
    dim3 grid(tri ? tiles : tcol, tri ? 1 : trow, (unsigned)nsplit);
    jdft_prof_begin(b, JDFT_K_GEMM_DOTK, st);
#define JDFT_DOTK_LAUNCH(...)                                                                                  \
    do {                                                                                                        \
        JDFT_CUDA(ensure_smem(k_gemm_dotk<__VA_ARGS__>, smem, b->device));                                      \
        k_gemm_dotk<__VA_ARGS__><<<grid, NTHREADS, smem, st>>>(tmX, tmY, (const double2 *)X, Rn, (const double2 *)Y, Cn, K, \
                                                               (int)per, (double2 *)scratch);                  \
    } while (0)
    if (tri && m3 && tma) JDFT_DOTK_LAUNCH(true, true, 48, true, ST3, BK3, true);
    else if (m3 && tma && conjY) JDFT_DOTK_LAUNCH(true, false, 48, true, ST3, BK3, true);
    else if (m3 && tma) JDFT_DOTK_LAUNCH(false, false, 48, true, ST3, BK3, true);
    else if (tri && m3) JDFT_DOTK_LAUNCH(true, true, 48, true, ST3, BK3);
    else if (tri) JDFT_DOTK_LAUNCH(true, true, 64);
    else if (m3 && conjY) JDFT_DOTK_LAUNCH(true, false, 48, true, ST3, BK3);
    else if (m3) JDFT_DOTK_LAUNCH(false, false, 48, true, ST3, BK3);
    else if (conjY && bn == 48) JDFT_DOTK_LAUNCH(true, false, 48);
    else if (conjY) JDFT_DOTK_LAUNCH(true, false, 64);
    else if (bn == 48) JDFT_DOTK_LAUNCH(false, false, 48);
    else JDFT_DOTK_LAUNCH(false, false, 64);
#undef JDFT_DOTK_LAUNCH
    jdft_prof_end(b, JDFT_K_GEMM_DOTK, st);
    JDFT_LAUNCH_CHECK("k_gemm_dotk");
    const int64_t total = (int64_t)Rn * Cn;
    int64_t blocks = (total + 255) / 256;
    if (blocks > b->num_sms * 8) blocks = b->num_sms * 8;
    jdft_prof_begin(b, JDFT_K_REDUCE, st);
    if (dblock) {
        const int64_t items = (int64_t)Rn * (Cn / nblk);
        int64_t bl = (items + 127) / 128;
        if (bl > b->num_sms * 8) bl = b->num_sms * 8;
        if (nblk <= 4)
            k_splitk_reduce_block<4><<<(int)bl, 128, 0, st>>>((const double2 *)scratch, (int)nsplit, Rn, Cn, nblk, scale, (const double2 *)dblock, (double2 *)Out);
        else if (nblk <= 9)
            k_splitk_reduce_block<9><<<(int)bl, 128, 0, st>>>((const double2 *)scratch, (int)nsplit, Rn, Cn, nblk, scale, (const double2 *)dblock, (double2 *)Out);
        else if (nblk <= 16)
            k_splitk_reduce_block<16><<<(int)bl, 128, 0, st>>>((const double2 *)scratch, (int)nsplit, Rn, Cn, nblk, scale, (const double2 *)dblock, (double2 *)Out);
        else
            k_splitk_reduce_block_any<<<(int)blocks, 256, 0, st>>>((const double2 *)scratch, (int)nsplit, Rn, Cn, nblk, scale, (const double2 *)dblock, (double2 *)Out);
    } else {
        k_splitk_reduce<<<(int)blocks, 256, 0, st>>>((const double2 *)scratch, (int)nsplit, total, Cn, scale, dscale, (double2 *)Out, tri ? bn : 0, accumulate);
    }
    jdft_prof_end(b, JDFT_K_REDUCE, st);
    JDFT_LAUNCH_CHECK("k_splitk_reduce");
    return JDFT_OK;
}

// Out[r][:] = scale * D . A[r][:] for projected coefficients A [Rn][Cn] that already exist (D_mode as in the ABI):
// the reduction kernels with a single "partial" (diagonal / block-diagonal D) or one small GEMM (dense D)
int jdft_apply_D(const jdft_basis *b, const double *A, int Rn, int Cn, const double *D, int D_mode, double scale, double *Out,
                 void *scratch, size_t scratch_bytes, cudaStream_t st) {
    if (Rn <= 0 || Cn <= 0) return JDFT_OK;
    if (D_mode == 1) return jdft_gemm_dotk(b, A, Rn, D, Cn, Cn, 0, scale, nullptr, Out, scratch, scratch_bytes, st);
    const int64_t total = (int64_t)Rn * Cn;
    jdft_prof_begin(b, JDFT_K_REDUCE, st);
    if (D_mode == 0) {
        int64_t blocks = (total + 255) / 256;
        if (blocks > b->num_sms * 8) blocks = b->num_sms * 8;
        k_splitk_reduce<<<(int)blocks, 256, 0, st>>>((const double2 *)A, 1, total, Cn, scale, D, (double2 *)Out, 0, 0);
    } else {
        const int nblk = D_mode;
        int64_t bl = ((int64_t)Rn * (Cn / nblk) + 127) / 128;
        if (bl > b->num_sms * 8) bl = b->num_sms * 8;
        if (nblk <= 4) k_splitk_reduce_block<4><<<(int)bl, 128, 0, st>>>((const double2 *)A, 1, Rn, Cn, nblk, scale, (const double2 *)D, (double2 *)Out);
        else if (nblk <= 9) k_splitk_reduce_block<9><<<(int)bl, 128, 0, st>>>((const double2 *)A, 1, Rn, Cn, nblk, scale, (const double2 *)D, (double2 *)Out);
        else if (nblk <= 16) k_splitk_reduce_block<16><<<(int)bl, 128, 0, st>>>((const double2 *)A, 1, Rn, Cn, nblk, scale, (const double2 *)D, (double2 *)Out);
        else {
            int64_t blocks = (total + 255) / 256;
            if (blocks > b->num_sms * 8) blocks = b->num_sms * 8;
            k_splitk_reduce_block_any<<<(int)blocks, 256, 0, st>>>((const double2 *)A, 1, Rn, Cn, nblk, scale, (const double2 *)D, (double2 *)Out);
        }
    }
    jdft_prof_end(b, JDFT_K_REDUCE, st);
    JDFT_LAUNCH_CHECK("apply_D");
    return JDFT_OK;
}

int jdft_gemm_expand(const jdft_basis *b, const double *A, int Rn, const double *Pm, int K, int64_t Nn, double *Out, int accumulate,
                     cudaStream_t st, const double *Add, double addscale) {
    if (Rn <= 0 || Nn <= 0) return JDFT_OK;
    if (accumulate) { Add = Out; addscale = 1.0; }   // Out += result; otherwise Out = result (+ addscale * Add)
    // tile width: 64, unless 56 fills the SMs x 3 CTA slots in whole waves noticeably better
    const int64_t slots = (int64_t)b->num_sms * 3, rt = (Rn + BM - 1) / BM;
    auto fill = [&](int bn) {
        const int64_t ctas = ((Nn + bn - 1) / bn) * rt, waves = (ctas + slots - 1) / slots;
        return (double)ctas / (double)(waves * slots);
    };
    const bool narrow = fill(56) > fill(64) + 0.05;
    jdft_prof_begin(b, JDFT_K_GEMM_EXPAND, st);
    if (b->opt_gemm3m && K >= 320) {   // 3M scheme: 64 x 48 tiles, 2 CTAs per SM (see k_gemm_dotk); measured neutral at K = 288, -8 % at 384, -12 % at 864
        constexpr int BNX = 48, ST3 = 6;
        const size_t smem = ST3 * (OPK_BYTES + BK * (BNX * 16 + 32));
        JDFT_CUDA(ensure_smem(k_gemm_expand<BNX, 2, 2, true, ST3>, smem, b->device));
        dim3 grid((unsigned)rt, (unsigned)((Nn + BNX - 1) / BNX));
        k_gemm_expand<BNX, 2, 2, true, ST3><<<grid, NTHREADS, smem, st>>>((const double2 *)A, Rn, (const double2 *)Pm, K, Nn, (double2 *)Out, (const double2 *)Add, addscale);
    } else if (narrow) {
        constexpr int BNX = 56;
        const size_t smem = STAGES * (OPK_BYTES + BK * (BNX * 16 + 32));
        JDFT_CUDA(ensure_smem(k_gemm_expand<BNX, 4, 1>, smem, b->device));
        dim3 grid((unsigned)rt, (unsigned)((Nn + BNX - 1) / BNX));
        k_gemm_expand<BNX, 4, 1><<<grid, NTHREADS, smem, st>>>((const double2 *)A, Rn, (const double2 *)Pm, K, Nn, (double2 *)Out, (const double2 *)Add, addscale);
    } else {
        const size_t smem = STAGES * (OPK_BYTES + OPN_BYTES);
        JDFT_CUDA(ensure_smem(k_gemm_expand<BN, 2, 2>, smem, b->device));
        dim3 grid((unsigned)rt, (unsigned)((Nn + BN - 1) / BN));
        k_gemm_expand<BN, 2, 2><<<grid, NTHREADS, smem, st>>>((const double2 *)A, Rn, (const double2 *)Pm, K, Nn, (double2 *)Out, (const double2 *)Add, addscale);
    }
    jdft_prof_end(b, JDFT_K_GEMM_EXPAND, st);
    JDFT_LAUNCH_CHECK("k_gemm_expand");
    return JDFT_OK;
}
