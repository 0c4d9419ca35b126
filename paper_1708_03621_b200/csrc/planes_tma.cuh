// K3 on Blackwell data movement (TMA): W2 -> inverse FFT along axis 0 -> * V_loc -> forward FFT along axis 0 -> W2.
// Included by local.cu only (uses Tuned<>, Hyb<>, dft8_in0167 / dft8_out0167 defined there).
//
// Same arithmetic as k_planes_fused_h (radix-8 first / last pass on pencil pairs, fused radix-R2 middle pass with the
// V multiply in registers), but the global side no longer goes global -> register -> shared through the LSU:
//   * a 3-D tensor map over W2 viewed as f64 [nbatch npl][S1][2 S2] describes the tile of one CTA step, the box
//     {32 doubles = 16 pencils, 1 row i1, npl planes}; `cp.async.bulk.tensor` lands it in shared memory as
//     [npl][16] c128 and signals an mbarrier; the write-back is a `cp.async.bulk.tensor` store of the same box;
//   * CTAs are persistent (grid = resident CTAs) and walk the tiles (i2 tile, i1, band) with stride gridDim; a
//     producer warp keeps ONE tile in flight ahead of the four compute warps (two in/out buffers), so the load of
//     tile i+1 and the store of tile i-1 overlap the butterflies of tile i;
//   * out-of-range pencils of a ragged last i2 tile are zero-filled on load and clipped on store by the TMA unit.
// Buffers: A = the [L][16] butterfly tile (in place), B[2] = in/out staging [npl][16]; B[s] receives the tile, is
// consumed by the first pass, and is re-used for the tile's result, which the producer stores before re-filling it.
#pragma once
#include "tma.cuh"


template <int LT>
struct PlanesTma {
    static constexpr int NTC = Hyb<LT>::NT;        // compute threads
    static constexpr int NT = NTC + 32;            // + one producer warp
    static constexpr int T = 16;
    static constexpr bool ok = Tuned<LT>::ok && Tuned<LT>::R1 == 8;
    static constexpr int MINB = LT >= 128 ? 3 : 4;   // resident CTAs per SM the registers are bounded for
    static size_t smem_bytes(int npl) { return ((size_t)LT * T + 2 * (size_t)npl * T) * sizeof(double2) + 128; }
};

template <int LT, bool PR>
__global__ void __launch_bounds__(PlanesTma<LT>::NT, PlanesTma<LT>::MINB)
    k_planes_tma(const __grid_constant__ CUtensorMap tmW, const double2 *__restrict__ tw, const int S1, const int S2,
                 const int npl, const int *__restrict__ planeof, const double *__restrict__ V, const int ntx,
                 const int ntiles) {
    using C = Tuned<LT>;
    constexpr int R1 = C::R1, R2 = C::R2, T = 16, H = 8, NTC = PlanesTma<LT>::NTC, L = LT;
    static_assert(R2 * H <= NTC && R1 * T <= NTC, "pair passes and the fused middle pass must each be one round");
    extern __shared__ unsigned char smem_raw[];
    double2 *A = reinterpret_cast<double2 *>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
    double2 *B[2] = {A + L * T, A + L * T + npl * T};
    __shared__ __align__(8) uint64_t full[2], outready[2];
    __shared__ int s_planeof[L];
    const int tid = threadIdx.x;
    for (int i = tid; i < L; i += PlanesTma<LT>::NT) s_planeof[i] = planeof[i];
    if (tid == 0) {
        for (int s = 0; s < 2; s++) {
            jtma::mbar_init(&full[s], 1);
            jtma::mbar_init(&outready[s], NTC);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int first = blockIdx.x, stride = gridDim.x;
    const int nmine = first < ntiles ? (ntiles - first + stride - 1) / stride : 0;
    const uint32_t box_bytes = (uint32_t)npl * T * sizeof(double2);

    if (tid >= NTC) {
        // ---------------------------------------------------------------- producer warp (one lane issues)
        if (tid == NTC) {
            auto coords = [&](int i, int &c0, int &c1, int &c2) {
                const int tile = first + i * stride;
                const int tx = tile % ntx, r = tile / ntx;
                c0 = tx * 2 * T;
                c1 = r % S1;
                c2 = (r / S1) * npl;
            };
            for (int i = 0; i < 2 && i < nmine; i++) {
                int c0, c1, c2;
                coords(i, c0, c1, c2);
                jtma::mbar_expect_tx(&full[i], box_bytes);
                jtma::tma_load_3d(B[i], &tmW, c0, c1, c2, &full[i]);
            }
            for (int i = 0; i < nmine; i++) {
                const int s = i & 1;
                jtma::mbar_wait(&outready[s], (i >> 1) & 1);   // every compute thread has written its part of the result
                int c0, c1, c2;
                coords(i, c0, c1, c2);
                jtma::tma_store_3d(&tmW, c0, c1, c2, B[s]);
                jtma::bulk_commit();
                if (i + 2 < nmine) {
                    jtma::bulk_wait_read0();                    // the store has read B[s]; it may be overwritten
                    coords(i + 2, c0, c1, c2);
                    jtma::mbar_expect_tx(&full[s], box_bytes);
                    jtma::tma_load_3d(B[s], &tmW, c0, c1, c2, &full[s]);
                }
            }
            jtma::bulk_wait0();
        }
        return;
    }

    // -------------------------------------------------------------------- compute warps
    for (int i = 0; i < nmine; i++) {
        const int s = i & 1;
        const int tile = first + i * stride;
        const int tx = tile % ntx, i1 = (tile / ntx) % S1;
        const int t0 = tx * T;
        const int tmax = S2 - t0;
        const size_t plane = (size_t)S1 * S2;
        const double *Vb = V + (size_t)i1 * S2 + t0;
        double2 *Bs = B[s];
        jtma::mbar_wait(&full[s], (i >> 1) & 1);
        // pass 0 of the inverse transform on the pencil pair (l, l + 8): rows bf + k R2 -> rows bf R1 + j
        if (tid < R2 * H) {
            const int l = tid % H, bf = tid / H;
            double2 a0[R1], a1[R1];
#pragma unroll
            for (int k = 0; k < R1; k++) {
                if (PR && k >= 2 && k < 6) continue;
                const int p = s_planeof[bf + k * R2];
                a0[k] = a1[k] = make_double2(0.0, 0.0);
                if (p >= 0) {
                    a0[k] = Bs[p * T + l];
                    a1[k] = Bs[p * T + H + l];
                }
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
        jtma::bar_compute<NTC>();
        {
            const int x = tid % T, bf = tid / T;
            const bool act = tid < R1 * T;
            double2 a[R2];
            if (act) {
#pragma unroll
                for (int k = 0; k < R2; k++) a[k] = A[(bf + k * R1) * T + x];
            }
            jtma::bar_compute<NTC>();
            if (act) {
                Dft<R2, +1>::run(a);
#pragma unroll
                for (int j = 0; j < R2; j++) {
                    const double f = x < tmax ? __ldg(Vb + (size_t)(bf + R1 * j) * plane + x) : 0.0;
                    a[j].x *= f;
                    a[j].y *= f;
                }
                Dft<R2, -1>::run(a);
                twiddle_rows<R2, -1>(a, tw, bf);
#pragma unroll
                for (int j = 0; j < R2; j++) A[(bf * R2 + j) * T + x] = a[j];
            }
        }
        jtma::bar_compute<NTC>();
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
                if (p >= 0) {
                    Bs[p * T + l] = a0[j];
                    Bs[p * T + H + l] = a1[j];
                }
            }
        }
        jtma::fence_proxy_async();          // make this thread's result visible to the TMA unit ...
        jtma::mbar_arrive(&outready[s]);    // ... then tell the producer; all NTC threads arrive
        jtma::bar_compute<NTC>();           // A is re-used by the next tile's first pass
    }
}
