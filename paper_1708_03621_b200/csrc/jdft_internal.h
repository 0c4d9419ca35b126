// Internal declarations shared by the translation units of libjdft_b200 (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <vector>
#include "../../include/jdft.h"

#define JDFT_MAX_PASSES 12

// Radix plan of one 1-D FFT length (Stockham autosort, one radix per pass).
struct FftPlan {
    int L;
    int npass;
    int radix[JDFT_MAX_PASSES];
};

// one captured jdft_apply_H call (option "graph"): replayed while every argument and the workspace stay the same
struct JdftGraphEntry {
    const void *V, *P, *D, *C, *HC, *ws;
    size_t ws_bytes;
    int nproj, D_mode, nb;
    int64_t launches;        // kernels in the graph (for jdft_launch_count)
    int seen;                // calls with this key so far (the first one runs directly and warms the kernel attributes)
    cudaGraphExec_t exec;    // nullptr until captured
};

struct jdft_basis {
    // geometry
    double R[9], k[3], Ecut, G[9], GGT[9], volume;
    int S[3];
    int64_t N, nG;
    int device;
    int num_sms;                              // multiProcessorCount of `device`, queried once at create
    // host copies of the sphere
    std::vector<int32_t> iG, index;
    std::vector<double> ke;
    // pruning structure: planes p <-> m0 = m0lo + p; columns c of plane p <-> m1 = pl_m1lo[p] + (c - pl_cbase[p])
    int npl, m0lo, ncol, maxcol_per_plane;
    int mmin[3], mmax[3];                     // extent of the sphere along each axis (signed m_d)
    std::vector<int> pl_m1lo, pl_cbase;       // [npl], [npl+1]
    std::vector<int> col_n0, col_m2lo;        // [ncol+1], [ncol]
    // device copies
    int32_t *d_index;
    int32_t *d_iG;                            // [nG][3] (gradient / divergence)
    double *d_ke;
    int *d_col_n0, *d_col_m2lo;               // [ncol+1], [ncol]
    int *d_rowcol;                            // [npl][S1]: column index of (plane p, i1) or -1
    int *d_planeof;                           // [S0]: plane index of i0 or -1
    double2 *d_tw[3];                         // exp(+2 pi i t / S_d), t = 0..S_d-1
    FftPlan plan[3];
    // workspace (caller-owned)
    void *ws;
    size_t ws_bytes;
    // options
    int64_t opt_band_batch, opt_force_generic;
    // fork/join resources of apply_H (option "overlap_gemm"): the projection GEMM runs on `side` while the FFT pipeline
    // runs on the caller's stream
    int64_t opt_overlap;
    int64_t opt_pair;                         // K3 with two pencils per thread where available ("planes_pair")
    int64_t opt_gemm3m;                       // GEMMs by the 3M complex-product scheme ("gemm_3m", default 1)
    int64_t opt_host_chunk;                   // bands per chunk of the *_host pipeline ("host_chunk", 0 = 128)
    int64_t opt_gemm_tma;                     // operand stages of the 3M GEMMs filled by TMA ("gemm_tma")
    int64_t opt_tma;                          // K3 through TMA tensor-map loads / stores ("planes_tma")
    int64_t opt_cols_direct;                  // K1: first pass reads the sphere straight from global memory ("cols_direct")
    int64_t opt_prune;                        // K3 hybrid: radix-8 butterflies pruned to the occupied planes ("planes_prune")
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_join;
    // optional per-kernel event timing (option "profile_kernel" = one of JDFT_K_*; 0 = off).  Diagnostics only.
    int64_t opt_profile_kernel;
    std::vector<cudaEvent_t> prof_ev;  // pairs (begin, end)
    size_t prof_used;
    // cached device buffers of the *_host entry points (library-owned, grow-only)
    void *hb[8];
    size_t hb_bytes[8];
    int64_t opt_graph;                        // "graph": -1 auto (small problems), 0 off, 1 on
    std::vector<JdftGraphEntry> graphs;
    cudaStream_t gstream;                     // capture stream
    cudaStream_t hs[3];                       // H2D, compute and D2H streams of the *_host pipeline (created on first use)
    std::vector<cudaEvent_t> hev;
    int h_C_nb;                               // bands of the last host call still valid in hb[0] (0: none)
    int h_ops_set, h_nproj, h_D_mode;         // resident operators of jdft_host_set_operators (in hb[2..4])
};

// kernel ids for the "profile_kernel" option
enum { JDFT_K_NONE = 0, JDFT_K_COLS_INV = 1, JDFT_K_ROWS_INV = 2, JDFT_K_PLANES = 3, JDFT_K_ROWS_FWD = 4,
       JDFT_K_COLS_FWD = 5, JDFT_K_GEMM_DOTK = 6, JDFT_K_GEMM_EXPAND = 7, JDFT_K_REDUCE = 8, JDFT_K_DIAG = 9 };
void jdft_prof_begin(const jdft_basis *b, int kid, cudaStream_t st);
void jdft_prof_end(const jdft_basis *b, int kid, cudaStream_t st);

// error plumbing
int jdft_fail(int code, const char *fmt, ...);
int jdft_cuda_fail(cudaError_t e, const char *what);
void jdft_count_launch(int n);
int64_t jdft_launch_count_peek();
void jdft_graphs_clear(jdft_basis *b);
#define JDFT_CUDA(call)                                           \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return jdft_cuda_fail(e__, #call); \
    } while (0)
#define JDFT_LAUNCH_CHECK(name)                                   \
    do {                                                          \
        jdft_count_launch(1);                                     \
        cudaError_t e__ = cudaGetLastError();                     \
        if (e__ != cudaSuccess) return jdft_cuda_fail(e__, name); \
    } while (0)

// Opt a kernel in to `bytes` of dynamic shared memory ONCE per (kernel, device): the first launch pays the
// cudaFuncSetAttribute, later launches only a table lookup (no driver call on the hot path).
cudaError_t jdft_ensure_smem(const void *kernel, size_t bytes, int device);

// per-band scratch of the FFT path (bytes)
size_t jdft_fft_bytes_per_band(const jdft_basis *b);
// bands per batch given the workspace and options; 0 if not even one fits
int jdft_band_batch(const jdft_basis *b, int nb, size_t ws_offset = 0);

// local.cu: FFT-based pieces
// out = scale * I^+ (Vloc .* I C) + kin * ke .* C; the FFT intermediates start ws_offset bytes into the workspace.
// kin < 0 selects the default Omega (the -1/2 L C term of H).  out may alias C when kin == 0.
int jdft_local_H(const jdft_basis *b, const double *Vloc, const double *C, int nb, double *HC, cudaStream_t st,
                 size_t ws_offset = 0, double scale = 1.0, double kin = -1.0);

// gemm.cu
// Out[r][c] = scale * dscale[c] * sum_k X[r][k] * (conjY ? conj(Y[c][k]) : Y[c][k]);  X [Rn][K], Y [Cn][K], Out [Rn][Cn]
// dblock != nullptr: instead of dscale, the block-diagonal matrix c128[Cn / nblk][nblk][nblk] multiplies each row's
// blocks, Out[r][a nblk + j] = scale sum_l dblock[a][j][l] (X Y^+)[r][a nblk + l].  accumulate: Out += (plain mode only).
int jdft_gemm_dotk(const jdft_basis *b, const double *X, int Rn, const double *Y, int Cn, int64_t K, int conjY,
                   double scale, const double *dscale, double *Out, void *scratch, size_t scratch_bytes,
                   cudaStream_t st, const double *dblock = nullptr, int nblk = 0, int accumulate = 0);
// Out[r][n] (+)= sum_j A[r][j] * Pm[j][n];  A [Rn][K] (K contiguous), Pm [K][Nn] (n contiguous), Out [Rn][Nn]
int jdft_apply_D(const jdft_basis *b, const double *A, int Rn, int Cn, const double *D, int D_mode, double scale, double *Out,
                 void *scratch, size_t scratch_bytes, cudaStream_t st);
// accumulate == 0 and Add != nullptr: Out = addscale * Add + A Pm  (Add [Rn][Nn]; may alias Out)
int jdft_gemm_expand(const jdft_basis *b, const double *A, int Rn, const double *Pm, int K, int64_t Nn, double *Out, int accumulate,
                     cudaStream_t st, const double *Add = nullptr, double addscale = 0.0);
