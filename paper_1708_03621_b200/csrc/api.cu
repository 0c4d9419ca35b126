// Composite entry points of the C ABI: Vnl, project, H, overlap, and the HOST-buffer variants.
#include <cstring>
#include "jdft_internal.h"

namespace {

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

int check_ptr16(const void *p, const char *who) {
    if (((uintptr_t)p) & 15) return jdft_fail(JDFT_EINVAL, "%s: data pointer not 16-byte aligned", who);
    return JDFT_OK;
}

// B1[ib][j] = scale * (D P^+ C)[j][ib] in the workspace; returns the array that holds it in *Bd
//   D_mode 0: real diagonal folded into the split-K reduction; 1: dense Hermitian, a second (small) GEMM;
//   nblk >= 2: per-atom blocks applied inside the reduction (k_splitk_reduce_block)
int project_D(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode, const double *C, int nb,
              double scale, double *B1, double *B2, void *part, size_t part_bytes, cudaStream_t st, const double **Bd) {
    int rc;
    *Bd = B1;
    if (D_mode >= 2)
        return jdft_gemm_dotk(b, C, nb, P, nproj, b->nG, 1, scale, nullptr, B1, part, part_bytes, st, D, D_mode);
    if ((rc = jdft_gemm_dotk(b, C, nb, P, nproj, b->nG, 1, scale, D_mode == 0 ? D : nullptr, B1, part, part_bytes, st))) return rc;
    if (D_mode == 1) {
        // B2[ib][j] = sum_l D[j][l] B1[ib][l]
        if ((rc = jdft_gemm_dotk(b, B1, nb, D, nproj, nproj, 0, 1.0, nullptr, B2, part, part_bytes, st))) return rc;
        *Bd = B2;
    }
    return JDFT_OK;
}

// out (+)= scale * P D P^+ C (+ addscale * Add) using the workspace for B = P^+ C, D B and the split-K partials
int vnl_impl(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode, const double *C, int nb,
             double *out, int accumulate, cudaStream_t st, const char *who, double scale = 1.0,
             const double *Add = nullptr, double addscale = 0.0) {
    if (nproj == 0 || nb == 0) {
        if (!accumulate && nb > 0) {
            if (Add) return jdft_fail(JDFT_EINVAL, "%s: internal: add-source without projectors", who);
            JDFT_CUDA(cudaMemsetAsync(out, 0, (size_t)nb * b->nG * 16, st));
        }
        return JDFT_OK;
    }
    const size_t bsz = align_up((size_t)nb * nproj * 16);
    if (!b->ws || b->ws_bytes < 3 * bsz) return jdft_fail(JDFT_EWORKSPACE, "%s: workspace missing or too small (%zu bytes needed)", who, 3 * bsz);
    char *ws = (char *)b->ws;
    double *B1 = (double *)ws, *B2 = (double *)(ws + bsz);
    void *part = ws + 2 * bsz;
    const size_t part_bytes = b->ws_bytes - 2 * bsz;
    int rc;
    const double *Bd;
    if ((rc = project_D(b, P, nproj, D, D_mode, C, nb, scale, B1, B2, part, part_bytes, st, &Bd))) return rc;
    // out[ib][n] (+)= sum_j Bd[ib][j] P[j][n]
    return jdft_gemm_expand(b, Bd, nb, P, nproj, b->nG, out, accumulate, st, Add, addscale);
}

int check_vnl_args(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode, const double *C, int nb,
                   const double *out, const char *who) {
    if (!b) return jdft_fail(JDFT_EINVAL, "%s: null basis", who);
    if (nb < 0 || nproj < 0) return jdft_fail(JDFT_EINVAL, "%s: negative size", who);
    if (D_mode < 0) return jdft_fail(JDFT_EINVAL, "%s: D_mode must be 0, 1 or a block size >= 2", who);
    if (D_mode >= 2 && nproj % D_mode != 0) return jdft_fail(JDFT_EINVAL, "%s: nproj = %d is not a multiple of the block size %d", who, nproj, D_mode);
    if (nb > 0 && (!C || !out)) return jdft_fail(JDFT_EINVAL, "%s: null data pointer", who);
    if (nproj > 0 && (!P || !D)) return jdft_fail(JDFT_EINVAL, "%s: null projector / D pointer", who);
    int rc;
    if ((rc = check_ptr16(C, who)) || (rc = check_ptr16(out, who)) || (rc = check_ptr16(P, who))) return rc;
    if (D_mode >= 1 && (rc = check_ptr16(D, who))) return rc;
    return JDFT_OK;
}

}  // namespace

extern "C" int jdft_apply_Vnl(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode,
                              const double *C, int nb, double *out, int accumulate, jdft_stream s) {
    int rc = check_vnl_args(b, P, nproj, D, D_mode, C, nb, out, "apply_Vnl");
    if (rc) return rc;
    return vnl_impl(b, P, nproj, D, D_mode, C, nb, out, accumulate, (cudaStream_t)s, "apply_Vnl");
}

extern "C" int jdft_project(const jdft_basis *b, const double *P, int nproj, const double *C, int nb, double *Bproj,
                            jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "project: null basis");
    if (nb < 0 || nproj < 0) return jdft_fail(JDFT_EINVAL, "project: negative size");
    if (nb == 0 || nproj == 0) return JDFT_OK;
    if (!P || !C || !Bproj) return jdft_fail(JDFT_EINVAL, "project: null data pointer");
    int rc;
    if ((rc = check_ptr16(C, "project")) || (rc = check_ptr16(P, "project")) || (rc = check_ptr16(Bproj, "project"))) return rc;
    if (!b->ws) return jdft_fail(JDFT_EWORKSPACE, "project: no workspace set");
    return jdft_gemm_dotk(b, C, nb, P, nproj, b->nG, 1, 1.0, nullptr, Bproj, b->ws, b->ws_bytes, (cudaStream_t)s);
}

namespace {
int apply_H_launch(const jdft_basis *b, const double *Vloc, const double *P, int nproj, const double *D, int D_mode,
                   const double *C, int nb, double *HC, cudaStream_t st) {
    int rc;
    if (nproj == 0) return jdft_local_H(b, Vloc, C, nb, HC, st);
    // Fork/join: B = D P^+ C (DMMA pipe) runs on the basis' side stream while the FFT pipeline (shared-memory / FP64
    // pipes) runs on the caller's stream; HC += P B follows both.  Needs separate workspace regions for the two.
    const size_t bsz = align_up((size_t)nb * nproj * 16);
    size_t part_bytes = b->ws_bytes / 4 < ((size_t)64 << 20) ? b->ws_bytes / 4 : ((size_t)64 << 20);
    part_bytes &= ~(size_t)255;
    const size_t gemm_bytes = 2 * bsz + part_bytes;
    const bool fork = b->opt_overlap && b->side && b->ws && part_bytes >= (size_t)nb * nproj * 16 &&
                      jdft_band_batch(b, nb, gemm_bytes) > 0;
    if (!fork) {
        if ((rc = jdft_local_H(b, Vloc, C, nb, HC, st))) return rc;
        return vnl_impl(b, P, nproj, D, D_mode, C, nb, HC, 1, st, "apply_H");
    }
    char *ws = (char *)b->ws;
    double *B1 = (double *)ws, *B2 = (double *)(ws + bsz);
    void *part = ws + 2 * bsz;
    JDFT_CUDA(cudaEventRecord(b->ev_fork, st));
    JDFT_CUDA(cudaStreamWaitEvent(b->side, b->ev_fork, 0));
    const double *Bd;
    int rc_side = project_D(b, P, nproj, D, D_mode, C, nb, 1.0, B1, B2, part, part_bytes, b->side, &Bd);
    cudaEventRecord(b->ev_join, b->side);
    rc = jdft_local_H(b, Vloc, C, nb, HC, st, gemm_bytes);
    JDFT_CUDA(cudaStreamWaitEvent(st, b->ev_join, 0));  // always join, also on error
    if (rc_side) return rc_side;
    if (rc) return rc;
    return jdft_gemm_expand(b, Bd, nb, P, nproj, b->nG, HC, 1, st);
}

}  // namespace

// CUDA-graph replay of small calls (option "graph"; automatic when nb * N <= 4 Mi points, where the ten launches of one
// call cost more than their kernels): the second call with the same arguments and workspace captures the launch
// sequence on a private stream; later calls replay it with one cudaGraphLaunch.  Capture failures fall back to direct
// launches for good.  Off while per-kernel profiling is on (events inside a graph cannot be timed).
extern "C" int jdft_apply_H(const jdft_basis *cb, const double *Vloc, const double *P, int nproj, const double *D,
                            int D_mode, const double *C, int nb, double *HC, jdft_stream s) {
    int rc = check_vnl_args(cb, P, nproj, D, D_mode, C, nb, HC, "apply_H");
    if (rc) return rc;
    if (!Vloc) return jdft_fail(JDFT_EINVAL, "apply_H: null Vloc");
    if (nb == 0) return JDFT_OK;
    cudaStream_t st = (cudaStream_t)s;
    const bool want_graph = cb->opt_graph > 0 || (cb->opt_graph < 0 && (int64_t)nb * cb->N <= ((int64_t)4 << 20));
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (want_graph) cudaStreamIsCapturing(st, &cap);
    if (!want_graph || cb->opt_profile_kernel || cb->opt_overlap || cap != cudaStreamCaptureStatusNone)
        return apply_H_launch(cb, Vloc, P, nproj, D, D_mode, C, nb, HC, st);
    jdft_basis *b = const_cast<jdft_basis *>(cb);   // the graph cache is bookkeeping, not state of the operator
    JdftGraphEntry *g = nullptr;
    for (JdftGraphEntry &e : b->graphs)
        if (e.V == Vloc && e.P == P && e.D == D && e.C == C && e.HC == HC && e.ws == b->ws && e.ws_bytes == b->ws_bytes &&
            e.nproj == nproj && e.D_mode == D_mode && e.nb == nb)
            g = &e;
    if (!g) {
        if (b->graphs.size() >= 8) {
            if (b->graphs.front().exec) cudaGraphExecDestroy(b->graphs.front().exec);
            b->graphs.erase(b->graphs.begin());
        }
        b->graphs.push_back(JdftGraphEntry{Vloc, P, D, C, HC, b->ws, b->ws_bytes, nproj, D_mode, nb, 0, 0, nullptr});
        g = &b->graphs.back();
    }
    if (g->exec) {
        JDFT_CUDA(cudaGraphLaunch(g->exec, st));
        jdft_count_launch((int)g->launches);
        return JDFT_OK;
    }
    if (g->seen++ == 0) return apply_H_launch(b, Vloc, P, nproj, D, D_mode, C, nb, HC, st);   // warms kernel attributes
    if (!b->gstream && cudaStreamCreateWithFlags(&b->gstream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError();
        b->opt_graph = 0;
        return apply_H_launch(b, Vloc, P, nproj, D, D_mode, C, nb, HC, st);
    }
    const int64_t before = jdft_launch_count_peek();
    cudaGraph_t graph = nullptr;
    bool ok = cudaStreamBeginCapture(b->gstream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
        rc = apply_H_launch(b, Vloc, P, nproj, D, D_mode, C, nb, HC, b->gstream);
        ok = cudaStreamEndCapture(b->gstream, &graph) == cudaSuccess && rc == JDFT_OK && graph;
    }
    const int64_t captured = jdft_launch_count_peek() - before;
    jdft_count_launch(-(int)captured);               // nothing ran yet
    if (ok) ok = cudaGraphInstantiate(&g->exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    if (!ok) {
        cudaGetLastError();
        g->exec = nullptr;
        b->opt_graph = 0;                            // do not try again on this basis
        return apply_H_launch(b, Vloc, P, nproj, D, D_mode, C, nb, HC, st);
    }
    g->launches = captured;
    JDFT_CUDA(cudaGraphLaunch(g->exec, st));
    jdft_count_launch((int)captured);
    return JDFT_OK;
}

extern "C" int jdft_overlap(const jdft_basis *b, const double *C1, int nb1, const double *C2, int nb2, double *M,
                            jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "overlap: null basis");
    if (nb1 < 0 || nb2 < 0) return jdft_fail(JDFT_EINVAL, "overlap: negative size");
    if (nb1 == 0 || nb2 == 0) return JDFT_OK;
    if (!C1 || !C2 || !M) return jdft_fail(JDFT_EINVAL, "overlap: null data pointer");
    int rc;
    if ((rc = check_ptr16(C1, "overlap")) || (rc = check_ptr16(C2, "overlap")) || (rc = check_ptr16(M, "overlap"))) return rc;
    if (!b->ws) return jdft_fail(JDFT_EWORKSPACE, "overlap: no workspace set");
    // M stored column-major nb1 x nb2 == row-major [nb2][nb1]:  M[bb][a] = Omega sum_n C2[bb][n] conj(C1[a][n])
    return jdft_gemm_dotk(b, C2, nb2, C1, nb1, b->nG, 1, b->volume, nullptr, M, b->ws, b->ws_bytes, (cudaStream_t)s);
}

extern "C" int jdft_subspace(const jdft_basis *b, const double *C1, int nb1, const double *X2, int nb2, double *M,
                             jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "subspace: null basis");
    if (nb1 < 0 || nb2 < 0) return jdft_fail(JDFT_EINVAL, "subspace: negative size");
    if (nb1 == 0 || nb2 == 0) return JDFT_OK;
    if (!C1 || !X2 || !M) return jdft_fail(JDFT_EINVAL, "subspace: null data pointer");
    int rc;
    if ((rc = check_ptr16(C1, "subspace")) || (rc = check_ptr16(X2, "subspace")) || (rc = check_ptr16(M, "subspace"))) return rc;
    if (!b->ws) return jdft_fail(JDFT_EWORKSPACE, "subspace: no workspace set");
    // column-major nb1 x nb2 == row-major [nb2][nb1]:  M[bb][a] = sum_n X2[bb][n] conj(C1[a][n])
    return jdft_gemm_dotk(b, X2, nb2, C1, nb1, b->nG, 1, 1.0, nullptr, M, b->ws, b->ws_bytes, (cudaStream_t)s);
}

// ---- ultrasoft generalised overlap (reading 24) ------------------
// O_us C = Omega (C + P Q P^+ C): B = Omega Q P^+ C (Q folded into the split-K reduction), then ONE expand GEMM whose
// epilogue adds Omega C, so OC is written once and C read once.
extern "C" int jdft_apply_O_us(const jdft_basis *b, const double *P, int nproj, const double *Q, int Q_mode,
                               const double *C, int nb, double *OC, jdft_stream s) {
    int rc = check_vnl_args(b, P, nproj, Q, Q_mode, C, nb, OC, "apply_O_us");
    if (rc) return rc;
    if (nb == 0) return JDFT_OK;
    if (nproj == 0) return jdft_apply_O(b, C, nb, OC, s);
    return vnl_impl(b, P, nproj, Q, Q_mode, C, nb, OC, 0, (cudaStream_t)s, "apply_O_us", b->volume, C, b->volume);
}

// M = C1^+ O_us C2 = Omega C1^+ C2 + (P^+ C1)^+ (Omega Q P^+ C2): the big K = nG contraction as in jdft_overlap, the
// projector term as two projections and one small K = nproj contraction accumulated into M by its reduction.
extern "C" int jdft_overlap_us(const jdft_basis *b, const double *P, int nproj, const double *Q, int Q_mode,
                               const double *C1, int nb1, const double *C2, int nb2, double *M, jdft_stream s) {
    if (!b) return jdft_fail(JDFT_EINVAL, "overlap_us: null basis");
    if (nb1 < 0 || nb2 < 0) return jdft_fail(JDFT_EINVAL, "overlap_us: negative size");
    if (nb1 == 0 || nb2 == 0) return JDFT_OK;
    int rc = check_vnl_args(b, P, nproj, Q, Q_mode, C1, nb1, M, "overlap_us");
    if (rc) return rc;
    if (!C2) return jdft_fail(JDFT_EINVAL, "overlap_us: null data pointer");
    if ((rc = check_ptr16(C2, "overlap_us"))) return rc;
    if ((rc = jdft_overlap(b, C1, nb1, C2, nb2, M, s))) return rc;
    if (nproj == 0) return JDFT_OK;
    cudaStream_t st = (cudaStream_t)s;
    const size_t bs1 = align_up((size_t)nb1 * nproj * 16), bs2 = align_up((size_t)nb2 * nproj * 16);
    if (b->ws_bytes < bs1 + 2 * bs2 + 16 * (size_t)(nb1 > nb2 ? nb1 : nb2) * nproj)
        return jdft_fail(JDFT_EWORKSPACE, "overlap_us: workspace too small (%zu bytes needed)", bs1 + 2 * bs2 + 16 * (size_t)(nb1 > nb2 ? nb1 : nb2) * nproj);
    char *ws = (char *)b->ws;
    double *A1 = (double *)ws, *B1 = (double *)(ws + bs1), *B2 = (double *)(ws + bs1 + bs2);
    void *part = ws + bs1 + 2 * bs2;
    const size_t part_bytes = b->ws_bytes - (bs1 + 2 * bs2);
    // A1[a][j] = (P^+ C1)[j][a];  Bd[bb][j] = Omega (Q P^+ C2)[j][bb]
    if ((rc = jdft_gemm_dotk(b, C1, nb1, P, nproj, b->nG, 1, 1.0, nullptr, A1, part, part_bytes, st))) return rc;
    const double *Bd;
    if (C1 == C2 && nb1 == nb2) {   // one projection serves both sides: Bd = Omega Q A1
        if ((rc = jdft_apply_D(b, A1, nb1, nproj, Q, Q_mode, b->volume, B1, part, part_bytes, st))) return rc;
        Bd = B1;
    } else if ((rc = project_D(b, P, nproj, Q, Q_mode, C2, nb2, b->volume, B1, B2, part, part_bytes, st, &Bd))) {
        return rc;
    }
    // M[bb][a] += sum_j Bd[bb][j] conj(A1[a][j])
    return jdft_gemm_dotk(b, Bd, nb2, A1, nb1, nproj, 1, 1.0, nullptr, M, part, part_bytes, st, nullptr, 0, 1);
}

// ---- HOST-buffer variants ----------------------------------------------------------------------------------
namespace {
int host_buf(jdft_basis *b, int slot, size_t bytes, void **out) {
    if (b->hb_bytes[slot] < bytes) {
        if (b->hb[slot]) cudaFree(b->hb[slot]);
        b->hb[slot] = nullptr;
        b->hb_bytes[slot] = 0;
        cudaError_t e = cudaMalloc(&b->hb[slot], bytes ? bytes : 16);
        if (e != cudaSuccess) { cudaGetLastError(); return jdft_fail(JDFT_ENOMEM, "host variant: cudaMalloc of %zu bytes failed", bytes); }
        b->hb_bytes[slot] = bytes;
    }
    *out = b->hb[slot];
    return JDFT_OK;
}
}  // namespace

namespace {

// streams / events of the HOST-buffer pipeline, created on first use (all non-blocking: no legacy-stream coupling)
int host_streams(jdft_basis *b, int nchunk) {
    for (int i = 0; i < 3; i++)
        if (!b->hs[i]) JDFT_CUDA(cudaStreamCreateWithFlags(&b->hs[i], cudaStreamNonBlocking));
    while ((int)b->hev.size() < 2 * nchunk + 2) {
        cudaEvent_t e;
        JDFT_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        b->hev.push_back(e);
    }
    return JDFT_OK;
}

// H C for HOST bands through device copies, pipelined over band chunks: the H2D copy of chunk i+1, the kernels of chunk i
// and the D2H copy of chunk i-1 run at the same time on three streams (PCIe is full duplex).  dV / dP / dD are DEVICE
// operands; with upload_ops they are first filled from the HOST arrays Vh / Ph / Dh, ordered so that the FFT pipeline of
// chunk 0 starts as soon as V_loc and the chunk have landed while the (larger) projector block is still in flight.
int host_H_pipeline(jdft_basis *b, bool upload_ops, const double *Vh, const double *Ph, const double *Dh, double *dV,
                    double *dP, double *dD, int nproj, int D_mode, size_t vb, size_t pb, size_t db, const double *C,
                    int nb, double *HC, const char *who) {
    const int64_t nG = b->nG;
    const size_t cb = (size_t)nb * nG * 16;
    void *dCv, *dHCv, *dW;
    int rc;
    b->h_C_nb = 0;
    if ((rc = host_buf(b, 0, cb, &dCv)) || (rc = host_buf(b, 1, cb, &dHCv))) return rc;
    double *dC = (double *)dCv, *dHC = (double *)dHCv;
    int nchunk = b->opt_host_chunk > 0 ? (int)((nb + b->opt_host_chunk - 1) / b->opt_host_chunk) : (nb + 63) / 64;   // chunks of <= 64 bands (option "host_chunk"; measured: config 5 73.3 / 70.5 / 91.0 ms at 128 / 64 / 32), at most 16
    if (nchunk > 16) nchunk = 16;
    const int nbc = (nb + nchunk - 1) / nchunk;
    nchunk = (nb + nbc - 1) / nbc;
    if ((rc = host_streams(b, nchunk))) return rc;
    void *saved_ws = b->ws;
    size_t saved_bytes = b->ws_bytes;
    if (!b->ws) {
        size_t need = jdft_workspace_bytes(b, nbc < 64 ? nbc : 64, nproj > nbc ? nproj : nbc);
        if ((rc = host_buf(b, 5, need, &dW))) return rc;
        b->ws = dW;
        b->ws_bytes = need;
    }
    // workspace split as in the fork/join path of jdft_apply_H: GEMM scratch in front, FFT intermediates behind
    const size_t bsz = align_up((size_t)nbc * nproj * 16);
    size_t part_bytes = b->ws_bytes / 4 < ((size_t)64 << 20) ? b->ws_bytes / 4 : ((size_t)64 << 20);
    part_bytes &= ~(size_t)255;
    const size_t gemm_bytes = nproj > 0 ? 2 * bsz + part_bytes : 0;
    if ((nproj > 0 && part_bytes < (size_t)nbc * nproj * 16) || jdft_band_batch(b, nbc, gemm_bytes) == 0) {
        b->ws = saved_ws;
        b->ws_bytes = saved_bytes;
        return jdft_fail(JDFT_EWORKSPACE, "%s: workspace too small", who);
    }
    char *ws = (char *)b->ws;
    double *B1 = (double *)ws, *B2 = (double *)(ws + bsz);
    cudaStream_t sin = b->hs[0], sc = b->hs[1], sout = b->hs[2];
    cudaEvent_t evV = b->hev[0], evOps = b->hev[1];
    cudaError_t e = cudaSuccess;
    rc = JDFT_OK;
    for (int i = 0; i < nchunk && e == cudaSuccess && !rc; i++) {
        const int b0 = i * nbc, nbt = nb - b0 < nbc ? nb - b0 : nbc;
        const size_t off = (size_t)b0 * nG * 2;          // in doubles
        cudaEvent_t evIn = b->hev[2 + 2 * i], evDone = b->hev[3 + 2 * i];
        if (i == 0 && upload_ops) {
            e = cudaMemcpyAsync(dV, Vh, vb, cudaMemcpyHostToDevice, sin);
            if (e == cudaSuccess) e = cudaEventRecord(evV, sin);
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(dC + off, C + off, (size_t)nbt * nG * 16, cudaMemcpyHostToDevice, sin);
        if (e == cudaSuccess) e = cudaEventRecord(evIn, sin);
        if (i == 0 && upload_ops && nproj > 0) {
            if (e == cudaSuccess) e = cudaMemcpyAsync(dP, Ph, pb, cudaMemcpyHostToDevice, sin);
            if (e == cudaSuccess) e = cudaMemcpyAsync(dD, Dh, db, cudaMemcpyHostToDevice, sin);
            if (e == cudaSuccess) e = cudaEventRecord(evOps, sin);
        }
        if (e == cudaSuccess && i == 0 && upload_ops) e = cudaStreamWaitEvent(sc, evV, 0);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(sc, evIn, 0);
        if (e != cudaSuccess) break;
        rc = jdft_local_H(b, dV, dC + off, nbt, dHC + off, sc, gemm_bytes);
        if (!rc && nproj > 0) {
            if (i == 0 && upload_ops) e = cudaStreamWaitEvent(sc, evOps, 0);
            const double *Bd = B1;
            if (e == cudaSuccess) rc = project_D(b, dP, nproj, dD, D_mode, dC + off, nbt, 1.0, B1, B2, ws + 2 * bsz, part_bytes, sc, &Bd);
            if (e == cudaSuccess && !rc) rc = jdft_gemm_expand(b, Bd, nbt, dP, nproj, nG, dHC + off, 1, sc);
        }
        if (e == cudaSuccess && !rc) e = cudaEventRecord(evDone, sc);
        if (e == cudaSuccess && !rc) e = cudaStreamWaitEvent(sout, evDone, 0);
        if (e == cudaSuccess && !rc) e = cudaMemcpyAsync(HC + off, dHC + off, (size_t)nbt * nG * 16, cudaMemcpyDeviceToHost, sout);
    }
    b->ws = saved_ws;
    b->ws_bytes = saved_bytes;
    // always drain the three streams before returning (also on error: the caller may free its buffers)
    cudaError_t e1 = cudaStreamSynchronize(sin), e2 = cudaStreamSynchronize(sc), e3 = cudaStreamSynchronize(sout);
    if (rc) return rc;
    if (e != cudaSuccess) return jdft_cuda_fail(e, who);
    if (e1 != cudaSuccess) return jdft_cuda_fail(e1, who);
    if (e2 != cudaSuccess) return jdft_cuda_fail(e2, who);
    if (e3 != cudaSuccess) return jdft_cuda_fail(e3, who);
    b->h_C_nb = nb;   // the band block stays on the device (hb[0]) for jdft_overlap_host_resident
    return JDFT_OK;
}

}  // namespace

extern "C" int jdft_apply_H_host(jdft_basis *b, const double *Vloc, const double *P, int nproj, const double *D,
                                 int D_mode, const double *C, int nb, double *HC) {
    if (!b) return jdft_fail(JDFT_EINVAL, "apply_H_host: null basis");
    if (nb < 0 || nproj < 0 || D_mode < 0 || (D_mode >= 2 && nproj % D_mode != 0)) return jdft_fail(JDFT_EINVAL, "apply_H_host: bad size or mode");
    if (!Vloc || (nb > 0 && (!C || !HC)) || (nproj > 0 && (!P || !D))) return jdft_fail(JDFT_EINVAL, "apply_H_host: null pointer");
    if (nb == 0) return JDFT_OK;
    JDFT_CUDA(cudaSetDevice(b->device));
    const size_t vb = (size_t)b->N * 8, pb = (size_t)nproj * b->nG * 16;
    const size_t db = D_mode == 0 ? (size_t)nproj * 8 : (D_mode == 1 ? (size_t)nproj * nproj * 16 : (size_t)nproj * D_mode * 16);
    void *dV, *dP, *dD;
    int rc;
    if ((rc = host_buf(b, 2, vb, &dV)) || (rc = host_buf(b, 3, pb, &dP)) || (rc = host_buf(b, 4, db, &dD))) return rc;
    b->h_ops_set = 0;   // the resident operators (if any) have just been overwritten
    return host_H_pipeline(b, true, Vloc, P, D, (double *)dV, (double *)dP, (double *)dD, nproj, D_mode, vb, pb, db, C, nb, HC,
                           "apply_H_host");
}

// Resident operators: V_loc, P and D are uploaded ONCE (they stay the same over the many H applications of one SCF
// iteration); jdft_apply_H_host_resident then moves only the bands in and H C out.
extern "C" int jdft_host_set_operators(jdft_basis *b, const double *Vloc, const double *P, int nproj, const double *D,
                                       int D_mode) {
    if (!b) return jdft_fail(JDFT_EINVAL, "host_set_operators: null basis");
    if (nproj < 0 || D_mode < 0 || (D_mode >= 2 && nproj % D_mode != 0)) return jdft_fail(JDFT_EINVAL, "host_set_operators: bad size or mode");
    if (!Vloc || (nproj > 0 && (!P || !D))) return jdft_fail(JDFT_EINVAL, "host_set_operators: null pointer");
    JDFT_CUDA(cudaSetDevice(b->device));
    const size_t vb = (size_t)b->N * 8, pb = (size_t)nproj * b->nG * 16;
    const size_t db = D_mode == 0 ? (size_t)nproj * 8 : (D_mode == 1 ? (size_t)nproj * nproj * 16 : (size_t)nproj * D_mode * 16);
    void *dV, *dP, *dD;
    int rc;
    if ((rc = host_buf(b, 2, vb, &dV)) || (rc = host_buf(b, 3, pb, &dP)) || (rc = host_buf(b, 4, db, &dD))) return rc;
    if ((rc = host_streams(b, 1))) return rc;
    b->h_ops_set = 0;
    JDFT_CUDA(cudaMemcpyAsync(dV, Vloc, vb, cudaMemcpyHostToDevice, b->hs[0]));
    if (nproj > 0) {
        JDFT_CUDA(cudaMemcpyAsync(dP, P, pb, cudaMemcpyHostToDevice, b->hs[0]));
        JDFT_CUDA(cudaMemcpyAsync(dD, D, db, cudaMemcpyHostToDevice, b->hs[0]));
    }
    JDFT_CUDA(cudaStreamSynchronize(b->hs[0]));
    b->h_ops_set = 1;
    b->h_nproj = nproj;
    b->h_D_mode = D_mode;
    return JDFT_OK;
}

extern "C" int jdft_apply_H_host_resident(jdft_basis *b, const double *C, int nb, double *HC) {
    if (!b) return jdft_fail(JDFT_EINVAL, "apply_H_host_resident: null basis");
    if (!b->h_ops_set) return jdft_fail(JDFT_EINVAL, "apply_H_host_resident: call jdft_host_set_operators first");
    if (nb < 0 || (nb > 0 && (!C || !HC))) return jdft_fail(JDFT_EINVAL, "apply_H_host_resident: bad size or null pointer");
    if (nb == 0) return JDFT_OK;
    JDFT_CUDA(cudaSetDevice(b->device));
    return host_H_pipeline(b, false, nullptr, nullptr, nullptr, (double *)b->hb[2], (double *)b->hb[3], (double *)b->hb[4],
                           b->h_nproj, b->h_D_mode, 0, 0, 0, C, nb, HC, "apply_H_host_resident");
}

extern "C" int jdft_overlap_host(jdft_basis *b, const double *C1, int nb1, const double *C2, int nb2, double *M) {
    if (!b) return jdft_fail(JDFT_EINVAL, "overlap_host: null basis");
    if (nb1 < 0 || nb2 < 0) return jdft_fail(JDFT_EINVAL, "overlap_host: negative size");
    if (nb1 == 0 || nb2 == 0) return JDFT_OK;
    if (!C1 || !C2 || !M) return jdft_fail(JDFT_EINVAL, "overlap_host: null pointer");
    JDFT_CUDA(cudaSetDevice(b->device));
    b->h_C_nb = 0;
    const bool same = C1 == C2 && nb1 == nb2;   // one upload; the device call then takes the Hermitian-triangle path
    const size_t b1 = (size_t)nb1 * b->nG * 16, b2 = (size_t)nb2 * b->nG * 16, mb = (size_t)nb1 * nb2 * 16;
    void *d1, *d2, *dM, *dW;
    int rc;
    if ((rc = host_buf(b, 0, b1, &d1)) || (rc = host_buf(b, 6, mb, &dM))) return rc;
    d2 = d1;
    if (!same && (rc = host_buf(b, 1, b2, &d2))) return rc;
    if ((rc = host_streams(b, 1))) return rc;
    void *saved_ws = b->ws;
    size_t saved_bytes = b->ws_bytes;
    if (!b->ws) {
        size_t need = jdft_workspace_bytes(b, 1, nb1 > nb2 ? nb1 : nb2);
        if ((rc = host_buf(b, 5, need, &dW))) return rc;
        b->ws = dW;
        b->ws_bytes = need;
    }
    cudaStream_t st = b->hs[1];
    cudaError_t e = cudaMemcpyAsync(d1, C1, b1, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && !same) e = cudaMemcpyAsync(d2, C2, b2, cudaMemcpyHostToDevice, st);
    rc = e == cudaSuccess ? jdft_overlap(b, (const double *)d1, nb1, (const double *)d2, nb2, (double *)dM, st)
                          : jdft_cuda_fail(e, "overlap_host H2D");
    b->ws = saved_ws;
    b->ws_bytes = saved_bytes;
    if (rc) { cudaStreamSynchronize(st); return rc; }
    JDFT_CUDA(cudaMemcpyAsync(M, dM, mb, cudaMemcpyDeviceToHost, st));
    JDFT_CUDA(cudaStreamSynchronize(st));
    return JDFT_OK;
}

// M = C^+ O C of the band block that the last jdft_apply_H_host / jdft_apply_H_host_resident call left on the device:
// H C and the overlap of the same bands are needed together in every SCF / minimiser step, so the second
// upload of C is skipped; only the nb x nb result crosses PCIe.
extern "C" int jdft_overlap_host_resident(jdft_basis *b, int nb, double *M) {
    if (!b) return jdft_fail(JDFT_EINVAL, "overlap_host_resident: null basis");
    if (nb <= 0 || !M) return jdft_fail(JDFT_EINVAL, "overlap_host_resident: bad size or null pointer");
    if (b->h_C_nb != nb) return jdft_fail(JDFT_EINVAL, "overlap_host_resident: the last apply_H_host call left %d bands on the device, not %d", b->h_C_nb, nb);
    JDFT_CUDA(cudaSetDevice(b->device));
    const size_t mb = (size_t)nb * nb * 16;
    void *dM, *dW;
    int rc;
    if ((rc = host_buf(b, 6, mb, &dM))) return rc;
    if ((rc = host_streams(b, 1))) return rc;
    void *saved_ws = b->ws;
    size_t saved_bytes = b->ws_bytes;
    if (!b->ws) {
        size_t need = jdft_workspace_bytes(b, 1, nb);
        if ((rc = host_buf(b, 5, need, &dW))) return rc;
        b->ws = dW;
        b->ws_bytes = need;
    }
    cudaStream_t st = b->hs[1];
    rc = jdft_overlap(b, (const double *)b->hb[0], nb, (const double *)b->hb[0], nb, (double *)dM, st);
    b->ws = saved_ws;
    b->ws_bytes = saved_bytes;
    if (rc) { cudaStreamSynchronize(st); return rc; }
    JDFT_CUDA(cudaMemcpyAsync(M, dM, mb, cudaMemcpyDeviceToHost, st));
    JDFT_CUDA(cudaStreamSynchronize(st));
    return JDFT_OK;
}
