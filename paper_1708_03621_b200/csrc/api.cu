// Composite entry points of the C ABI: Vnl, project, H, overlap, and the HOST-buffer variants.
#include <cstring>
#include "jdft_internal.h"

namespace {

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

int check_ptr16(const void *p, const char *who) {
    if (((uintptr_t)p) & 15) return jdft_fail(JDFT_EINVAL, "%s: data pointer not 16-byte aligned", who);
    return JDFT_OK;
}

// out (+)= P D P^+ C using the workspace for B = P^+ C, D B and the split-K partials
int vnl_impl(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode, const double *C, int nb,
             double *out, int accumulate, cudaStream_t st, const char *who) {
    if (nproj == 0 || nb == 0) {
        if (!accumulate && nb > 0)
            JDFT_CUDA(cudaMemsetAsync(out, 0, (size_t)nb * b->nG * 16, st));
        return JDFT_OK;
    }
    const size_t bsz = align_up((size_t)nb * nproj * 16);
    if (!b->ws || b->ws_bytes < 3 * bsz) return jdft_fail(JDFT_EWORKSPACE, "%s: workspace missing or too small (%zu bytes needed)", who, 3 * bsz);
    char *ws = (char *)b->ws;
    double *B1 = (double *)ws, *B2 = (double *)(ws + bsz);
    void *part = ws + 2 * bsz;
    const size_t part_bytes = b->ws_bytes - 2 * bsz;
    int rc;
    // B1[ib][j] = D_j * sum_n conj(P[j][n]) C[ib][n]   (D folded in when diagonal)
    if ((rc = jdft_gemm_dotk(b, C, nb, P, nproj, b->nG, 1, 1.0, D_mode == 0 ? D : nullptr, B1, part, part_bytes, st))) return rc;
    const double *Bd = B1;
    if (D_mode == 1) {
        // B2[ib][j] = sum_l D[j][l] B1[ib][l]
        if ((rc = jdft_gemm_dotk(b, B1, nb, D, nproj, nproj, 0, 1.0, nullptr, B2, part, part_bytes, st))) return rc;
        Bd = B2;
    }
    // out[ib][n] (+)= sum_j Bd[ib][j] P[j][n]
    return jdft_gemm_expand(b, Bd, nb, P, nproj, b->nG, out, accumulate, st);
}

int check_vnl_args(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode, const double *C, int nb,
                   const double *out, const char *who) {
    if (!b) return jdft_fail(JDFT_EINVAL, "%s: null basis", who);
    if (nb < 0 || nproj < 0) return jdft_fail(JDFT_EINVAL, "%s: negative size", who);
    if (D_mode != 0 && D_mode != 1) return jdft_fail(JDFT_EINVAL, "%s: D_mode must be 0 or 1", who);
    if (nb > 0 && (!C || !out)) return jdft_fail(JDFT_EINVAL, "%s: null data pointer", who);
    if (nproj > 0 && (!P || !D)) return jdft_fail(JDFT_EINVAL, "%s: null projector / D pointer", who);
    int rc;
    if ((rc = check_ptr16(C, who)) || (rc = check_ptr16(out, who)) || (rc = check_ptr16(P, who))) return rc;
    if (D_mode == 1 && (rc = check_ptr16(D, who))) return rc;
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

extern "C" int jdft_apply_H(const jdft_basis *b, const double *Vloc, const double *P, int nproj, const double *D,
                            int D_mode, const double *C, int nb, double *HC, jdft_stream s) {
    int rc = check_vnl_args(b, P, nproj, D, D_mode, C, nb, HC, "apply_H");
    if (rc) return rc;
    if (!Vloc) return jdft_fail(JDFT_EINVAL, "apply_H: null Vloc");
    if (nb == 0) return JDFT_OK;
    cudaStream_t st = (cudaStream_t)s;
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
    int rc_side = jdft_gemm_dotk(b, C, nb, P, nproj, b->nG, 1, 1.0, D_mode == 0 ? D : nullptr, B1, part, part_bytes, b->side);
    const double *Bd = B1;
    if (!rc_side && D_mode == 1) {
        rc_side = jdft_gemm_dotk(b, B1, nb, D, nproj, nproj, 0, 1.0, nullptr, B2, part, part_bytes, b->side);
        Bd = B2;
    }
    cudaEventRecord(b->ev_join, b->side);
    rc = jdft_local_H(b, Vloc, C, nb, HC, st, gemm_bytes);
    JDFT_CUDA(cudaStreamWaitEvent(st, b->ev_join, 0));  // always join, also on error
    if (rc_side) return rc_side;
    if (rc) return rc;
    return jdft_gemm_expand(b, Bd, nb, P, nproj, b->nG, HC, 1, st);
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

extern "C" int jdft_apply_H_host(jdft_basis *b, const double *Vloc, const double *P, int nproj, const double *D,
                                 int D_mode, const double *C, int nb, double *HC) {
    if (!b) return jdft_fail(JDFT_EINVAL, "apply_H_host: null basis");
    if (nb < 0 || nproj < 0 || (D_mode != 0 && D_mode != 1)) return jdft_fail(JDFT_EINVAL, "apply_H_host: bad size or mode");
    if (!Vloc || (nb > 0 && (!C || !HC)) || (nproj > 0 && (!P || !D))) return jdft_fail(JDFT_EINVAL, "apply_H_host: null pointer");
    if (nb == 0) return JDFT_OK;
    JDFT_CUDA(cudaSetDevice(b->device));
    const size_t cb = (size_t)nb * b->nG * 16, vb = (size_t)b->N * 8, pb = (size_t)nproj * b->nG * 16;
    const size_t db = D_mode == 0 ? (size_t)nproj * 8 : (size_t)nproj * nproj * 16;
    void *dC, *dHC, *dV, *dP, *dD, *dW;
    int rc;
    if ((rc = host_buf(b, 0, cb, &dC)) || (rc = host_buf(b, 1, cb, &dHC)) || (rc = host_buf(b, 2, vb, &dV)) ||
        (rc = host_buf(b, 3, pb, &dP)) || (rc = host_buf(b, 4, db, &dD)))
        return rc;
    void *saved_ws = b->ws;
    size_t saved_bytes = b->ws_bytes;
    if (!b->ws) {
        const int rows = nproj > nb ? nproj : nb;
        size_t need = jdft_workspace_bytes(b, 8, rows);
        if ((rc = host_buf(b, 5, need, &dW))) return rc;
        b->ws = dW;
        b->ws_bytes = need;
    }
    // Copy-in on the basis' side stream in the order the kernels need the data (C, Vloc, then P, D); the FFT pipeline
    // starts as soon as C and Vloc have landed and runs while the (larger) projector block is still in flight; the
    // projector GEMMs wait for the second event.  Pinned host buffers make the copies truly asynchronous.
    cudaStream_t st = 0, cp = b->side ? b->side : (cudaStream_t)0;
    cudaError_t e = cudaMemcpyAsync(dC, C, cb, cudaMemcpyHostToDevice, cp);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dV, Vloc, vb, cudaMemcpyHostToDevice, cp);
    if (e == cudaSuccess && cp != st) e = cudaEventRecord(b->ev_fork, cp);
    if (e == cudaSuccess && nproj > 0) e = cudaMemcpyAsync(dP, P, pb, cudaMemcpyHostToDevice, cp);
    if (e == cudaSuccess && nproj > 0) e = cudaMemcpyAsync(dD, D, db, cudaMemcpyHostToDevice, cp);
    if (e == cudaSuccess && cp != st) e = cudaEventRecord(b->ev_join, cp);
    if (e == cudaSuccess && cp != st) e = cudaStreamWaitEvent(st, b->ev_fork, 0);
    rc = e == cudaSuccess ? JDFT_OK : jdft_cuda_fail(e, "apply_H_host H2D");
    if (!rc) {
        if (nproj == 0) {
            rc = jdft_local_H(b, (const double *)dV, (const double *)dC, nb, (double *)dHC, st);
        } else {
            // same split of the workspace as the fork/join path of jdft_apply_H: GEMM scratch in front, FFT behind
            const size_t bsz = align_up((size_t)nb * nproj * 16);
            size_t part_bytes = b->ws_bytes / 4 < ((size_t)64 << 20) ? b->ws_bytes / 4 : ((size_t)64 << 20);
            part_bytes &= ~(size_t)255;
            const size_t gemm_bytes = 2 * bsz + part_bytes;
            if (part_bytes < (size_t)nb * nproj * 16 || jdft_band_batch(b, nb, gemm_bytes) == 0) {
                rc = jdft_fail(JDFT_EWORKSPACE, "apply_H_host: workspace too small");
            } else {
                char *ws = (char *)b->ws;
                double *B1 = (double *)ws, *B2 = (double *)(ws + bsz);
                rc = jdft_local_H(b, (const double *)dV, (const double *)dC, nb, (double *)dHC, st, gemm_bytes);
                if (cp != st) {
                    cudaError_t e2 = cudaStreamWaitEvent(st, b->ev_join, 0);
                    if (!rc && e2 != cudaSuccess) rc = jdft_cuda_fail(e2, "apply_H_host join");
                }
                if (!rc) rc = jdft_gemm_dotk(b, (const double *)dC, nb, (const double *)dP, nproj, b->nG, 1, 1.0,
                                             D_mode == 0 ? (const double *)dD : nullptr, B1, ws + 2 * bsz, part_bytes, st);
                const double *Bd = B1;
                if (!rc && D_mode == 1) {
                    rc = jdft_gemm_dotk(b, B1, nb, (const double *)dD, nproj, nproj, 0, 1.0, nullptr, B2, ws + 2 * bsz, part_bytes, st);
                    Bd = B2;
                }
                if (!rc) rc = jdft_gemm_expand(b, Bd, nb, (const double *)dP, nproj, b->nG, (double *)dHC, 1, st);
            }
        }
    }
    b->ws = saved_ws;
    b->ws_bytes = saved_bytes;
    if (rc) { cudaStreamSynchronize(cp); cudaStreamSynchronize(st); return rc; }
    JDFT_CUDA(cudaMemcpyAsync(HC, dHC, cb, cudaMemcpyDeviceToHost, st));
    JDFT_CUDA(cudaStreamSynchronize(st));
    JDFT_CUDA(cudaStreamSynchronize(cp));
    return JDFT_OK;
}

extern "C" int jdft_overlap_host(jdft_basis *b, const double *C1, int nb1, const double *C2, int nb2, double *M) {
    if (!b) return jdft_fail(JDFT_EINVAL, "overlap_host: null basis");
    if (nb1 < 0 || nb2 < 0) return jdft_fail(JDFT_EINVAL, "overlap_host: negative size");
    if (nb1 == 0 || nb2 == 0) return JDFT_OK;
    if (!C1 || !C2 || !M) return jdft_fail(JDFT_EINVAL, "overlap_host: null pointer");
    JDFT_CUDA(cudaSetDevice(b->device));
    const size_t b1 = (size_t)nb1 * b->nG * 16, b2 = (size_t)nb2 * b->nG * 16, mb = (size_t)nb1 * nb2 * 16;
    void *d1, *d2, *dM, *dW;
    int rc;
    if ((rc = host_buf(b, 0, b1, &d1)) || (rc = host_buf(b, 1, b2, &d2)) || (rc = host_buf(b, 6, mb, &dM))) return rc;
    void *saved_ws = b->ws;
    size_t saved_bytes = b->ws_bytes;
    if (!b->ws) {
        size_t need = jdft_workspace_bytes(b, 1, nb1 > nb2 ? nb1 : nb2);
        if ((rc = host_buf(b, 5, need, &dW))) return rc;
        b->ws = dW;
        b->ws_bytes = need;
    }
    cudaStream_t st = 0;
    cudaError_t e = cudaMemcpyAsync(d1, C1, b1, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d2, C2, b2, cudaMemcpyHostToDevice, st);
    rc = e == cudaSuccess ? jdft_overlap(b, (const double *)d1, nb1, (const double *)d2, nb2, (double *)dM, st)
                          : jdft_cuda_fail(e, "overlap_host H2D");
    b->ws = saved_ws;
    b->ws_bytes = saved_bytes;
    if (rc) return rc;
    JDFT_CUDA(cudaMemcpyAsync(M, dM, mb, cudaMemcpyDeviceToHost, st));
    JDFT_CUDA(cudaStreamSynchronize(st));
    return JDFT_OK;
}
