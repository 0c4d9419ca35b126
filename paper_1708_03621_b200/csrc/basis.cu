// Basis construction (host) and the bookkeeping entry points of the C ABI.
// Definitions: include/jdft.h (DESIGN.md section 3 readings 6-12).
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include "jdft_internal.h"
#include "tma.cuh"

static thread_local char g_err[512] = "";
static thread_local int64_t g_launches = 0;

int jdft_fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
int jdft_cuda_fail(cudaError_t e, const char *what) {
    return jdft_fail(JDFT_ECUDA, "CUDA error '%s' in %s", cudaGetErrorString(e), what);
}
void jdft_count_launch(int n) { g_launches += n; }
int64_t jdft_launch_count_peek() { return g_launches; }
void jdft_graphs_clear(jdft_basis *b) {
    for (JdftGraphEntry &g : b->graphs)
        if (g.exec) cudaGraphExecDestroy(g.exec);
    b->graphs.clear();
}

extern "C" const char *jdft_last_error(void) { return g_err; }
extern "C" int64_t jdft_launch_count(int reset) {
    int64_t v = g_launches;
    if (reset) g_launches = 0;
    return v;
}
extern "C" const char *jdft_version(void) { return "jdft-b200 0.1 (sm_100a)"; }

cudaError_t jdft_ensure_smem(const void *kernel, size_t bytes, int device) {
    static std::mutex mu;
    static std::map<std::pair<const void *, int>, size_t> done;
    std::lock_guard<std::mutex> lock(mu);
    size_t &have = done[std::make_pair(kernel, device)];
    if (have >= bytes && have > 0) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) have = bytes;
    return e;
}

JdftEncodeTiledFn jdft_tensor_map_encoder() {
    static JdftEncodeTiledFn fn = []() -> JdftEncodeTiledFn {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        return (JdftEncodeTiledFn)p;
    }();
    return fn;
}

static bool smooth235(int n) {
    if (n < 1) return false;
    for (int p : {2, 3, 5})
        while (n % p == 0) n /= p;
    return n == 1;
}

// Radix plan.  Specialised kernels exist for a few lengths (see fft.cuh: spec_plan); every other
// 2/3/5-smooth length runs on the runtime-radix kernels with radices 4, 2, 3, 5.
static FftPlan generic_plan(int L) {
    FftPlan p;
    memset(&p, 0, sizeof(p));
    p.L = L;
    int n = L;
    while (n % 4 == 0) { p.radix[p.npass++] = 4; n /= 4; }
    while (n % 2 == 0) { p.radix[p.npass++] = 2; n /= 2; }
    while (n % 3 == 0) { p.radix[p.npass++] = 3; n /= 3; }
    while (n % 5 == 0) { p.radix[p.npass++] = 5; n /= 5; }
    if (p.npass == 0) { p.radix[p.npass++] = 1; }
    return p;
}

static double det3(const double *A) {
    return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
           A[2] * (A[3] * A[7] - A[4] * A[6]);
}

static inline double ke_of(const double *GGT, const double *k, int m0, int m1, int m2) {
    const double x[3] = {m0 + k[0], m1 + k[1], m2 + k[2]};
    double s = 0.0;
    for (int a = 0; a < 3; a++)
        for (int c = 0; c < 3; c++) s += x[a] * GGT[3 * a + c] * x[c];
    return 0.5 * s;
}

static inline int wrap(int m, int S) {
    int r = m % S;
    return r < 0 ? r + S : r;
}

template <class T>
static cudaError_t upload(T **dst, const T *src, size_t n) {
    cudaError_t e = cudaMalloc((void **)dst, (n ? n : 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    if (n) e = cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice);
    return e;
}

extern "C" int jdft_basis_destroy(jdft_basis *b) {
    if (!b) return jdft_fail(JDFT_EINVAL, "basis_destroy: null basis");
    cudaSetDevice(b->device);
    cudaFree(b->d_index);
    cudaFree(b->d_iG);
    cudaFree(b->d_ke);
    cudaFree(b->d_col_n0);
    cudaFree(b->d_col_m2lo);
    cudaFree(b->d_rowcol);
    cudaFree(b->d_planeof);
    for (int d = 0; d < 3; d++) cudaFree(b->d_tw[d]);
    if (b->side) cudaStreamDestroy(b->side);
    if (b->ev_fork) cudaEventDestroy(b->ev_fork);
    if (b->ev_join) cudaEventDestroy(b->ev_join);
    for (int i = 0; i < 8; i++) cudaFree(b->hb[i]);
    for (int i = 0; i < 3; i++) if (b->hs[i]) cudaStreamDestroy(b->hs[i]);
    jdft_graphs_clear(b);
    if (b->gstream) cudaStreamDestroy(b->gstream);
    for (cudaEvent_t e : b->hev) cudaEventDestroy(e);
    for (cudaEvent_t e : b->prof_ev) cudaEventDestroy(e);
    delete b;
    return JDFT_OK;
}

extern "C" int jdft_basis_create(const double R[9], const double k[3], double Ecut, const int S[3], int device,
                                 jdft_basis **out) {
    if (!R || !k || !S || !out) return jdft_fail(JDFT_EINVAL, "basis_create: null argument");
    if (!(Ecut > 0.0)) return jdft_fail(JDFT_EINVAL, "basis_create: Ecut must be positive");
    for (int d = 0; d < 3; d++)
        if (!smooth235(S[d])) return jdft_fail(JDFT_EBOX, "basis_create: S[%d]=%d is not 2^a 3^b 5^c", d, S[d]);
    const double det = det3(R);
    if (det == 0.0 || !std::isfinite(det)) return jdft_fail(JDFT_EINVAL, "basis_create: singular lattice");
    if ((int64_t)S[0] * S[1] * S[2] >= (int64_t)1 << 31)
        return jdft_fail(JDFT_EBOX, "basis_create: box exceeds int32 indexing");

    jdft_basis *b = new (std::nothrow) jdft_basis();
    if (!b) return jdft_fail(JDFT_ENOMEM, "basis_create: out of host memory");
    memcpy(b->R, R, sizeof(b->R));
    memcpy(b->k, k, sizeof(b->k));
    memcpy(b->S, S, sizeof(b->S));
    b->Ecut = Ecut;
    b->device = device;
    b->volume = std::fabs(det);
    b->N = (int64_t)S[0] * S[1] * S[2];
    b->d_index = nullptr; b->d_iG = nullptr; b->d_ke = nullptr; b->d_col_n0 = nullptr; b->d_col_m2lo = nullptr;
    b->d_rowcol = nullptr; b->d_planeof = nullptr;
    for (int d = 0; d < 3; d++) b->d_tw[d] = nullptr;
    for (int i = 0; i < 8; i++) { b->hb[i] = nullptr; b->hb_bytes[i] = 0; }
    for (int i = 0; i < 3; i++) b->hs[i] = nullptr;
    b->opt_graph = -1; b->gstream = nullptr;
    b->h_ops_set = 0; b->h_nproj = 0; b->h_D_mode = 0; b->h_C_nb = 0;
    b->ws = nullptr; b->ws_bytes = 0; b->opt_band_batch = 0; b->opt_force_generic = 0;
    b->opt_profile_kernel = 0; b->prof_used = 0;
    b->opt_overlap = 0; b->opt_pair = 1; b->opt_prune = 1; b->opt_cols_direct = 1; b->opt_gemm3m = 1; b->opt_tma = 0; b->opt_gemm_tma = 0; b->opt_host_chunk = 0; b->side = nullptr; b->ev_fork = nullptr; b->ev_join = nullptr;

    // G = 2 pi R^-1 (adjugate / det): row i of G is the reciprocal vector b_i
    {
        const double adj[9] = {R[4] * R[8] - R[5] * R[7], R[2] * R[7] - R[1] * R[8], R[1] * R[5] - R[2] * R[4],
                               R[5] * R[6] - R[3] * R[8], R[0] * R[8] - R[2] * R[6], R[2] * R[3] - R[0] * R[5],
                               R[3] * R[7] - R[4] * R[6], R[1] * R[6] - R[0] * R[7], R[0] * R[4] - R[1] * R[3]};
        for (int i = 0; i < 9; i++) b->G[i] = 2.0 * M_PI * adj[i] / det;
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                double s = 0.0;
                for (int l = 0; l < 3; l++) s += b->G[3 * i + l] * b->G[3 * j + l];
                b->GGT[3 * i + j] = s;
            }
    }
    // integer bounding box of the ellipsoid: |m_d + k_d| <= sqrt(2 Ecut) |a_d| / (2 pi); one unit of slack
    int lo[3], hi[3];
    for (int d = 0; d < 3; d++) {
        const double len = std::sqrt(R[d] * R[d] + R[3 + d] * R[3 + d] + R[6 + d] * R[6 + d]);
        const double bound = std::sqrt(2.0 * Ecut) * len / (2.0 * M_PI);
        lo[d] = (int)std::floor(-k[d] - bound) - 1;
        hi[d] = (int)std::ceil(-k[d] + bound) + 1;
    }
    // sphere in lexicographic order (m0 slowest, m2 fastest), recording the plane / column structure:
    // all m0 between the first and last occupied plane are planes; within a plane all m1 between its first
    // and last occupied column are columns (possibly empty); within a column the m2 run is contiguous
    // because the cutoff region is convex.
    int mn[3] = {1 << 30, 1 << 30, 1 << 30}, mx[3] = {-(1 << 30), -(1 << 30), -(1 << 30)};
    struct Col { int m0, m1, m2lo, cnt; int64_t n0; };
    std::vector<Col> cols;
    try {
        for (int m0 = lo[0]; m0 <= hi[0]; m0++)
            for (int m1 = lo[1]; m1 <= hi[1]; m1++) {
                Col c = {m0, m1, 0, 0, (int64_t)b->ke.size()};
                int last = 0;
                for (int m2 = lo[2]; m2 <= hi[2]; m2++) {
                    const double e = ke_of(b->GGT, k, m0, m1, m2);
                    if (e < Ecut) {
                        if (c.cnt == 0) c.m2lo = m2;
                        else if (m2 != last + 1) { delete b; return jdft_fail(JDFT_EINVAL, "basis_create: non-contiguous column"); }
                        last = m2;
                        c.cnt++;
                        b->iG.push_back(m0); b->iG.push_back(m1); b->iG.push_back(m2);
                        b->ke.push_back(e);
                        const int m[3] = {m0, m1, m2};
                        for (int d = 0; d < 3; d++) { if (m[d] < mn[d]) mn[d] = m[d]; if (m[d] > mx[d]) mx[d] = m[d]; }
                    }
                }
                if (c.cnt) cols.push_back(c);
            }
    } catch (const std::bad_alloc &) { delete b; return jdft_fail(JDFT_ENOMEM, "basis_create: out of host memory"); }
    b->nG = (int64_t)b->ke.size();
    if (b->nG == 0) { delete b; return jdft_fail(JDFT_EINVAL, "basis_create: empty basis"); }
    for (int d = 0; d < 3; d++)
        if (mx[d] - mn[d] >= S[d]) {
            delete b;
            return jdft_fail(JDFT_EBOX, "basis_create: box axis %d too small (%d..%d does not fit %d)", d, mn[d], mx[d], S[d]);
        }
    b->index.resize(b->nG);
    for (int64_t n = 0; n < b->nG; n++)
        b->index[n] = (wrap(b->iG[3 * n], S[0]) * S[1] + wrap(b->iG[3 * n + 1], S[1])) * S[2] + wrap(b->iG[3 * n + 2], S[2]);

    for (int d = 0; d < 3; d++) { b->mmin[d] = mn[d]; b->mmax[d] = mx[d]; }
    // plane / column tables
    b->m0lo = mn[0];
    b->npl = mx[0] - mn[0] + 1;
    std::vector<int> pl_lo(b->npl, 1 << 30), pl_hi(b->npl, -(1 << 30));
    for (const Col &c : cols) {
        const int p = c.m0 - b->m0lo;
        if (c.m1 < pl_lo[p]) pl_lo[p] = c.m1;
        if (c.m1 > pl_hi[p]) pl_hi[p] = c.m1;
    }
    b->pl_m1lo.resize(b->npl);
    b->pl_cbase.resize(b->npl + 1);
    b->ncol = 0; b->maxcol_per_plane = 0;
    for (int p = 0; p < b->npl; p++) {
        const int cnt = pl_hi[p] >= pl_lo[p] ? pl_hi[p] - pl_lo[p] + 1 : 0;
        b->pl_m1lo[p] = cnt ? pl_lo[p] : 0;
        b->pl_cbase[p] = b->ncol;
        b->ncol += cnt;
        if (cnt > b->maxcol_per_plane) b->maxcol_per_plane = cnt;
    }
    b->pl_cbase[b->npl] = b->ncol;
    b->col_n0.assign(b->ncol + 1, 0);
    b->col_m2lo.assign(b->ncol, 0);
    std::vector<int> col_cnt(b->ncol, 0);
    for (const Col &c : cols) {
        const int p = c.m0 - b->m0lo;
        const int ci = b->pl_cbase[p] + (c.m1 - b->pl_m1lo[p]);
        col_cnt[ci] = c.cnt;
        b->col_m2lo[ci] = c.m2lo;
    }
    for (int c = 0; c < b->ncol; c++) b->col_n0[c + 1] = b->col_n0[c] + col_cnt[c];
    std::vector<int> rowcol((size_t)b->npl * S[1], -1), planeof(S[0], -1);
    for (int p = 0; p < b->npl; p++) {
        planeof[wrap(b->m0lo + p, S[0])] = p;
        for (int c = b->pl_cbase[p]; c < b->pl_cbase[p + 1]; c++)
            rowcol[(size_t)p * S[1] + wrap(b->pl_m1lo[p] + (c - b->pl_cbase[p]), S[1])] = c;
    }

    // twiddles exp(+2 pi i t / S_d) in long double with the argument reduced to the first octant
    std::vector<double2> tw[3];
    for (int d = 0; d < 3; d++) {
        const int n = S[d];
        tw[d].resize(n);
        const long double pi = 3.141592653589793238462643383279502884L;
        for (int t = 0; t < n; t++) {
            // angle = (pi/4) * (8 t / n) = (pi/4) * (oct + frac)
            const int64_t num = 8LL * t;
            const int oct = (int)(num / n);
            const int64_t rem = num % n;
            const long double phi = (oct & 1) ? (pi * (long double)(n - rem)) / (4.0L * n) : (pi * (long double)rem) / (4.0L * n);
            const long double c = cosl(phi), s = sinl(phi);
            long double cr, si;
            switch (oct) {
                case 0: cr = c; si = s; break;
                case 1: cr = s; si = c; break;
                case 2: cr = -s; si = c; break;
                case 3: cr = -c; si = s; break;
                case 4: cr = -c; si = -s; break;
                case 5: cr = -s; si = -c; break;
                case 6: cr = s; si = -c; break;
                default: cr = c; si = -s; break;
            }
            tw[d][t] = make_double2((double)cr, (double)si);
        }
        b->plan[d] = generic_plan(n);
    }

    // upload
    cudaError_t e = cudaSetDevice(device);
    b->num_sms = 148;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&b->num_sms, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = upload(&b->d_index, b->index.data(), b->index.size());
    if (e == cudaSuccess) e = upload(&b->d_iG, b->iG.data(), b->iG.size());
    if (e == cudaSuccess) e = upload(&b->d_ke, b->ke.data(), b->ke.size());
    if (e == cudaSuccess) e = upload(&b->d_col_n0, b->col_n0.data(), b->col_n0.size());
    if (e == cudaSuccess) e = upload(&b->d_col_m2lo, b->col_m2lo.data(), b->col_m2lo.size());
    if (e == cudaSuccess) e = upload(&b->d_rowcol, rowcol.data(), rowcol.size());
    if (e == cudaSuccess) e = upload(&b->d_planeof, planeof.data(), planeof.size());
    for (int d = 0; d < 3 && e == cudaSuccess; d++) e = upload(&b->d_tw[d], tw[d].data(), tw[d].size());
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&b->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&b->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&b->ev_join, cudaEventDisableTiming);
    if (e != cudaSuccess) {
        jdft_basis_destroy(b);
        return jdft_cuda_fail(e, "basis_create upload");
    }
    *out = b;
    return JDFT_OK;
}

extern "C" int jdft_basis_info(const jdft_basis *b, int64_t *nG, int64_t *N, double *volume) {
    if (!b) return jdft_fail(JDFT_EINVAL, "basis_info: null basis");
    if (nG) *nG = b->nG;
    if (N) *N = b->N;
    if (volume) *volume = b->volume;
    return JDFT_OK;
}

extern "C" int jdft_basis_structure(const jdft_basis *b, int64_t *npl, int64_t *ncol) {
    if (!b) return jdft_fail(JDFT_EINVAL, "basis_structure: null basis");
    if (npl) *npl = b->npl;
    if (ncol) *ncol = b->ncol;
    return JDFT_OK;
}

extern "C" int jdft_basis_export(const jdft_basis *b, int32_t *iG, int32_t *index, double *ke) {
    if (!b) return jdft_fail(JDFT_EINVAL, "basis_export: null basis");
    if (iG) memcpy(iG, b->iG.data(), sizeof(int32_t) * 3 * b->nG);
    if (index) memcpy(index, b->index.data(), sizeof(int32_t) * b->nG);
    if (ke) memcpy(ke, b->ke.data(), sizeof(double) * b->nG);
    return JDFT_OK;
}

extern "C" int jdft_basis_device_maps(const jdft_basis *b, const int32_t **index_dev, const double **ke_dev) {
    if (!b) return jdft_fail(JDFT_EINVAL, "basis_device_maps: null basis");
    if (index_dev) *index_dev = b->d_index;
    if (ke_dev) *ke_dev = b->d_ke;
    return JDFT_OK;
}

// ---- workspace ------------------------------------------------------------------------------------

size_t jdft_fft_bytes_per_band(const jdft_basis *b) {
    // W1: compact columns [ncol][S2]; W2: occupied planes [npl][S1][S2]; both c128
    return 16 * ((size_t)b->ncol * b->S[2] + (size_t)b->npl * b->S[1] * b->S[2]);
}

static size_t gemm_bytes(int nrows_max) {
    // projected coefficients B and D.B ([nb][np] each, bounded by nrows_max^2) + split-K partials (capped)
    const size_t r = (size_t)(nrows_max > 0 ? nrows_max : 0);
    return 2 * 16 * r * r + ((size_t)64 << 20);
}

extern "C" size_t jdft_workspace_bytes(const jdft_basis *b, int nbands_batch, int nrows_max) {
    if (!b) return 0;
    const size_t f = jdft_fft_bytes_per_band(b) * (size_t)(nbands_batch > 0 ? nbands_batch : 1);
    const size_t g = gemm_bytes(nrows_max);
    return f + g + 512;  // both at once: the projection GEMM overlaps the FFT pipeline in apply_H
}

extern "C" int jdft_set_workspace(jdft_basis *b, void *dev_ptr, size_t bytes) {
    if (!b) return jdft_fail(JDFT_EINVAL, "set_workspace: null basis");
    if (((uintptr_t)dev_ptr & 15) != 0) return jdft_fail(JDFT_EINVAL, "set_workspace: pointer not 16-byte aligned");
    b->ws = dev_ptr;
    b->ws_bytes = dev_ptr ? bytes : 0;
    jdft_graphs_clear(b);
    return JDFT_OK;
}

extern "C" int jdft_set_option(jdft_basis *b, const char *key, int64_t value) {
    if (!b || !key) return jdft_fail(JDFT_EINVAL, "set_option: null argument");
    jdft_graphs_clear(b);   // captured calls bake the options in
    if (!strcmp(key, "graph")) { b->opt_graph = value < 0 ? -1 : (value != 0); return JDFT_OK; }
    if (!strcmp(key, "band_batch")) { b->opt_band_batch = value < 0 ? 0 : value; return JDFT_OK; }
    if (!strcmp(key, "planes_pair")) { b->opt_pair = value != 0; return JDFT_OK; }
    if (!strcmp(key, "planes_prune")) { b->opt_prune = value != 0; return JDFT_OK; }
    if (!strcmp(key, "cols_direct")) { b->opt_cols_direct = value != 0; return JDFT_OK; }
    if (!strcmp(key, "host_chunk")) { b->opt_host_chunk = value < 0 ? 0 : value; return JDFT_OK; }
    if (!strcmp(key, "gemm_tma")) { b->opt_gemm_tma = value != 0; return JDFT_OK; }
    if (!strcmp(key, "planes_tma")) { b->opt_tma = value != 0; return JDFT_OK; }
    if (!strcmp(key, "gemm_3m")) { b->opt_gemm3m = value < 0 ? 0 : value; return JDFT_OK; }
    if (!strcmp(key, "overlap_gemm")) { b->opt_overlap = value != 0; return JDFT_OK; }
    if (!strcmp(key, "force_generic_fft")) { b->opt_force_generic = value != 0; return JDFT_OK; }
    if (!strcmp(key, "profile_kernel")) { b->opt_profile_kernel = value; b->prof_used = 0; return JDFT_OK; }
    return jdft_fail(JDFT_EINVAL, "set_option: unknown key '%s'", key);
}

int jdft_band_batch(const jdft_basis *b, int nb, size_t ws_offset) {
    const size_t per = jdft_fft_bytes_per_band(b);
    if (!b->ws || b->ws_bytes < ws_offset + per) return 0;
    size_t fit = (b->ws_bytes - ws_offset) / per;
    int64_t want = b->opt_band_batch;
    if (want <= 0) {
        // automatic: as many bands as the workspace holds, up to 256.  Measured on B200 (band-batch sweep):
        // filling the GPU (thousands of CTAs per launch, few tail waves) beats keeping a small batch L2-resident.
        want = 256;
    }
    if ((size_t)want > fit) want = (int64_t)fit;
    if (want > nb) want = nb;
    if (want < 1) want = 1;
    return (int)want;
}

// ---- optional per-kernel event timing (diagnostics; not thread-safe; off by default) ------------------

void jdft_prof_begin(const jdft_basis *cb, int kid, cudaStream_t st) {
    if (cb->opt_profile_kernel != kid) return;
    jdft_basis *b = const_cast<jdft_basis *>(cb);
    if (b->prof_used + 2 > b->prof_ev.size()) {
        if (b->prof_ev.size() >= 1 << 16) return;
        for (int i = 0; i < 2; i++) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return;
            b->prof_ev.push_back(e);
        }
    }
    cudaEventRecord(b->prof_ev[b->prof_used], st);
}

void jdft_prof_end(const jdft_basis *cb, int kid, cudaStream_t st) {
    if (cb->opt_profile_kernel != kid) return;
    jdft_basis *b = const_cast<jdft_basis *>(cb);
    if (b->prof_used + 2 > b->prof_ev.size()) return;
    cudaEventRecord(b->prof_ev[b->prof_used + 1], st);
    b->prof_used += 2;
}

extern "C" int jdft_profile_read(jdft_basis *b, int64_t *launches, double *total_ms) {
    if (!b) return jdft_fail(JDFT_EINVAL, "profile_read: null basis");
    double ms = 0.0;
    for (size_t i = 0; i + 1 < b->prof_used; i += 2) {
        JDFT_CUDA(cudaEventSynchronize(b->prof_ev[i + 1]));
        float t = 0.f;
        JDFT_CUDA(cudaEventElapsedTime(&t, b->prof_ev[i], b->prof_ev[i + 1]));
        ms += t;
    }
    if (launches) *launches = (int64_t)(b->prof_used / 2);
    if (total_ms) *total_ms = ms;
    b->prof_used = 0;
    return JDFT_OK;
}
