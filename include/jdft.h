/*
 * jdft.h -- C ABI of libjdft_b200: the data-parallel hot path of plane-wave DFT in the DFT++
 * operator language used by JDFTx (arXiv 1708.03621), hand-written for NVIDIA B200 (sm_100a).
 *
 *     H C = -1/2 L C + I^+ Diag(V_loc) I C + P D P^+ C        (BASELINE.json north_star)
 *
 * What the paper fixes.  PAPER.md:76 (section 2.1): "the operators I and J Fourier transform from
 * reciprocal to real space and vice versa (using Fast Fourier Transforms)"; gradient/divergence "apply in
 * reciprocal space (where they are diagonal)"; integrals are "a dot product with the overlap operator O",
 * which is "diagonal in the plane-wave basis".  PAPER.md:86: wavefunctions live in a ColumnBundle, the
 * grid and its Fourier transforms in GridInfo.  PAPER.md:127: SpeciesInfo holds the pseudopotentials
 * (the nonlocal projectors P and couplings D here).  PAPER.md:59 delegates every formula to the DFT++
 * paper (its Ref. [11]); the concrete conventions below are the readings listed in DESIGN.md section 3.
 *
 * Conventions.
 *   complex128  = double[2], (re, im) interleaved.
 *   R           = 3x3 row-major, COLUMNS are the lattice vectors (bohr).  Omega = |det R|.
 *   G           = 2 pi R^-1 (rows are reciprocal vectors); ke(m) = 1/2 (m+k)^T G G^T (m+k), k reduced.
 *   basis       = { m in Z^3 : ke(m) < Ecut } in ascending signed lexicographic order of (m0, m1, m2),
 *                 m2 fastest;  index[n] = ((m0 mod S0) S1 + (m1 mod S1)) S2 + (m2 mod S2).
 *   C           = [nb][nG] band-major, G-sphere index contiguous.
 *   psi         = [nb][S0][S1][S2] real-space block, axis 2 contiguous.
 *   I           (I C)[j]   = sum_n C[n] exp(+2 pi i sum_d iG[n]_d j_d / S_d)      (unnormalised)
 *   Idag        (I^+ f)[n] = sum_j exp(-2 pi i sum_d iG[n]_d j_d / S_d) f[j]
 *   J           = I^+ / N,   N = S0 S1 S2          (J I = 1 on the sphere)
 *   O C         = Omega C;   L C = -Omega |G+k|^2 C = -2 Omega ke C
 *   Vnl         = P D P^+ with P = [np][nG] (projector-major) and D given as data
 *
 * Pointers.  Unless marked HOST, every data pointer is a DEVICE pointer on the basis' device, owned by
 * the caller (e.g. a torch tensor's data_ptr()), 16-byte aligned (32-byte aligned arrays and workspace, as any
 * allocator gives, let the library pick its 256-bit load/store kernels; results are the same either way).  The library owns only the basis
 * object.  The hot path allocates nothing and never synchronises with the host: all scratch comes from
 * the caller-supplied workspace, and kernels are enqueued on the caller's stream.  Input and output
 * arrays must not alias unless stated.
 *
 * Errors.  Every call returns JDFT_OK (0) or a negative code; nothing throws, aborts or prints.
 * jdft_last_error() returns a thread-local message for the last failure.  Launches are asynchronous:
 * launch-time CUDA errors are returned, execution-time errors surface at the caller's next sync.
 *
 * The jdft_*_host entry points are the same operations taking HOST arrays: they allocate device
 * buffers, copy in, run the same kernels, copy out and synchronise (used for the end-to-end number);
 * jdft_apply_H_host pipelines band chunks over three streams (H2D of chunk i+1, kernels of chunk i, D2H of
 * chunk i-1 at once; pinned host arrays make the copies asynchronous).
 *
 * Concurrency.  A basis owns its workspace binding, its side streams and its events, so ONE stream (or host
 * thread) at a time may run calls on a given basis.  Callers that want concurrent streams create one basis per
 * stream (creation is cheap: an O(sphere) enumeration and a few small uploads).
 */
#ifndef JDFT_H
#define JDFT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define JDFT_OK 0
#define JDFT_EINVAL (-1)     /* null pointer, negative size, bad mode, singular R                      */
#define JDFT_EBOX (-2)       /* S[d] not 2^a 3^b 5^c, or box too small: two sphere points would collide */
#define JDFT_EWORKSPACE (-3) /* no workspace set, or too small for one band                             */
#define JDFT_ECUDA (-4)      /* a CUDA runtime call failed (see jdft_last_error)                        */
#define JDFT_ENOMEM (-5)     /* host or device allocation failed (basis creation / *_host calls only)   */

typedef struct jdft_basis jdft_basis; /* opaque; owned by the library */
typedef void *jdft_stream;            /* a cudaStream_t; NULL = the legacy default stream */

/* ---- basis (readings 6-12) --------------------------------------
 * Builds the G-sphere of the wavefunction cutoff inside FFT box S, uploads the index map, ke = 1/2|G+k|^2,
 * the per-axis twiddle tables and the column/plane structure used to prune the FFT passes.
 * R, k, S are HOST arrays.  Fails with JDFT_EBOX when max(m_d) - min(m_d) >= S[d] for some axis.      */
int jdft_basis_create(const double R[9], const double k[3], double Ecut, const int S[3], int device,
                      jdft_basis **out);
int jdft_basis_destroy(jdft_basis *b);
/* sizes: nG plane waves, N = S0 S1 S2 grid points, cell volume Omega (any pointer may be NULL)        */
int jdft_basis_info(const jdft_basis *b, int64_t *nG, int64_t *N, double *volume);
/* pruning structure: occupied i0 planes and (i0,i1) columns (npl, ncol)               */
int jdft_basis_structure(const jdft_basis *b, int64_t *npl, int64_t *ncol);
/* HOST copies for bit-exact checks: iG int32[nG][3], index int32[nG], ke f64[nG] (any may be NULL)    */
int jdft_basis_export(const jdft_basis *b, int32_t *iG_host, int32_t *index_host, double *ke_host);
/* device pointers to the resident index map / ke (valid until destroy)                                 */
int jdft_basis_device_maps(const jdft_basis *b, const int32_t **index_dev, const double **ke_dev);

/* ---- workspace -------------------------------------------------------------------------------------
 * Bytes needed to process `nbands_batch` bands at once (FFT intermediates) plus the projector / overlap GEMM
 * scratch for up to `nrows_max` rows (max of nproj, nb).
 * Calls with more bands than fit are split into band batches internally (results are identical).      */
size_t jdft_workspace_bytes(const jdft_basis *b, int nbands_batch, int nrows_max);
int jdft_set_workspace(jdft_basis *b, void *dev_ptr, size_t bytes);
/* tunables: "band_batch" (bands per FFT batch, 0 = automatic: what the workspace holds, at most 256),
 * "force_generic_fft" (0/1: use the runtime-radix FFT kernels even for lengths that have specialised ones; for
 * tests), "overlap_gemm" (0/1, default 0: apply_H forks B = D P^+ C onto a basis-owned side stream beside the FFT
 * pipeline and joins before HC += P B; uses basis-owned events, so not for concurrent calls on one basis),
 * "planes_pair" (0/1, default 1: K3 with two pencils per thread where that variant exists),
 * "planes_prune" (0/1, default 1: K3 hybrid with radix-8 butterflies pruned to the sphere's extent along axis 0
 * when planes [L/4, 3L/4) are empty),
 * "cols_direct" (0/1, default 1: K1's first pass reads the sphere and, at column length 128, K5's last pass writes it
 * straight from / to global memory instead of staging the scatter / gather through shared memory; same arithmetic, bit-identical),
 * "planes_tma" (0/1, default 0: K3 through tensor-map (TMA) loads / stores in persistent double-buffered CTAs; measured
 * slower than the LSU kernels on B200), "gemm_3m" (0/1, default 1: projector / overlap GEMMs by the
 * 3M complex-product scheme, three tensor instructions per complex tile product instead of four),
 * "gemm_tma" (0/1, default 0: operand stages of the 3M GEMMs filled by cp.async.bulk.tensor instead of cp.async; measured
 * 5 % slower),
 * "host_chunk" (bands per chunk of the jdft_apply_H_host pipeline; 0 = default 64),
 * "graph" (-1 auto / 0 off / 1 on: jdft_apply_H replays a captured CUDA graph when called again with the same pointers,
 * sizes and workspace; auto = calls of at most 4 Mi band x grid points, which are launch-bound),
 * "profile_kernel" (see diagnostics)                                                                    */
int jdft_set_option(jdft_basis *b, const char *key, int64_t value);

/* ---- operators ------------------------------------------------------ */
/* I ("the operators I and J Fourier transform from reciprocal to real space and vice versa (using Fast
 * Fourier Transforms)"; rows a1 + a2; readings 2, 3, 8, 9): C [nb][nG] -> psi [nb][N], sphere -> box
 * scatter + inverse 3-D FFT, unnormalised, sign +.                                                       */
int jdft_apply_I(const jdft_basis *b, const double *C, int nb, double *psi, jdft_stream s);
/* Idag (the adjoint of I that H C needs, BASELINE.json north_star; row a4 + the gather of a5): psi [nb][N] ->
 * C [nb][nG], forward 3-D FFT (sign -) + box -> sphere gather.  psi may hold components outside the sphere.  */
int jdft_apply_Idag(const jdft_basis *b, const double *psi, int nb, double *C, jdft_stream s);
/* J (the inverse transform of I; reading 2): J = Idag / N, so J I = 1 on the sphere.     */
int jdft_apply_J(const jdft_basis *b, const double *psi, int nb, double *C, jdft_stream s);
/* L (gradient / divergence "apply in reciprocal space (where they are diagonal)", L = div grad;
 * DESIGN.md readings 4, 6): L C = -Omega |G+k|^2 C = -2 Omega ke C.  May run in place (LC == C).               */
int jdft_apply_L(const jdft_basis *b, const double *C, int nb, double *LC, jdft_stream s);
/* O ("the integral is evaluated as a dot product with the overlap operator O", "diagonal in the
 * plane-wave basis"; reading 4): O C = Omega C.  May run in place.                                  */
int jdft_apply_O(const jdft_basis *b, const double *C, int nb, double *OC, jdft_stream s);
/* Vnl: out (+)= P D P^+ C (PAPER.md:127 SpeciesInfo pseudopotentials).  P c128[nproj][nG];
 * D_mode 0: D = f64[nproj] real diagonal;  D_mode 1: D = c128[nproj][nproj] row-major Hermitian;
 * D_mode = nblk >= 2: per-atom Hermitian blocks D = c128[nproj / nblk][nblk][nblk] (block a couples projectors
 * a nblk .. a nblk + nblk - 1 only -- the ultrasoft case of PAPER.md:95; nproj % nblk must be 0; reading 24).
 * The same three layouts are accepted wherever a D or Q is taken.  accumulate != 0 adds into out.              */
int jdft_apply_Vnl(const jdft_basis *b, const double *P, int nproj, const double *D, int D_mode,
                   const double *C, int nb, double *out, int accumulate, jdft_stream s);
/* projection alone (row a6): Bproj [nb][nproj] = (P^+ C)^T, i.e. Bproj[ib][j] = sum_n conj(P[j][n]) C[ib][n]    */
int jdft_project(const jdft_basis *b, const double *P, int nproj, const double *C, int nb, double *Bproj,
                 jdft_stream s);
/* H (BASELINE.json north_star; rows a1-a8 as one fused pipeline, the real-space psi never reaches HBM):
 * HC = -1/2 L C + I^+ (Vloc .* I C) + P D P^+ C.  Vloc f64[N] is used exactly as passed (the caller
 * folds in the quadrature weight Omega/N; reading 5).  nproj == 0 skips the nonlocal term.  */
int jdft_apply_H(const jdft_basis *b, const double *Vloc, const double *P, int nproj, const double *D,
                 int D_mode, const double *C, int nb, double *HC, jdft_stream s);
/* overlap (row a9; PAPER.md:76 integrals as dot(a, O b)): M[a + nb1*bb] = Omega sum_n conj(C1[a][n]) C2[bb][n]
 * (column-major nb1 x nb2, c128).  C1 == C2 (same pointer) computes the Hermitian triangle only and mirrors it.  */
int jdft_overlap(const jdft_basis *b, const double *C1, int nb1, const double *C2, int nb2, double *M,
                 jdft_stream s);

/* overlap without any allocation or workspace (same result as jdft_overlap): for callers that cannot call cudaMalloc or
 * hand over a workspace -- code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  The
 * split-K partials of the GEMM live in a 16 MiB file-scope static device array inside the library (held by every GPU that
 * loads the library until the process exits), so the call allocates nothing and ignores the basis' workspace.
 * LIMIT: nb1 * nb2 <= 65 536 entries (e.g. 256 x 256); larger sizes return JDFT_EINVAL with a message.  All calls on a
 * device share the array (it keeps the last call's contents; nothing needs clearing): calls that overlap on the GPU
 * (different streams) race -- use one stream at a time per device.  The first call per device resolves the array's
 * address and should be made outside graph capture.                                                                   */
int jdft_overlap_noalloc(const jdft_basis *b, const double *C1, int nb1, const double *C2, int nb2, double *M,
                         jdft_stream s);

/* ---- ultrasoft pseudopotentials ("norm-conserving and ultrasoft pseudopotentials",
 * PAPER.md:166-169 Listing 2 runs on the GBRV ultrasoft library; reading 24) ------------------------------
 * generalised overlap operator   O_us C = Omega (C + P Q P^+ C),   Q in the layouts of D (Q_mode as D_mode);
 * OC may alias C.  nproj == 0 gives O C = Omega C.                                                              */
int jdft_apply_O_us(const jdft_basis *b, const double *P, int nproj, const double *Q, int Q_mode, const double *C,
                    int nb, double *OC, jdft_stream s);
/* generalised overlap matrix     M[a + nb1*bb] = C1[a]^+ O_us C2[bb]   (column-major nb1 x nb2, c128)          */
int jdft_overlap_us(const jdft_basis *b, const double *P, int nproj, const double *Q, int Q_mode, const double *C1,
                    int nb1, const double *C2, int nb2, double *M, jdft_stream s);

/* ---- the steps next to H C in an SCF / minimiser iteration (PAPER.md:127 ElecVars:
 * wavefunctions -> density -> potential; PAPER.md:76 integrals as dot products) ------------------------------ */
/* subspace matrix: M[a + nb1*bb] = sum_n conj(C1[a][n]) X2[bb][n]  (column-major nb1 x nb2, c128; NO Omega --
 * with X2 = H C1 this is the subspace Hamiltonian C^+ H C)                                                   */
int jdft_subspace(const jdft_basis *b, const double *C1, int nb1, const double *X2, int nb2, double *M,
                  jdft_stream s);
/* density: n[j] (+)= sum_b f[b] |(I C_b)[j]|^2.  f = f64[nb] occupations (DEVICE), n = f64[N] (DEVICE), bands are
 * summed in index order (deterministic); accumulate != 0 adds to the existing n.  psi never reaches HBM.      */
int jdft_density(const jdft_basis *b, const double *C, int nb, const double *f, double *n, int accumulate,
                 jdft_stream s);

/* ---- scalar-field operators of the paper's Listing 1 --------
 * gradient:   out[d][b][n] = i q_d(n) C[b][n],  q = G^T (iG[n] + k) Cartesian, d = 0,1,2;  out is [3][nb][nG]
 * divergence: out[b][n]    = sum_d i q_d(n) X[d][b][n];                                     X   is [3][nb][nG]
 * pcm_hessian (Listing 1): out = (-1/(4 pi)) divergence(J(epsilon .* I(gradient(phi)))), epsilon f64[N] real,
 *   phi/out [nb][nG]; one fused pass: the epsilon multiply rides inside the FFT pipeline, nothing of size N per
 *   field reaches HBM.  Needs workspace for 3 nb nG c128 plus FFT scratch (jdft_workspace_bytes(b, 3 nb, 0) +
 *   48 nb nG is enough).                                                                                     */
int jdft_gradient(const jdft_basis *b, const double *C, int nb, double *out, jdft_stream s);
int jdft_divergence(const jdft_basis *b, const double *X, int nb, double *out, jdft_stream s);
int jdft_pcm_hessian(const jdft_basis *b, const double *epsilon, const double *phi, int nb, double *out,
                     jdft_stream s);
/* The same operator on REAL fields (epsilon, phi, rho are real ScalarFields, so phi~(-G) = conj(phi~(G)))
 * in half-sphere storage (reading 25).  Gamma-point bases only (k = 0, else JDFT_EINVAL): there the canonical
 * order is inversion symmetric, iG[nG-1-n] = -iG[n], the origin is n0 = (nG-1)/2 and the stored half is the tail:
 *     phi_h[ib][h] = phi~[n0 + h],  h = 0 .. nGh-1,  nGh = (nG+1)/2;   phi~[n0 - h] = conj(phi_h[ib][h]);  Im phi~[n0] ignored.
 * out_h has the same layout.  Two real gradient components share one complex transform (two-for-one), so the call moves
 * and computes half of what jdft_pcm_hessian does.  Workspace: ceil(3 nb / 2) nG c128 plus FFT scratch.               */
int jdft_pcm_hessian_real(const jdft_basis *b, const double *epsilon, const double *phi_h, int nb, double *out_h,
                          jdft_stream s);

/* ---- HOST-buffer variants (end-to-end path: H2D copy, kernels, D2H copy, sync) -------------------- */
int jdft_apply_H_host(jdft_basis *b, const double *Vloc_host, const double *P_host, int nproj,
                      const double *D_host, int D_mode, const double *C_host, int nb, double *HC_host);
int jdft_overlap_host(jdft_basis *b, const double *C1_host, int nb1, const double *C2_host, int nb2,
                      double *M_host);
/* Resident operators: V_loc, P, D stay the same over the many H applications of an SCF iteration, so
 * they are uploaded once into library-owned device buffers; jdft_apply_H_host_resident then moves only the bands in
 * and H C out (chunk-pipelined on three streams like jdft_apply_H_host).  A later jdft_apply_H_host call replaces them. */
int jdft_host_set_operators(jdft_basis *b, const double *Vloc_host, const double *P_host, int nproj,
                            const double *D_host, int D_mode);
int jdft_apply_H_host_resident(jdft_basis *b, const double *C_host, int nb, double *HC_host);
/* M = C^+ O C (column-major nb x nb, HOST) of the band block the last jdft_apply_H_host / _resident call uploaded: H C and
 * the overlap of the same bands are needed together in every SCF step, so C is not uploaded a second time.  JDFT_EINVAL
 * if no such block of nb bands is on the device (any other *_host call in between invalidates it).                  */
int jdft_overlap_host_resident(jdft_basis *b, int nb, double *M_host);

/* ---- diagnostics ---------------------------------------------------------------------------------- */
const char *jdft_last_error(void);
/* kernels launched by this thread since the last call with reset != 0 (bench.py's gpu_launches)       */
int64_t jdft_launch_count(int reset);
/* Diagnostics, off by default: jdft_set_option(b, "profile_kernel", id) brackets every later launch of ONE
 * kernel (1 cols_inv, 2 rows_inv, 3 planes, 4 rows_fwd, 5 cols_fwd, 6 gemm_dotk, 7 gemm_expand, 8 split-K
 * reduce, 9 diag; 0 = off) with CUDA events on the launch stream; jdft_profile_read waits for them, returns
 * the number of launches and their summed device time, and resets.  Not thread-safe.                   */
int jdft_profile_read(jdft_basis *b, int64_t *launches, double *total_ms);
const char *jdft_version(void);

#ifdef __cplusplus
}
#endif
#endif /* JDFT_H */
