/*
 * oracle/jdft_ref.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU implementation (fp64 data, long-double
 * twiddles and GEMM accumulators) of the plane-wave DFT++ operators whose CUDA
 * implementation lives in paper_1708_03621_b200/csrc/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, link, import or call anything in this directory.  It shares no
 * code, header, table or constant generator with the CUDA path.
 *
 * What it follows.  The paper (section 2.1) says only that "the
 * operators I and J Fourier transform from reciprocal to real space and vice
 * versa (using Fast Fourier Transforms)", that gradient/divergence "apply in
 * reciprocal space (where they are diagonal)", that "the integral is evaluated
 * as a dot product with the overlap operator O" and that O is "diagonal in the
 * plane-wave basis".  It delegates every formula to its Ref. [11] (DFT++,
 * PAPER.md:59, 329).  The concrete definitions implemented here are therefore
 * the readings fixed in DESIGN.md section 3 (= SURVEY.md section 8(c)):
 *
 *   geometry   R = 3x3, COLUMNS are lattice vectors; Omega = |det R|;
 *              G = 2 pi R^-1 (row i = reciprocal vector b_i); GGT = G G^T;
 *              ke(m) = 1/2 (m+k)^T GGT (m+k)                     [reading 6,10,11]
 *   basis      { m in Z^3 : ke(m) < Ecut }, ascending signed lexicographic
 *              (m0, m1, m2), m2 fastest; index = ((m0 mod S0) S1 + (m1 mod S1)) S2
 *              + (m2 mod S2)                                      [reading 7,8,9]
 *   I          (I C)[j]  = sum_n C[n] exp(+2 pi i sum_d iG[n]_d j_d / S_d)   [2,3]
 *   Idag       (I^+ f)[n] = sum_j exp(-2 pi i sum_d iG[n]_d j_d / S_d) f[j]
 *   J          J = I^+ / N
 *   O          O C = Omega C                                      [reading 4]
 *   L          (L C)[n] = -Omega |G+k|^2 C[n] = -2 Omega ke[n] C[n]
 *   Vnl        P D P^+ C, with P (nG x np) and D given as data    [reading 13,14]
 *   H          H C = -1/2 L C + I^+( Vloc .* (I C) ) + P D P^+ C  (BASELINE.json north_star)
 *   overlap    M = C1^+ O C2 = Omega C1^+ C2, column-major nb1 x nb2
 *
 * Algorithm (deliberately naive): the basis by a plain sweep of 2 S_d + 1 integers per axis (no ellipsoid
 * geometry) plus a literal collision check; a zero-filled full box per band; three
 * un-pruned passes of a recursive mixed-radix decimation-in-time 1-D FFT (any
 * prime factor; O(p) butterflies written as the plain DFT sum), pencils copied
 * to a contiguous buffer; separate V multiply, gather, kinetic passes; GEMMs
 * as triple loops with long double accumulators.  OpenMP over bands only.
 *
 * PINS (tests/test_oracle_pins.py, all "-m not gpu"): 1-D FFT vs O(n^2) DFT;
 * 3-D I/Idag vs the explicit N x nG matrix on small, non-cubic, k != 0 boxes;
 * J I = 1; I J idempotent; Parseval; adjointness; cos-potential closed form
 * (sign + wrap); translation covariance; L/ke closed forms; Omega values;
 * plane-wave eigenvalue ke + V0; Hermiticity; Vnl vs dense P D P^+, rank-1,
 * D = 0; basis vs exact counts, inversion symmetry, continuum count; block-diagonal D and the ultrasoft
 * O_us / overlap_us vs dense nG x nG matrices, positivity, Q = 0; density / subspace vs explicit matrices;
 * gradient / divergence / Listing-1 hessian vs finite differences and explicit matrices; the real-field
 * (half-sphere) hessian vs the complex path, realness of I, inversion symmetry of the order.
 * No function of this file is "parity unpinned".
 * Unpinned by the paper: the CHOICE of conventions (readings 2-11); see DESIGN.md.
 *
 * Layouts: complex128 = double[2] (re, im) interleaved.  C is [nb][nG]
 * (band-major, G contiguous); real-space block is [nb][S0][S1][S2], axis 2
 * fastest; P is [np][nG]; D is f64[np] (D_mode 0) or c128[np][np] row-major
 * Hermitian (D_mode 1); Bproj = P^+ C is [nb][np].
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex cplx;
typedef long double _Complex lcplx;

typedef struct jdft_ref_basis {
    double R[9], k[3], Ecut;
    int S[3];
    double G[9], GGT[9], volume;
    int64_t nG, N;
    int32_t *iG;    /* [nG][3] */
    int32_t *index; /* [nG]    */
    double *ke;     /* [nG]    */
} jdft_ref_basis;

#define REF_OK 0
#define REF_EINVAL (-1)
#define REF_EBOX (-2)
#define REF_ENOMEM (-5)

/* ------------------------------------------------------------------ geometry */

static double det3(const double *A) {
    return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
           A[2] * (A[3] * A[7] - A[4] * A[6]);
}

/* G = 2 pi R^-1 by the adjugate formula */
static void recip(const double *R, double *G) {
    double d = det3(R);
    double adj[9] = {
        R[4] * R[8] - R[5] * R[7], R[2] * R[7] - R[1] * R[8], R[1] * R[5] - R[2] * R[4],
        R[5] * R[6] - R[3] * R[8], R[0] * R[8] - R[2] * R[6], R[2] * R[3] - R[0] * R[5],
        R[3] * R[7] - R[4] * R[6], R[1] * R[6] - R[0] * R[7], R[0] * R[4] - R[1] * R[3]};
    for (int i = 0; i < 9; i++) G[i] = 2.0 * M_PI * adj[i] / d;
}

/* ke(m) = 1/2 (m+k)^T GGT (m+k) */
static double kinetic(const double *GGT, const double *k, int m0, int m1, int m2) {
    double x[3] = {m0 + k[0], m1 + k[1], m2 + k[2]};
    double s = 0.0;
    for (int a = 0; a < 3; a++)
        for (int b = 0; b < 3; b++) s += x[a] * GGT[3 * a + b] * x[b];
    return 0.5 * s;
}

static int smooth235(int n) {
    if (n < 1) return 0;
    while (n % 2 == 0) n /= 2;
    while (n % 3 == 0) n /= 3;
    while (n % 5 == 0) n /= 5;
    return n == 1;
}

static int posmod(int a, int n) {
    int r = a % n;
    return r < 0 ? r + n : r;
}

int jdft_ref_basis_destroy(jdft_ref_basis *b);

int jdft_ref_basis_create(const double *R, const double *k, double Ecut, const int *S,
                          jdft_ref_basis **out) {
    if (!R || !k || !S || !out || !(Ecut > 0.0)) return REF_EINVAL;
    for (int d = 0; d < 3; d++)
        if (!smooth235(S[d])) return REF_EBOX;
    if (det3(R) == 0.0) return REF_EINVAL;
    jdft_ref_basis *b = (jdft_ref_basis *)calloc(1, sizeof(*b));
    if (!b) return REF_ENOMEM;
    memcpy(b->R, R, sizeof(b->R));
    memcpy(b->k, k, sizeof(b->k));
    memcpy(b->S, S, sizeof(b->S));
    b->Ecut = Ecut;
    b->volume = fabs(det3(R));
    recip(R, b->G);
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double s = 0.0;
            for (int l = 0; l < 3; l++) s += b->G[3 * i + l] * b->G[3 * j + l];
            b->GGT[3 * i + j] = s;
        }
    b->N = (int64_t)S[0] * S[1] * S[2];
    /* Plain whole-range sweep ("brute force"): no ellipsoid geometry is used to bound the loop.
     * Per axis the range is the 2 S_d + 1 integers centred on the integer nearest to -k_d (the centre of the cutoff
     * region): any region that passes the box test below (extent < S_d) lies inside it, and a region that does not
     * still shows an extent >= S_d inside it (it is convex and centred within 1/2 of the range's centre).          */
    int lo[3], hi[3];
    for (int d = 0; d < 3; d++) {
        int c = (int)lround(-k[d]);
        lo[d] = c - S[d];
        hi[d] = c + S[d];
    }
    /* two brute-force sweeps: count, then fill, in (m0, m1, m2) lexicographic order, m2 fastest */
    for (int pass = 0; pass < 2; pass++) {
        int64_t n = 0;
        int mn[3] = {1 << 30, 1 << 30, 1 << 30}, mx[3] = {-(1 << 30), -(1 << 30), -(1 << 30)};
        for (int m0 = lo[0]; m0 <= hi[0]; m0++)
            for (int m1 = lo[1]; m1 <= hi[1]; m1++)
                for (int m2 = lo[2]; m2 <= hi[2]; m2++) {
                    double e = kinetic(b->GGT, k, m0, m1, m2);
                    if (e < Ecut) {
                        if (pass == 1) {
                            b->iG[3 * n + 0] = m0;
                            b->iG[3 * n + 1] = m1;
                            b->iG[3 * n + 2] = m2;
                            b->index[n] =
                                (posmod(m0, S[0]) * S[1] + posmod(m1, S[1])) * S[2] + posmod(m2, S[2]);
                            b->ke[n] = e;
                        }
                        int m[3] = {m0, m1, m2};
                        for (int d = 0; d < 3; d++) {
                            if (m[d] < mn[d]) mn[d] = m[d];
                            if (m[d] > mx[d]) mx[d] = m[d];
                        }
                        n++;
                    }
                }
        if (pass == 0) {
            if (n == 0) { free(b); return REF_EINVAL; }
            for (int d = 0; d < 3; d++)
                if (mx[d] - mn[d] >= S[d]) { free(b); return REF_EBOX; } /* two points would collide */
            b->nG = n;
            b->iG = (int32_t *)malloc(sizeof(int32_t) * 3 * n);
            b->index = (int32_t *)malloc(sizeof(int32_t) * n);
            b->ke = (double *)malloc(sizeof(double) * n);
            if (!b->iG || !b->index || !b->ke) return REF_ENOMEM;
        }
    }
    /* separate collision check, literally: no two sphere points may land on the same box offset */
    {
        unsigned char *seen = (unsigned char *)calloc((size_t)b->N, 1);
        if (!seen) return REF_ENOMEM;
        int dup = 0;
        for (int64_t n = 0; n < b->nG; n++) {
            if (seen[b->index[n]]) dup = 1;
            seen[b->index[n]] = 1;
        }
        free(seen);
        if (dup) { jdft_ref_basis_destroy(b); return REF_EBOX; }
    }
    *out = b;
    return REF_OK;
}

int jdft_ref_basis_destroy(jdft_ref_basis *b) {
    if (!b) return REF_EINVAL;
    free(b->iG);
    free(b->index);
    free(b->ke);
    free(b);
    return REF_OK;
}

int jdft_ref_basis_info(const jdft_ref_basis *b, int64_t *nG, int64_t *N, double *volume) {
    if (!b) return REF_EINVAL;
    if (nG) *nG = b->nG;
    if (N) *N = b->N;
    if (volume) *volume = b->volume;
    return REF_OK;
}

int jdft_ref_basis_export(const jdft_ref_basis *b, int32_t *iG, int32_t *index, double *ke) {
    if (!b) return REF_EINVAL;
    if (iG) memcpy(iG, b->iG, sizeof(int32_t) * 3 * b->nG);
    if (index) memcpy(index, b->index, sizeof(int32_t) * b->nG);
    if (ke) memcpy(ke, b->ke, sizeof(double) * b->nG);
    return REF_OK;
}

/* ---------------------------------------------------------------------- FFT */

/* w[t] = exp(sign 2 pi i t / n), t = 0..n-1, evaluated in long double */
static void twiddle_table(int n, int sign, cplx *w) {
    const long double twopi = 6.283185307179586476925286766559005768L;
    for (int t = 0; t < n; t++) {
        long double a = twopi * (long double)t / (long double)n;
        w[t] = (double)cosl(a) + I * (double)(sign * sinl(a));
    }
}

static int smallest_factor(int n) {
    for (int p = 2; p * p <= n; p++)
        if (n % p == 0) return p;
    return n;
}

/*
 * Recursive decimation in time.  X[q] = sum_j x[j] w_n^{jq}.  Split j = p*s + r:
 *   X[q] = sum_{r<p} w_n^{r q} Y_r[q mod m],  Y_r = DFT_m( x[r], x[r+p], ... ),  m = n/p.
 * in: stride `is`; out: contiguous; w: table for the TOP length nTop, ws = nTop / n.
 */
static void fft_rec(int n, const cplx *in, int is, cplx *out, const cplx *w, int nTop, cplx *scratch) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = smallest_factor(n), m = n / p, ws = nTop / n;
    cplx *Y = scratch; /* p blocks of m */
    for (int r = 0; r < p; r++) fft_rec(m, in + (size_t)r * is, is * p, Y + (size_t)r * m, w, nTop, scratch + n);
    for (int q = 0; q < n; q++) {
        cplx s = 0.0;
        for (int r = 0; r < p; r++) {
            int e = (int)(((int64_t)r * q) % n);
            s += w[(size_t)e * ws] * Y[(size_t)r * m + (q % m)];
        }
        out[q] = s;
    }
}

/* In-place 1-D DFT of `n` points with stride `stride`; sign = +1 or -1; unnormalised. */
int jdft_ref_fft1d(double *data, int n, int stride, int sign) {
    if (!data || n < 1 || (sign != 1 && sign != -1)) return REF_EINVAL;
    cplx *x = (cplx *)data;
    cplx *w = (cplx *)malloc(sizeof(cplx) * n);
    cplx *buf = (cplx *)malloc(sizeof(cplx) * n);
    cplx *scratch = (cplx *)malloc(sizeof(cplx) * 2 * (size_t)n + 64);
    if (!w || !buf || !scratch) return REF_ENOMEM;
    twiddle_table(n, sign, w);
    fft_rec(n, x, stride, buf, w, n, scratch);
    for (int q = 0; q < n; q++) x[(size_t)q * stride] = buf[q];
    free(w); free(buf); free(scratch);
    return REF_OK;
}

/* In-place 3-D DFT of one box [S0][S1][S2]: three passes, one axis each, every pencil. */
static int fft3d(cplx *box, const int *S, int sign) {
    const int64_t strides[3] = {(int64_t)S[1] * S[2], S[2], 1};
    for (int ax = 2; ax >= 0; ax--) {
        int n = S[ax];
        cplx *w = (cplx *)malloc(sizeof(cplx) * n);
        cplx *in = (cplx *)malloc(sizeof(cplx) * n);
        cplx *outb = (cplx *)malloc(sizeof(cplx) * n);
        cplx *scratch = (cplx *)malloc(sizeof(cplx) * 2 * (size_t)n + 64);
        if (!w || !in || !outb || !scratch) return REF_ENOMEM;
        twiddle_table(n, sign, w);
        int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
        for (int u = 0; u < S[a1]; u++)
            for (int v = 0; v < S[a2]; v++) {
                cplx *base = box + u * strides[a1] + v * strides[a2];
                for (int t = 0; t < n; t++) in[t] = base[t * strides[ax]];
                fft_rec(n, in, 1, outb, w, n, scratch);
                for (int t = 0; t < n; t++) base[t * strides[ax]] = outb[t];
            }
        free(w); free(in); free(outb); free(scratch);
    }
    return REF_OK;
}

/* ---------------------------------------------------------------- operators */

/* I: [nb][nG] -> [nb][N].  Scatter into a zeroed box, then DFT with sign +. */
int jdft_ref_apply_I(const jdft_ref_basis *b, const double *C_, int nb, double *psi_) {
    if (!b || !C_ || !psi_ || nb < 0) return REF_EINVAL;
    const cplx *C = (const cplx *)C_;
    cplx *psi = (cplx *)psi_;
    int err = 0;
#pragma omp parallel for schedule(dynamic)
    for (int ib = 0; ib < nb; ib++) {
        cplx *box = psi + (size_t)ib * b->N;
        memset(box, 0, sizeof(cplx) * b->N);
        for (int64_t n = 0; n < b->nG; n++) box[b->index[n]] = C[(size_t)ib * b->nG + n];
        if (fft3d(box, b->S, +1)) err = 1;
    }
    return err ? REF_ENOMEM : REF_OK;
}

/* Idag (scale = 1) and J (scale = 1/N): [nb][N] -> [nb][nG].  DFT with sign -, then gather. */
static int idag_scaled(const jdft_ref_basis *b, const double *psi_, int nb, double *C_, double scale) {
    if (!b || !C_ || !psi_ || nb < 0) return REF_EINVAL;
    const cplx *psi = (const cplx *)psi_;
    cplx *C = (cplx *)C_;
    int err = 0;
#pragma omp parallel for schedule(dynamic)
    for (int ib = 0; ib < nb; ib++) {
        cplx *box = (cplx *)malloc(sizeof(cplx) * b->N);
        if (!box) { err = 1; continue; }
        memcpy(box, psi + (size_t)ib * b->N, sizeof(cplx) * b->N);
        if (fft3d(box, b->S, -1)) err = 1;
        for (int64_t n = 0; n < b->nG; n++) C[(size_t)ib * b->nG + n] = scale * box[b->index[n]];
        free(box);
    }
    return err ? REF_ENOMEM : REF_OK;
}

int jdft_ref_apply_Idag(const jdft_ref_basis *b, const double *psi, int nb, double *C) {
    return idag_scaled(b, psi, nb, C, 1.0);
}

int jdft_ref_apply_J(const jdft_ref_basis *b, const double *psi, int nb, double *C) {
    if (!b) return REF_EINVAL;
    return idag_scaled(b, psi, nb, C, 1.0 / (double)b->N);
}

/* L C = -Omega |G+k|^2 C = -2 Omega ke C */
int jdft_ref_apply_L(const jdft_ref_basis *b, const double *C_, int nb, double *out_) {
    if (!b || !C_ || !out_ || nb < 0) return REF_EINVAL;
    const cplx *C = (const cplx *)C_;
    cplx *out = (cplx *)out_;
    for (int ib = 0; ib < nb; ib++)
        for (int64_t n = 0; n < b->nG; n++)
            out[(size_t)ib * b->nG + n] = (-2.0 * b->volume * b->ke[n]) * C[(size_t)ib * b->nG + n];
    return REF_OK;
}

/* O C = Omega C */
int jdft_ref_apply_O(const jdft_ref_basis *b, const double *C_, int nb, double *out_) {
    if (!b || !C_ || !out_ || nb < 0) return REF_EINVAL;
    const cplx *C = (const cplx *)C_;
    cplx *out = (cplx *)out_;
    for (int64_t i = 0; i < (int64_t)nb * b->nG; i++) out[i] = b->volume * C[i];
    return REF_OK;
}

/*
 * Vnl: out (+)= P D P^+ C.
 *   B[ib][j]  = sum_n conj(P[j][n]) C[ib][n]
 *   B'[ib][j] = D[j] B[ib][j]            (D_mode 0)   or   sum_l D[j][l] B[ib][l]   (D_mode 1)
 *   or, D_mode = nblk >= 2 (per-atom Hermitian blocks c128[np/nblk][nblk][nblk], reading 24; PAPER.md:95
 *   ultrasoft pseudopotentials couple the projectors of one atom only):
 *   B'[ib][a nblk + j'] = sum_l' D[a][j'][l'] B[ib][a nblk + l']
 *   out[ib][n] (+)= sum_j P[j][n] B'[ib][j]
 */
int jdft_ref_apply_Vnl(const jdft_ref_basis *b, const double *P_, int np, const double *D, int D_mode,
                       const double *C_, int nb, double *out_, int accumulate) {
    if (!b || !C_ || !out_ || nb < 0 || np < 0 || (np > 0 && (!P_ || !D)) || D_mode < 0 || (D_mode >= 2 && np % D_mode != 0))
        return REF_EINVAL;
    const cplx *P = (const cplx *)P_, *C = (const cplx *)C_;
    cplx *out = (cplx *)out_;
    const int64_t nG = b->nG;
    int err = 0;
#pragma omp parallel for schedule(dynamic)
    for (int ib = 0; ib < nb; ib++) {
        cplx *B = (cplx *)malloc(sizeof(cplx) * (np > 0 ? np : 1));
        cplx *B2 = (cplx *)malloc(sizeof(cplx) * (np > 0 ? np : 1));
        if (!B || !B2) { err = 1; free(B); free(B2); continue; }
        for (int j = 0; j < np; j++) {
            long double sr = 0.0L, si = 0.0L;
            for (int64_t n = 0; n < nG; n++) {
                long double pr = creal(P[(size_t)j * nG + n]), pi = cimag(P[(size_t)j * nG + n]);
                long double cr = creal(C[(size_t)ib * nG + n]), ci = cimag(C[(size_t)ib * nG + n]);
                sr += pr * cr + pi * ci; /* conj(p) * c */
                si += pr * ci - pi * cr;
            }
            B[j] = (double)sr + I * (double)si;
        }
        for (int j = 0; j < np; j++) {
            if (D_mode == 0) {
                B2[j] = D[j] * B[j];
            } else if (D_mode == 1) {
                const cplx *Dc = (const cplx *)D;
                lcplx s = 0.0L;
                for (int l = 0; l < np; l++) s += (lcplx)Dc[(size_t)j * np + l] * (lcplx)B[l];
                B2[j] = (cplx)s;
            } else { /* per-atom blocks: D[a][j'][l'], a = j / nblk, only projectors of the same atom couple */
                const int nblk = D_mode, a = j / nblk, jj = j % nblk;
                const cplx *Da = (const cplx *)D + (size_t)a * nblk * nblk;
                lcplx s = 0.0L;
                for (int l = 0; l < nblk; l++) s += (lcplx)Da[(size_t)jj * nblk + l] * (lcplx)B[(size_t)a * nblk + l];
                B2[j] = (cplx)s;
            }
        }
        for (int64_t n = 0; n < nG; n++) {
            long double sr = 0.0L, si = 0.0L;
            for (int j = 0; j < np; j++) {
                long double pr = creal(P[(size_t)j * nG + n]), pi = cimag(P[(size_t)j * nG + n]);
                long double br = creal(B2[j]), bi = cimag(B2[j]);
                sr += pr * br - pi * bi;
                si += pr * bi + pi * br;
            }
            cplx v = (double)sr + I * (double)si;
            if (accumulate) out[(size_t)ib * nG + n] += v;
            else out[(size_t)ib * nG + n] = v;
        }
        free(B); free(B2);
    }
    return err ? REF_ENOMEM : REF_OK;
}

/* P^+ C alone ([nb][np]); exposed so tests can compare the projection step by itself */
int jdft_ref_project(const jdft_ref_basis *b, const double *P_, int np, const double *C_, int nb, double *B_) {
    if (!b || !P_ || !C_ || !B_ || nb < 0 || np < 0) return REF_EINVAL;
    const cplx *P = (const cplx *)P_, *C = (const cplx *)C_;
    cplx *B = (cplx *)B_;
    const int64_t nG = b->nG;
#pragma omp parallel for schedule(dynamic) collapse(2)
    for (int ib = 0; ib < nb; ib++)
        for (int j = 0; j < np; j++) {
            long double sr = 0.0L, si = 0.0L;
            for (int64_t n = 0; n < nG; n++) {
                long double pr = creal(P[(size_t)j * nG + n]), pi = cimag(P[(size_t)j * nG + n]);
                long double cr = creal(C[(size_t)ib * nG + n]), ci = cimag(C[(size_t)ib * nG + n]);
                sr += pr * cr + pi * ci;
                si += pr * ci - pi * cr;
            }
            B[(size_t)ib * np + j] = (double)sr + I * (double)si;
        }
    return REF_OK;
}

/*
 * H C = -1/2 L C + I^+( Vloc .* (I C) ) + P D P^+ C       (BASELINE.json north_star)
 * Vloc is f64[N], used exactly as passed (the caller folds in the Omega/N weight; reading 5).
 */
int jdft_ref_apply_H(const jdft_ref_basis *b, const double *Vloc, const double *P, int np, const double *D,
                     int D_mode, const double *C_, int nb, double *HC_) {
    if (!b || !Vloc || !C_ || !HC_ || nb < 0 || np < 0) return REF_EINVAL;
    const cplx *C = (const cplx *)C_;
    cplx *HC = (cplx *)HC_;
    const int64_t nG = b->nG, N = b->N;
    int err = 0;
#pragma omp parallel for schedule(dynamic)
    for (int ib = 0; ib < nb; ib++) {
        cplx *box = (cplx *)calloc(N, sizeof(cplx));
        if (!box) { err = 1; continue; }
        /* I C */
        for (int64_t n = 0; n < nG; n++) box[b->index[n]] = C[(size_t)ib * nG + n];
        if (fft3d(box, b->S, +1)) err = 1;
        /* Diag(Vloc) */
        for (int64_t j = 0; j < N; j++) box[j] *= Vloc[j];
        /* I^+ */
        if (fft3d(box, b->S, -1)) err = 1;
        for (int64_t n = 0; n < nG; n++) HC[(size_t)ib * nG + n] = box[b->index[n]];
        /* -1/2 L C = Omega ke C */
        for (int64_t n = 0; n < nG; n++) HC[(size_t)ib * nG + n] += (b->volume * b->ke[n]) * C[(size_t)ib * nG + n];
        free(box);
    }
    if (err) return REF_ENOMEM;
    if (np > 0) return jdft_ref_apply_Vnl(b, P, np, D, D_mode, C_, nb, HC_, 1);
    return REF_OK;
}

/* M[a + nb1*bb] = Omega sum_n conj(C1[a][n]) C2[bb][n] */
int jdft_ref_overlap(const jdft_ref_basis *b, const double *C1_, int nb1, const double *C2_, int nb2, double *M_) {
    if (!b || !C1_ || !C2_ || !M_ || nb1 < 0 || nb2 < 0) return REF_EINVAL;
    const cplx *C1 = (const cplx *)C1_, *C2 = (const cplx *)C2_;
    cplx *M = (cplx *)M_;
    const int64_t nG = b->nG;
#pragma omp parallel for schedule(dynamic) collapse(2)
    for (int bb = 0; bb < nb2; bb++)
        for (int a = 0; a < nb1; a++) {
            long double sr = 0.0L, si = 0.0L;
            for (int64_t n = 0; n < nG; n++) {
                long double ar = creal(C1[(size_t)a * nG + n]), ai = cimag(C1[(size_t)a * nG + n]);
                long double cr = creal(C2[(size_t)bb * nG + n]), ci = cimag(C2[(size_t)bb * nG + n]);
                sr += ar * cr + ai * ci;
                si += ar * ci - ai * cr;
            }
            M[(size_t)a + (size_t)nb1 * bb] = b->volume * ((double)sr + I * (double)si);
        }
    return REF_OK;
}

/* one element of the overlap (for sampled full-size parity checks) */
int jdft_ref_overlap_entry(const jdft_ref_basis *b, const double *C1_, const double *C2_, int a, int bb, double *out2) {
    if (!b || !C1_ || !C2_ || !out2) return REF_EINVAL;
    const cplx *C1 = (const cplx *)C1_, *C2 = (const cplx *)C2_;
    const int64_t nG = b->nG;
    long double sr = 0.0L, si = 0.0L;
    for (int64_t n = 0; n < nG; n++) {
        long double ar = creal(C1[(size_t)a * nG + n]), ai = cimag(C1[(size_t)a * nG + n]);
        long double cr = creal(C2[(size_t)bb * nG + n]), ci = cimag(C2[(size_t)bb * nG + n]);
        sr += ar * cr + ai * ci;
        si += ar * ci - ai * cr;
    }
    out2[0] = b->volume * (double)sr;
    out2[1] = b->volume * (double)si;
    return REF_OK;
}

/* ---- the steps right after / before H C in every SCF or minimiser iteration
 * ("ElecVars": wavefunctions -> density -> potential; PAPER.md:76 integrals as dot products).
 *
 * subspace:  M[a + nb1*bb] = sum_n conj(C1[a][n]) X2[bb][n]      (no Omega: X2 = H C already carries it)
 * density:   n[j] (+)= sum_b f[b] |(I C_b)[j]|^2                 (I as defined above; f = occupations, real)  */
int jdft_ref_subspace(const jdft_ref_basis *b, const double *C1_, int nb1, const double *X2_, int nb2, double *M_) {
    if (!b || !C1_ || !X2_ || !M_ || nb1 < 0 || nb2 < 0) return REF_EINVAL;
    const cplx *C1 = (const cplx *)C1_, *X2 = (const cplx *)X2_;
    cplx *M = (cplx *)M_;
    const int64_t nG = b->nG;
#pragma omp parallel for schedule(dynamic) collapse(2)
    for (int bb = 0; bb < nb2; bb++)
        for (int a = 0; a < nb1; a++) {
            long double sr = 0.0L, si = 0.0L;
            for (int64_t n = 0; n < nG; n++) {
                long double ar = creal(C1[(size_t)a * nG + n]), ai = cimag(C1[(size_t)a * nG + n]);
                long double cr = creal(X2[(size_t)bb * nG + n]), ci = cimag(X2[(size_t)bb * nG + n]);
                sr += ar * cr + ai * ci;
                si += ar * ci - ai * cr;
            }
            M[(size_t)a + (size_t)nb1 * bb] = (double)sr + I * (double)si;
        }
    return REF_OK;
}

int jdft_ref_density(const jdft_ref_basis *b, const double *C_, int nb, const double *f, double *n, int accumulate) {
    if (!b || !n || nb < 0 || (nb > 0 && (!C_ || !f))) return REF_EINVAL;
    const cplx *C = (const cplx *)C_;
    if (!accumulate) memset(n, 0, sizeof(double) * b->N);
    cplx *box = (cplx *)malloc(sizeof(cplx) * b->N);
    if (!box) return REF_ENOMEM;
    for (int ib = 0; ib < nb; ib++) { /* bands one after the other, in order: a fixed summation order */
        memset(box, 0, sizeof(cplx) * b->N);
        for (int64_t g = 0; g < b->nG; g++) box[b->index[g]] = C[(size_t)ib * b->nG + g];
        if (fft3d(box, b->S, +1)) { free(box); return REF_ENOMEM; }
        for (int64_t j = 0; j < b->N; j++) {
            const double re = creal(box[j]), im = cimag(box[j]);
            n[j] += f[ib] * (re * re + im * im);
        }
    }
    free(box);
    return REF_OK;
}

/* ---- the scalar-field operators of the paper's Listing 1 and eq. (1)
 * (PAPER.md:63):  -4 pi rho = div( epsilon grad phi ),
 *     hessian(phi~) = (-1/(4 pi)) * divergence( J( epsilon * I( gradient(phi~) ) ) ).
 * "the gradient and divergence operators apply in reciprocal space (where they are diagonal)":
 *     gradient:   out[d][n] = i q_d(n) phi[n],  q(n) = G^T (iG[n] + k)  (Cartesian, d = 0,1,2)
 *     divergence: out[n]    = sum_d i q_d(n) X[d][n]
 * Layouts: a field block is [nb][nG]; a vector-field block is [3][nb][nG] (component slowest).  epsilon is f64[N].
 * Reading (#23): I, J exactly as above (J = I^+/N), no extra volume factors.               */
static void qvec(const jdft_ref_basis *b, int64_t n, double *q) {
    const double t[3] = {b->iG[3 * n] + b->k[0], b->iG[3 * n + 1] + b->k[1], b->iG[3 * n + 2] + b->k[2]};
    for (int d = 0; d < 3; d++) q[d] = b->G[0 + d] * t[0] + b->G[3 + d] * t[1] + b->G[6 + d] * t[2]; /* (G^T t)_d */
}

int jdft_ref_gradient(const jdft_ref_basis *b, const double *C_, int nb, double *out_) {
    if (!b || nb < 0 || (nb > 0 && (!C_ || !out_))) return REF_EINVAL;
    const cplx *C = (const cplx *)C_;
    cplx *out = (cplx *)out_;
    const size_t blk = (size_t)nb * b->nG;
    for (int ib = 0; ib < nb; ib++)
        for (int64_t n = 0; n < b->nG; n++) {
            double q[3];
            qvec(b, n, q);
            for (int d = 0; d < 3; d++) out[d * blk + (size_t)ib * b->nG + n] = (I * q[d]) * C[(size_t)ib * b->nG + n];
        }
    return REF_OK;
}

int jdft_ref_divergence(const jdft_ref_basis *b, const double *X_, int nb, double *out_) {
    if (!b || nb < 0 || (nb > 0 && (!X_ || !out_))) return REF_EINVAL;
    const cplx *X = (const cplx *)X_;
    cplx *out = (cplx *)out_;
    const size_t blk = (size_t)nb * b->nG;
    for (int ib = 0; ib < nb; ib++)
        for (int64_t n = 0; n < b->nG; n++) {
            double q[3];
            qvec(b, n, q);
            cplx s = 0.0;
            for (int d = 0; d < 3; d++) s += (I * q[d]) * X[d * blk + (size_t)ib * b->nG + n];
            out[(size_t)ib * b->nG + n] = s;
        }
    return REF_OK;
}

int jdft_ref_pcm_hessian(const jdft_ref_basis *b, const double *epsilon, const double *phi, int nb, double *out) {
    if (!b || nb < 0 || !epsilon || (nb > 0 && (!phi || !out))) return REF_EINVAL;
    const size_t blk = (size_t)nb * b->nG;
    double *g = (double *)malloc(sizeof(cplx) * 3 * blk);          /* gradient(phi) and later J(...)      */
    double *r = (double *)malloc(sizeof(cplx) * 3 * (size_t)nb * b->N); /* I(gradient(phi))             */
    if (!g || !r) { free(g); free(r); return REF_ENOMEM; }
    int rc = jdft_ref_gradient(b, phi, nb, g);
    if (!rc) rc = jdft_ref_apply_I(b, g, 3 * nb, r);
    if (!rc) {
        cplx *rr = (cplx *)r;
        for (size_t f = 0; f < (size_t)3 * nb; f++)
            for (int64_t j = 0; j < b->N; j++) rr[f * b->N + j] *= epsilon[j];      /* epsilon * (...)   */
        rc = jdft_ref_apply_J(b, r, 3 * nb, g);
    }
    if (!rc) rc = jdft_ref_divergence(b, g, nb, out);
    if (!rc) {
        cplx *o = (cplx *)out;
        for (size_t i = 0; i < blk; i++) o[i] *= -1.0 / (4.0 * M_PI);
    }
    free(g);
    free(r);
    return rc;
}

/* ---- ultrasoft pseudopotentials ("norm-conserving and ultrasoft
 * pseudopotentials"; Listing 2's own input uses the GBRV ultrasoft library).  The generalised
 * overlap operator carries a projector term (reading 24):
 *     O_us C = Omega ( C + P Q P^+ C ),        M_us = C1^+ O_us C2   (column-major nb1 x nb2),
 * with Q given as data in the same three layouts as D (Q_mode 0 real diagonal, 1 dense Hermitian, nblk >= 2 per-atom
 * blocks).  Written out literally: the nonlocal product first, then the sum, then the plain inner products.      */
int jdft_ref_apply_O_us(const jdft_ref_basis *b, const double *P, int np, const double *Q, int Q_mode,
                        const double *C_, int nb, double *out_) {
    if (!b || nb < 0 || np < 0 || (nb > 0 && (!C_ || !out_))) return REF_EINVAL;
    int rc = jdft_ref_apply_Vnl(b, P, np, Q, Q_mode, C_, nb, out_, 0);   /* out = P Q P^+ C   (0 when np = 0) */
    if (rc) return rc;
    if (np == 0) memset(out_, 0, sizeof(cplx) * (size_t)nb * b->nG);
    const cplx *C = (const cplx *)C_;
    cplx *out = (cplx *)out_;
    for (int64_t i = 0; i < (int64_t)nb * b->nG; i++) out[i] = b->volume * (C[i] + out[i]);
    return REF_OK;
}

int jdft_ref_overlap_us(const jdft_ref_basis *b, const double *P, int np, const double *Q, int Q_mode,
                        const double *C1, int nb1, const double *C2, int nb2, double *M) {
    if (!b || nb1 < 0 || nb2 < 0 || !C1 || !C2 || !M) return REF_EINVAL;
    double *X = (double *)malloc(sizeof(cplx) * (size_t)(nb2 > 0 ? nb2 : 1) * b->nG);
    if (!X) return REF_ENOMEM;
    int rc = jdft_ref_apply_O_us(b, P, np, Q, Q_mode, C2, nb2, X);       /* X = O_us C2 */
    if (!rc) rc = jdft_ref_subspace(b, C1, nb1, X, nb2, M);              /* M = C1^+ X  */
    free(X);
    return rc;
}

/* ---- Listing 1 on REAL fields (SURVEY.md 8(f) rank 3 "r2c/c2r variant"; `ScalarField epsilon`, phi and
 * rho are real fields, so their ScalarFieldTilde spectra are Hermitian-symmetric, phi~(-G) = conj(phi~(G))).
 * Half-sphere storage (reading 25): for a Gamma-point basis (k = 0) the canonical order is symmetric under
 * inversion, iG[nG-1-n] = -iG[n], the origin is n0 = (nG-1)/2, and the stored half is the tail n = n0 .. nG-1:
 *     phi_h[ib][h] = phi~[n0 + h],   h = 0 .. nGh-1,  nGh = n0 + 1;     phi~[n0 - h] = conj(phi_h[ib][h]);
 * the imaginary part of the G = 0 entry is ignored (a real field has none).  Written out literally: extend to the
 * full sphere, apply the complex operator, keep the stored half.                                                   */
int jdft_ref_pcm_hessian_real(const jdft_ref_basis *b, const double *epsilon, const double *phi_h, int nb, double *out_h) {
    if (!b || nb < 0 || !epsilon || (nb > 0 && (!phi_h || !out_h))) return REF_EINVAL;
    if (b->k[0] != 0.0 || b->k[1] != 0.0 || b->k[2] != 0.0 || b->nG % 2 == 0) return REF_EINVAL;
    const int64_t nG = b->nG, n0 = (nG - 1) / 2, nGh = n0 + 1;
    for (int64_t n = 0; n < nG; n++)                   /* the order really is inversion symmetric */
        for (int d = 0; d < 3; d++)
            if (b->iG[3 * n + d] != -b->iG[3 * (nG - 1 - n) + d]) return REF_EINVAL;
    cplx *full = (cplx *)malloc(sizeof(cplx) * (size_t)(nb > 0 ? nb : 1) * nG);
    cplx *res = (cplx *)malloc(sizeof(cplx) * (size_t)(nb > 0 ? nb : 1) * nG);
    if (!full || !res) { free(full); free(res); return REF_ENOMEM; }
    const cplx *ph = (const cplx *)phi_h;
    for (int ib = 0; ib < nb; ib++) {
        full[(size_t)ib * nG + n0] = creal(ph[(size_t)ib * nGh]);
        for (int64_t h = 1; h < nGh; h++) {
            full[(size_t)ib * nG + n0 + h] = ph[(size_t)ib * nGh + h];
            full[(size_t)ib * nG + n0 - h] = conj(ph[(size_t)ib * nGh + h]);
        }
    }
    int rc = jdft_ref_pcm_hessian(b, epsilon, (const double *)full, nb, (double *)res);
    if (!rc) {
        cplx *oh = (cplx *)out_h;
        for (int ib = 0; ib < nb; ib++)
            for (int64_t h = 0; h < nGh; h++) oh[(size_t)ib * nGh + h] = res[(size_t)ib * nG + n0 + h];
    }
    free(full);
    free(res);
    return rc;
}
