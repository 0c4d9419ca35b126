"""Pins for the CPU oracle (oracle/jdft_ref.c): each test checks it against something OTHER than itself --
brute-force definitions, closed forms, invariants the formulation fixes (BASELINE.json
north_star), and the exact basis sizes in tests/golden/basis_counts.txt.
All CPU-only ("-m 'not gpu'").  A plausible mistake in the oracle (dropped term, wrong sign, wrong index
order, transposed operand, missing Omega or 1/N) fails at least one of these.
"""
import os

import numpy as np
import pytest

import workloads

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rand_c(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _skew_lattice():
    # non-orthogonal cell, columns are lattice vectors
    return np.array([[5.0, 0.7, -0.4], [0.3, 6.0, 0.9], [-0.5, 0.2, 7.0]])


def _brute_I_matrix(b):
    """Explicit N x nG matrix exp(+2 pi i sum_d iG[n]_d j_d / S_d), j in row-major box order."""
    S = b.shape
    j = np.stack(np.meshgrid(np.arange(S[0]), np.arange(S[1]), np.arange(S[2]), indexing="ij"), -1).reshape(-1, 3)
    phase = (j[:, None, :] * b.iG[None, :, :].astype(np.float64) / np.asarray(S, dtype=np.float64)).sum(-1)
    return np.exp(2j * np.pi * phase)


# ------------------------------------------------------------------------------------------ 1-D FFT

@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 7, 8, 9, 10, 12, 15, 25, 27, 30, 32, 45, 60, 72, 80, 125, 128, 216])
@pytest.mark.parametrize("sign", [+1, -1])
def test_fft1d_vs_bruteforce_dft(ref, n, sign):
    rng = np.random.default_rng(n * 7 + sign)
    x = _rand_c(rng, n)
    jq = (np.arange(n)[:, None] * np.arange(n)[None, :]) % n
    W = np.exp(sign * 2j * np.pi * jq.astype(np.longdouble) / n).astype(np.clongdouble)
    want = (W @ x.astype(np.clongdouble)).astype(np.complex128)
    got = ref.fft1d(x, sign)
    assert np.max(np.abs(got - want)) <= 1e-13 * np.sqrt(n) * np.max(np.abs(want))


def test_fft1d_delta_and_constant(ref):
    n = 60
    x = np.zeros(n, complex); x[7] = 1.0
    got = ref.fft1d(x, +1)
    assert np.allclose(got, np.exp(2j * np.pi * 7 * np.arange(n) / n), atol=1e-15)
    got = ref.fft1d(np.ones(n, complex), -1)
    want = np.zeros(n, complex); want[0] = n
    assert np.allclose(got, want, atol=1e-13)


# ------------------------------------------------------------------------------------------ basis

def _golden_counts():
    rows = []
    with open(os.path.join(GOLDEN, "basis_counts.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([int(t) for t in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden_counts(), ids=lambda r: "cfg%d_k%d" % (r[0], r[1]))
def test_basis_exact_counts_and_extents(ref, row):
    cfg, ik, nG, *ext = row
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[ik], Ecut, S)
    assert b.nG == nG
    got = [b.iG[:, 0].min(), b.iG[:, 0].max(), b.iG[:, 1].min(), b.iG[:, 1].max(), b.iG[:, 2].min(), b.iG[:, 2].max()]
    assert got == ext
    # continuum estimate Omega (2 Ecut)^{3/2} / (6 pi^2) within 0.5 %
    cont = b.volume * (2 * Ecut) ** 1.5 / (6 * np.pi ** 2)
    assert abs(b.nG - cont) / cont < 5e-3


def test_basis_bruteforce_order_index_and_symmetry(ref):
    R = _skew_lattice()
    S = (12, 15, 16)
    for k in ([0.0, 0.0, 0.0], [0.25, -0.1, 0.4]):
        Ecut = 6.0
        b = ref.RefBasis(R, k, Ecut, S)
        # independent evaluation through CARTESIAN q = G^T (m + k) with numpy's inverse
        G = 2 * np.pi * np.linalg.inv(R)
        rng_ = [np.arange(-(s // 2), (s + 1) // 2) for s in S]
        m = np.stack(np.meshgrid(*rng_, indexing="ij"), -1).reshape(-1, 3)   # lexicographic, m2 fastest
        q = (m + np.asarray(k)) @ G                                           # rows: G^T (m+k)
        ke = 0.5 * (q * q).sum(1)
        keep = ke < Ecut
        assert b.nG == keep.sum()
        assert np.array_equal(b.iG, m[keep].astype(np.int32))
        assert np.allclose(b.ke, ke[keep], rtol=1e-13, atol=0)
        mm = m[keep] % np.asarray(S)
        assert np.array_equal(b.index, ((mm[:, 0] * S[1] + mm[:, 1]) * S[2] + mm[:, 2]).astype(np.int32))
        assert len(np.unique(b.index)) == b.nG
        if not any(k):
            have = {tuple(t) for t in b.iG.tolist()}
            assert all((-a, -bb, -c) in have for (a, bb, c) in have)   # Gamma: m in B <=> -m in B
    assert np.isclose(b.volume, abs(np.linalg.det(R)), rtol=1e-14)


def test_basis_cubic_gamma_closed_form_ke(ref):
    L = 10.0
    b = ref.RefBasis(np.diag([L, L, L]), [0, 0, 0], 10.0, (32, 32, 32))
    m2 = (b.iG.astype(np.int64) ** 2).sum(1)
    assert np.allclose(b.ke, 0.5 * (2 * np.pi / L) ** 2 * m2, rtol=1e-14)
    assert np.all(b.ke < 10.0) and b.nG == np.sum(0.5 * (2 * np.pi / L) ** 2 * ((np.indices((33, 33, 33)) - 16) ** 2).sum(0) < 10.0)


def test_volumes(ref):
    want = {1: 1000.0, 2: 8615.125, 3: 27000.0, 4: 24000.0, 5: 28934.443}
    for cfg, vol in want.items():
        R, kpts, Ecut, S = workloads.lattice(cfg)
        assert np.isclose(abs(np.linalg.det(R)), vol, rtol=1e-12)
    b = ref.RefBasis(np.diag([20.5] * 3), [0.25] * 3, 2.0, (20, 20, 20))
    assert np.isclose(b.volume, 8615.125, rtol=1e-14)


def test_basis_errors(ref):
    with pytest.raises(ref.RefError):      # 7 is not 2,3,5-smooth
        ref.RefBasis(np.eye(3) * 10, [0, 0, 0], 5.0, (14, 16, 16))
    with pytest.raises(ref.RefError):      # sphere wider than the box -> collision
        ref.RefBasis(np.eye(3) * 10, [0, 0, 0], 10.0, (8, 32, 32))


# ------------------------------------------------------------------------------------------ I, Idag, J

@pytest.mark.parametrize("S,k,R,Ecut", [((8, 8, 8), (0, 0, 0), np.eye(3) * 7.0, 3.0),
                                        ((4, 6, 5), (0.3, -0.2, 0.1), _skew_lattice(), 1.6),
                                        ((8, 9, 10), (0.5, 0.25, -0.125), _skew_lattice() * 1.3, 2.5)])
def test_I_Idag_vs_explicit_matrix(ref, S, k, R, Ecut):
    b = ref.RefBasis(R, k, Ecut, S)
    assert b.nG > 12
    rng = np.random.default_rng(11)
    E = _brute_I_matrix(b)
    C = _rand_c(rng, 3, b.nG)
    psi = b.apply_I(C).reshape(3, -1)
    want = C @ E.T
    assert np.max(np.abs(psi - want)) <= 1e-12 * np.max(np.abs(want))
    f = _rand_c(rng, 2, b.N)
    got = b.apply_Idag(f)
    want = f @ E.conj()
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))
    assert np.allclose(b.apply_J(f), want / b.N, rtol=0, atol=1e-13 * np.max(np.abs(want)))


def test_I_matches_numpy_ifftn(ref):
    R, kpts, Ecut, S = workloads.lattice(1)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    rng = np.random.default_rng(5)
    C = _rand_c(rng, 2, b.nG)
    box = np.zeros((2, b.N), complex)
    box[:, b.index] = C
    want = np.fft.ifftn(box.reshape((2,) + b.shape), axes=(1, 2, 3)) * b.N
    got = b.apply_I(C)
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))


def test_JI_identity_IJ_idempotent_parseval_adjoint(ref):
    R = _skew_lattice() * 2.0
    b = ref.RefBasis(R, [0.2, 0.1, -0.3], 5.0, (24, 30, 32))
    rng = np.random.default_rng(3)
    C = _rand_c(rng, 3, b.nG)
    psi = b.apply_I(C)
    # J I = 1 ("and vice versa")
    assert np.max(np.abs(b.apply_J(psi) - C)) <= 1e-13 * np.max(np.abs(C))
    # Parseval: sum_j |psi|^2 = N sum_n |C|^2
    assert np.allclose((np.abs(psi) ** 2).sum(axis=(1, 2, 3)), b.N * (np.abs(C) ** 2).sum(1), rtol=1e-13)
    # I J is idempotent
    f = _rand_c(rng, 2, b.N)
    g = b.apply_I(b.apply_J(f))
    g2 = b.apply_I(b.apply_J(g))
    assert np.max(np.abs(g2 - g)) <= 1e-13 * np.max(np.abs(g))
    # adjointness <f, I C> = <Idag f, C>
    lhs = np.vdot(f[0], psi[0].reshape(-1))
    rhs = np.vdot(b.apply_Idag(f[:1])[0], C[0])
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


def test_cos_potential_closed_form_sign_and_wrap(ref):
    """V[j] = cos(2 pi mv.j/S) => Idag(V .* I e_m) = (N/2)(e_{m+mv} + e_{m-mv}) restricted to the sphere."""
    R, kpts, Ecut, S = workloads.lattice(101)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    mv = np.array([1, -2, 1])
    j = np.stack(np.meshgrid(*[np.arange(s) for s in S], indexing="ij"), -1)
    V = np.cos(2 * np.pi * (j * mv / np.asarray(S)).sum(-1))
    lookup = {tuple(m): n for n, m in enumerate(b.iG.tolist())}
    for n0 in (0, b.nG // 2, b.nG - 1):
        C = np.zeros((1, b.nG), complex); C[0, n0] = 1.0
        got = b.apply_Idag(V[None] * b.apply_I(C))[0]
        want = np.zeros(b.nG, complex)
        for sgn in (+1, -1):
            t = tuple((b.iG[n0] + sgn * mv).tolist())
            if t in lookup:
                want[lookup[t]] += 0.5 * b.N
        assert np.max(np.abs(got - want)) <= 1e-12 * b.N
        # an asymmetric (complex) potential exp(+2 pi i mv.j/S) must shift m -> m + mv, not m - mv
        Vc = np.exp(2j * np.pi * (j * mv / np.asarray(S)).sum(-1))
        got = b.apply_Idag(Vc[None] * b.apply_I(C))[0]
        want = np.zeros(b.nG, complex)
        t = tuple((b.iG[n0] + mv).tolist())
        if t in lookup:
            want[lookup[t]] = b.N
        assert np.max(np.abs(got - want)) <= 1e-12 * b.N


# ------------------------------------------------------------------------------------------ L, O, overlap

def test_L_O_closed_forms(ref):
    R = _skew_lattice()
    k = np.array([0.1, 0.2, -0.3])
    b = ref.RefBasis(R, k, 5.0, (16, 18, 20))
    rng = np.random.default_rng(9)
    C = _rand_c(rng, 2, b.nG)
    G = 2 * np.pi * np.linalg.inv(R)
    q = (b.iG + k) @ G
    q2 = (q * q).sum(1)
    vol = abs(np.linalg.det(R))
    assert np.allclose(b.apply_L(C), -vol * q2[None, :] * C, rtol=1e-13)
    assert np.allclose(b.apply_O(C), vol * C, rtol=1e-15)


def test_overlap_orthonormal_bands_and_library_gemm(ref):
    cfg = 102
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    C = workloads.make_bands(cfg, b.nG)
    M = b.overlap(C, C)
    assert np.max(np.abs(M - np.eye(C.shape[0]))) <= 1e-13           # generator: C^+ O C = 1
    rng = np.random.default_rng(2)
    C1, C2 = _rand_c(rng, 4, b.nG), _rand_c(rng, 7, b.nG)
    M = b.overlap(C1, C2)
    want = b.volume * (C1.conj() @ C2.T)                              # M[a, b] = Omega sum_n conj(C1[a,n]) C2[b,n]
    assert M.shape == (4, 7) and np.max(np.abs(M - want)) <= 1e-13 * np.max(np.abs(want))
    assert abs(b.overlap_entry(C1, C2, 3, 5) - want[3, 5]) <= 1e-13 * abs(want[3, 5])
    assert np.allclose(b.overlap(C2, C1), M.conj().T, rtol=1e-14)


# ------------------------------------------------------------------------------------------ Vnl

def test_Vnl_dense_matrix_rank1_zeroD_denseD(ref):
    cfg = 101
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    assert b.nG <= 400
    inp = workloads.make_inputs(cfg, b.iG)
    P, D, C = inp["P"], inp["D"], inp["C"]
    Pm = P.T                                        # nG x np
    Vnl = Pm @ np.diag(D) @ Pm.conj().T             # dense nG x nG
    want = C @ Vnl.T                                 # row b: Vnl @ C[b]
    got = b.apply_Vnl(P, D, C)
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))
    # projection alone
    assert np.allclose(b.project(P, C), C @ Pm.conj(), rtol=1e-13, atol=1e-15)
    # rank one: d p (p^+ c)
    p, d = P[:1], np.array([0.7])
    got = b.apply_Vnl(p, d, C)
    want = np.stack([d[0] * p[0] * np.vdot(p[0], c) for c in C])
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))
    # D = 0 => 0 ; accumulate adds
    assert np.all(b.apply_Vnl(P, np.zeros_like(D), C) == 0)
    base = np.ones_like(C)
    assert np.allclose(b.apply_Vnl(P, D, C, out=base), 1.0 + b.apply_Vnl(P, D, C), rtol=1e-14)
    # dense Hermitian D
    rng = np.random.default_rng(4)
    A = _rand_c(rng, P.shape[0], P.shape[0]); Dd = A + A.conj().T
    got = b.apply_Vnl(P, Dd, C)
    want = C @ (Pm @ Dd @ Pm.conj().T).T
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))


# ------------------------------------------------------------------------------------------ H

def test_plane_wave_eigenvalue(ref):
    """C = e_n, V_loc = (Omega/N) V0, no projectors => HC = (ke[n] + V0) Omega e_n, zero elsewhere."""
    R, kpts, Ecut, S = workloads.lattice(101)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    V0 = -0.37
    V = np.full(b.shape, V0 * b.volume / b.N)
    for n0 in (0, 17, b.nG - 1):
        C = np.zeros((1, b.nG), complex); C[0, n0] = 1.0 - 0.5j
        HC = b.apply_H(V, None, None, C)[0]
        want = np.zeros(b.nG, complex); want[n0] = (b.ke[n0] + V0) * b.volume * C[0, n0]
        assert np.max(np.abs(HC - want)) <= 1e-13 * b.volume
        ray = np.vdot(C[0], HC) / np.vdot(C[0], b.apply_O(C)[0])
        assert abs(ray - (b.ke[n0] + V0)) <= 1e-13


def test_H_is_sum_of_its_terms_and_hermitian(ref):
    cfg = 102
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    inp = workloads.make_inputs(cfg, b.iG, nb=4)
    V, P, D, C = inp["Vloc"], inp["P"], inp["D"], inp["C"]
    HC = b.apply_H(V, P, D, C)
    terms = -0.5 * b.apply_L(C) + b.apply_Idag(V[None] * b.apply_I(C)) + b.apply_Vnl(P, D, C)
    assert np.max(np.abs(HC - terms)) <= 1e-13 * np.max(np.abs(HC))
    # Hermiticity to 1e-12 (north_star): a^+ H b = conj(b^+ H a)
    rng = np.random.default_rng(8)
    ab = _rand_c(rng, 2, b.nG)
    Hab = b.apply_H(V, P, D, ab)
    lhs, rhs = np.vdot(ab[0], Hab[1]), np.conj(np.vdot(ab[1], Hab[0]))
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(ab[0]) * np.linalg.norm(Hab[1])
    # and with a dense Hermitian D
    A = _rand_c(rng, P.shape[0], P.shape[0]); Dd = A + A.conj().T
    Hab = b.apply_H(V, P, Dd, ab)
    lhs, rhs = np.vdot(ab[0], Hab[1]), np.conj(np.vdot(ab[1], Hab[0]))
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(ab[0]) * np.linalg.norm(Hab[1])


def test_translation_covariance(ref):
    """Roll V_loc by grid vector s, move atoms by s/S, C'_m = exp(-2 pi i m.s/S) C_m
    => (H'C')_m = exp(-2 pi i m.s/S) (HC)_m.  Pins the FFT sign against the structure-factor sign."""
    cfg = 105
    R, kpts, Ecut, S = workloads.lattice(cfg)
    k = kpts[0]
    b = ref.RefBasis(R, k, Ecut, S)
    atoms = workloads.atoms_fractional(cfg)
    V = workloads.make_vloc(cfg, atoms)
    D = workloads.make_D(cfg)
    C = workloads.make_bands(cfg, b.nG, nb=3)
    P = workloads.make_projectors(cfg, b.iG, k, atoms)
    HC = b.apply_H(V, P, D, C)
    s = np.array([3, -4, 5])
    atoms2 = atoms + s / np.asarray(S, dtype=float)
    V2 = np.roll(V, shift=tuple(s), axis=(0, 1, 2))
    P2 = workloads.make_projectors(cfg, b.iG, k, atoms2)
    ph = np.exp(-2j * np.pi * (b.iG * (s / np.asarray(S, dtype=float))).sum(1))
    # projectors carry exp(-2 pi i (m + k).x): the k part is a global phase per atom and cancels in P D P^+
    HC2 = b.apply_H(V2, P2, D, C * ph[None, :])
    assert np.max(np.abs(HC2 - ph[None, :] * HC)) <= 1e-12 * np.max(np.abs(HC))


# ------------------------------------------------------------------------------------------ SURVEY 8(f) rank 1
# subspace matrix C1^+ X2 and density n = sum_b f_b |I C_b|^2 (PAPER.md:127 ElecVars: wavefunctions -> density)

def test_density_vs_explicit_matrix_closed_forms_and_invariants(ref):
    rng = np.random.default_rng(41)
    b = ref.RefBasis(_skew_lattice(), [0.2, -0.1, 0.3], 6.0, (8, 9, 10))
    nb = 4
    C = _rand_c(rng, nb, b.nG)
    f = np.array([2.0, 1.5, 0.25, 0.0])
    n = b.density(C, f)
    # brute force: explicit N x nG matrix of I (independent of the oracle's FFT)
    psi = (_brute_I_matrix(b) @ C.T).T.reshape((nb,) + b.shape)
    want = np.einsum("b,bijk->ijk", f, np.abs(psi) ** 2)
    assert np.max(np.abs(n - want)) <= 1e-11 * np.max(want)
    # Parseval: sum_j n[j] = N sum_b f_b sum_n |C_b[n]|^2 ; with quadrature weight Omega/N this is sum_b f_b C_b^+ O C_b
    assert abs(n.sum() - b.N * np.sum(f * np.sum(np.abs(C) ** 2, axis=1))) <= 1e-11 * n.sum()
    assert abs(n.sum() * b.volume / b.N - np.sum(f * np.real(np.diag(b.overlap(C, C))))) <= 1e-10 * n.sum()
    # real, non-negative, linear in f, accumulate adds, a band with f = 0 contributes nothing
    assert n.min() >= 0.0
    assert np.max(np.abs(b.density(C, 3.0 * f) - 3.0 * n)) <= 1e-12 * n.max()
    assert np.max(np.abs(b.density(C[:3], f[:3]) - n)) == 0.0
    acc = b.density(C[:2], f[:2])
    b.density(C[2:], f[2:], acc)
    assert np.max(np.abs(acc - n)) <= 1e-13 * n.max()
    # one plane wave: constant density f |c|^2 ; two plane waves: closed-form cosine with the + sign convention of I
    n1, n2 = 5, b.nG - 7
    e = np.zeros((1, b.nG), dtype=np.complex128)
    e[0, n1] = 0.3 - 0.4j
    assert np.max(np.abs(b.density(e, [2.0]) - 2.0 * 0.25)) <= 1e-14
    c1, c2 = 0.7 + 0.2j, -0.3 + 0.5j
    e[0, n1], e[0, n2] = c1, c2
    S = np.asarray(b.shape, dtype=np.float64)
    j = np.stack(np.meshgrid(*[np.arange(s) for s in b.shape], indexing="ij"), -1)
    dm = (b.iG[n1] - b.iG[n2]).astype(np.float64)
    phase = 2 * np.pi * (j * dm / S).sum(-1)
    want2 = abs(c1) ** 2 + abs(c2) ** 2 + 2 * np.real(c1 * np.conj(c2) * np.exp(1j * phase))
    assert np.max(np.abs(b.density(e, [1.0]) - want2)) <= 1e-13


def test_density_translation_covariance(ref):
    """C'_m = exp(-2 pi i m.s/S) C_m shifts psi, hence the density, by the grid vector s."""
    rng = np.random.default_rng(43)
    b = ref.RefBasis(np.diag([6.0, 7.0, 8.0]), [0.0, 0.0, 0.0], 5.0, (10, 12, 9))
    C = _rand_c(rng, 2, b.nG)
    f = np.array([1.0, 0.5])
    s = np.array([3, 5, 2])
    ph = np.exp(-2j * np.pi * (b.iG * s / np.asarray(b.shape, dtype=np.float64)).sum(-1))
    n0 = b.density(C, f)
    n1 = b.density(C * ph[None, :], f)
    assert np.max(np.abs(n1 - np.roll(n0, tuple(s), axis=(0, 1, 2)))) <= 1e-12 * n0.max()


def test_subspace_vs_numpy_and_hermitian_for_H(ref):
    rng = np.random.default_rng(47)
    cfg = 101
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    inp = workloads.make_inputs(cfg, b.iG)
    C, X = inp["C"], _rand_c(rng, 3, b.nG)
    M = b.subspace(C, X)
    assert M.shape == (C.shape[0], 3)
    assert np.max(np.abs(M - C.conj() @ X.T)) <= 1e-13 * np.max(np.abs(M))           # library matmul
    assert np.max(np.abs(b.subspace(C, C) * b.volume - b.overlap(C, C))) <= 1e-13    # overlap = Omega * subspace
    HC = b.apply_H(inp["Vloc"], inp["P"], inp["D"], C)
    Hs = b.subspace(C, HC)
    assert np.max(np.abs(Hs - Hs.conj().T)) <= 1e-12 * np.max(np.abs(Hs))            # Hermitian H => Hermitian C^+ H C
    # Rayleigh quotient of a plane wave under constant V0: (ke[n] + V0) Omega
    e = np.zeros((1, b.nG), dtype=np.complex128)
    e[0, 11] = 1.0
    V0 = 0.37
    Vc = np.full(b.shape, V0 * b.volume / b.N)
    assert abs(b.subspace(e, b.apply_H(Vc, None, None, e))[0, 0] - (b.ke[11] + V0) * b.volume) <= 1e-12 * b.volume


# ------------------------------------------------------------------------------------------ SURVEY 8(f) rank 3
# Listing 1 of the paper: hessian(phi) = (-1/4 pi) divergence(J(epsilon * I(gradient(phi))))

def _q_cart(b, R, k):
    """Cartesian q = 2 pi R^-T (m + k), computed here with numpy (not by the oracle)."""
    return (b.iG.astype(np.float64) + np.asarray(k, dtype=np.float64)) @ (2 * np.pi * np.linalg.inv(R))


def test_gradient_divergence_closed_forms_and_finite_differences(ref):
    rng = np.random.default_rng(71)
    R, k = _skew_lattice(), [0.0, 0.0, 0.0]
    b = ref.RefBasis(R, k, 5.0, (10, 12, 9))
    q = _q_cart(b, R, k)
    phi = _rand_c(rng, 2, b.nG)
    g = b.gradient(phi)
    assert g.shape == (3, 2, b.nG)
    for d in range(3):
        assert np.max(np.abs(g[d] - 1j * q[None, :, d] * phi)) <= 1e-13 * np.max(np.abs(g))
    # div grad = -|q|^2 = -2 ke = L / Omega
    lap = b.divergence(g)
    assert np.max(np.abs(lap - (-2.0 * b.ke)[None, :] * phi)) <= 1e-12 * np.max(np.abs(lap))
    assert np.max(np.abs(lap * b.volume - b.apply_L(phi))) <= 1e-12 * np.max(np.abs(lap)) * b.volume
    # real-space meaning: I(gradient(phi))_d is the Cartesian derivative of f(r) = sum_n phi_n exp(i q_n . r)
    # (central differences of the explicitly evaluated sum at three grid points; r_j = R (j / S))
    S = np.asarray(b.shape, dtype=np.float64)
    Ig = b.apply_I(g.reshape(6, b.nG)).reshape((3, 2) + b.shape)

    def f(r):
        return (phi[0] * np.exp(1j * (q @ r))).sum()

    h = 1e-5
    for j in [(0, 0, 0), (3, 7, 2), (9, 11, 8)]:
        r = R @ (np.asarray(j) / S)
        for d in range(3):
            e = np.zeros(3)
            e[d] = h
            fd = (f(r + e) - f(r - e)) / (2 * h)
            assert abs(Ig[d, 0][j] - fd) <= 1e-6 * max(1.0, abs(fd))


def test_pcm_hessian_vs_explicit_matrices_constant_epsilon_and_hermiticity(ref):
    rng = np.random.default_rng(73)
    R, k = _skew_lattice(), [0.0, 0.0, 0.0]
    b = ref.RefBasis(R, k, 4.0, (8, 9, 8))
    q = _q_cart(b, R, k)
    eps = 1.0 + 78.0 * rng.random(b.shape)                   # an inhomogeneous dielectric between 1 and 79
    phi = _rand_c(rng, 3, b.nG)
    got = b.pcm_hessian(eps, phi)
    # brute force from the explicit N x nG matrix of I: (-1/4pi) sum_d Dg_d (1/N) I^H diag(eps) I Dg_d
    Im = _brute_I_matrix(b)
    K = (Im.conj().T * eps.reshape(-1)[None, :]) @ Im / b.N
    want = np.zeros_like(phi)
    for d in range(3):
        Dg = 1j * q[:, d]
        want += (Dg[None, :] * ((K @ (Dg[None, :] * phi).T).T))
    want *= -1.0 / (4 * np.pi)
    assert np.max(np.abs(got - want)) <= 1e-11 * np.max(np.abs(want))
    # constant epsilon: J I = 1  =>  hessian = (eps0 / 4 pi) |q|^2 phi   (eq. (1) of the paper with constant epsilon)
    e0 = 78.4
    got0 = b.pcm_hessian(np.full(b.shape, e0), phi)
    assert np.max(np.abs(got0 - (e0 / (4 * np.pi)) * (2.0 * b.ke)[None, :] * phi)) <= 1e-12 * np.max(np.abs(got0))
    # Hermitian (and positive) for real positive epsilon
    a_, b_ = phi[0], phi[1]
    Ha, Hb = got[0], got[1]
    assert abs(np.vdot(a_, Hb) - np.conj(np.vdot(b_, Ha))) <= 1e-12 * np.linalg.norm(a_) * np.linalg.norm(Hb)
    assert np.real(np.vdot(a_, Ha)) > 0


# ------------------------------------------------------------------------------------------ ultrasoft (8(f) rank 2)

def _blocks(rng, natoms, nblk, psd=False):
    A = _rand_c(rng, natoms, nblk, nblk)
    if psd:
        return A @ A.conj().transpose(0, 2, 1)
    return A + A.conj().transpose(0, 2, 1)


def _block_diag(Q):
    na, n, _ = Q.shape
    out = np.zeros((na * n, na * n), complex)
    for a in range(na):
        out[a * n:(a + 1) * n, a * n:(a + 1) * n] = Q[a]
    return out


def test_block_diagonal_D_vs_dense_matrix(ref):
    """D_mode = nblk (per-atom Hermitian blocks, reading 24): P D P^+ against the dense nG x nG matrix built
    from the explicitly assembled block-diagonal D; a wrong block offset, a transposed block or coupling across atoms
    fails.  Blocks of one atom's 4 projectors, and 2-projector blocks (8 = 4 x 2)."""
    cfg = 101
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    assert b.nG <= 400
    inp = workloads.make_inputs(cfg, b.iG)
    P, C = inp["P"], inp["C"]
    Pm = P.T
    rng = np.random.default_rng(61)
    for nblk in (4, 2):
        Db = _blocks(rng, P.shape[0] // nblk, nblk)
        want = C @ (Pm @ _block_diag(Db) @ Pm.conj().T).T
        got = b.apply_Vnl(P, Db, C)
        assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))
        # same operator through the dense mode
        assert np.max(np.abs(got - b.apply_Vnl(P, _block_diag(Db), C))) <= 1e-12 * np.max(np.abs(want))
    # blocks that are diagonal reduce to the real-diagonal mode
    d = inp["D"]
    Dd = np.zeros((P.shape[0] // 4, 4, 4), complex)
    for a in range(Dd.shape[0]):
        Dd[a] = np.diag(d[4 * a:4 * a + 4])
    assert np.max(np.abs(b.apply_Vnl(P, Dd, C) - b.apply_Vnl(P, d, C))) <= 1e-13 * np.max(np.abs(C))
    # H with block D = sum of its terms
    V = inp["Vloc"]
    Db = _blocks(rng, P.shape[0] // 4, 4)
    assert np.allclose(b.apply_H(V, P, Db, C), b.apply_H(V, None, None, C) + b.apply_Vnl(P, Db, C), rtol=1e-13, atol=1e-16)


def test_ultrasoft_overlap_operator_vs_dense_matrix(ref):
    """O_us = Omega (1 + P Q P^+) (PAPER.md:95 ultrasoft pseudopotentials; reading 24) against the dense
    nG x nG matrix; Hermitian; positive definite for PSD Q; reduces to Omega at Q = 0 and at np = 0; the generalised
    overlap M = C1^+ O_us C2 against numpy; all three Q layouts."""
    cfg = 101
    R, kpts, Ecut, S = workloads.lattice(cfg)
    b = ref.RefBasis(R, kpts[0], Ecut, S)
    assert b.nG <= 400
    inp = workloads.make_inputs(cfg, b.iG)
    P, C = inp["P"], inp["C"]
    Pm = P.T
    rng = np.random.default_rng(67)
    C2 = _rand_c(rng, 3, b.nG)
    Qb = _blocks(rng, P.shape[0] // 4, 4, psd=True)
    Qdense = _rand_c(rng, P.shape[0], P.shape[0]); Qdense = Qdense + Qdense.conj().T
    qdiag = rng.uniform(0.1, 1.0, P.shape[0])
    for Q, Qfull in ((Qb, _block_diag(Qb)), (Qdense, Qdense), (qdiag, np.diag(qdiag))):
        Ous = b.volume * (np.eye(b.nG) + Pm @ Qfull @ Pm.conj().T)
        assert np.max(np.abs(Ous - Ous.conj().T)) <= 1e-12 * np.max(np.abs(Ous))
        got = b.apply_O_us(P, Q, C)
        want = C @ Ous.T
        assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))
        M = b.overlap_us(P, Q, C, C2)
        wantM = C.conj() @ Ous @ C2.T
        assert M.shape == (C.shape[0], 3)
        assert np.max(np.abs(M - wantM)) <= 1e-12 * np.max(np.abs(wantM))
        # Hermitian: M(C1, C2) = M(C2, C1)^+
        assert np.max(np.abs(b.overlap_us(P, Q, C2, C) - M.conj().T)) <= 1e-12 * np.max(np.abs(M))
    # PSD Q: every Rayleigh quotient of O_us is >= Omega |c|^2
    Mself = b.overlap_us(P, Qb, C2, C2)
    assert np.all(np.linalg.eigvalsh((Mself + Mself.conj().T) / 2) > 0)
    for c in C2:
        assert np.vdot(c, b.apply_O_us(P, Qb, c[None])[0]).real >= b.volume * np.vdot(c, c).real * (1 - 1e-12)
    # Q = 0 and no projectors: the norm-conserving O = Omega
    assert np.max(np.abs(b.apply_O_us(P, np.zeros(P.shape[0]), C) - b.apply_O(C))) == 0.0
    assert np.max(np.abs(b.apply_O_us(P[:0], np.zeros(0), C) - b.apply_O(C))) == 0.0
    assert np.max(np.abs(b.overlap_us(P, np.zeros(P.shape[0]), C, C2) - b.overlap(C, C2))) <= 1e-13 * b.volume
    # rank one: O_us c = Omega (c + q p (p^+ c))
    p, q = P[:1], np.array([0.3])
    want = b.volume * np.stack([c + q[0] * p[0] * np.vdot(p[0], c) for c in C])
    assert np.max(np.abs(b.apply_O_us(p, q, C) - want)) <= 1e-13 * np.max(np.abs(want))


# ------------------------------------------------------------------------------------------ real fields (8(f) rank 3)

def test_pcm_hessian_real_fields_half_sphere(ref):
    """Real-field variant (epsilon, phi, rho are real ScalarFields): half-sphere storage of a
    Hermitian-symmetric spectrum.  Pins: the canonical order is inversion symmetric with the origin in the middle; the
    Hermitian extension of the stored half IS a real field (I gives zero imaginary part); the complex operator maps
    it to a Hermitian-symmetric spectrum whose stored half is the real-variant result; for constant epsilon the closed
    form (eps0 / 4 pi) |q|^2 phi; k != 0 is refused."""
    R = _skew_lattice()
    S = (8, 9, 10)
    b = ref.RefBasis(R, [0.0, 0.0, 0.0], 6.0, S)
    nG, n0 = b.nG, (b.nG - 1) // 2
    assert nG % 2 == 1 and np.all(b.iG[n0] == 0)
    assert np.array_equal(b.iG[::-1], -b.iG)
    rng = np.random.default_rng(83)
    nb = 3
    ph = _rand_c(rng, nb, n0 + 1)
    ph[:, 0] = ph[:, 0].real + 0.77j                      # imaginary part of G = 0 must be ignored
    full = np.empty((nb, nG), complex)
    full[:, n0:] = ph
    full[:, n0] = ph[:, 0].real
    full[:, :n0] = ph[:, :0:-1].conj()
    psi = b.apply_I(full)
    assert np.max(np.abs(psi.imag)) <= 1e-12 * np.max(np.abs(psi.real))          # a real field
    eps = 1.0 + 5.0 * rng.random(S)
    want_full = b.pcm_hessian(eps, full)
    assert np.max(np.abs(want_full[:, ::-1].conj() - want_full)) <= 1e-12 * np.max(np.abs(want_full))   # stays Hermitian
    got = b.pcm_hessian_real(eps, ph)
    assert got.shape == ph.shape
    assert np.max(np.abs(got - want_full[:, n0:])) <= 1e-13 * np.max(np.abs(want_full))
    e0 = 3.25
    got0 = b.pcm_hessian_real(np.full(S, e0), ph)
    closed = (e0 / (4 * np.pi)) * (2.0 * b.ke[n0:])[None, :] * full[:, n0:]
    assert np.max(np.abs(got0 - closed)) <= 1e-12 * np.max(np.abs(closed))
    bk = ref.RefBasis(R, [0.25, 0.0, 0.0], 6.0, S)
    with pytest.raises(ref.RefError):
        bk.pcm_hessian_real(eps, np.zeros((1, (bk.nG + 1) // 2), complex))
