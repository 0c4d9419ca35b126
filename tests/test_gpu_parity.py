"""GPU parity: every exported call of libjdft_b200 (through the C ABI / ctypes binding) against the CPU oracle on
the same seeded inputs, element by element.  Acceptance (BASELINE.json north_star; reading 18):
per-band relative L2 error <= 1e-10 in fp64; index maps bit-exact.
"""
import numpy as np
import pytest
import torch

import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-10


def rel_err_per_band(got, want):
    got = np.asarray(got).reshape(got.shape[0], -1)
    want = np.asarray(want).reshape(want.shape[0], -1)
    num = np.linalg.norm(got - want, axis=1)
    den = np.linalg.norm(want, axis=1)
    den = np.where(den == 0, 1.0, den)
    return float(np.max(num / den))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Case:
    """One (config, k-point): oracle basis + GPU basis + seeded inputs (nb bands)."""

    def __init__(self, ref, jd, cfg_id, ik=0, nb=None, batch=None):
        R, kpts, Ecut, S = workloads.lattice(cfg_id)
        self.rb = ref.RefBasis(R, kpts[ik], Ecut, S)
        self.gb = jd.jdft_basis_create(R, kpts[ik], Ecut, S)
        inp = workloads.make_inputs(cfg_id, self.rb.iG, ik=ik, nb=nb)
        self.C, self.V, self.P, self.D = inp["C"], inp["Vloc"], inp["P"], inp["D"]
        self.nb = self.C.shape[0]
        jd.jdft_alloc_workspace(self.gb, batch if batch else min(self.nb, 8), max(self.nb, self.P.shape[0]))


SMALL = [101, 102, 103, 104, 105, 1]


@pytest.fixture(scope="module", params=SMALL)
def case(request, ref, jd):
    return Case(ref, jd, request.param)


# ------------------------------------------------------------------------------------------ basis (bit-exact)

@pytest.mark.parametrize("cfg_id,ik", [(c, 0) for c in SMALL] + [(103, 1), (2, 0), (3, 0), (4, 0), (4, 1), (4, 2), (4, 3), (5, 0)])
def test_basis_bit_exact(ref, jd, cfg_id, ik):
    R, kpts, Ecut, S = workloads.lattice(cfg_id)
    rb = ref.RefBasis(R, kpts[ik], Ecut, S)
    gb = jd.jdft_basis_create(R, kpts[ik], Ecut, S)
    iG, index, ke = jd.jdft_basis_export(gb)
    assert gb.nG == rb.nG and gb.N == rb.N
    assert np.array_equal(iG, rb.iG)
    assert np.array_equal(index, rb.index)
    assert np.max(np.abs(ke - rb.ke)) <= 1e-14 * np.max(rb.ke)
    assert abs(gb.volume - rb.volume) <= 1e-14 * rb.volume


def test_basis_errors(jd):
    R = np.diag([10.0, 10.0, 10.0])
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_basis_create(R, [0, 0, 0], 10.0, (14, 32, 32))     # 14 = 2 * 7
    assert e.value.code == jd.JDFT_EBOX
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_basis_create(R, [0, 0, 0], 10.0, (8, 32, 32))      # sphere spans -7..7 > 8
    assert e.value.code == jd.JDFT_EBOX
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_basis_create(np.zeros((3, 3)), [0, 0, 0], 10.0, (32, 32, 32))
    assert e.value.code == jd.JDFT_EINVAL
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_basis_create(R, [0, 0, 0], -1.0, (32, 32, 32))
    assert e.value.code == jd.JDFT_EINVAL


def test_workspace_errors(ref, jd):
    R, kpts, Ecut, S = workloads.lattice(101)
    gb = jd.jdft_basis_create(R, kpts[0], Ecut, S)
    C = torch.zeros((2, gb.nG), dtype=torch.complex128, device="cuda")
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_apply_I(gb, C)
    assert e.value.code == jd.JDFT_EWORKSPACE
    jd.jdft_set_workspace(gb, torch.empty(64, dtype=torch.uint8, device="cuda"))
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_apply_I(gb, C)
    assert e.value.code == jd.JDFT_EWORKSPACE
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_set_option(gb, "no_such_option", 1)
    assert e.value.code == jd.JDFT_EINVAL


# ------------------------------------------------------------------------------------------ operators

def test_apply_I(case, jd):
    want = case.rb.apply_I(case.C)
    got = jd.jdft_apply_I(case.gb, dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL


def test_apply_Idag_and_J(case, jd):
    rng = np.random.default_rng(5)
    nb = min(case.nb, 6)
    psi = rng.standard_normal((nb,) + case.rb.shape) + 1j * rng.standard_normal((nb,) + case.rb.shape)
    want = case.rb.apply_Idag(psi)
    got = jd.jdft_apply_Idag(case.gb, dev(psi)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL
    wantJ = case.rb.apply_J(psi)
    gotJ = jd.jdft_apply_J(case.gb, dev(psi)).cpu().numpy()
    assert rel_err_per_band(gotJ, wantJ) <= TOL


def test_apply_L_O(case, jd):
    C = dev(case.C)
    assert rel_err_per_band(jd.jdft_apply_L(case.gb, C).cpu().numpy(), case.rb.apply_L(case.C)) <= 1e-14
    assert rel_err_per_band(jd.jdft_apply_O(case.gb, C).cpu().numpy(), case.rb.apply_O(case.C)) <= 1e-14
    # in place
    C2 = C.clone()
    jd.jdft_apply_L(case.gb, C2, C2)
    assert rel_err_per_band(C2.cpu().numpy(), case.rb.apply_L(case.C)) <= 1e-14


def test_project(case, jd):
    want = case.rb.project(case.P, case.C)
    got = jd.jdft_project(case.gb, dev(case.P), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL


def test_apply_Vnl_diag(case, jd):
    want = case.rb.apply_Vnl(case.P, case.D, case.C)
    got = jd.jdft_apply_Vnl(case.gb, dev(case.P), dev(case.D), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL
    # accumulate into an existing array
    base = np.ascontiguousarray(case.C[::-1]) * 0.37
    out = dev(base)
    jd.jdft_apply_Vnl(case.gb, dev(case.P), dev(case.D), dev(case.C), out, accumulate=True)
    assert rel_err_per_band(out.cpu().numpy(), base + want) <= TOL


def test_apply_Vnl_dense_D(case, jd):
    rng = np.random.default_rng(11)
    n = case.P.shape[0]
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    D = (A + A.conj().T) / 2
    want = case.rb.apply_Vnl(case.P, D, case.C)
    got = jd.jdft_apply_Vnl(case.gb, dev(case.P), dev(D), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL


def test_apply_H_full(case, jd):
    want = case.rb.apply_H(case.V, case.P, case.D, case.C)
    got = jd.jdft_apply_H(case.gb, dev(case.V.reshape(-1)), dev(case.P), dev(case.D), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL


def test_apply_H_local_only(case, jd):
    want = case.rb.apply_H(case.V, None, None, case.C)
    got = jd.jdft_apply_H(case.gb, dev(case.V.reshape(-1)), None, None, dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL


def test_apply_H_zero_V(case, jd):
    V0 = np.zeros_like(case.V)
    want = case.rb.apply_H(V0, case.P, case.D, case.C)
    got = jd.jdft_apply_H(case.gb, dev(V0.reshape(-1)), dev(case.P), dev(case.D), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL


def test_overlap(case, jd):
    rng = np.random.default_rng(3)
    C2 = case.C[: max(1, case.nb // 2)] + 0.1 * (rng.standard_normal((max(1, case.nb // 2), case.rb.nG)) + 0j)
    want = case.rb.overlap(case.C, C2)                      # [nb1, nb2]
    got = jd.jdft_overlap(case.gb, dev(case.C), dev(C2)).cpu().numpy()
    assert got.shape == want.shape
    assert rel_err_per_band(got.T, want.T) <= TOL           # per column of M


@pytest.mark.parametrize("nb", [64, 65, 130, 200])
def test_overlap_hermitian_triangle_path(ref, jd, nb):
    """jdft_overlap(C, C) / jdft_subspace(C, C) with the SAME array on both sides compute the lower-triangle tiles only
    and mirror them; NON-orthonormal bands make every off-diagonal entry O(1), so a wrong mirror index or conjugation
    sign fails.  nb straddles one, two, three and four 64-wide tiles with ragged tails."""
    R, kpts, Ecut, S = workloads.lattice(104)
    rb = ref.RefBasis(R, kpts[0], Ecut, S)
    gb = jd.jdft_basis_create(R, kpts[0], Ecut, S)
    jd.jdft_alloc_workspace(gb, 1, nb)
    C = workloads.make_bands(104, rb.nG, nb=nb, orthonormalise=False)
    C = np.ascontiguousarray(C * (1.0 + np.arange(nb) % 5)[:, None] * np.exp(0.3j * np.arange(nb))[:, None])
    dC = dev(C)
    want = rb.overlap(C, C)
    got = jd.jdft_overlap(gb, dC, dC).cpu().numpy()
    assert rel_err_per_band(got.T, want.T) <= TOL
    assert np.max(np.abs(got - got.conj().T)) <= 1e-13 * np.max(np.abs(got))
    gots = jd.jdft_subspace(gb, dC, dC).cpu().numpy()
    assert rel_err_per_band(gots.T, rb.subspace(C, C).T) <= TOL
    # distinct arrays with equal contents take the full (non-triangle) path: same result
    got2 = jd.jdft_overlap(gb, dC, dC.clone()).cpu().numpy()
    assert rel_err_per_band(got2.T, want.T) <= TOL


def test_host_variants(case, jd):
    want = case.rb.apply_H(case.V, case.P, case.D, case.C)
    HC = torch.empty(case.C.shape, dtype=torch.complex128).pin_memory()
    jd.jdft_apply_H_host(case.gb, torch.from_numpy(case.V.reshape(-1).copy()), torch.from_numpy(case.P),
                         torch.from_numpy(case.D), torch.from_numpy(case.C), HC)
    assert rel_err_per_band(HC.numpy(), want) <= TOL
    M = torch.empty((case.nb, case.nb), dtype=torch.complex128)
    got = jd.jdft_overlap_host(case.gb, torch.from_numpy(case.C), torch.from_numpy(case.C), M).numpy()
    assert rel_err_per_band(got.T, case.rb.overlap(case.C, case.C).T) <= TOL


def test_host_pipeline_chunks_and_resident_operators(ref, jd):
    """jdft_apply_H_host pipelines band chunks (64 bands by default) over three streams; 300 bands of a small box span five
    chunks with a ragged last one.  jdft_host_set_operators + jdft_apply_H_host_resident give the same result; a dense and a
    block-diagonal D go through the same path; without a caller workspace the library allocates its own."""
    c = Case(ref, jd, 101, nb=300)
    want = c.rb.apply_H(c.V, c.P, c.D, c.C)
    Vt, Pt, Ct = torch.from_numpy(c.V.reshape(-1).copy()), torch.from_numpy(c.P), torch.from_numpy(c.C)
    for pinned in (False, True):
        HC = torch.empty(c.C.shape, dtype=torch.complex128)
        if pinned:
            HC = HC.pin_memory()
        jd.jdft_apply_H_host(c.gb, Vt, Pt, torch.from_numpy(c.D), Ct, HC)
        assert rel_err_per_band(HC.numpy(), want) <= TOL
    jd.jdft_host_set_operators(c.gb, Vt, Pt, torch.from_numpy(c.D))
    HC2 = torch.empty(c.C.shape, dtype=torch.complex128).pin_memory()
    jd.jdft_apply_H_host_resident(c.gb, Ct, HC2)
    assert rel_err_per_band(HC2.numpy(), want) <= TOL
    # the overlap of the block that call left on the device (no second upload)
    Mh = torch.empty((c.nb, c.nb), dtype=torch.complex128).pin_memory()
    gotM = jd.jdft_overlap_host_resident(c.gb, Mh).numpy()
    assert rel_err_per_band(gotM.T, c.rb.overlap(c.C, c.C).T) <= TOL
    with pytest.raises(jd.JdftError):                       # a different band count is refused
        jd.jdft_overlap_host_resident(c.gb, torch.empty((c.nb - 1, c.nb - 1), dtype=torch.complex128))
    rng = np.random.default_rng(3)
    n = c.P.shape[0]
    A = rng.standard_normal((n // 4, 4, 4)) + 1j * rng.standard_normal((n // 4, 4, 4))
    Db = np.ascontiguousarray(A + A.conj().transpose(0, 2, 1))
    jd.jdft_set_workspace(c.gb, None)                       # library-owned workspace
    jd.jdft_apply_H_host(c.gb, Vt, Pt, torch.from_numpy(Db), Ct, HC2)
    assert rel_err_per_band(HC2.numpy(), c.rb.apply_H(c.V, c.P, Db, c.C)) <= TOL
    with pytest.raises(jd.JdftError):                       # apply_H_host replaced the resident operators
        jd.jdft_apply_H_host_resident(c.gb, Ct, HC2)
    # no projectors
    jd.jdft_host_set_operators(c.gb, Vt, None, None)
    jd.jdft_apply_H_host_resident(c.gb, Ct, HC2)
    assert rel_err_per_band(HC2.numpy(), c.rb.apply_H(c.V, None, None, c.C)) <= TOL


# ------------------------------------------------------------------------------------------ GPU-side properties

def test_generic_fft_path_matches(ref, jd):
    """Lengths with specialised kernels (32, 64) also run on the runtime-radix kernels; both must match the oracle."""
    for cfg_id in (1, 104):
        c = Case(ref, jd, cfg_id, nb=4)
        want = c.rb.apply_H(c.V, c.P, c.D, c.C)
        args = (dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C))
        a = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
        jd.jdft_set_option(c.gb, "force_generic_fft", 1)
        b = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
        assert rel_err_per_band(a, want) <= TOL and rel_err_per_band(b, want) <= TOL
        assert rel_err_per_band(a, b) <= 1e-13


def test_band_batch_independence(ref, jd):
    c = Case(ref, jd, 102)
    args = (dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C))
    outs = []
    for batch in (1, 3, 7, 19):
        jd.jdft_set_option(c.gb, "band_batch", batch)
        outs.append(jd.jdft_apply_H(c.gb, *args).cpu().numpy())
    for o in outs[1:]:
        assert rel_err_per_band(o, outs[0]) <= 1e-13


def test_gpu_J_I_identity_and_hermiticity(case, jd):
    C = dev(case.C)
    back = jd.jdft_apply_J(case.gb, jd.jdft_apply_I(case.gb, C)).cpu().numpy()
    assert rel_err_per_band(back, case.C) <= 1e-13
    rng = np.random.default_rng(9)
    a = rng.standard_normal((1, case.rb.nG)) + 1j * rng.standard_normal((1, case.rb.nG))
    b = rng.standard_normal((1, case.rb.nG)) + 1j * rng.standard_normal((1, case.rb.nG))
    args = (dev(case.V.reshape(-1)), dev(case.P), dev(case.D))
    Ha = jd.jdft_apply_H(case.gb, *args, dev(a)).cpu().numpy()
    Hb = jd.jdft_apply_H(case.gb, *args, dev(b)).cpu().numpy()
    lhs = np.vdot(a, Hb)
    rhs = np.conj(np.vdot(b, Ha))
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(a) * np.linalg.norm(Hb)


def test_empty_inputs(case, jd):
    C0 = torch.empty((0, case.gb.nG), dtype=torch.complex128, device="cuda")
    assert jd.jdft_apply_H(case.gb, dev(case.V.reshape(-1)), dev(case.P), dev(case.D), C0).shape[0] == 0
    assert jd.jdft_apply_L(case.gb, C0).shape[0] == 0
    # no projectors: Vnl writes zeros
    out = jd.jdft_apply_Vnl(case.gb, None, None, dev(case.C))
    assert float(out.abs().max()) == 0.0


def test_launch_counter(case, jd):
    jd.jdft_launch_count(reset=True)
    jd.jdft_apply_H(case.gb, dev(case.V.reshape(-1)), dev(case.P), dev(case.D), dev(case.C))
    assert jd.jdft_launch_count() >= 8


def test_overlap_gemm_option_matches(ref, jd):
    """apply_H with the projection GEMM forked onto the side stream gives the same result (and matches the oracle)."""
    for D_dense in (False, True):
        c = Case(ref, jd, 102)
        D = c.D
        if D_dense:
            rng = np.random.default_rng(23)
            n = c.P.shape[0]
            A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
            D = (A + A.conj().T) / 2
        want = c.rb.apply_H(c.V, c.P, D, c.C)
        args = (dev(c.V.reshape(-1)), dev(c.P), dev(D), dev(c.C))
        a = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
        jd.jdft_set_option(c.gb, "overlap_gemm", 1)
        b = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
        assert rel_err_per_band(a, want) <= TOL and rel_err_per_band(b, want) <= TOL
        assert rel_err_per_band(a, b) <= 1e-13


# ------------------------------------------------------------------------------------------ SURVEY 8(f) rank 1

def test_subspace(case, jd):
    rng = np.random.default_rng(31)
    X = rng.standard_normal((3, case.rb.nG)) + 1j * rng.standard_normal((3, case.rb.nG))
    want = case.rb.subspace(case.C, X)
    got = jd.jdft_subspace(case.gb, dev(case.C), dev(X)).cpu().numpy()
    assert got.shape == want.shape
    assert rel_err_per_band(got.T, want.T) <= TOL
    # C^+ (H C) from the GPU's own H C is Hermitian
    HC = jd.jdft_apply_H(case.gb, dev(case.V.reshape(-1)), dev(case.P), dev(case.D), dev(case.C))
    Hs = jd.jdft_subspace(case.gb, dev(case.C), HC).cpu().numpy()
    assert np.max(np.abs(Hs - Hs.conj().T)) <= 1e-12 * np.max(np.abs(Hs))


def test_density(case, jd):
    rng = np.random.default_rng(37)
    f = rng.uniform(0.0, 2.0, case.nb)
    want = case.rb.density(case.C, f)
    got = jd.jdft_density(case.gb, dev(case.C), dev(f)).cpu().numpy()
    assert np.linalg.norm(got - want) <= TOL * np.linalg.norm(want)
    assert got.min() >= 0.0
    # accumulate into an existing array; batches of 1 and 3 bands give the same sum to rounding
    base = rng.uniform(0.0, 1.0, case.rb.shape)
    n = dev(base)
    jd.jdft_density(case.gb, dev(case.C), dev(f), n, accumulate=True)
    assert np.linalg.norm(n.cpu().numpy() - (base + want)) <= TOL * np.linalg.norm(base + want)
    for batch in (1, 3):
        jd.jdft_set_option(case.gb, "band_batch", batch)
        g2 = jd.jdft_density(case.gb, dev(case.C), dev(f)).cpu().numpy()
        assert np.linalg.norm(g2 - got) <= 1e-13 * np.linalg.norm(got)
    jd.jdft_set_option(case.gb, "band_batch", 0)
    # no bands: zeros
    C0 = torch.empty((0, case.gb.nG), dtype=torch.complex128, device="cuda")
    f0 = torch.empty((0,), dtype=torch.float64, device="cuda")
    assert float(jd.jdft_density(case.gb, C0, f0).abs().max()) == 0.0


# ------------------------------------------------------------------------------------------ general lattices

@pytest.mark.parametrize("S,k,Ecut", [((24, 20, 18), (0.2, -0.3, 0.1), 5.0), ((32, 27, 30), (0.0, 0.0, 0.0), 7.0),
                                      ((16, 16, 50), (0.5, 0.5, 0.25), 4.0)])
def test_skew_lattice_basis_and_H(ref, jd, S, k, Ecut):
    """Non-orthogonal cell (the workload generator only makes orthorhombic ones): index maps bit-exact, H, I, J, density
    against the oracle with random V, P, D."""
    R = np.array([[7.0, 0.9, -0.6], [0.4, 8.0, 1.1], [-0.7, 0.3, 9.0]])
    rb = ref.RefBasis(R, k, Ecut, S)
    gb = jd.jdft_basis_create(R, k, Ecut, S)
    iG, index, ke = jd.jdft_basis_export(gb)
    assert np.array_equal(iG, rb.iG) and np.array_equal(index, rb.index)
    assert np.max(np.abs(ke - rb.ke)) <= 1e-14 * np.max(rb.ke)
    rng = np.random.default_rng(61)
    nb, npj = 7, 5
    C = rng.standard_normal((nb, rb.nG)) + 1j * rng.standard_normal((nb, rb.nG))
    P = rng.standard_normal((npj, rb.nG)) + 1j * rng.standard_normal((npj, rb.nG))
    D = rng.uniform(-1, 1, npj)
    V = rng.standard_normal(S) * (rb.volume / rb.N)
    jd.jdft_alloc_workspace(gb, 4, 8)
    want = rb.apply_H(V, P, D, C)
    got = jd.jdft_apply_H(gb, dev(V.reshape(-1)), dev(P), dev(D), dev(C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL
    psi = jd.jdft_apply_I(gb, dev(C))
    assert rel_err_per_band(psi.cpu().numpy(), rb.apply_I(C)) <= TOL
    assert rel_err_per_band(jd.jdft_apply_J(gb, psi).cpu().numpy(), C) <= 1e-13
    f = rng.uniform(0, 2, nb)
    n_want = rb.density(C, f)
    n_got = jd.jdft_density(gb, dev(C), dev(f)).cpu().numpy()
    assert np.linalg.norm(n_got - n_want) <= TOL * np.linalg.norm(n_want)


# ------------------------------------------------------------------------------------------ SURVEY 8(f) rank 3 (Listing 1)

def test_gradient_divergence(case, jd):
    want = case.rb.gradient(case.C)
    got = jd.jdft_gradient(case.gb, dev(case.C)).cpu().numpy()
    assert got.shape == want.shape
    for d in range(3):
        assert rel_err_per_band(got[d], want[d]) <= 1e-14
    rng = np.random.default_rng(83)
    X = rng.standard_normal(want.shape) + 1j * rng.standard_normal(want.shape)
    assert rel_err_per_band(jd.jdft_divergence(case.gb, dev(X)).cpu().numpy(), case.rb.divergence(X)) <= 1e-14


def test_pcm_hessian(case, jd):
    rng = np.random.default_rng(89)
    eps = 1.0 + 78.0 * rng.random(case.rb.shape)
    nb = min(case.nb, 5)
    phi = np.ascontiguousarray(case.C[:nb])
    want = case.rb.pcm_hessian(eps, phi)
    ws = jd.jdft_workspace_bytes(case.gb, 3 * nb, 0) + 48 * nb * case.gb.nG
    jd.jdft_set_workspace(case.gb, torch.empty(ws, dtype=torch.uint8, device="cuda"))
    got = jd.jdft_pcm_hessian(case.gb, dev(eps.reshape(-1)), dev(phi)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL
    # several band batches inside the call give the same result
    jd.jdft_set_option(case.gb, "band_batch", 2)
    got2 = jd.jdft_pcm_hessian(case.gb, dev(eps.reshape(-1)), dev(phi)).cpu().numpy()
    jd.jdft_set_option(case.gb, "band_batch", 0)
    assert rel_err_per_band(got2, got) <= 1e-13
    # too small a workspace is refused
    jd.jdft_set_workspace(case.gb, torch.empty(48 * nb * case.gb.nG, dtype=torch.uint8, device="cuda"))
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_pcm_hessian(case.gb, dev(eps.reshape(-1)), dev(phi))
    assert e.value.code == jd.JDFT_EWORKSPACE
    jd.jdft_alloc_workspace(case.gb, min(case.nb, 8), max(case.nb, case.P.shape[0]))


# ------------------------------------------------------------------------------------------ every specialised length

@pytest.mark.parametrize("cfg_id", list(range(201, 210)))
def test_specialised_lengths_on_every_axis(ref, jd, cfg_id):
    """48 96 100 120 144 160 192 256 each as the column, row and plane length: H, I, J and the density."""
    c = Case(ref, jd, cfg_id)
    iG, index, _ = jd.jdft_basis_export(c.gb)
    assert np.array_equal(iG, c.rb.iG) and np.array_equal(index, c.rb.index)
    want = c.rb.apply_H(c.V, c.P, c.D, c.C)
    got = jd.jdft_apply_H(c.gb, dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL
    psi = jd.jdft_apply_I(c.gb, dev(c.C))
    assert rel_err_per_band(psi.cpu().numpy(), c.rb.apply_I(c.C)) <= TOL
    assert rel_err_per_band(jd.jdft_apply_J(c.gb, psi).cpu().numpy(), c.C) <= 1e-13
    f = np.array([1.0, 0.5, 2.0])
    n_want = c.rb.density(c.C, f)
    n_got = jd.jdft_density(c.gb, dev(c.C), dev(f)).cpu().numpy()
    assert np.linalg.norm(n_got - n_want) <= TOL * np.linalg.norm(n_want)


# ------------------------------------------------------------------------------------------ SURVEY 8(f) rank 2 (ultrasoft)

def _herm_blocks(rng, natoms, nblk, psd=False, scale=1.0):
    A = rng.standard_normal((natoms, nblk, nblk)) + 1j * rng.standard_normal((natoms, nblk, nblk))
    H = A @ A.conj().transpose(0, 2, 1) if psd else A + A.conj().transpose(0, 2, 1)
    return np.ascontiguousarray(scale * H)


def _nblk(case):
    n = case.P.shape[0]
    return 9 if n % 9 == 0 else 4


def test_block_diagonal_D(case, jd):
    """Per-atom Hermitian D blocks (D_mode = nblk, applied inside the split-K reduction) in apply_Vnl and apply_H
    against the oracle; every small shape (blocks of 4 and 9 projectors), accumulate mode included."""
    rng = np.random.default_rng(71)
    nblk = _nblk(case)
    Db = _herm_blocks(rng, case.P.shape[0] // nblk, nblk)
    want = case.rb.apply_Vnl(case.P, Db, case.C)
    got = jd.jdft_apply_Vnl(case.gb, dev(case.P), dev(Db), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(got, want) <= TOL
    wantH = case.rb.apply_H(case.V, case.P, Db, case.C)
    gotH = jd.jdft_apply_H(case.gb, dev(case.V.reshape(-1)), dev(case.P), dev(Db), dev(case.C)).cpu().numpy()
    assert rel_err_per_band(gotH, wantH) <= TOL
    # the smallest block size that divides the projector count, and ONE block of all projectors (> 16: generic kernel)
    n = case.P.shape[0]
    for nb2 in (min(d for d in range(2, n + 1) if n % d == 0), n):
        D2 = _herm_blocks(rng, case.P.shape[0] // nb2, nb2)
        got = jd.jdft_apply_Vnl(case.gb, dev(case.P), dev(D2), dev(case.C)).cpu().numpy()
        assert rel_err_per_band(got, case.rb.apply_Vnl(case.P, D2, case.C)) <= TOL
    with pytest.raises(jd.JdftError) as e:
        jd._chk(jd._lib.jdft_apply_Vnl(case.gb._h, dev(case.P).data_ptr(), case.P.shape[0], dev(Db).data_ptr(),
                                      case.P.shape[0] + 1, dev(case.C).data_ptr(), case.nb, dev(case.C).data_ptr(), 0, None))
    assert e.value.code == jd.JDFT_EINVAL


def test_ultrasoft_apply_O_us_and_overlap_us(case, jd):
    """O_us C = Omega (C + P Q P^+ C) and M = C1^+ O_us C2 against the oracle for all three Q layouts, plus the
    reduction to the norm-conserving O at np = 0, in-place operation, and Hermiticity / positivity of M for PSD Q."""
    rng = np.random.default_rng(101)
    n = case.P.shape[0]
    nblk = _nblk(case)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    Qs = [_herm_blocks(rng, n // nblk, nblk, psd=True, scale=0.05), 0.05 * (A + A.conj().T), rng.uniform(0.0, 0.3, n)]
    C2 = case.C[: max(1, case.nb // 2)] + 0.1 * (rng.standard_normal((max(1, case.nb // 2), case.rb.nG)) + 0j)
    dP, dC, dC2 = dev(case.P), dev(case.C), dev(C2)
    for Q in Qs:
        got = jd.jdft_apply_O_us(case.gb, dP, dev(Q), dC).cpu().numpy()
        assert rel_err_per_band(got, case.rb.apply_O_us(case.P, Q, case.C)) <= TOL
        M = jd.jdft_overlap_us(case.gb, dP, dev(Q), dC, dC2).cpu().numpy()
        want = case.rb.overlap_us(case.P, Q, case.C, C2)
        assert M.shape == want.shape
        assert rel_err_per_band(M.T, want.T) <= TOL
        Ms = jd.jdft_overlap_us(case.gb, dP, dev(Q), dC, dC).cpu().numpy()     # same array on both sides
        assert rel_err_per_band(Ms.T, case.rb.overlap_us(case.P, Q, case.C, case.C).T) <= TOL
        assert np.max(np.abs(Ms - Ms.conj().T)) <= 1e-12 * np.max(np.abs(Ms))
    Mpsd = jd.jdft_overlap_us(case.gb, dP, dev(Qs[0]), dC, dC).cpu().numpy()
    assert np.all(np.linalg.eigvalsh((Mpsd + Mpsd.conj().T) / 2) > 0)
    # in place
    buf = dC.clone()
    jd.jdft_apply_O_us(case.gb, dP, dev(Qs[0]), buf, buf)
    assert rel_err_per_band(buf.cpu().numpy(), case.rb.apply_O_us(case.P, Qs[0], case.C)) <= TOL
    # no projectors: O_us = O
    got0 = jd.jdft_apply_O_us(case.gb, None, None, dC).cpu().numpy()
    assert rel_err_per_band(got0, case.rb.apply_O(case.C)) <= 1e-14
    M0 = jd.jdft_overlap_us(case.gb, None, None, dC, dC2).cpu().numpy()
    assert rel_err_per_band(M0.T, case.rb.overlap(case.C, C2).T) <= TOL


@pytest.mark.parametrize("tma", [0, 1])
@pytest.mark.parametrize("cfg_id", [210, 211, 212, 213, 214, 215, 216])
def test_planes_pair_kernel_matches(ref, jd, cfg_id, tma):
    """Plane length 72 runs K3 with two pencils per thread (256-bit global accesses); same result as the one-pencil
    kernel and as the oracle; lengths 128 and 80 run the hybrid (pairs in the first and last pass only; also K2/K4 at row
    length 128).  214 and 215 have an odd S2, where the 256-bit variants must step aside for the one-pencil kernels."""
    c = Case(ref, jd, cfg_id)
    jd.jdft_set_option(c.gb, "planes_tma", tma)      # tma = 1: K3 takes the TMA kernel wherever the plane length has one
    want = c.rb.apply_H(c.V, c.P, c.D, c.C)
    args = (dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C))
    a = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
    jd.jdft_set_option(c.gb, "planes_pair", 0)
    b = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
    assert rel_err_per_band(a, want) <= TOL and rel_err_per_band(b, want) <= TOL
    assert rel_err_per_band(a, b) <= 1e-13
    # a workspace that is only 16-byte aligned (all the ABI requires): the 256-bit kernels must step aside
    jd.jdft_set_option(c.gb, "planes_pair", 1)
    ws = torch.empty(jd.jdft_workspace_bytes(c.gb, c.nb, max(c.nb, c.P.shape[0])) + 64, dtype=torch.uint8, device="cuda")
    jd.jdft_set_workspace(c.gb, ws[16:])
    d = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
    assert rel_err_per_band(d, want) <= TOL
    psi = jd.jdft_apply_I(c.gb, dev(c.C))
    assert rel_err_per_band(jd.jdft_apply_J(c.gb, psi).cpu().numpy(), c.C) <= 1e-13


# ------------------------------------------------------------------------------------------ 8(f) rank 4: band shards

@pytest.mark.gpu
@pytest.mark.parametrize("world", [1, 2, 3])
def test_band_shards_compose_on_one_gpu(case, jd, world):
    """The local operations each rank of sharding.py issues (one rank after the other on this one GPU, nothing waits
    on anything): per-shard apply_H rows, the ring schedule's row-shard x column-shard overlap blocks, per-shard
    density partial sums -- assembled, they equal the oracle on the unsharded arrays.  world = 1 goes through
    sharding.py itself (no process group)."""
    from paper_1708_03621_b200 import sharding as sh
    rng = np.random.default_rng(91)
    nb = case.nb
    X = case.C + 0.1 * (rng.standard_normal(case.C.shape) + 1j * rng.standard_normal(case.C.shape))
    f = rng.uniform(0.0, 2.0, nb)
    Cd, Xd, fd = dev(case.C), dev(X), dev(f)
    want_M, want_n = case.rb.overlap(case.C, X), case.rb.density(case.C, f)
    want_H = case.rb.apply_H(case.V, case.P, case.D, case.C)
    if world == 1:
        M = sh.sharded_overlap(case.gb, Cd, Xd, nb).cpu().numpy()
        n = sh.sharded_density(case.gb, Cd, fd).cpu().numpy()
        HC = sh.sharded_apply_H(case.gb, dev(case.V), dev(case.P), dev(case.D), Cd).cpu().numpy()
    else:
        ranges = [sh.shard_range(nb, world, r) for r in range(world)]
        M = np.zeros((nb, nb), dtype=np.complex128)
        n = torch.zeros(case.rb.shape, dtype=torch.float64, device="cuda")
        HC = np.zeros_like(case.C)
        for lo, hi in ranges:                       # "rank" owning bands lo:hi
            if hi == lo:
                continue
            for r0, r1 in ranges:                   # the row shard that is resident at this ring step
                if r1 > r0:
                    M[r0:r1, lo:hi] = jd.jdft_overlap(case.gb, Cd[r0:r1].contiguous(), Xd[lo:hi].contiguous()).cpu().numpy()
            n += jd.jdft_density(case.gb, Cd[lo:hi].contiguous(), fd[lo:hi].contiguous())   # the all-reduce's sum
            HC[lo:hi] = jd.jdft_apply_H(case.gb, dev(case.V), dev(case.P), dev(case.D), Cd[lo:hi].contiguous()).cpu().numpy()
        n = n.cpu().numpy()
    assert rel_err_per_band(M.T, want_M.T) <= TOL
    assert np.linalg.norm(n - want_n) <= TOL * np.linalg.norm(want_n)
    assert rel_err_per_band(HC, want_H) <= TOL


@pytest.mark.parametrize("cfg_id", [103, 101])
def test_bench_shard_step_on_one_gpu(ref, jd, cfg_id):
    """The step `bench.py --shard kb` times, as that mode builds it (bench.shard_inputs + sharding.sharded_step with the
    CUDA binding, one rank = every k-point, all bands): HC of every k-point and its overlap against the oracle.  The
    same step on 2 and 3 gloo ranks with the oracle as the local operation is tests/test_sharding_gloo.py."""
    import bench
    from paper_1708_03621_b200 import sharding as sh
    cfg = workloads.get_config(cfg_id)
    nk, nb = len(cfg["kpoints"]), cfg["nb"]
    lay = sh.KBLayout(nk, nb, 1, 0)

    def make_basis(R, k, Ecut, S):
        gb = jd.jdft_basis_create(R, k, Ecut, S)
        jd.jdft_alloc_workspace(gb, nb, max(nb, 64))
        return gb, jd.jdft_basis_export(gb)[0]

    kdata, V, D = bench.shard_inputs(cfg_id, lay, make_basis, lambda a: torch.from_numpy(a).cuda())
    for d in kdata.values():
        d["HC"] = torch.empty_like(d["C"])
    out = sh.sharded_step(lay, kdata, V, D, group=None, mode="allgather", overlap=True)
    assert sorted(out) == list(range(nk))
    R, kpts, Ecut, S = workloads.lattice(cfg_id)
    for k in range(nk):
        rb = ref.RefBasis(R, kpts[k], Ecut, S)
        inp = workloads.make_inputs(cfg_id, rb.iG, ik=k)
        HC, M = out[k]
        assert HC.data_ptr() == kdata[k]["HC"].data_ptr()                      # written in place, as the bench expects
        assert rel_err_per_band(HC.cpu().numpy(), rb.apply_H(inp["Vloc"], inp["P"], inp["D"], inp["C"])) <= TOL
        assert rel_err_per_band(M.cpu().numpy().T, rb.overlap(inp["C"], inp["C"]).T) <= TOL


@pytest.mark.parametrize("tma", [0, 1])
@pytest.mark.parametrize("cfg_id", [211, 212, 217])
def test_planes_pruned_butterflies_match(ref, jd, cfg_id, tma):
    """K3 hybrid (plane lengths 80, 128): radix-8 first/last butterflies pruned to the sphere's axis-0 extent (inputs /
    outputs 2..5 are empty planes).  211 (|m0| <= 13 of 80) and 212 (|m0| <= 21 of 128) take the pruned kernel, 217
    (|m0| <= 22 of 80, planes 20..22 occupied) must fall back; all equal the unpruned kernel and the oracle."""
    c = Case(ref, jd, cfg_id)
    jd.jdft_set_option(c.gb, "planes_tma", tma)
    m0 = c.rb.iG[:, 0]
    L, R2 = c.rb.shape[0], c.rb.shape[0] // 8
    assert (max(m0.max(), -m0.min()) < 2 * R2) == (cfg_id != 217)
    want = c.rb.apply_H(c.V, c.P, c.D, c.C)
    args = (dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C))
    a = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
    jd.jdft_set_option(c.gb, "planes_prune", 0)
    b = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
    jd.jdft_set_option(c.gb, "planes_prune", 1)
    assert rel_err_per_band(a, want) <= TOL and rel_err_per_band(b, want) <= TOL
    assert rel_err_per_band(a, b) <= 1e-13
    # stand-alone I: its first pass along axis 0 is pruned the same way
    want_psi = c.rb.apply_I(c.C).reshape(c.nb, -1)
    psi1 = jd.jdft_apply_I(c.gb, dev(c.C)).cpu().numpy().reshape(c.nb, -1)
    jd.jdft_set_option(c.gb, "planes_prune", 0)
    psi0 = jd.jdft_apply_I(c.gb, dev(c.C)).cpu().numpy().reshape(c.nb, -1)
    jd.jdft_set_option(c.gb, "planes_prune", 1)
    assert rel_err_per_band(psi1, want_psi) <= TOL and rel_err_per_band(psi0, want_psi) <= TOL


@pytest.mark.parametrize("cfg_id", [216, 209, 204, 104, 3])
def test_cols_direct_matches_staged(ref, jd, cfg_id):
    """K1 / K5 "cols_direct" (first pass reading the sphere, last pass writing it straight from / to global memory) against
    the staged scatter / gather: the arithmetic is the same, so the results are bit-identical; both match the oracle.
    Column lengths 128 (216: k != 0, runs that wrap; config 3 shape at 24 bands: pruned butterflies, K5 on the reversed
    plan), 256, 160, 64; stand-alone I^+ (K5 with no kinetic term) likewise."""
    c = Case(ref, jd, cfg_id, nb=24) if cfg_id == 3 else Case(ref, jd, cfg_id)
    want = c.rb.apply_H(c.V, c.P, c.D, c.C)
    args = (dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C))
    rng = np.random.default_rng(5)
    psi = dev(rng.standard_normal((2,) + tuple(c.rb.shape)) + 1j * rng.standard_normal((2,) + tuple(c.rb.shape)))
    a = jd.jdft_apply_H(c.gb, *args)
    ia = jd.jdft_apply_Idag(c.gb, psi)
    jd.jdft_set_option(c.gb, "cols_direct", 0)
    b = jd.jdft_apply_H(c.gb, *args)
    ib = jd.jdft_apply_Idag(c.gb, psi)
    jd.jdft_set_option(c.gb, "cols_direct", 1)
    assert torch.equal(a, b) and torch.equal(ia, ib)
    assert rel_err_per_band(a.cpu().numpy(), want) <= TOL


# ------------------------------------------------------------------------------------------ 3M complex GEMM scheme

@pytest.mark.parametrize("cfg_id", [102, 103, 104])
def test_gemm_3m_and_4m_schemes_match_the_oracle(ref, jd, cfg_id):
    """The projector GEMMs run the 3M complex-product scheme by default (three DMMAs per tile product, option
    "gemm_3m"); both schemes must meet the tolerance on the nonlocal term ALONE (where a GEMM error cannot hide behind
    the kinetic term), on the projection, and on a distinct-operand overlap."""
    c = Case(ref, jd, cfg_id)
    want = c.rb.apply_Vnl(c.P, c.D, c.C)
    wantB = c.rb.project(c.P, c.C)
    rng = np.random.default_rng(7)
    C2 = np.ascontiguousarray(c.C[::-1] * (1.0 + 0.5j)) + 0.1 * rng.standard_normal(c.C.shape)
    wantM = c.rb.overlap(c.C, C2)
    res = {}
    for m3 in (0, 1, 2):                                      # 2: the 3M kernels with TMA operand staging ("gemm_tma")
        jd.jdft_set_option(c.gb, "gemm_3m", min(m3, 1))
        jd.jdft_set_option(c.gb, "gemm_tma", 1 if m3 == 2 else 0)
        got = jd.jdft_apply_Vnl(c.gb, dev(c.P), dev(c.D), dev(c.C)).cpu().numpy()
        assert rel_err_per_band(got, want) <= TOL
        B = jd.jdft_project(c.gb, dev(c.P), dev(c.C)).cpu().numpy()
        assert rel_err_per_band(B, wantB) <= TOL
        M = jd.jdft_overlap(c.gb, dev(c.C), dev(C2)).cpu().numpy()
        assert rel_err_per_band(M.T, wantM.T) <= TOL
        res[m3] = got
    assert rel_err_per_band(res[0], res[1]) <= 1e-12
    assert rel_err_per_band(res[2], res[1]) <= 1e-13
    # the Hermitian-triangle overlap through the TMA-staged kernel
    Cn = workloads.make_bands(cfg_id, c.rb.nG, nb=130, orthonormalise=False)
    jd.jdft_alloc_workspace(c.gb, 1, 130)
    jd.jdft_set_option(c.gb, "gemm_tma", 1)
    dCn = dev(Cn)
    M = jd.jdft_overlap(c.gb, dCn, dCn).cpu().numpy()
    assert rel_err_per_band(M.T, c.rb.overlap(Cn, Cn).T) <= TOL


# ------------------------------------------------------------------------------------------ K3 through TMA

@pytest.mark.parametrize("cfg_id", [104, 210, 211, 212, 214, 215, 217, 204, 1])
def test_planes_tma_kernel_matches(ref, jd, cfg_id):
    """K3 with tensor-map (TMA) loads / stores and persistent double-buffered CTAs (plane lengths 64, 72, 80, 96, 120, 128)
    against the LSU kernels and the oracle: ragged last i2 tile (S2 = 27, 25, 50: zero-filled on load, clipped on
    store), odd S2, pruned and unpruned butterflies, several band batches (more tiles than resident CTAs or fewer),
    and a workspace that is only 16-byte aligned."""
    c = Case(ref, jd, cfg_id)
    want = c.rb.apply_H(c.V, c.P, c.D, c.C)
    args = (dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C))
    out = {}
    for tma in (1, 0):
        jd.jdft_set_option(c.gb, "planes_tma", tma)
        out[tma] = jd.jdft_apply_H(c.gb, *args).cpu().numpy()
        assert rel_err_per_band(out[tma], want) <= TOL
    assert rel_err_per_band(out[1], out[0]) <= 1e-13
    jd.jdft_set_option(c.gb, "planes_tma", 1)
    for batch in (1, 2):
        jd.jdft_set_option(c.gb, "band_batch", batch)
        assert rel_err_per_band(jd.jdft_apply_H(c.gb, *args).cpu().numpy(), out[1]) <= 1e-13
    jd.jdft_set_option(c.gb, "band_batch", 0)
    ws = torch.empty(jd.jdft_workspace_bytes(c.gb, c.nb, max(c.nb, c.P.shape[0])) + 64, dtype=torch.uint8, device="cuda")
    jd.jdft_set_workspace(c.gb, ws[16:])
    assert rel_err_per_band(jd.jdft_apply_H(c.gb, *args).cpu().numpy(), want) <= TOL
    # Listing 1 rides the same pipeline (epsilon in place of V_loc, 3 nb components)
    rng = np.random.default_rng(5)
    eps = 1.0 + 78.0 * rng.random(c.rb.shape)
    phi = c.C[:2]
    jd.jdft_set_workspace(c.gb, torch.empty(jd.jdft_workspace_bytes(c.gb, 6, 0) + 48 * 2 * c.gb.nG + 4096, dtype=torch.uint8, device="cuda"))
    got = jd.jdft_pcm_hessian(c.gb, dev(eps.reshape(-1)), dev(phi)).cpu().numpy()
    assert rel_err_per_band(got, c.rb.pcm_hessian(eps, phi)) <= TOL


# ------------------------------------------------------------------------------------------ CUDA-graph replay

def test_apply_H_graph_replay(ref, jd):
    """Small calls replay a captured CUDA graph from the third identical call on (option "graph", automatic for
    config 1): results equal the direct launches bit for bit, follow the CONTENTS of the arrays (same pointers, new
    data), a different output pointer gets its own capture, and options / a new workspace drop the captures."""
    c = Case(ref, jd, 1)
    V, P, D, C = dev(c.V.reshape(-1)), dev(c.P), dev(c.D), dev(c.C)
    HC = torch.empty_like(C)
    jd.jdft_set_option(c.gb, "graph", 0)
    jd.jdft_launch_count(reset=True)
    direct = jd.jdft_apply_H(c.gb, V, P, D, C, HC).clone()
    per_call = jd.jdft_launch_count()
    assert per_call >= 8
    jd.jdft_set_option(c.gb, "graph", -1)
    jd.jdft_launch_count(reset=True)
    for _ in range(4):                                       # direct, capture + replay, replay, replay
        HC.zero_()
        jd.jdft_apply_H(c.gb, V, P, D, C, HC)
        assert torch.equal(HC, direct)
    assert jd.jdft_launch_count() == 4 * per_call            # replays count their kernels
    C.mul_(2.0)                                              # same pointer, new contents
    jd.jdft_apply_H(c.gb, V, P, D, C, HC)
    assert torch.equal(HC, 2.0 * direct)
    C.mul_(0.5)
    HC2 = torch.empty_like(C)
    for _ in range(3):
        jd.jdft_apply_H(c.gb, V, P, D, C, HC2)
    assert torch.equal(HC2, direct)
    jd.jdft_set_option(c.gb, "band_batch", 3)                # drops the captures; 3 + 3 + 2 bands now
    for _ in range(3):
        jd.jdft_apply_H(c.gb, V, P, D, C, HC)
    assert rel_err_per_band(HC.cpu().numpy(), direct.cpu().numpy()) <= 1e-13
    assert rel_err_per_band(HC.cpu().numpy(), c.rb.apply_H(c.V, c.P, c.D, c.C)) <= TOL
    # replay on a non-default stream
    st = torch.cuda.Stream()
    jd.jdft_set_option(c.gb, "band_batch", 0)
    with torch.cuda.stream(st):
        for _ in range(3):
            jd.jdft_apply_H(c.gb, V, P, D, C, HC)
    st.synchronize()
    assert torch.equal(HC, direct)


# ------------------------------------------------------------------------------------------ Listing 1 on real fields

@pytest.mark.parametrize("cfg_id,nb", [(101, 1), (102, 2), (104, 5), (1, 3)])
def test_pcm_hessian_real_fields(ref, jd, cfg_id, nb):
    """jdft_pcm_hessian_real (half-sphere storage, two real gradient components per complex transform) against the
    oracle's real-field function and against the GPU's own complex path on the Hermitian extension; odd and even numbers
    of components (3 nb = 3, 6, 15, 9); k != 0 is refused."""
    R, kpts, Ecut, S = workloads.lattice(cfg_id)
    k0 = [0.0, 0.0, 0.0]
    rb = ref.RefBasis(R, k0, Ecut, S)
    gb = jd.jdft_basis_create(R, k0, Ecut, S)
    nG, n0 = rb.nG, (rb.nG - 1) // 2
    rng = np.random.default_rng(211 + cfg_id)
    ph = rng.standard_normal((nb, n0 + 1)) + 1j * rng.standard_normal((nb, n0 + 1))
    eps = 1.0 + 78.0 * rng.random(S)
    jd.jdft_set_workspace(gb, torch.empty(jd.jdft_workspace_bytes(gb, 3 * nb, 0) + 48 * nb * nG + 4096, dtype=torch.uint8, device="cuda"))
    got = jd.jdft_pcm_hessian_real(gb, dev(eps.reshape(-1)), dev(ph)).cpu().numpy()
    want = rb.pcm_hessian_real(eps, ph)
    assert rel_err_per_band(got, want) <= TOL
    full = np.empty((nb, nG), complex)
    full[:, n0:] = ph
    full[:, n0] = ph[:, 0].real
    full[:, :n0] = ph[:, :0:-1].conj()
    gfull = jd.jdft_pcm_hessian(gb, dev(eps.reshape(-1)), dev(full)).cpu().numpy()
    assert rel_err_per_band(got, gfull[:, n0:]) <= 1e-12
    if any(kpts[0] != 0):
        gk = jd.jdft_basis_create(R, kpts[0], Ecut, S)
        jd.jdft_alloc_workspace(gk, 8, 8)
        with pytest.raises(jd.JdftError) as e:
            jd.jdft_pcm_hessian_real(gk, dev(eps.reshape(-1)), torch.zeros((1, (gk.nG + 1) // 2), dtype=torch.complex128, device="cuda"))
        assert e.value.code == jd.JDFT_EINVAL


# ------------------------------------------------------------------------------------------ degenerate cases

@pytest.mark.parametrize("S,L,k,Ecut", [((32, 32, 32), 10.0, (0.0, 0.0, 0.0), 0.1),      # nG = 1: only G = 0
                                        ((32, 32, 32), 10.0, (0.0, 0.0, 0.0), 0.25),     # nG = 7: origin + 6 neighbours
                                        ((8, 8, 8), 10.0, (0.0, 0.0, 0.0), 3.1),         # m = -3..3 on every axis: extent 7 of 8, the collision limit
                                        ((12, 15, 20), 9.0, (0.5, 0.5, 0.5), 1.0)])      # k at the zone corner: asymmetric extents
def test_degenerate_spheres_single_band_single_projector(ref, jd, S, L, k, Ecut):
    """The smallest spheres (one plane wave; the origin and its six neighbours), a sphere that fills the box up to the
    collision limit, one band and one projector: H, Vnl, I / J, overlap, density against the oracle."""
    R = np.diag([L, L, L])
    rb = ref.RefBasis(R, k, Ecut, S)
    gb = jd.jdft_basis_create(R, k, Ecut, S)
    iG, index, _ = jd.jdft_basis_export(gb)
    assert np.array_equal(iG, rb.iG) and np.array_equal(index, rb.index)
    if Ecut == 0.1:
        assert rb.nG == 1
    if Ecut == 0.25:
        assert rb.nG == 7
    rng = np.random.default_rng(int(100 * Ecut) + S[0])
    C = rng.standard_normal((1, rb.nG)) + 1j * rng.standard_normal((1, rb.nG))
    P = rng.standard_normal((1, rb.nG)) + 1j * rng.standard_normal((1, rb.nG))
    D = np.array([0.7])
    V = rng.standard_normal(S) * (rb.volume / rb.N)
    jd.jdft_alloc_workspace(gb, 1, 1)
    args = (dev(V.reshape(-1)), dev(P), dev(D), dev(C))
    assert rel_err_per_band(jd.jdft_apply_H(gb, *args).cpu().numpy(), rb.apply_H(V, P, D, C)) <= TOL
    assert rel_err_per_band(jd.jdft_apply_Vnl(gb, dev(P), dev(D), dev(C)).cpu().numpy(), rb.apply_Vnl(P, D, C)) <= TOL
    psi = jd.jdft_apply_I(gb, dev(C))
    assert rel_err_per_band(psi.cpu().numpy(), rb.apply_I(C)) <= TOL
    assert rel_err_per_band(jd.jdft_apply_J(gb, psi).cpu().numpy(), C) <= 1e-13
    M = jd.jdft_overlap(gb, dev(C), dev(C)).cpu().numpy()
    assert abs(M[0, 0] - rb.overlap(C, C)[0, 0]) <= TOL * abs(M[0, 0])
    n = jd.jdft_density(gb, dev(C), dev(np.array([1.3]))).cpu().numpy()
    want_n = rb.density(C, np.array([1.3]))
    assert np.linalg.norm(n - want_n) <= TOL * np.linalg.norm(want_n)


def test_plane_wave_eigenvalue_on_the_gpu(ref, jd):
    """north_star's closed form directly on the CUDA path: C = e_n, V_loc = (Omega/N) V0, no projectors =>
    HC = (ke[n] + V0) Omega e_n and every other entry is zero to rounding."""
    R, kpts, Ecut, S = workloads.lattice(102)
    gb = jd.jdft_basis_create(R, kpts[0], Ecut, S)
    _, _, ke = jd.jdft_basis_export(gb)
    jd.jdft_alloc_workspace(gb, 3, 3)
    V0 = -0.37
    V = torch.full((gb.N,), V0 * gb.volume / gb.N, dtype=torch.float64, device="cuda")
    sel = [0, gb.nG // 3, gb.nG - 1]
    C = torch.zeros((3, gb.nG), dtype=torch.complex128, device="cuda")
    for i, n0 in enumerate(sel):
        C[i, n0] = 1.0 - 0.5j
    HC = jd.jdft_apply_H(gb, V, None, None, C).cpu().numpy()
    for i, n0 in enumerate(sel):
        want = np.zeros(gb.nG, complex)
        want[n0] = (ke[n0] + V0) * gb.volume * (1.0 - 0.5j)
        assert np.max(np.abs(HC[i] - want)) <= 1e-13 * gb.volume * max(1.0, ke[n0])
