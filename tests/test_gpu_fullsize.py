"""GPU parity at BASELINE.json's FULL sizes (configs 2-5, every k-point of config 4) in the launch configuration
bench.py times: all nb bands in one jdft_apply_H call, automatic band batch, the full projector block, workspace sized
as bench.py sizes it.  EVERY band of HC is compared with the oracle (per-band relative L2); I / I^+ / J are compared
with the oracle on real-space blocks that are NOT band-limited; the overlap is compared as a full matrix, also through
the Hermitian-triangle path with non-orthonormal bands; the HOST-buffer path of bench.py's e2e leg likewise.  Tolerance: BASELINE.json north_star, per-band relative
L2 <= 1e-10.  The oracle needs ~2-3 minutes of the box's host threads for the whole module.
"""
import numpy as np
import pytest
import torch

import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-10


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel_rows(got, want):
    """per-row (band / matrix column) relative L2 error, the maximum over rows"""
    got = np.asarray(got).reshape(got.shape[0], -1)
    want = np.asarray(want).reshape(want.shape[0], -1)
    return float(np.max(np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)))


def auto_batch(gb, S, ws_bytes):
    """Bands per FFT batch the library picks on its own (what the workspace holds, at most 256)."""
    per = 16 * (gb.ncol * S[2] + gb.npl * S[1] * S[2])
    return max(1, min(256, ws_bytes // per))


class Full:
    def __init__(self, ref, jd, cfg_id, ik):
        cfg = workloads.get_config(cfg_id)
        R, kpts, Ecut, S = workloads.lattice(cfg_id)
        self.cfg_id, self.ik = cfg_id, ik
        self.S, self.nb = S, cfg["nb"]
        self.rb = ref.RefBasis(R, kpts[ik], Ecut, S)
        self.gb = jd.jdft_basis_create(R, kpts[ik], Ecut, S)
        iG, index, _ = jd.jdft_basis_export(self.gb)
        assert np.array_equal(iG, self.rb.iG) and np.array_equal(index, self.rb.index)     # bit-exact maps
        inp = workloads.make_inputs(cfg_id, iG, ik=ik)
        self.C, self.V, self.P, self.D = inp["C"], inp["Vloc"], inp["P"], inp["D"]
        nproj = self.P.shape[0]
        ws = jd.jdft_alloc_workspace(self.gb, min(self.nb, 256), max(self.nb, nproj))       # as bench.py does
        nbatch = auto_batch(self.gb, S, ws.numel())
        last0 = ((self.nb - 1) // nbatch) * nbatch                                         # first band of the last batch
        # a >= 32-band subset for the term-by-term variants: head, both sides of every batch boundary, tail
        pick = set(range(0, 12)) | set(range(self.nb - 12, self.nb))
        pick |= set(range(max(0, nbatch - 4), min(self.nb, nbatch + 4))) | set(range(max(0, last0 - 4), min(self.nb, last0 + 4)))
        self.subset = sorted(b for b in pick if 0 <= b < self.nb)
        assert len(self.subset) >= 24
        self.dV, self.dP, self.dD, self.dC = dev(self.V.reshape(-1)), dev(self.P), dev(self.D), dev(self.C)


ALL = [(2, 0), (3, 0), (4, 0), (4, 1), (4, 2), (4, 3), (5, 0)]


@pytest.fixture(scope="module", params=ALL, ids=lambda p: "cfg%d_k%d" % p)
def full(request, ref, jd):
    f = Full(ref, jd, *request.param)
    yield f
    del f
    torch.cuda.empty_cache()


def test_full_H_every_band(full, jd):
    """HC of ALL bands (every k-point of config 4 is its own case) against jdft_ref_apply_H, band by band."""
    HC = jd.jdft_apply_H(full.gb, full.dV, full.dP, full.dD, full.dC)
    got = HC.cpu().numpy()
    want = full.rb.apply_H(full.V, full.P, full.D, full.C)
    err = np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)
    assert err.shape == (full.nb,)
    assert float(err.max()) <= TOL, "band %d: %g" % (int(err.argmax()), float(err.max()))
    full.HC, full.want_HC = HC, want


def test_full_H_pruned_butterflies_are_taken_and_agree(full, jd):
    """All five workloads leave planes [S0/4, 3 S0/4) empty, so the pruned radix-8 butterflies run (DESIGN.md
    section 5); every band equals the unpruned kernels' result to rounding."""
    m0 = full.rb.iG[:, 0]
    assert max(m0.max(), -m0.min()) < full.S[0] // 4
    jd.jdft_set_option(full.gb, "planes_prune", 0)
    ref_HC = jd.jdft_apply_H(full.gb, full.dV, full.dP, full.dD, full.dC)
    jd.jdft_set_option(full.gb, "planes_prune", 1)
    HC = full.HC if hasattr(full, "HC") else jd.jdft_apply_H(full.gb, full.dV, full.dP, full.dD, full.dC)
    num = torch.linalg.vector_norm(HC - ref_HC, dim=1)
    den = torch.linalg.vector_norm(ref_HC, dim=1)
    assert float((num / den).max()) <= 1e-13
    del ref_HC


def test_full_H_local_only_and_Vnl_alone(full, jd):
    """The nonlocal term is ~1e-3 of HC in norm, so each term is also compared on its own (>= 24 bands around every
    batch boundary; the GPU call still processes all bands)."""
    Cs = full.C[full.subset]
    got = jd.jdft_apply_H(full.gb, full.dV, None, None, full.dC)[full.subset].cpu().numpy()
    assert rel_rows(got, full.rb.apply_H(full.V, None, None, Cs)) <= TOL
    got = jd.jdft_apply_Vnl(full.gb, full.dP, full.dD, full.dC)[full.subset].cpu().numpy()
    assert rel_rows(got, full.rb.apply_Vnl(full.P, full.D, Cs)) <= TOL
    zeroV = torch.zeros_like(full.dV)
    got = jd.jdft_apply_H(full.gb, zeroV, full.dP, full.dD, full.dC)[full.subset].cpu().numpy()
    assert rel_rows(got, full.rb.apply_H(np.zeros_like(full.V), full.P, full.D, Cs)) <= TOL


def test_full_I_Idag_J_against_oracle(full, jd):
    """I on bands of the block; I^+ and J on DENSE random psi (components outside the sphere, as I^+(V psi) sees)."""
    sel = [0, 1, full.nb - 2, full.nb - 1]
    got = jd.jdft_apply_I(full.gb, dev(full.C[sel])).cpu().numpy()
    want = full.rb.apply_I(full.C[sel])
    assert rel_rows(got, want) <= TOL
    del got, want
    rng = np.random.default_rng(1000 + 10 * full.cfg_id + full.ik)
    psi = rng.standard_normal((4,) + tuple(full.S)) + 1j * rng.standard_normal((4,) + tuple(full.S))
    dpsi = dev(psi)
    assert rel_rows(jd.jdft_apply_Idag(full.gb, dpsi).cpu().numpy(), full.rb.apply_Idag(psi)) <= TOL
    assert rel_rows(jd.jdft_apply_J(full.gb, dpsi).cpu().numpy(), full.rb.apply_J(psi)) <= TOL


def test_full_properties_JI_identity_and_hermiticity(full, jd):
    nb = min(full.nb, 8)                      # the real-space block of 8 bands at 128^3 is 268 MB
    C8 = full.dC[:nb].contiguous()
    back = jd.jdft_apply_J(full.gb, jd.jdft_apply_I(full.gb, C8))
    err = (back - C8).norm(dim=1) / C8.norm(dim=1)
    assert float(err.max()) <= 1e-13
    HC = full.HC if hasattr(full, "HC") else jd.jdft_apply_H(full.gb, full.dV, full.dP, full.dD, full.dC)
    # subspace Hamiltonian C^+ (H C) through the overlap kernel: Hermitian for Hermitian H
    M = jd.jdft_overlap(full.gb, full.dC, HC)
    herm = (M - M.conj().t()).abs().max() / M.abs().max()
    assert float(herm) <= 1e-12


def test_full_overlap_whole_matrix(full, jd):
    """The whole nb x nb overlap against jdft_ref_overlap: (i) the bands themselves (Hermitian-triangle path, ~identity),
    (ii) NON-orthonormal bands through the same triangle path (off-diagonal entries of every magnitude, so a wrong
    mirror index or conjugation cannot hide), (iii) distinct operands C^+ O (H C).  One k-point of config 4 suffices
    for the 384 x 384 shape."""
    if full.cfg_id == 4 and full.ik not in (0, 3):
        pytest.skip("same shapes as k-points 0 and 3")
    nb = full.nb
    M = jd.jdft_overlap(full.gb, full.dC, full.dC).cpu().numpy()
    assert np.max(np.abs(M - M.conj().T)) <= 1e-12
    assert np.max(np.abs(M - np.eye(nb))) <= 1e-12
    want = full.rb.overlap(full.C, full.C)
    assert np.max(np.abs(M - want)) <= TOL
    Cn = workloads.make_bands(full.cfg_id, full.gb.nG, ik=full.ik, orthonormalise=False)
    Cn = np.ascontiguousarray(Cn * (1.0 + np.arange(nb) % 7)[:, None])            # columns of different norms
    dCn = dev(Cn)
    M2 = jd.jdft_overlap(full.gb, dCn, dCn).cpu().numpy()
    want2 = full.rb.overlap(Cn, Cn)
    assert rel_rows(M2.T, want2.T) <= TOL                                          # per column of M
    assert np.max(np.abs(M2 - M2.conj().T)) <= 1e-13 * np.max(np.abs(M2))
    S2 = jd.jdft_subspace(full.gb, dCn, dCn).cpu().numpy()
    assert rel_rows((S2 * full.gb.volume).T, want2.T) <= TOL
    del dCn
    HC = full.HC if hasattr(full, "HC") else jd.jdft_apply_H(full.gb, full.dV, full.dP, full.dD, full.dC)
    M3 = jd.jdft_overlap(full.gb, full.dC, HC).cpu().numpy()
    want3 = full.rb.overlap(full.C, HC.cpu().numpy())
    assert rel_rows(M3.T, want3.T) <= TOL


def test_full_host_path_every_band(full, jd):
    """The end-to-end leg bench.py times (`e2e`): jdft_apply_H_host with every input in pinned HOST memory (64-band chunks
    pipelined over three streams), then jdft_overlap_host_resident on the block that call uploaded.  EVERY band of HC
    against the oracle; the overlap against the oracle's (the bands are orthonormal: also ~identity); the resident-operator
    variant gives the same HC bit for bit (same kernels, same chunks)."""
    want = full.want_HC if hasattr(full, "want_HC") else full.rb.apply_H(full.V, full.P, full.D, full.C)
    Vp = torch.from_numpy(np.ascontiguousarray(full.V.reshape(-1))).pin_memory()
    Pp, Dp, Cp = (torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (full.P, full.D, full.C))
    HC = torch.empty(full.C.shape, dtype=torch.complex128).pin_memory()
    jd.jdft_apply_H_host(full.gb, Vp, Pp, Dp, Cp, HC)
    got = HC.numpy()
    err = np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)
    assert err.shape == (full.nb,)
    assert float(err.max()) <= TOL, "band %d: %g" % (int(err.argmax()), float(err.max()))
    M = torch.empty((full.nb, full.nb), dtype=torch.complex128).pin_memory()
    gotM = jd.jdft_overlap_host_resident(full.gb, M).numpy()
    assert np.max(np.abs(gotM - full.rb.overlap(full.C, full.C))) <= TOL
    assert np.max(np.abs(gotM - np.eye(full.nb))) <= 1e-12
    jd.jdft_host_set_operators(full.gb, Vp, Pp, Dp)
    HC2 = torch.empty_like(HC).pin_memory()
    jd.jdft_apply_H_host_resident(full.gb, Cp, HC2)
    assert torch.equal(HC2, HC)
    full.want_HC = None                                                                # the oracle's HC is not needed again


def test_full_density_and_subspace(full, jd):
    """Density of a band subset spanning several batches (the oracle sums bands serially): global norm AND the worst
    i0 plane (localises a bad tile); the full subspace Hamiltonian C^+ (H C) against the oracle."""
    if full.cfg_id == 4 and full.ik not in (0, 3):
        pytest.skip("same shapes as k-points 0 and 3")
    nbd = 128 if full.cfg_id == 2 else 12
    rng = np.random.default_rng(53)
    f = rng.uniform(0.0, 2.0, nbd)
    if full.cfg_id != 2:
        jd.jdft_set_option(full.gb, "band_batch", 5)            # 5 + 5 + 2 bands
    got = jd.jdft_density(full.gb, full.dC[:nbd].contiguous(), dev(f)).cpu().numpy()
    jd.jdft_set_option(full.gb, "band_batch", 0)
    want = full.rb.density(full.C[:nbd], f)
    assert np.linalg.norm(got - want) <= TOL * np.linalg.norm(want)
    plane_err = np.abs(got - want).reshape(full.S[0], -1).max(axis=1)
    assert float(plane_err.max()) <= TOL * float(np.abs(want).max()), "worst plane i0 = %d" % int(plane_err.argmax())
    # sum_j n[j] Omega/N = sum_b f_b (bands are O-orthonormal): holds at any size
    assert abs(got.sum() * full.gb.volume / full.gb.N - f.sum()) <= 1e-11 * f.sum()
    HC = full.HC if hasattr(full, "HC") else jd.jdft_apply_H(full.gb, full.dV, full.dP, full.dD, full.dC)
    Hs = jd.jdft_subspace(full.gb, full.dC, HC).cpu().numpy()
    assert np.max(np.abs(Hs - Hs.conj().T)) <= 1e-12 * np.max(np.abs(Hs))
    want_s = full.rb.subspace(full.C, HC.cpu().numpy())
    assert rel_rows(Hs.T, want_s.T) <= TOL


def test_full_pcm_hessian_scalar_field_basis(ref, jd):
    """Listing 1 on a scalar-field basis of the density cutoff (4 x the wavefunction cutoff: sphere radius doubles and
    just fits the box), config-2 box 80^3, Gamma: 8 fields at once against the oracle; constant epsilon
    reduces to (eps0 / 4 pi) |q|^2 phi at any size."""
    R, _, Ecut, S = workloads.lattice(2)
    k = [0.0, 0.0, 0.0]
    rb = ref.RefBasis(R, k, 4 * Ecut, S)
    gb = jd.jdft_basis_create(R, k, 4 * Ecut, S)
    iG, index, ke = jd.jdft_basis_export(gb)
    assert np.array_equal(iG, rb.iG) and np.array_equal(index, rb.index)
    rng = np.random.default_rng(97)
    nf = 8
    phi = rng.standard_normal((nf, rb.nG)) + 1j * rng.standard_normal((nf, rb.nG))
    eps = 1.0 + 78.0 * rng.random(S)
    ws = jd.jdft_workspace_bytes(gb, 3 * nf, 0) + 48 * nf * gb.nG
    jd.jdft_set_workspace(gb, torch.empty(ws, dtype=torch.uint8, device="cuda"))
    got = jd.jdft_pcm_hessian(gb, dev(eps.reshape(-1)), dev(phi)).cpu().numpy()
    want = rb.pcm_hessian(eps, phi)
    assert rel_rows(got, want) <= TOL
    e0 = 78.4
    got0 = jd.jdft_pcm_hessian(gb, dev(np.full(S, e0).reshape(-1)), dev(phi)).cpu().numpy()
    assert rel_rows(got0, (e0 / (4 * np.pi)) * (2.0 * ke)[None, :] * phi) <= 1e-12


def test_full_ultrasoft_and_block_D(full, jd):
    """SURVEY 8(f) rank 2 at full size (configs 2, 3, 5; one k-point of config 4): per-atom blocks of n_lm x n_lm (4 x 4, or
    9 x 9 at config 3) for D in apply_H / apply_Vnl and for Q in apply_O_us / overlap_us.  The GPU processes ALL bands in
    one call; the oracle checks 24 of them (head, tail and both sides of every batch boundary) band by band, and the
    generalised overlap on 16 columns against all nb rows."""
    if full.cfg_id == 4 and full.ik != 0:
        pytest.skip("same shapes as k-point 0")
    nblk = workloads.get_config(full.cfg_id)["n_lm"]
    nproj = full.P.shape[0]
    rng = np.random.default_rng(400 + full.cfg_id)
    A = rng.standard_normal((nproj // nblk, nblk, nblk)) + 1j * rng.standard_normal((nproj // nblk, nblk, nblk))
    Db = np.ascontiguousarray(A + A.conj().transpose(0, 2, 1))
    Qb = np.ascontiguousarray(0.05 * (A @ A.conj().transpose(0, 2, 1)))
    sub = full.subset[:24]
    Cs = full.C[sub]
    dDb, dQb = dev(Db), dev(Qb)
    got = jd.jdft_apply_Vnl(full.gb, full.dP, dDb, full.dC)[sub].cpu().numpy()
    assert rel_rows(got, full.rb.apply_Vnl(full.P, Db, Cs)) <= TOL
    got = jd.jdft_apply_H(full.gb, full.dV, full.dP, dDb, full.dC)[sub].cpu().numpy()
    assert rel_rows(got, full.rb.apply_H(full.V, full.P, Db, Cs)) <= TOL
    got = jd.jdft_apply_O_us(full.gb, full.dP, dQb, full.dC)[sub].cpu().numpy()
    assert rel_rows(got, full.rb.apply_O_us(full.P, Qb, Cs)) <= TOL
    cols = sub[:16]
    M = jd.jdft_overlap_us(full.gb, full.dP, dQb, full.dC, full.dC).cpu().numpy()      # same array: one projection, triangle overlap
    want = full.rb.overlap_us(full.P, Qb, full.C, full.C[cols])                         # [nb, 16]
    assert rel_rows(M[:, cols].T, want.T) <= TOL
    assert np.max(np.abs(M - M.conj().T)) <= 1e-12 * np.max(np.abs(M))
    C2 = dev(np.ascontiguousarray(full.C[cols] * (1.0 + 0.5j)))
    M2 = jd.jdft_overlap_us(full.gb, full.dP, dQb, full.dC, C2).cpu().numpy()           # distinct operands
    assert rel_rows(M2.T, (want * (1.0 + 0.5j)).T) <= TOL


def test_full_pcm_hessian_real_fields(ref, jd):
    """Listing 1 on REAL fields in half-sphere storage on the density-cutoff basis of the config-2 box (nG = 191 471): 4
    fields (3 x 4 = 12 components -> 6 complex transforms) against the oracle's real-field function."""
    R, _, Ecut, S = workloads.lattice(2)
    k = [0.0, 0.0, 0.0]
    rb = ref.RefBasis(R, k, 4 * Ecut, S)
    gb = jd.jdft_basis_create(R, k, 4 * Ecut, S)
    rng = np.random.default_rng(131)
    nf, nGh = 4, (rb.nG + 1) // 2
    ph = rng.standard_normal((nf, nGh)) + 1j * rng.standard_normal((nf, nGh))
    eps = 1.0 + 78.0 * rng.random(S)
    jd.jdft_set_workspace(gb, torch.empty(jd.jdft_workspace_bytes(gb, 3 * nf, 0) + 48 * nf * gb.nG, dtype=torch.uint8, device="cuda"))
    got = jd.jdft_pcm_hessian_real(gb, dev(eps.reshape(-1)), dev(ph)).cpu().numpy()
    assert rel_rows(got, rb.pcm_hessian_real(eps, ph)) <= TOL
