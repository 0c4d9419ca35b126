"""jdft_overlap_noalloc: the overlap whose split-K scratch is the library's static 16 MiB device array (no cudaMalloc, no
workspace; nb1 * nb2 <= 65 536) against the existing jdft_overlap path, on two calls in a row (the array is shared and
keeps the previous call's contents).  Collected last on purpose (the suite runs with pytest -x); passes alone in a
fresh process and after the other tests.  Tolerance: the suite's 1e-10 per column of M (BASELINE.json north_star).
"""
import numpy as np
import pytest
import torch

import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-10


def rel_cols(got, want):
    """max over the columns of M of the relative L2 error"""
    num = torch.linalg.vector_norm(got - want, dim=0)
    den = torch.linalg.vector_norm(want, dim=0)
    return float((num / den).max())


def _bands(cfg_id, nG, nb, seed):
    C = workloads.make_bands(cfg_id, nG, nb=nb, seed=seed, orthonormalise=False)
    return torch.from_numpy(np.ascontiguousarray(C * (1.0 + np.arange(nb) % 3)[:, None])).cuda()


def test_overlap_noalloc_matches_existing_path_two_calls_in_a_row(jd):
    R, kpts, Ecut, S = workloads.lattice(104)                      # 64^3 box, nG ~ 7 000
    ref_basis = jd.jdft_basis_create(R, kpts[0], Ecut, S)
    jd.jdft_alloc_workspace(ref_basis, 1, 256)                     # the existing path needs a caller workspace ...
    gb = jd.jdft_basis_create(R, kpts[0], Ecut, S)                 # ... the new entry point runs on a basis WITHOUT one
    # call 1: a large result (200 x 130 entries, several 64 x 48 tiles with ragged tails, many split-K slices);
    # call 2, right after it on the same stream: a small one that re-uses the front of the same static array;
    # call 3: the same array on both sides (Hermitian-triangle path: only part of each partial is written and read)
    shapes = [(200, 130, 1), (37, 19, 2), (130, 130, 3)]
    for nb1, nb2, seed in shapes:
        C1 = _bands(104, gb.nG, nb1, seed)
        C2 = C1 if seed == 3 else _bands(104, gb.nG, nb2, seed + 10)
        want = jd.jdft_overlap(ref_basis, C1, C2)
        M = torch.full((nb2, nb1), float("nan"), dtype=torch.complex128, device="cuda")
        got = jd.jdft_overlap_noalloc(gb, C1, C2, M)
        assert got.shape == want.shape
        assert rel_cols(got, want) <= TOL
        # a second call with the same inputs: bit-identical (fixed-order reduction, same scratch, stale contents ignored)
        M2 = torch.empty_like(M)
        got2 = jd.jdft_overlap_noalloc(gb, C1, C2, M2)
        assert torch.equal(got2, got)
    # the largest allowed size (256 x 256 = 65 536 entries) still works ...
    C = _bands(104, gb.nG, 256, 7)
    M = torch.empty((256, 256), dtype=torch.complex128, device="cuda")
    assert rel_cols(jd.jdft_overlap_noalloc(gb, C, C, M), jd.jdft_overlap(ref_basis, C, C)) <= TOL
    # ... and anything beyond it is refused with a clear message, not attempted
    C257 = _bands(104, gb.nG, 257, 8)
    with pytest.raises(jd.JdftError) as e:
        jd.jdft_overlap_noalloc(gb, C257, C, torch.empty((256, 257), dtype=torch.complex128, device="cuda"))
    assert e.value.code == jd.JDFT_EINVAL and "scratch limit" in str(e.value)
