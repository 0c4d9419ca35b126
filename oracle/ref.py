"""oracle/ref.py -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes wrapper around oracle/jdft_ref.c (the plain CPU oracle of the DFT++ operators; see that
file's header for the definitions and the PAPER.md / DESIGN.md passages they follow).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from the CUDA package and the CUDA package imports nothing from here.

All arrays are numpy, host memory: C is complex128 [nb, nG]; psi is complex128 [nb, S0, S1, S2];
Vloc is float64 [S0, S1, S2] (or flat [N]); P is complex128 [np, nG]; D is float64 [np] (diagonal),
complex128 [np, np] (dense Hermitian) or complex128 [natoms, nblk, nblk] (per-atom Hermitian blocks); the overlap is returned as M[a, b] (nb1 x nb2).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "jdft_ref.c")
_LIB = os.path.join(_HERE, "libjdft_ref.so")
_lib = None


def build(force=False):
    """Compile oracle/jdft_ref.c -> oracle/libjdft_ref.so with gcc (no fast-math; x87 long double kept)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math", "-Wall",
           "-o", tmp, _SRC, "-lm"]
    subprocess.check_call(cmd)
    os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        vp, ci, dp = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.jdft_ref_basis_create.argtypes = [vp, vp, dp, vp, ctypes.POINTER(vp)]
        L.jdft_ref_basis_destroy.argtypes = [vp]
        L.jdft_ref_basis_info.argtypes = [vp, vp, vp, vp]
        L.jdft_ref_basis_export.argtypes = [vp, vp, vp, vp]
        L.jdft_ref_fft1d.argtypes = [vp, ci, ci, ci]
        L.jdft_ref_apply_I.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_apply_Idag.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_apply_J.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_apply_L.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_apply_O.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_apply_Vnl.argtypes = [vp, vp, ci, vp, ci, vp, ci, vp, ci]
        L.jdft_ref_project.argtypes = [vp, vp, ci, vp, ci, vp]
        L.jdft_ref_apply_H.argtypes = [vp, vp, vp, ci, vp, ci, vp, ci, vp]
        L.jdft_ref_overlap.argtypes = [vp, vp, ci, vp, ci, vp]
        L.jdft_ref_overlap_entry.argtypes = [vp, vp, vp, ci, ci, vp]
        L.jdft_ref_subspace.argtypes = [vp, vp, ci, vp, ci, vp]
        L.jdft_ref_density.argtypes = [vp, vp, ci, vp, vp, ci]
        L.jdft_ref_gradient.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_divergence.argtypes = [vp, vp, ci, vp]
        L.jdft_ref_pcm_hessian.argtypes = [vp, vp, vp, ci, vp]
        L.jdft_ref_pcm_hessian_real.argtypes = [vp, vp, vp, ci, vp]
        L.jdft_ref_apply_O_us.argtypes = [vp, vp, ci, vp, ci, vp, ci, vp]
        L.jdft_ref_overlap_us.argtypes = [vp, vp, ci, vp, ci, vp, ci, vp, ci, vp]
        _lib = L
    return _lib


class RefError(RuntimeError):
    def __init__(self, code):
        super().__init__("oracle call failed with status %d" % code)
        self.code = code


def _chk(rc):
    if rc != 0:
        raise RefError(rc)


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def fft1d(x, sign):
    """Unnormalised 1-D DFT X[q] = sum_j x[j] exp(sign 2 pi i j q / n) by the oracle's own FFT."""
    x = _c128(x).copy()
    _chk(lib().jdft_ref_fft1d(_p(x), x.shape[0], 1, int(sign)))
    return x


class RefBasis:
    """The oracle's basis object (G-sphere index map + geometry)."""

    def __init__(self, R, k, Ecut, S):
        self.R = np.ascontiguousarray(R, dtype=np.float64).reshape(3, 3)
        self.k = np.ascontiguousarray(k, dtype=np.float64).reshape(3)
        self.S = np.ascontiguousarray(S, dtype=np.int32).reshape(3)
        self.Ecut = float(Ecut)
        h = ctypes.c_void_p()
        _chk(lib().jdft_ref_basis_create(_p(self.R), _p(self.k), self.Ecut, _p(self.S), ctypes.byref(h)))
        self._h = h
        nG, N, vol = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_double()
        _chk(lib().jdft_ref_basis_info(h, ctypes.byref(nG), ctypes.byref(N), ctypes.byref(vol)))
        self.nG, self.N, self.volume = nG.value, N.value, vol.value
        self.iG = np.empty((self.nG, 3), dtype=np.int32)
        self.index = np.empty(self.nG, dtype=np.int32)
        self.ke = np.empty(self.nG, dtype=np.float64)
        _chk(lib().jdft_ref_basis_export(h, _p(self.iG), _p(self.index), _p(self.ke)))

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            _lib.jdft_ref_basis_destroy(h)
            self._h = None

    @property
    def shape(self):
        return tuple(int(s) for s in self.S)

    def apply_I(self, C):
        C = _c128(C)
        nb = C.shape[0]
        psi = np.empty((nb,) + self.shape, dtype=np.complex128)
        _chk(lib().jdft_ref_apply_I(self._h, _p(C), nb, _p(psi)))
        return psi

    def _back(self, fn, psi):
        psi = _c128(psi).reshape(-1, self.N)
        nb = psi.shape[0]
        C = np.empty((nb, self.nG), dtype=np.complex128)
        _chk(fn(self._h, _p(psi), nb, _p(C)))
        return C

    def apply_Idag(self, psi):
        return self._back(lib().jdft_ref_apply_Idag, psi)

    def apply_J(self, psi):
        return self._back(lib().jdft_ref_apply_J, psi)

    def _diag(self, fn, C):
        C = _c128(C)
        out = np.empty_like(C)
        _chk(fn(self._h, _p(C), C.shape[0], _p(out)))
        return out

    def apply_L(self, C):
        return self._diag(lib().jdft_ref_apply_L, C)

    def apply_O(self, C):
        return self._diag(lib().jdft_ref_apply_O, C)

    @staticmethod
    def _D(D, nproj):
        if D is None:
            return None, 0
        D = np.asarray(D)
        if D.ndim == 1:
            return np.ascontiguousarray(D, dtype=np.float64), 0
        if D.ndim == 3:  # per-atom Hermitian blocks [natoms, nblk, nblk]: D_mode = nblk
            assert D.shape[1] == D.shape[2] >= 2 and D.shape[0] * D.shape[1] == nproj
            return _c128(D), int(D.shape[1])
        assert D.shape == (nproj, nproj)
        return _c128(D), 1

    def apply_Vnl(self, P, D, C, out=None):
        C = _c128(C)
        P = _c128(P)
        nproj = P.shape[0]
        Dm, mode = self._D(D, nproj)
        acc = 0 if out is None else 1
        res = np.empty_like(C) if out is None else _c128(out).copy()
        _chk(lib().jdft_ref_apply_Vnl(self._h, _p(P), nproj, _p(Dm), mode, _p(C), C.shape[0], _p(res), acc))
        return res

    def project(self, P, C):
        C = _c128(C)
        P = _c128(P)
        B = np.empty((C.shape[0], P.shape[0]), dtype=np.complex128)
        _chk(lib().jdft_ref_project(self._h, _p(P), P.shape[0], _p(C), C.shape[0], _p(B)))
        return B

    def apply_H(self, Vloc, P, D, C):
        C = _c128(C)
        V = np.ascontiguousarray(Vloc, dtype=np.float64).reshape(-1)
        assert V.shape[0] == self.N
        if P is None or len(P) == 0:
            Pm, Dm, mode, nproj = None, None, 0, 0
        else:
            Pm = _c128(P)
            nproj = Pm.shape[0]
            Dm, mode = self._D(D, nproj)
        HC = np.empty_like(C)
        _chk(lib().jdft_ref_apply_H(self._h, _p(V), _p(Pm), nproj, _p(Dm), mode, _p(C), C.shape[0], _p(HC)))
        return HC

    def overlap(self, C1, C2):
        C1, C2 = _c128(C1), _c128(C2)
        nb1, nb2 = C1.shape[0], C2.shape[0]
        M = np.empty((nb2, nb1), dtype=np.complex128)  # column-major nb1 x nb2 == C-order [nb2][nb1]
        _chk(lib().jdft_ref_overlap(self._h, _p(C1), nb1, _p(C2), nb2, _p(M)))
        return M.T  # M[a, b]

    def subspace(self, C1, X2):
        """M[a, b] = sum_n conj(C1[a, n]) X2[b, n] (no Omega); used as C^+ (H C)."""
        C1, X2 = _c128(C1), _c128(X2)
        nb1, nb2 = C1.shape[0], X2.shape[0]
        M = np.empty((nb2, nb1), dtype=np.complex128)
        _chk(lib().jdft_ref_subspace(self._h, _p(C1), nb1, _p(X2), nb2, _p(M)))
        return M.T

    def density(self, C, f, n=None):
        """n[j] (+)= sum_b f[b] |(I C_b)[j]|^2, float64 [S0, S1, S2]; accumulates into n if given."""
        C = _c128(C)
        f = np.ascontiguousarray(f, dtype=np.float64)
        acc = n is not None
        if n is None:
            n = np.zeros(self.shape, dtype=np.float64)
        assert n.flags.c_contiguous and n.dtype == np.float64
        _chk(lib().jdft_ref_density(self._h, _p(C), C.shape[0], _p(f), _p(n), 1 if acc else 0))
        return n

    def gradient(self, C):
        """[3, nb, nG]: i q_d C, q = G^T (iG + k) Cartesian."""
        C = _c128(C)
        out = np.empty((3,) + C.shape, dtype=np.complex128)
        _chk(lib().jdft_ref_gradient(self._h, _p(C), C.shape[0], _p(out)))
        return out

    def divergence(self, X):
        """[nb, nG]: sum_d i q_d X[d]."""
        X = _c128(X)
        out = np.empty(X.shape[1:], dtype=np.complex128)
        _chk(lib().jdft_ref_divergence(self._h, _p(X), X.shape[1], _p(out)))
        return out

    def pcm_hessian(self, epsilon, phi):
        """Listing 1 of the paper: (-1/4 pi) divergence(J(epsilon * I(gradient(phi)))); epsilon float64 [S0,S1,S2]."""
        phi = _c128(phi)
        eps = np.ascontiguousarray(epsilon, dtype=np.float64)
        assert eps.size == self.N
        out = np.empty_like(phi)
        _chk(lib().jdft_ref_pcm_hessian(self._h, _p(eps), _p(phi), phi.shape[0], _p(out)))
        return out

    def pcm_hessian_real(self, epsilon, phi_h):
        """Listing 1 on real fields in half-sphere storage: phi_h[ib, h] = phi~[n0 + h], n0 = (nG - 1) / 2 (k = 0 only)."""
        phi_h = _c128(phi_h)
        eps = np.ascontiguousarray(epsilon, dtype=np.float64)
        assert eps.size == self.N and phi_h.shape[1] == (self.nG + 1) // 2
        out = np.empty_like(phi_h)
        _chk(lib().jdft_ref_pcm_hessian_real(self._h, _p(eps), _p(phi_h), phi_h.shape[0], _p(out)))
        return out

    def apply_O_us(self, P, Q, C):
        """Ultrasoft generalised overlap operator: Omega (C + P Q P^+ C); Q like D (diag / dense / per-atom blocks)."""
        C, P = _c128(C), _c128(P)
        Qm, mode = self._D(Q, P.shape[0])
        out = np.empty_like(C)
        _chk(lib().jdft_ref_apply_O_us(self._h, _p(P), P.shape[0], _p(Qm), mode, _p(C), C.shape[0], _p(out)))
        return out

    def overlap_us(self, P, Q, C1, C2):
        """M[a, b] = C1[a]^+ O_us C2[b] with O_us = Omega (1 + P Q P^+)."""
        C1, C2, P = _c128(C1), _c128(C2), _c128(P)
        Qm, mode = self._D(Q, P.shape[0])
        nb1, nb2 = C1.shape[0], C2.shape[0]
        M = np.empty((nb2, nb1), dtype=np.complex128)
        _chk(lib().jdft_ref_overlap_us(self._h, _p(P), P.shape[0], _p(Qm), mode, _p(C1), nb1, _p(C2), nb2, _p(M)))
        return M.T

    def overlap_entry(self, C1, C2, a, b):
        C1, C2 = _c128(C1), _c128(C2)
        out = np.empty(2, dtype=np.float64)
        _chk(lib().jdft_ref_overlap_entry(self._h, _p(C1), _p(C2), int(a), int(b), _p(out)))
        return complex(out[0], out[1])


def threads():
    """Number of OpenMP threads the oracle will use (OMP_NUM_THREADS or the affinity count)."""
    v = os.environ.get("OMP_NUM_THREADS")
    if v:
        return int(v.split(",")[0])
    return len(os.sched_getaffinity(0))
