"""Thin ctypes binding of libjdft_b200.so (include/jdft.h): argument marshalling only.

Function names equal the C ABI's.  Tensors are torch CUDA tensors (complex128 / float64); every step of the
path runs in the library's CUDA kernels on the current torch stream.  There is no CPU fallback: importing
this module without the built library, or calling it without a CUDA device, raises.
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libjdft_b200.so")

JDFT_OK, JDFT_EINVAL, JDFT_EBOX, JDFT_EWORKSPACE, JDFT_ECUDA, JDFT_ENOMEM = 0, -1, -2, -3, -4, -5

EXPORTS = [
    "jdft_basis_create", "jdft_basis_destroy", "jdft_basis_info", "jdft_basis_structure", "jdft_basis_export",
    "jdft_basis_device_maps", "jdft_workspace_bytes", "jdft_set_workspace", "jdft_set_option",
    "jdft_apply_I", "jdft_apply_Idag", "jdft_apply_J", "jdft_apply_L", "jdft_apply_O", "jdft_apply_Vnl",
    "jdft_project", "jdft_apply_H", "jdft_overlap", "jdft_overlap_noalloc", "jdft_apply_O_us", "jdft_overlap_us", "jdft_subspace", "jdft_density", "jdft_gradient", "jdft_divergence", "jdft_pcm_hessian", "jdft_pcm_hessian_real", "jdft_apply_H_host", "jdft_overlap_host", "jdft_host_set_operators", "jdft_apply_H_host_resident", "jdft_overlap_host_resident",
    "jdft_last_error", "jdft_launch_count", "jdft_profile_read", "jdft_version",
]


class JdftError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libjdft_b200 status %d: %s" % (code, msg))
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libjdft_b200.so is not built: run `python -m paper_1708_03621_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, dp, i64, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_int64, ctypes.c_size_t
    L.jdft_basis_create.argtypes = [vp, vp, dp, vp, ci, ctypes.POINTER(vp)]
    L.jdft_basis_destroy.argtypes = [vp]
    L.jdft_basis_info.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64), ctypes.POINTER(dp)]
    L.jdft_basis_structure.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64)]
    L.jdft_basis_export.argtypes = [vp, vp, vp, vp]
    L.jdft_basis_device_maps.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp)]
    L.jdft_workspace_bytes.argtypes = [vp, ci, ci]
    L.jdft_workspace_bytes.restype = sz
    L.jdft_set_workspace.argtypes = [vp, vp, sz]
    L.jdft_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    for name in ("jdft_apply_I", "jdft_apply_Idag", "jdft_apply_J", "jdft_apply_L", "jdft_apply_O"):
        getattr(L, name).argtypes = [vp, vp, ci, vp, vp]
    L.jdft_apply_Vnl.argtypes = [vp, vp, ci, vp, ci, vp, ci, vp, ci, vp]
    L.jdft_project.argtypes = [vp, vp, ci, vp, ci, vp, vp]
    L.jdft_apply_H.argtypes = [vp, vp, vp, ci, vp, ci, vp, ci, vp, vp]
    L.jdft_overlap.argtypes = [vp, vp, ci, vp, ci, vp, vp]
    L.jdft_subspace.argtypes = [vp, vp, ci, vp, ci, vp, vp]
    L.jdft_overlap_noalloc.argtypes = [vp, vp, ci, vp, ci, vp, vp]
    L.jdft_apply_O_us.argtypes = [vp, vp, ci, vp, ci, vp, ci, vp, vp]
    L.jdft_overlap_us.argtypes = [vp, vp, ci, vp, ci, vp, ci, vp, ci, vp, vp]
    L.jdft_density.argtypes = [vp, vp, ci, vp, vp, ci, vp]
    L.jdft_gradient.argtypes = [vp, vp, ci, vp, vp]
    L.jdft_divergence.argtypes = [vp, vp, ci, vp, vp]
    L.jdft_pcm_hessian.argtypes = [vp, vp, vp, ci, vp, vp]
    L.jdft_pcm_hessian_real.argtypes = [vp, vp, vp, ci, vp, vp]
    L.jdft_apply_H_host.argtypes = [vp, vp, vp, ci, vp, ci, vp, ci, vp]
    L.jdft_overlap_host.argtypes = [vp, vp, ci, vp, ci, vp]
    L.jdft_host_set_operators.argtypes = [vp, vp, vp, ci, vp, ci]
    L.jdft_apply_H_host_resident.argtypes = [vp, vp, ci, vp]
    L.jdft_overlap_host_resident.argtypes = [vp, ci, vp]
    L.jdft_last_error.restype = ctypes.c_char_p
    L.jdft_launch_count.argtypes = [ci]
    L.jdft_launch_count.restype = i64
    L.jdft_profile_read.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(dp)]
    L.jdft_version.restype = ctypes.c_char_p
    return L


_lib = _load()


def _chk(rc):
    if rc != 0:
        raise JdftError(rc, _lib.jdft_last_error().decode())


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, dtype, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor of dtype %s" % (name, dtype))
    return ctypes.c_void_p(t.data_ptr())


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


class Basis:
    """Handle of a jdft_basis plus the torch-owned workspace it points at."""

    def __init__(self, handle, device, S):
        self._h = handle
        self.device = torch.device("cuda", device)
        self.S = tuple(int(s) for s in S)
        nG, N, vol = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_double()
        _chk(_lib.jdft_basis_info(handle, ctypes.byref(nG), ctypes.byref(N), ctypes.byref(vol)))
        self.nG, self.N, self.volume = nG.value, N.value, vol.value
        npl, ncol = ctypes.c_int64(), ctypes.c_int64()
        _chk(_lib.jdft_basis_structure(handle, ctypes.byref(npl), ctypes.byref(ncol)))
        self.npl, self.ncol = npl.value, ncol.value
        self._ws = None

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:  # at interpreter shutdown the module globals may already be gone
            _lib.jdft_basis_destroy(h)
            self._h = None


def jdft_basis_create(R, k, Ecut, S, device=0):
    if not torch.cuda.is_available():
        raise RuntimeError("jdft_basis_create needs a CUDA device (there is no CPU fallback)")
    R = _np(R, np.float64).reshape(9)
    k = _np(k, np.float64).reshape(3)
    S = _np(S, np.int32).reshape(3)
    h = ctypes.c_void_p()
    _chk(_lib.jdft_basis_create(R.ctypes.data, k.ctypes.data, float(Ecut), S.ctypes.data, int(device), ctypes.byref(h)))
    return Basis(h, int(device), S)


def jdft_basis_destroy(basis):
    if basis._h:
        _chk(_lib.jdft_basis_destroy(basis._h))
        basis._h = None


def jdft_basis_export(basis):
    """HOST copies (iG int32[nG,3], index int32[nG], ke float64[nG])."""
    iG = np.empty((basis.nG, 3), dtype=np.int32)
    index = np.empty(basis.nG, dtype=np.int32)
    ke = np.empty(basis.nG, dtype=np.float64)
    _chk(_lib.jdft_basis_export(basis._h, iG.ctypes.data, index.ctypes.data, ke.ctypes.data))
    return iG, index, ke


def jdft_workspace_bytes(basis, nbands_batch, nrows_max):
    return int(_lib.jdft_workspace_bytes(basis._h, int(nbands_batch), int(nrows_max)))


def jdft_set_workspace(basis, tensor):
    """tensor: a torch CUDA uint8 tensor (kept alive by the Basis), or None."""
    if tensor is None:
        _chk(_lib.jdft_set_workspace(basis._h, None, 0))
    else:
        _chk(_lib.jdft_set_workspace(basis._h, ctypes.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size()))
    basis._ws = tensor


def jdft_alloc_workspace(basis, nbands_batch, nrows_max):
    """Convenience: allocate the workspace with torch and attach it."""
    n = jdft_workspace_bytes(basis, nbands_batch, nrows_max)
    ws = torch.empty(n, dtype=torch.uint8, device=basis.device)
    jdft_set_workspace(basis, ws)
    return ws


def jdft_set_option(basis, key, value):
    _chk(_lib.jdft_set_option(basis._h, key.encode(), int(value)))


def _bands(C, basis, name):
    if C.dim() != 2 or C.shape[1] != basis.nG:
        raise ValueError("%s must have shape [nb, nG=%d]" % (name, basis.nG))
    return int(C.shape[0])


def jdft_apply_I(basis, C, psi=None):
    nb = _bands(C, basis, "C")
    if psi is None:
        psi = torch.empty((nb,) + basis.S, dtype=torch.complex128, device=C.device)
    _chk(_lib.jdft_apply_I(basis._h, _dev(C, torch.complex128, "C"), nb, _dev(psi, torch.complex128, "psi"), _stream()))
    return psi


def _back(fn, basis, psi, C):
    nb = int(psi.shape[0])
    if psi.numel() != nb * basis.N:
        raise ValueError("psi must have shape [nb, S0, S1, S2]")
    if C is None:
        C = torch.empty((nb, basis.nG), dtype=torch.complex128, device=psi.device)
    _chk(fn(basis._h, _dev(psi, torch.complex128, "psi"), nb, _dev(C, torch.complex128, "C"), _stream()))
    return C


def jdft_apply_Idag(basis, psi, C=None):
    return _back(_lib.jdft_apply_Idag, basis, psi, C)


def jdft_apply_J(basis, psi, C=None):
    return _back(_lib.jdft_apply_J, basis, psi, C)


def _diag(fn, basis, C, out):
    nb = _bands(C, basis, "C")
    if out is None:
        out = torch.empty_like(C)
    _chk(fn(basis._h, _dev(C, torch.complex128, "C"), nb, _dev(out, torch.complex128, "out"), _stream()))
    return out


def jdft_apply_L(basis, C, out=None):
    return _diag(_lib.jdft_apply_L, basis, C, out)


def jdft_apply_O(basis, C, out=None):
    return _diag(_lib.jdft_apply_O, basis, C, out)


def _PD(P, D, basis):
    if P is None or P.shape[0] == 0:
        return None, 0, None, 0
    nproj = int(P.shape[0])
    if P.dim() != 2 or P.shape[1] != basis.nG:
        raise ValueError("P must have shape [nproj, nG]")
    if D.dim() == 1:
        if D.shape[0] != nproj:
            raise ValueError("diagonal D must have nproj entries")
        return _dev(P, torch.complex128, "P"), nproj, _dev(D, torch.float64, "D"), 0
    if D.dim() == 3:  # per-atom Hermitian blocks [nproj / nblk, nblk, nblk]: D_mode = nblk
        nblk = int(D.shape[1])
        if nblk < 2 or D.shape[2] != nblk or D.shape[0] * nblk != nproj:
            raise ValueError("block D must be [nproj / nblk, nblk, nblk] with nblk >= 2")
        return _dev(P, torch.complex128, "P"), nproj, _dev(D, torch.complex128, "D"), nblk
    if tuple(D.shape) != (nproj, nproj):
        raise ValueError("dense D must be [nproj, nproj]")
    return _dev(P, torch.complex128, "P"), nproj, _dev(D, torch.complex128, "D"), 1


def jdft_apply_Vnl(basis, P, D, C, out=None, accumulate=False):
    nb = _bands(C, basis, "C")
    if out is None:
        out = torch.empty_like(C)
        accumulate = False
    Pp, nproj, Dp, mode = _PD(P, D, basis)
    _chk(_lib.jdft_apply_Vnl(basis._h, Pp, nproj, Dp, mode, _dev(C, torch.complex128, "C"), nb,
                             _dev(out, torch.complex128, "out"), 1 if accumulate else 0, _stream()))
    return out


def jdft_project(basis, P, C, Bproj=None):
    nb = _bands(C, basis, "C")
    nproj = int(P.shape[0])
    if Bproj is None:
        Bproj = torch.empty((nb, nproj), dtype=torch.complex128, device=C.device)
    _chk(_lib.jdft_project(basis._h, _dev(P, torch.complex128, "P"), nproj, _dev(C, torch.complex128, "C"), nb,
                           _dev(Bproj, torch.complex128, "Bproj"), _stream()))
    return Bproj


def jdft_apply_H(basis, Vloc, P, D, C, HC=None):
    nb = _bands(C, basis, "C")
    if Vloc.numel() != basis.N:
        raise ValueError("Vloc must have N = S0*S1*S2 entries")
    if HC is None:
        HC = torch.empty_like(C)
    Pp, nproj, Dp, mode = _PD(P, D, basis)
    _chk(_lib.jdft_apply_H(basis._h, _dev(Vloc, torch.float64, "Vloc"), Pp, nproj, Dp, mode,
                           _dev(C, torch.complex128, "C"), nb, _dev(HC, torch.complex128, "HC"), _stream()))
    return HC


def jdft_overlap(basis, C1, C2, M=None):
    """Returns M with M[a, b] = Omega sum_n conj(C1[a, n]) C2[b, n] (a view of the column-major result)."""
    nb1, nb2 = _bands(C1, basis, "C1"), _bands(C2, basis, "C2")
    if M is None:
        M = torch.empty((nb2, nb1), dtype=torch.complex128, device=C1.device)  # column-major nb1 x nb2
    _chk(_lib.jdft_overlap(basis._h, _dev(C1, torch.complex128, "C1"), nb1, _dev(C2, torch.complex128, "C2"), nb2,
                           _dev(M, torch.complex128, "M"), _stream()))
    return M.t()


def jdft_overlap_noalloc(basis, C1, C2, M):
    """jdft_overlap with the split-K scratch in the library's static 16 MiB device array: no allocation, no workspace;
    nb1 * nb2 <= 65536.  M: caller-provided CUDA complex128 [nb2, nb1] (column-major nb1 x nb2); returns the view M[a, b]."""
    nb1, nb2 = _bands(C1, basis, "C1"), _bands(C2, basis, "C2")
    if tuple(M.shape) != (nb2, nb1):
        raise ValueError("M must have shape [nb2, nb1]")
    _chk(_lib.jdft_overlap_noalloc(basis._h, _dev(C1, torch.complex128, "C1"), nb1, _dev(C2, torch.complex128, "C2"), nb2,
                                   _dev(M, torch.complex128, "M"), _stream()))
    return M.t()


def jdft_apply_O_us(basis, P, Q, C, OC=None):
    """Ultrasoft generalised overlap operator Omega (C + P Q P^+ C); Q: [np] real, [np, np] or [np / nblk, nblk, nblk]."""
    nb = _bands(C, basis, "C")
    if OC is None:
        OC = torch.empty_like(C)
    Pp, nproj, Qp, mode = _PD(P, Q, basis)
    _chk(_lib.jdft_apply_O_us(basis._h, Pp, nproj, Qp, mode, _dev(C, torch.complex128, "C"), nb,
                              _dev(OC, torch.complex128, "OC"), _stream()))
    return OC


def jdft_overlap_us(basis, P, Q, C1, C2, M=None):
    """M[a, b] = C1[a]^+ O_us C2[b], O_us = Omega (1 + P Q P^+) (a view of the column-major result)."""
    nb1, nb2 = _bands(C1, basis, "C1"), _bands(C2, basis, "C2")
    if M is None:
        M = torch.empty((nb2, nb1), dtype=torch.complex128, device=C1.device)
    Pp, nproj, Qp, mode = _PD(P, Q, basis)
    _chk(_lib.jdft_overlap_us(basis._h, Pp, nproj, Qp, mode, _dev(C1, torch.complex128, "C1"), nb1,
                              _dev(C2, torch.complex128, "C2"), nb2, _dev(M, torch.complex128, "M"), _stream()))
    return M.t()


def jdft_subspace(basis, C1, X2, M=None):
    """Returns M with M[a, b] = sum_n conj(C1[a, n]) X2[b, n] (no Omega; a view of the column-major result)."""
    nb1, nb2 = _bands(C1, basis, "C1"), _bands(X2, basis, "X2")
    if M is None:
        M = torch.empty((nb2, nb1), dtype=torch.complex128, device=C1.device)
    _chk(_lib.jdft_subspace(basis._h, _dev(C1, torch.complex128, "C1"), nb1, _dev(X2, torch.complex128, "X2"), nb2,
                            _dev(M, torch.complex128, "M"), _stream()))
    return M.t()


def jdft_density(basis, C, f, n=None, accumulate=False):
    """n[S0, S1, S2] (+)= sum_b f[b] |(I C_b)|^2 ; f is a CUDA float64 tensor [nb]."""
    nb = _bands(C, basis, "C")
    if f.numel() != nb:
        raise ValueError("f must have one entry per band")
    if n is None:
        n = torch.empty(basis.S, dtype=torch.float64, device=C.device)
        accumulate = False
    elif n.numel() != basis.N:
        raise ValueError("n must have N = S0*S1*S2 entries")
    _chk(_lib.jdft_density(basis._h, _dev(C, torch.complex128, "C"), nb, _dev(f, torch.float64, "f"),
                           _dev(n, torch.float64, "n"), 1 if accumulate else 0, _stream()))
    return n


def jdft_gradient(basis, C, out=None):
    """[3, nb, nG] = i q_d C."""
    nb = _bands(C, basis, "C")
    if out is None:
        out = torch.empty((3, nb, basis.nG), dtype=torch.complex128, device=C.device)
    _chk(_lib.jdft_gradient(basis._h, _dev(C, torch.complex128, "C"), nb, _dev(out, torch.complex128, "out"), _stream()))
    return out


def jdft_divergence(basis, X, out=None):
    """[nb, nG] = sum_d i q_d X[d];  X is [3, nb, nG]."""
    if X.dim() != 3 or X.shape[0] != 3 or X.shape[2] != basis.nG:
        raise ValueError("X must have shape [3, nb, nG]")
    nb = int(X.shape[1])
    if out is None:
        out = torch.empty((nb, basis.nG), dtype=torch.complex128, device=X.device)
    _chk(_lib.jdft_divergence(basis._h, _dev(X, torch.complex128, "X"), nb, _dev(out, torch.complex128, "out"), _stream()))
    return out


def jdft_pcm_hessian(basis, epsilon, phi, out=None):
    """Listing 1 of the paper: (-1/4 pi) divergence(J(epsilon * I(gradient(phi)))); epsilon float64 with N entries."""
    nb = _bands(phi, basis, "phi")
    if epsilon.numel() != basis.N:
        raise ValueError("epsilon must have N = S0*S1*S2 entries")
    if out is None:
        out = torch.empty_like(phi)
    _chk(_lib.jdft_pcm_hessian(basis._h, _dev(epsilon, torch.float64, "epsilon"), _dev(phi, torch.complex128, "phi"), nb,
                               _dev(out, torch.complex128, "out"), _stream()))
    return out


def jdft_pcm_hessian_real(basis, epsilon, phi_h, out_h=None):
    """Listing 1 on real fields in half-sphere storage: phi_h [nb, (nG + 1) / 2] = phi~[n0:], n0 = (nG - 1) / 2; k = 0 only."""
    nGh = (basis.nG + 1) // 2
    if phi_h.dim() != 2 or phi_h.shape[1] != nGh:
        raise ValueError("phi_h must have shape [nb, (nG + 1) / 2 = %d]" % nGh)
    if epsilon.numel() != basis.N:
        raise ValueError("epsilon must have N = S0*S1*S2 entries")
    if out_h is None:
        out_h = torch.empty_like(phi_h)
    _chk(_lib.jdft_pcm_hessian_real(basis._h, _dev(epsilon, torch.float64, "epsilon"), _dev(phi_h, torch.complex128, "phi_h"),
                                    int(phi_h.shape[0]), _dev(out_h, torch.complex128, "out_h"), _stream()))
    return out_h


def _host(a, dtype, name):
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != dtype or not a.is_contiguous():
            raise TypeError("%s must be a contiguous CPU tensor of dtype %s" % (name, dtype))
        return ctypes.c_void_p(a.data_ptr())
    raise TypeError("%s must be a CPU torch tensor" % name)


def jdft_apply_H_host(basis, Vloc, P, D, C, HC):
    """HOST tensors in and out (pinned for full copy speed); copies, kernels and sync happen inside the call."""
    nb = int(C.shape[0])
    if P is None or P.shape[0] == 0:
        Pp, nproj, Dp, mode = None, 0, None, 0
    else:
        nproj = int(P.shape[0])
        mode = 0 if D.dim() == 1 else (1 if D.dim() == 2 else int(D.shape[1]))
        Pp = _host(P, torch.complex128, "P")
        Dp = _host(D, torch.float64 if mode == 0 else torch.complex128, "D")
    _chk(_lib.jdft_apply_H_host(basis._h, _host(Vloc, torch.float64, "Vloc"), Pp, nproj, Dp, mode,
                                _host(C, torch.complex128, "C"), nb, _host(HC, torch.complex128, "HC")))
    return HC


def jdft_host_set_operators(basis, Vloc, P, D):
    """Upload V_loc, P, D once (HOST tensors); jdft_apply_H_host_resident then copies only the bands in and H C out."""
    if P is None or P.shape[0] == 0:
        Pp, nproj, Dp, mode = None, 0, None, 0
    else:
        nproj = int(P.shape[0])
        mode = 0 if D.dim() == 1 else (1 if D.dim() == 2 else int(D.shape[1]))
        Pp = _host(P, torch.complex128, "P")
        Dp = _host(D, torch.float64 if mode == 0 else torch.complex128, "D")
    _chk(_lib.jdft_host_set_operators(basis._h, _host(Vloc, torch.float64, "Vloc"), Pp, nproj, Dp, mode))


def jdft_apply_H_host_resident(basis, C, HC):
    _chk(_lib.jdft_apply_H_host_resident(basis._h, _host(C, torch.complex128, "C"), int(C.shape[0]),
                                         _host(HC, torch.complex128, "HC")))
    return HC


def jdft_overlap_host_resident(basis, M):
    """C^+ O C of the bands the last jdft_apply_H_host[_resident] call uploaded (no second upload); M: HOST [nb, nb]."""
    _chk(_lib.jdft_overlap_host_resident(basis._h, int(M.shape[0]), _host(M, torch.complex128, "M")))
    return M.t()


def jdft_overlap_host(basis, C1, C2, M):
    _chk(_lib.jdft_overlap_host(basis._h, _host(C1, torch.complex128, "C1"), int(C1.shape[0]),
                                _host(C2, torch.complex128, "C2"), int(C2.shape[0]), _host(M, torch.complex128, "M")))
    return M.t()


def jdft_launch_count(reset=False):
    return int(_lib.jdft_launch_count(1 if reset else 0))


KERNEL_IDS = {"cols_inv": 1, "rows_inv": 2, "planes": 3, "rows_fwd": 4, "cols_fwd": 5, "gemm_dotk": 6,
              "gemm_expand": 7, "splitk_reduce": 8, "diag": 9}


def jdft_profile_read(basis):
    """(launches, total_ms) of the kernel selected with jdft_set_option(basis, "profile_kernel", id); resets."""
    n, ms = ctypes.c_int64(), ctypes.c_double()
    _chk(_lib.jdft_profile_read(basis._h, ctypes.byref(n), ctypes.byref(ms)))
    return n.value, ms.value


def jdft_version():
    return _lib.jdft_version().decode()
