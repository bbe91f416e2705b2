"""B200-native direct-SCF J/K Fock build (arXiv 2406.14920) -- thin Python binding of the C ABI in
include/te_jk.h (libte_jk.so, hand-written CUDA for sm_100a).

Argument marshalling only: every step of the path runs in the library's kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: if the CUDA extension is missing the import of the
native library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))
NCLASS = 10
CLASS_NAMES = ["SS", "SP", "SD", "SF", "PP", "PD", "PF", "DD", "DF", "FF"]
CLASS_L = [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]

_lib = None


class TEError(RuntimeError):
    pass


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def lib():
    """Load libte_jk.so (building it with nvcc if the in-tree copy is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = os.path.join(HERE, "libte_jk.so")
    if not os.path.exists(path) or os.environ.get("TE_REBUILD"):
        path = _build.build()
    if not os.path.exists(path):
        raise TEError("libte_jk.so is missing and could not be built: the CUDA path is the only path")
    L = C.CDLL(path)
    vp, dpp, ipp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    L.te_basis_create.argtypes = [C.c_int, dpp, C.c_int, ipp, ipp, ipp, dpp, dpp, C.POINTER(vp)]
    L.te_basis_destroy.argtypes = [vp]
    L.te_basis_destroy.restype = None
    L.te_basis_nbf.argtypes = [vp]
    L.te_basis_nprim.argtypes = [vp]
    L.te_basis_shell_offsets.argtypes = [vp, ipp]
    L.te_basis_norm_coefs.argtypes = [vp, dpp]
    L.te_shellpair_build.argtypes = [vp, C.c_double, C.POINTER(vp)]
    L.te_pairs_destroy.argtypes = [vp]
    L.te_pairs_destroy.restype = None
    L.te_pairs_info.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.te_pairs_export.argtypes = [vp, C.c_int, ipp, ipp, ipp, ipp, dpp]
    L.te_pairs_export_geom.argtypes = [vp, C.c_int, dpp, dpp, dpp]
    L.te_build_jk.argtypes = [vp, vp, vp, vp, C.c_double, vp]
    L.te_build_jk_host.argtypes = [vp, dpp, dpp, dpp, C.c_double]
    L.te_build_jk_lr.argtypes = [vp, vp, vp, vp, C.c_double, C.c_double, vp]
    L.te_build_jk_mixed.argtypes = [vp, vp, vp, vp, C.c_double, C.c_double, vp]
    L.te_build_j.argtypes = [vp, vp, vp, C.c_double, vp]
    L.te_jk_precision_stats.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.te_nuclear_attraction.argtypes = [vp, C.c_int, dpp, dpp, vp, vp]
    L.te_nuclear_attraction_noalloc.argtypes = [vp, C.c_int, vp, vp, vp]
    L.te_jk_set_kernel_family.argtypes = [vp, C.c_int]
    L.te_measure_smem_dfma_rate.argtypes = [C.c_int, dpp]
    L.te_jk_stats.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_float)]
    L.te_jk_screening_stats.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.te_jk_set_profiling.argtypes = [vp, C.c_int]
    L.te_eri_block.argtypes = [vp, C.c_int, ipp, C.POINTER(C.c_longlong), vp]
    L.te_boys.argtypes = [C.c_int, vp, C.c_int, vp]
    L.te_measure_fp64_peak.argtypes = [dpp]
    L.te_last_error.restype = C.c_char_p
    _lib = L
    return L


def _check(rc, what):
    if rc != 0:
        raise TEError(f"{what} failed ({rc}): {lib().te_last_error().decode()}")


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


class Basis:
    """te_basis handle (te_basis_create / te_basis_destroy)."""

    def __init__(self, xyz, shell_atom, shell_l, shell_nprim, exponents, coefficients):
        L = lib()
        self.xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        self.shell_atom = np.ascontiguousarray(shell_atom, dtype=np.int32)
        self.shell_l = np.ascontiguousarray(shell_l, dtype=np.int32)
        self.shell_nprim = np.ascontiguousarray(shell_nprim, dtype=np.int32)
        ex = np.ascontiguousarray(exponents, dtype=np.float64)
        co = np.ascontiguousarray(coefficients, dtype=np.float64)
        self.handle = C.c_void_p()
        _check(L.te_basis_create(self.xyz.shape[0], _dp(self.xyz), len(self.shell_l), _ip(self.shell_atom),
                                 _ip(self.shell_l), _ip(self.shell_nprim), _dp(ex), _dp(co), C.byref(self.handle)),
               "te_basis_create")
        self.nshells = len(self.shell_l)
        self.nbf = int(L.te_basis_nbf(self.handle))
        self.nprim = int(L.te_basis_nprim(self.handle))

    @classmethod
    def from_problem(cls, prob):
        return cls(prob.xyz, prob.shell_atom, prob.shell_l, prob.shell_nprim, prob.exponents, prob.coefficients)

    def shell_offsets(self) -> np.ndarray:
        off = np.zeros(self.nshells + 1, dtype=np.int32)
        _check(lib().te_basis_shell_offsets(self.handle, _ip(off)), "te_basis_shell_offsets")
        return off

    def norm_coefs(self) -> np.ndarray:
        out = np.zeros(self.nprim)
        _check(lib().te_basis_norm_coefs(self.handle, _dp(out)), "te_basis_norm_coefs")
        return out

    def shellpair_build(self, pair_threshold: float) -> "Pairs":
        return Pairs(self, pair_threshold)

    def eri_block(self, quartets) -> list:
        """te_eri_block: list of [nA,nB,nC,nD] numpy blocks (A_i B_j|C_k D_l) for shell-id quartets."""
        import torch
        q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
        sizes = [int(np.prod([ncart(int(self.shell_l[s])) for s in row])) for row in q]
        offs = np.zeros(len(q) + 1, dtype=np.int64)
        offs[1:] = np.cumsum(sizes)
        out = torch.zeros(int(offs[-1]), dtype=torch.float64, device="cuda")
        _check(lib().te_eri_block(self.handle, len(q), _ip(q), offs.ctypes.data_as(C.POINTER(C.c_longlong)),
                                  C.c_void_p(out.data_ptr())), "te_eri_block")
        h = out.cpu().numpy()
        return [h[offs[i]:offs[i + 1]].reshape([ncart(int(self.shell_l[s])) for s in q[i]]) for i in range(len(q))]

    def close(self):
        if getattr(self, "handle", None):
            lib().te_basis_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Pairs:
    """te_pairs handle (te_shellpair_build / te_pairs_destroy)."""

    def __init__(self, basis: Basis, pair_threshold: float):
        self.basis = basis
        self.handle = C.c_void_p()
        _check(lib().te_shellpair_build(basis.handle, float(pair_threshold), C.byref(self.handle)), "te_shellpair_build")
        cnt = (C.c_longlong * NCLASS)()
        tot = C.c_longlong()
        _check(lib().te_pairs_info(self.handle, cnt, C.byref(tot)), "te_pairs_info")
        self.class_count = [int(x) for x in cnt]
        self.nkept = int(tot.value)

    def export(self, cls: int) -> dict:
        n = self.class_count[cls]
        out = {k: np.zeros(n, dtype=np.int32) for k in ("shellA", "shellB", "primA", "primB")}
        out["bound"] = np.zeros(n)
        out["P"] = np.zeros((n, 3))
        out["p"] = np.zeros(n)
        out["prefactor"] = np.zeros(n)
        L = lib()
        _check(L.te_pairs_export(self.handle, cls, _ip(out["shellA"]), _ip(out["shellB"]), _ip(out["primA"]),
                                 _ip(out["primB"]), _dp(out["bound"])), "te_pairs_export")
        _check(L.te_pairs_export_geom(self.handle, cls, _dp(out["P"]), _dp(out["p"]), _dp(out["prefactor"])),
               "te_pairs_export_geom")
        return out

    def build_jk(self, D, J=None, K=None, threshold: float = 0.0, stream=None, omega: float | None = None,
                 fp32_below: float | None = None):
        """te_build_jk (te_build_jk_lr when omega is given, te_build_jk_mixed when fp32_below is given) with torch CUDA
        tensors (float64, nbf x nbf, contiguous).  Asynchronous on `stream`."""
        import torch
        n = self.basis.nbf
        assert D.is_cuda and D.dtype == torch.float64 and D.is_contiguous() and tuple(D.shape) == (n, n)
        if J is None:
            J = torch.empty_like(D)
        if K is None:
            K = torch.empty_like(D)
        st = stream if stream is not None else torch.cuda.current_stream()
        if fp32_below is not None:
            assert omega is None
            _check(lib().te_build_jk_mixed(self.handle, C.c_void_p(D.data_ptr()), C.c_void_p(J.data_ptr()),
                                           C.c_void_p(K.data_ptr()), float(threshold), float(fp32_below),
                                           C.c_void_p(st.cuda_stream)), "te_build_jk_mixed")
        elif omega is None:
            _check(lib().te_build_jk(self.handle, C.c_void_p(D.data_ptr()), C.c_void_p(J.data_ptr()),
                                     C.c_void_p(K.data_ptr()), float(threshold), C.c_void_p(st.cuda_stream)), "te_build_jk")
        else:
            _check(lib().te_build_jk_lr(self.handle, C.c_void_p(D.data_ptr()), C.c_void_p(J.data_ptr()),
                                        C.c_void_p(K.data_ptr()), float(threshold), float(omega),
                                        C.c_void_p(st.cuda_stream)), "te_build_jk_lr")
        return J, K

    def build_j(self, D, J=None, threshold: float = 0.0, stream=None):
        """te_build_j: Coulomb matrix alone by the J-engine route (eq. 35).  Asynchronous on `stream`."""
        import torch
        n = self.basis.nbf
        assert D.is_cuda and D.dtype == torch.float64 and D.is_contiguous() and tuple(D.shape) == (n, n)
        if J is None:
            J = torch.empty_like(D)
        st = stream if stream is not None else torch.cuda.current_stream()
        _check(lib().te_build_j(self.handle, C.c_void_p(D.data_ptr()), C.c_void_p(J.data_ptr()), float(threshold),
                                C.c_void_p(st.cuda_stream)), "te_build_j")
        return J

    def nuclear_attraction(self, xyz_c, q_c, V=None, stream=None):
        """te_nuclear_attraction: V[nbf, nbf] (torch CUDA float64) for host point charges xyz_c[n, 3], q_c[n]."""
        import torch
        n = self.basis.nbf
        xyz_c = np.ascontiguousarray(xyz_c, dtype=np.float64).reshape(-1, 3)
        q_c = np.ascontiguousarray(q_c, dtype=np.float64)
        assert xyz_c.shape[0] == q_c.shape[0]
        if V is None:
            V = torch.empty((n, n), dtype=torch.float64, device="cuda")
        st = stream if stream is not None else torch.cuda.current_stream()
        _check(lib().te_nuclear_attraction(self.handle, int(q_c.shape[0]), _dp(xyz_c), _dp(q_c), C.c_void_p(V.data_ptr()),
                                           C.c_void_p(st.cuda_stream)), "te_nuclear_attraction")
        return V

    def nuclear_attraction_noalloc(self, xyzq, V, stream=None):
        """te_nuclear_attraction_noalloc: charges xyzq[n, 4] and output V[nbf, nbf] are caller-owned torch CUDA float64
        tensors; the call allocates nothing (nbf <= TE_NOALLOC_MAX_NBF = 512) and is asynchronous on `stream`."""
        import torch
        n = self.basis.nbf
        assert xyzq.is_cuda and xyzq.dtype == torch.float64 and xyzq.is_contiguous() and xyzq.dim() == 2 and xyzq.shape[1] == 4
        assert V.is_cuda and V.dtype == torch.float64 and V.is_contiguous() and tuple(V.shape) == (n, n)
        st = stream if stream is not None else torch.cuda.current_stream()
        _check(lib().te_nuclear_attraction_noalloc(self.handle, int(xyzq.shape[0]), C.c_void_p(xyzq.data_ptr()),
                                                   C.c_void_p(V.data_ptr()), C.c_void_p(st.cuda_stream)),
               "te_nuclear_attraction_noalloc")
        return V

    def set_kernel_family(self, family: int):
        _check(lib().te_jk_set_kernel_family(self.handle, int(family)), "te_jk_set_kernel_family")

    def precision_stats(self):
        """(fp64_quartets[10][10], fp32_quartets[10][10]) of the last build (te_jk_precision_stats)."""
        a = np.zeros((NCLASS, NCLASS), dtype=np.int64)
        b = np.zeros((NCLASS, NCLASS), dtype=np.int64)
        _check(lib().te_jk_precision_stats(self.handle, a.ctypes.data_as(C.POINTER(C.c_longlong)),
                                           b.ctypes.data_as(C.POINTER(C.c_longlong))), "te_jk_precision_stats")
        return a, b

    def build_jk_host(self, D: np.ndarray, threshold: float = 0.0, J=None, K=None):
        """te_build_jk_host: HOST numpy (or pinned torch CPU) buffers in, HOST buffers out (synchronous)."""
        n = self.basis.nbf

        def ptr(x):
            return C.cast(x.data_ptr(), C.POINTER(C.c_double)) if hasattr(x, "data_ptr") else _dp(x)
        if not hasattr(D, "data_ptr"):
            D = np.ascontiguousarray(D, dtype=np.float64)
        if J is None:
            J = np.empty((n, n))
        if K is None:
            K = np.empty((n, n))
        _check(lib().te_build_jk_host(self.handle, ptr(D), ptr(J), ptr(K), float(threshold)), "te_build_jk_host")
        return J, K

    def set_profiling(self, on: bool):
        _check(lib().te_jk_set_profiling(self.handle, int(on)), "te_jk_set_profiling")

    def stats(self):
        """(quartets[10][10], ms[10][10]) of the last build (synchronises)."""
        q = np.zeros((NCLASS, NCLASS), dtype=np.int64)
        ms = np.zeros((NCLASS, NCLASS), dtype=np.float32)
        _check(lib().te_jk_stats(self.handle, q.ctypes.data_as(C.POINTER(C.c_longlong)),
                                 ms.ctypes.data_as(C.POINTER(C.c_float))), "te_jk_stats")
        return q, ms

    def screening_stats(self):
        """(visited[10][10], slots[10][10]) of the last build (te_jk_screening_stats)."""
        v = np.zeros((NCLASS, NCLASS), dtype=np.int64)
        s = np.zeros((NCLASS, NCLASS), dtype=np.int64)
        _check(lib().te_jk_screening_stats(self.handle, v.ctypes.data_as(C.POINTER(C.c_longlong)),
                                           s.ctypes.data_as(C.POINTER(C.c_longlong))), "te_jk_screening_stats")
        return v, s

    def close(self):
        if getattr(self, "handle", None):
            lib().te_pairs_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- same names as the C calls --------------------------------------------------------------------------
def te_basis_create(xyz, shell_atom, shell_l, shell_nprim, exponents, coefficients) -> Basis:
    return Basis(xyz, shell_atom, shell_l, shell_nprim, exponents, coefficients)


def te_shellpair_build(basis: Basis, pair_threshold: float) -> Pairs:
    return Pairs(basis, pair_threshold)


def te_build_jk(pairs: Pairs, D, J=None, K=None, threshold: float = 0.0, stream=None):
    return pairs.build_jk(D, J, K, threshold, stream)


def te_build_j(pairs: Pairs, D, J=None, threshold: float = 0.0, stream=None):
    return pairs.build_j(D, J, threshold, stream)


def te_build_jk_lr(pairs: Pairs, D, omega: float, J=None, K=None, threshold: float = 0.0, stream=None):
    return pairs.build_jk(D, J, K, threshold, stream, omega=omega)


def te_build_jk_mixed(pairs: Pairs, D, fp32_below: float = 1e-5, J=None, K=None, threshold: float = 0.0, stream=None):
    return pairs.build_jk(D, J, K, threshold, stream, fp32_below=fp32_below)


def te_nuclear_attraction(pairs: Pairs, xyz_c, q_c, V=None, stream=None):
    return pairs.nuclear_attraction(xyz_c, q_c, V, stream)


def te_eri_block(basis: Basis, quartets):
    return basis.eri_block(quartets)


def te_boys(T, mmax: int):
    """F_0..F_mmax(T) by the device routine; T: 1-D torch CUDA float64 tensor -> [n, mmax+1] tensor."""
    import torch
    assert T.is_cuda and T.dtype == torch.float64 and T.is_contiguous()
    F = torch.empty((T.numel(), mmax + 1), dtype=torch.float64, device=T.device)
    _check(lib().te_boys(T.numel(), C.c_void_p(T.data_ptr()), mmax, C.c_void_p(F.data_ptr())), "te_boys")
    return F


def te_measure_smem_dfma_rate(warps_per_sm: int = 8) -> float:
    v = C.c_double()
    _check(lib().te_measure_smem_dfma_rate(int(warps_per_sm), C.byref(v)), "te_measure_smem_dfma_rate")
    return float(v.value)


def te_measure_fp64_peak() -> float:
    v = C.c_double()
    _check(lib().te_measure_fp64_peak(C.byref(v)), "te_measure_fp64_peak")
    return float(v.value)
