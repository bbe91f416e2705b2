"""CPU FP64 oracle (TEST INFRASTRUCTURE ONLY) -- ctypes binding of oracle/te_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It never imports the product package (paper_2406_14920_b200) and shares no code with it.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int),
                                 C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_nbf.argtypes = [C.c_void_p]
        L.orc_nprim.argtypes = [C.c_void_p]
        L.orc_norm_coefs.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.orc_boys.argtypes = [C.c_int, C.c_double, C.POINTER(C.c_double)]
        L.orc_build_pairs.restype = C.c_long
        L.orc_build_pairs.argtypes = [C.c_void_p, C.c_double]
        L.orc_get_pairs.argtypes = [C.c_void_p] + [C.POINTER(C.c_int)] * 5 + [C.POINTER(C.c_double)] * 4
        L.orc_all_bounds.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.orc_jk_o1.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_double, C.POINTER(C.c_double),
                                C.POINTER(C.c_double), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.orc_jk_o2.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_double, C.POINTER(C.c_double),
                                C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.orc_eri_shell_quartet.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.orc_overlap_shell.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.orc_prim_eri_raw.argtypes = ([C.c_int, C.c_double, C.POINTER(C.c_double)] * 4) + [C.POINTER(C.c_double)]
        L.orc_prim_eri_raw_lr.argtypes = ([C.c_int, C.c_double, C.POINTER(C.c_double)] * 4) + [C.c_double, C.POINTER(C.c_double)]
        L.orc_set_omega.argtypes = [C.c_void_p, C.c_double]
        L.orc_density_bounds.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_nuclear_attraction.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                             C.POINTER(C.c_double)]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


CLASS_NAMES = ["SS", "SP", "SD", "SF", "PP", "PD", "PF", "DD", "DF", "FF"]


def boys(mmax: int, T: float) -> np.ndarray:
    """F_0..F_mmax(T), eq. 18."""
    F = np.zeros(mmax + 1)
    lib().orc_boys(mmax, float(T), _dp(F))
    return F


def prim_eri_raw(la, a, A, lb, b, B, lc, c, Cc, ld, d, Dd, omega: float = 0.0) -> np.ndarray:
    """Block of UNNORMALISED primitive integrals (C_mu = 1), shape [nA,nB,nC,nD]: eq. 30, or the
    long-range erf(omega r)/r integrals of eq. 33 when omega > 0."""
    A, B, Cc, Dd = (np.ascontiguousarray(x, dtype=np.float64) for x in (A, B, Cc, Dd))
    out = np.zeros((ncart(la), ncart(lb), ncart(lc), ncart(ld)))
    lib().orc_prim_eri_raw_lr(la, float(a), _dp(A), lb, float(b), _dp(B), lc, float(c), _dp(Cc), ld, float(d), _dp(Dd),
                              float(omega), _dp(out))
    return out


def num_threads() -> int:
    return int(lib().orc_num_threads())


class Oracle:
    """Oracle context for one synth.Problem (or any object with the same array attributes)."""

    def __init__(self, prob):
        self.L = lib()
        self.xyz = np.ascontiguousarray(prob.xyz, dtype=np.float64)
        self.shell_atom = np.ascontiguousarray(prob.shell_atom, dtype=np.int32)
        self.shell_l = np.ascontiguousarray(prob.shell_l, dtype=np.int32)
        self.shell_nprim = np.ascontiguousarray(prob.shell_nprim, dtype=np.int32)
        self.ex = np.ascontiguousarray(prob.exponents, dtype=np.float64)
        self.co = np.ascontiguousarray(prob.coefficients, dtype=np.float64)
        self.ctx = self.L.orc_create(self.xyz.shape[0], _dp(self.xyz), len(self.shell_l), _ip(self.shell_atom),
                                     _ip(self.shell_l), _ip(self.shell_nprim), _dp(self.ex), _dp(self.co))
        if not self.ctx:
            raise ValueError("orc_create failed (l > 3 or empty shell)")
        self.nbf = int(self.L.orc_nbf(self.ctx))
        self.nprim = int(self.L.orc_nprim(self.ctx))
        self.nshells = len(self.shell_l)
        self.npairs = None

    def __del__(self):
        try:
            if getattr(self, "ctx", None):
                self.L.orc_destroy(self.ctx)
                self.ctx = None
        except Exception:
            pass

    def norm_coefs(self) -> np.ndarray:
        ct = np.zeros(self.nprim)
        self.L.orc_norm_coefs(self.ctx, _dp(ct))
        return ct

    def build_pairs(self, tau_pair: float) -> int:
        self.npairs = int(self.L.orc_build_pairs(self.ctx, float(tau_pair)))
        return self.npairs

    def pairs(self) -> dict:
        """Kept pairs in ascending canonical order (class, shellA/primA, shellB/primB)."""
        n = self.npairs
        out = {k: np.zeros(n, dtype=np.int32) for k in ("cls", "shellA", "shellB", "primA", "primB")}
        out["bound"] = np.zeros(n)
        out["P"] = np.zeros((n, 3))
        out["p"] = np.zeros(n)
        out["prefactor"] = np.zeros(n)
        self.L.orc_get_pairs(self.ctx, _ip(out["cls"]), _ip(out["shellA"]), _ip(out["shellB"]), _ip(out["primA"]),
                             _ip(out["primB"]), _dp(out["bound"]), _dp(out["P"]), _dp(out["p"]), _dp(out["prefactor"]))
        return out

    def all_bounds(self) -> np.ndarray:
        """Schwarz bound of every candidate primitive pair, index hi*(hi+1)/2+lo over global primitive ids."""
        q = np.zeros(self.nprim * (self.nprim + 1) // 2)
        self.L.orc_all_bounds(self.ctx, _dp(q))
        return q

    def set_omega(self, omega: float):
        """Operator of the J/K builds: 0 = 1/r, omega > 0 = erf(omega r)/r (eq. 32-33).  Pair lists are unaffected."""
        self.L.orc_set_omega(self.ctx, float(omega))

    def density_bounds(self, D) -> np.ndarray:
        """Dm[X][Y] = max |D| over the block of contracted shells (X,Y)."""
        D = np.ascontiguousarray(D, dtype=np.float64)
        Dm = np.zeros((self.nshells, self.nshells))
        self.L.orc_density_bounds(self.ctx, _dp(D), _dp(Dm))
        return Dm

    def nuclear_attraction(self, xyz_c, q_c) -> np.ndarray:
        """V_mu,nu = sum_C q_C (mu| 1/|r-C| |nu), eq. 14-26, over the kept primitive pairs (build_pairs first)."""
        xyz_c = np.ascontiguousarray(xyz_c, dtype=np.float64).reshape(-1, 3)
        q_c = np.ascontiguousarray(q_c, dtype=np.float64)
        V = np.zeros((self.nbf, self.nbf))
        self.L.orc_nuclear_attraction(self.ctx, len(q_c), _dp(xyz_c), _dp(q_c), _dp(V))
        return V

    def jk_o2(self, D, tau: float):
        """Production oracle: symmetry-unique quartets + per-term screening.  Returns J, K, stats."""
        D = np.ascontiguousarray(D, dtype=np.float64)
        J = np.zeros((self.nbf, self.nbf))
        K = np.zeros((self.nbf, self.nbf))
        st = np.zeros(3, dtype=np.int64)
        self.L.orc_jk_o2(self.ctx, _dp(D), float(tau), _dp(J), _dp(K), st.ctypes.data_as(C.POINTER(C.c_longlong)))
        return J, K, {"live_quartets": int(st[0]), "visited": int(st[1]), "borderline": int(st[2])}

    def jk_o1(self, D, tau: float, do_j=True, do_k=True, braA=-1, braB=-1, ketC=-1):
        """Definition oracle (eq. 34 / 36 over ordered primitive pairs, no symmetry)."""
        D = np.ascontiguousarray(D, dtype=np.float64)
        J = np.zeros((self.nbf, self.nbf))
        K = np.zeros((self.nbf, self.nbf))
        self.L.orc_jk_o1(self.ctx, _dp(D), float(tau), _dp(J), _dp(K), int(do_j), int(do_k), braA, braB, ketC)
        return J, K

    def shell_offsets(self) -> np.ndarray:
        off = np.zeros(self.nshells + 1, dtype=np.int64)
        off[1:] = np.cumsum([ncart(int(l)) for l in self.shell_l])
        return off

    def j_block(self, D, tau, A, B) -> np.ndarray:
        """J block of contracted shells (A,B) summed over ALL partners with the same per-term rule."""
        J, _ = self.jk_o1(D, tau, do_j=True, do_k=False, braA=A, braB=B)
        o = self.shell_offsets()
        return J[o[A]:o[A + 1], o[B]:o[B + 1]].copy()

    def k_block(self, D, tau, A, Cc) -> np.ndarray:
        _, K = self.jk_o1(D, tau, do_j=False, do_k=True, braA=A, ketC=Cc)
        o = self.shell_offsets()
        return K[o[A]:o[A + 1], o[Cc]:o[Cc + 1]].copy()

    def eri_shell_quartet(self, A, B, Cc, Dd) -> np.ndarray:
        shp = tuple(ncart(int(self.shell_l[s])) for s in (A, B, Cc, Dd))
        out = np.zeros(shp)
        self.L.orc_eri_shell_quartet(self.ctx, A, B, Cc, Dd, _dp(out))
        return out

    def overlap(self) -> np.ndarray:
        """Full overlap matrix by eq. 11."""
        o = self.shell_offsets()
        S = np.zeros((self.nbf, self.nbf))
        for A in range(self.nshells):
            for B in range(self.nshells):
                blk = np.zeros((o[A + 1] - o[A], o[B + 1] - o[B]))
                self.L.orc_overlap_shell(self.ctx, A, B, _dp(blk))
                S[o[A]:o[A + 1], o[B]:o[B + 1]] = blk
        return S
