"""ctypes front end of Oracle-B (plain C, oracle/mdwf_oracle.c).  Test infrastructure only.

Same ABI-level interface as oracle.Oracle (numpy Oracle-A); the two are independent
restatements of the paper and are cross-checked in tests/test_oracle_solvers.py (test_oracle_A_vs_B_cross_check).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build


class _Stats(C.Structure):
    _fields_ = [("iters", C.c_int), ("reliable_updates", C.c_int), ("converged", C.c_int),
                ("breakdown", C.c_int), ("inner_applies", C.c_long), ("true_res", C.c_double),
                ("seconds", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.ora_create.restype = C.c_void_p
        L.ora_create.argtypes = [ip, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, ip]
        L.ora_destroy.argtypes = [C.c_void_p]
        L.ora_get_matrix.argtypes = [C.c_void_p, C.c_int, dp]
        L.ora_get_gamma.argtypes = [C.c_void_p, dp]
        L.ora_load_gauge.argtypes = [C.c_void_p, dp, C.c_int]
        L.ora_apply_D.argtypes = [C.c_void_p, dp, dp, C.c_int]
        L.ora_apply_MdagM.argtypes = [C.c_void_p, dp, dp]
        L.ora_apply_A_block.argtypes = [C.c_void_p, dp, dp, C.c_int]
        L.ora_apply_precond.argtypes = [C.c_void_p, dp, dp, C.c_int, C.c_int]
        L.ora_solve.argtypes = [C.c_void_p, dp, dp, C.c_double, C.c_int, C.c_int, C.c_int, C.POINTER(_Stats), dp, C.c_int]
        L.ora_solve.restype = C.c_int
        L.ora_num_threads.restype = C.c_int
        L.ora_num_blocks.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class OracleC:
    def __init__(self, dims, Ls, b, c, M5, mf, block=None):
        self.dims = tuple(int(d) for d in dims)
        self.Ls = int(Ls)
        self.block = tuple(block) if block is not None else self.dims
        d = (C.c_int * 4)(*self.dims)
        B = (C.c_int * 4)(*self.block)
        self._h = lib().ora_create(d, self.Ls, b, c, M5, mf, B)
        if not self._h:
            raise ValueError("ora_create rejected the parameters")
        self.vh = int(np.prod(self.dims)) // 2

    def __del__(self):
        if getattr(self, "_h", None):
            lib().ora_destroy(self._h)
            self._h = None

    @property
    def threads(self):
        return lib().ora_num_threads()

    @property
    def num_blocks(self):
        return lib().ora_num_blocks(self._h)

    def matrix(self, which):
        out = np.empty((self.Ls, self.Ls))
        lib().ora_get_matrix(self._h, {"m5": 0, "mphi": 1, "m5inv": 2}[which], _dp(out))
        return out

    def gamma(self):
        out = np.empty((4, 4, 4, 2))
        lib().ora_get_gamma(self._h, _dp(out))
        return out[..., 0] + 1j * out[..., 1]

    def load_gauge(self, U_abi, t_boundary=-1):
        U = np.ascontiguousarray(U_abi, dtype=np.float64)
        assert U.size == 4 * 2 * self.vh * 18
        lib().ora_load_gauge(self._h, _dp(U), int(t_boundary))

    def _vec(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        assert v.size == self.Ls * self.vh * 24
        return v

    def apply_D(self, in_abi, dagger=False):
        v = self._vec(in_abi)
        out = np.empty_like(v)
        lib().ora_apply_D(self._h, _dp(v), _dp(out), int(dagger))
        return out

    def apply_MdagM(self, in_abi):
        v = self._vec(in_abi)
        out = np.empty_like(v)
        lib().ora_apply_MdagM(self._h, _dp(v), _dp(out))
        return out

    def apply_A_block(self, in_abi, block_index):
        v = self._vec(in_abi)
        out = np.empty_like(v)
        lib().ora_apply_A_block(self._h, _dp(v), _dp(out), int(block_index))
        return out

    def apply_precond(self, r_abi, n_inner, only_block=-1):
        v = self._vec(r_abi)
        out = np.empty_like(v)
        lib().ora_apply_precond(self._h, _dp(v), _dp(out), int(n_inner), int(only_block))
        return out

    def solve(self, b_abi, tol=1e-10, max_iter=100000, use_precond=False, n_inner=6, x0_abi=None, nhist=0):
        b = self._vec(b_abi)
        x = np.zeros_like(b) if x0_abi is None else self._vec(x0_abi).copy()
        st = _Stats()
        hist = np.zeros(max(nhist, 1))
        rc = lib().ora_solve(self._h, _dp(b), _dp(x), tol, max_iter, int(use_precond), n_inner, C.byref(st),
                             _dp(hist), int(nhist))
        stats = {k: getattr(st, k) for k, _ in _Stats._fields_}
        stats["rc"] = rc
        stats["history"] = hist[:min(nhist, st.iters)].copy()
        return x, stats
