"""CPU oracle for Fourier-accelerated Landau gauge fixing (arXiv 1301.3460).

TEST INFRASTRUCTURE ONLY.  May be imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  The product (paper_1301_3460_b200)
never imports this package, and this package never imports the product.

Thin ctypes wrapper over oracle/lgf_oracle.cpp (see its header for the algorithm, the
passages it follows and its pins).  Arrays are complex128 numpy arrays:
links [V,4,3,3], matrix fields [V,3,3], scalar complex fields [V]; x0 fastest.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        P = C.c_void_p
        D = C.POINTER(C.c_double)
        I4 = C.POINTER(C.c_int)
        L.orc_create.restype = P
        L.orc_create.argtypes = [I4, C.c_int, C.c_int]
        L.orc_destroy.argtypes = [P]
        L.orc_set_variant.argtypes = [P, C.c_int, C.c_int]
        L.orc_set_gauge.argtypes = [P, C.c_int]
        L.orc_load.argtypes = [P, P]
        L.orc_get.argtypes = [P, P]
        L.orc_measure.argtypes = [P, D, D]
        L.orc_delta.argtypes = [P, P]
        L.orc_fa_field.argtypes = [P, P]
        L.orc_g_field.argtypes = [P, C.c_double, P]
        L.orc_F_of_g.restype = C.c_double
        L.orc_F_of_g.argtypes = [P, P]
        L.orc_iterate.argtypes = [P, C.c_int, C.c_double, D, D]
        L.orc_fix.restype = C.c_int
        L.orc_fix.argtypes = [P, C.c_double, C.c_double, C.c_int, C.POINTER(C.c_int), D, D, P]
        L.orc_plaquette.restype = C.c_double
        L.orc_plaquette.argtypes = [P]
        L.orc_unitarity.argtypes = [P, D, D]
        L.orc_dft4.argtypes = [I4, P, P, C.c_int, C.c_int]
        L.orc_fa_weights.argtypes = [I4, P]
        L.orc_project.argtypes = [C.c_long, P, C.c_double, P]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _dims(dims):
    d = (C.c_int * 4)(*[int(v) for v in dims])
    return d


def _c128(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


class Oracle:
    """One lattice; mirrors the C ABI of include/lgf.h (create/load/iterate/fix/get/measure)."""

    def __init__(self, dims, storage: int = 18, fft_mode: int = 0):
        self.dims = tuple(int(v) for v in dims)
        self.V = int(np.prod(self.dims))
        self.storage = storage
        self._h = lib().orc_create(_dims(self.dims), storage, fft_mode)
        if not self._h:
            raise ValueError("orc_create failed")

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_destroy(self._h)
            self._h = None

    def set_variant(self, accel: int = 1, exp_sign: int = -1):
        lib().orc_set_variant(self._h, accel, exp_sign)

    def set_gauge(self, nd: int = 4):
        """nd = 4 Landau gauge (the paper); nd = 3 Coulomb gauge (gauge condition over mu = 0..2 only)."""
        lib().orc_set_gauge(self._h, nd)

    def load(self, U):
        U = _c128(U)
        assert U.shape == (self.V, 4, 3, 3)
        lib().orc_load(self._h, U.ctypes.data)

    def get(self):
        U = np.empty((self.V, 4, 3, 3), dtype=np.complex128)
        lib().orc_get(self._h, U.ctypes.data)
        return U

    def measure(self):
        F = C.c_double()
        th = C.c_double()
        lib().orc_measure(self._h, C.byref(F), C.byref(th))
        return F.value, th.value

    def _field(self, fn, *args):
        X = np.empty((self.V, 3, 3), dtype=np.complex128)
        fn(self._h, *args, X.ctypes.data)
        return X

    def delta(self):
        return self._field(lib().orc_delta)

    def fa_field(self):
        return self._field(lib().orc_fa_field)

    def g_field(self, alpha):
        return self._field(lib().orc_g_field, float(alpha))

    def F_of_g(self, g):
        g = _c128(g)
        assert g.shape == (self.V, 3, 3)
        return lib().orc_F_of_g(self._h, g.ctypes.data)

    def iterate(self, n, alpha):
        F = C.c_double()
        th = C.c_double()
        lib().orc_iterate(self._h, int(n), float(alpha), C.byref(F), C.byref(th))
        return F.value, th.value

    def fix(self, alpha, theta_tol, max_iter, history: bool = False):
        F = C.c_double()
        th = C.c_double()
        n = C.c_int()
        hist = np.zeros((max_iter + 1, 2)) if history else None
        st = lib().orc_fix(self._h, float(alpha), float(theta_tol), int(max_iter), C.byref(n), C.byref(F), C.byref(th),
                           hist.ctypes.data if history else None)
        out = dict(status=st, n_iter=n.value, F=F.value, theta=th.value)
        if history:
            out["history"] = hist[: n.value + 1]
        return out

    def plaquette(self):
        return lib().orc_plaquette(self._h)

    def unitarity(self):
        a = C.c_double()
        b = C.c_double()
        lib().orc_unitarity(self._h, C.byref(a), C.byref(b))
        return a.value, b.value


def dft4(dims, f, sign: int = -1, fft_mode: int = 0):
    f = _c128(f).reshape(-1)
    out = np.empty_like(f)
    lib().orc_dft4(_dims(dims), f.ctypes.data, out.ctypes.data, int(sign), int(fft_mode))
    return out


def fa_weights(dims):
    w = np.empty(int(np.prod(dims)), dtype=np.float64)
    lib().orc_fa_weights(_dims(dims), w.ctypes.data)
    return w


def project(X, alpha):
    X = _c128(X)
    g = np.empty_like(X)
    lib().orc_project(X.shape[0], X.ctypes.data, float(alpha), g.ctypes.data)
    return g


def num_threads():
    return lib().orc_num_threads()
