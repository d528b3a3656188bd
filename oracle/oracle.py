"""ctypes wrapper around oracle/msm_oracle.c (plain C, fp64). TEST INFRASTRUCTURE.

Argument marshalling only; every formula lives in msm_oracle.c with its PAPER.md citation.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "msm_oracle.c")
_SO = os.path.join(_HERE, "libmsm_oracle.so")
_lib = None


class _Params(C.Structure):
    _fields_ = [("box", C.c_double * 3), ("periodic", C.c_int * 3), ("h", C.c_double),
                ("a", C.c_double), ("p", C.c_int), ("levels", C.c_int), ("mu", C.c_int), ("pad", C.c_int)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp, no -ffast-math)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        d, i, p = C.c_double, C.c_int, C.c_void_p
        dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
        ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
        L = _lib
        for name in ("msmo_gamma", "msmo_dgamma"):
            getattr(L, name).restype = d; getattr(L, name).argtypes = [i, d]
        for name in ("msmo_kernel", "msmo_dkernel"):
            getattr(L, name).restype = d; getattr(L, name).argtypes = [i, d, i, i, d]
        for name in ("msmo_bspline", "msmo_dbspline"):
            getattr(L, name).restype = d; getattr(L, name).argtypes = [i, d]
        L.msmo_two_scale.argtypes = [i, dp]
        L.msmo_omega.restype = i; L.msmo_omega.argtypes = [i, i, dp]
        L.msmo_create.restype = p; L.msmo_create.argtypes = [C.POINTER(_Params), C.POINTER(i)]
        L.msmo_destroy.argtypes = [p]
        L.msmo_num_levels.restype = i; L.msmo_num_levels.argtypes = [p]
        L.msmo_omega_halfwidth.restype = i; L.msmo_omega_halfwidth.argtypes = [p]
        L.msmo_level_info.argtypes = [p, i, ip, ip, dp, ip]
        L.msmo_copy_grid.argtypes = [p, i, i, dp]
        L.msmo_copy_stencil.restype = i; L.msmo_copy_stencil.argtypes = [p, i, i, dp]
        L.msmo_anterpolate.argtypes = [p, i, dp, dp]
        L.msmo_interpolate.argtypes = [p, i, dp, dp, dp, dp]
        L.msmo_restrict.argtypes = [p, i]
        L.msmo_prolong_add.argtypes = [p, i]
        L.msmo_apply_stencil.argtypes = [p, i, i, dp, dp]
        L.msmo_short_range_brute.argtypes = [p, i, dp, dp, i, C.c_void_p, dp, dp, C.c_void_p]
        L.msmo_short_range_cells.argtypes = [p, i, dp, dp, dp, dp, C.c_void_p]
        L.msmo_grid_pass.argtypes = [p, C.c_void_p]
        L.msmo_set_grid.argtypes = [p, i, i, dp]
        L.msmo_evaluate.restype = i
        L.msmo_evaluate.argtypes = [p, i, dp, dp, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.msmo_direct_sum.restype = d
        L.msmo_direct_sum.argtypes = [i, dp, dp, dp, ip, i, C.c_void_p, C.c_void_p]
    return _lib


# ------------------------------------------------------------------ scalar functions

def gamma(p, rho): return lib().msmo_gamma(p, float(rho))
def dgamma(p, rho): return lib().msmo_dgamma(p, float(rho))
def kernel(p, a, L, l, r): return lib().msmo_kernel(p, float(a), L, l, float(r))
def dkernel(p, a, L, l, r): return lib().msmo_dkernel(p, float(a), L, l, float(r))
def bspline(p, u): return lib().msmo_bspline(p, float(u))
def dbspline(p, u): return lib().msmo_dbspline(p, float(u))


def two_scale(p):
    out = np.zeros(p + 1)
    lib().msmo_two_scale(p, out)
    return out


def omega(p, mu):
    out = np.zeros(2 * (p // 2 - 1 + mu) + 1)
    lib().msmo_omega(p, mu, out)
    return out


def direct_sum(pos, q, box=(1.0, 1.0, 1.0), periodic=(0, 0, 0), nimg=0, want_fv=True):
    pos = np.ascontiguousarray(pos, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
    n = len(q)
    F = np.zeros((n, 3)); V = np.zeros(n)
    U = lib().msmo_direct_sum(n, pos, q, np.asarray(box, dtype=np.float64),
                              np.asarray(periodic, dtype=np.int32), int(nimg),
                              F.ctypes.data if want_fv else None, V.ctypes.data if want_fv else None)
    return U, F, V


# ------------------------------------------------------------------ the method

class Oracle:
    """One MSM setup (the analogue of msm_plan_create on the CUDA side)."""

    def __init__(self, box, periodic, h, a, p, levels, mu=4, pad=0):
        """pad: extra grid nodes on both sides of every open axis at every level (the pin of
        reading G3: no output may depend on it beyond round-off)."""
        prm = _Params()
        prm.pad = int(pad)
        prm.box[:] = [float(b) for b in box]
        prm.periodic[:] = [int(b) for b in periodic]
        prm.h, prm.a, prm.p, prm.levels, prm.mu = float(h), float(a), int(p), int(levels), int(mu)
        st = C.c_int(0)
        self._ctx = lib().msmo_create(C.byref(prm), C.byref(st))
        if not self._ctx:
            raise ValueError(f"oracle setup failed with status {st.value}")
        self.p, self.a, self.mu = int(p), float(a), int(mu)
        self.L = lib().msmo_num_levels(self._ctx)
        self.w = lib().msmo_omega_halfwidth(self._ctx)

    def __del__(self):
        if getattr(self, "_ctx", None):
            lib().msmo_destroy(self._ctx); self._ctx = None

    def level_info(self, l):
        M = np.zeros(3, np.int32); lo = np.zeros(3, np.int32); h = np.zeros(3); Kr = np.zeros(3, np.int32)
        lib().msmo_level_info(self._ctx, l, M, lo, h, Kr)
        return {"M": tuple(int(v) for v in M), "lo": tuple(int(v) for v in lo),
                "h": tuple(float(v) for v in h), "Kr": tuple(int(v) for v in Kr)}

    def grid(self, l, kind):
        """kind 'Q' or 'E' of the last evaluate; array indexed [z, y, x]."""
        M = self.level_info(l)["M"]
        out = np.zeros((M[2], M[1], M[0]))
        lib().msmo_copy_grid(self._ctx, l, 0 if kind == "Q" else 1, out)
        return out

    def set_grid(self, l, kind, arr):
        lib().msmo_set_grid(self._ctx, l, 0 if kind == "Q" else 1, np.ascontiguousarray(arr, dtype=np.float64))

    def stencil(self, l, kind=0):
        """kind 0: K^l; 1..6: strain derivatives xx yy zz xy xz yz. Indexed [dz, dy, dx] + Kr."""
        Kr = self.level_info(l)["Kr"]
        out = np.zeros((2 * Kr[2] + 1, 2 * Kr[1] + 1, 2 * Kr[0] + 1))
        if lib().msmo_copy_stencil(self._ctx, l, kind, out):
            raise ValueError("no stencil at this level")
        return out

    def anterpolate(self, pos, q):
        pos = np.ascontiguousarray(pos, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
        lib().msmo_anterpolate(self._ctx, len(q), pos, q)
        return self.grid(1, "Q")

    def restrict(self, l):
        lib().msmo_restrict(self._ctx, l)
        return self.grid(l + 1, "Q")

    def prolong_add(self, l):
        lib().msmo_prolong_add(self._ctx, l)
        return self.grid(l, "E")

    def apply_stencil(self, l, q, kind=0):
        q = np.ascontiguousarray(q, dtype=np.float64)
        out = np.zeros_like(q)
        lib().msmo_apply_stencil(self._ctx, l, kind, q, out)
        return out

    def grid_pass(self, want_virial=False):
        W = np.zeros(6)
        lib().msmo_grid_pass(self._ctx, W.ctypes.data if want_virial else None)
        return W

    def interpolate(self, pos, q):
        pos = np.ascontiguousarray(pos, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
        F = np.zeros((len(q), 3)); V = np.zeros(len(q))
        lib().msmo_interpolate(self._ctx, len(q), pos, q, F, V)
        return F, V

    def short_range(self, pos, q, sel=None, method="brute", want_virial=True):
        pos = np.ascontiguousarray(pos, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
        n = len(q)
        W = np.zeros(6)
        wp = W.ctypes.data if want_virial else None
        if method == "cells":
            F = np.zeros((n, 3)); V = np.zeros(n)
            lib().msmo_short_range_cells(self._ctx, n, pos, q, F, V, wp)
        else:
            if sel is None:
                F = np.zeros((n, 3)); V = np.zeros(n)
                lib().msmo_short_range_brute(self._ctx, n, pos, q, 0, None, F, V, wp)
            else:
                sel = np.ascontiguousarray(sel, dtype=np.int32)
                F = np.zeros((len(sel), 3)); V = np.zeros(len(sel))
                lib().msmo_short_range_brute(self._ctx, n, pos, q, len(sel), sel.ctypes.data, F, V, wp)
        return F, V, W

    def evaluate(self, pos, q, want_virial=True):
        """-> dict(energy, forces (n,3), potentials (n,), virial (6,) or None)."""
        pos = np.ascontiguousarray(pos, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
        n = len(q)
        F = np.zeros((n, 3)); V = np.zeros(n); U = C.c_double(0.0); W = np.zeros(6)
        st = lib().msmo_evaluate(self._ctx, n, pos, q, F.ctypes.data, V.ctypes.data, C.addressof(U),
                                 W.ctypes.data if want_virial else None)
        if st:
            raise ValueError(f"oracle evaluate failed with status {st}")
        return {"energy": U.value, "forces": F, "potentials": V, "virial": W if want_virial else None}
