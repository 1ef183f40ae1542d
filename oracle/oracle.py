"""ctypes wrapper over oracle/alora_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this.  It imports nothing from the CUDA path.  ``build()`` compiles the C file with gcc (plain C,
-O2, no OpenMP: the oracle runs on exactly one thread).

Part 1 (quantities with a plain definition) lives in the C file, one function per definition;
Part 2 (the ALORA iteration, Algorithm 1) lives in oracle/alm.py.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "alora_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Prob(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("m", C.c_int64),
        ("nnzC", C.c_int64), ("C_row", C.c_void_p), ("C_col", C.c_void_p), ("C_val", C.c_void_p),
        ("pC", C.c_int32), ("C_U", C.c_void_p), ("C_s", C.c_void_p),
        ("nnzA", C.c_int64), ("A_ptr", C.c_void_p), ("A_row", C.c_void_p), ("A_col", C.c_void_p),
        ("A_val", C.c_void_p), ("b", C.c_void_p),
    ]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_f.restype = C.c_double
        _lib.oracle_inner_C.restype = C.c_double
        _lib.oracle_normC_sq.restype = C.c_double
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """Holds one problem (inputs.Problem-shaped object) and evaluates the definitions on it."""

    def __init__(self, prob):
        self.lib = _load()
        self.n, self.m = int(prob.n), int(prob.m)
        k = self._keep = {}
        k["C_row"] = np.ascontiguousarray(prob.C_row, np.int32)
        k["C_col"] = np.ascontiguousarray(prob.C_col, np.int32)
        k["C_val"] = _f64(prob.C_val)
        k["A_ptr"] = np.ascontiguousarray(prob.A_ptr, np.int64)
        k["A_row"] = np.ascontiguousarray(prob.A_row, np.int32)
        k["A_col"] = np.ascontiguousarray(prob.A_col, np.int32)
        k["A_val"] = _f64(prob.A_val)
        k["b"] = _f64(prob.b)
        pC = 0 if getattr(prob, "C_s", None) is None else int(len(prob.C_s))
        if pC:
            k["C_U"] = np.asfortranarray(prob.C_U, dtype=np.float64)  # n x pC column-major
            k["C_s"] = _f64(prob.C_s)
        self.b = k["b"]
        self.P = _Prob(
            n=self.n, m=self.m, nnzC=len(k["C_val"]), C_row=_p(k["C_row"]), C_col=_p(k["C_col"]),
            C_val=_p(k["C_val"]), pC=pC, C_U=_p(k["C_U"]) if pC else None,
            C_s=_p(k["C_s"]) if pC else None, nnzA=len(k["A_val"]), A_ptr=_p(k["A_ptr"]),
            A_row=_p(k["A_row"]), A_col=_p(k["A_col"]), A_val=_p(k["A_val"]), b=_p(k["b"]))
        self._normC = None

    # --- Part 1: definitions -------------------------------------------------------------
    def A_op(self, R):
        """z = A(RR^T)."""
        R = _f64(R); z = np.empty(self.m)
        self.lib.oracle_A_op(C.byref(self.P), _p(R), C.c_int32(R.shape[1]), _p(z))
        return z

    def A_sym(self, X, Y):
        """<A_i, XY^T + YX^T>/2 for every i."""
        X, Y = _f64(X), _f64(Y); out = np.empty(self.m)
        self.lib.oracle_A_sym(C.byref(self.P), _p(X), _p(Y), C.c_int32(X.shape[1]), _p(out))
        return out

    def inner_C(self, X, Y):
        X, Y = _f64(X), _f64(Y)
        return float(self.lib.oracle_inner_C(C.byref(self.P), _p(X), _p(Y), C.c_int32(X.shape[1])))

    def f(self, y, sigma, R, parts=False):
        """f(R) of (AL-BM).  parts=True -> dict(cx, yq, qq, f)."""
        y, R = _f64(y), _f64(R); out = np.empty(4)
        v = float(self.lib.oracle_f(C.byref(self.P), _p(y), C.c_double(sigma), _p(R),
                                    C.c_int32(R.shape[1]), _p(out)))
        return dict(cx=out[0], yq=out[1], qq=out[2], f=out[3]) if parts else v

    def lam(self, y, sigma, R):
        """lambda = y - sigma (A(RR^T) - b);  returns (lambda, z)."""
        y, R = _f64(y), _f64(R); lam = np.empty(self.m); z = np.empty(self.m)
        self.lib.oracle_lambda(C.byref(self.P), _p(y), C.c_double(sigma), _p(R), C.c_int32(R.shape[1]),
                               _p(lam), _p(z))
        return lam, z

    def grad(self, y, sigma, R):
        """nabla f(R) = 2 (C - A^*(lambda)) R."""
        y, R = _f64(y), _f64(R); G = np.empty_like(R)
        self.lib.oracle_grad(C.byref(self.P), _p(y), C.c_double(sigma), _p(R), C.c_int32(R.shape[1]), _p(G))
        return G

    def linesearch(self, y, sigma, R, D):
        """p0..p4 of alpha -> f(R + alpha D)."""
        y, R, D = _f64(y), _f64(R), _f64(D); p = np.empty(5)
        self.lib.oracle_linesearch(C.byref(self.P), _p(y), C.c_double(sigma), _p(R), _p(D),
                                   C.c_int32(R.shape[1]), _p(p))
        return p

    def smatvec(self, w, V):
        """(C - A^*(w)) V,  V is [n] or [n,p]."""
        w = _f64(w); V = _f64(V)
        V2 = V.reshape(self.n, -1); W = np.empty_like(V2)
        self.lib.oracle_smatvec(C.byref(self.P), _p(w), _p(V2), C.c_int32(V2.shape[1]), _p(W))
        return W.reshape(V.shape)

    def normC(self):
        """||C||_F with duplicate COO entries summed first (they denote one matrix entry)."""
        if self._normC is None:
            k = self._keep
            key = k["C_row"].astype(np.int64) * self.n + k["C_col"]
            uniq, inv = np.unique(key, return_inverse=True)
            val = np.bincount(inv, weights=k["C_val"], minlength=len(uniq)) if len(uniq) else np.zeros(0)
            rows = np.ascontiguousarray(uniq // self.n, np.int32)
            cols = np.ascontiguousarray(uniq % self.n, np.int32)
            val = _f64(val)
            P2 = _Prob.from_buffer_copy(self.P)
            P2.nnzC, P2.C_row, P2.C_col, P2.C_val = len(val), _p(rows), _p(cols), _p(val)
            self._normC = float(np.sqrt(max(0.0, self.lib.oracle_normC_sq(C.byref(P2)))))
        return self._normC
