"""Thin ctypes binding over the C ABI of include/alora.h (csrc/libalora.so).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.  Device
buffers are torch tensors (PyTorch is used for device memory and streams, nothing else); the
binding passes ``tensor.data_ptr()``.  There is no CPU fallback: if the shared library is missing
the import of this module fails, and without a CUDA device ``Context(...)`` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libalora.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} not found: build it with `python -m paper_2505_15775_b200.build` "
        "(there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENOTCONV = range(6)
F32, F64 = 0, 1


class AloraError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"alora status {status} ({_lib.alora_strerror(status).decode()}): {msg}")
        self.status = status


class _Problem(C.Structure):
    _fields_ = [("n", C.c_int64), ("m", C.c_int64), ("nnzC", C.c_int64), ("C_row", C.c_void_p),
                ("C_col", C.c_void_p), ("C_val", C.c_void_p), ("pC", C.c_int32), ("C_U", C.c_void_p),
                ("C_s", C.c_void_p), ("nnzA", C.c_int64), ("A_ptr", C.c_void_p), ("A_row", C.c_void_p),
                ("A_col", C.c_void_p), ("A_val", C.c_void_p), ("b", C.c_void_p)]


class Params(C.Structure):
    """alora_params (include/alora.h); defaults from alora_default_params."""
    _fields_ = [("eps", C.c_double), ("stop_mode", C.c_int32), ("T_max", C.c_int32), ("tol0", C.c_double),
                ("c_in", C.c_double), ("tol_min", C.c_double), ("it_max", C.c_int32), ("lbfgs_mem", C.c_int32),
                ("p_max", C.c_int32), ("k_max", C.c_int32), ("tau_neg", C.c_double), ("tol_eig", C.c_double),
                ("gamma", C.c_double), ("kappa", C.c_double), ("sigma_max", C.c_double),
                ("tau_shrink", C.c_double), ("s_max", C.c_double), ("seed", C.c_uint64),
                ("stall_tol", C.c_double), ("stall_iters", C.c_int32), ("pad_", C.c_int32)]

    def __init__(self, **kw):
        super().__init__()
        _lib.alora_default_params(C.byref(self))
        for k, v in kw.items():
            if not hasattr(self, k):
                raise AttributeError(k)
            setattr(self, k, v)


    @classmethod
    def preset(cls, dtype, **kw):
        """alora_preset_params for the context dtype (F32: bounded inexact inner solves), then overrides."""
        p = cls()
        _lib.alora_preset_params(C.byref(p), {"f32": F32, "f64": F64, F32: F32, F64: F64}[dtype])
        for k, v in kw.items():
            if not hasattr(p, k):
                raise AttributeError(k)
            setattr(p, k, v)
        return p


class IterRecord(C.Structure):
    _fields_ = [("t", C.c_int32), ("r", C.c_int32), ("inner_iters", C.c_int32), ("n_evals", C.c_int32),
                ("lanczos_steps", C.c_int32), ("grew", C.c_int32), ("shrank", C.c_int32), ("pad_", C.c_int32),
                ("sigma", C.c_double), ("cx", C.c_double), ("f", C.c_double), ("qnorm", C.c_double),
                ("gnorm", C.c_double), ("theta1", C.c_double), ("kkt", C.c_double * 3)]


class Result(C.Structure):
    _fields_ = [("converged", C.c_int32), ("outer_iters", C.c_int32), ("n_evals", C.c_int32),
                ("n_linesearch", C.c_int32), ("n_matvec", C.c_int32), ("r_final", C.c_int32),
                ("kkt", C.c_double * 3), ("sigma_final", C.c_double), ("seconds", C.c_double)]


_lib.alora_strerror.restype = C.c_char_p
_lib.alora_strerror.argtypes = [C.c_int]
_lib.alora_last_error.restype = C.c_char_p
_lib.alora_last_error.argtypes = [C.c_void_p]
_lib.alora_destroy.restype = None
_lib.alora_destroy.argtypes = [C.c_void_p]
_lib.alora_default_params.restype = None
_lib.alora_preset_params.restype = None
_lib.alora_preset_params.argtypes = [C.c_void_p, C.c_int]
_vp, _i32, _i64, _dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
_lib.alora_create.argtypes = [C.POINTER(_Problem), C.c_int, C.c_int, _vp, C.POINTER(_vp)]
_lib.alora_info.argtypes = [_vp, _vp]
_lib.alora_set_dual.argtypes = [_vp, _vp, _dbl]
_lib.alora_eval.argtypes = [_vp, _vp, _i32, _i64, _vp, _vp, _vp]
_lib.alora_get_stats.argtypes = [_vp, _vp]
_lib.alora_get_lambda.argtypes = [_vp, _vp]
_lib.alora_dual_terms.argtypes = [_vp, _vp, _vp, _vp]
_lib.alora_rowdots.argtypes = [_vp, _vp, _vp, _i64, _i32, _i64, _vp]
_lib.alora_rowdots_static.argtypes = [_vp, _vp, _vp, _i64, _i32, _i64, _vp]
ROWDOTS_STATIC_MAX_ELEMS = 1 << 26   # ALORA_ROWDOTS_STATIC_MAX_ELEMS
_lib.alora_eval_host.argtypes = [_vp, _vp, _i32, _i64, _vp, _vp, _vp]
_lib.alora_step_host.argtypes = [_vp, _vp, _vp, _vp, _i32, _i64, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.alora_linesearch.argtypes = [_vp, _vp, _vp, _i32, _i64, _i32, _vp]
_lib.alora_get_linesearch.argtypes = [_vp, _vp]
_lib.alora_smatvec.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp]
_lib.alora_kernel_timing.argtypes = [_vp, C.c_int]
_lib.alora_kernel_timing_read.argtypes = [_vp, _vp, _vp]
_lib.alora_lanczos.argtypes = [_vp, _vp, _i32, _dbl, C.c_uint64, _i32, _vp, _vp, _vp, _vp, _vp]
_lib.alora_solve.argtypes = [_vp, C.POINTER(Params), _vp, _vp, _i32, _vp, _vp, _vp, _i32, _vp]


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _ptr(t):
    """device/host pointer of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


class Context:
    """alora_ctx: one per (problem, dtype, device, stream).  `problem` is an inputs.Problem-shaped
    object with host numpy arrays (sym-upper COO)."""

    def __init__(self, problem, dtype, device: int = 0, stream: int | None = None):
        self._h = None
        dt = {"f32": F32, "f64": F64, F32: F32, F64: F64}[dtype]
        self.dtype = dt
        k = {}
        k["C_row"], k["C_col"] = _np(problem.C_row, np.int32), _np(problem.C_col, np.int32)
        k["C_val"] = _np(problem.C_val, np.float64)
        k["A_ptr"] = _np(problem.A_ptr, np.int64)
        k["A_row"], k["A_col"] = _np(problem.A_row, np.int32), _np(problem.A_col, np.int32)
        k["A_val"], k["b"] = _np(problem.A_val, np.float64), _np(problem.b, np.float64)
        pC = 0 if getattr(problem, "C_s", None) is None else len(problem.C_s)
        if pC:
            k["C_U"] = np.asfortranarray(problem.C_U, dtype=np.float64)
            k["C_s"] = _np(problem.C_s, np.float64)
        P = _Problem(n=problem.n, m=problem.m, nnzC=len(k["C_val"]), C_row=k["C_row"].ctypes.data,
                     C_col=k["C_col"].ctypes.data, C_val=k["C_val"].ctypes.data, pC=pC,
                     C_U=k["C_U"].ctypes.data if pC else None, C_s=k["C_s"].ctypes.data if pC else None,
                     nnzA=len(k["A_val"]), A_ptr=k["A_ptr"].ctypes.data, A_row=k["A_row"].ctypes.data,
                     A_col=k["A_col"].ctypes.data, A_val=k["A_val"].ctypes.data, b=k["b"].ctypes.data)
        if stream is None:
            import torch
            stream = torch.cuda.current_stream(device).cuda_stream if torch.cuda.is_available() else 0
        h = _vp()
        st = _lib.alora_create(C.byref(P), dt, device, _vp(stream), C.byref(h))
        if st != OK:
            raise AloraError(st, _lib.alora_last_error(None).decode())
        self._h = h
        self.n, self.m = int(problem.n), int(problem.m)
        self._keep = None  # tensors the library reads later (y)

    def close(self):
        if self._h:
            _lib.alora_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, st, allow=()):
        if st != OK and st not in allow:
            raise AloraError(st, _lib.alora_last_error(self._h).decode())
        return st

    def info(self):
        a = np.zeros(16, np.int64)
        self._chk(_lib.alora_info(self._h, a.ctypes.data))
        keys = ["cls", "n", "m", "c_nnz", "a_nnz", "nf_A", "nlong", "launches", "dev_bytes", "num_sms", "nf_C"]
        return dict(zip(keys, (int(v) for v in a)))

    def set_dual(self, y, sigma: float):
        self._keep = y
        self._chk(_lib.alora_set_dual(self._h, _ptr(y), float(sigma)))

    def eval(self, R, r: int, ld: int, G=None, z=None, stats: bool = True):
        out = np.zeros(8) if stats else None
        self._chk(_lib.alora_eval(self._h, _ptr(R), r, ld, _ptr(G), _ptr(z), _ptr(out)))
        return out

    def get_stats(self):
        out = np.zeros(8)
        self._chk(_lib.alora_get_stats(self._h, out.ctypes.data))
        return out

    def get_lambda(self, lam):
        self._chk(_lib.alora_get_lambda(self._h, _ptr(lam)))

    def dual_terms(self, z, lam=None):
        """(y.q, ||q||^2, lambda.z) for a caller-supplied device z (q = z - b); lam (device, m) receives lambda."""
        out = np.zeros(3)
        self._chk(_lib.alora_dual_terms(self._h, _ptr(z), _ptr(lam), out.ctypes.data))
        return out

    def rowdots(self, X, Y, n_rows: int, r: int, ld: int):
        """(sum X^2, sum X Y) over the first n_rows rows."""
        out = np.zeros(2)
        self._chk(_lib.alora_rowdots(self._h, _ptr(X), _ptr(Y), n_rows, r, ld, out.ctypes.data))
        return out

    def rowdots_static(self, X, Y, n_rows: int, r: int, ld: int, out):
        """alora_rowdots_static: the same two sums into `out` (device fp64[2]); allocates nothing, does not synchronise."""
        self._chk(_lib.alora_rowdots_static(self._h, _ptr(X), _ptr(Y), n_rows, r, ld, _ptr(out)))

    def eval_host(self, R_host, r: int, ld: int, G_host=None, z_host=None):
        out = np.zeros(8)
        self._chk(_lib.alora_eval_host(self._h, _ptr(R_host), r, ld, _ptr(G_host), _ptr(z_host), out.ctypes.data))
        return out

    def step_host(self, R_host, D_host, V_host, r: int, ld: int, G_host=None, z_host=None, W_host=None):
        """One whole step (f + grad, line-search coefficients, S(lambda) V) through HOST buffers.
        Returns (stats[8], p[5], <V,W>)."""
        st, p, vw = np.zeros(8), np.zeros(5), C.c_double()
        self._chk(_lib.alora_step_host(self._h, _ptr(R_host), _ptr(D_host), _ptr(V_host), r, ld, _ptr(G_host), _ptr(z_host),
                                       _ptr(W_host), st.ctypes.data, p.ctypes.data, C.addressof(vw)))
        return st, p, vw.value

    def linesearch(self, R, D, r: int, ld: int, fetch: bool = True, warm: bool = False):
        """warm=True: the ctx still holds an alora_eval of this same R (same tensor, r, ld, dual)."""
        out = np.zeros(5) if fetch else None
        self._chk(_lib.alora_linesearch(self._h, _ptr(R), _ptr(D), r, ld, 1 if warm else 0, _ptr(out)))
        return out

    def get_linesearch(self):
        out = np.zeros(5)
        self._chk(_lib.alora_get_linesearch(self._h, out.ctypes.data))
        return out

    def smatvec(self, mu, V, p: int, W, fetch: bool = True):
        out = np.zeros(1) if fetch else None
        self._chk(_lib.alora_smatvec(self._h, _ptr(mu), _ptr(V), p, _ptr(W), _ptr(out)))
        return None if out is None else float(out[0])

    def kernel_timing(self, enable):
        """False / True, or an int k > 1: bracket every k-th evaluation only."""
        self._chk(_lib.alora_kernel_timing(self._h, int(enable)))

    def kernel_timing_read(self):
        ms, cnt = C.c_double(), C.c_int64()
        self._chk(_lib.alora_kernel_timing_read(self._h, C.addressof(ms), C.addressof(cnt)))
        return ms.value, cnt.value

    def lanczos(self, mu, kmax: int, tol_abs: float, seed: int, v=None, p_want: int = 1):
        """p_want == 1: returns (theta, k_used, resid, converged); v: device [n] or None.
        p_want > 1: returns (theta[p_found], k_used, resid[p_found], converged); v: device buffer of p_want * n
        elements (Ritz vector j at v[j*n:(j+1)*n]) or None.  mu=None: lambda of the last eval."""
        theta, resid = np.zeros(p_want), np.zeros(p_want)
        k, pf = C.c_int32(), C.c_int32()
        st = self._chk(_lib.alora_lanczos(self._h, _ptr(mu), kmax, float(tol_abs), C.c_uint64(seed), p_want,
                                          theta.ctypes.data, _ptr(v), C.addressof(pf), C.addressof(k), resid.ctypes.data),
                       allow=(ENOTCONV,))
        if p_want == 1:
            return float(theta[0]), k.value, float(resid[0]), st == OK
        return theta[: pf.value].copy(), k.value, resid[: pf.value].copy(), st == OK

    def solve(self, params: Params, R, r: int, r_cap: int, y, sigma: float, log_cap: int = 256):
        """Returns (Result, [IterRecord], r_final, sigma_final, converged)."""
        rr, sg = C.c_int32(r), C.c_double(sigma)
        log = (IterRecord * log_cap)()
        res = Result()
        st = self._chk(_lib.alora_solve(self._h, C.byref(params), _ptr(R), C.addressof(rr), r_cap, _ptr(y),
                                        C.addressof(sg), C.addressof(log), log_cap, C.addressof(res)),
                       allow=(ENOTCONV,))
        return res, list(log[: min(res.outer_iters, log_cap)]), rr.value, sg.value, st == OK
