"""ctypes wrapper around the oracle (oracle/hawkes_ref.cpp).  TEST INFRASTRUCTURE ONLY: imported by
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs; never by the
product package."""
from __future__ import annotations

import ctypes
import dataclasses

import numpy as np

from . import build as _build

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.hawkes_ref_eval.restype = ctypes.c_int
        _lib.hawkes_ref_eval.argtypes = [ctypes.c_int64, ctypes.c_int] + [_dp] * 14 + [ctypes.c_int, ctypes.c_int]
        _lib.hawkes_ref_rows.restype = ctypes.c_int
        _lib.hawkes_ref_rows.argtypes = [ctypes.c_int64, ctypes.c_int, _dp, _dp, _dp, _dp,
                                         ctypes.c_int64, _ip, _dp, _dp, _dp, ctypes.c_int, ctypes.c_int]
        _lib.hawkes_ref_integral.restype = ctypes.c_int
        _lib.hawkes_ref_integral.argtypes = [ctypes.c_int64, ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp, ctypes.c_int]
        _lib.hawkes_ref_cols.restype = ctypes.c_int
        _lib.hawkes_ref_cols.argtypes = [ctypes.c_int64, ctypes.c_int, _dp, _dp, _dp, _dp,
                                         ctypes.c_int64, _ip, _dp, _dp, ctypes.c_int]
        _lib.hawkes_ref_max_threads.restype = ctypes.c_int
    return _lib


def max_threads() -> int:
    return int(lib().hawkes_ref_max_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


@dataclasses.dataclass
class RefResult:
    status: int
    ll: float | None = None
    integral: float | None = None
    lam: np.ndarray | None = None
    grad_theta: np.ndarray | None = None
    grad_hyper: np.ndarray | None = None
    hess_theta_diag: np.ndarray | None = None
    hess_hyper: np.ndarray | None = None
    hess_cross: np.ndarray | None = None
    hess_theta_dense: np.ndarray | None = None
    row_d1: np.ndarray | None = None


def _bg(bg: str) -> int:
    """"ST" (default model) or "S" (paper-literal space-only background) -> the C argument."""
    if bg not in ("ST", "S"):
        raise ValueError("bg must be 'ST' or 'S'")
    return 1 if bg == "S" else 0


def evaluate(x, t, theta, params, *, grad=True, hess=False, cross=False, dense=False,
             row_d1=False, threads: int = 1, bg: str = "ST") -> RefResult:
    """x: [dim, n] SoA; t: [n] sorted; theta: [n]; params: 6 floats.  Always returns ll, the
    integral Lambda(t_N) and lambda[n]; gradient / Hessian pieces on request.  bg: background model, "ST" or "S"."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    t = np.ascontiguousarray(t, dtype=np.float64)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    prm = np.asarray(params, dtype=np.float64)
    dim, n = x.shape
    ll = np.zeros(1)
    integ = np.zeros(1)
    lam = np.zeros(n)
    gth = np.zeros(n) if grad else None
    ghy = np.zeros(6) if grad else None
    hth = np.zeros(n) if hess else None
    hhy = np.zeros(36) if hess else None
    hcr = np.zeros(n * 6) if cross else None
    hde = np.zeros(n * n) if dense else None
    rd1 = np.zeros(n * 6) if row_d1 else None
    st = lib().hawkes_ref_eval(n, dim, _p(x), _p(t), _p(theta), _p(prm), _p(ll), _p(integ), _p(lam),
                               _p(gth), _p(ghy), _p(hth), _p(hhy), _p(hcr), _p(hde), _p(rd1), threads, _bg(bg))
    if st < 0:
        raise ValueError(f"hawkes_ref_eval: bad argument (status {st})")
    return RefResult(status=st, ll=float(ll[0]), integral=float(integ[0]), lam=lam, grad_theta=gth,
                     grad_hyper=ghy, hess_theta_diag=hth,
                     hess_hyper=None if hhy is None else hhy.reshape(6, 6),
                     hess_cross=None if hcr is None else hcr.reshape(n, 6),
                     hess_theta_dense=None if hde is None else hde.reshape(n, n),
                     row_d1=None if rd1 is None else rd1.reshape(n, 6))


def rows(x, t, theta, params, idx, *, derivs=True, second=False, threads: int = 1, bg: str = "ST"):
    """lambda_n and d lambda_n / dp for the listed target rows; with second=True a third value, d2 lambda_n / dp dq
    as [rows, 6, 6]."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    t = np.ascontiguousarray(t, dtype=np.float64)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    prm = np.asarray(params, dtype=np.float64)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    dim, n = x.shape
    lam = np.zeros(len(idx))
    d1 = np.zeros(len(idx) * 6) if derivs else None
    d2 = np.zeros(len(idx) * 36) if second else None
    st = lib().hawkes_ref_rows(n, dim, _p(x), _p(t), _p(theta), _p(prm), len(idx),
                               idx.ctypes.data_as(_ip), _p(lam), _p(d1), _p(d2), threads, _bg(bg))
    if st != 0:
        raise ValueError(f"hawkes_ref_rows: status {st}")
    if second:
        return lam, (None if d1 is None else d1.reshape(-1, 6)), d2.reshape(-1, 6, 6)
    return lam, (None if d1 is None else d1.reshape(-1, 6))


def integral(t, theta, params, dim: int, *, bg: str = "ST"):
    """Lambda(t_N) and its first [6] and second [6, 6] derivatives in the hyperparameters (O(N))."""
    t = np.ascontiguousarray(t, dtype=np.float64)
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    prm = np.asarray(params, dtype=np.float64)
    lam, d1, d2 = np.zeros(1), np.zeros(6), np.zeros(36)
    st = lib().hawkes_ref_integral(len(t), dim, _p(t), _p(theta), _p(prm), _p(lam), _p(d1), _p(d2), _bg(bg))
    if st != 0:
        raise ValueError(f"hawkes_ref_integral: status {st}")
    return float(lam[0]), d1, d2.reshape(6, 6)


def cross_abs(x, t, params, lam, row_d1, *, threads: int = 1):
    """Error scale of the cross block (tests only): abs[m, p] = sum_{t_m<t_n} (k_nm/lambda_n) (T_p + |lambda_{n,p}|/lambda_n),
    T = (0, 0, 0, 1/xi0, r^2/h^3 + D/h, 1/omega + dt) -- the magnitudes of the terms of entry (m, p), SURVEY.md 8(c) B16."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    t = np.ascontiguousarray(t, dtype=np.float64)
    prm = np.asarray(params, dtype=np.float64)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    rd1 = np.ascontiguousarray(row_d1, dtype=np.float64)
    dim, n = x.shape
    out = np.zeros(n * 6)
    fn = lib().hawkes_ref_cross_abs
    fn.restype = ctypes.c_int
    fn.argtypes = [ctypes.c_int64, ctypes.c_int] + [_dp] * 6 + [ctypes.c_int]
    st = fn(n, dim, _p(x), _p(t), _p(prm), _p(lam), _p(rd1), _p(out), threads)
    if st != 0:
        raise ValueError(f"hawkes_ref_cross_abs: status {st}")
    return out.reshape(n, 6)


def cols(x, t, params, lam, idx, *, threads: int = 1):
    """c_m = sum_{t_m<t_n} k_nm / lambda_n and d_m = sum (k_nm/lambda_n)^2 for the listed columns."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    t = np.ascontiguousarray(t, dtype=np.float64)
    prm = np.asarray(params, dtype=np.float64)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    dim, n = x.shape
    c = np.zeros(len(idx))
    d = np.zeros(len(idx))
    st = lib().hawkes_ref_cols(n, dim, _p(x), _p(t), _p(prm), _p(lam), len(idx),
                               idx.ctypes.data_as(_ip), _p(c), _p(d), threads)
    if st != 0:
        raise ValueError(f"hawkes_ref_cols: status {st}")
    return c, d
