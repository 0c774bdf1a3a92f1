"""Oracle of the phylogenetic-diffusion prior and of the z-parametrisation of the rates (section 2.2).
TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs; never by the product package.

Dense arithmetic lives in oracle/tree_ref.cpp (long double path sums and Cholesky); the rest is the printed
formula written out in numpy fp64:

    theta_n = exp(z_n + beta f(t_n)), n in M;  theta_n = 1 otherwise;  f(t) = t
    d ell / d z_m      = theta_m d ell / d theta_m                                       (chain rule)
    d2 ell / d z_m^2   = theta_m^2 d2 ell / d theta_m^2 + theta_m d ell / d theta_m
    d ell / d beta     = sum_m t_m theta_m d ell / d theta_m
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import lib as _lib

_dp = ctypes.POINTER(ctypes.c_double)
_i32p = ctypes.POINTER(ctypes.c_int32)
_ready = False


def _l():
    global _ready
    l = _lib()
    if not _ready:
        l.tree_ref_vg.restype = ctypes.c_int
        l.tree_ref_vg.argtypes = [ctypes.c_int32, _i32p, _dp, ctypes.c_double, _dp]
        l.tree_ref_logp.restype = ctypes.c_int
        l.tree_ref_logp.argtypes = [ctypes.c_int32, _dp, _dp, ctypes.c_double, _dp, _dp]
        l.tree_ref_precision_diag.restype = ctypes.c_int
        l.tree_ref_precision_diag.argtypes = [ctypes.c_int32, _dp, ctypes.c_double, _dp]
        _ready = True
    return l


def vg(parent, branch, n_tips: int, tau0: float) -> np.ndarray:
    """V_G [M, M] from the path-length definition."""
    parent = np.ascontiguousarray(parent, dtype=np.int32)
    branch = np.ascontiguousarray(branch, dtype=np.float64)
    assert parent.shape == branch.shape == (2 * n_tips - 1,)
    V = np.empty((n_tips, n_tips), dtype=np.float64)
    rc = _l().tree_ref_vg(n_tips, parent.ctypes.data_as(_i32p), branch.ctypes.data_as(_dp), float(tau0),
                          V.ctypes.data_as(_dp))
    if rc != 0:
        raise ValueError("malformed tree")
    return V


def log_prior(V: np.ndarray, z, sigma2: float, grad: bool = True):
    """Eq. 2: returns (log p, d log p / d z or None)."""
    V = np.ascontiguousarray(V, dtype=np.float64)
    z = np.ascontiguousarray(z, dtype=np.float64)
    M = z.shape[0]
    assert V.shape == (M, M)
    lp = ctypes.c_double(0.0)
    g = np.empty(M, dtype=np.float64) if grad else None
    _l().tree_ref_logp(M, V.ctypes.data_as(_dp), z.ctypes.data_as(_dp), float(sigma2), ctypes.byref(lp),
                       g.ctypes.data_as(_dp) if grad else None)
    return float(lp.value), g


def precision_diag(V: np.ndarray, sigma2: float) -> np.ndarray:
    """diag(V_G^-1) / sigma2 = -d2 log p / d z_m^2 of Eq. 2."""
    V = np.ascontiguousarray(V, dtype=np.float64)
    M = V.shape[0]
    out = np.empty(M, dtype=np.float64)
    if _l().tree_ref_precision_diag(M, V.ctypes.data_as(_dp), float(sigma2), out.ctypes.data_as(_dp)) != 0:
        raise ValueError("V is not positive definite")
    return out


def theta_from_z(n: int, idx, z, beta: float, t) -> np.ndarray:
    """PAPER.md:97 with f(t) = t."""
    theta = np.ones(n, dtype=np.float64)
    idx = np.asarray(idx, dtype=np.int64)
    theta[idx] = np.exp(np.asarray(z, dtype=np.float64) + beta * np.asarray(t, dtype=np.float64)[idx])
    return theta


def z_chain(theta, t, idx, grad_theta, hess_theta_diag=None):
    """Chain rule through theta(z): (d ell/d z [M], d2 ell/d z^2 [M] or None, d ell/d beta)."""
    idx = np.asarray(idx, dtype=np.int64)
    th = np.asarray(theta, dtype=np.float64)[idx]
    g = np.asarray(grad_theta, dtype=np.float64)[idx]
    gz = th * g
    hz = None
    if hess_theta_diag is not None:
        hz = th * th * np.asarray(hess_theta_diag, dtype=np.float64)[idx] + th * g
    gbeta = float(np.sum(np.asarray(t, dtype=np.float64)[idx] * gz))
    return gz, hz, gbeta
