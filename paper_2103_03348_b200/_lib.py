"""Loader of the in-tree CUDA library.  There is no fallback: if the library cannot be loaded the
import of the binding fails loudly."""
from __future__ import annotations

import ctypes
import os

from . import build as _build

_dp = ctypes.c_void_p   # device or host pointer to fp64
_lib = None

# every symbol include/hawkes.h declares: name -> (restype, argtypes)
i64, cint, u32, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_uint32, ctypes.c_void_p


class Params(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double) for k in ("mu0", "tau_x", "tau_t", "xi0", "h", "omega")]


PP = ctypes.POINTER(Params)


class HmcOpts(ctypes.Structure):
    _fields_ = [("n_iter", ctypes.c_int32), ("n_leapfrog", ctypes.c_int32), ("precond_every", ctypes.c_int32),
                ("n_refresh_done", ctypes.c_int32), ("step", ctypes.c_double), ("mass_floor", ctypes.c_double),
                ("cache_background", ctypes.c_int32), ("flags", ctypes.c_int32)]
SYMBOLS = {
    "hawkes_create": (cint, [ctypes.POINTER(vp), i64, cint, cint]),
    "hawkes_destroy": (None, [vp]),
    "hawkes_strerror": (ctypes.c_char_p, [cint]),
    "hawkes_last_status": (cint, [vp, vp]),
    "hawkes_loglik": (cint, [vp, i64, _dp, _dp, _dp, PP, _dp, vp]),
    "hawkes_loglik_static": (cint, [i64, cint, _dp, _dp, _dp, PP, _dp, vp, vp]),
    "hawkes_grad": (cint, [vp, i64, _dp, _dp, _dp, PP, _dp, _dp, _dp, vp]),
    "hawkes_hessian": (cint, [vp, i64, _dp, _dp, _dp, PP, _dp, _dp, _dp, vp]),
    "hawkes_eval": (cint, [vp, i64, _dp, _dp, _dp, PP, u32, _dp, _dp, _dp, _dp, _dp, _dp, vp]),
    "hawkes_eval_host": (cint, [vp, i64, _dp, _dp, _dp, PP, u32, _dp, _dp, _dp, _dp, _dp, _dp, vp]),
    "hawkes_hessian_theta_dense": (cint, [vp, i64, _dp, _dp, _dp, PP, _dp, vp]),
    "hawkes_sort_events": (cint, [vp, i64, cint, _dp, _dp, _dp, _dp, _dp, _dp, vp, vp]),
    "hawkes_get_lambda": (cint, [vp, i64, _dp, vp]),
    "hawkes_set_pass1_mode": (cint, [vp, cint]),
    "hawkes_pass1_is_symmetric": (cint, [vp, cint]),
    "hawkes_row_moments_enable": (cint, [vp, cint]),
    "hawkes_get_row_moments": (cint, [vp, i64, _dp, _dp, vp]),
    "hawkes_skip_plan": (cint, [vp, i64, _dp, _dp, PP]),
    "hawkes_eval_skip": (cint, [vp, i64, _dp, _dp, _dp, PP, u32, _dp, _dp, _dp, _dp, _dp, vp]),
    "hawkes_skip_stats": (cint, [vp, vp]),
    "hawkes_skip_perm": (cint, [vp, i64, vp]),
    "hawkes_set_background_mode": (cint, [vp, cint]),
    "hawkes_hessian_theta_block": (cint, [vp, i64, _dp, _dp, _dp, PP, i64, vp, _dp, vp]),
    "hawkes_shard_part_doubles": (i64, [i64, u32, cint]),
    "hawkes_shard_pass1": (cint, [vp, i64, _dp, _dp, _dp, PP, u32, cint, cint, _dp, vp]),
    "hawkes_shard_reduce1": (cint, [vp, i64, PP, u32, cint, _dp, _dp, _dp, _dp, vp]),
    "hawkes_shard_pass2": (cint, [vp, i64, PP, u32, cint, cint, _dp, vp]),
    "hawkes_shard_finish": (cint, [vp, i64, PP, u32, cint, _dp, _dp, _dp, vp]),
    "hawkes_shard_workers": (cint, [vp, u32, ctypes.POINTER(cint), ctypes.POINTER(cint)]),
    "hawkes_plan_segments": (i64, [i64, cint, cint, cint, cint, cint, cint, vp, i64]),
    "hawkes_debug_guard_check": (i64, [vp]),
    "hawkes_launch_count": (i64, [vp]),
    "hawkes_graph_launch_count": (i64, [vp]),
    "hawkes_profile_enable": (cint, [vp, cint]),
    "hawkes_profile_read": (cint, [vp, ctypes.POINTER(ctypes.c_double)]),
    "hawkes_fp64_peak": (cint, [vp, ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]),
    "hawkes_tree_create": (cint, [ctypes.POINTER(vp), ctypes.c_int32, vp, vp, cint]),
    "hawkes_tree_destroy": (None, [vp]),
    "hawkes_tree_prior": (cint, [vp, _dp, ctypes.c_double, ctypes.c_double, _dp, _dp, vp]),
    "hawkes_tree_levels": (ctypes.c_int32, [vp]),
    "hawkes_tree_launch_count": (i64, [vp]),
    "hawkes_theta_from_z": (cint, [vp, i64, i64, vp, _dp, ctypes.c_double, _dp, _dp, vp]),
    "hawkes_z_chain": (cint, [vp, i64, i64, vp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp, vp]),
    "hawkes_posterior_z": (cint, [vp, vp, i64, _dp, _dp, i64, vp, _dp, ctypes.c_double, PP, ctypes.c_double,
                                  ctypes.c_double, _dp, _dp, _dp, vp]),
    "hawkes_posterior_z_skip": (cint, [vp, vp, i64, _dp, _dp, i64, vp, _dp, ctypes.c_double, PP, ctypes.c_double,
                                  ctypes.c_double, _dp, _dp, _dp, vp]),
    "hawkes_hmc_run": (cint, [vp, vp, i64, _dp, _dp, i64, vp, _dp, ctypes.c_double, PP, ctypes.c_double,
                              ctypes.c_double, ctypes.POINTER(HmcOpts), _dp, _dp, _dp, _dp, _dp, vp]),
    "hawkes_tree_precision_diag": (cint, [vp, ctypes.c_double, ctypes.c_double, _dp, vp]),
}


def lib_path() -> str:
    return _build.LIB


def load():
    """Load (building first if the .so is missing or stale and nvcc is available)."""
    global _lib
    if _lib is not None:
        return _lib
    guard = os.environ.get("HAWKES_B200_GUARD") == "1"   # the debug build with guard bands (hawkes_debug_guard_check)
    path = _build.LIB_GUARD if guard else _build.LIB
    if not _build.up_to_date(guard):
        try:
            _build.build(guard=guard)
        except Exception as exc:   # no nvcc on this machine, or compile error: never run a stale library silently
            stamp = path + ".srchash"
            unstamped = os.path.exists(path) and not os.path.exists(stamp)
            if unstamped and os.environ.get("HAWKES_B200_ALLOW_UNSTAMPED") == "1":
                # a library copied without its source stamp: staleness unknown.  Loaded only on this explicit request.
                import warnings
                warnings.warn(f"paper_2103_03348_b200: {path} has no source stamp and could not be rebuilt ({exc}); "
                              f"loading it because HAWKES_B200_ALLOW_UNSTAMPED=1 -- it may not match csrc/", RuntimeWarning)
            else:
                what = ("has no source stamp (it cannot be checked against csrc/; set HAWKES_B200_ALLOW_UNSTAMPED=1 to load it anyway)"
                        if unstamped else "is older than its sources" if os.path.exists(path) else "is missing")
                raise ImportError(
                    f"paper_2103_03348_b200: CUDA library {path} {what} and could not be rebuilt "
                    f"({exc}); run `python -m paper_2103_03348_b200.build` on a machine with nvcc") from exc
    lib = ctypes.CDLL(path)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)   # AttributeError if the symbol is not exported
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib
