"""paper_2103_03348_b200 -- thin Python binding of the B200-native phylogenetic-Hawkes likelihood
library (include/hawkes.h).  Argument marshalling only: every step of the evaluation runs in the
CUDA kernels of csrc/hawkes.cu; PyTorch supplies device memory and the stream.  There is no CPU
fallback -- without the CUDA library (or without a GPU) the calls fail."""
from __future__ import annotations

import ctypes
import dataclasses

from . import synth  # noqa: F401  (seeded inputs; no method arithmetic)
from ._lib import HmcOpts, Params, load, lib_path  # noqa: F401

OK = 0
ERR_ARG, ERR_PARAM, ERR_UNSORTED, ERR_CUDA, ERR_NOMEM, ERR_UNSUPPORTED, ERR_NONFINITE = -1, -2, -3, -4, -5, -6, -7
ERR_TOO_LARGE = -8
STATIC_N_MAX = 32768   # HAWKES_STATIC_N_MAX: the largest problem loglik_static() takes
STATIC_BIT_UNSORTED, STATIC_BIT_NONFINITE, STATIC_BIT_ZERO_RATE = 1, 2, 4
WARN_ZERO_RATE = 1
WANT_LL, WANT_GRAD_THETA, WANT_GRAD_HYPER, WANT_HESS_THETA, WANT_HESS_HYPER, WANT_HESS_CROSS = 1, 2, 4, 8, 16, 32
WANT_GRAD = WANT_LL | WANT_GRAD_THETA | WANT_GRAD_HYPER
WANT_ALL = 63
BG_SPACE_TIME, BG_SPACE_ONLY = 0, 1
PASS1_AUTO, PASS1_DENSE = 0, 1
HMC_NO_GRAPH = 1


class HawkesError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {load().hawkes_strerror(status).decode()} (status {status})")


@dataclasses.dataclass
class EvalResult:
    """Device tensors (or host tensors for eval_host) of the requested outputs; None if not wanted."""
    ll: object = None
    grad_theta: object = None
    grad_hyper: object = None
    hess_theta_diag: object = None
    hess_hyper: object = None
    hess_cross: object = None
    status: int | None = None


def _params(p) -> Params:
    if isinstance(p, Params):
        return p
    return Params(*[float(v) for v in p])


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def loglik_static(x, t, theta, params, out, status_out=None):
    """hawkes_loglik_static: the log-likelihood for callers that cannot allocate GPU memory -- no HawkesContext (whose
    creation cudaMallocs its scratch) is involved, and neither this wrapper nor the C call behind it allocates: the
    intermediates sit in a fixed array inside the library, which limits the problem to STATIC_N_MAX events
    (HawkesError with ERR_TOO_LARGE beyond that).  Meant for code running inside a host application that owns all
    device memory, or that must not trigger the device-wide stall of an allocation.

    x [dim, n], t [n], theta [n]: float64 CUDA tensors on the current device; `out`: a float64 CUDA tensor of one
    element that receives ell (the caller provides it, for the same reason); `status_out`: optional int32 CUDA tensor of
    one element for the STATIC_BIT_* flags of this evaluation.  Asynchronous on the current stream.  The first call on
    a device does a one-off set-up with a small blocking copy, so make it before any stream capture.  All calls share
    the library's one array: do not let two of them run on the GPU at the same time (two streams, two threads)."""
    import torch
    for name, a, dt in (("x", x, torch.float64), ("t", t, torch.float64), ("theta", theta, torch.float64),
                        ("out", out, torch.float64), ("status_out", status_out, torch.int32)):
        if a is None and name == "status_out":
            continue
        if not a.is_cuda or a.device.index != torch.cuda.current_device() or a.dtype != dt or not a.is_contiguous():
            raise ValueError(f"{name} must be a contiguous {dt} CUDA tensor on the current device")
    n = t.shape[0]
    if x.dim() != 2 or x.shape[1] != n or theta.shape != (n,) or out.numel() != 1 or (status_out is not None and status_out.numel() != 1):
        raise ValueError("expected x [dim, n] (SoA), t [n], theta [n], out [1], status_out [1]")
    p = _params(params)
    rc = load().hawkes_loglik_static(n, x.shape[0], _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), _ptr(out), _ptr(status_out),
                                     ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != 0:
        raise HawkesError(rc, "hawkes_loglik_static")
    return out


class HawkesContext:
    """Owns one hawkes_ctx (device scratch for problems of up to n_max events in `dim` dimensions)."""

    def __init__(self, n_max: int, dim: int = 2, device: int = 0):
        import torch
        self._torch = torch
        self._lib = load()
        self.n_max, self.dim, self.device = int(n_max), int(dim), int(device)
        h = ctypes.c_void_p()
        rc = self._lib.hawkes_create(ctypes.byref(h), self.n_max, self.dim, self.device)
        if rc != 0:
            raise HawkesError(rc, "hawkes_create")
        self._h = h
        self._dev = torch.device("cuda", self.device)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.hawkes_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers ---------------------------------------------------------------------------------
    def _stream(self):
        return ctypes.c_void_p(self._torch.cuda.current_stream(self._dev).cuda_stream)

    def _check_dev(self, a, name, shape=None, dtype=None, optional=False):
        """Every pointer handed to a device-pointer entry point: a contiguous tensor of the expected dtype (float64
        unless given) and shape on this context's device.  A host tensor or an int32 index would otherwise reach
        the kernels as a wild address."""
        torch = self._torch
        if a is None:
            if optional:
                return
            raise ValueError(f"{name} is required")
        dtype = torch.float64 if dtype is None else dtype
        if not a.is_cuda or a.device.index != self.device:
            raise ValueError(f"{name} must be a CUDA tensor on device {self.device}")
        if a.dtype != dtype or not a.is_contiguous():
            raise ValueError(f"{name} must be a contiguous {dtype} tensor")
        if shape is not None and tuple(a.shape) != tuple(shape):
            raise ValueError(f"{name} must have shape {tuple(shape)}, got {tuple(a.shape)}")

    def _check_inputs(self, x, t, theta, host=False):
        torch = self._torch
        for a in (x, t, theta):
            if a.dtype != torch.float64 or not a.is_contiguous():
                raise ValueError("x, t, theta must be contiguous float64 tensors")
            if host and a.is_cuda:
                raise ValueError("eval_host() takes host tensors")
            if not host and (not a.is_cuda or a.device.index != self.device):
                raise ValueError(f"x, t, theta must be CUDA tensors on device {self.device}; use eval_host() for host buffers")
        n = t.shape[0]
        if x.shape != (self.dim, n) or theta.shape != (n,):
            raise ValueError("expected x [dim, n] (SoA), t [n], theta [n]")
        return n

    def _check_out(self, r, n):
        for name, shape in (("ll", (1,)), ("grad_theta", (n,)), ("grad_hyper", (6,)), ("hess_theta_diag", (n,)),
                            ("hess_hyper", (6, 6)), ("hess_cross", (n, 6))):
            self._check_dev(getattr(r, name), "out." + name, shape, optional=True)

    def _outputs(self, n, want, device, pinned=False):
        torch = self._torch
        mk = lambda *s: torch.empty(*s, dtype=torch.float64, device=device, pin_memory=pinned)
        return EvalResult(
            ll=mk(1) if want & WANT_LL else None,
            grad_theta=mk(n) if want & WANT_GRAD_THETA else None,
            grad_hyper=mk(6) if want & WANT_GRAD_HYPER else None,
            hess_theta_diag=mk(n) if want & WANT_HESS_THETA else None,
            hess_hyper=mk(6, 6) if want & WANT_HESS_HYPER else None,
            hess_cross=mk(n, 6) if want & WANT_HESS_CROSS else None)

    def new_outputs(self, n, want, device=None, pinned=False) -> EvalResult:
        """Output buffers for `want`, to be reused across calls through the `out=` arguments."""
        return self._outputs(n, want, self._dev if device is None else device, pinned)

    # -- the C-ABI calls ---------------------------------------------------------------------------
    def eval(self, x, t, theta, params, want: int = WANT_GRAD, out: EvalResult | None = None) -> EvalResult:
        """hawkes_eval: device tensors in, device tensors out, asynchronous on the current stream."""
        n = self._check_inputs(x, t, theta)
        r = out if out is not None else self._outputs(n, want, self._dev)
        self._check_out(r, n)
        p = _params(params)
        rc = self._lib.hawkes_eval(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), want,
                                   _ptr(r.ll), _ptr(r.grad_theta), _ptr(r.grad_hyper), _ptr(r.hess_theta_diag),
                                   _ptr(r.hess_hyper), _ptr(r.hess_cross), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_eval")
        return r

    def skip_plan(self, x, t, params) -> dict:
        """hawkes_skip_plan: k-d order, boxes and work lists of the exact-zero-skipping variant for these events
        and hyperparameters (synchronous, host work).  Returns the item counts of hawkes_skip_stats."""
        if x.dim() != 2 or x.shape[0] != self.dim or t.shape[0] != x.shape[1]:
            raise ValueError("x must be (dim, n) and t (n,)")
        for a in (x, t):
            if a.dtype != self._torch.float64 or not a.is_contiguous():
                raise ValueError("x and t must be contiguous float64 tensors (host or device)")
        n = int(t.shape[0])
        p = _params(params)
        rc = self._lib.hawkes_skip_plan(self._h, n, _ptr(x), _ptr(t), ctypes.byref(p))
        if rc != 0:
            raise HawkesError(rc, "hawkes_skip_plan")
        st = (ctypes.c_int64 * 9)()
        rc = self._lib.hawkes_skip_stats(self._h, st)
        if rc != 0:
            raise HawkesError(rc, "hawkes_skip_stats")
        return {"items_background": st[0], "items_excitation": st[1], "items_dense_pass1": st[2],
                "items_pass2": st[3], "items_dense_pass2": st[4], "workers_pass1": st[5], "workers_pass2": st[6],
                "items_background_unordered": st[7], "order_reused": st[8]}

    def skip_perm(self, n: int):
        """The k-d order of the current plan: record i is the caller's event perm[i] (host int64 tensor)."""
        perm = self._torch.empty(n, dtype=self._torch.int64)
        rc = self._lib.hawkes_skip_perm(self._h, n, perm.data_ptr())
        if rc != 0:
            raise HawkesError(rc, "hawkes_skip_perm")
        return perm

    def eval_skip(self, x, t, theta, params, want: int = WANT_GRAD, out: EvalResult | None = None) -> EvalResult:
        """hawkes_eval_skip: hawkes_eval over the work lists of skip_plan (same arguments, same outputs in the
        caller's event order, no cross block); the events need not be sorted by time."""
        n = self._check_inputs(x, t, theta)
        r = out if out is not None else self._outputs(n, want, self._dev)
        self._check_out(r, n)
        p = _params(params)
        rc = self._lib.hawkes_eval_skip(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), want,
                                        _ptr(r.ll), _ptr(r.grad_theta), _ptr(r.grad_hyper), _ptr(r.hess_theta_diag),
                                        _ptr(r.hess_hyper), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_eval_skip")
        return r

    def loglik(self, x, t, theta, params):
        n = self._check_inputs(x, t, theta)
        r = self._outputs(n, WANT_LL, self._dev)
        p = _params(params)
        rc = self._lib.hawkes_loglik(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), _ptr(r.ll), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_loglik")
        return r.ll

    def grad(self, x, t, theta, params, out: EvalResult | None = None) -> EvalResult:
        n = self._check_inputs(x, t, theta)
        r = out if out is not None else self._outputs(n, WANT_GRAD, self._dev)
        self._check_out(r, n)
        p = _params(params)
        rc = self._lib.hawkes_grad(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), _ptr(r.ll),
                                   _ptr(r.grad_theta), _ptr(r.grad_hyper), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_grad")
        return r

    def hessian(self, x, t, theta, params, cross: bool = False, out: EvalResult | None = None) -> EvalResult:
        n = self._check_inputs(x, t, theta)
        want = WANT_HESS_THETA | WANT_HESS_HYPER | (WANT_HESS_CROSS if cross else 0)
        r = out if out is not None else self._outputs(n, want, self._dev)
        self._check_out(r, n)
        p = _params(params)
        rc = self._lib.hawkes_hessian(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p),
                                      _ptr(r.hess_theta_diag), _ptr(r.hess_hyper), _ptr(r.hess_cross), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_hessian")
        return r

    def eval_host(self, x, t, theta, params, want: int = WANT_GRAD, out: EvalResult | None = None) -> EvalResult:
        """hawkes_eval_host: HOST tensors (pinned or pageable) in and out; copies run inside the call,
        which synchronises the stream and returns the evaluation's device status in `.status`."""
        n = self._check_inputs(x, t, theta, host=True)
        r = out if out is not None else self._outputs(n, want, "cpu")
        for name in ("ll", "grad_theta", "grad_hyper", "hess_theta_diag", "hess_hyper", "hess_cross"):
            o = getattr(r, name)
            if o is not None and (o.is_cuda or o.dtype != self._torch.float64 or not o.is_contiguous()):
                raise ValueError(f"out.{name} must be a contiguous float64 host tensor")
        p = _params(params)
        rc = self._lib.hawkes_eval_host(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), want,
                                        _ptr(r.ll), _ptr(r.grad_theta), _ptr(r.grad_hyper), _ptr(r.hess_theta_diag),
                                        _ptr(r.hess_hyper), _ptr(r.hess_cross), self._stream())
        if rc < 0:
            raise HawkesError(rc, "hawkes_eval_host")
        r.status = rc
        return r

    def hessian_theta_dense(self, x, t, theta, params):
        n = self._check_inputs(x, t, theta)
        H = self._torch.empty(n, n, dtype=self._torch.float64, device=self._dev)
        p = _params(params)
        rc = self._lib.hawkes_hessian_theta_dense(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), _ptr(H), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_hessian_theta_dense")
        return H

    def hessian_theta_block(self, x, t, theta, params, idx):
        """hawkes_hessian_theta_block: the dense m x m Hessian of ell in the rates of the events idx (device tensor)."""
        n = self._check_inputs(x, t, theta)
        m = int(idx.shape[0])
        self._check_dev(idx, "idx", (m,), self._torch.int64)
        H = self._torch.empty(m, m, dtype=self._torch.float64, device=self._dev)
        p = _params(params)
        rc = self._lib.hawkes_hessian_theta_block(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), m, _ptr(idx),
                                                  _ptr(H), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_hessian_theta_block")
        return H

    def sort_events(self, x, t, theta):
        """Stable sort by time on the device; returns (x_sorted, t_sorted, theta_sorted, perm)."""
        torch = self._torch
        n = self._check_inputs(x, t, theta)
        xo, to, tho = torch.empty_like(x), torch.empty_like(t), torch.empty_like(theta)
        perm = torch.empty(n, dtype=torch.int64, device=self._dev)
        rc = self._lib.hawkes_sort_events(self._h, n, self.dim, _ptr(x), _ptr(t), _ptr(theta), _ptr(xo), _ptr(to),
                                          _ptr(tho), _ptr(perm), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_sort_events")
        return xo, to, tho, perm

    # -- z-parametrisation and the fused z-posterior (include/hawkes.h, "Phylogenetic ... prior") ------------
    def theta_from_z(self, n: int, idx, z, beta: float, t, out=None):
        """hawkes_theta_from_z: idx int64 [m], z [m], t [n] device tensors -> theta [n]."""
        theta = out if out is not None else self._torch.empty(n, dtype=self._torch.float64, device=self._dev)
        m = int(idx.shape[0])
        self._check_dev(idx, "idx", (m,), self._torch.int64)
        self._check_dev(z, "z", (m,))
        self._check_dev(t, "t", (n,))
        self._check_dev(theta, "theta", (n,))
        rc = self._lib.hawkes_theta_from_z(self._h, n, int(idx.shape[0]), _ptr(idx), _ptr(z), float(beta), _ptr(t),
                                           _ptr(theta), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_theta_from_z")
        return theta

    def z_chain(self, idx, theta, t, grad_theta, hess_theta_diag=None, prior_grad_z=None, want_beta: bool = False):
        """hawkes_z_chain: returns (grad_z [m], hess_z [m] or None, grad_beta [1] or None)."""
        torch = self._torch
        n, m = int(theta.shape[0]), int(idx.shape[0])
        self._check_dev(idx, "idx", (m,), torch.int64)
        self._check_dev(theta, "theta", (n,))
        self._check_dev(t, "t", (n,), optional=not want_beta)
        self._check_dev(grad_theta, "grad_theta", (n,))
        self._check_dev(hess_theta_diag, "hess_theta_diag", (n,), optional=True)
        self._check_dev(prior_grad_z, "prior_grad_z", (m,), optional=True)
        gz = torch.empty(m, dtype=torch.float64, device=self._dev)
        hz = torch.empty(m, dtype=torch.float64, device=self._dev) if hess_theta_diag is not None else None
        gb = torch.empty(1, dtype=torch.float64, device=self._dev) if want_beta else None
        rc = self._lib.hawkes_z_chain(self._h, n, m, _ptr(idx), _ptr(theta), _ptr(t), _ptr(grad_theta),
                                      _ptr(hess_theta_diag), _ptr(prior_grad_z), _ptr(gz), _ptr(hz), _ptr(gb), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_z_chain")
        return gz, hz, gb

    def posterior_z(self, tree: "HawkesTree", x, t, idx, z, beta: float, params, sigma2: float, tau0: float,
                    hess: bool = False, out=None, skip: bool = False):
        """hawkes_posterior_z: returns (out3 [ell, log prior, sum], grad_z [m], hess_z [m] or None), device tensors;
        `out` = a previous return value to reuse its buffers; skip=True: hawkes_posterior_z_skip (after skip_plan)."""
        torch = self._torch
        n, m = int(t.shape[0]), int(idx.shape[0])
        self._check_dev(x, "x", (self.dim, n))
        self._check_dev(t, "t", (n,))
        self._check_dev(idx, "idx", (m,), torch.int64)
        self._check_dev(z, "z", (m,))
        if out is None:
            mk = lambda k: torch.empty(k, dtype=torch.float64, device=self._dev)
            out = (mk(3), mk(m), mk(m) if hess else None)
        self._check_dev(out[0], "out[0]", (3,), optional=True)
        self._check_dev(out[1], "out[1]", (m,), optional=True)
        self._check_dev(out[2], "out[2]", (m,), optional=True)
        p = _params(params)
        fn = self._lib.hawkes_posterior_z_skip if skip else self._lib.hawkes_posterior_z
        rc = fn(self._h, tree._h, n, _ptr(x), _ptr(t), m, _ptr(idx), _ptr(z), float(beta),
                                          ctypes.byref(p), float(sigma2), float(tau0), _ptr(out[0]), _ptr(out[1]),
                                          _ptr(out[2]), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_posterior_z")
        return out

    def hmc_run(self, tree: "HawkesTree", x, t, idx, z, beta: float, params, sigma2: float, tau0: float, *, n_iter: int,
                n_leapfrog: int, step: float, precond_every: int, mass, mass_floor: float, normals, uniforms,
                n_refresh_done: int = 0, cache_background: int = 0, prior_prec=None, trace=None, graph: bool = True):
        """hawkes_hmc_run: z [m] and mass [m] are updated in place (device tensors); normals [n_iter, m] and
        uniforms [n_iter] are device tensors; returns the trace [n_iter, 4] (device).  graph=False: HAWKES_HMC_NO_GRAPH."""
        torch = self._torch
        n, m = int(t.shape[0]), int(idx.shape[0])
        if normals.shape != (n_iter, m) or uniforms.shape != (n_iter,) or not normals.is_contiguous():
            raise ValueError("normals must be [n_iter, m] contiguous and uniforms [n_iter]")
        if trace is None:
            trace = torch.empty(n_iter, 4, dtype=torch.float64, device=self._dev)
        self._check_dev(x, "x", (self.dim, n))
        self._check_dev(t, "t", (n,))
        self._check_dev(idx, "idx", (m,), torch.int64)
        self._check_dev(z, "z", (m,))
        self._check_dev(mass, "mass", (m,))
        self._check_dev(normals, "normals", (n_iter, m))
        self._check_dev(uniforms, "uniforms", (n_iter,))
        self._check_dev(prior_prec, "prior_prec", (m,), optional=True)
        self._check_dev(trace, "trace", (n_iter, 4))
        o = HmcOpts(int(n_iter), int(n_leapfrog), int(precond_every), int(n_refresh_done), float(step),
                    float(mass_floor), int(cache_background), 0 if graph else HMC_NO_GRAPH)
        p = _params(params)
        rc = self._lib.hawkes_hmc_run(self._h, tree._h, n, _ptr(x), _ptr(t), m, _ptr(idx), _ptr(z), float(beta),
                                      ctypes.byref(p), float(sigma2), float(tau0), ctypes.byref(o), _ptr(normals),
                                      _ptr(uniforms), _ptr(mass), _ptr(prior_prec), _ptr(trace), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_hmc_run")
        return trace

    def set_background_mode(self, mode: int):
        """hawkes_set_background_mode: BG_SPACE_TIME (default) or BG_SPACE_ONLY (the paper's background as printed)."""
        rc = self._lib.hawkes_set_background_mode(self._h, int(mode))
        if rc != 0:
            raise HawkesError(rc, "hawkes_set_background_mode")

    # -- one evaluation sharded across GPUs (include/hawkes.h, "One evaluation sharded ...") ---------------------
    def shard_part_doubles(self, n: int, want: int, phase: int) -> int:
        return int(self._lib.hawkes_shard_part_doubles(n, want, phase))

    def shard_pass1(self, x, t, theta, params, want: int, rank: int, world: int, part_out):
        n = self._check_inputs(x, t, theta)
        self._check_dev(part_out, "part_out", (self.shard_part_doubles(n, want, 1),))
        p = _params(params)
        rc = self._lib.hawkes_shard_pass1(self._h, n, _ptr(x), _ptr(t), _ptr(theta), ctypes.byref(p), want, rank, world,
                                          _ptr(part_out), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_shard_pass1")

    def shard_reduce1(self, n: int, params, want: int, world: int, parts_all, out: EvalResult):
        self._check_dev(parts_all, "parts_all", (world, self.shard_part_doubles(n, want, 1)))
        self._check_out(out, n)
        p = _params(params)
        rc = self._lib.hawkes_shard_reduce1(self._h, n, ctypes.byref(p), want, world, _ptr(parts_all), _ptr(out.ll),
                                            _ptr(out.grad_hyper), _ptr(out.hess_hyper), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_shard_reduce1")

    def shard_pass2(self, n: int, params, want: int, rank: int, world: int, part2_out):
        self._check_dev(part2_out, "part2_out", (self.shard_part_doubles(n, want, 2),))
        p = _params(params)
        rc = self._lib.hawkes_shard_pass2(self._h, n, ctypes.byref(p), want, rank, world, _ptr(part2_out), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_shard_pass2")

    def shard_finish(self, n: int, params, want: int, world: int, parts2_all, out: EvalResult):
        self._check_dev(parts2_all, "parts2_all", (world, self.shard_part_doubles(n, want, 2)))
        p = _params(params)
        rc = self._lib.hawkes_shard_finish(self._h, n, ctypes.byref(p), want, world, _ptr(parts2_all),
                                           _ptr(out.grad_theta), _ptr(out.hess_theta_diag), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_shard_finish")

    def shard_workers(self, want: int):
        a, b = ctypes.c_int(0), ctypes.c_int(0)
        rc = self._lib.hawkes_shard_workers(self._h, want, ctypes.byref(a), ctypes.byref(b))
        if rc != 0:
            raise HawkesError(rc, "hawkes_shard_workers")
        return int(a.value), int(b.value)

    def set_pass1_mode(self, mode: int):
        """hawkes_set_pass1_mode: PASS1_AUTO (background once per unordered pair where it applies) or PASS1_DENSE."""
        rc = self._lib.hawkes_set_pass1_mode(self._h, int(mode))
        if rc != 0:
            raise HawkesError(rc, "hawkes_set_pass1_mode")

    def pass1_is_symmetric(self, level: int) -> bool:
        return bool(self._lib.hawkes_pass1_is_symmetric(self._h, int(level)))

    def row_moments_enable(self, enable: bool = True):
        rc = self._lib.hawkes_row_moments_enable(self._h, 1 if enable else 0)
        if rc != 0:
            raise HawkesError(rc, "hawkes_row_moments_enable")

    def get_row_moments(self, n: int, second: bool = False):
        """hawkes_get_row_moments: d lambda_n/dp [n, 6] (and d2 lambda_n/dp dq [n, 21], upper triangle) of the last
        evaluation; device tensors."""
        torch = self._torch
        d1 = torch.empty(n, 6, dtype=torch.float64, device=self._dev)
        d2 = torch.empty(n, 21, dtype=torch.float64, device=self._dev) if second else None
        rc = self._lib.hawkes_get_row_moments(self._h, n, _ptr(d1), _ptr(d2), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_get_row_moments")
        return (d1, d2) if second else d1

    def get_lambda(self, n: int):
        lam = self._torch.empty(n, dtype=self._torch.float64, device=self._dev)
        rc = self._lib.hawkes_get_lambda(self._h, n, _ptr(lam), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_get_lambda")
        return lam

    def last_status(self) -> int:
        return int(self._lib.hawkes_last_status(self._h, self._stream()))

    def debug_guard_check(self) -> int:
        """hawkes_debug_guard_check: corrupted guard-band bytes (guard build, HAWKES_B200_GUARD=1), else raises."""
        rc = int(self._lib.hawkes_debug_guard_check(self._h))
        if rc < 0:
            raise HawkesError(rc, "hawkes_debug_guard_check")
        return rc

    def launch_count(self) -> int:
        return int(self._lib.hawkes_launch_count(self._h))

    def graph_launch_count(self) -> int:
        return int(self._lib.hawkes_graph_launch_count(self._h))

    def profile_enable(self, enable: bool = True):
        rc = self._lib.hawkes_profile_enable(self._h, 1 if enable else 0)
        if rc != 0:
            raise HawkesError(rc, "hawkes_profile_enable")

    def profile_read(self) -> dict:
        """Sums over the evaluations recorded since the last read (at most 256)."""
        out = (ctypes.c_double * 7)()
        rc = self._lib.hawkes_profile_read(self._h, out)
        if rc != 0:
            raise HawkesError(rc, "hawkes_profile_read")
        return {"evals": int(out[0]), "pass1_ms": out[1], "pass2_ms": out[2], "total_ms": out[3],
                "prep_ms": out[4], "mid_ms": out[5], "tail_ms": out[6]}

    def fp64_peak(self, millis: float = 200.0) -> float:
        v = ctypes.c_double(0.0)
        rc = self._lib.hawkes_fp64_peak(self._h, float(millis), ctypes.byref(v), self._stream())
        if rc != 0:
            raise HawkesError(rc, "hawkes_fp64_peak")
        return float(v.value)


class HawkesTree:
    """Owns one hawkes_tree: the device copy of a rooted binary tree over M tips (nodes 0..M-1 are the tips;
    parent[root] = -1; branch[v] = edge weight to the parent), for the O(M) phylogenetic-diffusion prior."""

    def __init__(self, parent, branch, device: int = 0):
        import numpy as np
        import torch
        self._torch = torch
        self._lib = load()
        par = np.ascontiguousarray(parent, dtype=np.int32)
        br = np.ascontiguousarray(branch, dtype=np.float64)
        if par.shape != br.shape or par.ndim != 1 or par.shape[0] % 2 != 1:
            raise ValueError("parent and branch must be 1-D arrays of 2M-1 entries")
        self.n_tips = (par.shape[0] + 1) // 2
        self.device = int(device)
        h = ctypes.c_void_p()
        rc = self._lib.hawkes_tree_create(ctypes.byref(h), self.n_tips, par.ctypes.data_as(ctypes.c_void_p),
                                          br.ctypes.data_as(ctypes.c_void_p), self.device)
        if rc != 0:
            raise HawkesError(rc, "hawkes_tree_create")
        self._h = h
        self._dev = torch.device("cuda", self.device)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.hawkes_tree_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def prior(self, z, sigma2: float, tau0: float, grad: bool = True):
        """hawkes_tree_prior: z [M] device tensor -> (log p [1], d log p / d z [M] or None), device tensors."""
        torch = self._torch
        lp = torch.empty(1, dtype=torch.float64, device=self._dev)
        g = torch.empty(self.n_tips, dtype=torch.float64, device=self._dev) if grad else None
        if (not z.is_cuda or z.device.index != self.device or z.dtype != torch.float64 or not z.is_contiguous()
                or tuple(z.shape) != (self.n_tips,)):
            raise ValueError(f"z must be a contiguous float64 CUDA tensor of {self.n_tips} entries on device {self.device}")
        st = ctypes.c_void_p(torch.cuda.current_stream(self._dev).cuda_stream)
        rc = self._lib.hawkes_tree_prior(self._h, _ptr(z), float(sigma2), float(tau0), _ptr(lp), _ptr(g), st)
        if rc != 0:
            raise HawkesError(rc, "hawkes_tree_prior")
        return lp, g

    def precision_diag(self, sigma2: float, tau0: float):
        """hawkes_tree_precision_diag: diag(V_G^-1)/sigma2 [M] (device tensor)."""
        torch = self._torch
        out = torch.empty(self.n_tips, dtype=torch.float64, device=self._dev)
        st = ctypes.c_void_p(torch.cuda.current_stream(self._dev).cuda_stream)
        rc = self._lib.hawkes_tree_precision_diag(self._h, float(sigma2), float(tau0), _ptr(out), st)
        if rc != 0:
            raise HawkesError(rc, "hawkes_tree_precision_diag")
        return out

    def levels(self) -> int:
        return int(self._lib.hawkes_tree_levels(self._h))

    def launch_count(self) -> int:
        return int(self._lib.hawkes_tree_launch_count(self._h))


def plan_segments(n: int, pass_: int, level: int, symmetric: bool, workers_total: int, w_begin: int, w_end: int):
    """hawkes_plan_segments (host-only, no GPU): int64 array [rows, 5] = (worker, tile, j_begin, j_end, partial slot)."""
    import numpy as np
    lib = load()
    cap = 1024
    while True:
        seg = np.zeros((cap, 5), dtype=np.int64)
        cnt = int(lib.hawkes_plan_segments(n, pass_, level, 1 if symmetric else 0, workers_total, w_begin, w_end,
                                           seg.ctypes.data, cap))
        if cnt < 0:
            raise HawkesError(cnt, "hawkes_plan_segments")
        if cnt <= cap:
            return seg[:cnt]
        cap = cnt


def shard_eval(ctx, dist, rank: int, world: int, x, t, theta, params, want: int = WANT_GRAD, out: EvalResult | None = None):
    """One evaluation sharded across the `world` processes of `dist` (torch.distributed, one process per GPU; or None
    with world == 1): the four hawkes_shard_* phases of `ctx` with one all-gather between pass and reduction.  Every rank
    returns the full, replicated outputs.  Orchestration only: `ctx` does the arithmetic."""
    import torch
    n = int(t.shape[0])
    r = out if out is not None else ctx.new_outputs(n, want)
    mk = lambda k: torch.empty(k, dtype=torch.float64, device=t.device)

    def gather(part):
        allp = mk(world * part.numel()).view(world, part.numel())
        if dist is None or world == 1:
            allp.copy_(part.view(1, -1))
        else:
            dist.all_gather_into_tensor(allp.view(-1), part)
        return allp

    part1 = mk(ctx.shard_part_doubles(n, want, 1))
    ctx.shard_pass1(x, t, theta, params, want, rank, world, part1)
    ctx.shard_reduce1(n, params, want, world, gather(part1), r)
    if want & (WANT_GRAD_THETA | WANT_HESS_THETA):
        part2 = mk(ctx.shard_part_doubles(n, want, 2))
        ctx.shard_pass2(n, params, want, rank, world, part2)
        ctx.shard_finish(n, params, want, world, gather(part2), r)
    return r
