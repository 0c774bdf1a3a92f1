"""Oracle of the preconditioned HMC update of the log-rates z (section 2.3.2, l.127-145).
TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs; never by the product package.

The algorithm, step by step in the paper's notation (numpy fp64; plain Python loops):

    H(z, p) = -log pi(z) + 1/2 p^T M^-1 p                      (l.129; M diagonal, l.141)
    dz/dt = M^-1 p,   dp/dt = grad log pi(z)                   (l.133; the printed factor 1/2 in dz/dt is a typo:
                                                                DESIGN.md reading R7 -- it is not the derivative of H)
    leapfrog (Leimkuhler & Reich, cited l.131):  p += eps/2 grad;  L times { z += eps M^-1 p;  p += eps grad }
                                                  with the last kick eps/2
    accept the proposal with probability min(1, exp(H_old - H_new))            (standard HMC, Neal 2011 cited l.117)
    preconditioner: M = A + P, A = running average of the negative diagonal Hessian of the log-likelihood in z,
    refreshed at a fixed interval and floor-clamped (l.143-145; reading R6), P = the prior's own diagonal
    curvature diag(V_G^-1)/sigma^2 (constant; optional, reading R20: without it the dynamics are unstable on
    trees with very short branches) -- the paper gives no step size, averaging weights or floor: those choices are
    "parity unpinned".

Random numbers are INPUTS (normals [n_iter, M] for the momenta, uniforms [n_iter] for the accept test), so that the
CUDA path and this oracle consume the same draws.

`target(z, hess)` returns (log pi(z), grad log pi(z) [M], h [M] or None) with h = -d2 ell/dz_m^2 (likelihood part).
"""
from __future__ import annotations

import numpy as np


def leapfrog(target, z, p, grad, mass, eps: float, n_steps: int):
    """n_steps leapfrog steps from (z, p) with grad = grad log pi(z); returns (z, p, logpi, grad) at the end."""
    z = np.array(z, dtype=np.float64)
    p = np.array(p, dtype=np.float64)
    p = p + 0.5 * eps * grad
    logpi = None
    for step in range(n_steps):
        z = z + eps * p / mass
        logpi, grad, _ = target(z, False)
        p = p + (eps if step + 1 < n_steps else 0.5 * eps) * grad
    return z, p, logpi, grad


def run(target, z0, normals, uniforms, n_iter: int, n_leapfrog: int, eps: float, precond_every: int, mass0,
        mass_floor: float, prior_prec=None):
    """Returns dict(z [M], mass [M] (the running average A), trace [n_iter, 4] = (log pi after the iteration, H_old,
    H_new, accepted)).  The mass matrix used by the dynamics is A + prior_prec."""
    z = np.array(z0, dtype=np.float64)
    avg = np.array(mass0, dtype=np.float64)
    pp = np.zeros_like(avg) if prior_prec is None else np.asarray(prior_prec, dtype=np.float64)
    mass = avg + pp
    logpi, grad, _ = target(z, False)
    n_refresh = 0
    trace = np.zeros((n_iter, 4))
    for it in range(n_iter):
        if precond_every > 0 and it % precond_every == 0:
            _, _, h = target(z, True)
            n_refresh += 1
            avg = avg + (np.maximum(h, mass_floor) - avg) / n_refresh     # running average of the clamped Hessians
            mass = avg + pp
        p0 = np.sqrt(mass) * normals[it]
        h_old = -logpi + 0.5 * float(np.sum(p0 * p0 / mass))
        z1, p1, logpi1, grad1 = leapfrog(target, z, p0, grad, mass, eps, n_leapfrog)
        h_new = -logpi1 + 0.5 * float(np.sum(p1 * p1 / mass))
        with np.errstate(divide="ignore"):
            accept = bool(np.isfinite(h_new) and np.log(uniforms[it]) < h_old - h_new)
        if accept:
            z, logpi, grad = z1, logpi1, grad1
        trace[it] = (logpi, h_old, h_new, 1.0 if accept else 0.0)
    return {"z": z, "mass": avg, "trace": trace}


def hawkes_target(x, t, idx, beta, params, V, sigma2, threads: int = 1):
    """log pi(z) = ell(theta(z)) + log p(z | V_G, sigma2, tau0) (Eq. 3 restricted to z) from the oracles."""
    import oracle
    from oracle import tree as otree
    n = t.shape[0]

    def target(z, hess):
        th = otree.theta_from_z(n, idx, z, beta, t)
        r = oracle.evaluate(x, t, th, params, hess=hess, threads=threads)
        lp, pg = otree.log_prior(V, z, sigma2)
        gz, hz, _ = otree.z_chain(th, t, idx, r.grad_theta, r.hess_theta_diag if hess else None)
        return r.ll + lp, gz + pg, (-hz if hess else None)

    return target
