"""Parity criteria shared by the GPU tests (SURVEY.md 8(c) B16 / DESIGN.md "Tolerance").

Every comparison is  |gpu - oracle| <= TOL * max(|oracle|, scale)  with TOL = 1e-10 (BASELINE.json
north_star) and `scale` = the sum of the magnitudes of the terms whose difference forms the entry, so
that an entry that cancels to ~0 (a gradient at an optimum) is still tested at the accuracy its terms
allow.  All scales are computed from ORACLE quantities only."""
import numpy as np

TOL = 1e-10


def check(name, g, o, scale=None, tol=TOL, floor=0.0):
    g, o = np.asarray(g, float), np.asarray(o, float)
    assert g.shape == o.shape, (name, g.shape, o.shape)
    ref = np.abs(o)
    if scale is not None:
        ref = np.maximum(ref, np.abs(scale))
    ref = np.maximum(ref, floor)
    err = np.abs(g - o)
    bad = ~(err <= tol * ref)
    if np.any(bad):
        i = np.argmax(np.where(bad, err / np.maximum(ref, 1e-300), 0))
        raise AssertionError(f"{name}: {bad.sum()} entries off; worst idx {np.unravel_index(i, g.shape)} "
                             f"gpu {g.flat[i]!r} oracle {o.flat[i]!r} rel-to-scale {err.flat[i] / max(ref.flat[i], 1e-300):.3e}")
    return float(np.max(err / np.maximum(ref, 1e-300))) if err.size else 0.0


def scales(ev, ref):
    """Error scales from the oracle's result `ref` (needs lam, integral, row_d1, grad_theta)."""
    mu0, tx, tt, xi0, h, om = ev.params
    n, D = ev.n, ev.dim
    lam = ref.lam
    s = {}
    s["ll"] = float(np.sum(np.abs(np.log(lam)))) + abs(ref.integral)
    T = ev.t[-1] - ev.t
    integ_theta = xi0 * (-np.expm1(-om * T))
    s["grad_theta"] = np.abs(ref.grad_theta + integ_theta) + integ_theta      # |c_m| + |xi0 (1-E_m)|
    if ref.row_d1 is not None:
        r = ref.row_d1 / lam[:, None]
        bfrac = float(np.sum(mu0 * r[:, 0]))       # sum_n SB_n / lambda_n
        sfrac = float(np.sum(xi0 * r[:, 3]))       # sum_n SS_n / lambda_n
        base = np.sum(np.abs(r), axis=0)
        a = (ev.t[-1] - ev.t) / tt
        b = -ev.t / tt
        phi = lambda z: np.exp(-0.5 * z * z) / np.sqrt(2 * np.pi)
        lam_tt = mu0 / tt * float(np.sum(np.abs(a * phi(a)) + np.abs(b * phi(b))))
        lam_om = xi0 * float(np.sum(ev.theta * T * np.exp(-om * T)))
        s["grad_hyper"] = base + np.array([n / mu0, 2 * D * bfrac / tx, 2 * bfrac / tt + lam_tt,
                                           float(np.sum(ev.theta * (-np.expm1(-om * T)))), 2 * D * sfrac / h,
                                           2 * sfrac / om + lam_om])
    return s


def hess_hyper_scale(H):
    d = np.sqrt(np.abs(np.diag(H)))
    return np.outer(d, d)


TRIU = [(p, q) for p in range(6) for q in range(p, 6)]


def scalars_from_rows(lam, d1, d2_triu, Lam, L1, L2):
    """ell, the hyper-gradient and the 6x6 Hessian as the plain O(N) sums of SURVEY.md 8(c) A2 / A6 / A7 over
    per-event values (long-double accumulation):
        ell = sum log lambda_n - Lambda,   g_p = sum lambda_{n,p}/lambda_n - Lambda_p,
        H_pq = sum [lambda_{n,pq}/lambda_n - lambda_{n,p} lambda_{n,q}/lambda_n^2] - Lambda_pq,
    with the error scales (sums of the magnitudes of the terms) beside them.  Used at sizes where the oracle can
    afford only a sample of rows: the per-event values are the GPU's own, validated on that sample; Lambda and its
    derivatives are the oracle's (oracle.integral)."""
    ld = np.longdouble
    lam = lam.astype(ld)
    ll = float(np.sum(np.log(lam)) - ld(Lam))
    s_ll = float(np.sum(np.abs(np.log(lam)))) + abs(Lam)
    out = {"ll": ll, "s_ll": s_ll}
    if d1 is not None:
        r = d1.astype(ld) / lam[:, None]
        out["grad_hyper"] = np.array(r.sum(0) - L1.astype(ld), dtype=float)
        out["s_grad_hyper"] = np.array(np.abs(r).sum(0), dtype=float) + np.abs(L1)
        if d2_triu is not None:
            H = np.zeros((6, 6))
            for k, (p, q) in enumerate(TRIU):
                v = float(np.sum(d2_triu[:, k].astype(ld) / lam - r[:, p] * r[:, q]) - ld(L2[p, q]))
                H[p, q] = H[q, p] = v
            out["hess_hyper"] = H
    return out
