"""Pins for the oracle (oracle/hawkes_ref.cpp): everything here checks the oracle against something
other than itself -- closed forms, numbers worked out independently, quadrature, finite differences,
invariances the model must have, and a library KDE.  CPU only.

Pin numbering follows SURVEY.md section 8(c); PAPER.md line numbers in the docstrings."""
import json
import math
import os

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_2103_03348_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))
CFG = synth.CONFIG_PARAMS


def Phi(z):
    return 0.5 * math.erfc(-z / math.sqrt(2.0))


def rel(a, b):
    a, b = np.asarray(a, float), np.asarray(b, float)
    return np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-300))


# ------------------------------------------------------------------ P1: N = 1 closed form
def test_p1_single_event():
    """N=1: the only source is the event itself, excluded from the background (I[x != x_n],
    PAPER.md:60) and not earlier than itself (l.78) => lambda_1 = 0, ell = -inf, status 1;
    Lambda = mu0 [Phi(0) - Phi(-t_1/tau_t)]; the theta-gradient's integral part is xi0 (1-e^0) = 0."""
    t1 = 3.7
    r = oracle.evaluate(np.array([[1.0], [2.0]]), np.array([t1]), np.array([1.3]), CFG)
    assert r.status == 1
    assert r.lam[0] == 0.0
    assert r.ll == -math.inf
    assert abs(r.integral - CFG[0] * (0.5 - Phi(-t1 / CFG[2]))) < 1e-15
    assert r.grad_theta[0] == 0.0


# ------------------------------------------------------------------ P2: N = 2 closed form
@pytest.mark.parametrize("dim", [1, 2, 3])
def test_p2_two_events_closed_form(dim):
    """N=2, t_1<t_2, x_1!=x_2: lambda_1 = B (background from the LATER event: the background sums
    over all n', l.60), lambda_2 = B + theta_1 k.  Constants typed out from l.60-62."""
    mu0, tx, tt, xi0, h, om = 0.4, 2.5, 3.0, 0.6, 1.3, 0.45
    xs = np.array([[0.3, 1.9], [-0.4, 0.8], [0.25, -0.6]])[:dim]
    t = np.array([1.2, 2.9])
    th = np.array([1.7, 0.6])
    r2 = float(np.sum((xs[:, 0] - xs[:, 1]) ** 2))
    dt = t[1] - t[0]
    B = mu0 * (2 * math.pi) ** (-(dim + 1) / 2) * tx ** (-dim) / tt * math.exp(-r2 / (2 * tx * tx) - dt * dt / (2 * tt * tt))
    k = xi0 * om * (2 * math.pi * h * h) ** (-dim / 2) * math.exp(-om * dt - r2 / (2 * h * h))
    Lam = mu0 * ((Phi(dt / tt) - Phi(-t[0] / tt)) + (Phi(0.0) - Phi(-t[1] / tt))) + xi0 * th[0] * (1 - math.exp(-om * dt))
    ll = math.log(B) + math.log(B + th[0] * k) - Lam
    r = oracle.evaluate(xs, t, th, (mu0, tx, tt, xi0, h, om), hess=True, dense=True)
    assert r.status == 0
    assert rel(r.lam, [B, B + th[0] * k]) < 1e-14
    assert abs(r.integral - Lam) < 1e-14
    assert abs(r.ll - ll) < 1e-13
    a = k / (B + th[0] * k)
    assert rel(r.grad_theta[0], a - xi0 * (1 - math.exp(-om * dt))) < 1e-13
    assert r.grad_theta[1] == 0.0            # last event: no later target, 1 - e^0 = 0
    assert rel(r.hess_theta_diag[0], -a * a) < 1e-13
    assert r.hess_theta_diag[1] == 0.0
    assert rel(r.hess_theta_dense[0, 0], -a * a) < 1e-13
    assert r.hess_theta_dense[0, 1] == 0.0 and r.hess_theta_dense[1, 1] == 0.0


# ------------------------------------------------------------------ P2': worked numbers
def test_p2_worked_examples_golden():
    with open(os.path.join(HERE, "golden", "worked_examples.json")) as f:
        g = json.load(f)
    prm = g["params"]
    for name, c in g["cases"].items():
        r = oracle.evaluate(np.array(c["x"]), np.array(c["t"]), np.array(c["theta"]), prm, hess=True)
        assert abs(r.ll - c["ll"]) < 2e-13, name
        if "integral" in c:
            assert abs(r.integral - c["integral"]) < 1e-14, name
        if "lambda" in c:
            assert rel(r.lam, c["lambda"]) < 1e-13, name
        assert np.allclose(r.grad_theta, c["grad_theta"], rtol=1e-12, atol=1e-15), name
        if "hess_theta_diag" in c:
            assert np.allclose(r.hess_theta_diag, c["hess_theta_diag"], rtol=1e-12, atol=1e-18), name
        if "grad_hyper" in c:
            assert np.allclose(r.grad_hyper, c["grad_hyper"], rtol=1e-12), name
        if "B" in c:
            assert rel(r.lam[0], c["B"]) < 1e-13, name
            assert rel(r.lam[1] - r.lam[0], c["theta1_k"]) < 1e-9, name


# ------------------------------------------------------------------ P3: quadrature of Lambda
@pytest.mark.parametrize("seed", [1, 2])
def test_p3_integral_by_quadrature(seed):
    """Lambda(t_N) = int_0^{t_N} int_{R^D} lambda dx dt.  Space integrates analytically
    to 1 per event (Gaussians), leaving a 1-D integrand in s with kinks at the event times; adaptive
    quadrature with breakpoints at the t_n must reproduce the closed form (l.72 / Eq. 7 l.253 for the
    excitation part, DESIGN R1/R2 for the time-Gaussian background)."""
    ev = synth.small_random(7, seed)
    mu0, tx, tt, xi0, h, om = ev.params
    t, th = ev.t, ev.theta

    def f(s):
        bg = mu0 / tt * np.sum(np.exp(-0.5 * ((s - t) / tt) ** 2)) / math.sqrt(2 * math.pi)
        ex = xi0 * om * np.sum(th[t < s] * np.exp(-om * (s - t[t < s])))
        return bg + ex

    q, _ = integrate.quad(f, 0.0, t[-1], points=list(t[:-1]), epsabs=1e-13, epsrel=1e-13, limit=400)
    r = oracle.evaluate(ev.x, t, th, ev.params, grad=False)
    assert abs(r.integral - q) < 1e-11 * max(1.0, abs(q))


def test_p3_space_time_normalisation_1d():
    """D=1 brute-force 2-D (x, t) quadrature of the intensity surface itself on a box wide enough
    that the truncated tails are < 1e-12: confirms the tau_x^-D tau_t^-1 / h^-D normalisations and that
    the measure-zero indicator does not matter.  lambda(x,s) is typed from PAPER.md:56-60."""
    xs = np.array([[0.0, 0.9, -0.7]])
    t = np.array([0.5, 1.1, 2.0])
    th = np.array([1.4, 0.7, 1.0])
    mu0, tx, tt, xi0, h, om = 0.8, 0.6, 0.9, 0.5, 0.4, 1.1

    def lam(x, s):
        bg = mu0 / (tx * tt) * np.sum(np.exp(-0.5 * ((x - xs[0]) / tx) ** 2 - 0.5 * ((s - t) / tt) ** 2)) / (2 * math.pi)
        m = t < s
        ex = xi0 * om / h * np.sum(th[m] * np.exp(-om * (s - t[m]) - 0.5 * ((x - xs[0][m]) / h) ** 2)) / math.sqrt(2 * math.pi)
        return bg + ex

    total = 0.0
    edges = [0.0] + list(t)
    for a, b in zip(edges[:-1], edges[1:]):
        v, _ = integrate.dblquad(lam, a, b, -8.0, 8.0, epsabs=1e-11, epsrel=1e-11)
        total += v
    r = oracle.evaluate(xs, t, th, (mu0, tx, tt, xi0, h, om), grad=False)
    assert abs(r.integral - total) < 5e-9


# ------------------------------------------------------------------ P4: finite differences
def _ll(ev, theta, params):
    return oracle.evaluate(ev.x, ev.t, theta, params, grad=False).ll


def _grad(ev, theta, params):
    r = oracle.evaluate(ev.x, ev.t, theta, params)
    return np.concatenate([r.grad_theta, r.grad_hyper])


def _fd5(fun, z, i, h):
    """4th-order central difference of fun along coordinate i."""
    def at(s):
        zz = z.copy()
        zz[i] += s
        return fun(zz)
    return (-at(2 * h) + 8 * at(h) - 8 * at(-h) + at(-2 * h)) / (12 * h)


@pytest.mark.parametrize("regime,seed,dim,ties,dup", [
    ("mixed", 3, 2, False, False), ("excite", 4, 2, True, False), ("background", 5, 2, False, True),
    ("mixed", 6, 1, False, False), ("mixed", 7, 3, True, True)])
def test_p4_gradient_vs_finite_differences(regime, seed, dim, ties, dup):
    """Eq. 4 (l.137) and the derived hyperparameter gradient against central differences of Eq. 1."""
    ev = synth.small_random(24, seed, dim=dim, regime=regime, ties=ties, duplicates=dup)
    n = ev.n
    z0 = np.concatenate([ev.theta, np.array(ev.params)])
    fun = lambda z: _ll(ev, z[:n], tuple(z[n:]))
    g = _grad(ev, ev.theta, ev.params)
    for i in range(n + 6):
        h = 1e-3 * max(abs(z0[i]), 0.1)
        fd = _fd5(fun, z0, i, h)
        assert abs(fd - g[i]) < 2e-8 * max(1.0, abs(g[i])), (i, fd, g[i])


@pytest.mark.parametrize("regime,seed,dim,ties,dup", [
    ("mixed", 13, 2, False, False), ("excite", 14, 2, True, True), ("background", 15, 2, False, False),
    ("mixed", 16, 1, True, False), ("mixed", 17, 3, False, True)])
def test_p4_hessian_vs_finite_differences(regime, seed, dim, ties, dup):
    """Eq. 5 (l.143; strict '<', DESIGN R5), the dense theta-theta block, the 6x6 hyperparameter
    block and the N x 6 cross block against central differences of the GRADIENT."""
    ev = synth.small_random(14, seed, dim=dim, regime=regime, ties=ties, duplicates=dup)
    n = ev.n
    z0 = np.concatenate([ev.theta, np.array(ev.params)])
    r = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, cross=True, dense=True)
    H = np.zeros((n + 6, n + 6))
    H[:n, :n] = r.hess_theta_dense
    H[n:, n:] = r.hess_hyper
    H[:n, n:] = r.hess_cross
    H[n:, :n] = r.hess_cross.T
    assert np.allclose(np.diag(r.hess_theta_dense), r.hess_theta_diag, rtol=1e-13, atol=0)
    assert np.allclose(r.hess_hyper, r.hess_hyper.T, rtol=1e-12, atol=1e-12)
    fun = lambda z: _grad(ev, z[:n], tuple(z[n:]))
    scale = np.sqrt(np.abs(np.diag(H))) + 1e-3
    for i in range(n + 6):
        h = 1e-3 * max(abs(z0[i]), 0.1)
        col = _fd5(fun, z0, i, h)
        err = np.abs(col - H[:, i])
        tol = 5e-8 * np.maximum(np.maximum(np.abs(H[:, i]), scale * scale[i]), 1.0)
        assert np.all(err < tol), (i, np.argmax(err / tol), col, H[:, i])


# ------------------------------------------------------------------ P5: invariances
def test_p5_translation_rotation():
    ev = synth.small_random(30, 21)
    base = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params)
    c, s = math.cos(0.7), math.sin(0.7)
    R = np.array([[c, -s], [s, c]])
    x2 = R @ ev.x + np.array([[123.0], [-45.0]])
    r = oracle.evaluate(x2, ev.t, ev.theta, ev.params)
    assert abs(r.ll - base.ll) < 1e-9 * abs(base.ll)
    assert np.allclose(r.grad_theta, base.grad_theta, rtol=1e-9, atol=1e-12)
    assert np.allclose(r.grad_hyper, base.grad_hyper, rtol=1e-9, atol=1e-10)


@pytest.mark.parametrize("dim", [1, 2, 3])
def test_p5_space_scaling(dim):
    """x -> a x, tau_x -> a tau_x, h -> a h: every density picks up a^-D, ell -> ell - N D log a."""
    ev = synth.small_random(20, 22, dim=dim)
    a = 3.7
    mu0, tx, tt, xi0, h, om = ev.params
    base = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, grad=False)
    r = oracle.evaluate(a * ev.x, ev.t, ev.theta, (mu0, a * tx, tt, xi0, a * h, om), grad=False)
    assert abs(r.ll - (base.ll - ev.n * dim * math.log(a))) < 1e-10 * abs(base.ll)
    assert abs(r.integral - base.integral) < 1e-13


def test_p5_time_scaling():
    """t -> a t, tau_t -> a tau_t, omega -> omega/a: ell -> ell - N log a, Lambda unchanged."""
    ev = synth.small_random(20, 23)
    a = 2.3
    mu0, tx, tt, xi0, h, om = ev.params
    base = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, grad=False)
    r = oracle.evaluate(ev.x, a * ev.t, ev.theta, (mu0, tx, a * tt, xi0, h, om / a), grad=False)
    assert abs(r.ll - (base.ll - ev.n * math.log(a))) < 1e-10 * abs(base.ll)
    assert abs(r.integral - base.integral) < 1e-12


def test_p5_lambda_affine_in_theta():
    """lambda_n is affine in theta (l.60): lambda(theta_a + theta_b)/2 = mean of the lambdas;
    and its theta-slope row is k_{nm}: checked through Eq. 4 at a single source."""
    ev = synth.small_random(25, 24)
    tha, thb = ev.theta, ev.theta[::-1].copy()
    la = oracle.evaluate(ev.x, ev.t, tha, ev.params, grad=False).lam
    lb = oracle.evaluate(ev.x, ev.t, thb, ev.params, grad=False).lam
    lm = oracle.evaluate(ev.x, ev.t, 0.5 * (tha + thb), ev.params, grad=False).lam
    assert np.allclose(lm, 0.5 * (la + lb), rtol=1e-13)


def test_p5_ordering_of_tied_events_is_irrelevant():
    """Events with equal times may be listed in either order (strict '<', DESIGN R4)."""
    ev = synth.small_random(12, 25, ties=True)
    base = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True)
    perm = np.arange(ev.n)
    perm[[1, 2]] = perm[[2, 1]]
    r = oracle.evaluate(ev.x[:, perm], ev.t[perm], ev.theta[perm], ev.params, hess=True)
    assert abs(r.ll - base.ll) < 1e-12 * abs(base.ll)
    assert np.allclose(r.grad_theta[perm.argsort()], base.grad_theta, rtol=1e-12, atol=1e-14)
    assert np.allclose(r.hess_theta_diag[perm.argsort()], base.hess_theta_diag, rtol=1e-12, atol=1e-14)


def test_p5_tied_events_do_not_excite_each_other_and_duplicates_are_excluded():
    """Two simultaneous events at one place with nothing else: neither is earlier (l.78) and the
    coincident location is excluded from the background (l.60) => both rates are exactly zero.
    An EARLIER event at the same place does excite (k has no location indicator)."""
    x = np.array([[1.0, 1.0], [2.0, 2.0]])
    r = oracle.evaluate(x, np.array([1.0, 1.0]), np.array([1.0, 1.0]), CFG, grad=False)
    assert r.status == 1 and np.all(r.lam == 0.0)
    r = oracle.evaluate(x, np.array([1.0, 1.5]), np.array([2.0, 1.0]), CFG, grad=False)
    mu0, tx, tt, xi0, h, om = CFG
    k = xi0 * om / (2 * math.pi * h * h) * math.exp(-om * 0.5)
    assert r.lam[0] == 0.0 and rel(r.lam[1], 2.0 * k) < 1e-14


def test_p5_pure_excitation_and_pure_background_limits():
    """mu0 -> 0: only the excitation sum survives; xi0 -> 0: only the KDE background survives."""
    ev = synth.small_random(15, 26)
    mu0, tx, tt, xi0, h, om = ev.params
    full = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, grad=False).lam
    ex = oracle.evaluate(ev.x, ev.t, ev.theta, (1e-300, tx, tt, xi0, h, om), grad=False).lam
    bg = oracle.evaluate(ev.x, ev.t, ev.theta, (mu0, tx, tt, 1e-300, h, om), grad=False).lam
    assert np.allclose(ex + bg, full, rtol=1e-13)
    assert ex[0] < 1e-290          # first event has no earlier source
    assert np.all(ex[1:] > 0)


# ------------------------------------------------------------------ P7: library KDE special case
def test_p7_background_is_leave_one_out_gaussian_kde():
    """xi0 -> 0: lambda_n / mu0 is a leave-one-out Gaussian product-kernel KDE in (x/tau_x, t/tau_t)
    space (Habbema et al. indicator).  scikit-learn's KernelDensity (bandwidth 1 on the
    rescaled coordinates) is the independent evaluator."""
    from sklearn.neighbors import KernelDensity
    ev = synth.small_random(40, 31)
    mu0, tx, tt, xi0, h, om = ev.params
    lam = oracle.evaluate(ev.x, ev.t, ev.theta, (mu0, tx, tt, 1e-300, h, om), grad=False).lam
    Z = np.column_stack([ev.x[0] / tx, ev.x[1] / tx, ev.t / tt])
    n = ev.n
    for i in (0, 7, 19, 39):
        others = np.delete(Z, i, axis=0)
        kde = KernelDensity(kernel="gaussian", bandwidth=1.0, rtol=0, atol=0).fit(others)
        dens = math.exp(kde.score_samples(Z[i:i + 1])[0])       # mean of N-1 unit-bandwidth kernels
        expect = mu0 * dens * (n - 1) / (tx * tx * tt)           # Jacobian of the rescaling
        assert abs(lam[i] - expect) < 1e-10 * expect


# ------------------------------------------------------------------ internal consistency of helpers
def test_threads_do_not_change_results_and_sampled_rows_cols_agree():
    ev = synth.small_random(60, 41)
    a = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, cross=True, threads=1)
    b = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, cross=True, threads=4)
    for f in ("ll", "integral"):
        assert getattr(a, f) == getattr(b, f)
    for f in ("lam", "grad_theta", "grad_hyper", "hess_theta_diag", "hess_hyper", "hess_cross"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    idx = np.array([0, 5, 17, 59])
    lam, d1 = oracle.rows(ev.x, ev.t, ev.theta, ev.params, idx)
    assert np.array_equal(lam, a.lam[idx])
    c, d = oracle.cols(ev.x, ev.t, ev.params, a.lam, idx)
    assert np.allclose(-d, a.hess_theta_diag[idx], rtol=1e-14, atol=0)   # cols() divides by the double-rounded lambda
    # Eq. 4: grad_theta = c - xi0 (1 - exp(-omega (t_N - t_m)))
    xi0, om = ev.params[3], ev.params[5]
    assert np.allclose(c - xi0 * (1 - np.exp(-om * (ev.t[-1] - ev.t[idx]))), a.grad_theta[idx], rtol=1e-13, atol=1e-15)
    # row derivative sums reproduce the hyper-gradient's data part: sum_n d1/lambda - dLambda/dp
    lam_all, d1_all = oracle.rows(ev.x, ev.t, ev.theta, ev.params, np.arange(ev.n))
    assert np.allclose((d1_all / lam_all[:, None]).sum(0)[[1, 4]], a.grad_hyper[[1, 4]], rtol=1e-12)
    # rows(second=True) and integral(): together they rebuild the pinned evaluate()'s ell, hyper-gradient and 6x6
    # Hessian (sum_n [lambda_pq/lambda - lambda_p lambda_q/lambda^2] - Lambda_pq), in both background modes
    for bg in ("ST", "S"):
        e = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, bg=bg)
        lam_r, d1_r, d2_r = oracle.rows(ev.x, ev.t, ev.theta, ev.params, np.arange(ev.n), second=True, bg=bg)
        Lam, L1, L2 = oracle.integral(ev.t, ev.theta, ev.params, ev.dim, bg=bg)
        assert np.array_equal(lam_r, e.lam) and Lam == e.integral
        assert abs(np.sum(np.log(lam_r)) - Lam - e.ll) <= 1e-13 * abs(e.ll)
        g = (d1_r / lam_r[:, None]).sum(0) - L1
        assert np.allclose(g, e.grad_hyper, rtol=1e-11, atol=1e-11 * np.abs(d1_r / lam_r[:, None]).sum(0).max())
        r = d1_r / lam_r[:, None]
        H = (d2_r / lam_r[:, None, None] - r[:, :, None] * r[:, None, :]).sum(0) - L2
        sc = np.sqrt(np.abs(np.diag(e.hess_hyper)))
        assert np.all(np.abs(H - e.hess_hyper) <= 1e-11 * np.maximum(np.outer(sc, sc), np.abs(e.hess_hyper)) + 1e-300)
        assert np.array_equal(d2_r, np.transpose(d2_r, (0, 2, 1)))


def test_bad_arguments_are_rejected():
    ev = synth.small_random(5, 1)
    with pytest.raises(ValueError):
        oracle.evaluate(ev.x, ev.t[::-1].copy(), ev.theta, ev.params)
    with pytest.raises(ValueError):
        oracle.evaluate(ev.x, ev.t, ev.theta, (0.0, 1, 1, 1, 1, 1))


def test_generator_is_reproducible_and_has_the_configured_shape():
    a = synth.config(0)
    b = synth.config(0)
    assert np.array_equal(a.x, b.x) and np.array_equal(a.t, b.t) and np.array_equal(a.theta, b.theta)
    assert a.n == 1000 and a.dim == 2 and len(a.free_idx) == 70
    assert np.all(np.diff(a.t) >= 0) and a.t.min() >= 0 and a.t.max() <= 700
    assert np.sum(a.theta != 1.0) == 70
    c = synth.config(0, seed=1)
    assert not np.array_equal(a.t, c.t)
    u = synth.uniforms(0, 1, 200000)
    assert abs(u.mean() - 0.5) < 5e-3 and abs(u.var() - 1 / 12) < 2e-3
    z = synth.normals(0, 1, 200000)
    assert abs(z.mean()) < 1e-2 and abs(z.var() - 1) < 1e-2


# ------------------------------------------------------------------ S mode: the paper's background as printed
def test_s_mode_two_events_closed_form_and_printed_integral():
    """Paper-literal background: mu(x) = mu0 tau_x^-D sum phi_D((x-x_n)/tau_x) I[x != x_n], no time
    factor, with the integral printed at l.72, mu0 t_N (DESIGN R2).  N = 2 typed out; tau_t drops out."""
    mu0, tx, tt, xi0, h, om = 0.4, 2.5, 3.0, 0.6, 1.3, 0.45
    x = np.array([[0.3, 1.9], [-0.4, 0.8]])
    t = np.array([1.2, 2.9])
    th = np.array([1.7, 0.6])
    r2, dt = 1.6 ** 2 + 1.2 ** 2, 1.7
    B = mu0 / (2 * math.pi * tx * tx) * math.exp(-r2 / (2 * tx * tx))
    k = xi0 * om / (2 * math.pi * h * h) * math.exp(-om * dt - r2 / (2 * h * h))
    Lam = mu0 * t[1] + xi0 * th[0] * (1 - math.exp(-om * dt))
    r = oracle.evaluate(x, t, th, (mu0, tx, tt, xi0, h, om), hess=True, bg="S")
    r_tt = oracle.evaluate(x, t, th, (mu0, tx, 7.7, xi0, h, om), bg="S")
    assert abs(r.lam[0] - B) < 1e-16 and abs(r.lam[1] - (B + th[0] * k)) < 1e-16
    assert abs(r.integral - Lam) < 1e-15
    assert abs(r.ll - (math.log(B) + math.log(B + th[0] * k) - Lam)) < 1e-14
    assert r.ll == r_tt.ll                                   # tau_t is not in the model
    assert r.grad_hyper[2] == 0.0 and np.all(r.hess_hyper[2, :] == 0.0) and np.all(r.hess_hyper[:, 2] == 0.0)
    assert abs(r.grad_theta[0] - (k / (B + th[0] * k) - xi0 * (1 - math.exp(-om * dt)))) < 1e-14
    # the mode is an argument, not a state: the default model is another likelihood
    assert abs(oracle.evaluate(x, t, th, (mu0, tx, tt, xi0, h, om)).ll - r.ll) > 1.0


def test_s_mode_gradient_and_hessian_by_finite_differences():
    ev = synth.small_random(18, seed=31, regime="mixed", ties=True, duplicates=True)
    prm = np.array(ev.params)
    S = dict(bg="S")
    r = oracle.evaluate(ev.x, ev.t, ev.theta, prm, hess=True, **S)
    for a in range(6):
        e = np.zeros(6)
        e[a] = 1e-6 * prm[a]
        lp = oracle.evaluate(ev.x, ev.t, ev.theta, prm + e, **S)
        lm = oracle.evaluate(ev.x, ev.t, ev.theta, prm - e, **S)
        fd = (lp.ll - lm.ll) / (2 * e[a])
        assert abs(fd - r.grad_hyper[a]) <= 1e-7 * max(1.0, abs(r.grad_hyper[a]))
        fdh = (lp.grad_hyper - lm.grad_hyper) / (2 * e[a])
        assert np.max(np.abs(fdh - r.hess_hyper[a]) / np.maximum(1.0, np.abs(r.hess_hyper[a]))) <= 2e-6
    for m in (0, 5, 17):
        e = np.zeros(ev.n)
        e[m] = 1e-6
        fd = (oracle.evaluate(ev.x, ev.t, ev.theta + e, prm, **S).ll - oracle.evaluate(ev.x, ev.t, ev.theta - e, prm, **S).ll) / 2e-6
        assert abs(fd - r.grad_theta[m]) <= 1e-7 * max(1.0, abs(r.grad_theta[m]))


def test_s_mode_background_is_the_leave_one_out_kde():
    """With xi0 -> 0 every lambda_n is mu0 N' times the leave-one-out Gaussian KDE of the other locations
    (scikit-learn's KernelDensity, an independent library routine)."""
    from sklearn.neighbors import KernelDensity
    ev = synth.small_random(40, seed=33, regime="background")
    mu0, tx = 0.7, 0.9
    r = oracle.evaluate(ev.x, ev.t, ev.theta, (mu0, tx, 1.0, 1e-300, 0.5, 1.0), bg="S")
    X = ev.x.T
    for n in (0, 7, 39):
        others = np.delete(X, n, axis=0)
        kde = KernelDensity(kernel="gaussian", bandwidth=tx).fit(others)
        dens = math.exp(kde.score_samples(X[n:n + 1])[0])      # mean of the kernels
        assert abs(r.lam[n] - mu0 * len(others) * dens) <= 1e-10 * r.lam[n]


def test_cross_abs_scale_brute_force_and_triangle_inequality():
    """oracle.cross_abs, the entry-wise error scale of the cross block (used by the GPU parity tests,
    not an output of the method): typed out here as a double loop from its definition, bounded below by the block itself
    (triangle inequality) and equal to it where no term changes sign (column mu0: the bracket is -SB_n / (mu0 lambda_n))."""
    ev = synth.small_random(40, seed=77, ties=True, duplicates=True)
    ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, cross=True, row_d1=True)
    A = oracle.cross_abs(ev.x, ev.t, ev.params, ref.lam, ref.row_d1)
    mu0, tx, tt, xi0, h, om = ev.params
    n, D = ev.n, ev.dim
    B = np.zeros((n, 6))
    for m in range(n):
        for i in range(n):
            dt = ev.t[i] - ev.t[m]
            if not dt > 0:
                continue
            r2 = float(np.sum((ev.x[:, i] - ev.x[:, m]) ** 2))
            k = xi0 * om * (2 * np.pi) ** (-D / 2) * h ** (-D) * np.exp(-om * dt - r2 / (2 * h * h))
            a = k / ref.lam[i]
            T = np.array([0, 0, 0, 1 / xi0, r2 / h ** 3 + D / h, 1 / om + dt])
            B[m] += a * (T + np.abs(ref.row_d1[i]) / ref.lam[i])
    assert np.allclose(A, B, rtol=1e-12, atol=0)
    Tm = ev.t[-1] - ev.t
    S = ref.hess_cross.copy()                     # the pair sums alone: add the integral part back
    S[:, 3] += -np.expm1(-om * Tm)
    S[:, 5] += xi0 * Tm * np.exp(-om * Tm)
    assert np.all(np.abs(S) <= A * (1 + 1e-12) + 1e-300)
    assert np.allclose(np.abs(S[:, 0]), A[:, 0], rtol=1e-12, atol=1e-300)
    assert np.all(A[:, 3:] > np.abs(S[:, 3:])[:, :] - 1e-300) and A[:-2].min() >= 0
