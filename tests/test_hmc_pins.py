"""Pins for the HMC oracle (oracle/hmc.py): the leapfrog map against its closed form on a quadratic potential,
time reversibility, second-order energy error, the accept rule on hand-made energies, the running-average
preconditioner, and one iteration on a Hawkes posterior re-traced by hand.  CPU only."""
import math

import numpy as np

from oracle import hmc
from oracle import tree as otree
from paper_2103_03348_b200 import synth


def gaussian_target(prec):
    prec = np.asarray(prec, float)

    def target(z, hess):
        return -0.5 * float(np.sum(prec * z * z)), -prec * z, (prec.copy() if hess else None)

    return target


def test_h1_leapfrog_closed_form_harmonic_oscillator():
    """For log pi = -a z^2/2 and mass m one leapfrog step is the linear map
    z' = (1 - eps^2 a/(2m)) z + (eps/m) p,  p' = -eps a (1 - eps^2 a/(4m)) z + (1 - eps^2 a/(2m)) p  (textbook)."""
    a, m, eps = 2.3, 0.7, 0.11
    z0, p0 = np.array([0.8]), np.array([-0.4])
    tgt = gaussian_target([a])
    A = np.array([[1 - eps * eps * a / (2 * m), eps / m],
                  [-eps * a * (1 - eps * eps * a / (4 * m)), 1 - eps * eps * a / (2 * m)]])
    s = np.array([z0[0], p0[0]])
    for steps in (1, 2, 7):
        z, p, logpi, grad = hmc.leapfrog(tgt, z0, p0, -a * z0, np.array([m]), eps, steps)
        s_expected = np.linalg.matrix_power(A, steps) @ s
        assert abs(z[0] - s_expected[0]) < 1e-14 and abs(p[0] - s_expected[1]) < 1e-14
        assert abs(logpi + 0.5 * a * z[0] ** 2) < 1e-15 and abs(grad[0] + a * z[0]) < 1e-15


def test_h2_leapfrog_reversible_and_second_order():
    M = 6
    prec = 0.5 + synth.uniforms(1, 300, M) * 3
    mass = 0.3 + synth.uniforms(1, 301, M)
    z0 = synth.normals(1, 302, M)
    p0 = synth.normals(1, 303, M)
    tgt = gaussian_target(prec)
    z1, p1, _, g1 = hmc.leapfrog(tgt, z0, p0, -prec * z0, mass, 0.05, 9)
    z2, p2, _, _ = hmc.leapfrog(tgt, z1, -p1, g1, mass, 0.05, 9)
    assert np.allclose(z2, z0, rtol=0, atol=1e-13) and np.allclose(-p2, p0, rtol=0, atol=1e-13)
    H = lambda z, p: 0.5 * np.sum(prec * z * z) + 0.5 * np.sum(p * p / mass)
    errs = []
    for eps, steps in ((0.08, 10), (0.04, 20), (0.02, 40)):
        z, p, _, _ = hmc.leapfrog(tgt, z0, p0, -prec * z0, mass, eps, steps)
        errs.append(abs(H(z, p) - H(z0, p0)))
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0      # error ~ eps^2


def test_h3_accept_rule_trace_and_preconditioner():
    """One-dimensional Gaussian target, so that every quantity of two iterations can be re-traced by hand."""
    a, eps, L, floor = 1.7, 0.2, 3, 0.5
    tgt = gaussian_target([a])
    normals = np.array([[0.9], [-1.3], [0.4]])
    z0 = np.array([0.6])
    out_acc = hmc.run(tgt, z0, normals, np.array([1e-300, 1e-300, 1e-300]), 3, L, eps, 2, np.array([1.0]), floor)
    out_rej = hmc.run(tgt, z0, normals, np.array([1.0, 1.0, 1.0]), 3, L, eps, 2, np.array([1.0]), floor)
    # by hand: refresh at it = 0 and it = 2 with h = a (> floor): mass = 1 + (a - 1)/1 = a, then a + (a - a)/2 = a
    assert abs(out_acc["mass"][0] - a) < 1e-15
    A = lambda m: np.array([[1 - eps * eps * a / (2 * m), eps / m],
                            [-eps * a * (1 - eps * eps * a / (4 * m)), 1 - eps * eps * a / (2 * m)]])
    z = z0[0]
    for it in range(3):
        p = math.sqrt(a) * normals[it, 0]
        h_old = 0.5 * a * z * z + 0.5 * p * p / a
        z1, p1 = np.linalg.matrix_power(A(a), L) @ np.array([z, p])
        h_new = 0.5 * a * z1 * z1 + 0.5 * p1 * p1 / a
        assert abs(out_acc["trace"][it, 1] - h_old) < 1e-13 and abs(out_acc["trace"][it, 2] - h_new) < 1e-13
        assert out_acc["trace"][it, 3] == 1.0 and abs(out_acc["trace"][it, 0] + 0.5 * a * z1 * z1) < 1e-13
        z = z1
    assert abs(out_acc["z"][0] - z) < 1e-13
    # u = 1: log u = 0 < H_old - H_new only if the energy went down
    zr = z0[0]
    for it in range(3):
        went_down = out_rej["trace"][it, 2] < out_rej["trace"][it, 1]
        assert out_rej["trace"][it, 3] == (1.0 if went_down else 0.0)
    # floor: a target flatter than the floor gets mass = floor
    out_f = hmc.run(gaussian_target([0.1]), z0, normals, np.ones(3), 1, 1, 0.1, 1, np.array([3.0]), floor)
    assert out_f["mass"][0] == floor


def test_h4_hawkes_target_is_ell_plus_prior():
    """hawkes_target = ell(theta(z)) + Eq. 2, gradient by the chain rule: finite-difference check of the sum."""
    ev = synth.small_random(20, seed=9, regime="mixed")
    idx = np.array([2, 5, 11, 17], dtype=np.int64)
    tree = synth.make_tree(ev.t[idx], 9)
    V = otree.vg(tree.parent, tree.branch, 4, 0.1)
    tgt = hmc.hawkes_target(ev.x, ev.t, idx, 0.01, ev.params, V, 0.25)
    z = np.array([0.2, -0.3, 0.4, 0.05])
    lp, g, h = tgt(z, True)
    for k in range(4):
        e = np.zeros(4)
        e[k] = 1e-5
        fd = (tgt(z + e, False)[0] - tgt(z - e, False)[0]) / 2e-5
        assert abs(fd - g[k]) <= 2e-7 * max(1.0, abs(g[k]))
    assert h.shape == (4,)


def test_h5_prior_precision_adds_to_the_mass():
    """With prior_prec = P the dynamics use M = A + P: one-dimensional Gaussian target re-traced by hand."""
    a, P, eps, L = 1.7, 0.9, 0.2, 2
    tgt = gaussian_target([a])
    out = hmc.run(tgt, np.array([0.6]), np.array([[0.9]]), np.array([1e-300]), 1, L, eps, 1, np.array([1.0]), 0.5,
                  prior_prec=np.array([P]))
    m = a + P                                  # A = a after the first refresh
    assert abs(out["mass"][0] - a) < 1e-15
    A = np.array([[1 - eps * eps * a / (2 * m), eps / m],
                  [-eps * a * (1 - eps * eps * a / (4 * m)), 1 - eps * eps * a / (2 * m)]])
    p = math.sqrt(m) * 0.9
    z1, p1 = np.linalg.matrix_power(A, L) @ np.array([0.6, p])
    assert abs(out["z"][0] - z1) < 1e-14
    assert abs(out["trace"][0, 1] - (0.5 * a * 0.36 + 0.5 * p * p / m)) < 1e-14
    assert abs(out["trace"][0, 2] - (0.5 * a * z1 * z1 + 0.5 * p1 * p1 / m)) < 1e-14
