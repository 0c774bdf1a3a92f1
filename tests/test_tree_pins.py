"""Pins for the oracle of the phylogenetic-diffusion prior and of the z-parametrisation (oracle/tree_ref.cpp,
oracle/tree.py): closed forms, a hand-written V_G, the generative description of the Brownian process
marginalised with dense linear algebra, a library multivariate-normal density, Sherman-Morrison on a star tree,
finite differences.  CPU only.  PAPER.md line numbers in the docstrings."""
import json
import math
import os

import numpy as np
import pytest
from scipy import stats

import oracle
from oracle import tree as otree
from paper_2103_03348_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def test_t1_single_tip_closed_form():
    """M=1: the tip is the root, d_F(root, tip) = 0 => V_G = [tau0] and Eq. 2 (l.101) is the
    N(0, sigma^2 tau0) density (root value ~ N(0, tau0 sigma^2), l.99)."""
    tau0, s2, z = 0.3, 0.7, 0.45
    V = otree.vg([-1], [0.0], 1, tau0)
    assert V.shape == (1, 1) and V[0, 0] == tau0
    lp, g = otree.log_prior(V, [z], s2)
    assert abs(lp - (-0.5 * math.log(2 * math.pi * s2 * tau0) - z * z / (2 * s2 * tau0))) < 1e-15
    assert abs(g[0] + z / (s2 * tau0)) < 1e-15


def test_t2_two_tips_closed_form():
    """M=2: root with two tips on branches w1, w2: V = [[tau0+w1, tau0], [tau0, tau0+w2]] (l.103: diagonal =
    tau0 + root-to-tip, off-diagonal = tau0 + root-to-MRCA = tau0); bivariate normal typed out from Eq. 2."""
    tau0, s2, w1, w2 = 0.1, 0.25, 0.5, 0.7
    z1, z2 = 0.3, -0.2
    V = otree.vg([2, 2, -1], [w1, w2, 0.0], 2, tau0)
    assert np.allclose(V, [[tau0 + w1, tau0], [tau0, tau0 + w2]], rtol=0, atol=1e-16)
    det = (tau0 + w1) * (tau0 + w2) - tau0 * tau0
    quad = (z1 * z1 * (tau0 + w2) - 2 * z1 * z2 * tau0 + z2 * z2 * (tau0 + w1)) / det
    lp_expected = -math.log(2 * math.pi * s2) - 0.5 * math.log(det) - quad / (2 * s2)
    lp, g = otree.log_prior(V, [z1, z2], s2)
    assert abs(lp - lp_expected) < 1e-14
    g_expected = [-((tau0 + w2) * z1 - tau0 * z2) / det / s2, -((tau0 + w1) * z2 - tau0 * z1) / det / s2]
    assert np.allclose(g, g_expected, rtol=1e-14, atol=0)


def test_t3_hand_written_four_tip_vg():
    """V_G of the tree ((0:1.0, 1:2.0):0.5, (2:0.3, 3:0.4):1.5) written by hand from l.103
    (tests/golden/tree_examples.json)."""
    ex = json.load(open(os.path.join(HERE, "golden", "tree_examples.json")))["four_tips"]
    V = otree.vg(ex["parent"], ex["branch"], 4, ex["tau0"])
    assert np.allclose(V, np.array(ex["V"]), rtol=0, atol=1e-15)


def _joint_precision(parent, branch, tau0, s2):
    """Precision matrix of ALL node values from the generative description: root ~ N(0, tau0 s2),
    child | parent ~ N(parent, w_child s2)."""
    nn = len(parent)
    Q = np.zeros((nn, nn))
    for v in range(nn):
        p = parent[v]
        if p < 0:
            Q[v, v] += 1.0 / (tau0 * s2)
        else:
            q = 1.0 / (branch[v] * s2)
            Q[v, v] += q
            Q[p, p] += q
            Q[v, p] -= q
            Q[p, v] -= q
    return Q


@pytest.mark.parametrize("M,seed", [(2, 0), (5, 1), (12, 2), (40, 3)])
def test_t4_generative_process_marginalised_to_tips(M, seed):
    """The covariance of the tips under the Brownian process on the tree, obtained by inverting the joint precision
    of all 2M-1 nodes, equals sigma^2 V_G, and Eq. 2 equals scipy's multivariate normal log-density."""
    times = np.sort(synth.uniforms(seed, 200, M) * 300.0)
    tr = synth.make_tree(times, seed)
    tau0, s2 = 0.15, 0.4
    V = otree.vg(tr.parent, tr.branch, M, tau0)
    cov_all = np.linalg.inv(_joint_precision(tr.parent, tr.branch, tau0, s2))
    assert np.allclose(cov_all[:M, :M], s2 * V, rtol=1e-9, atol=1e-12)
    z = synth.normals(seed, 210, M) * 0.6
    lp, _ = otree.log_prior(V, z, s2)
    lp_lib = stats.multivariate_normal(mean=np.zeros(M), cov=s2 * V, allow_singular=False).logpdf(z)
    assert abs(lp - lp_lib) <= 1e-9 * max(1.0, abs(lp_lib))


def test_t5_star_tree_sherman_morrison():
    """Caterpillar whose internal branches have length 0 is a star: V = tau0 11^T + diag(w) (l.103), so
    |V| = prod w (1 + tau0 sum 1/w) and z^T V^-1 z = sum z^2/w - tau0 (sum z/w)^2 / (1 + tau0 sum 1/w)."""
    M, tau0, s2 = 6, 0.2, 0.3
    w = np.array([0.5, 0.9, 0.3, 1.4, 0.7, 1.1])
    z = np.array([0.2, -0.5, 0.9, 0.1, -0.3, 0.4])
    # tips 0..5; internal 6 = (0,1), 7 = (6,2), 8 = (7,3), 9 = (8,4), 10 = (9,5) = root; internal branches 0
    parent = [6, 6, 7, 8, 9, 10, 7, 8, 9, 10, -1]
    branch = list(w) + [0.0, 0.0, 0.0, 0.0, 0.0]
    V = otree.vg(parent, branch, M, tau0)
    assert np.allclose(V, tau0 * np.ones((M, M)) + np.diag(w), rtol=0, atol=1e-15)
    denom = 1 + tau0 * np.sum(1 / w)
    logdet = np.sum(np.log(w)) + math.log(denom)
    quad = np.sum(z * z / w) - tau0 * np.sum(z / w) ** 2 / denom
    lp_expected = -0.5 * M * math.log(2 * math.pi * s2) - 0.5 * logdet - quad / (2 * s2)
    lp, g = otree.log_prior(V, z, s2)
    assert abs(lp - lp_expected) < 1e-13
    g_expected = -(z / w - tau0 * np.sum(z / w) / denom / w) / s2
    assert np.allclose(g, g_expected, rtol=1e-13, atol=0)


def test_t6_gradient_by_finite_differences():
    M, seed = 25, 7
    tr = synth.make_tree(np.sort(synth.uniforms(seed, 200, M) * 500.0), seed)
    V = otree.vg(tr.parent, tr.branch, M, 0.1)
    z = synth.normals(seed, 210, M) * 0.5
    _, g = otree.log_prior(V, z, 0.25)
    for k in range(M):
        e = np.zeros(M)
        e[k] = 1e-5
        fd = (otree.log_prior(V, z + e, 0.25, grad=False)[0] - otree.log_prior(V, z - e, 0.25, grad=False)[0]) / 2e-5
        assert abs(fd - g[k]) <= 1e-7 * max(1.0, abs(g[k]))


def test_t7_vg_path_sums_equal_mrca_form():
    """l.103 gives two descriptions of the off-diagonal entries (path-length formula; root-to-MRCA time).
    The oracle uses the first; here the second is written independently in Python."""
    M, seed, tau0 = 30, 11, 0.05
    tr = synth.make_tree(np.sort(synth.uniforms(seed, 200, M) * 400.0), seed)
    par, br = tr.parent, tr.branch
    nn = 2 * M - 1
    dist = np.zeros(nn)
    for v in range(nn - 2, -1, -1):
        dist[v] = dist[par[v]] + br[v]

    def ancestors(v):
        out = [v]
        while par[v] >= 0:
            v = par[v]
            out.append(v)
        return out

    V2 = np.zeros((M, M))
    for i in range(M):
        ai = ancestors(i)
        for j in range(M):
            aj = set(ancestors(j))
            mrca = next(a for a in ai if a in aj)
            V2[i, j] = tau0 + dist[mrca]
    assert np.allclose(otree.vg(par, br, M, tau0), V2, rtol=1e-13, atol=1e-15)


def test_t8_z_parametrisation_chain_rule_by_finite_differences():
    """theta(z) of PAPER.md:97 with f(t) = t (l.202); d ell/dz, d2 ell/dz^2 (diagonal) and d ell/dbeta of
    oracle.tree.z_chain against central differences of the oracle's log-likelihood / gradient."""
    ev = synth.small_random(24, seed=5, regime="mixed")
    idx = np.array([1, 4, 5, 9, 16, 23], dtype=np.int64)
    z = np.array([0.3, -0.2, 0.5, 0.1, -0.4, 0.25])
    beta = 0.03
    n = ev.n

    def ell(zv, b):
        th = otree.theta_from_z(n, idx, zv, b, ev.t)
        return oracle.evaluate(ev.x, ev.t, th, ev.params, grad=False).ll

    th = otree.theta_from_z(n, idx, z, beta, ev.t)
    assert np.all(np.delete(th, idx) == 1.0) and np.allclose(th[idx], np.exp(z + beta * ev.t[idx]), rtol=1e-15)
    r = oracle.evaluate(ev.x, ev.t, th, ev.params, hess=True)
    gz, hz, gb = otree.z_chain(th, ev.t, idx, r.grad_theta, r.hess_theta_diag)
    for k in range(len(idx)):
        e = np.zeros(len(idx))
        e[k] = 1e-5
        fd1 = (ell(z + e, beta) - ell(z - e, beta)) / 2e-5
        assert abs(fd1 - gz[k]) <= 2e-7 * max(1.0, abs(gz[k]))
        fd2 = (ell(z + e, beta) - 2 * ell(z, beta) + ell(z - e, beta)) / 1e-10
        assert abs(fd2 - hz[k]) <= 2e-4 * max(1.0, abs(hz[k]))
    fdb = (ell(z, beta + 1e-6) - ell(z, beta - 1e-6)) / 2e-6
    assert abs(fdb - gb) <= 1e-6 * max(1.0, abs(gb))


def test_t9_config_tree_generator_shape():
    """BASELINE.json configs[2] stand-in: 1,610 tips dated by the sequenced events, rooted binary tree, mean
    root-to-tip distance 1, z with marginal variance about sigma^2 (tau0 + 1) ~ 0.27."""
    ev, tr, z = synth.config_tree(seed=0, n=3000, n_centres=8, n_free=200)
    M = tr.n_tips
    assert M == 200 and tr.parent.shape == (2 * M - 1,) and np.sum(tr.parent < 0) == 1
    assert np.all(np.bincount(tr.parent[tr.parent >= 0], minlength=2 * M - 1)[M:] == 2)
    assert np.all(tr.branch >= 0)
    assert np.allclose(ev.theta[ev.free_idx], np.exp(z)) and np.all(np.delete(ev.theta, ev.free_idx) == 1.0)
    V = otree.vg(tr.parent, tr.branch, M, 0.0)
    assert abs(np.mean(np.diag(V)) - 1.0) < 1e-12


def test_t10_prior_precision_diagonal():
    """diag(V_G^-1)/sigma^2 (the prior's own curvature, -d2 log p/dz_m^2): 2x2 closed form, the star tree by
    Sherman-Morrison ((V^-1)_ii = 1/w_i - tau0 / (w_i^2 (1 + tau0 sum 1/w))), numpy's inverse on a random tree, and
    central differences of the oracle's own gradient."""
    tau0, s2, w1, w2 = 0.1, 0.25, 0.5, 0.7
    V = otree.vg([2, 2, -1], [w1, w2, 0.0], 2, tau0)
    det = (tau0 + w1) * (tau0 + w2) - tau0 * tau0
    assert np.allclose(otree.precision_diag(V, s2), [(tau0 + w2) / det / s2, (tau0 + w1) / det / s2], rtol=1e-14)
    w = np.array([0.5, 0.9, 0.3, 1.4, 0.7, 1.1])
    parent = [6, 6, 7, 8, 9, 10, 7, 8, 9, 10, -1]
    V = otree.vg(parent, list(w) + [0.0] * 5, 6, 0.2)
    denom = 1 + 0.2 * np.sum(1 / w)
    assert np.allclose(otree.precision_diag(V, 0.3), (1 / w - 0.2 / (w * w * denom)) / 0.3, rtol=1e-13)
    M, seed = 35, 13
    tr = synth.make_tree(np.sort(synth.uniforms(seed, 200, M) * 500.0), seed)
    V = otree.vg(tr.parent, tr.branch, M, 0.1)
    pd = otree.precision_diag(V, 0.25)
    assert np.allclose(pd, np.diag(np.linalg.inv(V)) / 0.25, rtol=1e-8)
    z = synth.normals(seed, 210, M) * 0.5
    for k in (0, 7, 34):
        e = np.zeros(M)
        e[k] = 1e-4
        fd = (otree.log_prior(V, z + e, 0.25)[1][k] - otree.log_prior(V, z - e, 0.25)[1][k]) / 2e-4
        assert abs(-fd - pd[k]) <= 1e-7 * pd[k]
