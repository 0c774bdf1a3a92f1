"""GPU parity of the O(M) phylogenetic-diffusion prior, the z-parametrisation and the fused z-posterior
(include/hawkes.h: hawkes_tree_*, hawkes_theta_from_z, hawkes_z_chain, hawkes_posterior_z) against the dense
oracle (oracle/tree_ref.cpp, oracle/tree.py, oracle/hawkes_ref.cpp).  Same 1e-10 bar as the likelihood:
|gpu - oracle| <= 1e-10 max(|oracle|, scale), scale = sum of the magnitudes of the terms that form the entry."""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import tree as otree
from paper_2103_03348_b200 import synth
from parity import check

pytestmark = pytest.mark.gpu
THREADS = min(os.cpu_count() or 1, 32)


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def prior_scales(V, z, s2):
    """log p = -M/2 log(2 pi s2) - 1/2 log|V| - q/(2 s2): scale = sum of the three magnitudes; gradient entry
    k = -(V^-1 z)_k / s2: scale = sum_j |V^-1_kj z_j| / s2."""
    M = len(z)
    Vi = np.linalg.inv(V)
    sign, logdet = np.linalg.slogdet(V)
    q = float(z @ Vi @ z)
    lp_scale = 0.5 * M * abs(math.log(2 * math.pi * s2)) + 0.5 * abs(logdet) + q / (2 * s2)
    g_scale = (np.abs(Vi) @ np.abs(z)) / s2
    return lp_scale, g_scale


def run_prior(torch, hp, parent, branch, z, s2, tau0):
    tr = hp.HawkesTree(parent, branch, 0)
    lp, g = tr.prior(dev(torch, z), s2, tau0)
    torch.cuda.synchronize()
    return tr, float(lp.item()), g.cpu().numpy()


@pytest.mark.parametrize("M,seed,tau0", [(1, 0, 0.3), (2, 1, 0.1), (3, 2, 0.1), (7, 3, 0.0), (64, 4, 0.1), (333, 5, 0.02)])
def test_tree_prior_small_trees(torch, M, seed, tau0):
    import paper_2103_03348_b200 as hp
    tt = np.sort(synth.uniforms(seed, 200, M) * 600.0)
    tree = synth.make_tree(tt, seed)
    z = synth.normals(seed, 210, M) * 0.5
    s2 = 0.25
    if M == 1 and tau0 == 0.0:
        tau0 = 0.3
    V = otree.vg(tree.parent, tree.branch, M, tau0)
    lp_o, g_o = otree.log_prior(V, z, s2)
    _, lp, g = run_prior(torch, hp, tree.parent, tree.branch, z, s2, tau0)
    lps, gs = prior_scales(V, z, s2)
    check("logp", lp, lp_o, lps)
    check("grad_z", g, g_o, gs)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    check("prior precision diagonal", tr.precision_diag(s2, tau0).cpu().numpy(), otree.precision_diag(V, s2))


def test_tree_prior_config2_full_size_and_determinism(torch):
    """BASELINE.json configs[2]: 1,610 tips (147 levels deep), sigma^2 = 0.25, tau0 = 0.1."""
    import paper_2103_03348_b200 as hp
    ev, tree, z = synth.config_tree(0)
    M = tree.n_tips
    assert M == 1610
    V = otree.vg(tree.parent, tree.branch, M, synth.TREE_TAU0)
    lp_o, g_o = otree.log_prior(V, z, synth.TREE_SIGMA2)
    tr, lp, g = run_prior(torch, hp, tree.parent, tree.branch, z, synth.TREE_SIGMA2, synth.TREE_TAU0)
    lps, gs = prior_scales(V, z, synth.TREE_SIGMA2)
    check("logp", lp, lp_o, lps)
    check("grad_z", g, g_o, gs)
    assert tr.levels() >= 10
    lp2, g2 = tr.prior(dev(torch, z), synth.TREE_SIGMA2, synth.TREE_TAU0)
    assert float(lp2.item()) == lp and np.array_equal(g2.cpu().numpy(), g)      # bit-identical run to run
    lp3, none = tr.prior(dev(torch, z), synth.TREE_SIGMA2, synth.TREE_TAU0, grad=False)
    assert none is None and float(lp3.item()) == lp
    pd = tr.precision_diag(synth.TREE_SIGMA2, synth.TREE_TAU0).cpu().numpy()
    check("prior precision diagonal", pd, otree.precision_diag(V, synth.TREE_SIGMA2))


@pytest.mark.parametrize("M", [500, 8000])
def test_tree_prior_star_caterpillar_closed_form(torch, M):
    """Caterpillar with zero-length internal branches = star tree: closed form by Sherman-Morrison (pinned in
    tests/test_tree_pins.py::test_t5).  M-1 levels deep; M = 8000 exceeds the shared-memory node store and takes
    the global-scratch path."""
    import paper_2103_03348_b200 as hp
    tau0, s2 = 0.2, 0.3
    w = 0.2 + synth.uniforms(9, 220, M)
    z = synth.normals(9, 221, M) * 0.4
    parent = np.empty(2 * M - 1, dtype=np.int32)
    branch = np.zeros(2 * M - 1)
    branch[:M] = w
    parent[0] = parent[1] = M
    for k in range(2, M):
        parent[k] = M + k - 1          # tip k joins internal node M + k - 1
        parent[M + k - 2] = M + k - 1  # previous internal node joins it too
    parent[2 * M - 2] = -1
    denom = 1 + tau0 * np.sum(1 / w)
    logdet = np.sum(np.log(w)) + math.log(denom)
    quad = np.sum(z * z / w) - tau0 * np.sum(z / w) ** 2 / denom
    lp_o = -0.5 * M * math.log(2 * math.pi * s2) - 0.5 * logdet - quad / (2 * s2)
    g_o = -(z / w - tau0 * np.sum(z / w) / denom / w) / s2
    tr, lp, g = run_prior(torch, hp, parent, branch, z, s2, tau0)
    assert tr.levels() == M - 1
    lps = 0.5 * M * abs(math.log(2 * math.pi * s2)) + 0.5 * (np.sum(np.abs(np.log(w))) + math.log(denom)) + \
        (np.sum(z * z / w) + tau0 * np.sum(z / w) ** 2 / denom) / (2 * s2)
    gs = (np.abs(z) / w + tau0 * np.sum(np.abs(z) / w) / denom / w) / s2
    check("logp", lp, lp_o, lps)
    check("grad_z", g, g_o, gs)


def test_tree_create_rejects_malformed_trees(torch):
    import paper_2103_03348_b200 as hp
    good_parent, good_branch = [4, 4, 5, 5, 6, 6, -1], [1.0, 2.0, 0.3, 0.4, 0.5, 1.5, 0.0]
    hp.HawkesTree(good_parent, good_branch, 0).close()
    bad = [
        ([4, 4, 5, 5, 6, 6, 6], good_branch),            # no root
        ([4, 4, 5, 5, -1, 6, -1], good_branch),          # two roots
        ([4, 4, 4, 5, 6, 6, -1], good_branch),           # three children / one child
        ([4, 4, 5, 5, 5, 4, -1], good_branch),           # cycle between internal nodes
        ([1, 4, 5, 5, 6, 6, -1], good_branch),           # a tip as parent
        (good_parent, [1.0, -2.0, 0.3, 0.4, 0.5, 1.5, 0.0]),          # negative branch
        (good_parent, [1.0, float("nan"), 0.3, 0.4, 0.5, 1.5, 0.0]),  # non-finite branch
    ]
    for par, br in bad:
        with pytest.raises(hp.HawkesError) as e:
            hp.HawkesTree(par, br, 0)
        assert e.value.status == hp.ERR_ARG
    tr = hp.HawkesTree(good_parent, good_branch, 0)
    z = dev(torch, np.zeros(4))
    for s2, t0 in [(0.0, 0.1), (-1.0, 0.1), (float("nan"), 0.1), (0.25, -0.1)]:
        with pytest.raises(hp.HawkesError) as e:
            tr.prior(z, s2, t0)
        assert e.value.status == hp.ERR_PARAM


def test_theta_from_z_and_chain_rule(torch):
    import paper_2103_03348_b200 as hp
    ev = synth.make_events(3000, seed=4, n_centres=10, n_free=200)
    ev.x *= 0.05
    n, idx = ev.n, ev.free_idx
    z = synth.normals(4, 230, len(idx)) * 0.5
    beta = 0.002
    ctx = hp.HawkesContext(n, ev.dim, 0)
    th = ctx.theta_from_z(n, dev(torch, idx), dev(torch, z), beta, dev(torch, ev.t))
    th_o = otree.theta_from_z(n, idx, z, beta, ev.t)
    # exp: same argument on both sides, library exp on both: a few ulp
    check("theta", th.cpu().numpy(), th_o, tol=1e-14)
    ref = oracle.evaluate(ev.x, ev.t, th_o, ev.params, hess=True, threads=THREADS)
    gz_o, hz_o, gb_o = otree.z_chain(th_o, ev.t, idx, ref.grad_theta, ref.hess_theta_diag)
    r = ctx.eval(dev(torch, ev.x), dev(torch, ev.t), dev(torch, th_o), ev.params,
                 hp.WANT_LL | hp.WANT_GRAD_THETA | hp.WANT_HESS_THETA)
    gz, hz, gb = ctx.z_chain(dev(torch, idx), dev(torch, th_o), dev(torch, ev.t), r.grad_theta, r.hess_theta_diag,
                             want_beta=True)
    xi0, om = ev.params[3], ev.params[5]
    integ = xi0 * (-np.expm1(-om * (ev.t[-1] - ev.t)))
    gscale = (np.abs(ref.grad_theta + integ) + integ)[idx] * th_o[idx]          # theta (|c_m| + |xi0 (1 - E_m)|)
    check("grad_z", gz.cpu().numpy(), gz_o, gscale)
    check("hess_z", hz.cpu().numpy(), hz_o, th_o[idx] ** 2 * np.abs(ref.hess_theta_diag[idx]) + gscale)
    check("grad_beta", gb.item(), gb_o, float(np.sum(ev.t[idx] * gscale)))


def posterior_case(torch, ev, tree, z, s2, tau0, beta=0.0):
    import paper_2103_03348_b200 as hp
    n, idx = ev.n, ev.free_idx
    ctx = hp.HawkesContext(n, ev.dim, 0)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    out = ctx.posterior_z(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), dev(torch, z), beta, ev.params, s2,
                          tau0, hess=True)
    assert ctx.last_status() == 0
    out3, gz, hz = (o.cpu().numpy() for o in out)
    th_o = otree.theta_from_z(n, idx, z, beta, ev.t)
    ref = oracle.evaluate(ev.x, ev.t, th_o, ev.params, hess=True, threads=THREADS)
    V = otree.vg(tree.parent, tree.branch, tree.n_tips, tau0)
    lp_o, pg_o = otree.log_prior(V, z, s2)
    gz_o, hz_o, _ = otree.z_chain(th_o, ev.t, idx, ref.grad_theta, ref.hess_theta_diag)
    lps, pgs = prior_scales(V, z, s2)
    ll_scale = float(np.sum(np.abs(np.log(ref.lam)))) + abs(ref.integral)
    check("ell", out3[0], ref.ll, ll_scale)
    check("log prior", out3[1], lp_o, lps)
    check("log posterior", out3[2], ref.ll + lp_o, ll_scale + lps)
    xi0, om = ev.params[3], ev.params[5]
    integ = xi0 * (-np.expm1(-om * (ev.t[-1] - ev.t)))
    gscale = (np.abs(ref.grad_theta + integ) + integ)[idx] * th_o[idx]
    check("grad_z", gz, gz_o + pg_o, gscale + pgs)
    check("hess_z", hz, hz_o, th_o[idx] ** 2 * np.abs(ref.hess_theta_diag[idx]) + gscale)
    # buffers are reusable and the call is deterministic
    out_b = ctx.posterior_z(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), dev(torch, z), beta, ev.params, s2,
                            tau0, hess=True)
    assert all(np.array_equal(a.cpu().numpy(), b) for a, b in zip(out_b, (out3, gz, hz)))
    # hawkes_posterior_z_skip: the same posterior over the work lists of hawkes_skip_plan, against the same oracle values
    with pytest.raises(hp.HawkesError):
        ctx.posterior_z(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), dev(torch, z), beta, ev.params, s2, tau0,
                        hess=True, skip=True)
    ctx.skip_plan(dev(torch, ev.x), dev(torch, ev.t), ev.params)
    out_s = ctx.posterior_z(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), dev(torch, z), beta, ev.params, s2,
                            tau0, hess=True, skip=True)
    assert ctx.last_status() == 0
    o3s, gzs, hzs = (o.cpu().numpy() for o in out_s)
    check("ell (skip)", o3s[0], ref.ll, ll_scale)
    check("log posterior (skip)", o3s[2], ref.ll + lp_o, ll_scale + lps)
    check("grad_z (skip)", gzs, gz_o + pg_o, gscale + pgs)
    check("hess_z (skip)", hzs, hz_o, th_o[idx] ** 2 * np.abs(ref.hess_theta_diag[idx]) + gscale)


def test_posterior_z_small_problem(torch):
    ev = synth.make_events(2500, seed=6, n_centres=8, n_free=150)
    ev.x *= 0.05
    tree = synth.make_tree(ev.t[ev.free_idx], 6)
    z = synth.draw_z(tree, 0.25, 0.1, 6)
    posterior_case(torch, ev, tree, z, 0.25, 0.1, beta=0.001)


def subset_events(n, m, shuffle, seed=61):
    """A dense little problem (ties, duplicated locations) whose sequenced set is an arbitrary subset of m events that
    always holds the first event and, for m >= 2, the last one; shuffle: idx in no particular order."""
    ev = synth.small_random(n, seed=seed, ties=True, duplicates=True)
    ev.x *= np.sqrt(n / 16.0)
    ev.t *= n / 40.0
    rest = np.argsort(synth.uniforms(seed, 700, n), kind="stable")
    rest = rest[(rest != 0) & (rest != n - 1)]
    idx = np.concatenate([[0, n - 1][:min(m, 2)], rest[:max(m - 2, 0)]]).astype(np.int64)
    if not shuffle:
        idx = np.sort(idx)
    ev.free_idx = idx
    return ev


@pytest.mark.parametrize("m,shuffle", [(1, False), (2, True), (97, True), (256, False), (257, True), (750, True), (751, False),
                                       (1500, False)])
def test_posterior_z_source_subsets(torch, m, shuffle):
    """Pass 2 runs over the m sequenced sources only when 2 m <= n (the O(NM) gradient; Alg. 2 step 2), over
    all n otherwise: m = 1, one and two source tiles, a ragged tile, both sides of the switch, m = n; idx sorted and not;
    the subset holds event 0 and event n - 1; ties in time and duplicated locations.  Every output against the oracle."""
    ev = subset_events(1500, m, shuffle)
    tree = synth.make_tree(ev.t[ev.free_idx], 61)
    z = synth.draw_z(tree, 0.25, 0.1, 61)
    posterior_case(torch, ev, tree, z, 0.25, 0.1, beta=0.002)


def test_posterior_z_config2_full_size(torch):
    """BASELINE.json configs[2] at full size: N = 23,422, M = 1,610."""
    ev, tree, z = synth.config_tree(0)
    posterior_case(torch, ev, tree, z, synth.TREE_SIGMA2, synth.TREE_TAU0)
