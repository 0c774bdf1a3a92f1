"""GPU parity of hawkes_hmc_run (include/hawkes.h) against the HMC oracle (oracle/hmc.py) driven by the likelihood
and prior oracles, on the same seeded inputs and the same random numbers."""
import os

import numpy as np
import pytest

from oracle import hmc as ohmc
from oracle import tree as otree
from paper_2103_03348_b200 import synth

pytestmark = pytest.mark.gpu
THREADS = min(os.cpu_count() or 1, 32)


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


@pytest.mark.parametrize("cache_bg,with_prior_prec", [(0, False), (1, False), (1, True), (2, False), (2, True),
                                                      (3, False), (4, False), (4, True), (5, False), (5, True)])
def test_hmc_matches_oracle_trajectory(torch, cache_bg, with_prior_prec):
    """1,500 events, 90 sequenced; 6 iterations x 5 leapfrog steps, preconditioner refreshed every 3 iterations.
    Tolerance: the state after 30 leapfrog steps inherits the 1e-10 bar of the gradient through a mildly expanding
    map; 1e-8 relative to the scale of z and of the energies leaves two orders of margin (measured ~1e-12)."""
    import paper_2103_03348_b200 as hp
    ev = synth.make_events(1500, seed=12, n_centres=6, n_free=90)
    ev.x *= 0.05
    idx = ev.free_idx
    M = len(idx)
    tree = synth.make_tree(ev.t[idx], 12)
    s2, tau0, beta = 0.25, 0.1, 0.0005
    z0 = synth.draw_z(tree, s2, tau0, 12)
    n_iter, L, eps, every, floor = 6, 5, 0.04, 3, 0.5
    normals = synth.normals(12, 400, n_iter * M).reshape(n_iter, M)
    uniforms = synth.uniforms(12, 401, n_iter)
    uniforms[1] = 1.0      # forces a comparison log(1) = 0 < H_old - H_new: rejects whenever the energy went up
    mass0 = np.ones(M)
    V = otree.vg(tree.parent, tree.branch, M, tau0)
    target = ohmc.hawkes_target(ev.x, ev.t, idx, beta, ev.params, V, s2, threads=THREADS)
    pp = otree.precision_diag(V, s2) if with_prior_prec else None
    if with_prior_prec:
        eps = 0.3          # the preconditioned dynamics take a far larger step
    ref = ohmc.run(target, z0, normals, uniforms, n_iter, L, eps, every, mass0, floor, prior_prec=pp)

    ctx = hp.HawkesContext(ev.n, ev.dim, 0)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    z = dev(torch, z0.copy())
    mass = dev(torch, mass0.copy())
    pp_d = tr.precision_diag(s2, tau0) if with_prior_prec else None
    if with_prior_prec:
        assert np.max(np.abs(pp_d.cpu().numpy() - pp) / pp) <= 1e-10
    if cache_bg in (3, 4):     # variants 0 / 1 over the work lists of hawkes_skip_plan (exact zeros left out)
        with pytest.raises(hp.HawkesError):
            ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z.clone(), beta, ev.params, s2, tau0,
                        n_iter=1, n_leapfrog=1, step=eps, precond_every=0, mass=mass.clone(), mass_floor=floor,
                        normals=dev(torch, normals[:1]), uniforms=dev(torch, uniforms[:1]), cache_background=cache_bg)
        stats = ctx.skip_plan(dev(torch, ev.x), dev(torch, ev.t), ev.params)
        assert stats["items_excitation"] < stats["items_dense_pass1"]
    trace = ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z, beta, ev.params, s2, tau0,
                        n_iter=n_iter, n_leapfrog=L, step=eps, precond_every=every, mass=mass, mass_floor=floor,
                        normals=dev(torch, normals), uniforms=dev(torch, uniforms), cache_background=cache_bg,
                        prior_prec=pp_d)
    torch.cuda.synchronize()
    assert ctx.last_status() == 0
    trace = trace.cpu().numpy()
    assert np.array_equal(trace[:, 3], ref["trace"][:, 3]), (trace[:, 3], ref["trace"][:, 3])
    assert 0 < ref["trace"][:, 3].sum()                     # the case exercises accepted proposals ...
    escale = np.max(np.abs(ref["trace"][:, 1:3]))
    assert np.max(np.abs(trace[:, :3] - ref["trace"][:, :3])) <= 1e-8 * escale
    assert np.max(np.abs(z.cpu().numpy() - ref["z"])) <= 1e-8 * np.max(np.abs(ref["z"]))
    assert np.max(np.abs(mass.cpu().numpy() - ref["mass"]) / ref["mass"]) <= 1e-8
    # the call replays captured CUDA graphs (one host launch per iteration); enqueuing every kernel directly
    # (HAWKES_HMC_NO_GRAPH) runs the same kernels in the same order: bit-identical state, preconditioner and trace
    # (a kind of iteration -- with / without a preconditioner refresh -- that the call runs fewer than 3 times is enqueued
    # directly: here the 2 refresh iterations, so 4 of the 6 iterations are graph launches)
    n_refresh = -(-n_iter // every)
    n_graph = sum(k for k in (n_refresh, n_iter - n_refresh) if k >= 3)
    assert ctx.graph_launch_count() == n_graph == 4
    z2, mass2 = dev(torch, z0.copy()), dev(torch, mass0.copy())
    l0 = ctx.launch_count()
    trace2 = ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z2, beta, ev.params, s2, tau0,
                         n_iter=n_iter, n_leapfrog=L, step=eps, precond_every=every, mass=mass2, mass_floor=floor,
                         normals=dev(torch, normals), uniforms=dev(torch, uniforms), cache_background=cache_bg,
                         prior_prec=pp_d, graph=False)
    torch.cuda.synchronize()
    assert ctx.graph_launch_count() == n_graph
    assert torch.equal(z2, z) and torch.equal(mass2, mass) and np.array_equal(trace2.cpu().numpy(), trace)
    # ... and the launch bookkeeping counts the replayed kernels: a second graph run adds as many as the direct run did
    direct = ctx.launch_count() - l0
    z3, mass3 = dev(torch, z0.copy()), dev(torch, mass0.copy())
    l1 = ctx.launch_count()
    ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z3, beta, ev.params, s2, tau0,
                n_iter=n_iter, n_leapfrog=L, step=eps, precond_every=every, mass=mass3, mass_floor=floor,
                normals=dev(torch, normals), uniforms=dev(torch, uniforms), cache_background=cache_bg, prior_prec=pp_d)
    torch.cuda.synchronize()
    assert ctx.launch_count() - l1 == direct
    assert torch.equal(z3, z)
    # with the timing ring on nothing is captured (its event records would be frozen into the graph): same results, no
    # graph launch, and the ring has seen every evaluation of the call -- the first, 5 per iteration, one per refresh
    if cache_bg == 0:
        g0 = ctx.graph_launch_count()
        ctx.profile_enable(True)
        z4, mass4 = dev(torch, z0.copy()), dev(torch, mass0.copy())
        ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z4, beta, ev.params, s2, tau0,
                    n_iter=n_iter, n_leapfrog=L, step=eps, precond_every=every, mass=mass4, mass_floor=floor,
                    normals=dev(torch, normals), uniforms=dev(torch, uniforms), cache_background=cache_bg, prior_prec=pp_d)
        torch.cuda.synchronize()
        prof = ctx.profile_read()
        ctx.profile_enable(False)
        assert ctx.graph_launch_count() == g0 and torch.equal(z4, z)
        assert prof["evals"] == 1 + n_iter * L + n_refresh and prof["pass1_ms"] > 0


def test_hmc_full_size_single_iteration(torch):
    """BASELINE.json configs[3] inputs (N = 23,422, M = 1,610): one iteration of hawkes_hmc_run -- a preconditioner
    refresh, the momentum draw, 6 leapfrog steps, the accept test -- against oracle/hmc.py on the full likelihood
    oracle and the dense Cholesky prior oracle (8 oracle evaluations), with the paper's preconditioner
    (prior_prec = NULL) and the recompute-every-pair variant bench.py reports as the headline."""
    import paper_2103_03348_b200 as hp
    ev, tree, z0 = synth.config_tree(0)
    idx = ev.free_idx
    M = len(idx)
    s2, tau0 = synth.TREE_SIGMA2, synth.TREE_TAU0
    n_iter, L, eps, every, floor = 1, 6, 0.01, 1, 1.0
    normals = synth.normals(0, 500, n_iter * M).reshape(n_iter, M)
    uniforms = synth.uniforms(0, 501, n_iter)
    V = otree.vg(tree.parent, tree.branch, M, tau0)
    target = ohmc.hawkes_target(ev.x, ev.t, idx, 0.0, ev.params, V, s2, threads=THREADS)
    ref = ohmc.run(target, z0, normals, uniforms, n_iter, L, eps, every, np.ones(M), floor)
    ctx = hp.HawkesContext(ev.n, ev.dim, 0)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    z, mass = dev(torch, z0.copy()), dev(torch, np.ones(M))
    trace = ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z, 0.0, ev.params, s2, tau0,
                        n_iter=n_iter, n_leapfrog=L, step=eps, precond_every=every, mass=mass, mass_floor=floor,
                        normals=dev(torch, normals), uniforms=dev(torch, uniforms), cache_background=0)
    torch.cuda.synchronize()
    assert ctx.last_status() == 0
    trace = trace.cpu().numpy()
    assert np.array_equal(trace[:, 3], ref["trace"][:, 3])
    escale = np.max(np.abs(ref["trace"][:, 1:3]))
    assert np.max(np.abs(trace[:, :3] - ref["trace"][:, :3])) <= 1e-8 * escale
    assert np.max(np.abs(z.cpu().numpy() - ref["z"])) <= 1e-8 * np.max(np.abs(ref["z"]))
    assert np.max(np.abs(mass.cpu().numpy() - ref["mass"]) / ref["mass"]) <= 1e-8


def test_hmc_rejects_bad_options(torch):
    import paper_2103_03348_b200 as hp
    ev = synth.make_events(300, seed=3, n_centres=3, n_free=20)
    idx = ev.free_idx
    M = len(idx)
    tree = synth.make_tree(ev.t[idx], 3)
    ctx = hp.HawkesContext(ev.n, ev.dim, 0)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    args = (tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), dev(torch, np.zeros(M)), 0.0, ev.params, 0.25, 0.1)
    kw = dict(n_iter=2, n_leapfrog=2, step=0.1, precond_every=1, mass=dev(torch, np.ones(M)), mass_floor=0.1,
              normals=dev(torch, np.zeros((2, M))), uniforms=dev(torch, np.full(2, 0.5)))
    for bad in (dict(step=0.0), dict(step=float("nan")), dict(mass_floor=0.0)):
        with pytest.raises(hp.HawkesError) as e:
            ctx.hmc_run(*args, **{**kw, **bad})
        assert e.value.status == hp.ERR_PARAM
    with pytest.raises(hp.HawkesError) as e:
        ctx.hmc_run(*args, **{**kw, "n_leapfrog": 0})
    assert e.value.status == hp.ERR_ARG


def test_hmc_sparse_kernel_matrix_edge_cases(torch):
    """Variant 5 against variant 2 (the dense cached kernel matrix, itself checked against the oracle above) where
    the compression is degenerate: a self-excitation reach so short that K has no non-zero at all, and a second call
    on the same context (buffers kept from the first)."""
    import paper_2103_03348_b200 as hp
    ev = synth.make_events(1200, seed=21, n_centres=5, n_free=64)
    idx = ev.free_idx
    M = len(idx)
    tree = synth.make_tree(ev.t[idx], 21)
    s2, tau0 = 0.25, 0.1
    z0 = synth.draw_z(tree, s2, tau0, 21)
    n_iter, L = 3, 4
    normals = synth.normals(21, 400, n_iter * M).reshape(n_iter, M)
    uniforms = synth.uniforms(21, 401, n_iter)
    ctx = hp.HawkesContext(ev.n, ev.dim, 0)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    pp = tr.precision_diag(s2, tau0)
    for params in (ev.params[:4] + (1e-4,) + ev.params[5:], ev.params):
        out = {}
        for variant in (2, 5):
            z, mass = dev(torch, z0.copy()), dev(torch, np.ones(M))
            trace = ctx.hmc_run(tr, dev(torch, ev.x), dev(torch, ev.t), dev(torch, idx), z, 0.0, params, s2, tau0,
                                n_iter=n_iter, n_leapfrog=L, step=0.2, precond_every=2, mass=mass, mass_floor=0.5,
                                normals=dev(torch, normals), uniforms=dev(torch, uniforms), cache_background=variant,
                                prior_prec=pp)
            torch.cuda.synchronize()
            out[variant] = (ctx.last_status(), trace.cpu().numpy(), z.cpu().numpy(), mass.cpu().numpy())
        assert out[2][0] == out[5][0] == 0
        for a, b in zip(out[2][1:], out[5][1:]):
            assert np.max(np.abs(a - b)) <= 1e-11 * max(np.max(np.abs(a)), 1.0)
