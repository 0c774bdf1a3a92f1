"""One pass over every kernel family of the library at small sizes, for `compute-sanitizer`:

    compute-sanitizer --tool memcheck  --error-exitcode 9 python tests/sanitizer_run.py
    compute-sanitizer --tool racecheck --error-exitcode 9 python tests/sanitizer_run.py

With the guard-band build (`python -m paper_2103_03348_b200.build --guard`, then HAWKES_B200_GUARD=1) the run ends with
hawkes_debug_guard_check on its contexts.  Not a pytest file (the sanitizers slow every kernel 10-100x, so this is run on demand and its tails are kept in
profiles/r02_sanitizers.md).  It only calls the C ABI through the binding and checks that the results are finite;
parity is the job of the test-suite proper.  Families touched: prep / pass1s (levels 0, 1, masked and plain blocks,
ragged tile) / dense pass 1 (level 2 and PASS1_DENSE) / reduce1 / scalars / pass 2 (factorised and not, levels 0, 1) /
theta / cross pass / dense theta-theta / theta block / S mode / D = 3 / sort / skip plan + list kernels (symmetric
background lists included) / tree prior + precision diagonal / z chain / posterior_z (+ skip) / one HMC iteration of each
of the six variants."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import paper_2103_03348_b200 as hp            # noqa: E402
from paper_2103_03348_b200 import synth       # noqa: E402


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def finite(*tensors):
    for t in tensors:
        if t is not None:
            assert bool(torch.isfinite(t).all()), "non-finite output"


def main():
    n = int(os.environ.get("HAWKES_SANITIZE_N", "1000"))
    ev = synth.config(0) if n == 1000 else synth.make_events(n, seed=0)
    x, t, th = dev(ev.x), dev(ev.t), dev(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim, 0)
    ctx.row_moments_enable(True)
    for want in (hp.WANT_LL, hp.WANT_LL | hp.WANT_GRAD_THETA, hp.WANT_GRAD, hp.WANT_ALL, hp.WANT_HESS_CROSS):
        r = ctx.eval(x, t, th, ev.params, want)
        finite(r.ll, r.grad_theta, r.grad_hyper, r.hess_theta_diag, r.hess_hyper, r.hess_cross)
    d1, d2 = ctx.get_row_moments(ev.n, second=True)
    finite(d1, d2, ctx.get_lambda(ev.n))
    ctx.set_pass1_mode(hp.PASS1_DENSE)
    finite(ctx.grad(x, t, th, ev.params).grad_theta)
    ctx.set_pass1_mode(hp.PASS1_AUTO)
    ctx.set_background_mode(hp.BG_SPACE_ONLY)
    finite(ctx.eval(x, t, th, ev.params, hp.WANT_ALL).hess_cross)
    ctx.set_background_mode(hp.BG_SPACE_TIME)
    # a long time axis: pass 2 keeps the unfactorised exponent
    finite(ctx.eval(x, dev(ev.t * 60.0), th, (0.3, 10.0, 1.0e5, 0.7, 1.0, 1 / 3), hp.WANT_GRAD | hp.WANT_HESS_THETA).grad_theta)
    finite(ctx.hessian_theta_dense(x, t, th, ev.params))
    idx = dev(ev.free_idx.astype(np.int64))
    finite(ctx.hessian_theta_block(x, t, th, ev.params, idx))
    perm = np.argsort(synth.uniforms(5, 5, ev.n), kind="stable")
    finite(*ctx.sort_events(dev(ev.x[:, perm]), dev(ev.t[perm]), dev(ev.theta[perm]))[:3])
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    finite(ctx.eval_host(pin(ev.x), pin(ev.t), pin(ev.theta), ev.params, hp.WANT_GRAD).grad_theta)
    # exact-zero skipping: plan + list kernels at every level, re-plan, shuffled input
    ctx.skip_plan(x, t, ev.params)
    for want in (hp.WANT_LL | hp.WANT_GRAD_THETA, hp.WANT_GRAD, hp.WANT_ALL & ~hp.WANT_HESS_CROSS):
        r = ctx.eval_skip(x, t, th, ev.params, want)
        finite(r.ll, r.grad_theta, r.grad_hyper, r.hess_theta_diag, r.hess_hyper)
    p2 = (0.3, 12.0, 14.0, 0.7, 1.2, 1 / 3)
    ctx.skip_plan(x, t, p2)
    finite(ctx.eval_skip(x, t, th, p2, hp.WANT_GRAD).grad_theta)
    # D = 3
    e3 = synth.small_random(300, 7, dim=3, regime="mixed", ties=True, duplicates=True)
    c3 = hp.HawkesContext(e3.n, 3, 0)
    r = c3.eval(dev(e3.x), dev(e3.t), dev(e3.theta), e3.params, hp.WANT_ALL)
    finite(r.ll, r.grad_theta, r.hess_cross)
    # tree prior, z-parametrisation, posterior, HMC (one iteration per variant)
    m = len(ev.free_idx)
    tree = synth.make_tree(ev.t[ev.free_idx], 0)
    z0 = synth.draw_z(tree, 0.25, 0.1, 0)
    tr = hp.HawkesTree(tree.parent, tree.branch, 0)
    zd = dev(z0)
    finite(*tr.prior(zd, 0.25, 0.1))
    pp = tr.precision_diag(0.25, 0.1)
    finite(pp)
    theta = ctx.theta_from_z(ev.n, idx, zd, 0.001, t)
    g = ctx.grad(x, t, theta, ev.params)
    h = ctx.hessian(x, t, theta, ev.params)
    finite(*[a for a in ctx.z_chain(idx, theta, t, g.grad_theta, h.hess_theta_diag, want_beta=True)])
    finite(*ctx.posterior_z(tr, x, t, idx, zd, 0.0, ev.params, 0.25, 0.1, hess=True))
    ctx.skip_plan(x, t, ev.params)
    finite(*ctx.posterior_z(tr, x, t, idx, zd, 0.0, ev.params, 0.25, 0.1, hess=True, skip=True))
    nrm = dev(synth.normals(0, 500, 2 * m).reshape(2, m))
    uni = dev(synth.uniforms(0, 501, 2))
    for variant in range(6):
        z, mass = dev(z0.copy()), dev(np.ones(m))
        trace = ctx.hmc_run(tr, x, t, idx, z, 0.0, ev.params, 0.25, 0.1, n_iter=2, n_leapfrog=3, step=0.1,
                            precond_every=1, mass=mass, mass_floor=0.5, normals=nrm, uniforms=uni,
                            cache_background=variant, prior_prec=pp)
        finite(trace, z, mass)
    torch.cuda.synchronize()
    assert ctx.last_status() == 0
    if os.environ.get("HAWKES_B200_GUARD") == "1":     # the guard-band build: no scratch buffer was overrun
        bad = ctx.debug_guard_check() + c3.debug_guard_check()
        assert bad == 0, f"{bad} guard-band bytes overwritten"
        print("guard bands intact: 0 bytes overwritten around the scratch buffers of both contexts")
    print("sanitizer_run ok: n=%d, %d + %d launches" % (ev.n, ctx.launch_count() + c3.launch_count(), tr.launch_count()))


if __name__ == "__main__":
    main()
