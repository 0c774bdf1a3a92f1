"""GPU parity of the exact-zero-skipping variant (hawkes_skip_plan + hawkes_eval_skip) against the
oracle, element by element, at the tolerance of the dense path (1e-10 relative, tests/parity.py).  The oracle knows
nothing of tiles, orders or lists: it sums every pair of Eq. 1 / Eq. 4."""
import math
import os

import numpy as np
import pytest

import oracle
import paper_2103_03348_b200 as hp
from paper_2103_03348_b200 import synth
from parity import TOL, check, hess_hyper_scale, scales

pytestmark = pytest.mark.gpu
THREADS = max(1, min(os.cpu_count() or 1, 64))
WANT = hp.WANT_LL | hp.WANT_GRAD_THETA | hp.WANT_GRAD_HYPER | hp.WANT_HESS_THETA | hp.WANT_HESS_HYPER


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def run_skip(torch, ev, want=WANT, order=None, ctx=None):
    """Evaluate through the skip variant; `order` presents the events to the library in that (unsorted) order and
    the per-event outputs are brought back to the order of `ev`."""
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    o = np.arange(ev.n) if order is None else order
    x, t, th = f(ev.x[:, o]), f(ev.t[o]), f(ev.theta[o])
    ctx = ctx or hp.HawkesContext(ev.n, ev.dim)
    stats = ctx.skip_plan(x, t, ev.params)
    r = ctx.eval_skip(x, t, th, ev.params, want)
    st = ctx.last_status()
    lam_rec = ctx.get_lambda(ev.n).cpu().numpy()          # in record (k-d tree) order
    perm = ctx.skip_perm(ev.n).numpy()
    assert np.array_equal(np.sort(perm), np.arange(ev.n))
    lam = np.empty(ev.n)
    lam[o[perm]] = lam_rec
    back = lambda v: None if v is None else _unpermute(v.cpu().numpy(), o)
    return r, st, lam, back(r.grad_theta), back(r.hess_theta_diag), stats, ctx


def _unpermute(v, o):
    out = np.empty_like(v)
    out[o] = v
    return out


def zero_rates_agree(lam, lam_ref):
    """Rates the oracle holds above the subnormal range agree to TOL; where it holds a subnormal or zero, the GPU
    (which flushes terms below 2^-1020, reading B15) holds nothing larger."""
    ok = lam_ref > 1e-290
    assert np.max(np.abs(lam[ok] - lam_ref[ok]) / lam_ref[ok]) <= TOL
    assert np.all(lam[~ok] <= 1e-290)


def compare(ev, ref, r, lam, g, hd):
    s = scales(ev, ref)
    check("lambda", lam, ref.lam)
    check("ll", r.ll.cpu().numpy()[0], ref.ll, s["ll"])
    check("grad_theta", g, ref.grad_theta, s["grad_theta"])
    assert np.max(np.abs(g - ref.grad_theta)) <= TOL * np.max(np.abs(ref.grad_theta))
    check("grad_hyper", r.grad_hyper.cpu().numpy(), ref.grad_hyper, s["grad_hyper"])
    check("hess_theta_diag", hd, ref.hess_theta_diag, floor=1e-280)
    H = r.hess_hyper.cpu().numpy()
    assert np.array_equal(H, H.T)
    check("hess_hyper", H, ref.hess_hyper, hess_hyper_scale(ref.hess_hyper))


@pytest.mark.parametrize("n,seed,dim,regime,ties,dup,spread", [
    (2, 1, 2, "mixed", False, False, 1.0), (3, 2, 2, "excite", False, False, 1.0),
    (129, 4, 2, "mixed", False, False, 1.0), (257, 5, 2, "background", True, False, 16.0),
    (300, 6, 1, "mixed", False, True, 300.0), (300, 7, 3, "excite", True, True, 16.0),
    (777, 8, 2, "mixed", True, True, 16.0), (1500, 9, 3, "mixed", False, False, 4.0),
    (2100, 10, 2, "mixed", True, True, 8.0), (777, 8, 2, "mixed", True, True, 60.0)])
def test_skip_small_problems_shuffled_input(torch, n, seed, dim, regime, ties, dup, spread):
    """One thread to several tiles with ragged tails; D = 1, 2, 3; ties and duplicated locations; the events handed
    over in a shuffled order (this variant does not need them sorted); `spread` stretches space and time so that
    boxes really fall outside the cut-off radii."""
    ev = synth.small_random(n, seed, dim=dim, regime=regime, ties=ties, duplicates=dup)
    if n > 64:
        ev.x *= math.sqrt(n / 16.0) * spread
        ev.t *= n / 40.0
    ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS)
    order = np.argsort(synth.uniforms(seed, 77, n), kind="stable")
    r, st, lam, g, hd, stats, ctx = run_skip(torch, ev, order=order)
    assert st == ref.status
    if ref.status == 0:
        compare(ev, ref, r, lam, g, hd)
        # the gradient level and the likelihood level take the background once per unordered pair (another kernel):
        # same oracle values
        s = scales(ev, ref)
        for want in (hp.WANT_GRAD, hp.WANT_LL | hp.WANT_GRAD_THETA):
            r1, st1, lam1, g1, _, stats1, _ = run_skip(torch, ev, want=want, order=order, ctx=ctx)
            assert st1 == 0 and stats1["items_background_unordered"] > 0 and stats1["order_reused"] == 1
            check("lambda", lam1, ref.lam)
            check("ll", r1.ll.cpu().numpy()[0], ref.ll, s["ll"])
            check("grad_theta", g1, ref.grad_theta, s["grad_theta"])
            if want & hp.WANT_GRAD_HYPER:
                check("grad_hyper", r1.grad_hyper.cpu().numpy(), ref.grad_hyper, s["grad_hyper"])
    else:   # (last case) some lambda_n is exactly zero in the oracle as well: ll = -inf on both sides
        assert r.ll.item() == ref.ll == -math.inf
        zero_rates_agree(lam, ref.lam)


def test_skip_n1_and_empty_pass2(torch):
    """N = 1: lambda_1 = 0 (reading B14), the pass-2 list is empty."""
    ev = synth.small_random(1, 3)
    ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=1)
    r, st, lam, g, hd, stats, _ = run_skip(torch, ev)
    assert stats["items_pass2"] == 0
    assert st == ref.status != 0 and r.ll.item() == -math.inf
    assert abs(g[0] - ref.grad_theta[0]) <= TOL * abs(ref.grad_theta[0]) and hd[0] == 0.0


def test_skip_config0_really_skips_and_matches(torch):
    """BASELINE.json configs[0] (N = 1,000): at its scales part of the tile pairs hold exact zeros only; with a
    shorter background length scale most do.  All outputs against the oracle in both settings."""
    ev = synth.config(0)
    ev0_params = ev.params
    for params in (ev0_params, (0.3, 2.0, 14.0, 0.7, 0.5, 1.0 / 3.0)):
        ev.params = params
        ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS)
        r, st, lam, g, hd, stats, _ = run_skip(torch, ev)
        assert st == ref.status
        assert stats["items_excitation"] < stats["items_dense_pass1"] and stats["items_pass2"] < stats["items_dense_pass2"]
        if params is not ev0_params:     # four tiles of 256 events: the background's 386 km reach spans them all
            assert stats["items_background"] < stats["items_dense_pass1"]
        if ref.status == 0:
            compare(ev, ref, r, lam, g, hd)
        else:
            zero_rates_agree(lam, ref.lam)


def test_skip_long_time_axis(torch):
    """A record ten times longer than the temporal cut-offs: boxes separate in time as well as in space."""
    ev = synth.config(0)
    ev.t = ev.t * 40.0
    ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS)
    r, st, lam, g, hd, stats, _ = run_skip(torch, ev)
    assert st == ref.status
    assert stats["items_background"] < stats["items_dense_pass1"]
    if ref.status == 0:
        compare(ev, ref, r, lam, g, hd)
    else:
        zero_rates_agree(lam, ref.lam)


def test_skip_space_only_background(torch):
    """Paper-literal S mode through the lists."""
    ev = synth.config(0)
    ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS, bg="S")
    ctx = hp.HawkesContext(ev.n, ev.dim)
    ctx.set_background_mode(hp.BG_SPACE_ONLY)
    r, st, lam, g, hd, stats, _ = run_skip(torch, ev, ctx=ctx)
    assert st == ref.status == 0
    compare(ev, ref, r, lam, g, hd)
    r1, st1, lam1, g1, _, stats1, _ = run_skip(torch, ev, want=hp.WANT_GRAD, ctx=ctx)   # symmetric background lists
    assert st1 == 0 and stats1["items_background_unordered"] > 0
    s = scales(ev, ref)
    check("lambda", lam1, ref.lam)
    check("ll", r1.ll.cpu().numpy()[0], ref.ll, s["ll"])
    check("grad_theta", g1, ref.grad_theta, s["grad_theta"])
    check("grad_hyper", r1.grad_hyper.cpu().numpy(), ref.grad_hyper, s["grad_hyper"])


def test_skip_full_size_against_dense_gpu_and_sampled_oracle(torch):
    """BASELINE.json configs[1] (N = 23,422) in the launch configuration bench.py times: every output against the dense
    CUDA path (summation order is the only difference), and 192 sampled rows / columns against the oracle."""
    ev = synth.config(1)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    x, t, th = f(ev.x), f(ev.t), f(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    stats = ctx.skip_plan(x, t, ev.params)
    assert stats["items_background"] < 0.8 * stats["items_dense_pass1"]
    assert stats["items_excitation"] < 0.3 * stats["items_dense_pass1"]
    rs = ctx.eval_skip(x, t, th, ev.params, WANT)
    assert ctx.last_status() == 0
    lam_rec = ctx.get_lambda(ev.n).cpu().numpy()
    perm = ctx.skip_perm(ev.n).numpy()
    lam = np.empty(ev.n)
    lam[perm] = lam_rec
    rd = ctx.eval(x, t, th, ev.params, WANT)
    assert ctx.last_status() == 0
    torch.cuda.synchronize()
    for name in ("ll", "grad_theta", "grad_hyper", "hess_theta_diag", "hess_hyper"):
        a, b = getattr(rs, name).cpu().numpy(), getattr(rd, name).cpu().numpy()
        assert np.max(np.abs(a - b)) <= 1e-12 * np.max(np.abs(b)), name
    idx = np.unique(np.concatenate([np.arange(0, ev.n, 123), [ev.n - 1]]))
    lam_ref, _ = oracle.rows(ev.x, ev.t, ev.theta, ev.params, idx, derivs=False, threads=THREADS)
    assert np.max(np.abs(lam[idx] - lam_ref) / lam_ref) <= TOL
    c_ref, d_ref = oracle.cols(ev.x, ev.t, ev.params, lam, idx, threads=THREADS)
    xi0, om = ev.params[3], ev.params[5]
    integ = xi0 * (-np.expm1(-om * (ev.t[-1] - ev.t[idx])))
    g = rs.grad_theta.cpu().numpy()[idx]
    assert np.max(np.abs(g - (c_ref - integ)) / np.maximum(np.abs(c_ref) + integ, 1e-300)) <= TOL
    hd = rs.hess_theta_diag.cpu().numpy()[idx]
    assert np.max(np.abs(hd + d_ref) / np.maximum(d_ref, 1e-280)) <= TOL


def test_skip_plan_is_checked(torch):
    """No plan, or a plan for other hyperparameters / another n: HAWKES_ERR_ARG, nothing is launched."""
    ev = synth.config(0)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    x, t, th = f(ev.x), f(ev.t), f(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    with pytest.raises(hp.HawkesError):
        ctx.eval_skip(x, t, th, ev.params)
    ctx.skip_plan(x, t, ev.params)
    ctx.eval_skip(x, t, th, ev.params)
    other = tuple(ev.params[:4]) + (ev.params[4] * 1.01, ev.params[5])
    with pytest.raises(hp.HawkesError):
        ctx.eval_skip(x, t, th, other)
    with pytest.raises(hp.HawkesError):
        ctx.eval_skip(x[:, :500].contiguous(), t[:500].contiguous(), th[:500].contiguous(), ev.params)
    ctx.skip_plan(x, t, other)               # re-planning replaces the plan
    ctx.eval_skip(x, t, th, other)
    assert ctx.last_status() == 0


def test_skip_replan_keeps_order_for_nearby_hyperparameters(torch):
    """An MCMC sweep re-plans the same events for new hyperparameters: the order and boxes are kept while the cut-off
    radii stay within a factor 2, rebuilt otherwise or for other events; results match the oracle either way."""
    ev = synth.config(0)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    x, t, th = f(ev.x), f(ev.t), f(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    assert ctx.skip_plan(x, t, ev.params)["order_reused"] == 0
    perm0 = ctx.skip_perm(ev.n).numpy().copy()
    near = (0.35, 12.0, 11.0, 0.6, 1.3, 0.4)
    far = (0.35, 2.0, 11.0, 0.6, 0.2, 0.4)
    for params, reused in ((near, 1), (far, 0), (far, 1)):
        st = ctx.skip_plan(x, t, params)
        assert st["order_reused"] == reused
        if params is near:
            assert np.array_equal(ctx.skip_perm(ev.n).numpy(), perm0)
        ev.params = params
        ref = oracle.evaluate(ev.x, ev.t, ev.theta, ev.params, hess=True, row_d1=True, threads=THREADS)
        r = ctx.eval_skip(x, t, th, params, WANT)
        assert ctx.last_status() == ref.status
        if ref.status == 0:
            lam = np.empty(ev.n)
            lam[ctx.skip_perm(ev.n).numpy()] = ctx.get_lambda(ev.n).cpu().numpy()
            compare(ev, ref, r, lam, r.grad_theta.cpu().numpy(), r.hess_theta_diag.cpu().numpy())
    x2 = x.clone()
    x2[0, 0] += 1.0
    assert ctx.skip_plan(x2, t, far)["order_reused"] == 0        # other events: a fresh order


def test_skip_rejects_bad_data(torch):
    """Non-finite events are refused when planning (host check); a negative or non-finite theta is a device status
    of the evaluation, as in the dense path."""
    ev = synth.config(0)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    x, t, th = f(ev.x), f(ev.t), f(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    xb = x.clone()
    xb[1, 17] = float("nan")
    with pytest.raises(hp.HawkesError):
        ctx.skip_plan(xb, t, ev.params)
    tb = t.clone()
    tb[3] = float("inf")
    with pytest.raises(hp.HawkesError):
        ctx.skip_plan(x, tb, ev.params)
    with pytest.raises(hp.HawkesError):
        ctx.skip_plan(x, t, ev.params[:4] + (-1.0,) + ev.params[5:])
    ctx.skip_plan(x, t, ev.params)
    thb = th.clone()
    thb[5] = -0.5
    ctx.eval_skip(x, t, thb, ev.params)
    assert ctx.last_status() == hp.ERR_NONFINITE
    ctx.eval_skip(x, t, th, ev.params)
    assert ctx.last_status() == 0


@pytest.mark.parametrize("n", [50000, 250000])
def test_skip_scaling_sweep_sampled_rows_and_columns(torch, n):
    """BASELINE.json configs[4] sizes through the lists: 1,024 sampled target rows (lambda_n) and, with the GPU's
    lambda, 1,024 source columns (c_m, d_m) against the oracle; properties that hold at any size."""
    ev = synth.config(4, n=n)
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to("cuda")
    x, t, th = f(ev.x), f(ev.t), f(ev.theta)
    ctx = hp.HawkesContext(ev.n, ev.dim)
    stats = ctx.skip_plan(x, t, ev.params)
    assert stats["items_background"] < 0.6 * stats["items_dense_pass1"]
    assert stats["items_pass2"] < 0.1 * stats["items_dense_pass2"]
    r = ctx.eval_skip(x, t, th, ev.params, hp.WANT_GRAD | hp.WANT_HESS_THETA)
    assert ctx.last_status() == 0
    lam = np.empty(ev.n)
    lam[ctx.skip_perm(ev.n).numpy()] = ctx.get_lambda(ev.n).cpu().numpy()
    k = 1024
    idx = np.sort((synth.uniforms(123, 7, k) * n).astype(np.int64))
    idx[0], idx[-1] = 0, n - 1
    lam_o, _ = oracle.rows(ev.x, ev.t, ev.theta, ev.params, idx, derivs=False, threads=THREADS)
    check("lambda rows", lam[idx], lam_o)
    c_o, d_o = oracle.cols(ev.x, ev.t, ev.params, lam, idx, threads=THREADS)
    xi0, om = ev.params[3], ev.params[5]
    integ = xi0 * (-np.expm1(-om * (ev.t[-1] - ev.t[idx])))
    gt = r.grad_theta.cpu().numpy()
    hd = r.hess_theta_diag.cpu().numpy()
    check("grad_theta cols", gt[idx], c_o - integ, np.abs(c_o) + integ)
    check("hess_theta cols", hd[idx], -d_o, floor=1e-280)
    assert gt[-1] == 0.0 and np.all(np.isfinite(gt)) and np.all(hd <= 0)
    assert np.all(lam > 0) and math.isfinite(r.ll.item())
